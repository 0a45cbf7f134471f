// dc_narrow.cuh -- S5 (narrow phase) and S6 (decide) as a short sequence of uniform kernels over global queues.
//
// Every kernel does one kind of operation and compacts its output into a global queue (warp-aggregated
// atomics), so warps stay full and no kernel carries another's registers:
//
//   k_np_stage      thread / (element, patch) : monomial coefficients and Bezier box of a boundary patch -> ecoef, pbox
//                                         (best[b] = reach and the seed item come from k_pairs)
//   k_np_solve      thread / leaf       : projected Newton (Eq. 3-5 L256-L270 generalised to two patches, clamp
//                                         L272-L278), both patches' coefficients in registers; a pass hands its
//                                         stragglers to the next pass through a continuation queue; min into best /
//                                         dmin / pair_key; the sub-leaves of an unconverged leaf go to an overflow queue
//   k_np_roots      thread / pair       : (pair, patch) whose boxes are within best + t_tie (A.2, L689-L709)
//                                         become the items of round 0
//   k_np_bound      thread / item       : bound_node -> prune / 4 children / leaf (+ the leaf's starting point and
//                                         lower bound); <ROOT> for round 0
//   k_np_bound_tail one CTA             : the sparse late rounds, until one comes up empty
//   k_np_compact    thread / leaf       : drops the leaves whose lower bound the element's best distance has passed
//   k_np_decide     thread / band elem  : S6 (L215 nearest face and its normal; tie rule L294)
//
// Launch order (dc_classify): stage, solve(seeds), roots, bound<ROOT>, bound x 3, bound_tail, compact, solve(leaves),
// solve(continuations) x 2, [bound(overflow), solve] x 2, decide.  Every item of bound round r has lP + lQ = r, so
// 2 max_level + 1 rounds always terminate the branch and bound.
#pragma once

#define NPW_THREADS 128
#define DC_STATUS_INVALID (DC_STATUS_PAIR_OVERFLOW | DC_STATUS_QUEUE_OVERFLOW | DC_STATUS_BAND_OVERFLOW)
#define DC_MAX_ROUNDS 25            /* 2 * 12 + 1 */


// what a leaf carries beside its item (16 bytes): the starting point of its solve (the first step k_np_bound took from
// the centre, local coordinates in [-1,1] as 16-bit fixed point: +-32767 = on the bound) and its lower bound (the solve
// is skipped when the element's best distance has dropped below it by the time a lane picks it up)
struct __align__(16) NLeafX { short x[4]; double lb; };

struct NpCounters { unsigned nodes, newton, iters, fail, depth; };

__device__ __forceinline__ double u2d(unsigned long long b) { return __longlong_as_double((long long)b); }
__device__ __forceinline__ unsigned long long d2u(double d) { return (unsigned long long)__double_as_longlong(d); }

__device__ __forceinline__ void nitem_box(const NItem &it, double &uc, double &vc, double &hP,
                                          double &sc, double &tc, double &hQ)
{
    const int lP = it.w2 & 15, lQ = (it.w2 >> 4) & 15;
    const int iu = (it.w2 >> 8) & 0xfff, iv = (it.w2 >> 20) & 0xfff;
    const int is = it.w3 & 0xfff, itt = (it.w3 >> 12) & 0xfff;
    hP = __longlong_as_double((long long)(1023 - lP) << 52);
    hQ = __longlong_as_double((long long)(1023 - lQ) << 52);
    uc = fma((double)(2 * iu + 1), hP, -1.0); vc = fma((double)(2 * iv + 1), hP, -1.0);
    sc = fma((double)(2 * is + 1), hQ, -1.0); tc = fma((double)(2 * itt + 1), hQ, -1.0);
}

__device__ __forceinline__ NItem nitem_child(const NItem &it, bool splitP, int c)
{
    const unsigned lP = it.w2 & 15, lQ = (it.w2 >> 4) & 15;
    const unsigned iu = (it.w2 >> 8) & 0xfff, iv = (it.w2 >> 20) & 0xfff;
    const unsigned is = it.w3 & 0xfff, itt = (it.w3 >> 12) & 0xfff;
    NItem ch; ch.p = it.p; ch.ak = it.ak;
    if (splitP) {
        ch.w2 = (lP + 1) | (lQ << 4) | ((2 * iu + (c & 1)) << 8) | ((2 * iv + (c >> 1)) << 20);
        ch.w3 = it.w3 & 0x00ffffffu;
    } else {
        ch.w2 = lP | ((lQ + 1) << 4) | (iu << 8) | (iv << 20);
        ch.w3 = (2 * is + (c & 1)) | ((2 * itt + (c >> 1)) << 12);
    }
    return ch;
}

// choose which patch a node splits (never beyond max_level); false = nothing left to split
__device__ __forceinline__ bool choose_split(const NItem &it, bool wantP, int max_level, bool &splitP)
{
    const int lP = it.w2 & 15, lQ = (it.w2 >> 4) & 15;
    splitP = wantP;
    if (splitP && lP >= max_level) splitP = false;
    if (!splitP && lQ >= max_level) {
        if (lP < max_level) splitP = true;
        else return false;
    }
    return true;
}

// warp-aggregated append of `n_mine` (0 or `per`) items per lane; returns this lane's first slot or -1
__device__ __forceinline__ long long warp_reserve(int *counter, bool mine, int per, long long cap, int *status)
{
    const unsigned m = __ballot_sync(0xffffffffu, mine);
    if (!m) return -1;
    const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(counter, __popc(m) * per);
    base = __shfl_sync(0xffffffffu, base, leader);
    if (!mine) return -1;
    const long long slot = (long long)base + (long long)__popc(m & ((1u << lane) - 1)) * per;
    if (slot + per > cap) { atomicOr(status, DC_STATUS_QUEUE_OVERFLOW); return -1; }
    return slot;
}

__device__ __forceinline__ void np_flush_counters(DcScalars *S, const NpCounters &c)
{
    unsigned v[5] = { c.nodes, c.newton, c.iters, c.fail, c.depth };
#pragma unroll
    for (int i = 0; i < 5; ++i)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], o);
    if ((threadIdx.x & 31) == 0) {
        if (v[0]) atomicAdd(&S->c_bnb_nodes, (unsigned long long)v[0]);
        if (v[1]) atomicAdd(&S->c_newton, (unsigned long long)v[1]);
        if (v[2]) atomicAdd(&S->c_newton_iters, (unsigned long long)v[2]);
        if (v[3]) atomicAdd(&S->c_newton_fail, (unsigned long long)v[3]);
        if (v[4]) atomicAdd(&S->c_depth_exceeded, (unsigned long long)v[4]);
    }
}

// ------------------------------------------------------------------------------------------
// Stage: one thread per (band element, boundary patch).  ecoef [b][6][28] (27 monomial coefficients [coord][9] + the
// higher-order constant K), pbox [b][6][8] floats (Bezier box of each boundary patch, rounded outward).  (best[b], dmin[b] and the seed item
// are written by k_pairs, which meets every candidate pair anyway.)
__global__ void __launch_bounds__(128) k_np_stage(const DcScalars *S, const double *__restrict__ xyz, const int *__restrict__ conn,
                                                  const int *__restrict__ band_elem, double *__restrict__ ecoef,
                                                  float *__restrict__ pbox)
{
    pdl_start();
    const int n_band = min(S->n_band, S->max_band);
    const long long n = (long long)n_band * 6;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(i / 6), k = (int)(i - (long long)b * 6);
        const int *cn = conn + (size_t)__ldg(band_elem + b) * 27;
        // nodes of boundary patch k (c_face_node[k][a + 3 b] = base + sa a + sb b; the table itself is not used here: with a
        // runtime k the compiler pairs its 36-byte rows into 64-bit constant loads, misaligned for odd k)
        const int nbase = k == 1 ? 2 : (k == 3 ? 6 : (k == 5 ? 18 : 0)), sa = k < 2 ? 3 : 1, sb = k < 4 ? 9 : 3;
        int id[9];
#pragma unroll
        for (int m = 0; m < 9; ++m) id[m] = __ldg(cn + nbase + sa * (m % 3) + sb * (m / 3));
        double A[28], box[6];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double x[9];
#pragma unroll
            for (int m = 0; m < 9; ++m) x[m] = __ldg(xyz + (size_t)id[m] * 3 + c);
            nodes_to_mono9(x, A + 9 * c);
            // Bezier box of the patch (convex-hull property)
#pragma unroll
            for (int j = 0; j < 3; ++j) x[3 * j + 1] = bez_mid(x[3 * j], x[3 * j + 1], x[3 * j + 2]);
#pragma unroll
            for (int q = 0; q < 3; ++q) x[q + 3] = bez_mid(x[q], x[q + 3], x[q + 6]);
            double lo = x[0], hi = x[0];
#pragma unroll
            for (int m = 1; m < 9; ++m) { lo = dmin2(lo, x[m]); hi = dmax2(hi, x[m]); }
            box[c] = lo; box[3 + c] = hi;
        }
        A[27] = higher_order_const(A);
        double2 *out = reinterpret_cast<double2 *>(ecoef + (size_t)i * 28);
#pragma unroll
        for (int m = 0; m < 14; ++m) out[m] = make_double2(A[2 * m], A[2 * m + 1]);
        // the patch's box in single precision, rounded OUTWARD (it only feeds k_np_roots' filter)
        float4 *ob = reinterpret_cast<float4 *>(pbox + (size_t)i * 8);
        ob[0] = make_float4(__double2float_rd(box[0]), __double2float_rd(box[1]), __double2float_rd(box[2]), 0.f);
        ob[1] = make_float4(__double2float_ru(box[3]), __double2float_ru(box[4]), __double2float_ru(box[5]), 0.f);
    }
}

// ------------------------------------------------------------------------------------------
// Solve: projected Newton (dc_newton.cuh), ONE THREAD PER LEAF, both patches' 54 root monomial coefficients in
// REGISTERS (two CTAs of 128 threads per SM at <= 255 registers: the FP64 pipe issues one warp instruction every other
// cycle, so two warps per scheduler with the instruction-level parallelism of six independent jets keep it busy; no
// shared memory, no refill machinery).  Iteration counts differ between the lanes of a warp (2 to 5 evaluations from the
// starting point k_np_bound hands over, rarely many more), so a pass gives every solve a BUDGET of evaluations; a solve
// that needs more is handed, with its state, to the next pass through a continuation queue (64 bytes), where it
// meets other long solves: three passes (budgets NW_BUDGET1, NW_BUDGET2, the rest) keep the lanes of every pass busy.
// Unconverged leaves (NW_MAXIT evaluations, or a stalled step) keep their attained distance as an upper bound and
// are quartered: the four sub-leaves go to an overflow queue, back through one k_np_bound pass (best[b] is final by
// then: most are pruned) and one more solve launch, twice; the last launch finishes what still fails from a small
// local stack.
#define NW_THREADS 128
#define NW_STACK 12                 /* sub-leaves a lane of the last launch may hold (3 levels of quartering) */
#ifndef NW_OVF_MAXIT
#define NW_OVF_MAXIT 20              /* evaluations a sub-leaf of an unconverged leaf may take (a quarter of the box) */
#endif
#define NW_SEED_MAXIT 5              /* evaluations a seed solve may take */
#ifndef NW_BUDGET1
#define NW_BUDGET1 20                 /* busy lanes below which a warp of pass 1 hands its stragglers on */
#endif
#ifndef NW_BUDGET2
#define NW_BUDGET2 12
#endif

struct __align__(16) NCont { NItem it; double x[4]; double lb; short iters, ls, phase, pad; };

// warp-aggregated append of one entry per lane that asks; -1 if the queue is full (no status bit: the caller copes)
__device__ __forceinline__ long long warp_reserve_try(int *counter, int per, long long cap)
{
    const unsigned m = __activemask();           // (every lane that calls wants `per` entries)
    const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(counter, __popc(m) * per);
    base = __shfl_sync(m, base, leader);
    const long long slot = (long long)base + (long long)__popc(m & ((1u << lane) - 1)) * per;
    return slot + per <= cap ? slot : -1;
}

// Leaves are queued with the lower bound they had when k_np_bound met them; by the end of the branch and bound the
// element's best distance has usually dropped below most of them (two thirds at config 2).  One streaming pass drops
// those (and the leaves of elements found CUT) so that the solve launches get dense warps.
__global__ void __launch_bounds__(256) k_np_compact(const DcScalars *S, const int *__restrict__ n_in, long long in_cap,
                                                    const NItem *__restrict__ nq, const NLeafX *__restrict__ nqx,
                                                    const unsigned long long *__restrict__ best,
                                                    NItem *__restrict__ nq_out, NLeafX *__restrict__ nqx_out, int *__restrict__ n_out)
{
    pdl_start();
    if (S->status & DC_STATUS_INVALID) return;
    const int n = min(*n_in, (int)min(in_cap, (long long)0x7fffffff));
    const double tau_exit = S->tau_exit, t_tie = S->t_tie;
    const int n_round = (n + 31) & ~31;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += gridDim.x * blockDim.x) {
        bool keep = false;
        uint4 w = make_uint4(0, 0, 0, 0), xw = make_uint4(0, 0, 0, 0);
        if (i < n) {
            w = __ldg(reinterpret_cast<const uint4 *>(nq + i));
            xw = __ldg(reinterpret_cast<const uint4 *>(nqx + i));
            const double bst = u2d(__ldcg(best + (w.y & 0x1fffffffu)));
            keep = bst > tau_exit && __hiloint2double((int)xw.w, (int)xw.z) <= bst + t_tie;
        }
        const unsigned m = __ballot_sync(0xffffffffu, keep);
        if (!m) continue;
        const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
        int base = 0;
        if (lane == leader) base = atomicAdd(n_out, __popc(m));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (keep) {
            const int sl = base + __popc(m & ((1u << lane) - 1));
            reinterpret_cast<uint4 *>(nq_out)[sl] = w;
            reinterpret_cast<uint4 *>(nqx_out)[sl] = xw;
        }
    }
}

// MODE 0: items are leaves (nq + nqx: starting point and lower bound; nqx == nullptr: seeds, started at the centre)
// MODE 1: items are continuations (cin)
template <int MODE>
__global__ void __launch_bounds__(NW_THREADS, 2) k_np_solve(DcScalars *S, const int *__restrict__ n_items, long long in_cap,
                                                           const NItem *__restrict__ nq, const NLeafX *__restrict__ nqx,
                                                           const NCont *__restrict__ cin,
                                                           const int *__restrict__ pair_face, const double *__restrict__ fcoef,
                                                           const double *__restrict__ ecoef, unsigned long long *__restrict__ best,
                                                           unsigned long long *__restrict__ dmin, unsigned long long *__restrict__ pair_key,
                                                           NCont *__restrict__ cout, int *__restrict__ cout_n, long long cout_cap,
                                                           NItem *__restrict__ ovf, int *__restrict__ ovf_n, long long ovf_cap,
                                                           int budget, int maxit)
{
    pdl_start();
    if (S->status & DC_STATUS_INVALID) return;
    const int n = min(*n_items, (int)min(in_cap, (long long)0x7fffffff));
    const double tau_exit = S->tau_exit, tol_d2 = S->tol_d * S->tol_d, t_tie = S->t_tie;
    const double tau_exit2 = tau_exit > 0.0 ? tau_exit * tau_exit : -1.0;
    const int max_level = S->max_level;
    NpCounters cnt = { 0, 0, 0, 0, 0 };
    const int stride = gridDim.x * blockDim.x;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        NItem it;
        dcn::NwState s; s.iters = 0; s.ls = 0; s.phase = 1;
        double lb = 0.0;
        int a4[4] = { 0, 0, 0, 0 };
        if (MODE == 0) {
            const uint4 w = __ldg(reinterpret_cast<const uint4 *>(nq + i));
            it.p = w.x; it.ak = w.y; it.w2 = w.z; it.w3 = w.w;
            if (nqx) {
                const uint4 xw = __ldg(reinterpret_cast<const uint4 *>(nqx + i));
                a4[0] = (short)(xw.x & 0xffff); a4[1] = (short)(xw.x >> 16); a4[2] = (short)(xw.y & 0xffff); a4[3] = (short)(xw.y >> 16);
                lb = __hiloint2double((int)xw.w, (int)xw.z);
            }
        } else {
            const uint4 *cp = reinterpret_cast<const uint4 *>(cin + i);
            const uint4 w = __ldg(cp), x01 = __ldg(cp + 1), x23 = __ldg(cp + 2), st = __ldg(cp + 3);
            it.p = w.x; it.ak = w.y; it.w2 = w.z; it.w3 = w.w;
            s.x[0] = __hiloint2double((int)x01.y, (int)x01.x); s.x[1] = __hiloint2double((int)x01.w, (int)x01.z);
            s.x[2] = __hiloint2double((int)x23.y, (int)x23.x); s.x[3] = __hiloint2double((int)x23.w, (int)x23.z);
            lb = __hiloint2double((int)st.y, (int)st.x);
            s.iters = (int)(st.z & 0xffff); s.ls = (int)(st.z >> 16); s.phase = (int)(st.w & 0xffff);
        }
        const unsigned b = it.ak & 0x1fffffffu;
        unsigned k = it.ak >> 29;
        const double bst0 = u2d(__ldcg(best + b));
        // dropped: the element is already CUT, or its best distance is below this leaf's lower bound by now
        if (!(bst0 > tau_exit) || lb > bst0 + t_tie) continue;
        double AP[28], AQ[28];
        {
            const double2 *AQg = reinterpret_cast<const double2 *>(fcoef + (size_t)__ldg(pair_face + it.p) * 28);
#pragma unroll
            for (int m = 0; m < 14; ++m) { const double2 vq = __ldg(AQg + m); AQ[2 * m] = vq.x; AQ[2 * m + 1] = vq.y; }
            if (k == 7) {
                // a seed names the pair with the nearest face BOX (k_pairs); its patch is the one whose centre is nearest
                // to the face's centre
                double dbest = INFINITY;
                k = 0;
#pragma unroll
                for (int kk = 0; kk < 6; ++kk) {
                    const double *c = ecoef + ((size_t)b * 6 + kk) * 28;
                    const double dx = __ldg(c) - AQ[0], dy = __ldg(c + 9) - AQ[9], dz = __ldg(c + 18) - AQ[18];
                    const double d2 = dx * dx + dy * dy + dz * dz;
                    if (d2 < dbest) { dbest = d2; k = kk; }
                }
                it.ak = b | (k << 29);
            }
            const double2 *APg = reinterpret_cast<const double2 *>(ecoef + ((size_t)b * 6 + k) * 28);
#pragma unroll
            for (int m = 0; m < 14; ++m) { const double2 vp = __ldg(APg + m); AP[2 * m] = vp.x; AP[2 * m + 1] = vp.y; }
        }
        auto cf = [&](int m) { return m < 27 ? AP[m] : AQ[m - 27]; };
        double uc, vc, hP, sc, tc, hQ;
        nitem_box(it, uc, vc, hP, sc, tc, hQ);
        double lo[4] = { uc - hP, vc - hP, sc - hQ, tc - hQ }, hi[4] = { uc + hP, vc + hP, sc + hQ, tc + hQ };
        if (MODE == 0 && !nqx) {
            // a seed (a whole patch pair, centre (0,0)): its own first-order model from the coefficients themselves
            const double r[3] = { cf(0) - cf(27), cf(9) - cf(36), cf(18) - cf(45) };
            const double pu[3] = { cf(1), cf(10), cf(19) }, pv[3] = { cf(3), cf(12), cf(21) };
            const double qs[3] = { cf(28), cf(37), cf(46) }, qt[3] = { cf(30), cf(39), cf(48) };
            double a[4];
            model_closest_pair(r, pu, pv, qs, qt, pu[0] * pu[0] + pu[1] * pu[1] + pu[2] * pu[2], pv[0] * pv[0] + pv[1] * pv[1] + pv[2] * pv[2],
                               qs[0] * qs[0] + qs[1] * qs[1] + qs[2] * qs[2], qt[0] * qt[0] + qt[1] * qt[1] + qt[2] * qt[2], 1.0, 1.0, a);
#pragma unroll
            for (int j = 0; j < 4; ++j) s.x[j] = a[j];
        } else if (MODE == 0) {
            // start at the closest pair of the leaf's first-order model (on a bound when the fixed point says so)
            const double q15 = 1.0 / 32767.0;
            const double cen[4] = { uc, vc, sc, tc }, hw[4] = { hP, hP, hQ, hQ };
#pragma unroll
            for (int j = 0; j < 4; ++j)
                s.x[j] = a4[j] >= 32767 ? hi[j] : (a4[j] <= -32767 ? lo[j] : fma(hw[j] * q15, (double)a4[j], cen[j]));
        }
        const bool seed = (it.w3 >> 24) & 1;
        NItem stk[NW_STACK];            // (last launch only: sub-leaves of an unconverged solve; local memory, rarely touched)
        int sp = 0;
        int left = maxit;
        while (true) {
            dcn::NwResult R; R.dist = 0.0; R.cosv = 0.0; R.converged = 0;
            bool fin = false, dropped = false;
            while (left > 0 && !fin) {
                // a solve that drags on looks, every 4th evaluation, whether its element has been found CUT meanwhile (by
                // another of its pairs), or its best distance has dropped below this leaf's lower bound: nothing it could
                // still find would matter then
                if (s.iters >= 4 && (s.iters & 3) == 0) {
                    const double bnow = u2d(__ldcg(best + b));
                    if (bnow <= tau_exit || lb > bnow + t_tie) { dropped = true; break; }
                }
                fin = dcn::iterate(cf, s, lo, hi, tol_d2, tau_exit2, R, maxit);
                --left;
                // the budget of a pass is not a number of evaluations but a number of busy lanes: a warp goes on while at
                // least `budget` of its lanes are still iterating, then hands the stragglers to the next pass
                if (!fin && cout && __popc(__activemask()) < budget) left = 0;
            }
            if (dropped) break;
            if (!fin) {
                // out of budget: hand the solve to the next pass (or go on here if its queue is full)
                const long long sl = cout ? warp_reserve_try(cout_n, 1, cout_cap) : -1;
                if (sl >= 0) {
                    uint4 *cp = reinterpret_cast<uint4 *>(cout + sl);
                    cp[0] = make_uint4(it.p, it.ak, it.w2, it.w3);
                    cp[1] = make_uint4((unsigned)__double2loint(s.x[0]), (unsigned)__double2hiint(s.x[0]), (unsigned)__double2loint(s.x[1]), (unsigned)__double2hiint(s.x[1]));
                    cp[2] = make_uint4((unsigned)__double2loint(s.x[2]), (unsigned)__double2hiint(s.x[2]), (unsigned)__double2loint(s.x[3]), (unsigned)__double2hiint(s.x[3]));
                    cp[3] = make_uint4((unsigned)__double2loint(lb), (unsigned)__double2hiint(lb), (unsigned)s.iters | ((unsigned)s.ls << 16), (unsigned)s.phase);
                    break;
                }
                left = maxit;
                continue;
            }
            // ---- result of the finished solve (an attained distance is an upper bound whether converged or not)
            cnt.newton++; cnt.iters += s.iters;
            atomicMin(best + b, d2u(R.dist));
            // (a seed only tightens best[b]: its pair comes back as a leaf, and which pair is the seed depends on the
            // arrival order of the faces in their bins -- results must not: dmin and the keys come from leaves alone)
            if (R.dist > tau_exit && !seed) {
                atomicMin(dmin + b, d2u(R.dist));
                const unsigned long long key = (d2u(R.dist) & ~0xffull) | (unsigned long long)cos_code(R.cosv);
                atomicMin(pair_key + it.p, key);
                if (!R.converged) {
                    // unconverged: the distance above stands as an upper bound and the leaf is quartered (a seed solve is
                    // never split: the roots cover its pair)
                    cnt.fail++;
                    bool splitP = false;
                    if (u2d(__ldcg(best + b)) <= tau_exit) { /* the element is CUT by now: no sub-leaves */ }
                    else if (choose_split(it, (it.w2 & 15) <= ((it.w2 >> 4) & 15), max_level, splitP)) {
                        if (ovf) {
                            const long long sl = warp_reserve_try(ovf_n, 4, ovf_cap);
                            if (sl >= 0) {
#pragma unroll
                                for (int c = 0; c < 4; ++c) ovf[sl + c] = nitem_child(it, splitP, c);
                            } else { atomicOr(&S->status, DC_STATUS_QUEUE_OVERFLOW); }
                        } else if (sp + 4 <= NW_STACK) {
#pragma unroll
                            for (int c = 0; c < 4; ++c) stk[sp++] = nitem_child(it, splitP, c);
                        } else cnt.depth++;
                    } else cnt.depth++;
                }
            }
            if (sp == 0) break;
            // (last launch) next sub-leaf of this lane's own: same pair, the coefficients are in place
            it = stk[--sp];
            nitem_box(it, uc, vc, hP, sc, tc, hQ);
            lo[0] = uc - hP; lo[1] = vc - hP; lo[2] = sc - hQ; lo[3] = tc - hQ;
            hi[0] = uc + hP; hi[1] = vc + hP; hi[2] = sc + hQ; hi[3] = tc + hQ;
            s.x[0] = uc; s.x[1] = vc; s.x[2] = sc; s.x[3] = tc;
            s.iters = 0; s.ls = 0; s.phase = 1;
            left = maxit;
        }
    }
    np_flush_counters(S, cnt);
}

// ------------------------------------------------------------------------------------------
// Roots: one thread per candidate pair.  (pair, patch k) survives when the box distance (Algorithm A.2) of
// the patch's Bezier box and the face's Bezier box is within best + t_tie; survivors become the items of round 0
// (warp-aggregated append: a scan of the lanes' counts, one atomic per warp).
__global__ void __launch_bounds__(256) k_np_roots(DcScalars *S, const int *__restrict__ pair_band, const int *__restrict__ pair_face,
                                                  const float *__restrict__ fbox, const float *__restrict__ pbox,
                                                  const unsigned long long *__restrict__ best, long long max_pairs,
                                                  NItem *__restrict__ qout, int *__restrict__ qout_n, long long qcap)
{
    pdl_start();
    __shared__ int s_wsum[8];
    __shared__ int s_base, s_total;
    if (S->status & DC_STATUS_INVALID) return;       // an overflow upstream left holes in the lists: nothing here can be trusted (or safely read)
    const long long n_pairs = min((long long)S->n_pairs, max_pairs);
    const long long n_round = (n_pairs + 255) & ~255LL;          // (uniform trip count inside a CTA: barriers below)
    const double t_tie = S->t_tie, tau_exit = S->tau_exit;
    const int lane = threadIdx.x & 31;
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < n_round; p += (long long)gridDim.x * blockDim.x) {
        unsigned mask = 0;
        int b = 0;
        if (p < n_pairs) {
            b = __ldg(pair_band + p);
            const double bst = u2d(__ldg(best + b));
            if (bst > tau_exit) {                                   // (else: already CUT)
                // single precision, conservative: boxes rounded outward, gaps and their squares rounded down, the cutoff up
                const float cutf = __double2float_ru(bst + t_tie), cut2 = __fmul_ru(cutf, cutf);
                const float4 *fp = reinterpret_cast<const float4 *>(fbox) + (size_t)__ldg(pair_face + p) * 2;
                const float4 flo = __ldg(fp), fhi = __ldg(fp + 1);
                const float4 *pb = reinterpret_cast<const float4 *>(pbox) + (size_t)b * 12;
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    const float4 plo = __ldg(pb + 2 * k), phi = __ldg(pb + 2 * k + 1);
                    const float gx = fmaxf(0.f, fmaxf(__fsub_rd(flo.x, phi.x), __fsub_rd(plo.x, fhi.x)));
                    const float gy = fmaxf(0.f, fmaxf(__fsub_rd(flo.y, phi.y), __fsub_rd(plo.y, fhi.y)));
                    const float gz = fmaxf(0.f, fmaxf(__fsub_rd(flo.z, phi.z), __fsub_rd(plo.z, fhi.z)));
                    const float d2 = __fadd_rd(__fadd_rd(__fmul_rd(gx, gx), __fmul_rd(gy, gy)), __fmul_rd(gz, gz));
                    if (d2 <= cut2) mask |= 1u << k;
                }
            }
        }
        const int mine = __popc(mask);
        int incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
        // one atomic per CTA and round (a returning atomic on ONE address costs about a third of a nanosecond of the whole
        // GPU's time: one per warp was a third of this kernel)
        if (lane == 31) s_wsum[threadIdx.x >> 5] = incl;
        __syncthreads();
        if (threadIdx.x == 0) {
            int t = 0;
#pragma unroll
            for (int w2 = 0; w2 < 8; ++w2) { const int v = s_wsum[w2]; s_wsum[w2] = t; t += v; }
            s_base = t ? atomicAdd(qout_n, t) : 0;
            s_total = t;
        }
        __syncthreads();
        const int cbase = s_base, start = cbase + s_wsum[threadIdx.x >> 5], total = s_total;
        __syncthreads();
        if (total == 0) continue;
        if ((long long)cbase + total > qcap) { if (threadIdx.x == 0) atomicOr(&S->status, DC_STATUS_QUEUE_OVERFLOW); continue; }
        long long slot = (long long)start + incl - mine;
        while (mask) {
            const int k = __ffs(mask) - 1; mask &= mask - 1;
            NItem it; it.p = (unsigned)p; it.ak = (unsigned)b | ((unsigned)k << 29); it.w2 = 0; it.w3 = 0;
            qout[slot++] = it;
        }
    }
}

// ------------------------------------------------------------------------------------------
// Bound: one thread per item of qin[0 .. n): prune, or 4 children -> qout, or leaf -> the ONE leaf queue nq
// (all rounds append to it; the Newton kernel runs once, after the last round).  Items i0, i0 + stride, ...
template <bool ROOT>
__device__ __forceinline__ void np_bound_items(DcScalars *S, int n, const NItem *__restrict__ qin,
                                               const int *__restrict__ pair_face, const double *__restrict__ fcoef,
                                               const double *__restrict__ ecoef, unsigned long long *__restrict__ best,
                                               NItem *__restrict__ qout, int *__restrict__ qout_n,
                                               NItem *__restrict__ nq, NLeafX *__restrict__ nqx, int *__restrict__ nq_n, long long qcap,
                                               int i0, int stride, NpCounters &cnt, bool force_leaf = false)
{
    const double t_tie = S->t_tie, tau_exit = S->tau_exit, theta2 = S->theta * S->theta;
    const int max_level = S->max_level;
    const int n_round = (n + 31) & ~31;
    for (int i = i0; i < n_round; i += stride) {
        bool split = false, leaf = false, splitP = false;
        NItem it; it.p = it.ak = it.w2 = it.w3 = 0;
        float4 x0 = make_float4(0.f, 0.f, 0.f, 0.f);
        double lbq = 0.0;                      // the leaf's lower bound
        if (i < n) {
            // (L2 load: the tail kernel reads items the same launch wrote)
            const uint4 w = __ldcg(reinterpret_cast<const uint4 *>(qin + i));
            it.p = w.x; it.ak = w.y; it.w2 = w.z; it.w3 = w.w;
            const unsigned b = it.ak & 0x1fffffffu, k = it.ak >> 29;
            double bst = u2d(__ldcg(best + b));
            if (bst > tau_exit) {
                double uc, vc, hP, sc, tc, hQ;
                nitem_box(it, uc, vc, hP, sc, tc, hQ);
                const double *APg = ecoef + ((size_t)b * 6 + k) * 28;
                const double *AQg = fcoef + (size_t)__ldg(pair_face + it.p) * 28;
                double AP[28], AQ[28];
#pragma unroll
                for (int m = 0; m < 14; ++m) {
                    const double2 vp = __ldg(reinterpret_cast<const double2 *>(APg) + m);
                    const double2 vq = __ldg(reinterpret_cast<const double2 *>(AQg) + m);
                    AP[2 * m] = vp.x; AP[2 * m + 1] = vp.y; AQ[2 * m] = vq.x; AQ[2 * m + 1] = vq.y;
                }
                const NodeOut o = bound_node<ROOT>([&](int m) { return AP[m]; }, [&](int m) { return AQ[m]; }, AP[27], AQ[27],
                                             uc, vc, hP, sc, tc, hQ, theta2);
                cnt.nodes++;
                if (o.ub < bst) { atomicMin(best + b, d2u(o.ub)); bst = o.ub; }
                const bool alive = o.ub > tau_exit && o.lb <= bst + t_tie;
                lbq = o.lb;
                x0 = make_float4((float)o.x0[0], (float)o.x0[1], (float)o.x0[2], (float)o.x0[3]);
                if (alive) {
                    leaf = o.leaf || force_leaf;     // (sub-leaves of an unconverged leaf stay leaves)
                    if (!leaf) {
                        split = choose_split(it, o.splitP, max_level, splitP);
                        if (!split) { leaf = true; cnt.depth++; }
                    }
                }
            }
        }
        const long long sl = warp_reserve(nq_n, leaf, 1, qcap, &S->status);
        if (sl >= 0) {
            NLeafX lx;
            lx.x[0] = (short)__float2int_rn(x0.x * 32767.f); lx.x[1] = (short)__float2int_rn(x0.y * 32767.f);
            lx.x[2] = (short)__float2int_rn(x0.z * 32767.f); lx.x[3] = (short)__float2int_rn(x0.w * 32767.f);
            lx.lb = lbq;
            nq[sl] = it; nqx[sl] = lx;
        }
        const long long slot = warp_reserve(qout_n, split, 4, qcap, &S->status);
        if (slot >= 0) {
#pragma unroll
            for (int c = 0; c < 4; ++c) qout[slot + c] = nitem_child(it, splitP, c);
        }
    }
}

template <bool ROOT>
__global__ void __launch_bounds__(NPW_THREADS, ROOT ? 3 : 2) k_np_bound(DcScalars *S, const int *__restrict__ n_in, const NItem *__restrict__ qin,
                                                          const int *__restrict__ pair_face, const double *__restrict__ fcoef,
                                                          const double *__restrict__ ecoef, unsigned long long *__restrict__ best,
                                                          NItem *__restrict__ qout, int *__restrict__ qout_n,
                                                          NItem *__restrict__ nq, NLeafX *__restrict__ nqx, int *__restrict__ nq_n, long long qcap, int force_leaf)
{
    pdl_start();
    if (S->status & DC_STATUS_INVALID) return;
    const int n = min(*n_in, (int)min(qcap, (long long)0x7fffffff));
    if (n == 0) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicMax(&S->c_queue_peak, (unsigned long long)n);
    NpCounters cnt = { 0, 0, 0, 0, 0 };
    np_bound_items<ROOT>(S, n, qin, pair_face, fcoef, ecoef, best, qout, qout_n, nq, nqx, nq_n, qcap,
                   blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x, cnt, force_leaf != 0);
    np_flush_counters(S, cnt);
}

// The rounds after the first few hold few items (deep levels exist only where the surface curves fast): ONE CTA
// walks them all, round after round, until a round comes up empty -- no launch per round, no empty launches.
#define NP_TAIL_THREADS 256
__global__ void __launch_bounds__(NP_TAIL_THREADS) k_np_bound_tail(DcScalars *S, int r_begin, int r_end, NItem *q0, NItem *q1,
                                                                   const int *__restrict__ pair_face, const double *__restrict__ fcoef,
                                                                   const double *__restrict__ ecoef, unsigned long long *__restrict__ best,
                                                                   NItem *__restrict__ nq, NLeafX *__restrict__ nqx, int *__restrict__ nq_n, long long qcap)
{
    pdl_start();
    if (S->status & DC_STATUS_INVALID) return;
    NpCounters cnt = { 0, 0, 0, 0, 0 };
    for (int r = r_begin; r < r_end; ++r) {
        const int n = min(*(volatile int *)&S->qn[r], (int)min(qcap, (long long)0x7fffffff));
        if (n == 0) break;
        if (threadIdx.x == 0) atomicMax(&S->c_queue_peak, (unsigned long long)n);
        np_bound_items<false>(S, n, (r & 1) ? q1 : q0, pair_face, fcoef, ecoef, best, (r & 1) ? q0 : q1, &S->qn[r + 1], nq, nqx, nq_n, qcap,
                       threadIdx.x, NP_TAIL_THREADS, cnt);
        __threadfence();
        __syncthreads();
    }
    np_flush_counters(S, cnt);
}

// ------------------------------------------------------------------------------------------
// S6 decide (L215: nearest face, dot of the minimal vector with its outward normal; ties L294):
// a group of 8 lanes per band element (its ~25 pair keys are one contiguous run: the lanes read it side by side).
#define ND_W 8
__global__ void k_np_decide(DcScalars *S, const int *__restrict__ band_elem, const long long *__restrict__ band_start,
                            const int *__restrict__ band_cnt, const unsigned long long *__restrict__ best,
                            const unsigned long long *__restrict__ dmin_arr, const unsigned long long *__restrict__ pair_key,
                            signed char *__restrict__ labels, double *__restrict__ sdist)
{
    pdl_start();
    const int n_band = min(S->n_band, S->max_band);
    const double tau = S->tau, tau_exit = S->tau_exit, amb = S->amb, t_tie = S->t_tie, d_band = S->d_band;
    unsigned n_amb = 0, n_samb = 0;
    const int sub = threadIdx.x & (ND_W - 1);
    const unsigned gmask = ((1u << ND_W) - 1u) << ((threadIdx.x & 31) & ~(ND_W - 1));
    const int ngroups = gridDim.x * blockDim.x / ND_W;
    const int n_round = (n_band + ngroups - 1) / ngroups * ngroups;          // (uniform trip count: group shuffles below)
    for (int b = (blockIdx.x * blockDim.x + threadIdx.x) / ND_W; b < n_round; b += ngroups) {   // (n_band is only known on the device)
        if (b >= n_band) continue;
        const int e = band_elem[b];
        const double dmin = u2d(dmin_arr[b]);
        if (u2d(best[b]) <= tau_exit) { if (sub == 0) { labels[e] = DC_CUT; sdist[e] = 0.0; } }
        else if (dmin <= tau) { if (sub == 0) { labels[e] = DC_CUT; sdist[e] = 0.0; if (dmin >= tau - amb) ++n_amb; } }
        else if (dmin <= d_band) {
            // (an element whose distance exceeds the band keeps label -1 and takes its sign from the flood fill: beyond
            // best[b] = reach the branch and bound has pruned freely, so the faces it did solve need not include the
            // nearest one, and on a body thinner than the band a far-side face could win the sign)
            int bestkey = -1, bneg = 0, npos = 0, nneg = 0;   // the largest magnitude wins
            const long long p0 = band_start[b];
            const int cnt = band_cnt[b];
            for (int p = sub; p < cnt; p += ND_W) {
                const unsigned long long key = pair_key[p0 + p];
                const double dk = u2d(key & ~0xffull);
                if (dk <= dmin + t_tie) {
                    const int code = (int)(key & 0xff), mag = code & 0x7f, ng = code >> 7;
                    if (ng) ++nneg; else ++npos;
                    // ties in magnitude go to the first pair of the run, as a single thread walking it would decide:
                    // (mag, -p) ordered, kept as one integer
                    const int k2 = (mag << 24) | (0xffffff - min(p, 0xffffff));
                    if (k2 > bestkey) { bestkey = k2; bneg = ng; }
                }
            }
#pragma unroll
            for (int o = ND_W / 2; o > 0; o >>= 1) {
                const int ob = __shfl_xor_sync(gmask, bestkey, o), on = __shfl_xor_sync(gmask, bneg, o);
                npos += __shfl_xor_sync(gmask, npos, o); nneg += __shfl_xor_sync(gmask, nneg, o);
                if (ob > bestkey) { bestkey = ob; bneg = on; }
            }
            if (sub == 0) {
                if (dmin <= tau + amb) ++n_amb;
                if (npos && nneg) ++n_samb;
                const int neg = bneg;
                labels[e] = neg ? DC_HOLE : DC_NORMAL;
                const double d = dmin2(dmin, d_band);
                sdist[e] = neg ? -d : d;
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { n_amb += __shfl_xor_sync(0xffffffffu, n_amb, o); n_samb += __shfl_xor_sync(0xffffffffu, n_samb, o); }
    if ((threadIdx.x & 31) == 0) {
        if (n_amb) atomicAdd(&S->c_ambiguous, (unsigned long long)n_amb);
        if (n_samb) atomicAdd(&S->c_sign_ambiguous, (unsigned long long)n_samb);
    }
}
