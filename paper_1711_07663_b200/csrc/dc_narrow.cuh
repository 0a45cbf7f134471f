// dc_narrow.cuh -- S5 (narrow phase) and S6 (decide) as a short sequence of uniform kernels over global queues.
//
// Every kernel does one kind of operation and compacts its output into a global queue (warp-aggregated
// atomics), so warps stay full and no kernel carries another's registers:
//
//   k_np_stage      warp / band element : gather the 27 nodes, monomial coefficients and Bezier boxes of the 6
//                                         boundary patches -> ecoef, pbox; centre-centre distances of all
//                                         (pair, patch) -> first upper bound best[b] and ONE seed item per element
//   k_np_newton     persistent warps    : projected Newton (Eq. 3-5 L256-L270 generalised to two patches, clamp
//                                         L272-L278), one solve per lane in lockstep, lanes refilled from the
//                                         queue; min into best / dmin / pair_key; the sub-leaves of an unconverged
//                                         leaf go to an overflow queue
//   k_np_roots      warp / band element : (pair, patch) whose boxes are within best + t_tie (A.2, L689-L709)
//                                         become the items of round 0
//   k_np_bound      thread / item       : bound_node -> prune / 4 children / leaf (+ the leaf's first step)
//   k_np_bound_tail one CTA             : the sparse late rounds, until one comes up empty
//   k_np_decide     thread / band elem  : S6 (L215 nearest face and its normal; tie rule L294)
//
// Launch order (dc_classify): stage, newton(seeds), roots, bound x 4, bound_tail, newton(leaves),
// [bound(overflow), newton] x 2, decide.  Every item of bound round r has lP + lQ = r, so 2 max_level + 1
// rounds always terminate the branch and bound.
#pragma once

#define NPW_THREADS 128
#define DC_MAX_ROUNDS 25            /* 2 * 12 + 1 */

struct __align__(16) NItem { unsigned p, ak, w2, w3; };
// p : global pair index (face = pair_face[p], key slot = pair_key[p])
// ak: band index b (29 bits) | boundary patch k << 29
// w2: lP(4) | lQ(4)<<4 | iu(12)<<8 | iv(12)<<20
// w3: is(12) | it(12)<<12 | flags(8)<<24      flags bit0: seed solve (no re-split on failure)

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
// Stage: one warp per band element.  ecoef [b][6][28] (27 monomial coefficients [coord][9] + the
// higher-order constant K), pbox [b][6][6] (Bezier box of each boundary patch).
#define ST_WARPS (NPW_THREADS / 32)
__global__ void __launch_bounds__(NPW_THREADS) k_np_stage(DcScalars *S, const double *__restrict__ xyz, const int *__restrict__ conn,
                                                          const int *__restrict__ band_elem, const long long *__restrict__ band_start,
                                                          const int *__restrict__ band_cnt, const int *__restrict__ pair_face,
                                                          const double *__restrict__ fcoef, double *__restrict__ ecoef,
                                                          double *__restrict__ pbox, unsigned long long *__restrict__ best,
                                                          unsigned long long *__restrict__ dmin, NItem *__restrict__ nq)
{
    __shared__ double s_nodes[ST_WARPS][81];
    __shared__ double s_coef[ST_WARPS][6 * 28];
    __shared__ double s_box[ST_WARPS][36];
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * blockDim.x) >> 5;
    const int n_band = min(S->n_band, S->max_band);
    const double reach = S->reach;
    double *nd = s_nodes[wl], *cf = s_coef[wl], *bx = s_box[wl];
    // the node gather (band_elem -> conn -> xyz: three dependent loads) of the NEXT element of this warp is issued
    // before the current one is processed
    double cx = 0.0, cy = 0.0, cz = 0.0;
    if (warp < n_band && lane < 27) {
        const int id = __ldg(conn + (size_t)band_elem[warp] * 27 + lane);
        const double *p = xyz + (size_t)id * 3;
        cx = __ldg(p); cy = __ldg(p + 1); cz = __ldg(p + 2);
    }
    for (int b = warp; b < n_band; b += nwarps) {
        if (lane < 27) { nd[lane * 3 + 0] = cx; nd[lane * 3 + 1] = cy; nd[lane * 3 + 2] = cz; }
        if (b + nwarps < n_band && lane < 27) {
            const int id = __ldg(conn + (size_t)band_elem[b + nwarps] * 27 + lane);
            const double *p = xyz + (size_t)id * 3;
            cx = __ldg(p); cy = __ldg(p + 1); cz = __ldg(p + 2);
        }
        __syncwarp();
        if (lane < 18) {
            const int k = lane / 3, c = lane % 3;
            double x[9], a[9];
#pragma unroll
            for (int m = 0; m < 9; ++m) x[m] = nd[c_face_node[k][m] * 3 + c];
            nodes_to_mono9(x, a);
#pragma unroll
            for (int m = 0; m < 9; ++m) cf[k * 28 + c * 9 + m] = a[m];
            // Bezier box of the patch (convex-hull property)
#pragma unroll
            for (int j = 0; j < 3; ++j) x[3 * j + 1] = bez_mid(x[3 * j], x[3 * j + 1], x[3 * j + 2]);
#pragma unroll
            for (int i = 0; i < 3; ++i) x[i + 3] = bez_mid(x[i], x[i + 3], x[i + 6]);
            double lo = x[0], hi = x[0];
#pragma unroll
            for (int m = 1; m < 9; ++m) { lo = dmin2(lo, x[m]); hi = dmax2(hi, x[m]); }
            bx[k * 6 + c] = lo; bx[k * 6 + 3 + c] = hi;
        }
        __syncwarp();
        // constants K of the 6 patches (dc_geom.cuh higher_order_const): the 6 x 6 coefficient norms it needs are
        // spread over the warp (a lane per norm) instead of 9 square roots in a row on 6 lanes
        {
            // weights of |A20| |A02| |A11| |A21| |A12| |A22| (m = 2, 6, 4, 5, 7, 8) in K
            const int mm[6] = { 2, 6, 4, 5, 7, 8 };
            const double ww[6] = { 1.0, 1.0, 1.0, 4.0, 4.0, 11.0 };
            double part = 0.0, part2 = 0.0;
            {
                const int k = lane / 6, j = lane % 6;           // lanes 0..31 -> (patch, norm) 0..31
                const double *A = cf + k * 28;
                const int m = mm[j];
                part = ww[j] * sqrt(A[m] * A[m] + A[9 + m] * A[9 + m] + A[18 + m] * A[18 + m]);
            }
            if (lane < 4) {                                     // (patch 5, norms 2..5) = items 32..35
                const int j = lane + 2;
                const double *A = cf + 5 * 28;
                const int m = mm[j];
                part2 = ww[j] * sqrt(A[m] * A[m] + A[9 + m] * A[9 + m] + A[18 + m] * A[18 + m]);
            }
            // sum the 6 norms of each patch: lanes 6k .. 6k+5 (patch 5: lanes 30, 31 + part2 of lanes 0..3)
            double sum = part;
#pragma unroll
            for (int o = 1; o < 6; ++o) {
                const double v = __shfl_down_sync(0xffffffffu, part, o);
                if (lane % 6 + o < 6 && lane + o < 32) sum += v;
            }
            double tail = part2;
            tail += __shfl_down_sync(0xffffffffu, tail, 2);
            tail += __shfl_down_sync(0xffffffffu, tail, 1);
            tail = __shfl_sync(0xffffffffu, tail, 0);
            if (lane % 6 == 0 && lane < 30) cf[(lane / 6) * 28 + 27] = sum;
            if (lane == 30) cf[5 * 28 + 27] = sum + tail;
        }
        __syncwarp();
        for (int i = lane; i < 6 * 28; i += 32) ecoef[(size_t)b * (6 * 28) + i] = cf[i];
        for (int i = lane; i < 36; i += 32) pbox[(size_t)b * 36 + i] = bx[i];
        // centre-centre distances of every (pair, patch): attained => upper bound; the smallest seeds Newton.
        // A lane per pair (its face centre is loaded once), the 6 patch centres come from shared memory.
        const long long p0 = band_start[b];
        const int npair = band_cnt[b];
        unsigned long long key = ~0ull;
        for (int pl = lane; pl < npair; pl += 32) {
            const int f = __ldg(pair_face + p0 + pl);
            const double *AQ = fcoef + (size_t)f * 28;
            const double qx = __ldg(AQ), qy = __ldg(AQ + 9), qz = __ldg(AQ + 18);
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                const double dx = cf[k * 28] - qx, dy = cf[k * 28 + 9] - qy, dz = cf[k * 28 + 18] - qz;
                const double d2 = dx * dx + dy * dy + dz * dz;           // (squared: one sqrt per element, below)
                const unsigned long long kk = (d2u(d2) & ~0xfffffull) | (unsigned long long)min(pl * 6 + k, 0xfffff);
                key = kk < key ? kk : key;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { const unsigned long long v = __shfl_xor_sync(0xffffffffu, key, o); key = v < key ? v : key; }
        if (lane == 0) {
            // the truncated key is <= the attained squared distance: round up to stay an upper bound
            const double dkey = sqrt(u2d((key & ~0xfffffull) + 0x100000ull)) * (1.0 + 4e-16);
            best[b] = d2u(dmin2(reach, dkey));
            dmin[b] = 0x7ff0000000000000ull;
            const int t = (int)(key & 0xfffffull);
            const int pl = t / 6, k = t - pl * 6;
            NItem it; it.p = (unsigned)(p0 + pl); it.ak = (unsigned)b | ((unsigned)k << 29); it.w2 = 0; it.w3 = 1u << 24;
            nq[b] = it;
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------
// Newton: PERSISTENT warps over the leaf queue nq[0 .. *n_items), one solve per lane, all lanes of a warp
// in lockstep (dcn::iterate = exactly one value+gradient+Hessian evaluation), lanes whose solve has
// finished are refilled from the queue (one warp-aggregated atomic on *head), so the iteration count of
// one solve never holds up the other 31.  The two patches' 54 root monomial coefficients of every lane
// live in shared memory, transposed (coefficient-major, lane-minor: conflict-free reads), which keeps the
// kernel at <= 128 registers and 16 warps per SM; a refill is a warp-cooperative coalesced copy of the
// 2 x 216 B of the new item (the odd stride makes the transposed store 2-way conflicted instead of 32).
#define NW_THREADS 128
#define NW_STRIDE 129
#define NW_SMEM_BYTES (54 * NW_STRIDE * 8)
#define NW_STACK 12                 /* sub-leaves a lane may hold (3 levels of quartering) */
#define NW_TICKETS 64                /* queue tickets a warp draws per atomic on the queue head */
#define NW_OVF_MAXIT 20              /* evaluations a sub-leaf of an unconverged leaf may take (a quarter of the box) */
#define NW_SEED_MAXIT 8              /* evaluations a seed solve may take */
#define NW_REFILL 1                 /* idle lanes that trigger a refill while others are still iterating */

__global__ void __launch_bounds__(NW_THREADS, 4) k_np_newton(DcScalars *S, const int *__restrict__ n_items, long long in_cap, int *head,
                                                            const NItem *__restrict__ nq, const float4 *__restrict__ nqx,
                                                            const int *__restrict__ pair_face, const double *__restrict__ fcoef,
                                                            const double *__restrict__ ecoef, unsigned long long *__restrict__ best,
                                                            unsigned long long *__restrict__ dmin, unsigned long long *__restrict__ pair_key,
                                                            NItem *__restrict__ ovf, int *__restrict__ ovf_n, long long ovf_cap, int maxit)
{
    extern __shared__ double nw_sm[];
    const int n = min(*n_items, (int)min(in_cap, (long long)0x7fffffff));
    if (n == 0) return;
    const int tid = threadIdx.x, lane = tid & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    const double *slot = nw_sm + tid;
    const volatile double *vslot = slot;   // volatile: re-read in the line search instead of keeping 54 values live
    auto cf = [&](int m) { return vslot[m * NW_STRIDE]; };
    const double tau_exit = S->tau_exit, tol_d2 = S->tol_d * S->tol_d;
    const double tau_exit2 = tau_exit > 0.0 ? tau_exit * tau_exit : -1.0;
    const int max_level = S->max_level;
    NpCounters cnt = { 0, 0, 0, 0, 0 };
    dcn::NwState s; s.phase = 0; s.iters = 0; s.ls = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) s.x[i] = 0.0;
    NItem it; it.p = it.ak = it.w2 = it.w3 = 0;
    NItem nxt; nxt.p = nxt.ak = nxt.w2 = nxt.w3 = 0;       // prefetched next item of this lane
    // 0 no ticket, 2 ticket in hand, 3 item asked for, 4 face id and best[b] asked for (ready), 9 queue exhausted
    int nst = 0, nface = 0, tk = 0, pbase = 0;
    int pool_next = 0, pool_end = 0;    // (warp-uniform) tickets this warp holds
    // tickets per draw: half a warp's share of the queue, between 8 and NW_TICKETS (short queues stay spread out)
    const int chunk = max(8, min(NW_TICKETS, n / (int)(gridDim.x * (NW_THREADS / 32) * 2)));
    unsigned long long nbest = 0;
    float4 nx0 = make_float4(0.f, 0.f, 0.f, 0.f);   // its starting point (local coordinates; zero = the centre, for seeds)
    bool pend = false;              // (warp-uniform) a ticket atomic is in flight
    NItem stk[NW_STACK];            // sub-leaves of an unconverged solve, solved by the same lane (local memory, rarely touched)
    int sp = 0;
    while (true) {
        // ---- a lane with sub-leaves of its own goes on with those (same pair: its coefficients are already in place)
        if (s.phase == 0 && sp > 0) {
            it = stk[--sp];
            double uc, vc, hP, sc, tc, hQ;
            nitem_box(it, uc, vc, hP, sc, tc, hQ);
            s.x[0] = uc; s.x[1] = vc; s.x[2] = sc; s.x[3] = tc;
            s.iters = 0; s.ls = 0; s.phase = 1;
        }
        // ---- every lane runs a small pipeline that fetches its NEXT item while it solves the current one, one
        // stage per trip, so that no trip waits for more than one memory round trip: ticket (warp-aggregated
        // atomic) -> item -> face id, best[b], L2 prefetch of the element coefficients -> ready.
        if (nst == 3) {
            const unsigned nb = nxt.ak & 0x1fffffffu;
            nface = __ldg(pair_face + nxt.p);
            nbest = __ldcg(best + nb);
            const char *pn = reinterpret_cast<const char *>(ecoef + ((size_t)nb * 6 + (nxt.ak >> 29)) * 28);
            asm volatile("prefetch.global.L2 [%0];" :: "l"(pn));
            asm volatile("prefetch.global.L2 [%0];" :: "l"(pn + 128));
            nst = 4;
        } else if (nst == 2) {
            if (tk >= n) nst = 9;
            else {
                const uint4 w = __ldg(reinterpret_cast<const uint4 *>(nq + tk));
                nxt.p = w.x; nxt.ak = w.y; nxt.w2 = w.z; nxt.w3 = w.w;
                if (nqx) nx0 = __ldg(nqx + tk);
                nst = 3;
            }
        }
        if (pend) {                                   // (uniform) the ticket atomic of an earlier trip has landed
            pool_next = __shfl_sync(0xffffffffu, pbase, 0);
            pool_end = pool_next + chunk;
            pend = false;
        }
        // ---- idle lanes whose next item is ready take it
        bool fresh = false;
        unsigned long long pA = 0, pQ = 0;
        {
            const bool ready = s.phase == 0 && nst == 4;
            const unsigned mready = __ballot_sync(0xffffffffu, ready);
            const unsigned mbusy = __ballot_sync(0xffffffffu, s.phase != 0);
            if (mready && (__popc(mready) >= NW_REFILL || mbusy == 0)) {
                if (ready) {
                    it = nxt; nst = 0;
                    if (u2d(nbest) > tau_exit) {      // else: the element is already CUT, drop the item
                        const unsigned b = it.ak & 0x1fffffffu, k = it.ak >> 29;
                        fresh = true;
                        double uc, vc, hP, sc, tc, hQ;
                        nitem_box(it, uc, vc, hP, sc, tc, hQ);
                        // start at the first step k_np_bound took from the centre (local coordinates; on a bound when within float rounding of it)
                        const double a0 = nx0.x, a1 = nx0.y, a2 = nx0.z, a3 = nx0.w, e1 = 1.0 - 1e-6;
                        s.x[0] = a0 >= e1 ? uc + hP : (a0 <= -e1 ? uc - hP : fma(hP, a0, uc));
                        s.x[1] = a1 >= e1 ? vc + hP : (a1 <= -e1 ? vc - hP : fma(hP, a1, vc));
                        s.x[2] = a2 >= e1 ? sc + hQ : (a2 <= -e1 ? sc - hQ : fma(hQ, a2, sc));
                        s.x[3] = a3 >= e1 ? tc + hQ : (a3 <= -e1 ? tc - hQ : fma(hQ, a3, tc));
                        s.iters = 0; s.ls = 0; s.phase = 1;
                        pA = (unsigned long long)(ecoef + ((size_t)b * 6 + k) * 28);
                        pQ = (unsigned long long)(fcoef + (size_t)nface * 28);
                    }
                }
            }
        }
        // ---- lanes without a next item draw a ticket from the warp's pool; the pool is refilled NW_TICKETS at a time by
        // one atomic on the queue head whose result is looked at on a later trip (a ticket per lane per trip from the
        // head itself made 2 368 warps queue up on ONE address: the kernel ran at the pace of that atomic)
        {
            const unsigned m0 = __ballot_sync(0xffffffffu, nst == 0);
            if (m0) {
                const int avail = pool_end - pool_next, rank = __popc(m0 & lt_mask);
                if (nst == 0 && rank < avail) { tk = pool_next + rank; nst = 2; }
                pool_next += min(__popc(m0), avail);
            }
            if (pool_next == pool_end && !pend) {
                if (lane == 0) pbase = atomicAdd(head, chunk);
                pend = true;
            }
        }
        // ---- the new items' coefficients go into their lanes' slots by asynchronous copies (cp.async, 8 bytes per
        // lane), ALL issued before the one wait, so the new lanes of a trip cost one memory round trip together.
        // Warp-cooperative: the warp copies one new lane's 2 x 216 contiguous bytes at a time (~5 L1 wavefronts per new
        // lane; every new lane copying its own 54 coefficients cost 54, and the L1 data pipe -- shared-memory reads
        // of the coefficients plus these copies -- is the resource this kernel saturates).
        {
            unsigned mf = __ballot_sync(0xffffffffu, fresh);
            if (mf) {
                double *wslot = nw_sm + (tid & ~31);
                do {
                    const int L = __ffs(mf) - 1; mf &= mf - 1;
                    const double *a = (const double *)__shfl_sync(0xffffffffu, pA, L);
                    const double *q = (const double *)__shfl_sync(0xffffffffu, pQ, L);
                    const unsigned d0 = (unsigned)__cvta_generic_to_shared(wslot + L + lane * NW_STRIDE);
                    const double *g0 = lane < 27 ? a + lane : q + (lane - 27);
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(d0), "l"(g0));
                    if (lane < 22)
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(d0 + 32 * NW_STRIDE * 8), "l"(q + (lane + 5)));
                } while (mf);
                asm volatile("cp.async.wait_all;" ::: "memory");
            }
            __syncwarp();
        }
        if (__ballot_sync(0xffffffffu, s.phase != 0) == 0) {
            if (__ballot_sync(0xffffffffu, nst != 9 || sp > 0) == 0) break;
            continue;
        }
        // ---- one evaluation per busy lane
        bool fin = false;
        dcn::NwResult R; R.dist = 0.0; R.cosv = 0.0; R.converged = 0;
        // a solve that drags on looks, every 4th evaluation, whether its element has been found CUT meanwhile (by
        // another of its pairs): nothing it could still find would matter then.  The solves that do not converge are
        // almost all of this kind -- other patch pairs of an element the surface passes through, where the minimum
        // is a curve of zeros and the Hessian is singular -- and each used to cost two extra launches of sub-leaves.
        if (s.phase == 1 && s.iters >= 4 && (s.iters & 3) == 0 && u2d(__ldcg(best + (it.ak & 0x1fffffffu))) <= tau_exit) s.phase = 0;
        if (s.phase != 0) {
            // the leaf's box (dyadic, exact) is re-derived from the item every time instead of living in registers
            double uc, vc, hP, sc, tc, hQ;
            nitem_box(it, uc, vc, hP, sc, tc, hQ);
            const double lo[4] = { uc - hP, vc - hP, sc - hQ, tc - hQ }, hi[4] = { uc + hP, vc + hP, sc + hQ, tc + hQ };
            fin = dcn::iterate(cf, s, lo, hi, tol_d2, tau_exit2, R, maxit);
        }
        // ---- results of the solves that finished (an attained distance is an upper bound whether converged or not)
        bool resplit = false, splitP = false;
        if (fin) {
            const unsigned b = it.ak & 0x1fffffffu;
            cnt.newton++; cnt.iters += s.iters;
            s.phase = 0;
            atomicMin(best + b, d2u(R.dist));
            if (R.dist > tau_exit) {
                atomicMin(dmin + b, d2u(R.dist));
                const unsigned long long key = (d2u(R.dist) & ~0xffull) | (unsigned long long)cos_code(R.cosv);
                atomicMin(pair_key + it.p, key);
                if (!R.converged && !((it.w3 >> 24) & 1)) {
                    // unconverged: the distance above stands as an upper bound and the leaf is quartered (a seed solve is
                    // never split: the roots cover its pair).  With an overflow queue the four sub-leaves go there, for
                    // the next launch to spread over the machine: solved one after the other by this lane they were a
                    // serial chain of up to 5 x NW_MAXIT evaluations that the whole launch waited for (175 us of 690).
                    cnt.fail++;
                    if (u2d(__ldcg(best + b)) <= tau_exit) { /* the element is CUT by now: no sub-leaves */ }
                    else if (choose_split(it, (it.w2 & 15) <= ((it.w2 >> 4) & 15), max_level, splitP)) {
                        if (ovf) resplit = true;
                        else if (sp + 4 <= NW_STACK) {
#pragma unroll
                            for (int c = 0; c < 4; ++c) stk[sp++] = nitem_child(it, splitP, c);
                        } else cnt.depth++;
                    } else cnt.depth++;
                }
            }
        }
        if (ovf) {
            const long long sl = warp_reserve(ovf_n, resplit, 4, ovf_cap, &S->status);
            if (sl >= 0) {
#pragma unroll
                for (int c = 0; c < 4; ++c) ovf[sl + c] = nitem_child(it, splitP, c);
            }
        }
    }
    np_flush_counters(S, cnt);
}

// ------------------------------------------------------------------------------------------
// Roots: one warp per band element, lanes over its pairs.  (pair, patch k) survives when the
// box distance (Algorithm A.2) of the patch's Bezier box and the face's Bezier box is
// within best + t_tie; survivors become the items of round 0.
__global__ void __launch_bounds__(NPW_THREADS) k_np_roots(DcScalars *S, const long long *__restrict__ band_start,
                                                          const int *__restrict__ band_cnt, const int *__restrict__ pair_face,
                                                          const double *__restrict__ fbox, const double *__restrict__ pbox,
                                                          const unsigned long long *__restrict__ best,
                                                          NItem *__restrict__ qout, int *__restrict__ qout_n, long long qcap)
{
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * blockDim.x) >> 5;
    const int n_band = min(S->n_band, S->max_band);
    const double t_tie = S->t_tie, tau_exit = S->tau_exit;
    for (int b = warp; b < n_band; b += nwarps) {
        const double bst = u2d(best[b]);
        if (bst <= tau_exit) continue;                      // already CUT
        const double cut = bst + t_tie, cut2 = cut * cut;
        const long long p0 = band_start[b];
        const int cnt = band_cnt[b];
        const double *pb = pbox + (size_t)b * 36;
        for (int base = 0; base < cnt; base += 32) {
            const int pl = base + lane;
            unsigned mask = 0;
            if (pl < cnt) {
                const int f = __ldg(pair_face + p0 + pl);
                double fb[6];
#pragma unroll
                for (int m = 0; m < 6; ++m) fb[m] = __ldg(fbox + (size_t)f * 6 + m);
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    double d2 = 0.0;
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const double g = dmax2(0.0, dmax2(fb[c] - __ldg(pb + k * 6 + 3 + c), __ldg(pb + k * 6 + c) - fb[3 + c]));
                        d2 = fma(g, g, d2);
                    }
                    if (d2 <= cut2) mask |= 1u << k;
                }
            }
            const int mine = __popc(mask);
            int incl = mine;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            if (total == 0) continue;
            int start = 0;
            if (lane == 31) start = atomicAdd(qout_n, total);
            start = __shfl_sync(0xffffffffu, start, 31);
            long long slot = (long long)start + incl - mine;
            if ((long long)start + total > qcap) { if (lane == 0) atomicOr(&S->status, DC_STATUS_QUEUE_OVERFLOW); continue; }
            while (mask) {
                const int k = __ffs(mask) - 1; mask &= mask - 1;
                NItem it; it.p = (unsigned)(p0 + pl); it.ak = (unsigned)b | ((unsigned)k << 29); it.w2 = 0; it.w3 = 0;
                qout[slot++] = it;
            }
        }
    }
}

// First step of a leaf's closest-point solve, taken here where the centre evaluation already exists: the
// Gauss-Newton step of |r + P_u du + P_v dv - Q_s ds - Q_t dt|^2 from the centre, clamped to the leaf's box, in the
// leaf's local coordinates [-1,1]^4 (floats: it is a starting point).  Saves k_np_newton its evaluation at the centre.
__device__ __forceinline__ float4 leaf_first_step(const NodeOut &o, double hP, double hQ)
{
#define DOT3(A, B) (A[0] * B[0] + A[1] * B[1] + A[2] * B[2])
    // local variables a = du / hP ... : columns scaled by the half-widths
    const double h00 = hP * hP * DOT3(o.pu, o.pu), h01 = hP * hP * DOT3(o.pu, o.pv), h02 = -hP * hQ * DOT3(o.pu, o.qs), h03 = -hP * hQ * DOT3(o.pu, o.qt);
    const double h11 = hP * hP * DOT3(o.pv, o.pv), h12 = -hP * hQ * DOT3(o.pv, o.qs), h13 = -hP * hQ * DOT3(o.pv, o.qt);
    const double h22 = hQ * hQ * DOT3(o.qs, o.qs), h23 = hQ * hQ * DOT3(o.qs, o.qt), h33 = hQ * hQ * DOT3(o.qt, o.qt);
    const double g[4] = { hP * DOT3(o.r, o.pu), hP * DOT3(o.r, o.pv), -hQ * DOT3(o.r, o.qs), -hQ * DOT3(o.r, o.qt) };
#undef DOT3
    const double tr = h00 + h11 + h22 + h33;
    double p[4] = { 0.0, 0.0, 0.0, 0.0 };
    if (tr > 0.0) dcn::ldl4_mod(h00, h01, h02, h03, h11, h12, h13, h22, h23, h33, g, 1e-6 * tr, p);
    float4 x;
    x.x = (float)dmax2(-1.0, dmin2(1.0, p[0])); x.y = (float)dmax2(-1.0, dmin2(1.0, p[1]));
    x.z = (float)dmax2(-1.0, dmin2(1.0, p[2])); x.w = (float)dmax2(-1.0, dmin2(1.0, p[3]));
    return x;
}

// ------------------------------------------------------------------------------------------
// Bound: one thread per item of qin[0 .. n): prune, or 4 children -> qout, or leaf -> the ONE leaf queue nq
// (all rounds append to it; the Newton kernel runs once, after the last round).  Items i0, i0 + stride, ...
__device__ __forceinline__ void np_bound_items(DcScalars *S, int n, const NItem *__restrict__ qin,
                                               const int *__restrict__ pair_face, const double *__restrict__ fcoef,
                                               const double *__restrict__ ecoef, unsigned long long *__restrict__ best,
                                               NItem *__restrict__ qout, int *__restrict__ qout_n,
                                               NItem *__restrict__ nq, float4 *__restrict__ nqx, int *__restrict__ nq_n, long long qcap,
                                               int i0, int stride, NpCounters &cnt, bool force_leaf = false)
{
    const double t_tie = S->t_tie, tau_exit = S->tau_exit, theta2 = S->theta * S->theta;
    const int max_level = S->max_level;
    const int n_round = (n + 31) & ~31;
    for (int i = i0; i < n_round; i += stride) {
        bool split = false, leaf = false, splitP = false;
        NItem it; it.p = it.ak = it.w2 = it.w3 = 0;
        float4 x0 = make_float4(0.f, 0.f, 0.f, 0.f);
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
                const NodeOut o = bound_node(AP, AQ, AP[27], AQ[27], uc, vc, hP, sc, tc, hQ, theta2);
                cnt.nodes++;
                if (o.dist_c < bst) { atomicMin(best + b, d2u(o.dist_c)); bst = o.dist_c; }
                if (o.dist_c > tau_exit && o.lb <= bst + t_tie) {
                    leaf = o.leaf || force_leaf;     // (sub-leaves of an unconverged leaf stay leaves)
                    if (!leaf) {
                        split = choose_split(it, o.splitP, max_level, splitP);
                        if (!split) { leaf = true; cnt.depth++; }
                    }
                    if (leaf) x0 = leaf_first_step(o, hP, hQ);
                }
            }
        }
        const long long sl = warp_reserve(nq_n, leaf, 1, qcap, &S->status);
        if (sl >= 0) { nq[sl] = it; nqx[sl] = x0; }
        const long long slot = warp_reserve(qout_n, split, 4, qcap, &S->status);
        if (slot >= 0) {
#pragma unroll
            for (int c = 0; c < 4; ++c) qout[slot + c] = nitem_child(it, splitP, c);
        }
    }
}

__global__ void __launch_bounds__(NPW_THREADS) k_np_bound(DcScalars *S, const int *__restrict__ n_in, const NItem *__restrict__ qin,
                                                          const int *__restrict__ pair_face, const double *__restrict__ fcoef,
                                                          const double *__restrict__ ecoef, unsigned long long *__restrict__ best,
                                                          NItem *__restrict__ qout, int *__restrict__ qout_n,
                                                          NItem *__restrict__ nq, float4 *__restrict__ nqx, int *__restrict__ nq_n, long long qcap, int force_leaf)
{
    const int n = min(*n_in, (int)min(qcap, (long long)0x7fffffff));
    if (n == 0) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicMax(&S->c_queue_peak, (unsigned long long)n);
    NpCounters cnt = { 0, 0, 0, 0, 0 };
    np_bound_items(S, n, qin, pair_face, fcoef, ecoef, best, qout, qout_n, nq, nqx, nq_n, qcap,
                   blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x, cnt, force_leaf != 0);
    np_flush_counters(S, cnt);
}

// The rounds after the first few hold few items (deep levels exist only where the surface curves fast): ONE CTA
// walks them all, round after round, until a round comes up empty -- no launch per round, no empty launches.
#define NP_TAIL_THREADS 256
__global__ void __launch_bounds__(NP_TAIL_THREADS) k_np_bound_tail(DcScalars *S, int r_begin, int r_end, NItem *q0, NItem *q1,
                                                                   const int *__restrict__ pair_face, const double *__restrict__ fcoef,
                                                                   const double *__restrict__ ecoef, unsigned long long *__restrict__ best,
                                                                   NItem *__restrict__ nq, float4 *__restrict__ nqx, int *__restrict__ nq_n, long long qcap)
{
    NpCounters cnt = { 0, 0, 0, 0, 0 };
    for (int r = r_begin; r < r_end; ++r) {
        const int n = min(*(volatile int *)&S->qn[r], (int)min(qcap, (long long)0x7fffffff));
        if (n == 0) break;
        if (threadIdx.x == 0) atomicMax(&S->c_queue_peak, (unsigned long long)n);
        np_bound_items(S, n, (r & 1) ? q1 : q0, pair_face, fcoef, ecoef, best, (r & 1) ? q0 : q1, &S->qn[r + 1], nq, nqx, nq_n, qcap,
                       threadIdx.x, NP_TAIL_THREADS, cnt);
        __threadfence();
        __syncthreads();
    }
    np_flush_counters(S, cnt);
}

// ------------------------------------------------------------------------------------------
// S6 decide (L215: nearest face, dot of the minimal vector with its outward normal; ties L294):
// one thread per band element.
__global__ void k_np_decide(DcScalars *S, const int *__restrict__ band_elem, const long long *__restrict__ band_start,
                            const int *__restrict__ band_cnt, const unsigned long long *__restrict__ best,
                            const unsigned long long *__restrict__ dmin_arr, const unsigned long long *__restrict__ pair_key,
                            signed char *__restrict__ labels, double *__restrict__ sdist)
{
    const int n_band = min(S->n_band, S->max_band);
    const double tau = S->tau, tau_exit = S->tau_exit, amb = S->amb, t_tie = S->t_tie, d_band = S->d_band;
    unsigned n_amb = 0, n_samb = 0;
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < n_band; b += gridDim.x * blockDim.x) {   // (n_band is only known on the device)
        const int e = band_elem[b];
        const double dmin = u2d(dmin_arr[b]);
        if (u2d(best[b]) <= tau_exit) { labels[e] = DC_CUT; sdist[e] = 0.0; }
        else if (dmin <= tau) { labels[e] = DC_CUT; sdist[e] = 0.0; if (dmin >= tau - amb) ++n_amb; }
        else if (dmin < INFINITY) {
            if (dmin <= tau + amb) ++n_amb;
            int bestmag = -1, neg = 0, npos = 0, nneg = 0;
            const long long p0 = band_start[b];
            const int cnt = band_cnt[b];
            for (int p = 0; p < cnt; ++p) {
                const unsigned long long key = pair_key[p0 + p];
                const double dk = u2d(key & ~0xffull);
                if (dk <= dmin + t_tie) {
                    const int code = (int)(key & 0xff), mag = code & 0x7f, ng = code >> 7;
                    if (ng) ++nneg; else ++npos;
                    if (mag > bestmag) { bestmag = mag; neg = ng; }
                }
            }
            if (npos && nneg) ++n_samb;
            labels[e] = neg ? DC_HOLE : DC_NORMAL;
            const double d = dmin2(dmin, d_band);
            sdist[e] = neg ? -d : d;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { n_amb += __shfl_xor_sync(0xffffffffu, n_amb, o); n_samb += __shfl_xor_sync(0xffffffffu, n_samb, o); }
    if ((threadIdx.x & 31) == 0) {
        if (n_amb) atomicAdd(&S->c_ambiguous, (unsigned long long)n_amb);
        if (n_samb) atomicAdd(&S->c_sign_ambiguous, (unsigned long long)n_samb);
    }
}
