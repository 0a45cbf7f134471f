// dc_far.cuh -- DC_FLAG_EXACT_FAR: the exact distance of the elements BEYOND the band (second half;
// reading A5's alternative "exact everywhere, d_band = infinity").  The banded cut leaves those elements their label (flood
// fill, S7) and the clamp +-d_band; this pass replaces the clamp by +-d_e without a pair list of N_e x N_f entries.
//
// The face bins of S3 (64^3 cells, faces sorted by cell) get an octree on top (k_far_pyramid: levels 32^3 ... 1, one
// byte per cube = which of its 8 children hold faces).  The far elements walk that tree depth first, a WARP per 32
// consecutive elements with one walk for all of them (uniform control flow; each lane tests a face against its own
// element); the tests are single precision, rounded so that a distance is never overestimated:
//
//   k_far_nearest : nearest-bin traversal -- the child octant nearest to the element first, a subtree skipped once its box
//                   is no nearer than the nearest face BOX found so far.  That face becomes the element's seed pair; the seed
//                   solve of the narrow phase (k_np_solve, unchanged) turns it into an ATTAINED distance ub >= d_e.
//   k_far_count / : every face whose box is within ub (the box test of Algorithm A.2, with the
//   k_far_pairs     element's own cutoff instead of the band's) AND which a second bound along the line of centres does not
//                   put beyond ub (far_dir_lb) is a candidate pair: subtrees farther than ub are skipped, so the walk
//                   costs about the candidates it finds, not N_f.
//
// The candidate pairs then go through the SAME narrow phase as the band's (k_np_roots, k_np_bound, k_np_solve: nothing
// is pruned below the true minimum because best[] starts at the attained ub, not at the band's reach), and k_far_decide
// writes sdist = +-d_e with the sign the flood fill gave.
//
// Far elements have many more candidates than band elements (far from a round body a hundred faces are about as near as
// the nearest), so the pairs are made and solved in PASSES sized to the workspace: in each pass the warps that still wait
// ask for the slots of their 32 elements at one counter, all or nothing, until the list is full; the host reads two
// counters per pass.  Deep inside a round body EVERY face is about as near as the next one: an element with more than
// FAR_HEAVY candidates, or whose warp has walked past n_face / 24 faces, leaves the walk and is counted and listed by
// brute force instead (k_far_heavy_count / k_far_heavy_pairs: a CTA per element, a thread per face) -- a pass lasts as
// long as its slowest warp.
//
// Launch order (run_exact_far): pyramid, faces, list, [codes, scan, sort], nearest; per slice of max_band elements:
// slots, k_np_stage, k_np_solve(seeds), count(refine: a better seed face), k_np_solve(seeds), count, heavy_count; per pass: pairs, heavy_pairs, fix, k_np_roots ... the last
// k_np_solve, decide.
#pragma once

#define DC_FAR_STACK 48             /* 7 pushed siblings per level x 6 levels + 1 */
#define DC_PYR_TOTAL 37449          /* 32^3 + 16^3 + 8^3 + 4^3 + 2^3 + 1 */

__device__ __forceinline__ int pyr_off(int L)    // first entry of level L (1 .. 6); level L has (64 >> L)^3 entries
{
    return L == 1 ? 0 : (L == 2 ? 32768 : (L == 3 ? 36864 : (L == 4 ? 37376 : (L == 5 ? 37440 : 37448))));
}

// which children of a cube of 2^L cells hold faces (bit k: child (k & 1, k >> 1 & 1, k >> 2)); a row of cells along x is
// one range of the sorted faces
__global__ void k_far_pyramid(const int *__restrict__ cell_start, unsigned char *__restrict__ pmask)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= DC_PYR_TOTAL) return;
    int L = 1;
    while (L < 6 && t >= pyr_off(L + 1)) ++L;
    const int n = DC_GRID_MAX >> L, h = 1 << (L - 1), idx = t - pyr_off(L);
    const int x = idx % n, y = (idx / n) % n, z = idx / (n * n);
    unsigned mask = 0;
    for (int k = 0; k < 8; ++k) {
        const int x0 = (2 * x + (k & 1)) * h, y0 = (2 * y + ((k >> 1) & 1)) * h, z0 = (2 * z + (k >> 2)) * h;
        int cnt = 0;
        for (int zz = z0; zz < z0 + h && !cnt; ++zz)
            for (int yy = y0; yy < y0 + h; ++yy) {
                const int c0 = cell_code(x0, yy, zz);
                cnt += __ldg(cell_start + c0 + h) - __ldg(cell_start + c0);
            }
        if (cnt) mask |= 1u << k;
    }
    pmask[t] = (unsigned char)mask;
}

// ---- the walk.  A WARP takes 32 consecutive far elements (consecutive in the list = neighbours in the grid, mostly) and
// walks the tree ONCE for all of them, with the box that holds all 32 and the largest of their cutoffs: control flow is
// uniform, a face's data is loaded once per warp (broadcast), and each lane tests the face against its OWN element.
struct FarLane {
    float lo[3], hi[3];     // the element box in units of cells relative to the grid origin (from the doubles), rounded outward
    float cen[3], half[3];  // a centre and half-edges that hold the box about it (rounded up)
    float glo[3], ghi[3];   // the box grown by what a face may overhang its cell (faces are binned by box centre: at most fhalf)
    bool on;
};

__device__ __forceinline__ FarLane far_lane(const DcScalars *S, const double *__restrict__ ebox, long long n_elem, long long e, bool on)
{
    FarLane q; q.on = on;
    const double inv = S->inv_cell;
    const float infl = __double2float_ru(S->fhalf * S->inv_cell + 1e-6);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        q.lo[c] = on ? __double2float_rd((ebox[(size_t)c * n_elem + e] - S->origin[c]) * inv - 1e-9) : 0.f;
        q.hi[c] = on ? __double2float_ru((ebox[(size_t)(3 + c) * n_elem + e] - S->origin[c]) * inv + 1e-9) : 0.f;
        q.cen[c] = 0.5f * (q.lo[c] + q.hi[c]);
        q.half[c] = fmaxf(__fsub_ru(q.hi[c], q.cen[c]), __fsub_ru(q.cen[c], q.lo[c]));
        q.glo[c] = __fsub_rd(q.lo[c], infl); q.ghi[c] = __fadd_ru(q.hi[c], infl);
    }
    return q;
}
// a distance (double, length units) as a cutoff in cell units, rounded up
__device__ __forceinline__ float far_cut(const DcScalars *S, double d) { return __double2float_ru(d * S->inv_cell * (1.0 + 1e-9)); }

__device__ __forceinline__ float warp_min_f(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ float warp_max_f(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// the centre of the warp's elements (the octant order of the nearest-first walk)
struct FarGroup { float cen[3]; };

__device__ __forceinline__ FarGroup far_group(const FarLane &q)
{
    FarGroup g;
#pragma unroll
    for (int c = 0; c < 3; ++c) g.cen[c] = 0.5f * (warp_min_f(q.on ? q.lo[c] : INFINITY) + warp_max_f(q.on ? q.hi[c] : -INFINITY));
    return g;
}

// squared distance (cell units, never overestimated) between the lane's grown box and the cube (x, y, z) of level L
__device__ __forceinline__ float far_lb2(const FarLane &q, int L, int x, int y, int z)
{
    const float s = (float)(1 << L);
    const int xi[3] = { x, y, z };
    float d2 = 0.f;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float nlo = (float)xi[c] * s, nhi = nlo + s;            // (exact)
        const float gp = fmaxf(0.f, fmaxf(__fsub_rd(nlo, q.ghi[c]), __fsub_rd(q.glo[c], nhi)));
        d2 = __fadd_rd(d2, __fmul_rd(gp, gp));
    }
    return d2;
}

// squared box distance (cell units) of the lane's element and a face (boxes rounded outward, gaps and squares rounded
// down: never overestimated)
__device__ __forceinline__ float far_box_d2(const FarLane &q, const float4 flo, const float4 fhi)
{
    const float gx = fmaxf(0.f, fmaxf(__fsub_rd(flo.x, q.hi[0]), __fsub_rd(q.lo[0], fhi.x)));
    const float gy = fmaxf(0.f, fmaxf(__fsub_rd(flo.y, q.hi[1]), __fsub_rd(q.lo[1], fhi.y)));
    const float gz = fmaxf(0.f, fmaxf(__fsub_rd(flo.z, q.hi[2]), __fsub_rd(q.lo[2], fhi.z)));
    return __fadd_rd(__fadd_rd(__fmul_rd(gx, gx), __fmul_rd(gy, gy)), __fmul_rd(gz, gz));
}

// A second lower bound, along the line of centres n (any unit n gives one: dist >= n.(c_f - c_e) - supp_e(n) - supp_f(-n)).
// The element is its box (support sum |n_c| half_c); the face lies in a flat cylinder about its centre (k_far_faces: axis =
// the normal at the centre, half-thickness t, radius r; support |n.axis| t + sqrt(1 - (n.axis)^2) r).  Seen from far away a
// face's own box is as thick as the face is wide whenever its normal is off the axes, and every face within a wide cap
// of the surface passes the box test; along the line of centres the nearby faces are seen face on and only their real
// thickness counts.  Cell units relative to the grid origin (coordinates are O(64) or O(distance): single precision is
// good to 1e-7 of that), with the slack below: never overestimated.
__device__ __forceinline__ float far_dir_lb(const FarLane &q, float cx, float cy, float cz, const float4 ax, const float4 tr)
{
    const float dx = cx - q.cen[0], dy = cy - q.cen[1], dz = cz - q.cen[2];
    const float D2 = dx * dx + dy * dy + dz * dz;
    if (!(D2 > 0.f)) return 0.f;
    const float rD = rsqrtf(D2), D = D2 * rD;
    const float nx = dx * rD, ny = dy * rD, nz = dz * rD;
    const float se = fabsf(nx) * q.half[0] + fabsf(ny) * q.half[1] + fabsf(nz) * q.half[2];
    const float ca = fabsf(nx * ax.x + ny * ax.y + nz * ax.z);
    const float sa = sqrtf(fmaxf(0.f, 1.f - ca * ca) + 1e-5f);
    const float sf = fminf(ca, 1.f) * tr.x + sa * tr.y;
    return D - se - sf - 1e-5f * (D + se + sf) - 1e-4f;
}

// Depth-first walk, uniform over the warp, of the cubes that hold faces and are within the cutoff of AT LEAST ONE lane
// (each lane tests the cube against its own box and its own squared cutoff cut2, cell units; one vote): the cubes walked
// are the union of what the 32 elements would walk alone.  cell(p0, p1) is called (by all lanes) for every such cell with
// the range of its faces; it returns true (uniformly) to end the walk, and may switch lanes off (q.on).  ORDERED: nearest
// octant first, strict test, and the lanes' cutoffs may shrink on the way.
// (Fetching for 32 cubes at a time, lane by lane, with the face records prefetched into L1, was tried: no gain -- a step
// costs what its hundred dependent instructions cost a lone warp, not its loads; the throughput comes from the warps.)
template <bool ORDERED, class F>
__device__ __forceinline__ void far_walk(const FarLane &q, const FarGroup &g, const float &cut2, const int *__restrict__ cell_start,
                                         const unsigned char *__restrict__ pmask, unsigned *stack, F &&cell)
{
    int top = 0;
    stack[top++] = 6u << 18;            // (level << 18) | (z << 12) | (y << 6) | x; every lane writes the same words
    while (top > 0) {
        const unsigned nd = stack[--top];
        const int L = (int)(nd >> 18), x = (int)(nd & 63u), y = (int)((nd >> 6) & 63u), z = (int)((nd >> 12) & 63u);
        if (ORDERED && !__any_sync(0xffffffffu, q.on && far_lb2(q, L, x, y, z) < cut2)) continue;   // (the cutoffs have shrunk since the push)
        if (L == 0) {
            const int c = cell_code(x, y, z);
            if (cell(__ldg(cell_start + c), __ldg(cell_start + c + 1))) break;      // (the caller has seen enough)
            continue;
        }
        const unsigned mask = __ldg(pmask + pyr_off(L) + x + (DC_GRID_MAX >> L) * (y + (DC_GRID_MAX >> L) * z));
        // the octant of this cube nearest to the group: pushed last, popped first
        const float half = (float)(1 << (L - 1));
        const int oct = (g.cen[0] >= (float)(2 * x + 1) * half ? 1 : 0) | (g.cen[1] >= (float)(2 * y + 1) * half ? 2 : 0) |
                        (g.cen[2] >= (float)(2 * z + 1) * half ? 4 : 0);
#pragma unroll
        for (int j = 7; j >= 0; --j) {
            const int k = ORDERED ? (j ^ oct) : j;
            if (!((mask >> k) & 1u)) continue;
            const int cx = 2 * x + (k & 1), cy = 2 * y + ((k >> 1) & 1), cz = 2 * z + (k >> 2);
            const float lb2 = far_lb2(q, L - 1, cx, cy, cz);
            if (!__any_sync(0xffffffffu, q.on && (ORDERED ? lb2 < cut2 : lb2 <= cut2))) continue;
            if (top < DC_FAR_STACK) stack[top++] = ((unsigned)(L - 1) << 18) | ((unsigned)cz << 12) | ((unsigned)cy << 6) | (unsigned)cx;
        }
    }
}

// per face (sorted order), in units of cells relative to the grid origin: its box, its centre, the unit normal at the
// centre, and the flat cylinder about them that holds the patch's Bezier control points (hence the patch):
// ffar[p] = { box lo | c.x }, { box hi | c.y }, { n | c.z }, { t, r, -, - }; boxes rounded outward, t and r up
__global__ void k_far_faces(const DcScalars *S, const double *__restrict__ fcoef, const double *__restrict__ fbox, int n_face,
                            float *__restrict__ ffar)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_face) return;
    const double inv = S->inv_cell;
    const double *A = fcoef + (size_t)p * 28;
    double B[3][9];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double *a = A + 9 * c;
        double r[3][3];
#pragma unroll
        for (int j = 0; j < 3; ++j) mono_to_bern(a[3 * j], a[3 * j + 1], a[3 * j + 2], r[j][0], r[j][1], r[j][2]);
#pragma unroll
        for (int i = 0; i < 3; ++i) mono_to_bern(r[0][i], r[1][i], r[2][i], B[c][i], B[c][3 + i], B[c][6 + i]);
    }
    const float cf[3] = { (float)((A[0] - S->origin[0]) * inv), (float)((A[9] - S->origin[1]) * inv), (float)((A[18] - S->origin[2]) * inv) };
    const double ux = A[1], uy = A[10], uz = A[19], vx = A[3], vy = A[12], vz = A[21];
    double nx = uy * vz - uz * vy, ny = uz * vx - ux * vz, nz = ux * vy - uy * vx;
    const double nn = sqrt(nx * nx + ny * ny + nz * nz);
    if (nn > 0.0) { nx /= nn; ny /= nn; nz /= nn; } else { nx = 1.0; ny = 0.0; nz = 0.0; }
    // t and r are measured against the single-precision centre and axis the test will use
    const float fx = (float)nx, fy = (float)ny, fz = (float)nz;
    const double ax = fx, ay = fy, az = fz, an = sqrt(ax * ax + ay * ay + az * az);
    double t = 0.0, r2 = 0.0;
#pragma unroll
    for (int m = 0; m < 9; ++m) {
        const double dx = (B[0][m] - S->origin[0]) * inv - (double)cf[0], dy = (B[1][m] - S->origin[1]) * inv - (double)cf[1],
                     dz = (B[2][m] - S->origin[2]) * inv - (double)cf[2];
        const double h = (dx * ax + dy * ay + dz * az) / an;
        t = dmax2(t, fabs(h));
        r2 = dmax2(r2, dx * dx + dy * dy + dz * dz - h * h);
    }
    float4 *o = reinterpret_cast<float4 *>(ffar) + (size_t)p * 4;
    const double *fb = fbox + (size_t)p * 6;
    o[0] = make_float4(__double2float_rd((fb[0] - S->origin[0]) * inv - 1e-9), __double2float_rd((fb[1] - S->origin[1]) * inv - 1e-9),
                       __double2float_rd((fb[2] - S->origin[2]) * inv - 1e-9), cf[0]);
    o[1] = make_float4(__double2float_ru((fb[3] - S->origin[0]) * inv + 1e-9), __double2float_ru((fb[4] - S->origin[1]) * inv + 1e-9),
                       __double2float_ru((fb[5] - S->origin[2]) * inv + 1e-9), cf[1]);
    o[2] = make_float4(fx, fy, fz, cf[2]);
    o[3] = make_float4(__double2float_ru(t * 1.000001 + 1e-9), __double2float_ru(sqrt(dmax2(r2, 0.0)) * 1.000001 + 1e-9), 0.f, 0.f);
}

// the elements the banded cut left clamped: not CUT and |sdist| = d_band (elements of the band whose distance turned out
// to exceed d_band included); also the box that holds their centres (for the ordering below)
__global__ void k_far_list(DcScalars *S, long long n_elem, const signed char *__restrict__ labels, const double *__restrict__ sdist,
                           const double *__restrict__ ebox, int *__restrict__ list)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const double d_band = S->d_band;
    const bool far = e < n_elem && labels[e] != DC_CUT && labels[e] >= 0 && fabs(sdist[e]) >= d_band;
    const unsigned m = __ballot_sync(0xffffffffu, far);
    if (!m) return;
    const int lane = threadIdx.x & 31;
    int base = 0;
    if (lane == (__ffs(m) - 1)) base = atomicAdd(&S->far_n[0], __popc(m));
    base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
    if (far) list[base + __popc(m & ((1u << lane) - 1))] = (int)e;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double lo = far ? 0.5 * (ebox[(size_t)c * n_elem + e] + ebox[(size_t)(3 + c) * n_elem + e]) : INFINITY, hi = far ? lo : -INFINITY;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { lo = dmin2(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = dmax2(hi, __shfl_xor_sync(0xffffffffu, hi, o)); }
        if (lane == 0) { atomicMin(&S->far_lo[c], enc_ord(lo)); atomicMax(&S->far_hi[c], enc_ord(hi)); }
    }
}

// The walks below take 32 elements at a time, and pay for the box that holds all 32: the far elements are put in the order
// of the Morton code of their centre in a 64^3 grid over their bounding box (counting sort: histogram, the scan of S3,
// scatter), so that 32 neighbours in the list are a compact block in space whatever the numbering of the grid.
__device__ __forceinline__ unsigned spread3(unsigned v)
{
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000ffu; v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;  v = (v | (v << 2)) & 0x09249249u;
    return v;
}
__global__ void k_far_codes(const DcScalars *S, const int *__restrict__ list, const double *__restrict__ ebox, long long n_elem,
                            int *__restrict__ code, int *bin_count)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S->far_n[0]) return;
    const long long e = list[i];
    unsigned b[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double lo = dec_ord(S->far_lo[c]), hi = dec_ord(S->far_hi[c]);
        const double x = 0.5 * (ebox[(size_t)c * n_elem + e] + ebox[(size_t)(3 + c) * n_elem + e]);
        const int k = hi > lo ? (int)((x - lo) / (hi - lo) * 64.0) : 0;
        b[c] = (unsigned)(k < 0 ? 0 : (k > 63 ? 63 : k));
    }
    const int cd = (int)(spread3(b[0]) | (spread3(b[1]) << 1) | (spread3(b[2]) << 2));
    code[i] = cd;
    atomicAdd(&bin_count[cd], 1);
}
__global__ void k_far_sort(const DcScalars *S, const int *__restrict__ list, const int *__restrict__ code,
                           const int *__restrict__ bin_start, int *bin_fill, int *__restrict__ sorted)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S->far_n[0]) return;
    const int cd = code[i];
    sorted[bin_start[cd] + atomicAdd(&bin_fill[cd], 1)] = list[i];
}

// every far element at once: the face with the nearest box (one warp per 32 elements of the list)
#define FAR_WARPS 4
#define FAR_NEAREST_CAP 1024        /* faces a warp looks at for its 32 seeds */
#ifndef FAR_HEAVY
#define FAR_HEAVY 128               /* candidates beyond which an element leaves the walk for the brute-force kernels */
#endif
#ifndef FAR_WARP_CAP_DIV
#define FAR_WARP_CAP_DIV 24         /* a warp that has visited n_face / 24 faces (at least 1024) gives up its walk: the elements it still
                                       walks for go to the brute-force kernels, which cost n_face tests each */
#endif
#ifndef FAR_REFINE_CAP_MUL
#define FAR_REFINE_CAP_MUL 4        /* the walk for a better seed may visit this many times as many */
#endif
#define FAR_HEAVY_BIT (1 << 30)
__global__ void __launch_bounds__(FAR_WARPS * 32) k_far_nearest(DcScalars *S, const int *__restrict__ list, int n,
                                                                const double *__restrict__ ebox, long long n_elem,
                                                                const int *__restrict__ cell_start, const unsigned char *__restrict__ pmask,
                                                                const float *__restrict__ ffar, int *__restrict__ fstar)
{
    __shared__ unsigned s_stack[FAR_WARPS][DC_FAR_STACK];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if ((i & ~31) >= n) return;                         // (whole warps only)
    const bool on = i < n;
    const FarLane q = far_lane(S, ebox, n_elem, on ? list[i] : 0, on);
    const FarGroup g = far_group(q);
    float best = on ? INFINITY : 0.f;                   // squared box distance of the nearest face box so far
    float cut2 = best;                                  // (+ a hair: a lane's nearest cube must not be lost to rounding)
    int f = 0;
    // (the seed only has to be near: where every face is about as near as the next one -- deep inside a round body -- the
    // walk would visit them all; the nearest octant comes first, so what FAR_NEAREST_CAP faces have shown is near enough)
    int seen = 0;
    far_walk<true>(q, g, cut2, cell_start, pmask, s_stack[threadIdx.x >> 5], [&](int p0, int p1) {
        for (int p = p0; p < p1; ++p) {
            const float4 *fp = reinterpret_cast<const float4 *>(ffar) + (size_t)p * 4;
            const float d2 = far_box_d2(q, __ldg(fp), __ldg(fp + 1));
            if (d2 < best) { best = d2; f = p; cut2 = best * 1.0001f + 1e-6f; }
        }
        seen += p1 - p0;
        return seen >= FAR_NEAREST_CAP;
    });
    if (on) fstar[i] = f;
}

// start of a slice of m far elements: they are the "band" of the narrow-phase launches that follow, slot i = position in
// the slice; pair i is element i's seed pair until the first pass overwrites the pair list
__global__ void k_far_reset(DcScalars *S, int m, int first)
{
    if (first) S->n_band = m;
    S->n_pairs = first ? (unsigned long long)m : 0ull;
    S->far_end = 0ull;
    for (int i = 0; i < DC_NQN; ++i) { S->qn[i] = 0; S->nn[i] = 0; S->nh[i] = 0; }
    S->nh[DC_NQN] = 0;
    S->far_pass_done = 0;
    if (first) S->far_nheavy = 0;
    S->far_nheavy_pass = 0;
}

__global__ void k_far_slots(const int *__restrict__ list, const int *__restrict__ fstar, int m,
                            int *__restrict__ band_elem, long long *__restrict__ band_start, int *__restrict__ band_cnt,
                            int *__restrict__ pair_face, unsigned long long *__restrict__ pair_key,
                            int *__restrict__ pair_band, NItem *__restrict__ seed_q,
                            unsigned long long *__restrict__ best, unsigned long long *__restrict__ dmin)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    band_elem[i] = list[i]; band_start[i] = -1; band_cnt[i] = 0;
    pair_face[i] = fstar[i]; pair_key[i] = 0x7ff0000000000000ull; pair_band[i] = i;
    best[i] = 0x7fe0000000000000ull;            // (no cutoff yet: the seed solve sets it)
    dmin[i] = 0x7ff0000000000000ull;
    NItem it; it.p = (unsigned)i; it.ak = (unsigned)i | (7u << 29); it.w2 = 0; it.w3 = 1u << 24;
    seed_q[i] = it;
}

// after the seed solves: how many faces pass both tests against the element's attained distance (the seed's face is one)
__device__ __forceinline__ bool far_hit(const FarLane &q, float cutf, float cut2f, const float *__restrict__ ffar, int p)
{
    const float4 *fp = reinterpret_cast<const float4 *>(ffar) + (size_t)p * 4;
    const float4 blo = __ldg(fp), bhi = __ldg(fp + 1);
    if (!(far_box_d2(q, blo, bhi) <= cut2f)) return false;
    const float4 ax = __ldg(fp + 2);
    return far_dir_lb(q, blo.w, bhi.w, ax.w, ax, __ldg(fp + 3)) <= cutf;
}

__global__ void __launch_bounds__(FAR_WARPS * 32) k_far_count(DcScalars *S, const double *__restrict__ ebox, long long n_elem,
                                                              const int *__restrict__ cell_start, const unsigned char *__restrict__ pmask,
                                                              const float *__restrict__ ffar, const int *__restrict__ band_elem,
                                                              int *__restrict__ band_cnt, const unsigned long long *__restrict__ best,
                                                              int *__restrict__ heavy_list, int *__restrict__ pair_face, int refine)
{
    __shared__ unsigned s_stack[FAR_WARPS][DC_FAR_STACK];
    const int i = blockIdx.x * blockDim.x + threadIdx.x, n = S->n_band;
    if ((i & ~31) >= n) return;
    const bool on = i < n;
    FarLane q = far_lane(S, ebox, n_elem, on ? band_elem[i] : 0, on);
    // refine: no count -- among the candidates, the face (other than the seed's) whose CENTRE is nearest becomes the pair of a
    // second seed solve.  The first seed is the face with the nearest box, a bound from below that a tilted face wins for
    // the wrong reason; among the faces that bound has not excluded, the centre distance (a proxy from above) picks better,
    // and every bit the attained distance comes down by takes candidates off the list.
    const int seed_face = (refine && on) ? pair_face[i] : -1;
    int alt = -1;
    float alt_d2 = INFINITY;
    const FarGroup g = far_group(q);
    const float cutf = on ? far_cut(S, u2d(best[i]) + S->t_tie) : 0.f, cut2f = __fmul_ru(cutf, cutf);
    const float cutg = cut2f * 1.0001f + 1e-6f;        // (for the cubes: + a hair against the rounding of two distances)
    int cnt = 0;
    // An element with more than FAR_HEAVY candidates (deep inside a round body every face is about as near as the next
    // one) leaves the walk -- it would drag its whole warp over most of the surface -- and is counted, and later listed,
    // by the brute-force kernels below, a CTA per element over all faces.  So do the elements a warp is still walking
    // for after warp_cap faces: a pass lasts as long as its slowest warp.
    int seen = 0;
    const int warp_cap = max(1024, S->n_face / FAR_WARP_CAP_DIV);
    far_walk<false>(q, g, cutg, cell_start, pmask, s_stack[threadIdx.x >> 5], [&](int p0, int p1) {
        if (refine) {
            for (int p = p0; p < p1; ++p)
                if (q.on && p != seed_face && far_hit(q, cutf, cut2f, ffar, p)) {
                    const float4 *fp = reinterpret_cast<const float4 *>(ffar) + (size_t)p * 4;
                    const float ex = __ldg(fp).w - q.cen[0], ey = __ldg(fp + 1).w - q.cen[1], ez = __ldg(fp + 2).w - q.cen[2];
                    const float d2 = ex * ex + ey * ey + ez * ez;
                    if (d2 < alt_d2) { alt_d2 = d2; alt = p; }
                }
            seen += p1 - p0;
            return seen > warp_cap * FAR_REFINE_CAP_MUL;
        }
        for (int p = p0; p < p1; ++p) if (q.on && far_hit(q, cutf, cut2f, ffar, p) && ++cnt > FAR_HEAVY) q.on = false;
        seen += p1 - p0;
        if (seen > warp_cap && q.on) { cnt = FAR_HEAVY + 1; q.on = false; }
        return !__any_sync(0xffffffffu, q.on);
    });
    if (refine) { if (on && alt >= 0) pair_face[i] = alt; return; }
    if (on) {
        const bool heavy = cnt > FAR_HEAVY;
        band_cnt[i] = heavy ? FAR_HEAVY_BIT : cnt;
        if (heavy) heavy_list[atomicAdd(&S->far_nheavy, 1)] = i;
    }
}

// brute force for the heavy elements: a CTA per element, a thread per face
#define FAR_HEAVY_THREADS 256
__global__ void __launch_bounds__(FAR_HEAVY_THREADS) k_far_heavy_count(const DcScalars *S, const double *__restrict__ ebox, long long n_elem,
                                                                       const float *__restrict__ ffar, const int *__restrict__ band_elem,
                                                                       int *__restrict__ band_cnt, const unsigned long long *__restrict__ best,
                                                                       const int *__restrict__ heavy_list)
{
    __shared__ int s_warp[FAR_HEAVY_THREADS / 32];
    const int nh = S->far_nheavy, nf = S->n_face;
    for (int h = blockIdx.x; h < nh; h += gridDim.x) {
        const int i = heavy_list[h];
        const FarLane q = far_lane(S, ebox, n_elem, band_elem[i], true);
        const float cutf = far_cut(S, u2d(best[i]) + S->t_tie), cut2f = __fmul_ru(cutf, cutf);
        int cnt = 0;
        for (int p = threadIdx.x; p < nf; p += FAR_HEAVY_THREADS) cnt += far_hit(q, cutf, cut2f, ffar, p) ? 1 : 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
        if ((threadIdx.x & 31) == 0) s_warp[threadIdx.x >> 5] = cnt;
        __syncthreads();
        if (threadIdx.x == 0) {
            int t = 0;
            for (int w = 0; w < FAR_HEAVY_THREADS / 32; ++w) t += s_warp[w];
            band_cnt[i] = t | FAR_HEAVY_BIT;
        }
        __syncthreads();
    }
}
// ... and the pairs of the heavy elements that got their slots in this pass (k_far_pairs lists them): faces in order
__global__ void __launch_bounds__(FAR_HEAVY_THREADS) k_far_heavy_pairs(const DcScalars *S, const double *__restrict__ ebox, long long n_elem,
                                                                       const float *__restrict__ ffar, const int *__restrict__ band_elem,
                                                                       const long long *__restrict__ band_start,
                                                                       const unsigned long long *__restrict__ best,
                                                                       const int *__restrict__ pass_list,
                                                                       int *__restrict__ pair_face, unsigned long long *__restrict__ pair_key,
                                                                       int *__restrict__ pair_band)
{
    __shared__ int s_warp[FAR_HEAVY_THREADS / 32];
    const int nh = S->far_nheavy_pass, nf = S->n_face;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int h = blockIdx.x; h < nh; h += gridDim.x) {
        const int i = pass_list[h];
        const FarLane q = far_lane(S, ebox, n_elem, band_elem[i], true);
        const float cutf = far_cut(S, u2d(best[i]) + S->t_tie), cut2f = __fmul_ru(cutf, cutf);
        long long j = band_start[i];
        for (int p0 = 0; p0 < nf; p0 += FAR_HEAVY_THREADS) {
            const int p = p0 + threadIdx.x;
            const bool hit = p < nf && far_hit(q, cutf, cut2f, ffar, p);
            const unsigned hm = __ballot_sync(0xffffffffu, hit);
            if (lane == 0) s_warp[wid] = __popc(hm);
            __syncthreads();
            int before = 0, total = 0;
#pragma unroll
            for (int w = 0; w < FAR_HEAVY_THREADS / 32; ++w) { const int v = s_warp[w]; if (w < wid) before += v; total += v; }
            if (hit) { const long long w = j + before + __popc(hm & ((1u << lane) - 1u)); pair_face[w] = p; pair_key[w] = 0x7ff0000000000000ull; pair_band[w] = i; }
            j += total;
            __syncthreads();
        }
    }
}

// One pass: every waiting element (band_cnt > 0) asks for its pair slots at ONE counter that is never wound back -- the
// first element that does not fit pushes it past the capacity, so every later one fails too and the slots given out are
// exactly [0, far_end) without holes.  The lanes that got their slots walk the tree again (as a group) and write their
// pairs; the others wait for the next pass (the first to ask always fits, unless its candidates alone exceed a pass:
// far_want).
__global__ void __launch_bounds__(FAR_WARPS * 32) k_far_pairs(DcScalars *S, const double *__restrict__ ebox, long long n_elem,
                                                              const int *__restrict__ cell_start, const unsigned char *__restrict__ pmask,
                                                              const float *__restrict__ ffar, const int *__restrict__ band_elem,
                                                              long long *__restrict__ band_start, const int *__restrict__ band_cnt,
                                                              int *__restrict__ pair_face, unsigned long long *__restrict__ pair_key,
                                                              int *__restrict__ pair_band, const unsigned long long *__restrict__ best,
                                                              long long cap_pairs, int *__restrict__ pass_list)
{
    __shared__ unsigned s_stack[FAR_WARPS][DC_FAR_STACK];
    const int i = blockIdx.x * blockDim.x + threadIdx.x, n = S->n_band;
    if ((i & ~31) >= n) return;
    const int raw = i < n ? band_cnt[i] : -1;         // (-1: done in an earlier pass)
    bool heavy = raw >= 0 && (raw & FAR_HEAVY_BIT) != 0;
    int cnt = raw >= 0 ? (raw & ~FAR_HEAVY_BIT) : 0;
    if (cnt > cap_pairs) { atomicMax(&S->far_want, (unsigned long long)cnt); cnt = 0; }
    // the warp asks for the slots of all its waiting lanes at once, all or nothing: the lanes of a pass are whole warps
    // (a walk costs the same for one lane as for 32), and the counter sees one atomic per warp.  The warp's range holds
    // first the pairs of its light lanes, in the order the walk meets them, then a range per heavy lane.
    const int lane = threadIdx.x & 31;
    int incl_h = heavy ? cnt : 0, light = heavy ? 0 : cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl_h, o); if (lane >= o) incl_h += v; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) light += __shfl_xor_sync(0xffffffffu, light, o);
    const int total = light + __shfl_sync(0xffffffffu, incl_h, 31);
    if (total == 0) return;
    unsigned long long old = 0;
    if (lane == 0) {
        old = total <= cap_pairs ? atomicAdd(&S->n_pairs, (unsigned long long)total) : ~0ull;
        if (old != ~0ull && old + (unsigned long long)total > (unsigned long long)cap_pairs) old = ~0ull;
        if (old != ~0ull) atomicMax(&S->far_end, old + (unsigned long long)total);
    }
    old = __shfl_sync(0xffffffffu, old, 0);
    long long hbase = 0;
    if (old == ~0ull) {
        // (a warp whose lanes together exceed a pass, though none does alone: one lane per pass, the first that waits)
        if (total <= cap_pairs) return;
        const unsigned waiting = __ballot_sync(0xffffffffu, cnt > 0);
        const int leader = __ffs(waiting) - 1;
        if (lane == leader) {
            old = atomicAdd(&S->n_pairs, (unsigned long long)cnt);
            if (old + (unsigned long long)cnt > (unsigned long long)cap_pairs) old = ~0ull;
            else atomicMax(&S->far_end, old + (unsigned long long)cnt);
        } else cnt = 0;
        old = __shfl_sync(0xffffffffu, old, leader);
        if (old == ~0ull) return;
        hbase = (long long)old;
    } else hbase = (long long)old + light + incl_h - cnt;
    if (cnt == 0) heavy = false;
    if (heavy) { band_start[i] = hbase; pass_list[atomicAdd(&S->far_nheavy_pass, 1)] = i; }
    const bool on = cnt > 0 && !heavy;
    if (on) band_start[i] = (long long)old;           // (>= 0: this element's pairs are in the list of this pass)
    if (!__any_sync(0xffffffffu, on)) return;
    const FarLane q = far_lane(S, ebox, n_elem, on ? band_elem[i] : 0, on);
    const FarGroup g = far_group(q);
    // (best[i] has not moved since k_far_count: same candidates)
    const float cutf = on ? far_cut(S, u2d(best[i]) + S->t_tie) : 0.f, cut2f = __fmul_ru(cutf, cutf);
    const float cutg = cut2f * 1.0001f + 1e-6f;
    // the warp's pairs fill its range in the order the walk meets them: the lanes that hit a face write neighbouring
    // entries (the narrow phase goes by pair_band, not by ranges per element)
    long long j = (long long)old;
    const unsigned lt = (1u << (threadIdx.x & 31)) - 1u;
    far_walk<false>(q, g, cutg, cell_start, pmask, s_stack[threadIdx.x >> 5], [&](int p0, int p1) {
        for (int p = p0; p < p1; ++p) {
            const bool hit = on && far_hit(q, cutf, cut2f, ffar, p);
            const unsigned hm = __ballot_sync(0xffffffffu, hit);
            if (hit) { const long long w = j + __popc(hm & lt); pair_face[w] = p; pair_key[w] = 0x7ff0000000000000ull; pair_band[w] = i; }
            j += __popc(hm);
        }
        return false;
    });
}

__global__ void k_far_fix(DcScalars *S)
{
    S->far_pairs_total += S->far_end;
    S->n_pairs = S->far_end;
}

// sdist = +-d_e for the elements of this pass: the magnitude from the narrow phase, the sign from the label the flood
// fill gave
__global__ void k_far_decide(DcScalars *S, const int *__restrict__ band_elem, long long *__restrict__ band_start, int *__restrict__ band_cnt,
                             const unsigned long long *__restrict__ dmin, const signed char *__restrict__ labels,
                             double *__restrict__ sdist)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    int done = 0, bad = 0;
    if (i < S->n_band && band_start[i] >= 0 && !(S->status & DC_STATUS_INVALID)) {
        const int e = band_elem[i];
        const double d = u2d(dmin[i]);
        if (d < 1e300) { sdist[e] = labels[e] == DC_HOLE ? -d : d; done = 1; }
        else bad = 1;                                // (no leaf was solved: cannot happen; counted, clamp kept)
        band_start[i] = -1; band_cnt[i] = -1;
    }
    const unsigned md = __ballot_sync(0xffffffffu, done), mb = __ballot_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0) {
        if (md) { atomicAdd(&S->far_pass_done, __popc(md)); atomicAdd(&S->far_done, __popc(md)); }
        if (mb) { atomicAdd(&S->far_pass_done, __popc(mb)); atomicAdd(&S->far_unresolved, __popc(mb)); }
    }
}
