// dc_kernels.cu -- libdc: direct-cut hole cutting on B200 (sm_100a).  Kernels S1..S7 + C ABI.
//
// Step names follow SURVEY.md 8(a) / DESIGN.md:
//   S1 face prep      k_face_boxes, k_setup_surface
//   S3 face bins      k_face_hist, k_scan_sums, k_scan_cells, k_cell_occ, k_face_scatter   (uniform bins, rows along x contiguous)
//   S2 element boxes  k_elem_boxes                                    (HBM-bound stream)
//   S4 candidates     k_filter (thread/element), k_pairs (16 lanes/active element, one append per element)
//   S5 narrow phase   dc_narrow.cuh: k_np_stage, k_np_solve, k_np_roots, k_np_bound, k_np_bound_tail, k_np_compact (FP64)
//   (DC_FLAG_PAPER_MODE: dc_paper.cuh, the paper's approximate A.1 / A.3 / A.4 in place of S5 and S6)
//   S6 decide         k_np_decide
//   S7 flood fill     k_uf_tiles, k_uf_seed, k_uf_resolve, k_uf_assign, k_seedless, k_uf_fix
//
// PAPER.md citations are given where an operation is defined; the kernel design itself is new
// (the paper's A.1-A.4 kernels were written for Kepler K80 and are prior art, not the blueprint).
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <new>
#include <algorithm>
#include <vector>
#include <mutex>

#include "../../include/dc.h"
#include "dc_geom.cuh"
#include "dc_newton.cuh"

using namespace dcg;

#define DC_MAX_GRAPHS 64                /* launch sequences dc_cut keeps as CUDA graphs (least recently used goes) */
#define DC_MAX_SEEDLESS 1024           /* seedless components resolved per cut (each by one exhaustive query) */
#define DC_GRID_MAX 64              /* face-bin cells per axis; cell (x,y,z) has code x + 64 (y + 64 z): a row along x is contiguous */
#define DC_OCC (DC_GRID_MAX / 4)    /* coarse occupancy grid: 4 x 4 x 4 cells per entry */
#define DC_NCELL (DC_GRID_MAX * DC_GRID_MAX * DC_GRID_MAX)
#define DC_NQN 28                   /* >= DC_MAX_ROUNDS + 2 */
#define DC_GRID_ROUNDS 4             /* branch-and-bound rounds launched as grids; the rest run inside one CTA */

// ------------------------------------------------------------------------------------------
// device-resident scalars and counters
struct DcScalars {
    // reductions over the surface (ordered-uint encodings), reset by dc_set_cut_surface
    unsigned long long node_min[3], node_max[3];   // AABB of the surface NODES -> L_ref
    unsigned long long fbox_min[3], fbox_max[3];   // AABB of the face Bezier boxes
    unsigned long long max_face_edge;              // max face-box edge
    unsigned long long grid_max_diag2;             // max element-box diagonal^2 (set by S2)
    // derived by k_setup_surface
    double l_ref_auto;
    double smin[3], smax[3];
    double origin[3], cell, inv_cell, fhalf;
    int dims[3];
    int n_face;
    // derived by k_setup_classify
    double l_ref, tau, tau_exit, t_tie, d_band, reach, theta, tol_d, amb;
    int max_level;
    int pad0;
    // work state
    int n_active;
    int n_band;                     // elements with >= 1 candidate pair (the narrow-phase band)
    int max_band;                   // capacity of the per-band-element arrays
    int n_seedless;
    int uf_tile;                    // next tile of k_uf_tiles (tiles are taken in launch order)
    int n_lroots;                   // tile-local roots listed by k_uf_tiles
    int epoch;                      // number of the cut (k_uf_tiles' flags); lives on the device so that a replayed CUDA graph counts too
    int surface_small;              // DC_STATUS_SURFACE_SMALL (kept apart from status: k_setup_classify resets that later)
    int status;
    int qn[DC_NQN];                 // items of round r (children queue, ping-pong buffers)
    int nn[DC_NQN];                 // leaves of round r (Newton queue)
    int nh[DC_NQN + 1];             // Newton queue heads: [0] seed pass, [r + 1] round r
    unsigned long long n_pairs;
    int seedless_elem[DC_MAX_SEEDLESS];
    // counters
    unsigned long long c_box_tests, c_bnb_nodes, c_newton, c_newton_iters, c_newton_fail,
        c_depth_exceeded, c_cut, c_hole, c_normal, c_ambiguous, c_sign_ambiguous,
        c_fill_conflicts, c_queue_peak, c_seedless_total;
    // DC_FLAG_EXACT_FAR (dc_far.cuh): the two lists of far elements still to do (ping-pong), the chunk's and the pass's tallies
    int far_n[2];
    int far_pass_done, far_done, far_unresolved, far_pad;
    int far_nheavy, far_nheavy_pass;   // heavy elements of the slice / of those, the ones served in this pass
    unsigned long long far_end;         // end of the pair slots handed out in this chunk
    unsigned long long far_want;        // most candidates a deferred element asked for
    unsigned long long far_pairs_total;
    unsigned long long far_lo[3], far_hi[3];    // box of the far elements' centres (ordered-uint encodings)
};

// first statement of every kernel of a cut (see launch_pdl): let the next kernel start launching, then wait for the previous
// one (a no-op for a kernel launched the plain way)
__device__ __forceinline__ void pdl_start()
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

__device__ __forceinline__ void atomic_min_d(unsigned long long *addr, double v) { atomicMin(addr, enc_ord(v)); }
__device__ __forceinline__ void atomic_max_d(unsigned long long *addr, double v) { atomicMax(addr, enc_ord(v)); }

__device__ __forceinline__ int cell_code(int x, int y, int z) { return x + DC_GRID_MAX * (y + DC_GRID_MAX * z); }

// Bezier control values of a 1-D quadratic through nodes (-1,0,1): b0 = x0, b1 = 2 x1 - (x0+x2)/2,
// b2 = x2 (convex-hull property => conservative boxes; Lagrange NODES do not bound the patch).
__device__ __forceinline__ double bez_mid(double x0, double x1, double x2) { return 2.0 * x1 - 0.5 * (x0 + x2); }

// ------------------------------------------------------------------------------------------
// S1: per-face Bezier box + surface reductions.  face_nodes [n_face][9][3].
__global__ void k_face_boxes(DcScalars *S, const double *__restrict__ face_nodes, int n_face,
                             double *__restrict__ fbox_orig /*[n_face][6]*/)
{
    pdl_start();
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    double lo[3] = { INFINITY, INFINITY, INFINITY }, hi[3] = { -INFINITY, -INFINITY, -INFINITY };
    double nlo[3] = { INFINITY, INFINITY, INFINITY }, nhi[3] = { -INFINITY, -INFINITY, -INFINITY };
    double edge = 0.0;
    if (f < n_face) {
        const double *X = face_nodes + (size_t)f * 27;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double x[9], b[9];
#pragma unroll
            for (int m = 0; m < 9; ++m) { x[m] = __ldg(X + 3 * m + c); nlo[c] = dmin2(nlo[c], x[m]); nhi[c] = dmax2(nhi[c], x[m]); }
#pragma unroll
            for (int j = 0; j < 3; ++j) { b[3*j] = x[3*j]; b[3*j+1] = bez_mid(x[3*j], x[3*j+1], x[3*j+2]); b[3*j+2] = x[3*j+2]; }
#pragma unroll
            for (int i = 0; i < 3; ++i) { const double m1 = bez_mid(b[i], b[i+3], b[i+6]); b[i+3] = m1; }
#pragma unroll
            for (int m = 0; m < 9; ++m) { lo[c] = dmin2(lo[c], b[m]); hi[c] = dmax2(hi[c], b[m]); }
            fbox_orig[(size_t)f * 6 + c] = lo[c];
            fbox_orig[(size_t)f * 6 + 3 + c] = hi[c];
            edge = dmax2(edge, hi[c] - lo[c]);
        }
    }
    // warp reduce then one atomic per warp
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            lo[c] = dmin2(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], o));
            hi[c] = dmax2(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], o));
            nlo[c] = dmin2(nlo[c], __shfl_xor_sync(0xffffffffu, nlo[c], o));
            nhi[c] = dmax2(nhi[c], __shfl_xor_sync(0xffffffffu, nhi[c], o));
        }
        edge = dmax2(edge, __shfl_xor_sync(0xffffffffu, edge, o));
    }
    if ((threadIdx.x & 31) == 0 && lo[0] != INFINITY) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            atomic_min_d(&S->fbox_min[c], lo[c]); atomic_max_d(&S->fbox_max[c], hi[c]);
            atomic_min_d(&S->node_min[c], nlo[c]); atomic_max_d(&S->node_max[c], nhi[c]);
        }
        atomic_max_d(&S->max_face_edge, edge);
    }
}

__global__ void k_reset_surface(DcScalars *S)
{
    pdl_start();
    for (int c = 0; c < 3; ++c) {
        S->node_min[c] = S->fbox_min[c] = ~0ull;
        S->node_max[c] = S->fbox_max[c] = 0ull;
    }
    S->max_face_edge = 0ull;
}

__global__ void k_setup_surface(DcScalars *S, int n_face)
{
    pdl_start();
    double ext = 0.0, lref = 0.0;
    for (int c = 0; c < 3; ++c) {
        S->smin[c] = dec_ord(S->fbox_min[c]); S->smax[c] = dec_ord(S->fbox_max[c]);
        ext = dmax2(ext, S->smax[c] - S->smin[c]);
        lref = dmax2(lref, dec_ord(S->node_max[c]) - dec_ord(S->node_min[c]));
    }
    S->l_ref_auto = lref;
    const double edge = dec_ord(S->max_face_edge);
    double cell = dmax2(edge, ext / DC_GRID_MAX) * (1.0 + 1e-9);
    if (!(cell > 0.0)) cell = 1.0;
    S->cell = cell; S->inv_cell = 1.0 / cell; S->fhalf = 0.5 * edge;
    for (int c = 0; c < 3; ++c) {
        S->origin[c] = S->smin[c];
        int d = (int)floor((S->smax[c] - S->smin[c]) * S->inv_cell) + 1;
        S->dims[c] = d < 1 ? 1 : (d > DC_GRID_MAX ? DC_GRID_MAX : d);
    }
    S->n_face = n_face;
}

__device__ __forceinline__ int cell_coord(const DcScalars *S, double x, int c)
{
    int i = (int)floor((x - S->origin[c]) * S->inv_cell);
    return i < 0 ? 0 : (i >= S->dims[c] ? S->dims[c] - 1 : i);
}

// S3: histogram of faces over cells keyed by the code of the box-centre cell
__global__ void k_face_hist(const DcScalars *S, const double *__restrict__ fbox_orig, int n_face,
                            int *__restrict__ fcell, int *cell_count)
{
    pdl_start();
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_face) return;
    int ic[3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
        ic[c] = cell_coord(S, 0.5 * (fbox_orig[(size_t)f * 6 + c] + fbox_orig[(size_t)f * 6 + 3 + c]), c);
    const int code = cell_code(ic[0], ic[1], ic[2]);
    fcell[f] = code;
    atomicAdd(&cell_count[code], 1);
}

// exclusive scan over the DC_NCELL cells in two coalesced passes: per-chunk sums (one CTA of
// 256 threads per 1024 cells, int4 loads), then every CTA adds the sums of the chunks before it to a local scan.
#define SCAN_CHUNK 1024
#define SCAN_NCHUNK (DC_NCELL / SCAN_CHUNK)
__device__ __forceinline__ int block_sum_256(int v, int *s_warp)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) s_warp[threadIdx.x >> 5] = v;
    __syncthreads();
    int t = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) t += s_warp[w];
    __syncthreads();
    return t;
}
__global__ void __launch_bounds__(256) k_scan_sums(const int *__restrict__ cell_count, int *__restrict__ chunk_sum)
{
    pdl_start();
    __shared__ int s_warp[8];
    const int4 v = reinterpret_cast<const int4 *>(cell_count)[blockIdx.x * 256 + threadIdx.x];
    const int t = block_sum_256(v.x + v.y + v.z + v.w, s_warp);
    if (threadIdx.x == 0) chunk_sum[blockIdx.x] = t;
}
__global__ void __launch_bounds__(256) k_scan_cells(const int *__restrict__ cell_count, const int *__restrict__ chunk_sum,
                                                    int *__restrict__ cell_start)
{
    pdl_start();
    __shared__ int s_warp[8];
    __shared__ int s_incl[8];
    // sum of the chunks before this one (SCAN_NCHUNK = 256 values: one per thread)
    const int before = block_sum_256((int)threadIdx.x < (int)blockIdx.x ? chunk_sum[threadIdx.x] : 0, s_warp);
    const int4 v = reinterpret_cast<const int4 *>(cell_count)[blockIdx.x * 256 + threadIdx.x];
    const int mine = v.x + v.y + v.z + v.w;
    int incl = mine;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += u; }
    if (lane == 31) s_incl[wid] = incl;
    __syncthreads();
    int woff = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) if (w < wid) woff += s_incl[w];
    int4 o;
    o.x = before + woff + incl - mine; o.y = o.x + v.x; o.z = o.y + v.y; o.w = o.z + v.z;
    reinterpret_cast<int4 *>(cell_start)[blockIdx.x * 256 + threadIdx.x] = o;
    if (blockIdx.x == SCAN_NCHUNK - 1 && threadIdx.x == 255) cell_start[DC_NCELL] = o.w + v.w;
}

// coarse occupancy: does any face sit in the 4 x 4 x 4 cells of a coarse entry (k_filter's first look: most elements
// near the surface's box are in empty space)
__global__ void k_cell_occ(const int *__restrict__ cell_start, unsigned char *__restrict__ occ)
{
    pdl_start();
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= DC_OCC * DC_OCC * DC_OCC) return;
    const int X = t % DC_OCC, Y = (t / DC_OCC) % DC_OCC, Z = t / (DC_OCC * DC_OCC);
    int n = 0;
    for (int z = 4 * Z; z < 4 * Z + 4; ++z)
        for (int y = 4 * Y; y < 4 * Y + 4; ++y) {
            const int c0 = cell_code(4 * X, y, z);
            n += cell_start[c0 + 4] - cell_start[c0];
        }
    occ[t] = n > 0;
}

// scatter faces into cell order; write sorted boxes and monomial coefficients (stride 28 doubles)
__global__ void k_face_scatter(const double *__restrict__ face_nodes, const double *__restrict__ fbox_orig,
                               const int *__restrict__ fcell, const int *__restrict__ cell_start,
                               int *cell_fill, int n_face, int *__restrict__ fperm,
                               double *__restrict__ fbox, double *__restrict__ fcoef, float *__restrict__ fboxf)
{
    pdl_start();
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_face) return;
    const int code = fcell[f];
    const int pos = cell_start[code] + atomicAdd(&cell_fill[code], 1);
    fperm[pos] = f;
#pragma unroll
    for (int m = 0; m < 6; ++m) fbox[(size_t)pos * 6 + m] = fbox_orig[(size_t)f * 6 + m];
    // the same box in single precision, rounded OUTWARD (k_np_roots' filter: 32 bytes per face instead of 48)
    {
        float4 lo4, hi4;
        lo4.x = __double2float_rd(fbox_orig[(size_t)f * 6]); lo4.y = __double2float_rd(fbox_orig[(size_t)f * 6 + 1]); lo4.z = __double2float_rd(fbox_orig[(size_t)f * 6 + 2]); lo4.w = 0.f;
        hi4.x = __double2float_ru(fbox_orig[(size_t)f * 6 + 3]); hi4.y = __double2float_ru(fbox_orig[(size_t)f * 6 + 4]); hi4.z = __double2float_ru(fbox_orig[(size_t)f * 6 + 5]); hi4.w = 0.f;
        reinterpret_cast<float4 *>(fboxf)[(size_t)pos * 2] = lo4; reinterpret_cast<float4 *>(fboxf)[(size_t)pos * 2 + 1] = hi4;
    }
    const double *X = face_nodes + (size_t)f * 27;
    double A[27];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double x[9];
#pragma unroll
        for (int m = 0; m < 9; ++m) x[m] = __ldg(X + 3 * m + c);
        nodes_to_mono9(x, A + 9 * c);
#pragma unroll
        for (int m = 0; m < 9; ++m) fcoef[(size_t)pos * 28 + c * 9 + m] = A[9 * c + m];
    }
    fcoef[(size_t)pos * 28 + 27] = higher_order_const(A);   // slot 27: see dc_geom.cuh bound_node
}

// ------------------------------------------------------------------------------------------
// S2: conservative element boxes from the 26 boundary control points of the Bezier net.
// conn rows are staged through shared memory so the global reads are fully coalesced.
// ebox is SoA: ebox[c*n_elem + e] (c = 0..5: min xyz, max xyz).
#ifndef EB_THREADS
#define EB_THREADS 128
#endif
#ifndef EB_UNROLL
#define EB_UNROLL 3
#endif
constexpr int kEbUnroll = EB_UNROLL;
__global__ void __launch_bounds__(EB_THREADS) k_elem_boxes(DcScalars *S, const double *__restrict__ xyz,
                                                           const int *__restrict__ conn, long long n_elem,
                                                           double *__restrict__ ebox)
{
    pdl_start();
    // One (element, coordinate) pair per work item, 3 items per thread: consecutive lanes read CONSECUTIVE
    // doubles of a node (x, y, z of one element, then the next element), so one warp load touches a third
    // of the sectors a lane-per-element gather would, and the Lagrange -> Bezier conversion is per coordinate
    // anyway.  conn rows are staged through shared memory (coalesced).
    __shared__ int s_conn[EB_THREADS * 27];
    __shared__ double s_ext2[EB_THREADS * 3];
    const long long e0 = (long long)blockIdx.x * EB_THREADS;
    const int nloc = (int)min((long long)EB_THREADS, n_elem - e0);
    for (int i = threadIdx.x; i < nloc * 27; i += EB_THREADS) s_conn[i] = __ldg(conn + e0 * 27 + i);
    __syncthreads();
    const int wbase = (threadIdx.x >> 5) * 32, lane = threadIdx.x & 31;
#pragma unroll kEbUnroll
    for (int j = 0; j < 3; ++j) {
        const int idx = j * 32 + lane;               // 0..95 within the warp's 32 elements
        const int el = wbase + idx / 3, c = idx % 3;
        if (el < nloc) {
            const int *cn = s_conn + el * 27;
            double b[27];
#pragma unroll
            for (int m = 0; m < 27; ++m) b[m] = __ldg(xyz + (size_t)cn[m] * 3 + c);
            // Lagrange -> Bezier along i, then j, then k (only the middle layer of each line changes)
#pragma unroll
            for (int m = 0; m < 9; ++m) b[3*m+1] = bez_mid(b[3*m], b[3*m+1], b[3*m+2]);
#pragma unroll
            for (int k = 0; k < 3; ++k)
#pragma unroll
                for (int i = 0; i < 3; ++i) b[i+3+9*k] = bez_mid(b[i+9*k], b[i+3+9*k], b[i+6+9*k]);
#pragma unroll
            for (int m = 0; m < 9; ++m) b[m+9] = bez_mid(b[m], b[m+9], b[m+18]);
            // (plain compare-and-select: fmin / fmax of doubles expand to a NaN-aware sequence twice as long)
            double lo = b[0], hi = b[0];
#pragma unroll
            for (int m = 1; m < 27; ++m) if (m != 13) { lo = b[m] < lo ? b[m] : lo; hi = b[m] > hi ? b[m] : hi; }
            const long long e = e0 + el;
            ebox[(size_t)c * n_elem + e] = lo;
            ebox[(size_t)(3 + c) * n_elem + e] = hi;
            s_ext2[el * 3 + c] = (hi - lo) * (hi - lo);
        }
    }
    __syncthreads();
    double diag2 = 0.0;
    if (threadIdx.x < nloc) diag2 = s_ext2[threadIdx.x * 3] + s_ext2[threadIdx.x * 3 + 1] + s_ext2[threadIdx.x * 3 + 2];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) diag2 = dmax2(diag2, __shfl_xor_sync(0xffffffffu, diag2, o));
    if ((threadIdx.x & 31) == 0) atomicMax(&S->grid_max_diag2, (unsigned long long)__double_as_longlong(diag2));
}

// ------------------------------------------------------------------------------------------
// adjacency from shared face-centre nodes (only when the caller passes adj6 = NULL)
__constant__ int c_face_centre[6] = { 12, 14, 10, 16, 4, 22 };
__global__ void k_adj_pass1(const int *__restrict__ conn, long long n_elem, int *first, int *second)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_elem * 6) return;
    const long long e = t / 6; const int k = (int)(t % 6);
    const int c = conn[e * 27 + c_face_centre[k]];
    const int code = (int)t;
    const int old = atomicCAS(&first[c], -1, code);
    if (old != -1) second[c] = code;
}
__global__ void k_adj_pass2(const int *__restrict__ conn, long long n_elem, const int *__restrict__ first,
                            const int *__restrict__ second, int *__restrict__ adj)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_elem * 6) return;
    const long long e = t / 6; const int k = (int)(t % 6);
    const int c = conn[e * 27 + c_face_centre[k]];
    const int a = first[c], b = second[c];
    const int other = (a == (int)t) ? b : a;
    adj[t] = other < 0 ? -1 : other / 6;
}

// ------------------------------------------------------------------------------------------
// per-classify scalar setup
__global__ void k_setup_classify(DcScalars *S, dc_params P, int max_band)
{
    pdl_start();
    S->max_band = max_band;
    S->epoch = S->epoch == 0x7fffffff ? 1 : S->epoch + 1;
    const double lref = P.l_ref > 0.0 ? P.l_ref : S->l_ref_auto;
    S->l_ref = lref;
    S->tau = (P.tau_cut_rel > 0.0 ? P.tau_cut_rel : 1e-7) * lref;
    S->amb = 1e-9 * lref;
    S->tau_exit = S->tau - S->amb;
    S->t_tie = 1e-9 * lref;
    S->tol_d = 1e-13 * lref;
    S->d_band = P.d_band > 0.0 ? P.d_band : sqrt(__longlong_as_double((long long)S->grid_max_diag2));
    S->reach = S->d_band + 2.0 * S->tau + S->t_tie;
    {
        // precondition of reading A7 (SURVEY 8(a) note ii), checked where it is cheap: the WHOLE surface against the
        // largest element (a cube of diagonal D has edge D / sqrt 3)
        double ext = 0.0;
        for (int c = 0; c < 3; ++c) ext = dmax2(ext, S->smax[c] - S->smin[c]);
        const double dg = sqrt(__longlong_as_double((long long)S->grid_max_diag2));
        S->surface_small = ext < dg * 0.5773502691896258 ? 1 : 0;
    }
    S->theta = P.theta_leaf > 0.0 ? P.theta_leaf : 0.25;
    S->max_level = (P.max_level > 0 && P.max_level <= 12) ? P.max_level : 12;
    S->n_active = 0; S->n_band = 0; S->n_seedless = 0; S->uf_tile = 0; S->n_lroots = 0; S->n_pairs = 0ull;
    S->status = S->surface_small ? DC_STATUS_SURFACE_SMALL : 0;
    for (int i = 0; i < DC_NQN; ++i) { S->qn[i] = 0; S->nn[i] = 0; S->nh[i] = 0; }
    S->nh[DC_NQN] = 0;
    S->c_box_tests = S->c_bnb_nodes = S->c_newton = S->c_newton_iters = S->c_newton_fail = 0ull;
    S->c_depth_exceeded = S->c_cut = S->c_hole = S->c_normal = S->c_ambiguous = 0ull;
    S->c_sign_ambiguous = S->c_fill_conflicts = S->c_queue_peak = S->c_seedless_total = 0ull;
    S->far_n[0] = S->far_n[1] = 0; S->far_pass_done = S->far_done = S->far_unresolved = 0;
    S->far_end = S->far_want = S->far_pairs_total = 0ull;
    for (int c = 0; c < 3; ++c) { S->far_lo[c] = ~0ull; S->far_hi[c] = 0ull; }
}

// ------------------------------------------------------------------------------------------
// S4a: one thread per element.  Initialises the per-element state of this cut and appends the elements whose inflated
// box meets a face cell that is not empty to the active list (warp-aggregated atomic append).  Coarse to fine: most
// elements near the surface's box sit in empty space, and the (at most 27, usually 8) coarse occupancy bytes say so;
// only the others look at the cell rows k_pairs will walk (a row of cells along x is ONE contiguous face range).
__device__ __forceinline__ bool filter_test(const DcScalars *S, const int *__restrict__ cell_start,
                                            const unsigned char *__restrict__ occ, const double *lo, const double *hi)
{
    double d2 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double g = dmax2(0.0, dmax2(S->smin[c] - hi[c], lo[c] - S->smax[c]));
        d2 = fma(g, g, d2);
    }
    const double reach = S->reach;
    if (!(d2 <= reach * reach)) return false;
    const double pad = reach + S->fhalf;
    int i0[3], i1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) { i0[c] = cell_coord(S, lo[c] - pad, c); i1[c] = cell_coord(S, hi[c] + pad, c); }
    bool maybe = false;
    for (int z = i0[2] >> 2; z <= (i1[2] >> 2) && !maybe; ++z)
        for (int y = i0[1] >> 2; y <= (i1[1] >> 2) && !maybe; ++y)
            for (int x = i0[0] >> 2; x <= (i1[0] >> 2); ++x)
                if (__ldg(occ + x + DC_OCC * (y + DC_OCC * z))) { maybe = true; break; }
    if (!maybe) return false;
    for (int z = i0[2]; z <= i1[2]; ++z)
        for (int y = i0[1]; y <= i1[1]; ++y) {
            const int c0 = cell_code(0, y, z);
            if (__ldg(cell_start + c0 + i1[0] + 1) - __ldg(cell_start + c0 + i0[0]) > 0) return true;
        }
    return false;
}

__global__ void k_filter(DcScalars *S, const double *__restrict__ ebox, long long n_elem,
                         signed char *__restrict__ labels, int *__restrict__ parent,
                         unsigned char *__restrict__ comp, const int *__restrict__ cell_start,
                         const unsigned char *__restrict__ occ, int *__restrict__ act_elem)
{
    pdl_start();
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    bool active = false;
    if (e < n_elem) {
        labels[e] = -1; comp[e] = 0;       // (parent[] is initialised by k_uf_tiles)
        double lo[3], hi[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) { lo[c] = ebox[(size_t)c * n_elem + e]; hi[c] = ebox[(size_t)(3 + c) * n_elem + e]; }
        active = filter_test(S, cell_start, occ, lo, hi);
    }
    const unsigned m = __ballot_sync(0xffffffffu, active);
    if (m) {
        const int lane = threadIdx.x & 31;
        int base = 0;
        if (lane == (__ffs(m) - 1)) base = atomicAdd(&S->n_active, __popc(m));
        base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
        if (active) act_elem[base + __popc(m & ((1u << lane) - 1))] = (int)e;
    }
}

// S4b: a group of 16 lanes per active element.  The cells its inflated box overlaps are (ny x nz) ROWS along x, one
// contiguous face range each: one lane per row fetches its range, the ranges are concatenated by a scan over the
// group, and the lanes then walk the concatenation 16 faces at a time (coalesced face-box loads, every lane busy)
// applying the box test of Algorithm A.2.  Survivors are staged in shared memory and written as
// ONE contiguous segment of the pair list (one atomic per element); an element with more survivors than the stage
// holds re-walks its ranges and writes directly.  pair_key is initialised to +inf for S5.
__device__ __forceinline__ double box_dist2(const double *lo, const double *hi, const double *fb)
{
    double d2 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double g = dmax2(0.0, dmax2(fb[c] - hi[c], lo[c] - fb[3 + c]));
        d2 = fma(g, g, d2);
    }
    return d2;
}

#define PR_WARPS 8
#define PR_CAP 224
#define PR_W 16                     /* lanes per element: two elements in flight per warp (the walk is latency bound) */
#define PR_GROUPS (PR_WARPS * 32 / PR_W)
__global__ void __launch_bounds__(PR_WARPS * 32) k_pairs(DcScalars *S, const double *__restrict__ ebox, long long n_elem,
                                               const int *__restrict__ act_elem, const int *__restrict__ cell_start,
                                               const double *__restrict__ fbox, long long max_pairs,
                                               int *__restrict__ band_elem, long long *__restrict__ band_start,
                                               int *__restrict__ band_cnt,
                                               int *__restrict__ pair_face, unsigned long long *__restrict__ pair_key,
                                               int *__restrict__ pair_band, NItem *__restrict__ seed_q,
                                               unsigned long long *__restrict__ best, unsigned long long *__restrict__ dmin)
{
    pdl_start();
    __shared__ int s_list[PR_GROUPS][PR_CAP];
    __shared__ int s_off[PR_GROUPS][PR_W + 1];
    __shared__ int s_first[PR_GROUPS][PR_W];
    // a GROUP of PR_W lanes per element; every warp primitive below is confined to the group's lanes
    const int lane = threadIdx.x & (PR_W - 1), wl = threadIdx.x / PR_W;
    const int gshift = (threadIdx.x & 31) & ~(PR_W - 1);
    const unsigned gmask = (PR_W == 32 ? 0xffffffffu : ((1u << PR_W) - 1u)) << gshift;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) / PR_W;
    const int nwarps = (gridDim.x * blockDim.x) / PR_W;
    const int n_active = S->n_active;
    const double reach = S->reach, reach2 = reach * reach, pad = reach + S->fhalf;
    int *list = s_list[wl], *off = s_off[wl], *firsts = s_first[wl];
    unsigned long long tests = 0;
    for (int a = warp; a < n_active; a += nwarps) {
        const long long e = act_elem[a];
        double lo[3], hi[3];
        int i0[3], i1[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            lo[c] = ebox[(size_t)c * n_elem + e]; hi[c] = ebox[(size_t)(3 + c) * n_elem + e];
            i0[c] = cell_coord(S, lo[c] - pad, c); i1[c] = cell_coord(S, hi[c] + pad, c);
        }
        const int ny = i1[1] - i0[1] + 1, nblk = ny * (i1[2] - i0[2] + 1);      // rows of cells along x
        long long base = 0;
        int total = 0, bslot = 0;
        unsigned long long skey = ~0ull;
        for (int phase = 0; phase < 2; ++phase) {
            int running = 0;
            for (int bbase = 0; bbase < nblk; bbase += PR_W) {
                const int bi = bbase + lane;
                int cnt = 0, first = 0;
                if (bi < nblk) {
                    const int c0 = cell_code(0, i0[1] + bi % ny, i0[2] + bi / ny);
                    first = __ldg(cell_start + c0 + i0[0]);
                    cnt = __ldg(cell_start + c0 + i1[0] + 1) - first;
                }
                int incl = cnt;
#pragma unroll
                for (int o = 1; o < PR_W; o <<= 1) { const int v = __shfl_up_sync(gmask, incl, o, PR_W); if (lane >= o) incl += v; }
                const int T = __shfl_sync(gmask, incl, PR_W - 1, PR_W);
                if (lane == 0) off[0] = 0;
                off[lane + 1] = incl; firsts[lane] = first;
                __syncwarp(gmask);
                for (int j0 = 0; j0 < T; j0 += PR_W) {
                    const int j = j0 + lane;
                    bool hit = false;
                    int p = -1;
                    double d2 = 0.0;
                    if (j < T) {
                        int L = 0;                       // largest L with off[L] <= j
#pragma unroll
                        for (int st = PR_W / 2; st > 0; st >>= 1) if (off[L + st] <= j) L += st;
                        p = firsts[L] + (j - off[L]);
                        double fb[6];
#pragma unroll
                        for (int m = 0; m < 6; m += 2) {
                            const double2 v = __ldg(reinterpret_cast<const double2 *>(fbox + (size_t)p * 6 + m));
                            fb[m] = v.x; fb[m + 1] = v.y;
                        }
                        d2 = box_dist2(lo, hi, fb);
                        hit = d2 <= reach2;
                        if (phase == 0) ++tests;
                    }
                    const unsigned m = (__ballot_sync(gmask, hit) >> gshift) & (PR_W == 32 ? 0xffffffffu : ((1u << PR_W) - 1u));
                    const int pos = running + __popc(m & lt_mask);
                    if (hit) {
                        if (phase == 0) {
                            if (pos < PR_CAP) list[pos] = p;
                            // (the seed of the narrow phase: the pair with the nearest face box)
                            const unsigned long long kk = ((unsigned long long)__double_as_longlong(d2) & ~0xfffffull) | (unsigned long long)min(pos, 0xfffff);
                            skey = kk < skey ? kk : skey;
                        }
                        else { pair_face[base + pos] = p; pair_key[base + pos] = 0x7ff0000000000000ull; pair_band[base + pos] = (int)bslot; }
                    }
                    running += __popc(m);
                }
                __syncwarp(gmask);
            }
            if (phase == 1) break;
            total = running;
#pragma unroll
            for (int o = PR_W / 2; o > 0; o >>= 1) { const unsigned long long v = __shfl_xor_sync(gmask, skey, o, PR_W); skey = v < skey ? v : skey; }
            if (lane == 0) {
                long long b = (long long)atomicAdd(&S->n_pairs, (unsigned long long)total);
                if (b + total > max_pairs) { atomicOr(&S->status, DC_STATUS_PAIR_OVERFLOW); b = -1; }
                if (b >= 0 && total > 0) {
                    const int slot = atomicAdd(&S->n_band, 1);
                    if (slot < S->max_band) {
                        band_elem[slot] = (int)e; band_start[slot] = b; band_cnt[slot] = total;
                        best[slot] = (unsigned long long)__double_as_longlong(reach);
                        dmin[slot] = 0x7ff0000000000000ull;
                        NItem it; it.p = (unsigned)(b + (long long)(skey & 0xfffffull)); it.ak = (unsigned)slot | (7u << 29); it.w2 = 0; it.w3 = 1u << 24;
                        seed_q[slot] = it;
                        bslot = slot;
                    } else { atomicOr(&S->status, DC_STATUS_BAND_OVERFLOW); b = -1; }
                }
                base = b;
            }
            base = __shfl_sync(gmask, base, 0, PR_W);
            bslot = __shfl_sync(gmask, bslot, 0, PR_W);
            if (base < 0 || total == 0) break;
            if (total <= PR_CAP) {
                for (int i = lane; i < total; i += PR_W) { pair_face[base + i] = list[i]; pair_key[base + i] = 0x7ff0000000000000ull; pair_band[base + i] = bslot; }
                break;
            }
        }
        __syncwarp(gmask);
    }
    __syncwarp();
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tests += __shfl_xor_sync(0xffffffffu, tests, o);
    if ((threadIdx.x & 31) == 0 && tests) atomicAdd(&S->c_box_tests, tests);
}

// ------------------------------------------------------------------------------------------
// S5 + S6: narrow phase -> dc_narrow.cuh.
__constant__ int c_face_node[6][9] = {
    { 0, 3, 6, 9, 12, 15, 18, 21, 24 },      // xi = -1 : (a,b) = (j,k)
    { 2, 5, 8, 11, 14, 17, 20, 23, 26 },     // xi = +1
    { 0, 1, 2, 9, 10, 11, 18, 19, 20 },      // eta = -1 : (a,b) = (i,k)
    { 6, 7, 8, 15, 16, 17, 24, 25, 26 },     // eta = +1
    { 0, 1, 2, 3, 4, 5, 6, 7, 8 },           // zeta = -1 : (a,b) = (i,j)
    { 18, 19, 20, 21, 22, 23, 24, 25, 26 },  // zeta = +1
};

#include "dc_narrow.cuh"
#include "dc_paper.cuh"
#include "dc_far.cuh"

// ------------------------------------------------------------------------------------------
// S7: flood fill = connected components of the face-adjacency graph of non-CUT elements
// (lock-free union-find), seeded by the signs found in S5/S6 (the classical paint-fill,
// PAPER.md L143 / Fig. 5c, without its O(diameter) sweeps).
__device__ __forceinline__ int uf_find(int *parent, int x)
{
    volatile int *P = parent;
    while (true) {
        const int p = P[x];
        if (p == x) return x;
        const int gp = P[p];
        if (gp != p) P[x] = gp;   // path halving (benign race: always points to an ancestor)
        x = p;
    }
}
__device__ __forceinline__ void uf_union(int *parent, int a, int b)
{
    while (true) {
        a = uf_find(parent, a); b = uf_find(parent, b);
        if (a == b) return;
        if (a < b) { const int t = a; a = b; b = t; }
        if (atomicCAS(&parent[a], a, b) == a) return;   // hook the larger root under the smaller
    }
}

__device__ __forceinline__ int ld_acquire(const int *p) { int v; asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v; }
__device__ __forceinline__ void st_release(int *p, int v) { asm volatile("st.release.gpu.global.s32 [%0], %1;" :: "l"(p), "r"(v) : "memory"); }

// One kernel for the whole forest.  Components INSIDE a tile of UF_TILE consecutive elements are found in shared memory
// (neighbours mostly have nearby ids, so most edges are settled there); every element then points at its tile-local root.
// Only the edges that leave the tile (towards LOWER tiles: each edge is handled by its upper end) go through the global
// forest.  They need the lower tile's local roots: tiles are handed out in launch order by a counter, a tile publishes a
// flag (the cut's epoch) once its local roots are written, and an upper tile waits for the flags of the lower tiles it
// touches -- those started earlier and never wait for an upper tile, so the wait cannot deadlock (the chained-scan
// argument).  Per tile, a (local root, other root) pair already united is remembered in shared memory, so a slab of
// 1024 elements facing one component of the slab below costs one union, not a thousand.
#define UF_TILE 1024
__global__ void __launch_bounds__(UF_TILE) k_uf_tiles(DcScalars *S, const signed char *__restrict__ labels, const int *__restrict__ adj,
                                                      long long n_elem, int *parent, int *tile_flag,
                                                      int *__restrict__ lroot_list)
{
    pdl_start();
    __shared__ int sp[UF_TILE];
    __shared__ int s_last[UF_TILE];
    __shared__ signed char s_lab[UF_TILE];
    __shared__ int s_tile;
    const int tid = threadIdx.x, lane = tid & 31;
    const int epoch = S->epoch;
    if (tid == 0) s_tile = atomicAdd(&S->uf_tile, 1);
    s_last[tid] = -1;
    __syncthreads();
    const int tile = s_tile;
    const long long base = (long long)tile * UF_TILE, e = base + tid;
    const int lab = e < n_elem ? labels[e] : DC_CUT;
    s_lab[tid] = (signed char)lab;
    const bool live = lab != DC_CUT;
    int nbs[6] = { -1, -1, -1, -1, -1, -1 };
    if (live) {
        const int2 *ap = reinterpret_cast<const int2 *>(adj + e * 6);
#pragma unroll
        for (int k = 0; k < 3; ++k) { const int2 v = __ldg(ap + k); nbs[2 * k] = v.x; nbs[2 * k + 1] = v.y; }
    }
    // Runs of consecutive ids that are neighbours (rows of a structured numbering) are merged inside the warp with one
    // ballot: every lane starts hooked under the first lane of its run, and the run's edges to other runs are issued once
    // per pair of runs, not once per element (a thousand threads hooking a row one element at a time was the cost here).
    bool to_prev = false;
#pragma unroll
    for (int k = 0; k < 6; ++k) to_prev = to_prev || nbs[k] == (int)e - 1;
    const unsigned mlive = __ballot_sync(0xffffffffu, live);
    to_prev = to_prev && live && lane > 0 && ((mlive >> (lane - 1)) & 1u);
    const unsigned mconn = __ballot_sync(0xffffffffu, to_prev);
    const int head = (tid & ~31) + (31 - __clz((~mconn) & (0xffffffffu >> (31 - lane))));
    sp[tid] = head;
    __syncthreads();
    if (live) {
        int hn[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const int nb = nbs[k];
            const bool in_tile = nb >= base && nb < e && !(to_prev && nb == (int)e - 1) && s_lab[nb - (int)base] != DC_CUT;
            hn[k] = in_tile ? sp[nb - (int)base] : -1;           // (its run's head, or already something above it)
        }
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const int ph = __shfl_up_sync(__activemask(), hn[k], 1);
            if (hn[k] >= 0 && !(to_prev && ph == hn[k])) uf_union(sp, head, hn[k]);
        }
    }
    __syncthreads();
    const int lr = uf_find(sp, tid);
    if (e < n_elem) parent[e] = (int)base + lr;
    if (live && lr == tid) lroot_list[atomicAdd(&S->n_lroots, 1)] = (int)e;
    __syncthreads();
    if (tid == 0) st_release(tile_flag + tile, epoch);       // (release after the barrier: the tile's stores come before it)
    // edges to lower tiles: all the gathers first (independent loads in flight together), the unions after
    const int mine = (int)base + lr;
    int other[6];
    bool edge[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const int nb = nbs[k];
        const bool cross = live && nb >= 0 && nb < base;
        edge[k] = cross && labels[nb] != DC_CUT;
        other[k] = -1 - lane;
        if (edge[k]) {
            const int *fl = tile_flag + nb / UF_TILE;
            while (ld_acquire(fl) != epoch) { }
            other[k] = ((volatile int *)parent)[nb];
        }
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        // a lane whose (root, root) pair equals that of the lane before it leaves the union to that lane; the others ask the
        // tile's memory of the last root united with their local root
        const int pm = __shfl_up_sync(0xffffffffu, mine, 1), po = __shfl_up_sync(0xffffffffu, other[k], 1);
        if (edge[k] && !(lane > 0 && pm == mine && po == other[k])) {
            if (atomicExch(&s_last[lr], other[k]) != other[k]) uf_union(parent, mine, other[k]);
        }
    }
}

// seeds: only the band elements carry a sign from S6 (one thread per band element, not per element)
__global__ void k_uf_seed(const DcScalars *S, const int *__restrict__ band_elem, const signed char *__restrict__ labels,
                          int *parent, unsigned char *comp)
{
    pdl_start();
    const int n_band = min(S->n_band, S->max_band);
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < n_band; b += gridDim.x * blockDim.x) {
        const int e = band_elem[b];
        const int lab = labels[e];
        if (lab == DC_HOLE || lab == DC_NORMAL) {
            const int r = uf_find(parent, e);
            // byte-wide OR through a 32-bit atomic; tested first (two giant components take almost every seed: the
            // atomics on their two words were the whole duration of this kernel)
            const unsigned bit = lab == DC_HOLE ? 1u : 2u;
            if ((((volatile unsigned char *)comp)[r] & bit) == 0) {
                unsigned *w = reinterpret_cast<unsigned *>(comp + (r & ~3));
                atomicOr(w, bit << (8 * (r & 3)));
            }
        }
    }
}

// A component no band element touches (surface misses the grid, or a pocket cut off by the grid
// boundary): one exhaustive nearest-face query for its representative element (SURVEY 8(a) note iii).
// One CTA per component; each thread runs a private depth-first branch and bound per (face, patch).
#define SL_THREADS 256
__global__ void __launch_bounds__(SL_THREADS) k_seedless(DcScalars *S, const double *__restrict__ xyz, const int *__restrict__ conn,
                                                         const double *__restrict__ fcoef, int n_face, unsigned char *comp)
{
    pdl_start();
    __shared__ double s_ecoef[6][28];
    __shared__ double s_nodes[81];
    __shared__ unsigned long long s_best;
    __shared__ double s_d[SL_THREADS], s_c[SL_THREADS];
    const int ns = min(S->n_seedless, DC_MAX_SEEDLESS);
    const int tid = threadIdx.x;
    for (int comp_i = blockIdx.x; comp_i < ns; comp_i += gridDim.x) {
    const int e = S->seedless_elem[comp_i];
    __syncthreads();
    if (tid < 27) {
        const int id = conn[(size_t)e * 27 + tid];
        for (int c = 0; c < 3; ++c) s_nodes[tid * 3 + c] = xyz[(size_t)id * 3 + c];
    }
    if (tid == 0) s_best = 0x7ff0000000000000ull;
    __syncthreads();
    if (tid < 18) {
        const int k = tid / 3, c = tid % 3;
        double x[9], a[9];
        for (int m = 0; m < 9; ++m) x[m] = s_nodes[c_face_node[k][m] * 3 + c];
        nodes_to_mono9(x, a);
        for (int m = 0; m < 9; ++m) s_ecoef[k][c * 9 + m] = a[m];
    }
    __syncthreads();
    if (tid < 6) s_ecoef[tid][27] = higher_order_const(s_ecoef[tid]);
    __syncthreads();
    const double t_tie = S->t_tie, theta2 = S->theta * S->theta, tol_d2 = S->tol_d * S->tol_d;
    const int max_level = S->max_level;
    double my_d = INFINITY, my_c = 0.0;
    for (int f = tid; f < n_face; f += SL_THREADS) {
        double AQ[28];
        for (int m = 0; m < 28; ++m) AQ[m] = __ldg(fcoef + (size_t)f * 28 + m);
        for (int k = 0; k < 6; ++k) {
            const double *AP = s_ecoef[k];
            NItem st[80];
            int top = 0;
            st[top].p = (unsigned)f; st[top].ak = 0; st[top].w2 = 0; st[top].w3 = 0; ++top;
            while (top > 0) {
                const NItem it = st[--top];
                double uc, vc, hP, sc, tc, hQ;
                nitem_box(it, uc, vc, hP, sc, tc, hQ);
                const NodeOut nb = bound_node<false>([&](int m) { return AP[m]; }, [&](int m) { return AQ[m]; }, AP[27], AQ[27], uc, vc, hP, sc, tc, hQ, theta2);
                double best = u2d(s_best);
                if (nb.ub < best) { atomicMin(&s_best, d2u(nb.ub)); best = nb.ub; }
                if (nb.lb > best + t_tie) continue;
                bool leaf = nb.leaf, splitP = false;
                if (!leaf) leaf = !choose_split(it, nb.splitP, max_level, splitP);
                if (leaf || top + 4 > 80) {
                    // the same iteration as k_np_solve, run to the end by this thread (an unconverged
                    // solve still yields an attained distance; a seedless component only needs the sign)
                    dcn::NwState s; s.x[0] = uc; s.x[1] = vc; s.x[2] = sc; s.x[3] = tc; s.iters = 0; s.ls = 0; s.phase = 1;
                    const double lo[4] = { uc - hP, vc - hP, sc - hQ, tc - hQ }, hi[4] = { uc + hP, vc + hP, sc + hQ, tc + hQ };
                    dcn::NwResult R; R.dist = INFINITY; R.cosv = 0.0; R.converged = 0;
                    auto cf = [&](int m) { return m < 27 ? AP[m] : AQ[m - 27]; };
                    while (!dcn::iterate(cf, s, lo, hi, tol_d2, -1.0, R)) { }
                    atomicMin(&s_best, d2u(R.dist));
                    if (R.dist < my_d - t_tie || (R.dist <= my_d + t_tie && fabs(R.cosv) > fabs(my_c))) {
                        my_d = dmin2(my_d, R.dist); my_c = R.cosv;
                    }
                } else {
                    for (int c = 0; c < 4; ++c) st[top++] = nitem_child(it, splitP, c);
                }
            }
        }
    }
    s_d[tid] = my_d; s_c[tid] = my_c;
    __syncthreads();
    if (tid == 0) {
        double dmin = INFINITY;
        for (int i = 0; i < SL_THREADS; ++i) dmin = dmin2(dmin, s_d[i]);
        double bc = 0.0;
        for (int i = 0; i < SL_THREADS; ++i) if (s_d[i] <= dmin + t_tie && fabs(s_c[i]) > fabs(bc)) bc = s_c[i];
        comp[e] = bc < 0.0 ? 1 : 2;
        atomicAdd(&S->c_seedless_total, 1ull);
    }
    }
}

// Labels of the elements S6 left undecided.  An element points at its tile-local root (or, a hooked root or a band
// element whose path k_uf_seed has halved, at some root above it), and every such root is in the list k_uf_tiles made:
// k_uf_resolve walks the global forest once per listed root and leaves the component's seed bits at the root itself
// (comp[] of a hooked root is otherwise unused), so k_uf_assign is a plain stream: labels, parent, comp[parent].
// A component with no seed at all is listed (by its global root) for k_seedless and its elements are left to k_uf_fix.
__device__ __forceinline__ void uf_label(DcScalars *S, long long e, int lab, int bits, signed char *labels, double *sdist, bool &conflict, int &out)
{
    out = lab;
    if (lab < 0) {
        if (bits == 0) return;                         // seedless: k_uf_fix
        conflict = bits == 3;
        out = (bits == 1) ? DC_HOLE : DC_NORMAL;
        labels[e] = (signed char)out;
        sdist[e] = out == DC_HOLE ? -S->d_band : S->d_band;
    } else if (bits == 3) conflict = true;
}
// census of the labels: ballots, then shared-memory counters, then one atomic per counter and CTA (a warp-level atomic
// on three global addresses was most of the duration of the old assign kernel)
__device__ __forceinline__ void uf_census(DcScalars *S, int lab, bool conflict)
{
    __shared__ unsigned s_cnt[4];
    if (threadIdx.x < 4) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const unsigned mc = __ballot_sync(0xffffffffu, lab == DC_CUT);
    const unsigned mh = __ballot_sync(0xffffffffu, lab == DC_HOLE);
    const unsigned mn = __ballot_sync(0xffffffffu, lab == DC_NORMAL);
    const unsigned mf = __ballot_sync(0xffffffffu, conflict);
    if ((threadIdx.x & 31) == 0) {
        if (mc) atomicAdd(&s_cnt[0], __popc(mc));
        if (mh) atomicAdd(&s_cnt[1], __popc(mh));
        if (mn) atomicAdd(&s_cnt[2], __popc(mn));
        if (mf) atomicAdd(&s_cnt[3], __popc(mf));
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_cnt[0]) atomicAdd(&S->c_cut, (unsigned long long)s_cnt[0]);
        if (s_cnt[1]) atomicAdd(&S->c_hole, (unsigned long long)s_cnt[1]);
        if (s_cnt[2]) atomicAdd(&S->c_normal, (unsigned long long)s_cnt[2]);
        if (s_cnt[3]) { atomicAdd(&S->c_fill_conflicts, (unsigned long long)s_cnt[3]); atomicOr(&S->status, DC_STATUS_FILL_CONFLICT); }
    }
}
__global__ void k_uf_resolve(DcScalars *S, const int *__restrict__ lroot_list, int *parent, unsigned char *comp)
{
    pdl_start();
    const int n = S->n_lroots;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int r = lroot_list[i];
        const int g = uf_find(parent, r);
        const int bits = ((volatile unsigned char *)comp)[g];
        if (g != r) comp[r] = (unsigned char)bits;        // (global roots keep their own; nobody reads a hooked root's before this)
        else if (bits == 0) {
            const int k = atomicAdd(&S->n_seedless, 1);
            if (k < DC_MAX_SEEDLESS) S->seedless_elem[k] = r;
            else atomicOr(&S->status, DC_STATUS_SEEDLESS_OVERFLOW);
        }
    }
}
__global__ void k_uf_assign(DcScalars *S, long long n_elem, const int *__restrict__ parent,
                            const unsigned char *__restrict__ comp, signed char *__restrict__ labels,
                            double *__restrict__ sdist)
{
    pdl_start();
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int lab = -2, out = -2;
    bool conflict = false;
    if (e < n_elem) {
        lab = labels[e]; out = lab;
        if (lab != DC_CUT) uf_label(S, e, lab, comp[parent[e]], labels, sdist, conflict, out);
    }
    uf_census(S, out, conflict);
}

// the elements of seedless components, once k_seedless has given those a sign (nothing to do on most cuts)
__global__ void k_uf_fix(DcScalars *S, long long n_elem, int *parent, const unsigned char *__restrict__ comp,
                         signed char *__restrict__ labels, double *__restrict__ sdist)
{
    pdl_start();
    if (S->n_seedless == 0) return;
    for (long long e0 = (long long)blockIdx.x * blockDim.x; e0 < n_elem; e0 += (long long)gridDim.x * blockDim.x) {
        const long long e = e0 + threadIdx.x;
        bool conflict = false;
        int out = -2;
        if (e < n_elem && labels[e] < 0) {
            int bits = comp[uf_find(parent, (int)e)];
            if (bits == 0) bits = 2;                    // (more seedless components than DC_MAX_SEEDLESS: status bit set)
            uf_label(S, e, -1, bits, labels, sdist, conflict, out);
        }
        uf_census(S, out, conflict);
    }
}

// small helpers
__global__ void k_boxes_to_aos(const double *__restrict__ ebox, long long n_elem, double *__restrict__ out)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_elem) return;
    for (int c = 0; c < 6; ++c) out[e * 6 + c] = ebox[(size_t)c * n_elem + e];
}

// FP64 FMA peak: 8 independent register-resident chains per thread
__global__ void __launch_bounds__(256) k_dfma_peak(double *out, int iters, double a, double b)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    const double s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

#include "dc_donor.cuh"

// ==========================================================================================
// host side
// ==========================================================================================
struct dc_ctx {
    int device, num_sms;
    int grid_roots, grid_bound_root, grid_decide;   // grid-stride grids of uniform-work kernels: whole waves of resident CTAs
    long long n_nodes, n_elem, max_faces, max_pairs, n_face, max_band, qcap;
    const double *xyz; const int *conn; const int *adj;
    const double *face_nodes;
    // workspace partition
    unsigned char *ws; size_t ws_bytes;
    DcScalars *S;
    double *ebox;             // [6][n_elem]
    int *adj_own;             // [n_elem][6] (derived) or NULL
    int *parent; unsigned char *comp; int *tile_flag;
    int *act_elem;
    int *band_elem; long long *band_start; int *band_cnt;
    double *ecoef; float *pbox; unsigned long long *best, *dmin;
    NItem *q[2], *nq; NLeafX *nqx;
    int *pair_face; unsigned long long *pair_key; int *pair_band;
    double *fbox_orig, *fbox, *fcoef; int *fcell, *fperm; float *fboxf;
    int *cell_count, *cell_start, *cell_fill; unsigned char *occ;
    int *pyr;                 // octree over the face bins (DC_FLAG_EXACT_FAR)
    float *ffar;              // [max_faces][16]: per-face records of the far pass
    int *far_sorted, *far_bins;   // the far elements in Morton order; the bins of the counting sort that makes it
    int *far_heavy;               // [n_elem]: the heavy elements served in a pass (the slice's are listed in act_elem)
    double *h_faces_dev; signed char *h_labels_dev; double *h_sdist_dev;   // staging for dc_classify_host
    cudaEvent_t ev[14], evk[10];
    cudaStream_t side; cudaEvent_t ev_fork, ev_join;   // second branch of dc_cut's graph (capture only)    // evk: boundaries between the kernels of S5/S6
    cudaStream_t last_stream;
    bool have_surface, have_cut;
    int launches_surface, launches_classify;   // kernels launched by the last dc_set_cut_surface / dc_classify
    DcScalars *S_host;        // pinned
    DcScalars *S_band_host;   // pinned: the scalars as the banded cut left them, when a far pass has run since
    bool last_was_graph;      // the last cut was a graph replay: no stage times
    bool far_ran; int far_passes; long long far_n_total; int far_error;
    // dc_cut with DC_FLAG_GRAPH: the launch sequences captured so far, by what they were captured for
    struct GraphEntry {
        const double *faces; long long n_face; dc_params P; signed char *labels; double *sdist; cudaStream_t stream;
        const double *h_faces; signed char *h_labels; double *h_sdist;     // dc_classify_host's buffers (copies inside the graph), else NULL
        cudaGraphExec_t exec; unsigned long long stamp; int launches_surface, launches_classify;
    } graphs[DC_MAX_GRAPHS];
    int n_graphs; unsigned long long graph_clock;
    const AdtNode *adt; int adt_nodes;   // donor search tree (dc_adt_build), caller's memory
};

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

struct WsLayout {
    size_t off_S, off_ebox, off_adj, off_parent, off_comp, off_tile_flag, off_act_elem, off_band_elem, off_band_start, off_band_cnt,
        off_ecoef, off_pbox, off_best, off_dmin, off_q0, off_q1, off_nq, off_nqx,
        off_pair_face, off_pair_key, off_pair_band, off_fbox_orig, off_fbox, off_fboxf, off_fcoef, off_fcell, off_fperm,
        off_cell_count, off_cell_start, off_cell_fill, off_occ, off_pyr, off_ffar, off_far_sorted, off_far_bins, off_far_heavy, off_hfaces, off_hlabels, off_hsdist, total;
    long long max_band, qcap;
};

// capacities derived from max_pairs: band elements (each has >= 1 pair, ~25 in the configs) and
// narrow-phase queue items per round
static long long band_capacity(long long n_elem, long long max_pairs)
{
    long long b = max_pairs / 8; if (b < 65536) b = 65536; if (b > n_elem) b = n_elem; return b;
}
static long long queue_capacity(long long max_pairs) { return max_pairs < (1LL << 20) ? (1LL << 20) : max_pairs; }

static WsLayout ws_layout(long long n_nodes, long long n_elem, long long max_faces, long long max_pairs)
{
    WsLayout L; size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o += align_up(bytes); return r; };
    L.off_S = take(sizeof(DcScalars));
    L.off_ebox = take((size_t)n_elem * 6 * 8);
    L.off_adj = take((size_t)n_elem * 6 * 4);
    L.off_parent = take((size_t)n_elem * 4);
    L.off_comp = take((size_t)n_elem + 4);
    L.off_tile_flag = take((size_t)(n_elem / UF_TILE + 2) * 4);
    L.off_act_elem = take((size_t)n_elem * 4);
    L.max_band = band_capacity(n_elem, max_pairs);
    L.qcap = queue_capacity(max_pairs);
    L.off_band_elem = take((size_t)L.max_band * 4);
    L.off_band_start = take((size_t)L.max_band * 8);
    L.off_band_cnt = take((size_t)L.max_band * 4);
    L.off_ecoef = take((size_t)L.max_band * 6 * 28 * 8);
    L.off_pbox = take((size_t)L.max_band * 36 * 8);
    L.off_best = take((size_t)L.max_band * 8);
    L.off_dmin = take((size_t)L.max_band * 8);
    L.off_q0 = take((size_t)L.qcap * sizeof(NItem));
    L.off_q1 = take((size_t)L.qcap * sizeof(NItem));
    L.off_nq = take((size_t)(L.qcap > L.max_band ? L.qcap : L.max_band) * sizeof(NItem));
    L.off_nqx = take((size_t)(L.qcap > L.max_band ? L.qcap : L.max_band) * sizeof(NLeafX));
    // pair arrays double as the scratch of the adjacency derivation (2 x n_nodes ints)
    size_t pf = (size_t)max_pairs * 4, pk = (size_t)max_pairs * 8;
    size_t need_adj = (size_t)n_nodes * 8;
    if (pf + pk < need_adj) pk = need_adj - pf;
    L.off_pair_face = take(pf);
    L.off_pair_key = take(pk);
    L.off_pair_band = take((size_t)max_pairs * 4);
    L.off_fbox_orig = take((size_t)max_faces * 6 * 8);
    L.off_fbox = take((size_t)max_faces * 6 * 8);
    L.off_fboxf = take((size_t)max_faces * 8 * 4);
    L.off_fcoef = take((size_t)max_faces * 28 * 8);
    L.off_fcell = take((size_t)max_faces * 4);
    L.off_fperm = take((size_t)max_faces * 4);
    L.off_cell_count = take((size_t)(DC_NCELL + 1) * 4);
    L.off_cell_start = take((size_t)(DC_NCELL + 1) * 4);
    L.off_cell_fill = take((size_t)(DC_NCELL + 8 + SCAN_NCHUNK) * 4);   // + the scan's chunk sums
    L.off_occ = take((size_t)DC_OCC * DC_OCC * DC_OCC);
    L.off_pyr = take((size_t)DC_PYR_TOTAL * 4);
    L.off_ffar = take((size_t)max_faces * 16 * 4);
    L.off_far_sorted = take((size_t)n_elem * 4);
    L.off_far_heavy = take((size_t)n_elem * 4);
    L.off_far_bins = take((size_t)(3 * (DC_NCELL + 8) + SCAN_NCHUNK) * 4);
    L.off_hfaces = take((size_t)max_faces * 27 * 8);
    L.off_hlabels = take((size_t)n_elem);
    L.off_hsdist = take((size_t)n_elem * 8);
    L.total = o;
    return L;
}

extern "C" size_t dc_workspace_bytes(long long n_nodes, long long n_elem, long long max_faces, long long max_pairs)
{
    if (n_nodes <= 0 || n_elem <= 0 || max_faces <= 0 || max_pairs <= 0) return 0;
    // (element, node, face and pair indices are 32-bit on the device; a work item keeps the band index in 29 bits)
    if (n_elem > 300000000LL || n_nodes > 2000000000LL || max_faces >= (1LL << 31) || max_pairs >= (1LL << 31)) return 0;
    return ws_layout(n_nodes, n_elem, max_faces, max_pairs).total;
}

#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { \
    fprintf(stderr, "libdc: %s failed: %s (%s:%d)\n", #call, cudaGetErrorString(e_), __FILE__, __LINE__); return DC_ERR_CUDA; } } while (0)

static inline unsigned nblk(long long n, int t) { return (unsigned)((n + t - 1) / t); }

// Every kernel of a cut is launched with programmatic stream serialisation: it starts as its predecessor's CTAs drain
// (each kernel raises griddepcontrol.launch_dependents on entry) and waits at griddepcontrol.wait -- its first
// instruction after that -- until the predecessor has completed and its writes are visible.  What overlaps is the launch
// latency and the tail of one kernel with the ramp of the next: a cut is ~38 short dependent kernels.
template <class... KArgs, class... Args>
static cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t st, Args &&... args)
{
    cudaLaunchConfig_t cfg; memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

// The events that time the stages (dc_stats.ms_stage / ms_kernel).  On a stream that is being captured into a CUDA graph
// (dc_cut with DC_FLAG_GRAPH, or the caller's own capture) they are left out: a plain record would only mark a dependency,
// and as nodes of the graph (cudaEventRecordExternal) the 22 of them cost 3 us each -- most of what the graph saves.
// dc_get_stats reports no stage times for a replayed cut; a plain dc_cut / dc_classify gives them.
static cudaError_t ev_record(cudaEvent_t ev, cudaStream_t st)
{
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    cudaError_t e = cudaStreamIsCapturing(st, &cs);
    if (e != cudaSuccess) return e;
    return cs == cudaStreamCaptureStatusActive ? cudaSuccess : cudaEventRecord(ev, st);
}

static int run_elem_boxes(dc_ctx *c, cudaStream_t st)
{
    CK(cudaMemsetAsync(&c->S->grid_max_diag2, 0, 8, st));
    CK(launch_pdl(k_elem_boxes, nblk(c->n_elem, EB_THREADS), EB_THREADS, st, c->S, c->xyz, c->conn, c->n_elem, c->ebox));
    CK(cudaGetLastError());
    return DC_OK;
}

extern "C" void dc_destroy(dc_ctx *c);

static int create_grid_body(dc_ctx *c, int num_sms, int device, long long n_nodes, const double *xyz_dev,
                            long long n_elem, const int *conn27_dev, const int *adj6_dev,
                            void *workspace_dev, size_t workspace_bytes, long long max_faces, long long max_pairs, cudaStream_t st)
{
    c->device = device; c->num_sms = num_sms;
    c->n_nodes = n_nodes; c->n_elem = n_elem; c->max_faces = max_faces; c->max_pairs = max_pairs;
    c->xyz = xyz_dev; c->conn = conn27_dev;
    c->ws = (unsigned char *)workspace_dev; c->ws_bytes = workspace_bytes;
    const WsLayout L = ws_layout(n_nodes, n_elem, max_faces, max_pairs);
    c->S = (DcScalars *)(c->ws + L.off_S);
    c->ebox = (double *)(c->ws + L.off_ebox);
    c->adj_own = (int *)(c->ws + L.off_adj);
    c->parent = (int *)(c->ws + L.off_parent);
    c->comp = c->ws + L.off_comp;
    c->tile_flag = (int *)(c->ws + L.off_tile_flag);
    c->act_elem = (int *)(c->ws + L.off_act_elem);
    c->max_band = L.max_band; c->qcap = L.qcap;
    c->band_elem = (int *)(c->ws + L.off_band_elem);
    c->band_start = (long long *)(c->ws + L.off_band_start);
    c->band_cnt = (int *)(c->ws + L.off_band_cnt);
    c->ecoef = (double *)(c->ws + L.off_ecoef);
    c->pbox = (float *)(c->ws + L.off_pbox);
    c->best = (unsigned long long *)(c->ws + L.off_best);
    c->dmin = (unsigned long long *)(c->ws + L.off_dmin);
    c->q[0] = (NItem *)(c->ws + L.off_q0);
    c->q[1] = (NItem *)(c->ws + L.off_q1);
    c->nq = (NItem *)(c->ws + L.off_nq);
    c->nqx = (NLeafX *)(c->ws + L.off_nqx);
    c->pair_face = (int *)(c->ws + L.off_pair_face);
    c->pair_key = (unsigned long long *)(c->ws + L.off_pair_key);
    c->pair_band = (int *)(c->ws + L.off_pair_band);
    c->fbox_orig = (double *)(c->ws + L.off_fbox_orig);
    c->fbox = (double *)(c->ws + L.off_fbox);
    c->fboxf = (float *)(c->ws + L.off_fboxf);
    c->fcoef = (double *)(c->ws + L.off_fcoef);
    c->fcell = (int *)(c->ws + L.off_fcell);
    c->fperm = (int *)(c->ws + L.off_fperm);
    c->cell_count = (int *)(c->ws + L.off_cell_count);
    c->cell_start = (int *)(c->ws + L.off_cell_start);
    c->cell_fill = (int *)(c->ws + L.off_cell_fill);
    c->occ = c->ws + L.off_occ;
    c->pyr = (int *)(c->ws + L.off_pyr);
    c->ffar = (float *)(c->ws + L.off_ffar);
    c->far_sorted = (int *)(c->ws + L.off_far_sorted);
    c->far_heavy = (int *)(c->ws + L.off_far_heavy);
    c->far_bins = (int *)(c->ws + L.off_far_bins);
    c->h_faces_dev = (double *)(c->ws + L.off_hfaces);
    c->h_labels_dev = (signed char *)(c->ws + L.off_hlabels);
    c->h_sdist_dev = (double *)(c->ws + L.off_hsdist);
    c->last_stream = st;
    {
        // A grid-stride kernel whose items all cost the same runs as long as its waves of resident CTAs: a grid that is not
        // a whole number of waves idles part of the GPU through its last one (k_np_roots at 8 CTAs per SM with 6 resident:
        // 1.33 waves, 0.086 ms; at 6: 0.066 ms).  Resident CTAs per SM from the occupancy calculator, not from a guess at
        // the register count.
        int occ = 0;
        CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_np_roots, 256, 0));
        c->grid_roots = num_sms * (occ > 0 ? occ : 1);
        CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_np_bound<true>, NPW_THREADS, 0));
        c->grid_bound_root = num_sms * (occ > 0 ? occ : 1) * 2;
        CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_np_decide, 256, 0));
        c->grid_decide = num_sms * (occ > 0 ? occ : 1);
    }
    for (int i = 0; i < 14; ++i) CK(cudaEventCreate(&c->ev[i]));
    CK(cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking));
    CK(cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
    for (int i = 0; i < 10; ++i) CK(cudaEventCreate(&c->evk[i]));
    CK(cudaMallocHost((void **)&c->S_host, sizeof(DcScalars)));
    CK(cudaMallocHost((void **)&c->S_band_host, sizeof(DcScalars)));
    CK(cudaMemsetAsync(c->S, 0, sizeof(DcScalars), st));
    CK(cudaMemsetAsync(c->tile_flag, 0, (size_t)(n_elem / UF_TILE + 2) * 4, st));
    int rc = run_elem_boxes(c, st);
    if (rc != DC_OK) return rc;
    if (adj6_dev) c->adj = adj6_dev;
    else {
        int *first = (int *)(c->ws + L.off_pair_face);
        int *second = first + n_nodes;
        CK(cudaMemsetAsync(first, 0xff, (size_t)n_nodes * 8, st));
        k_adj_pass1<<<nblk(n_elem * 6, 256), 256, 0, st>>>(c->conn, n_elem, first, second);
        k_adj_pass2<<<nblk(n_elem * 6, 256), 256, 0, st>>>(c->conn, n_elem, first, second, c->adj_own);
        CK(cudaGetLastError());
        c->adj = c->adj_own;
    }
    return DC_OK;
}


extern "C" int dc_create_grid(dc_ctx **out, int device, long long n_nodes, const double *xyz_dev,
                              long long n_elem, const int *conn27_dev, const int *adj6_dev,
                              void *workspace_dev, size_t workspace_bytes,
                              long long max_faces, long long max_pairs, void *stream)
{
    if (!out || !xyz_dev || !conn27_dev || !workspace_dev) return DC_ERR_ARG;
    const size_t need = dc_workspace_bytes(n_nodes, n_elem, max_faces, max_pairs);
    if (need == 0) return DC_ERR_ARG;
    if (workspace_bytes < need) return DC_ERR_WORKSPACE;
    if (((uintptr_t)workspace_dev & 255) != 0) return DC_ERR_ARG;
    CK(cudaSetDevice(device));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10 || prop.minor != 0) return DC_ERR_UNSUPPORTED;   // sm_100a only (the one cubin built): no fallback path exists
    dc_ctx *c = new (std::nothrow) dc_ctx();
    if (!c) return DC_ERR_ARG;
    memset(c, 0, sizeof *c);
    const int rc = create_grid_body(c, prop.multiProcessorCount, device, n_nodes, xyz_dev, n_elem, conn27_dev, adj6_dev,
                                    workspace_dev, workspace_bytes, max_faces, max_pairs, (cudaStream_t)stream);
    if (rc != DC_OK) { dc_destroy(c); return rc; }     // (events, pinned buffer and the context itself: one cleanup path)
    *out = c;
    return DC_OK;
}

extern "C" int dc_set_cut_surface(dc_ctx *c, long long n_face, const double *face_nodes_dev, void *stream)
{
    if (!c || !face_nodes_dev || n_face <= 0) return DC_ERR_ARG;
    if (n_face > c->max_faces) return DC_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    c->last_stream = st;
    CK(cudaSetDevice(c->device));
    CK(ev_record(c->ev[8], st));
    c->last_was_graph = false;
    c->face_nodes = face_nodes_dev; c->n_face = n_face;
    const int nf = (int)n_face;
    CK(launch_pdl(k_reset_surface, 1, 1, st, c->S));
    CK(launch_pdl(k_face_boxes, nblk(nf, 128), 128, st, c->S, face_nodes_dev, nf, c->fbox_orig));
    CK(launch_pdl(k_setup_surface, 1, 1, st, c->S, nf));
    CK(cudaMemsetAsync(c->cell_count, 0, (size_t)(DC_NCELL + 1) * 4, st));
    CK(cudaMemsetAsync(c->cell_fill, 0, (size_t)(DC_NCELL + 1) * 4, st));
    CK(launch_pdl(k_face_hist, nblk(nf, 128), 128, st, c->S, c->fbox_orig, nf, c->fcell, c->cell_count));
    CK(launch_pdl(k_scan_sums, SCAN_NCHUNK, 256, st, c->cell_count, c->cell_fill + DC_NCELL + 8));
    CK(launch_pdl(k_scan_cells, SCAN_NCHUNK, 256, st, c->cell_count, c->cell_fill + DC_NCELL + 8, c->cell_start));
    CK(launch_pdl(k_cell_occ, (DC_OCC * DC_OCC * DC_OCC + 127) / 128, 128, st, c->cell_start, c->occ));
    CK(launch_pdl(k_face_scatter, nblk(nf, 128), 128, st, face_nodes_dev, c->fbox_orig, c->fcell, c->cell_start, c->cell_fill,
                                                   nf, c->fperm, c->fbox, c->fcoef, c->fboxf));
    CK(cudaGetLastError());
    CK(ev_record(c->ev[9], st));
    c->launches_surface = 8;
    c->have_surface = true;
    return DC_OK;
}

// S5 as a launch sequence (dc_narrow.cuh).  part 0: the band's narrow phase, with the events that time it.  The exact far
// pass (dc_far.cuh) runs the same kernels on its own elements: part 1 = stage + seed solves (once per slice), part 3 = the
// seed solves again (on better faces), part 2 = roots to the last solve (once per pass, after the pass's candidate pairs
// have been written).
#define EVREC(ev_, st_) do { if (part == 0) CK(ev_record(ev_, st_)); } while (0)
static int launch_narrow(dc_ctx *c, cudaStream_t st, int rounds, int grid_rounds, int part)
{
    // ---- S5: wavefront narrow phase (dc_narrow.cuh)
    const int gw = c->num_sms * 8;     // grid-stride grids: 8 CTAs of 128 threads per SM
    DcScalars *S = c->S;
    if (part != 2 && part != 3) CK(launch_pdl(k_np_stage, gw, 128, st, S, c->xyz, c->conn, c->band_elem, c->ecoef, c->pbox));
    // seed solves: one per band element, queue = nq[0 .. n_band); never re-split, and cut short after NW_SEED_MAXIT
    // evaluations (a seed only has to leave an attained upper bound: its pair comes back as a leaf)
    const int gs = c->num_sms * 2 * 4;     // solve grids: grid-stride, 2 resident CTAs of 128 threads per SM
    EVREC(c->ev[7], st);
    if (part != 2)
        CK(launch_pdl(k_np_solve<0>, gs, NW_THREADS, st, S, &S->n_band, c->max_band, c->nq, nullptr, nullptr, c->pair_face, c->fcoef, c->ecoef,
                                                 c->best, c->dmin, c->pair_key, nullptr, nullptr, 0, nullptr, nullptr, 0, 0, NW_SEED_MAXIT));
    if (part == 1 || part == 3) { CK(cudaGetLastError()); return DC_OK; }
    EVREC(c->ev[10], st);
    CK(launch_pdl(k_np_roots, c->grid_roots, 256, st, S, c->pair_band, c->pair_face, c->fboxf, c->pbox, c->best, c->max_pairs,
                                               c->q[0], &S->qn[0], c->qcap));
    // branch and bound, level by level (every item of round r has lP + lQ = r, so 2 max_level + 1 rounds end it):
    // the first rounds as grids, the sparse rest inside one CTA; every round appends its leaves to ONE queue
    EVREC(c->evk[0], st);
    CK(launch_pdl(k_np_bound<true>, c->grid_bound_root, NPW_THREADS, st, S, &S->qn[0], c->q[0], c->pair_face, c->fcoef, c->ecoef, c->best,
                                                 c->q[1], &S->qn[1], c->nq, c->nqx, &S->nn[0], c->qcap, 0));
    for (int r = 1; r < grid_rounds; ++r)
        CK(launch_pdl(k_np_bound<false>, gw, NPW_THREADS, st, S, &S->qn[r], c->q[r & 1], c->pair_face, c->fcoef, c->ecoef, c->best,
                                                      c->q[(r + 1) & 1], &S->qn[r + 1], c->nq, c->nqx, &S->nn[0], c->qcap, 0));
    if (rounds > grid_rounds)
        CK(launch_pdl(k_np_bound_tail, 1, NP_TAIL_THREADS, st, S, grid_rounds, rounds, c->q[0], c->q[1], c->pair_face, c->fcoef, c->ecoef, c->best,
                                                       c->nq, c->nqx, &S->nn[0], c->qcap));
    // all leaves: first dropped if their element's best distance has fallen below their lower bound meanwhile (the two
    // bound queues are free by now and take the compacted leaf queue), then three solve passes (the old leaf queue's
    // memory holds the continuations and the overflow queue of sub-leaves)
    EVREC(c->ev[5], st);
    NItem *lq = c->q[0]; NLeafX *lqx = (NLeafX *)c->q[1];
    NCont *contA = (NCont *)c->nq, *contB = (NCont *)c->nqx;
    const long long capA = c->qcap / 4, capB = c->qcap / 8;
    NItem *ovf1 = (NItem *)c->nqx + c->qcap / 2;
    const long long cap_ovf1 = c->qcap / 2;
    CK(launch_pdl(k_np_compact, c->num_sms * 8, 256, st, S, &S->nn[0], c->qcap, c->nq, c->nqx, c->best, lq, lqx, &S->nn[5]));
    EVREC(c->evk[1], st);
    CK(launch_pdl(k_np_solve<0>, gs, NW_THREADS, st, S, &S->nn[5], c->qcap, lq, lqx, nullptr, c->pair_face, c->fcoef, c->ecoef,
                                             c->best, c->dmin, c->pair_key, contA, &S->nh[0], capA, ovf1, &S->nn[1], cap_ovf1, NW_BUDGET1, NW_MAXIT));
    CK(launch_pdl(k_np_solve<1>, gs, NW_THREADS, st, S, &S->nh[0], capA, nullptr, nullptr, contA, c->pair_face, c->fcoef, c->ecoef,
                                             c->best, c->dmin, c->pair_key, contB, &S->nh[1], capB, ovf1, &S->nn[1], cap_ovf1, NW_BUDGET2, NW_MAXIT));
    CK(launch_pdl(k_np_solve<1>, gs, NW_THREADS, st, S, &S->nh[1], capB, nullptr, nullptr, contB, c->pair_face, c->fcoef, c->ecoef,
                                             c->best, c->dmin, c->pair_key, nullptr, nullptr, 0, ovf1, &S->nn[1], cap_ovf1, 0, NW_MAXIT));
    EVREC(c->evk[2], st);
    // The sub-leaves of unconverged solves come back through one bound pass (best[b] is final or nearly so: most of them
    // are pruned) and one solve launch, twice; the last launch finishes whatever still fails on the lane that held it.
    CK(launch_pdl(k_np_bound<false>, gw, NPW_THREADS, st, S, &S->nn[1], ovf1, c->pair_face, c->fcoef, c->ecoef, c->best,
                                           nullptr, &S->qn[DC_NQN - 1], lq, lqx, &S->nn[2], c->qcap, 1));
    CK(launch_pdl(k_np_solve<0>, gs, NW_THREADS, st, S, &S->nn[2], c->qcap, lq, lqx, nullptr, c->pair_face, c->fcoef, c->ecoef,
                                             c->best, c->dmin, c->pair_key, nullptr, nullptr, 0, c->nq, &S->nn[3], c->qcap, 0, NW_OVF_MAXIT));
    CK(launch_pdl(k_np_bound<false>, gw, NPW_THREADS, st, S, &S->nn[3], c->nq, c->pair_face, c->fcoef, c->ecoef, c->best,
                                           nullptr, &S->qn[DC_NQN - 1], lq, lqx, &S->nn[4], c->qcap, 1));
    CK(launch_pdl(k_np_solve<0>, gs, NW_THREADS, st, S, &S->nn[4], c->qcap, lq, lqx, nullptr, c->pair_face, c->fcoef, c->ecoef,
                                             c->best, c->dmin, c->pair_key, nullptr, nullptr, 0, nullptr, nullptr, 0, 0, NW_OVF_MAXIT));
    EVREC(c->ev[6], st);
    CK(cudaGetLastError());
    return DC_OK;
}
#undef EVREC

// DC_FLAG_EXACT_FAR: the exact distance of the elements the banded cut left clamped (dc_far.cuh).  Slices of at most
// max_band elements (the narrow phase keeps 1.3 KB of patch coefficients per element), passes sized to the pair list within a
// slice.  Synchronises the stream (two counters are read back per pass).
static int run_exact_far(dc_ctx *c, cudaStream_t st, const signed char *labels_dev, double *sdist_dev, int rounds, int grid_rounds)
{
    DcScalars *S = c->S;
    const long long ne = c->n_elem;
    unsigned char *pmask = (unsigned char *)c->pyr;
    CK(ev_record(c->ev[11], st));
    k_far_pyramid<<<nblk(DC_PYR_TOTAL, 128), 128, 0, st>>>(c->cell_start, pmask);
    k_far_faces<<<nblk(c->n_face, 128), 128, 0, st>>>(S, c->fcoef, c->fbox, (int)c->n_face, c->ffar);
    k_far_list<<<nblk(ne, 256), 256, 0, st>>>(S, ne, labels_dev, sdist_dev, c->ebox, c->act_elem);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(c->S_band_host, S, sizeof(DcScalars), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    c->far_ran = true; c->far_passes = 0; c->far_error = 0;
    long long n_far = c->S_band_host->far_n[0];
    c->far_n_total = n_far;
    if (c->S_band_host->status & DC_STATUS_INVALID) n_far = 0;       // (the banded cut itself failed: nothing to refine)
    // the union-find arrays are free by now: act_elem holds the far elements as found, parent their Morton codes and, once
    // they are sorted by those, their nearest faces
    int *list = c->far_sorted, *fstar = c->parent;
    if (n_far > 0) {
        int *bin_count = c->far_bins, *bin_start = bin_count + DC_NCELL + 8, *bin_fill = bin_start + DC_NCELL + 8, *chunk = bin_fill + DC_NCELL + 8;
        CK(cudaMemsetAsync(bin_count, 0, (size_t)(DC_NCELL + 8) * 4, st));
        CK(cudaMemsetAsync(bin_fill, 0, (size_t)(DC_NCELL + 8) * 4, st));
        k_far_codes<<<nblk(n_far, 256), 256, 0, st>>>(S, c->act_elem, c->ebox, ne, c->parent, bin_count);
        k_scan_sums<<<SCAN_NCHUNK, 256, 0, st>>>(bin_count, chunk);
        k_scan_cells<<<SCAN_NCHUNK, 256, 0, st>>>(bin_count, chunk, bin_start);
        k_far_sort<<<nblk(n_far, 256), 256, 0, st>>>(S, c->act_elem, c->parent, bin_start, bin_fill, list);
    }
    if (n_far > 0)
        k_far_nearest<<<nblk(n_far, 128), 128, 0, st>>>(S, list, (int)n_far, c->ebox, ne, c->cell_start, pmask, c->ffar, fstar);
    // pair slots of one pass: a sixth of the list, so that the root items (up to 6 per pair: the patches of a small distant
    // element are all about as near as each other) fit the queues
    const long long cap = (c->max_pairs < c->qcap ? c->max_pairs : c->qcap) / 6;
    for (long long s0 = 0; s0 < n_far && !c->far_error; s0 += c->max_band) {
        const long long m = n_far - s0 < c->max_band ? n_far - s0 : c->max_band;
        k_far_reset<<<1, 1, 0, st>>>(S, (int)m, 1);
        k_far_slots<<<nblk(m, 256), 256, 0, st>>>(list + s0, fstar + s0, (int)m, c->band_elem, c->band_start, c->band_cnt, c->pair_face,
                                                   c->pair_key, c->pair_band, c->nq, c->best, c->dmin);
        { const int rc = launch_narrow(c, st, rounds, grid_rounds, 1); if (rc) return rc; }
        k_far_count<<<nblk(m, 128), 128, 0, st>>>(S, c->ebox, ne, c->cell_start, pmask, c->ffar, c->band_elem, c->band_cnt, c->best, c->act_elem, c->pair_face, 1);
        { const int rc = launch_narrow(c, st, rounds, grid_rounds, 3); if (rc) return rc; }      // (second seed solve)
        k_far_count<<<nblk(m, 128), 128, 0, st>>>(S, c->ebox, ne, c->cell_start, pmask, c->ffar, c->band_elem, c->band_cnt, c->best, c->act_elem, c->pair_face, 0);
        k_far_heavy_count<<<c->num_sms * 4, FAR_HEAVY_THREADS, 0, st>>>(S, c->ebox, ne, c->ffar, c->band_elem, c->band_cnt, c->best, c->act_elem);
        long long pending = m;
        while (pending > 0 && !c->far_error) {
            k_far_reset<<<1, 1, 0, st>>>(S, (int)m, 0);
            k_far_pairs<<<nblk(m, 128), 128, 0, st>>>(S, c->ebox, ne, c->cell_start, pmask, c->ffar, c->band_elem, c->band_start, c->band_cnt,
                                                       c->pair_face, c->pair_key, c->pair_band, c->best, cap, c->far_heavy);
            k_far_heavy_pairs<<<c->num_sms * 4, FAR_HEAVY_THREADS, 0, st>>>(S, c->ebox, ne, c->ffar, c->band_elem, c->band_start, c->best, c->far_heavy,
                                                                             c->pair_face, c->pair_key, c->pair_band);
            k_far_fix<<<1, 1, 0, st>>>(S);
            { const int rc = launch_narrow(c, st, rounds, grid_rounds, 2); if (rc) return rc; }
            k_far_decide<<<nblk(m, 256), 256, 0, st>>>(S, c->band_elem, c->band_start, c->band_cnt, c->dmin, labels_dev, sdist_dev);
            CK(cudaGetLastError());
            CK(cudaMemcpyAsync(c->S_host, S, sizeof(DcScalars), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            ++c->far_passes;
            const int done = c->S_host->far_pass_done;
            if (c->S_host->status & DC_STATUS_INVALID) c->far_error = 1;          // (a queue of the narrow phase overflowed)
            else if (done == 0) c->far_error = 2;                                    // (an element's candidates exceed a pass)
            pending -= done;
        }
    }
    CK(ev_record(c->ev[12], st));
    return DC_OK;
}

extern "C" int dc_classify(dc_ctx *c, const dc_params *params, signed char *labels_dev, double *sdist_dev, void *stream)
{
    if (!c || !labels_dev || !sdist_dev) return DC_ERR_ARG;
    if (!c->have_surface) return DC_ERR_STATE;
    cudaStream_t st = (cudaStream_t)stream;
    c->last_stream = st;
    CK(cudaSetDevice(c->device));
    dc_params P; memset(&P, 0, sizeof P);
    if (params) P = *params;
    const long long ne = c->n_elem;
    c->last_was_graph = false;
    CK(ev_record(c->ev[0], st));
    if (P.flags & DC_FLAG_RECOMPUTE_BOXES) { int rc = run_elem_boxes(c, st); if (rc) return rc; }
    CK(ev_record(c->ev[1], st));
    CK(launch_pdl(k_setup_classify, 1, 1, st, c->S, P, (int)c->max_band));
    CK(launch_pdl(k_filter, nblk(ne, 256), 256, st, c->S, c->ebox, ne, labels_dev, c->parent, c->comp, c->cell_start, c->occ, c->act_elem));
    CK(launch_pdl(k_pairs, c->num_sms * 16, 256, st, c->S, c->ebox, ne, c->act_elem, c->cell_start, c->fbox, c->max_pairs,
                                           c->band_elem, c->band_start, c->band_cnt, c->pair_face, c->pair_key,
                                           c->pair_band, c->nq, c->best, c->dmin));
    CK(ev_record(c->ev[2], st));
    const int max_level = (P.max_level > 0 && P.max_level <= 12) ? P.max_level : 12;
    const int rounds = 2 * max_level + 1;
    const int grid_rounds = rounds < DC_GRID_ROUNDS ? rounds : DC_GRID_ROUNDS;
    if (P.flags & DC_FLAG_PAPER_MODE) {
        // ---- the paper's approximate cut of the band elements (dc_paper.cuh) in place of S5/S6; its work arrays live in the
        // memory of the exact mode's per-element coefficients (1344 bytes per band element there, 656 here)
        DcScalars *S = c->S;
        PmWork W;
        unsigned char *base = (unsigned char *)c->ecoef;
        const size_t mb = (size_t)c->max_band;
        W.sel1 = (int *)base; base += mb * PM_NF1 * 4;
        W.corner = (int *)base; base += mb * PM_NF1 * 4;
        W.sel2 = (int *)base; base += mb * PM_NF2 * 4;
        W.d1 = (double *)base; base += mb * PM_NF1 * 8;
        W.d2 = (double *)base; base += mb * PM_NF2 * 3 * 8;
        W.v2 = (double *)base;
        const int g = c->num_sms * 8;
        CK(launch_pdl(k_pm_rank, g, 128, st, S, c->xyz, c->conn, c->band_elem, c->band_start, c->band_cnt, c->pair_face, c->fperm, c->face_nodes, W));
        CK(launch_pdl(k_pm_pass1, g, 128, st, S, c->xyz, c->conn, c->band_elem, c->face_nodes, W));
        CK(launch_pdl(k_pm_select, g, 128, st, S, W));
        CK(launch_pdl(k_pm_pass2, g, 128, st, S, c->xyz, c->conn, c->band_elem, c->face_nodes, W));
        CK(launch_pdl(k_pm_decide, g, 128, st, S, c->band_elem, c->face_nodes, W, labels_dev, sdist_dev));
        CK(ev_record(c->ev[3], st));
    } else {
    { const int rc = launch_narrow(c, st, rounds, grid_rounds, 0); if (rc) return rc; }
    DcScalars *S = c->S;
    CK(launch_pdl(k_np_decide, c->grid_decide, 256, st, S, c->band_elem, c->band_start, c->band_cnt, c->best, c->dmin,
                                                                              c->pair_key, labels_dev, sdist_dev));
    CK(ev_record(c->ev[3], st));
    }
    CK(launch_pdl(k_uf_tiles, nblk(ne, UF_TILE), UF_TILE, st, c->S, labels_dev, c->adj, ne, c->parent, c->tile_flag, c->act_elem));
    CK(launch_pdl(k_uf_seed, c->num_sms * 8, 256, st, c->S, c->band_elem, labels_dev, c->parent, c->comp));
    CK(launch_pdl(k_uf_resolve, c->num_sms * 4, 256, st, c->S, c->act_elem, c->parent, c->comp));
    CK(launch_pdl(k_uf_assign, nblk(ne, 256), 256, st, c->S, ne, c->parent, c->comp, labels_dev, sdist_dev));
    CK(launch_pdl(k_seedless, 32, SL_THREADS, st, c->S, c->xyz, c->conn, c->fcoef, (int)c->n_face, c->comp));
    CK(launch_pdl(k_uf_fix, c->num_sms * 4, 256, st, c->S, ne, c->parent, c->comp, labels_dev, sdist_dev));
    CK(cudaGetLastError());
    CK(ev_record(c->ev[4], st));
    c->far_ran = false;
    if ((P.flags & DC_FLAG_EXACT_FAR) && !(P.flags & DC_FLAG_PAPER_MODE)) {
        const int rc = run_exact_far(c, st, labels_dev, sdist_dev, rounds, grid_rounds);
        if (rc) return rc;
    }
    c->launches_classify = ((P.flags & DC_FLAG_PAPER_MODE) ? 13 : 21 + grid_rounds + (rounds > grid_rounds ? 1 : 0)) + ((P.flags & DC_FLAG_RECOMPUTE_BOXES) ? 1 : 0);
    c->have_cut = true;
    return DC_OK;
}

// One cut in one call: dc_set_cut_surface + dc_classify.  With DC_FLAG_GRAPH the launch sequence (about 35 short kernels,
// two memsets, the stage events) is captured into a CUDA graph the first time it is asked for with these arguments, and
// replayed afterwards: the gaps between dependent launches go (config 2: 1.22 -> 1.11 ms per cut; config 0: 0.28 -> 0.17).
// Everything a replay must see anew is on the device (the cut's counters, the epoch of the flood fill's flags); what the
// graph fixes is what it was captured for: the surface's address and face count, the parameters, the output addresses, the
// stream.  The surface's CONTENTS may change between calls (a moving body updated in place: the re-cut of PAPER.md L233).
// (h_faces / h_labels / h_sdist: dc_classify_host's pinned host buffers, or all NULL -- the copies then become nodes of the
// graph: the faces' upload at the head of the surface's branch, next to S2, the results' download at the end)
static int cut_impl(dc_ctx *c, const dc_params *params, long long n_face, const double *face_nodes_dev,
                    signed char *labels_dev, double *sdist_dev, void *stream,
                    const double *h_faces, signed char *h_labels, double *h_sdist)
{
    if (!c || !face_nodes_dev || !labels_dev || !sdist_dev || n_face <= 0) return DC_ERR_ARG;
    if (n_face > c->max_faces) return DC_ERR_WORKSPACE;
    dc_params P; memset(&P, 0, sizeof P);
    if (params) P = *params;
    cudaStream_t st = (cudaStream_t)stream;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    CK(cudaSetDevice(c->device));
    CK(cudaStreamIsCapturing(st, &cs));
    // no graph of our own: not asked for; the far pass reads counters back between its passes; the caller is capturing
    // already (our launches then go into the caller's graph); the legacy default stream cannot be captured
    if (!(P.flags & DC_FLAG_GRAPH) || (P.flags & DC_FLAG_EXACT_FAR) || cs != cudaStreamCaptureStatusNone || st == nullptr) {
        if (h_faces) CK(cudaMemcpyAsync((void *)face_nodes_dev, h_faces, (size_t)n_face * 27 * 8, cudaMemcpyHostToDevice, st));
        int rc = dc_set_cut_surface(c, n_face, face_nodes_dev, stream);
        if (!rc) rc = dc_classify(c, &P, labels_dev, sdist_dev, stream);
        if (rc) return rc;
        if (h_labels) CK(cudaMemcpyAsync(h_labels, labels_dev, (size_t)c->n_elem, cudaMemcpyDeviceToHost, st));
        if (h_sdist) CK(cudaMemcpyAsync(h_sdist, sdist_dev, (size_t)c->n_elem * 8, cudaMemcpyDeviceToHost, st));
        return DC_OK;
    }
    dc_ctx::GraphEntry *g = nullptr;
    for (int i = 0; i < c->n_graphs; ++i) {
        dc_ctx::GraphEntry &q = c->graphs[i];
        if (q.faces == face_nodes_dev && q.n_face == n_face && q.labels == labels_dev && q.sdist == sdist_dev && q.stream == st &&
            q.h_faces == h_faces && q.h_labels == h_labels && q.h_sdist == h_sdist && memcmp(&q.P, &P, sizeof P) == 0) { g = &q; break; }
    }
    if (!g) {
        CK(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
        // Two branches: the surface's own preparation (S1 + S3: ten short dependent launches over the faces, a few dozen
        // microseconds that leave most of the GPU idle) does not depend on the element boxes (S2: one pass over the raw
        // nodes at HBM speed) nor S2 on it, so the graph runs them side by side and joins them in front of S4.
        int rc = DC_OK;
        const bool fork = (P.flags & DC_FLAG_RECOMPUTE_BOXES) != 0;
        if (fork) {
            cudaError_t e1 = cudaEventRecord(c->ev_fork, st);
            if (e1 == cudaSuccess) e1 = cudaStreamWaitEvent(c->side, c->ev_fork, 0);
            if (e1 == cudaSuccess && h_faces)
                e1 = cudaMemcpyAsync((void *)face_nodes_dev, h_faces, (size_t)n_face * 27 * 8, cudaMemcpyHostToDevice, c->side);
            if (e1 != cudaSuccess) rc = DC_ERR_CUDA;
            if (!rc) rc = dc_set_cut_surface(c, n_face, face_nodes_dev, (void *)c->side);
            if (!rc) rc = run_elem_boxes(c, st);
            if (!rc) {
                e1 = cudaEventRecord(c->ev_join, c->side);
                if (e1 == cudaSuccess) e1 = cudaStreamWaitEvent(st, c->ev_join, 0);
                if (e1 != cudaSuccess) rc = DC_ERR_CUDA;
            }
            dc_params Q = P; Q.flags &= ~DC_FLAG_RECOMPUTE_BOXES;
            if (!rc) rc = dc_classify(c, &Q, labels_dev, sdist_dev, stream);
            c->launches_classify += 1;          // (k_elem_boxes)
        } else {
            if (h_faces && cudaMemcpyAsync((void *)face_nodes_dev, h_faces, (size_t)n_face * 27 * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) rc = DC_ERR_CUDA;
            if (!rc) rc = dc_set_cut_surface(c, n_face, face_nodes_dev, stream);
            if (!rc) rc = dc_classify(c, &P, labels_dev, sdist_dev, stream);
        }
        if (!rc && h_labels && cudaMemcpyAsync(h_labels, labels_dev, (size_t)c->n_elem, cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = DC_ERR_CUDA;
        if (!rc && h_sdist && cudaMemcpyAsync(h_sdist, sdist_dev, (size_t)c->n_elem * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = DC_ERR_CUDA;
        cudaGraph_t graph = nullptr;
        const cudaError_t e = cudaStreamEndCapture(st, &graph);
        if (rc || e != cudaSuccess || !graph) {
            if (graph) cudaGraphDestroy(graph);
            (void)cudaGetLastError();
            c->have_cut = false;
            return rc ? rc : DC_ERR_CUDA;
        }
        cudaGraphExec_t exec = nullptr;
        const cudaError_t ei = cudaGraphInstantiate(&exec, graph, 0);
        cudaGraphDestroy(graph);
        if (ei != cudaSuccess) { fprintf(stderr, "libdc: cudaGraphInstantiate failed: %s\n", cudaGetErrorString(ei)); return DC_ERR_CUDA; }
        if (c->n_graphs < DC_MAX_GRAPHS) g = &c->graphs[c->n_graphs++];
        else {
            g = &c->graphs[0];
            for (int i = 1; i < DC_MAX_GRAPHS; ++i) if (c->graphs[i].stamp < g->stamp) g = &c->graphs[i];
            cudaGraphExecDestroy(g->exec);
        }
        g->faces = face_nodes_dev; g->n_face = n_face; g->P = P; g->labels = labels_dev; g->sdist = sdist_dev; g->stream = st;
        g->h_faces = h_faces; g->h_labels = h_labels; g->h_sdist = h_sdist;
        g->exec = exec; g->launches_surface = c->launches_surface; g->launches_classify = c->launches_classify;
    }
    g->stamp = ++c->graph_clock;
    // what the two calls leave on the host
    c->face_nodes = face_nodes_dev; c->n_face = n_face; c->last_stream = st;
    c->launches_surface = g->launches_surface; c->launches_classify = g->launches_classify;
    c->have_surface = true; c->have_cut = true; c->far_ran = false; c->last_was_graph = true;
    CK(cudaGraphLaunch(g->exec, st));
    return DC_OK;
}

extern "C" int dc_cut(dc_ctx *c, const dc_params *params, long long n_face, const double *face_nodes_dev,
                      signed char *labels_dev, double *sdist_dev, void *stream)
{
    return cut_impl(c, params, n_face, face_nodes_dev, labels_dev, sdist_dev, stream, nullptr, nullptr, nullptr);
}

// is this host pointer page-locked (cudaMallocHost / cudaHostRegister)?  Only then can its copies be nodes of a graph that
// run asynchronously.
static bool host_pinned(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeHost;
}

extern "C" int dc_classify_host(dc_ctx *c, const dc_params *params, long long n_face, const double *face_nodes_host,
                                signed char *labels_host, double *sdist_host, void *stream)
{
    if (!c || !face_nodes_host || !labels_host || !sdist_host || n_face <= 0) return DC_ERR_ARG;
    if (n_face > c->max_faces) return DC_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(c->device));
    if (params && (params->flags & DC_FLAG_GRAPH) && host_pinned(face_nodes_host) && host_pinned(labels_host) && host_pinned(sdist_host)) {
        // copies and cut in ONE graph: the faces' upload runs beside S2, which does not need them
        const int rc = cut_impl(c, params, n_face, c->h_faces_dev, c->h_labels_dev, c->h_sdist_dev, stream,
                                face_nodes_host, labels_host, sdist_host);
        if (rc) return rc;
        CK(cudaStreamSynchronize(st));
        return DC_OK;
    }
    CK(cudaMemcpyAsync(c->h_faces_dev, face_nodes_host, (size_t)n_face * 27 * 8, cudaMemcpyHostToDevice, st));
    const int rc = dc_cut(c, params, n_face, c->h_faces_dev, c->h_labels_dev, c->h_sdist_dev, stream);
    if (rc) return rc;
    CK(cudaMemcpyAsync(labels_host, c->h_labels_dev, (size_t)c->n_elem, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(sdist_host, c->h_sdist_dev, (size_t)c->n_elem * 8, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return DC_OK;
}

extern "C" int dc_get_element_boxes(dc_ctx *c, double *out_dev, void *stream)
{
    if (!c || !out_dev) return DC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    k_boxes_to_aos<<<nblk(c->n_elem, 256), 256, 0, st>>>(c->ebox, c->n_elem, out_dev);
    CK(cudaGetLastError());
    return DC_OK;
}

extern "C" int dc_get_adjacency(dc_ctx *c, int *out_dev, void *stream)
{
    if (!c || !out_dev) return DC_ERR_ARG;
    CK(cudaMemcpyAsync(out_dev, c->adj, (size_t)c->n_elem * 6 * 4, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return DC_OK;
}

extern "C" long long dc_get_pairs(dc_ctx *c, int *elem_host, int *face_host, long long cap)
{
    if (!c || !elem_host || !face_host) return DC_ERR_ARG;
    if (!c->have_cut || c->far_ran) return DC_ERR_STATE;     // (the chunks of an exact far pass have overwritten the band's lists)
    CK(cudaStreamSynchronize(c->last_stream));
    CK(cudaMemcpy(c->S_host, c->S, sizeof(DcScalars), cudaMemcpyDeviceToHost));
    const int na = c->S_host->n_band < (int)c->max_band ? c->S_host->n_band : (int)c->max_band;
    long long np = (long long)c->S_host->n_pairs; if (np > c->max_pairs) np = c->max_pairs;
    int *ae = new (std::nothrow) int[na > 0 ? na : 1]; long long *as = new (std::nothrow) long long[na > 0 ? na : 1];
    int *ac = new (std::nothrow) int[na > 0 ? na : 1]; int *perm = new (std::nothrow) int[c->n_face > 0 ? c->n_face : 1];
    int *pf = new (std::nothrow) int[np > 0 ? np : 1];
    long long n = DC_ERR_ARG;
    if (ae && as && ac && perm && pf) {
        n = DC_ERR_CUDA;
        if (cudaMemcpy(ae, c->band_elem, (size_t)na * 4, cudaMemcpyDeviceToHost) == cudaSuccess &&
            cudaMemcpy(as, c->band_start, (size_t)na * 8, cudaMemcpyDeviceToHost) == cudaSuccess &&
            cudaMemcpy(ac, c->band_cnt, (size_t)na * 4, cudaMemcpyDeviceToHost) == cudaSuccess &&
            cudaMemcpy(perm, c->fperm, (size_t)c->n_face * 4, cudaMemcpyDeviceToHost) == cudaSuccess &&
            cudaMemcpy(pf, c->pair_face, (size_t)np * 4, cudaMemcpyDeviceToHost) == cudaSuccess) {
            n = 0;
            for (int a = 0; a < na; ++a)
                for (int i = 0; i < ac[a]; ++i) {
                    if (n < cap && as[a] + i < np) { elem_host[n] = ae[a]; face_host[n] = perm[pf[as[a] + i]]; }
                    ++n;
                }
        } else fprintf(stderr, "libdc: dc_get_pairs: a device-to-host copy failed: %s\n", cudaGetErrorString(cudaGetLastError()));
    }
    delete[] ae; delete[] as; delete[] ac; delete[] perm; delete[] pf;
    return n;
}

extern "C" int dc_get_stats(dc_ctx *c, dc_stats *o)
{
    if (!c || !o) return DC_ERR_ARG;
    CK(cudaSetDevice(c->device));
    CK(cudaStreamSynchronize(c->last_stream));
    CK(cudaMemcpy(c->S_host, c->S, sizeof(DcScalars), cudaMemcpyDeviceToHost));
    // after an exact far pass the band's counters are the ones saved before it (its chunks reuse the band's lists)
    const bool far = c->have_cut && c->far_ran;
    DcScalars &S = far ? *c->S_band_host : *c->S_host;
    memset(o, 0, sizeof *o);
    if (far) {
        const DcScalars &F = *c->S_host;
        S.status |= F.status;
        o->n_far = c->far_n_total; o->n_far_done = F.far_done; o->n_far_unresolved = F.far_unresolved;
        o->far_pairs = (long long)F.far_pairs_total; o->far_passes = c->far_passes;
        if (c->far_error == 2) {            // one element's candidates do not fit a chunk (a third of max_pairs)
            S.status |= DC_STATUS_PAIR_OVERFLOW;
            S.n_pairs = 6ull * (F.far_want + 1ull) + 16ull;
        }
        float ms;
        if (cudaEventElapsedTime(&ms, c->ev[11], c->ev[12]) == cudaSuccess) o->ms_far = ms;
    }
    o->n_elem = c->n_elem; o->n_face = c->n_face;
    o->n_active = S.n_active; o->n_box_tests = (long long)S.c_box_tests;
    o->n_pairs = (long long)S.n_pairs > c->max_pairs ? c->max_pairs : (long long)S.n_pairs;
    o->pairs_needed = (long long)S.n_pairs;
    o->n_bnb_nodes = (long long)S.c_bnb_nodes; o->n_newton = (long long)S.c_newton;
    o->n_newton_iters = (long long)S.c_newton_iters; o->n_newton_fail = (long long)S.c_newton_fail;
    o->n_depth_exceeded = (long long)S.c_depth_exceeded;
    o->n_cut = (long long)S.c_cut; o->n_hole = (long long)S.c_hole; o->n_normal = (long long)S.c_normal;
    o->n_ambiguous = (long long)S.c_ambiguous; o->n_sign_ambiguous = (long long)S.c_sign_ambiguous;
    o->n_seedless_components = S.n_seedless; o->n_fill_conflicts = (long long)S.c_fill_conflicts;
    o->queue_peak = (long long)S.c_queue_peak;
    o->n_root_nodes = S.qn[0]; o->band_needed = S.n_band;
    for (int i = 0; i < DC_NQN; ++i) { if (S.qn[i] > o->queue_needed) o->queue_needed = S.qn[i]; if (S.nn[i] > o->queue_needed) o->queue_needed = S.nn[i]; }
    if (far)        // (the last pass of the far pass: on DC_STATUS_QUEUE_OVERFLOW, what its largest queue wanted)
        for (int i = 0; i < DC_NQN; ++i) {
            if (c->S_host->qn[i] > o->queue_needed) o->queue_needed = c->S_host->qn[i];
            if (c->S_host->nn[i] > o->queue_needed) o->queue_needed = c->S_host->nn[i];
        }
    o->l_ref = S.l_ref; o->tau_cut = S.tau; o->d_band = S.d_band;
    o->status = S.status;
    o->n_launches = (c->have_surface ? c->launches_surface : 0) + (c->have_cut ? c->launches_classify : 0);
    if (c->have_cut && !c->last_was_graph) {
        float ms;
        if (cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]) == cudaSuccess) o->ms_stage[1] = ms;
        if (cudaEventElapsedTime(&ms, c->ev[1], c->ev[2]) == cudaSuccess) o->ms_stage[2] = ms;
        if (cudaEventElapsedTime(&ms, c->ev[2], c->ev[3]) == cudaSuccess) o->ms_stage[3] = ms;
        if (cudaEventElapsedTime(&ms, c->ev[3], c->ev[4]) == cudaSuccess) o->ms_stage[4] = ms;
        if (cudaEventElapsedTime(&ms, c->ev[0], c->ev[4]) == cudaSuccess) o->ms_stage[5] = ms;
        if (cudaEventElapsedTime(&ms, c->ev[5], c->ev[6]) == cudaSuccess) o->ms_stage[7] = ms;
        if (cudaEventElapsedTime(&ms, c->ev[7], c->ev[10]) == cudaSuccess) { o->ms_stage[7] += ms; o->ms_kernel[1] = ms; }
        if (cudaEventElapsedTime(&ms, c->ev[2], c->ev[7]) == cudaSuccess) o->ms_kernel[0] = ms;
        if (cudaEventElapsedTime(&ms, c->ev[10], c->evk[0]) == cudaSuccess) o->ms_kernel[2] = ms;
        if (cudaEventElapsedTime(&ms, c->evk[0], c->ev[5]) == cudaSuccess) o->ms_kernel[3] = ms;
        if (cudaEventElapsedTime(&ms, c->ev[5], c->evk[1]) == cudaSuccess) o->ms_kernel[4] = ms;
        if (cudaEventElapsedTime(&ms, c->evk[1], c->evk[2]) == cudaSuccess) o->ms_kernel[5] = ms;
        if (cudaEventElapsedTime(&ms, c->evk[2], c->ev[6]) == cudaSuccess) o->ms_kernel[6] = ms;
        if (cudaEventElapsedTime(&ms, c->ev[6], c->ev[3]) == cudaSuccess) o->ms_kernel[7] = ms;
        // (ms_stage[7]: every k_np_solve launch = seeds + leaf passes + overflow rounds; the compaction pass is not in it)
        o->ms_stage[7] = o->ms_kernel[1] + o->ms_kernel[5] + o->ms_kernel[6];
    }
    if (c->have_surface && !c->last_was_graph) {
        float ms;
        if (cudaEventElapsedTime(&ms, c->ev[8], c->ev[9]) == cudaSuccess) { o->ms_stage[0] = ms; o->ms_stage[6] = ms; }
    }
    (void)cudaGetLastError();
    if (S.status & (DC_STATUS_PAIR_OVERFLOW | DC_STATUS_QUEUE_OVERFLOW | DC_STATUS_BAND_OVERFLOW)) return DC_ERR_WORKSPACE;
    if (S.status & (DC_STATUS_FILL_CONFLICT | DC_STATUS_SEEDLESS_OVERFLOW)) return DC_ERR_RESULT;
    if (S.status & DC_STATUS_SURFACE_SMALL) return DC_ERR_UNSUPPORTED;
    return DC_OK;
}

extern "C" void dc_destroy(dc_ctx *c)
{
    if (!c) return;
    cudaSetDevice(c->device);
    if (c->last_stream || true) cudaStreamSynchronize(c->last_stream);
    for (int i = 0; i < 14; ++i) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    for (int i = 0; i < 10; ++i) if (c->evk[i]) cudaEventDestroy(c->evk[i]);
    if (c->side) cudaStreamDestroy(c->side);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->S_host) cudaFreeHost(c->S_host);
    if (c->S_band_host) cudaFreeHost(c->S_band_host);
    for (int i = 0; i < c->n_graphs; ++i) if (c->graphs[i].exec) cudaGraphExecDestroy(c->graphs[i].exec);
    delete c;
}

extern "C" const char *dc_error_string(int code)
{
    switch (code) {
    case DC_OK: return "ok";
    case DC_ERR_ARG: return "bad argument";
    case DC_ERR_WORKSPACE: return "workspace too small or device-side list overflow";
    case DC_ERR_UNSUPPORTED: return "unsupported device (libdc needs an sm_100 GPU) or input (cutting surface smaller than an element)";
    case DC_ERR_CUDA: return "CUDA runtime error";
    case DC_ERR_STATE: return "call order error";
    case DC_ERR_RESULT: return "device-side consistency check failed (fill conflict or too many seedless components): results not to be trusted";
    default: return "unknown error";
    }
}

extern "C" double dc_measure_fp64_tflops(int device, int iters)
{
    if (cudaSetDevice(device) != cudaSuccess) return -1.0;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return -1.0;
    const int blocks = prop.multiProcessorCount * 8, threads = 256;
    double *out = nullptr;
    if (cudaMalloc(&out, (size_t)blocks * threads * 8) != cudaSuccess) return -1.0;
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    if (iters <= 0) iters = 2000;
    k_dfma_peak<<<blocks, threads>>>(out, iters / 10 + 1, 1.0000001, 1e-9);
    cudaDeviceSynchronize();
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(a);
        k_dfma_peak<<<blocks, threads>>>(out, iters, 1.0000001, 1e-9);
        cudaEventRecord(b);
        cudaEventSynchronize(b);
        float ms = 0; cudaEventElapsedTime(&ms, a, b);
        const double flop = 2.0 * 8 * 16 * (double)iters * blocks * threads;
        const double tf = flop / (ms * 1e-3) / 1e12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(out);
    if (cudaGetLastError() != cudaSuccess) return -1.0;
    return best;
}

#include "dc_blank.cuh"

// ---- donor search (dc_donor.cuh)
extern "C" size_t dc_adt_bytes(long long n_elem) { return n_elem > 0 ? (size_t)n_elem * sizeof(AdtNode) : 0; }
extern "C" size_t dc_donor_scratch_bytes(long long n_pts) { return n_pts > 0 ? (size_t)n_pts * (DC_DONOR_CAND + 1) * 4 : 0; }

extern "C" int dc_adt_build(dc_ctx *c, void *adt_dev, size_t adt_bytes, void *stream)
{
    if (!c || !adt_dev) return DC_ERR_ARG;
    if (adt_bytes < dc_adt_bytes(c->n_elem) || ((uintptr_t)adt_dev & 15) != 0) return DC_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(c->device));
    CK(cudaStreamSynchronize(st));
    const long long n = c->n_elem;
    std::vector<double> soa((size_t)n * 6), box((size_t)n * 6);
    CK(cudaMemcpy(soa.data(), c->ebox, (size_t)n * 6 * 8, cudaMemcpyDeviceToHost));
    for (long long e = 0; e < n; ++e) for (int k = 0; k < 6; ++k) box[(size_t)e * 6 + k] = soa[(size_t)k * n + e];
    std::vector<int> ids((size_t)n);
    for (long long e = 0; e < n; ++e) ids[(size_t)e] = (int)e;
    std::vector<AdtNode> nodes((size_t)n);
    dcadt::Builder B; B.box = box.data(); B.nodes = nodes.data(); B.next = 0;
    B.build(ids.data(), 0, (int)n, 0);
    CK(cudaMemcpy(adt_dev, nodes.data(), (size_t)n * sizeof(AdtNode), cudaMemcpyHostToDevice));
    c->adt = (const AdtNode *)adt_dev; c->adt_nodes = (int)n;
    return DC_OK;
}

extern "C" int dc_find_donors(dc_ctx *c, long long n_pts, const double *pts_dev, const double *rot9_host, const double *off3_host,
                              int *donor_dev, double *ref_dev, void *scratch_dev, size_t scratch_bytes, void *stream)
{
    if (!c || !pts_dev || !donor_dev || !ref_dev || !scratch_dev || n_pts < 0) return DC_ERR_ARG;
    if (!c->adt) return DC_ERR_STATE;
    if (scratch_bytes < dc_donor_scratch_bytes(n_pts)) return DC_ERR_WORKSPACE;
    if (n_pts == 0) return DC_OK;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(c->device));
    const double I[9] = { 1, 0, 0, 0, 1, 0, 0, 0, 1 }, Z[3] = { 0, 0, 0 };
    const double *R = rot9_host ? rot9_host : I, *o = off3_host ? off3_host : Z;
    int *cand = (int *)scratch_dev, *cand_n = cand + (size_t)n_pts * DC_DONOR_CAND;
    k_adt_search<<<nblk(n_pts, 128), 128, 0, st>>>(c->adt, c->adt_nodes, c->ebox, c->n_elem, pts_dev, n_pts, R[0], R[1], R[2], R[3], R[4],
                                                   R[5], R[6], R[7], R[8], o[0], o[1], o[2], 1e-12, cand, cand_n);
    k_donor_newton<<<nblk(n_pts, 128), 128, 0, st>>>(c->xyz, c->conn, c->ebox, c->n_elem, pts_dev, n_pts, R[0], R[1], R[2], R[3], R[4],
                                                     R[5], R[6], R[7], R[8], o[0], o[1], o[2], cand, cand_n, donor_dev, ref_dev);
    CK(cudaGetLastError());
    return DC_OK;
}

// ---- dc_find_donors_noalloc: the donor search for callers that cannot allocate (code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc).  Same two kernels as dc_find_donors; the candidate lists that call
// takes as caller-allocated scratch live here in ONE file-scope device array of fixed size: DC_NOALLOC_MAX_POINTS points x
// (DC_DONOR_CAND candidates + 1 count) x 4 bytes = 4 456 448 bytes, held by every GPU that loads the library until exit.
// In host code the array's name is only a stand-in for the symbol, not a device address: the address is asked for once
// per device (cudaGetSymbolAddress with that device current, return code checked) and handed to the kernels.
// Every call on a device shares the array: calls that overlap on the GPU (two streams) race; calls on one stream do not.
static __device__ __align__(256) int g_noalloc_donor_scratch[(size_t)DC_NOALLOC_MAX_POINTS * (DC_DONOR_CAND + 1)];

#define DC_NOALLOC_MAX_DEVICES 64
static std::mutex g_noalloc_mutex;
static int *g_noalloc_ptr[DC_NOALLOC_MAX_DEVICES];          // device address of the array on each device, once resolved

// set-up, once per device: the caller has made `device` current
static int noalloc_scratch_address(int device, int **out)
{
    if (device < 0 || device >= DC_NOALLOC_MAX_DEVICES) return DC_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_donor_scratch);
        if (e != cudaSuccess || !p) {
            fprintf(stderr, "libdc: cudaGetSymbolAddress(g_noalloc_donor_scratch) failed on device %d: %s\n", device, cudaGetErrorString(e));
            return DC_ERR_CUDA;
        }
        g_noalloc_ptr[device] = (int *)p;
    }
    *out = g_noalloc_ptr[device];
    return DC_OK;
}

extern "C" int dc_find_donors_noalloc(dc_ctx *c, long long n_pts, const double *pts_dev, const double *rot9_host, const double *off3_host,
                                      int *donor_dev, double *ref_dev, void *stream)
{
    if (!c || !pts_dev || !donor_dev || !ref_dev || n_pts < 0) return DC_ERR_ARG;
    if (!c->adt) return DC_ERR_STATE;
    if (n_pts > DC_NOALLOC_MAX_POINTS) {
        fprintf(stderr, "libdc: dc_find_donors_noalloc: %lld points exceed the built-in scratch of %d points; split the batch or call "
                        "dc_find_donors with scratch of your own\n", n_pts, DC_NOALLOC_MAX_POINTS);
        return DC_ERR_WORKSPACE;
    }
    if (n_pts == 0) return DC_OK;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(c->device));
    int *scratch = nullptr;
    { const int rc = noalloc_scratch_address(c->device, &scratch); if (rc) return rc; }
    const double I[9] = { 1, 0, 0, 0, 1, 0, 0, 0, 1 }, Z[3] = { 0, 0, 0 };
    const double *R = rot9_host ? rot9_host : I, *o = off3_host ? off3_host : Z;
    int *cand = scratch, *cand_n = cand + (size_t)n_pts * DC_DONOR_CAND;
    // The array keeps the last call's contents.  Nothing in it has to start at zero for the result (k_adt_search writes
    // cand_n[i] for every point, and cand[i][0 .. cand_n[i]) before k_donor_newton reads them), but the counts are cleared
    // all the same: a stale count must never be taken for this call's, whatever happens to the first kernel.
    CK(cudaMemsetAsync(cand_n, 0, (size_t)n_pts * 4, st));
    k_adt_search<<<nblk(n_pts, 128), 128, 0, st>>>(c->adt, c->adt_nodes, c->ebox, c->n_elem, pts_dev, n_pts, R[0], R[1], R[2], R[3], R[4],
                                                   R[5], R[6], R[7], R[8], o[0], o[1], o[2], 1e-12, cand, cand_n);
    k_donor_newton<<<nblk(n_pts, 128), 128, 0, st>>>(c->xyz, c->conn, c->ebox, c->n_elem, pts_dev, n_pts, R[0], R[1], R[2], R[3], R[4],
                                                     R[5], R[6], R[7], R[8], o[0], o[1], o[2], cand, cand_n, donor_dev, ref_dev);
    CK(cudaGetLastError());
    return DC_OK;
}

extern "C" int dc_version(void) { return 4; }

