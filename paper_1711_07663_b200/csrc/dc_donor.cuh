// dc_donor.cuh -- donor search for receptor points (PAPER.md 4.3 L229-L278; SURVEY.md 8(f) "(later)"): the paper's OTHER
// GPU algorithm, a different path from the direct cut, built on the same context (it needs the element boxes of S2).
//
//   dc_adt_build   host  : alternating digital tree over the element boxes, built ONCE on the CPU ("the ADT can be
//                          constructed once during preprocessing on the CPU and copied onto the GPU", L233) and valid
//                          under rigid motion of the grid: queries are rotated / shifted into the grid's frame instead.
//                          Balanced by construction (median splits, L247): a stack of (height + 1) entries suffices.
//   k_adt_search   thread / point : stack-based depth-first traversal with a fixed-size local LIFO array (L241-L247);
//                          an element whose box holds the point is APPENDED to the point's candidate list -- the
//                          work-intensive containment check is not done at the tree node (L247, against divergence)
//   k_donor_newton thread / point : Newton iterations on the isoparametric map of each candidate (Eq. 1-5:
//                          Delta = x_p - x(X_n), X_{n+1} = X_n + J^-1 Delta), X limited to a small tolerance around
//                          [-1,1]^3 (L272-L278: outside the element the iteration stalls on the boundary and cannot
//                          converge), at most 10 iterations (L272); the first candidate that converges is the donor.
#pragma once

#define DC_DONOR_CAND 16            /* candidate elements kept per point (boxes holding the point) */
#define DC_ADT_STACK 40             /* LIFO depth: height of a balanced tree of 2^39 nodes */
#define DC_DONOR_MAXIT 10           /* L272 */

struct __align__(16) AdtNode { double split; int elem, left, right, pad; };   // dimension = depth mod 6 (implicit)

// ------------------------------------------------------------------------------------------ host: build
namespace dcadt {
struct Builder {
    const double *box;      // [n][6] min xyz, max xyz
    AdtNode *nodes;
    int next;
    // median of ids[lo, hi) along dimension d becomes the node; returns its index
    int build(int *ids, int lo, int hi, int depth)
    {
        if (lo >= hi) return -1;
        const int d = depth % 6, mid = lo + (hi - lo) / 2;
        const double *B = box;
        std::nth_element(ids + lo, ids + mid, ids + hi, [B, d](int a, int b) {
            const double xa = B[(size_t)a * 6 + d], xb = B[(size_t)b * 6 + d];
            return xa < xb || (xa == xb && a < b);
        });
        const int me = next++;
        nodes[me].elem = ids[mid]; nodes[me].split = box[(size_t)ids[mid] * 6 + d]; nodes[me].pad = 0;
        const int l = build(ids, lo, mid, depth + 1);
        const int r = build(ids, mid + 1, hi, depth + 1);
        nodes[me].left = l; nodes[me].right = r;
        return me;
    }
};
} // namespace dcadt

// ------------------------------------------------------------------------------------------ device: search
// Elements whose box holds p: in the 6-D box space the query is  min_c <= p_c  (dimensions 0-2) and  max_c >= p_c
// (dimensions 3-5).  At a node splitting dimension d at value s: the left subtree has coordinate_d <= s, the right
// one >= s.  d < 3 (a minimum): the right subtree can only hold hits if s <= p_d.  d >= 3 (a maximum): the left
// subtree only if s >= p_(d-3).
__global__ void k_adt_search(const AdtNode *__restrict__ nodes, int n_nodes, const double *__restrict__ ebox, long long n_elem,
                             const double *__restrict__ pts, long long n_pts, double r00, double r01, double r02, double r10,
                             double r11, double r12, double r20, double r21, double r22, double ox, double oy, double oz,
                             double tol, int *__restrict__ cand, int *__restrict__ cand_n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pts) return;
    // the point in the grid's frame: x_grid = R^T (x - o)
    const double wx = pts[3 * i] - ox, wy = pts[3 * i + 1] - oy, wz = pts[3 * i + 2] - oz;
    const double p[3] = { r00 * wx + r10 * wy + r20 * wz, r01 * wx + r11 * wy + r21 * wz, r02 * wx + r12 * wy + r22 * wz };
    int stack[DC_ADT_STACK], depth[DC_ADT_STACK];
    int top = 0, nc = 0;
    if (n_nodes > 0) { stack[top] = 0; depth[top] = 0; ++top; }
    while (top > 0) {
        --top;
        const int node = stack[top], dep = depth[top];
        const AdtNode nd = nodes[node];
        const int e = nd.elem;
        bool in = true;
#pragma unroll
        for (int c = 0; c < 3; ++c)
            in = in && ebox[(size_t)c * n_elem + e] - tol <= p[c] && p[c] <= ebox[(size_t)(3 + c) * n_elem + e] + tol;
        if (in) { if (nc < DC_DONOR_CAND) cand[i * DC_DONOR_CAND + nc] = e; ++nc; }
        const int d = dep % 6;
        const bool go_left = nd.left >= 0 && (d < 3 || nd.split + tol >= p[d - 3]);
        const bool go_right = nd.right >= 0 && (d >= 3 || nd.split - tol <= p[d]);
        if (go_right && top < DC_ADT_STACK) { stack[top] = nd.right; depth[top] = dep + 1; ++top; }
        if (go_left && top < DC_ADT_STACK) { stack[top] = nd.left; depth[top] = dep + 1; ++top; }
    }
    cand_n[i] = nc;
}

// 1-D quadratic Lagrange basis on nodes (-1, 0, +1) and its derivative (Eq. 1 with K = 2)
__device__ __forceinline__ void lag3(double t, double *l, double *dl)
{
    l[0] = 0.5 * t * (t - 1.0); l[1] = 1.0 - t * t; l[2] = 0.5 * t * (t + 1.0);
    dl[0] = t - 0.5; dl[1] = -2.0 * t; dl[2] = t + 0.5;
}

__global__ void k_donor_newton(const double *__restrict__ xyz, const int *__restrict__ conn, const double *__restrict__ ebox,
                               long long n_elem, const double *__restrict__ pts, long long n_pts, double r00, double r01,
                               double r02, double r10, double r11, double r12, double r20, double r21, double r22, double ox,
                               double oy, double oz, const int *__restrict__ cand, const int *__restrict__ cand_n,
                               int *__restrict__ donor, double *__restrict__ ref)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pts) return;
    const double wx = pts[3 * i] - ox, wy = pts[3 * i + 1] - oy, wz = pts[3 * i + 2] - oz;
    const double p[3] = { r00 * wx + r10 * wy + r20 * wz, r01 * wx + r11 * wy + r21 * wz, r02 * wx + r12 * wy + r22 * wz };
    const int nc = min(cand_n[i], DC_DONOR_CAND);
    int found = -1;
    double X[3] = { 0.0, 0.0, 0.0 };
    for (int ci = 0; ci < nc && found < 0; ++ci) {
        const int e = cand[i * DC_DONOR_CAND + ci];
        // element size (box diagonal) scales the convergence tolerance
        double diag2 = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) { const double w = ebox[(size_t)(3 + c) * n_elem + e] - ebox[(size_t)c * n_elem + e]; diag2 += w * w; }
        const double tol2 = 1e-24 * diag2;             // |Delta| <= 1e-12 x element size
        double x[3] = { 0.0, 0.0, 0.0 };                // initial guess: the element's centre
        bool ok = false;
        for (int it = 0; it <= DC_DONOR_MAXIT; ++it) {
            double lx[3], dx[3], ly[3], dy[3], lz[3], dz[3];
            lag3(x[0], lx, dx); lag3(x[1], ly, dy); lag3(x[2], lz, dz);
            double f[3] = { 0.0, 0.0, 0.0 }, J[3][3] = { { 0, 0, 0 }, { 0, 0, 0 }, { 0, 0, 0 } };
            for (int k = 0; k < 3; ++k)
                for (int j = 0; j < 3; ++j)
#pragma unroll
                    for (int ii = 0; ii < 3; ++ii) {
                        const double *nd = xyz + (size_t)__ldg(conn + (size_t)e * 27 + ii + 3 * j + 9 * k) * 3;
                        const double N = lx[ii] * ly[j] * lz[k];
                        const double Nx = dx[ii] * ly[j] * lz[k], Ny = lx[ii] * dy[j] * lz[k], Nz = lx[ii] * ly[j] * dz[k];
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            const double v = __ldg(nd + c);
                            f[c] = fma(N, v, f[c]);
                            J[c][0] = fma(Nx, v, J[c][0]); J[c][1] = fma(Ny, v, J[c][1]); J[c][2] = fma(Nz, v, J[c][2]);
                        }
                    }
            const double D[3] = { p[0] - f[0], p[1] - f[1], p[2] - f[2] };                       // Eq. 3
            if (D[0] * D[0] + D[1] * D[1] + D[2] * D[2] <= tol2) { ok = true; break; }
            if (it == DC_DONOR_MAXIT) break;
            // Eq. 4: X += J^-1 Delta (cofactors)
            const double c00 = J[1][1] * J[2][2] - J[1][2] * J[2][1], c01 = J[1][2] * J[2][0] - J[1][0] * J[2][2], c02 = J[1][0] * J[2][1] - J[1][1] * J[2][0];
            const double det = J[0][0] * c00 + J[0][1] * c01 + J[0][2] * c02;
            if (det == 0.0) break;
            const double inv = 1.0 / det;
            const double s0 = (c00 * D[0] + (J[0][2] * J[2][1] - J[0][1] * J[2][2]) * D[1] + (J[0][1] * J[1][2] - J[0][2] * J[1][1]) * D[2]) * inv;
            const double s1 = (c01 * D[0] + (J[0][0] * J[2][2] - J[0][2] * J[2][0]) * D[1] + (J[0][2] * J[1][0] - J[0][0] * J[1][2]) * D[2]) * inv;
            const double s2 = (c02 * D[0] + (J[0][1] * J[2][0] - J[0][0] * J[2][1]) * D[1] + (J[0][0] * J[1][1] - J[0][1] * J[1][0]) * D[2]) * inv;
            // L272-L278: X is limited to a small tolerance around [-1,1]
            const double lim = 1.0 + 1e-10;
            x[0] = fmax(-lim, fmin(lim, x[0] + s0)); x[1] = fmax(-lim, fmin(lim, x[1] + s1)); x[2] = fmax(-lim, fmin(lim, x[2] + s2));
        }
        if (ok) { found = e; X[0] = x[0]; X[1] = x[1]; X[2] = x[2]; }
    }
    donor[i] = found;
    ref[3 * i] = X[0]; ref[3 * i + 1] = X[1]; ref[3 * i + 2] = X[2];
}
