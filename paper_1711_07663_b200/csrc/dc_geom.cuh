// dc_geom.cuh -- device-side patch mathematics of the narrow phase (S5), sm_100a.
//
// A biquadratic patch (9-node Lagrange quad, Eq. 1 L241 with K = 2) is held in the
// MONOMIAL basis  P(u,v) = sum_{i,j<=2} A[i+3j] u^i v^j,  (u,v) in [-1,1]^2, one 9-vector per
// coordinate.  Restricting it to a dyadic sub-rectangle (centre (uc,vc), half-widths (hu,hv))
// and re-centring gives local coefficients C with  P = sum C[i+3j] a^i b^j, (a,b) in [-1,1]^2:
// this one representation yields the point at the centre (an attained distance, hence an upper
// bound), range bounds of any projection n.P (the lower bound of the branch and bound) and all
// derivatives the projected Newton solve needs (the two-patch generalisation of Eq. 3-5,
// L256-L270, with the paper's clamp to the reference box, L272-L278).
//
// No code is shared with oracle/ (which uses Bezier nets and triangle-triangle distances).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dcg {

// min / max of two finite doubles as one compare and a select (fmin / fmax expand to a NaN-aware sequence about
// twice as long; every value compared on the hot path is finite)
__host__ __device__ __forceinline__ double dmin2(double a, double b) { return a < b ? a : b; }
__host__ __device__ __forceinline__ double dmax2(double a, double b) { return a > b ? a : b; }

// ---------------------------------------------------------------------------------------------
// 1-D quadratic through nodes (-1, 0, +1): a0 + a1 t + a2 t^2
__device__ __forceinline__ void lag_to_mono(double x0, double x1, double x2,
                                            double &a0, double &a1, double &a2)
{
    a0 = x1;
    a1 = 0.5 * (x2 - x0);
    a2 = 0.5 * (x0 + x2) - x1;
}

// 9 Lagrange node values X[i+3j] (one coordinate) -> 9 monomial coefficients A[i+3j].
__device__ __forceinline__ void nodes_to_mono9(const double *X, double *A)
{
    double T[9];
#pragma unroll
    for (int j = 0; j < 3; ++j)
        lag_to_mono(X[0 + 3 * j], X[1 + 3 * j], X[2 + 3 * j], T[0 + 3 * j], T[1 + 3 * j], T[2 + 3 * j]);
#pragma unroll
    for (int i = 0; i < 3; ++i)
        lag_to_mono(T[i], T[i + 3], T[i + 6], A[i], A[i + 3], A[i + 6]);
}

// Re-centre one coordinate: A[9] on [-1,1]^2 -> C[9] on the sub-rectangle (uc,vc,hu,hv).
__device__ __forceinline__ void recentre9(const double *A, double uc, double vc, double hu, double hv,
                                          double *C)
{
    double R[9];
    const double hu2 = hu * hu, hv2 = hv * hv;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const double a0 = A[3 * j], a1 = A[3 * j + 1], a2 = A[3 * j + 2];
        R[3 * j]     = fma(uc, fma(uc, a2, a1), a0);
        R[3 * j + 1] = hu * fma(2.0 * uc, a2, a1);
        R[3 * j + 2] = hu2 * a2;
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const double r0 = R[i], r1 = R[i + 3], r2 = R[i + 6];
        C[i]     = fma(vc, fma(vc, r2, r1), r0);
        C[i + 3] = hv * fma(2.0 * vc, r2, r1);
        C[i + 6] = hv2 * r2;
    }
}

// value of one coordinate at (u,v)
__device__ __forceinline__ double eval9(const double *A, double u, double v)
{
    const double r0 = fma(u, fma(u, A[2], A[1]), A[0]);
    const double r1 = fma(u, fma(u, A[5], A[4]), A[3]);
    const double r2 = fma(u, fma(u, A[8], A[7]), A[6]);
    return fma(v, fma(v, r2, r1), r0);
}

// value and all derivatives up to second order of one coordinate at (a,b)
struct Jet { double p, pa, pb, paa, pab, pbb; };
__device__ __forceinline__ Jet jet9(const double *C, double a, double b)
{
    const double r0 = fma(a, fma(a, C[2], C[1]), C[0]);
    const double r1 = fma(a, fma(a, C[5], C[4]), C[3]);
    const double r2 = fma(a, fma(a, C[8], C[7]), C[6]);
    const double d0 = fma(2.0 * a, C[2], C[1]);
    const double d1 = fma(2.0 * a, C[5], C[4]);
    const double d2 = fma(2.0 * a, C[8], C[7]);
    Jet J;
    J.p   = fma(b, fma(b, r2, r1), r0);
    J.pb  = fma(2.0 * b, r2, r1);
    J.pbb = 2.0 * r2;
    J.pa  = fma(b, fma(b, d2, d1), d0);
    J.pab = fma(2.0 * b, d2, d1);
    J.paa = 2.0 * fma(b, fma(b, C[8], C[5]), C[2]);
    return J;
}

// ---------------------------------------------------------------------------------------------
// ordered-uint encoding of doubles for atomicMin/atomicMax
__device__ __forceinline__ unsigned long long enc_ord(double x)
{
    unsigned long long b = (unsigned long long)__double_as_longlong(x);
    return (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __host__ __forceinline__ double dec_ord(unsigned long long e)
{
    unsigned long long b = (e & 0x8000000000000000ull) ? (e & 0x7fffffffffffffffull) : ~e;
#ifdef __CUDA_ARCH__
    return __longlong_as_double((long long)b);
#else
    double d; memcpy(&d, &b, 8); return d;
#endif
}

// ---------------------------------------------------------------------------------------------
// Sub-pair bound.  Inputs: root monomial coefficients AP[27], AQ[27] laid out [coord][9]
// (coord-major), and the two dyadic sub-rectangles.  Outputs everything the branch and bound
// needs to decide prune / split / leaf.
struct NodeBound {
    double dist_c;   // |P_c - Q_c|: attained by real points -> valid upper bound
    double lb;       // slab lower bound of the distance over the sub-pair
    double s1P, s2P; // first-order size (max |C10|,|C01|) and higher-order radius of P's sub-patch
    double s1Q, s2Q;
};

// lower bound of  m(a,b) = sum_{(i,j)!=(0,0)} g[i+3j] a^i b^j  over [-1,1]^2  (g[0] ignored)
__device__ __forceinline__ double poly_lower(const double *g)
{
    return -fabs(g[1]) - fabs(g[3]) + dmin2(0.0, g[2]) + dmin2(0.0, g[6]) - fabs(g[4])
           - fabs(g[5]) - fabs(g[7]) + dmin2(0.0, g[8]);
}
__device__ __forceinline__ double poly_upper(const double *g)
{
    return fabs(g[1]) + fabs(g[3]) + dmax2(0.0, g[2]) + dmax2(0.0, g[6]) + fabs(g[4])
           + fabs(g[5]) + fabs(g[7]) + dmax2(0.0, g[8]);
}

template <typename LoadP, typename LoadQ>
__device__ __forceinline__ NodeBound bound_subpair(LoadP ldP, LoadQ ldQ,
                                                   double uc, double vc, double hP,
                                                   double sc, double tc, double hQ)
{
    // pass 1: centres -> r, n
    double r[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double A[9];
#pragma unroll
        for (int m = 0; m < 9; ++m) A[m] = ldP(c * 9 + m);
        const double p = eval9(A, uc, vc);
#pragma unroll
        for (int m = 0; m < 9; ++m) A[m] = ldQ(c * 9 + m);
        r[c] = p - eval9(A, sc, tc);
    }
    NodeBound nb;
    const double d2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
    nb.dist_c = sqrt(d2);
    const double inv = nb.dist_c > 0.0 ? 1.0 / nb.dist_c : 0.0;
    const double n[3] = { r[0] * inv, r[1] * inv, r[2] * inv };
    // pass 2: projections of the re-centred coefficients on n, and coefficient norms
    double gP[9], gQ[9], nP[9], nQ[9];
#pragma unroll
    for (int m = 0; m < 9; ++m) { gP[m] = gQ[m] = nP[m] = nQ[m] = 0.0; }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double A[9], C[9];
#pragma unroll
        for (int m = 0; m < 9; ++m) A[m] = ldP(c * 9 + m);
        recentre9(A, uc, vc, hP, hP, C);
#pragma unroll
        for (int m = 1; m < 9; ++m) { gP[m] = fma(n[c], C[m], gP[m]); nP[m] = fma(C[m], C[m], nP[m]); }
#pragma unroll
        for (int m = 0; m < 9; ++m) A[m] = ldQ(c * 9 + m);
        recentre9(A, sc, tc, hQ, hQ, C);
#pragma unroll
        for (int m = 1; m < 9; ++m) { gQ[m] = fma(n[c], C[m], gQ[m]); nQ[m] = fma(C[m], C[m], nQ[m]); }
    }
    nb.lb = nb.dist_c + poly_lower(gP) - poly_upper(gQ);
    nb.s1P = sqrt(dmax2(nP[1], nP[3]));
    nb.s1Q = sqrt(dmax2(nQ[1], nQ[3]));
    nb.s2P = sqrt(nP[2]) + sqrt(nP[6]) + sqrt(nP[4]) + sqrt(nP[5]) + sqrt(nP[7]) + sqrt(nP[8]);
    nb.s2Q = sqrt(nQ[2]) + sqrt(nQ[6]) + sqrt(nQ[4]) + sqrt(nQ[5]) + sqrt(nQ[7]) + sqrt(nQ[8]);
    return nb;
}

// ---------------------------------------------------------------------------------------------
// Projected Newton on f(a,b,c,d) = 1/2 |P(a,b) - Q(c,d)|^2 over the LOCAL box [-1,1]^4 of a leaf
// (the leaf's own sub-rectangles).  CP, CQ: local coefficients [coord][9] (27 each).
struct NewtonOut {
    double dist;      // attained distance at the final iterate
    double cosv;      // (r . n)/(|r||n|), n = Q_c x Q_d (same orientation as Q_s x Q_t)
    int iters;
    int converged;    // 1: predicted decrease below tolerance; 0: cap hit / stalled
};

__device__ __forceinline__ double f_only(const double *CP, const double *CQ, const double *x)
{
    double f = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double r = eval9(CP + 9 * c, x[0], x[1]) - eval9(CQ + 9 * c, x[2], x[3]);
        f = fma(r, r, f);
    }
    return 0.5 * f;
}

// Cholesky solve of the 4x4 SPD system H p = -g (H given by its upper triangle h[10] in row
// order 00 01 02 03 11 12 13 22 23 33).  Returns false if not positive definite.
__device__ __forceinline__ bool chol4_solve(const double *h, const double *g, double *p)
{
    double l00, l10, l20, l30, l11, l21, l31, l22, l32, l33;
    if (!(h[0] > 0.0)) return false;
    l00 = sqrt(h[0]); const double i00 = 1.0 / l00;
    l10 = h[1] * i00; l20 = h[2] * i00; l30 = h[3] * i00;
    double t = h[4] - l10 * l10; if (!(t > 0.0)) return false;
    l11 = sqrt(t); const double i11 = 1.0 / l11;
    l21 = (h[5] - l20 * l10) * i11; l31 = (h[6] - l30 * l10) * i11;
    t = h[7] - l20 * l20 - l21 * l21; if (!(t > 0.0)) return false;
    l22 = sqrt(t); const double i22 = 1.0 / l22;
    l32 = (h[8] - l30 * l20 - l31 * l21) * i22;
    t = h[9] - l30 * l30 - l31 * l31 - l32 * l32; if (!(t > 0.0)) return false;
    l33 = sqrt(t); const double i33 = 1.0 / l33;
    // forward: L y = -g
    const double y0 = -g[0] * i00;
    const double y1 = (-g[1] - l10 * y0) * i11;
    const double y2 = (-g[2] - l20 * y0 - l21 * y1) * i22;
    const double y3 = (-g[3] - l30 * y0 - l31 * y1 - l32 * y2) * i33;
    // backward: L^T p = y
    p[3] = y3 * i33;
    p[2] = (y2 - l32 * p[3]) * i22;
    p[1] = (y1 - l21 * p[2] - l31 * p[3]) * i11;
    p[0] = (y0 - l10 * p[1] - l20 * p[2] - l30 * p[3]) * i00;
    return true;
}

__device__ __forceinline__ double clamp1(double x) { return dmin2(1.0, dmax2(-1.0, x)); }

__device__ inline NewtonOut newton_leaf(const double *CP, const double *CQ, double tol_d,
                                        double tau_exit, int max_iter)
{
    double x[4] = { 0.0, 0.0, 0.0, 0.0 };
    NewtonOut out; out.iters = 0; out.converged = 0;
    double f = 0.0, r[3], Qc[3], Qd[3];
    for (int it = 0; it < max_iter; ++it) {
        out.iters = it + 1;
        // jets
        double Pa[3], Pb[3], Paa[3], Pab[3], Pbb[3], Qcc[3], Qcd[3], Qdd[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const Jet JP = jet9(CP + 9 * c, x[0], x[1]);
            const Jet JQ = jet9(CQ + 9 * c, x[2], x[3]);
            r[c] = JP.p - JQ.p;
            Pa[c] = JP.pa; Pb[c] = JP.pb; Paa[c] = JP.paa; Pab[c] = JP.pab; Pbb[c] = JP.pbb;
            Qc[c] = JQ.pa; Qd[c] = JQ.pb; Qcc[c] = JQ.paa; Qcd[c] = JQ.pab; Qdd[c] = JQ.pbb;
        }
#define DOT(A, B) (A[0] * B[0] + A[1] * B[1] + A[2] * B[2])
        f = 0.5 * DOT(r, r);
        const double dist = sqrt(2.0 * f);
        if (dist <= tau_exit) { out.converged = 1; break; }
        double g[4] = { DOT(r, Pa), DOT(r, Pb), -DOT(r, Qc), -DOT(r, Qd) };
        double h[10];
        h[0] = DOT(Pa, Pa) + DOT(r, Paa);
        h[1] = DOT(Pa, Pb) + DOT(r, Pab);
        h[2] = -DOT(Pa, Qc);
        h[3] = -DOT(Pa, Qd);
        h[4] = DOT(Pb, Pb) + DOT(r, Pbb);
        h[5] = -DOT(Pb, Qc);
        h[6] = -DOT(Pb, Qd);
        h[7] = DOT(Qc, Qc) - DOT(r, Qcc);
        h[8] = DOT(Qc, Qd) - DOT(r, Qcd);
        h[9] = DOT(Qd, Qd) - DOT(r, Qdd);
        // active set: variables at a bound whose gradient pushes outward are held (L272-L278)
        bool fixed[4];
#pragma unroll
        for (int i = 0; i < 4; ++i)
            fixed[i] = (x[i] <= -1.0 && g[i] > 0.0) || (x[i] >= 1.0 && g[i] < 0.0);
        const int di[4] = { 0, 4, 7, 9 };
        // decouple held variables
        if (fixed[0]) { h[1] = h[2] = h[3] = 0.0; h[0] = 1.0; g[0] = 0.0; }
        if (fixed[1]) { h[1] = h[5] = h[6] = 0.0; h[4] = 1.0; g[1] = 0.0; }
        if (fixed[2]) { h[2] = h[5] = h[8] = 0.0; h[7] = 1.0; g[2] = 0.0; }
        if (fixed[3]) { h[3] = h[6] = h[8] = 0.0; h[9] = 1.0; g[3] = 0.0; }
        const double gg = g[0] * g[0] + g[1] * g[1] + g[2] * g[2] + g[3] * g[3];
        if (gg == 0.0) { out.converged = 1; break; }
        // Levenberg damping only if the (reduced) Hessian is not positive definite
        double tr = 0.0;
#pragma unroll
        for (int i = 0; i < 4; ++i) if (!fixed[i]) tr += fabs(h[di[i]]);
        double p[4];
        double lam = 0.0;
        bool ok = false;
        for (int tries = 0; tries < 6 && !ok; ++tries) {
            double hd[10];
#pragma unroll
            for (int i = 0; i < 10; ++i) hd[i] = h[i];
#pragma unroll
            for (int i = 0; i < 4; ++i) if (!fixed[i]) hd[di[i]] += lam;
            ok = chol4_solve(hd, g, p);
            lam = (lam == 0.0) ? 1e-6 * tr + 1e-300 : lam * 100.0;
        }
        if (!ok) { // steepest descent fallback, scaled by the trace
            const double s = tr > 0.0 ? 1.0 / tr : 1.0;
#pragma unroll
            for (int i = 0; i < 4; ++i) p[i] = -g[i] * s;
        }
        const double pred = -0.5 * (g[0] * p[0] + g[1] * p[1] + g[2] * p[2] + g[3] * p[3]);
        // projected step with backtracking on f
        double xn[4], fn = f, alpha = 1.0;
        bool dec = false;
        for (int ls = 0; ls < 6; ++ls) {
#pragma unroll
            for (int i = 0; i < 4; ++i) xn[i] = clamp1(fma(alpha, p[i], x[i]));
            fn = f_only(CP, CQ, xn);
            if (fn <= f) { dec = true; break; }
            alpha *= 0.25;
        }
        double step = 0.0;
        if (dec) {
#pragma unroll
            for (int i = 0; i < 4; ++i) { step = dmax2(step, fabs(xn[i] - x[i])); x[i] = xn[i]; }
            f = fn;
        }
        // converged when the predicted decrease of the DISTANCE is below tol_d
        if (pred <= tol_d * dmax2(dist, tol_d)) { out.converged = 1; break; }
        if (!dec || step < 1e-15) { break; }
    }
    // final evaluation at x: distance and the sign cosine
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const Jet JP = jet9(CP + 9 * c, x[0], x[1]);
        const Jet JQ = jet9(CQ + 9 * c, x[2], x[3]);
        r[c] = JP.p - JQ.p; Qc[c] = JQ.pa; Qd[c] = JQ.pb;
    }
    const double nx = Qc[1] * Qd[2] - Qc[2] * Qd[1];
    const double ny = Qc[2] * Qd[0] - Qc[0] * Qd[2];
    const double nz = Qc[0] * Qd[1] - Qc[1] * Qd[0];
    const double rr = DOT(r, r), nn = nx * nx + ny * ny + nz * nz;
    out.dist = sqrt(rr);
    const double den = sqrt(rr * nn);
    out.cosv = den > 0.0 ? (r[0] * nx + r[1] * ny + r[2] * nz) / den : 0.0;
#undef DOT
    return out;
}

// 8-bit code of the sign cosine: bit 7 = negative, bits 0-6 = round(|cos| * 127)
__device__ __forceinline__ unsigned cos_code(double cosv)
{
    const double a = dmin2(1.0, fabs(cosv));
    unsigned m = (unsigned)(a * 127.0 + 0.5);
    return (cosv < 0.0 ? 0x80u : 0u) | m;
}

} // namespace dcg

// =============================================================================================
// Wavefront narrow phase (dc_narrow.cuh): one branch-and-bound node, sqrt-free.
//
// A node is a pair of dyadic sub-rectangles (centre, half-width) of a root patch pair given by
// root monomial coefficients AP, AQ ([coord][9]) and the root constants KP, KQ (see
// higher_order_const).  It returns
//   dist_c : |P(centre) - Q(centre)|, attained by real points => an upper bound of the minimum;
//   lb     : a lower bound of the distance over the node: with n = r/|r| (r = centre difference)
//            min |P - Q| >= n.(P - Q) >= dist_c + min n.(P - Pc) - max n.(Q - Qc), the ranges of
//            the two SCALAR biquadratics n.P, n.Q re-centred on the node (project first, re-centre
//            the 8 non-constant scalar coefficients after: 3x cheaper than re-centring vectors);
//   leaf / splitP : the subdivision rule.  s1^2 = h^2 max(|P_u|^2,|P_v|^2) at the centre is the
//            squared first-order size, s2 = h^2 K bounds the sum of the norms of the node's six
//            higher-order coefficients.  leaf <=> max(kP,kQ) max(s1P,s1Q) <= theta, k = s2/s1^2,
//            tested in squared form (no sqrt, no divide).
namespace dcg {

// Upper bound K of (sum of the norms of the 6 higher-order re-centred coefficients)/h^2 over every
// sub-rectangle of [-1,1]^2 (|uc|,|vc| <= 1, h <= 1), from the root coefficients A [coord][9]:
//   |C20| <= h^2(|A20|+|A21|+|A22|), |C02| <= h^2(|A02|+|A12|+|A22|),
//   |C11| <= h^2(|A11|+2|A21|+2|A12|+4|A22|), |C21| <= h^3(|A21|+2|A22|), |C12| <= h^3(|A12|+2|A22|),
//   |C22| <= h^4 |A22|      (index m = i + 3 j for u^i v^j).
__device__ __forceinline__ double higher_order_const(const double *A /*[27]*/)
{
    double nrm[9];
#pragma unroll
    for (int m = 0; m < 9; ++m) nrm[m] = sqrt(A[m] * A[m] + A[9 + m] * A[9 + m] + A[18 + m] * A[18 + m]);
    const double a20 = nrm[2], a02 = nrm[6], a11 = nrm[4], a21 = nrm[5], a12 = nrm[7], a22 = nrm[8];
    return (a20 + a21 + a22) + (a02 + a12 + a22) + (a11 + 2.0 * a21 + 2.0 * a12 + 4.0 * a22)
           + (a21 + 2.0 * a22) + (a12 + 2.0 * a22) + a22;
}

// value and first derivatives of one coordinate at (u,v)
__device__ __forceinline__ void eval_d1(const double *A, double u, double v, double &p, double &pu, double &pv)
{
    const double u2 = u + u, v2 = v + v;
    const double r0 = fma(u, fma(u, A[2], A[1]), A[0]);
    const double r1 = fma(u, fma(u, A[5], A[4]), A[3]);
    const double r2 = fma(u, fma(u, A[8], A[7]), A[6]);
    const double d0 = fma(u2, A[2], A[1]);
    const double d1 = fma(u2, A[5], A[4]);
    const double d2 = fma(u2, A[8], A[7]);
    p = fma(v, fma(v, r2, r1), r0);
    pv = fma(v2, r2, r1);
    pu = fma(v, fma(v, d2, d1), d0);
}

// range [lo, hi] of the non-constant part of the scalar biquadratic g (g[0] ignored) over the
// sub-rectangle (uc, vc, h): re-centre, then bound term by term.
__device__ __forceinline__ void scalar_range(const double *g, double uc, double vc, double h, double &lo, double &hi)
{
    const double h2 = h * h, uc2 = uc + uc, vc2 = vc + vc;
    // rows j = 0,1,2 (powers of v): R_j0 (only j = 1,2 feed non-constant terms), R_j1, R_j2
    const double R01 = h * fma(uc2, g[2], g[1]), R02 = h2 * g[2];
    const double R10 = fma(uc, fma(uc, g[5], g[4]), g[3]), R11 = h * fma(uc2, g[5], g[4]), R12 = h2 * g[5];
    const double R20 = fma(uc, fma(uc, g[8], g[7]), g[6]), R21 = h * fma(uc2, g[8], g[7]), R22 = h2 * g[8];
    const double c1 = fma(vc, fma(vc, R21, R11), R01);       // u
    const double c2 = fma(vc, fma(vc, R22, R12), R02);       // u^2
    const double c3 = h * fma(vc2, R20, R10);                // v
    const double c4 = h * fma(vc2, R21, R11);                // u v
    const double c5 = h * fma(vc2, R22, R12);                // u^2 v
    const double c6 = h2 * R20, c7 = h2 * R21, c8 = h2 * R22; // v^2, u v^2, u^2 v^2
    const double odd = fabs(c1) + fabs(c3) + fabs(c4) + fabs(c5) + fabs(c7);
    lo = dmin2(0.0, c2) + dmin2(0.0, c6) + dmin2(0.0, c8) - odd;
    hi = dmax2(0.0, c2) + dmax2(0.0, c6) + dmax2(0.0, c8) + odd;
}

struct NodeOut { double dist_c, lb; bool leaf, splitP; };

__device__ __forceinline__ NodeOut bound_node(const double *AP, const double *AQ, double KP, double KQ,
                                              double uc, double vc, double hP, double sc, double tc, double hQ,
                                              double theta2)
{
    double r[3], pu[3], pv[3], qs[3], qt[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double p, q;
        eval_d1(AP + 9 * c, uc, vc, p, pu[c], pv[c]);
        eval_d1(AQ + 9 * c, sc, tc, q, qs[c], qt[c]);
        r[c] = p - q;
    }
    NodeOut o;
    const double d2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
    const double inv = d2 > 0.0 ? rsqrt(d2) : 0.0;
    o.dist_c = d2 * inv;
    const double n0 = r[0] * inv, n1 = r[1] * inv, n2 = r[2] * inv;
    double gP[9], gQ[9];
#pragma unroll
    for (int m = 1; m < 9; ++m) {
        gP[m] = fma(n2, AP[18 + m], fma(n1, AP[9 + m], n0 * AP[m]));
        gQ[m] = fma(n2, AQ[18 + m], fma(n1, AQ[9 + m], n0 * AQ[m]));
    }
    double loP, hiP, loQ, hiQ;
    scalar_range(gP, uc, vc, hP, loP, hiP);
    scalar_range(gQ, sc, tc, hQ, loQ, hiQ);
    o.lb = o.dist_c + loP - hiQ;
    // subdivision rule (squared form)
    const double hP2 = hP * hP, hQ2 = hQ * hQ;
    const double S1P = hP2 * dmax2(pu[0] * pu[0] + pu[1] * pu[1] + pu[2] * pu[2], pv[0] * pv[0] + pv[1] * pv[1] + pv[2] * pv[2]);
    const double S1Q = hQ2 * dmax2(qs[0] * qs[0] + qs[1] * qs[1] + qs[2] * qs[2], qt[0] * qt[0] + qt[1] * qt[1] + qt[2] * qt[2]);
    const double s2P = hP2 * KP, s2Q = hQ2 * KQ;
    const double M = dmax2(S1P, S1Q);
    const bool okP = !(S1P > 0.0) || s2P * s2P * M <= theta2 * S1P * S1P;
    const bool okQ = !(S1Q > 0.0) || s2Q * s2Q * M <= theta2 * S1Q * S1Q;
    o.leaf = okP && okQ;
    o.splitP = S1P >= S1Q;
    return o;
}

} // namespace dcg
