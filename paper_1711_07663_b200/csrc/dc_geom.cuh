// dc_geom.cuh -- device-side patch mathematics of the narrow phase (S5), sm_100a.
//
// A biquadratic patch (9-node Lagrange quad, Eq. 1 L241 with K = 2) is held in the
// MONOMIAL basis  P(u,v) = sum_{i,j<=2} A[i+3j] u^i v^j,  (u,v) in [-1,1]^2, one 9-vector per
// coordinate, plus one constant K bounding its higher-order part.  A sub-patch is a dyadic
// sub-rectangle (centre (uc,vc), half-width h) of its root patch and is never re-centred: the
// branch-and-bound node (bound_node, below) evaluates the centre (an attained distance, hence an
// upper bound) and the range of the projections n.P, n.Q on the sub-rectangles (the lower bound)
// straight from the root coefficients; the projected Newton solve lives in dc_newton.cuh.
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

struct NodeOut {
    double dist_c, lb; bool leaf, splitP;
    double r[3], pu[3], pv[3], qs[3], qt[3];     // centre difference and first derivatives there (for the leaf's first step)
};

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
#pragma unroll
    for (int c = 0; c < 3; ++c) { o.r[c] = r[c]; o.pu[c] = pu[c]; o.pv[c] = pv[c]; o.qs[c] = qs[c]; o.qt[c] = qt[c]; }
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
