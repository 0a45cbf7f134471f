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

// a work item of the narrow phase: a candidate pair, a boundary patch of its element, and a dyadic sub-rectangle of each
struct __align__(16) NItem { unsigned p, ak, w2, w3; };
// p : global pair index (face = pair_face[p], key slot = pair_key[p])
// ak: band index b (29 bits) | boundary patch k << 29
// w2: lP(4) | lQ(4)<<4 | iu(12)<<8 | iv(12)<<20
// w3: is(12) | it(12)<<12 | flags(8)<<24      flags bit0: seed solve (no re-split on failure)

namespace dcg {

// min / max of two finite doubles as one compare and a select (fmin / fmax expand to a NaN-aware sequence about
// twice as long; every value compared on the hot path is finite)
__device__ __forceinline__ double dmin2(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax2(double a, double b) { return a > b ? a : b; }

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
__device__ __forceinline__ double dec_ord(unsigned long long e)
{
    const unsigned long long b = (e & 0x8000000000000000ull) ? (e & 0x7fffffffffffffffull) : ~e;
    return __longlong_as_double((long long)b);
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
//   ub     : an ATTAINED distance (hence an upper bound of the minimum): the smaller of the centre distance and the
//            distance of the TRUE patches at x0, the closest pair of the node's first-order model
//            min |r_c + J a|, a in [-1,1]^4, J = [h P_u, h P_v, -h Q_s, -h Q_t] at the centre (a few sweeps of exact
//            coordinate minimisation with the clamp of L272-L278: the model is a box-constrained 4-variable least
//            squares problem whose J^T J is singular -- two patches can slide along each other -- so a plain
//            Gauss-Newton step lands anywhere; the sweeps only ever decrease |r|);
//   lb     : a lower bound of the distance over the node: for ANY unit n,
//            min |P - Q| >= n.(P_c - Q_c) + min n.(P - P_c) - max n.(Q - Q_c); with n = r(x0)/|r(x0)|, the direction
//            of the closest pair, the first-order part of the bound is tight (the centre direction loses 13 % of the
//            distance in the median on config 2, this one 1 %), and the ranges of the two SCALAR biquadratics n.P,
//            n.Q over the sub-rectangles come from their Bernstein coefficients (convex-hull property; exact for a
//            bilinear function, where bounding term by term is not: the twist u v is coupled to u and v);
//   x0     : that point in the node's local coordinates [-1,1]^4 (a leaf's solve starts there);
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
// (coefficients come through an accessor A(m), m = i + 3 j: registers, shared memory or a pointer)
template <class CF>
__device__ __forceinline__ void eval_d1(CF A, double u, double v, double &p, double &pu, double &pv)
{
    const double u2 = u + u, v2 = v + v;
    const double a0 = A(0), a1 = A(1), a2 = A(2), a3 = A(3), a4 = A(4), a5 = A(5), a6 = A(6), a7 = A(7), a8 = A(8);
    const double r0 = fma(u, fma(u, a2, a1), a0);
    const double r1 = fma(u, fma(u, a5, a4), a3);
    const double r2 = fma(u, fma(u, a8, a7), a6);
    const double d0 = fma(u2, a2, a1);
    const double d1 = fma(u2, a5, a4);
    const double d2 = fma(u2, a8, a7);
    p = fma(v, fma(v, r2, r1), r0);
    pv = fma(v2, r2, r1);
    pu = fma(v, fma(v, d2, d1), d0);
}

// value of one coordinate at (u,v)
template <class CF>
__device__ __forceinline__ double eval_d0(CF A, double u, double v)
{
    const double r0 = fma(u, fma(u, A(2), A(1)), A(0));
    const double r1 = fma(u, fma(u, A(5), A(4)), A(3));
    const double r2 = fma(u, fma(u, A(8), A(7)), A(6));
    return fma(v, fma(v, r2, r1), r0);
}

// Bernstein coefficients on [-1,1] of a0 + a1 t + a2 t^2
__device__ __forceinline__ void mono_to_bern(double a0, double a1, double a2, double &b0, double &b1, double &b2)
{
    const double s = a0 + a2;
    b0 = s - a1; b1 = a0 - a2; b2 = s + a1;
}

// range [lo, hi] of the non-constant part of the scalar biquadratic g (g[0] ignored) over the sub-rectangle
// (uc, vc, h): re-centre and scale to [-1,1]^2, convert to the Bernstein basis, take the smallest and the largest
// of the 9 coefficients (the function lies in their convex hull).
template <bool ROOT>
__device__ __forceinline__ void scalar_range(const double *g, double uc, double vc, double h, double &lo, double &hi)
{
    double c01, c02, c10, c11, c12, c20, c21, c22;
    if (ROOT) {
        // the whole patch (centre (0,0), half-width 1): the coefficients are already the local ones
        c01 = g[1]; c02 = g[2]; c10 = g[3]; c11 = g[4]; c12 = g[5]; c20 = g[6]; c21 = g[7]; c22 = g[8];
    } else {
        const double h2 = h * h, uc2 = uc + uc, vc2 = vc + vc;
        // rows j = 0,1,2 (powers of v) re-centred in u: R_j0, R_j1, R_j2
        const double R01 = h * fma(uc2, g[2], g[1]), R02 = h2 * g[2];
        const double R10 = fma(uc, fma(uc, g[5], g[4]), g[3]), R11 = h * fma(uc2, g[5], g[4]), R12 = h2 * g[5];
        const double R20 = fma(uc, fma(uc, g[8], g[7]), g[6]), R21 = h * fma(uc2, g[8], g[7]), R22 = h2 * g[8];
        // columns re-centred in v: c[j][i], constant term dropped
        c01 = fma(vc, fma(vc, R21, R11), R01); c02 = fma(vc, fma(vc, R22, R12), R02);
        c10 = h * fma(vc2, R20, R10); c11 = h * fma(vc2, R21, R11); c12 = h * fma(vc2, R22, R12);
        c20 = h2 * R20; c21 = h2 * R21; c22 = h2 * R22;
    }
    // Bernstein in u (rows), then in v (columns)
    double r0[3], r1[3], r2[3];
    mono_to_bern(0.0, c01, c02, r0[0], r0[1], r0[2]);
    mono_to_bern(c10, c11, c12, r1[0], r1[1], r1[2]);
    mono_to_bern(c20, c21, c22, r2[0], r2[1], r2[2]);
    lo = 0.0; hi = 0.0;                 // (the centre value, 0, is attained)
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        double b0, b1, b2;
        mono_to_bern(r0[i], r1[i], r2[i], b0, b1, b2);
        lo = dmin2(lo, dmin2(b0, dmin2(b1, b2)));
        hi = dmax2(hi, dmax2(b0, dmax2(b1, b2)));
    }
}

#ifndef DC_CD_SWEEPS
#define DC_CD_SWEEPS 4
#endif

// reciprocal of a positive normal-range double: hardware seed + two Newton steps (no slow path)
__device__ __forceinline__ double rcp_pos(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    y = fma(fma(-x, y, 1.0), y, y);
    y = fma(fma(-x, y, 1.0), y, y);
    return y;
}

// Closest pair of the first-order model min |r + J a|, a in [-1,1]^4, J = [h P_u, h P_v, -h Q_s, -h Q_t]: DC_CD_SWEEPS
// sweeps of exact coordinate minimisation with clamping (rho = r + J a only ever shrinks).  nrm[i] = |J_i|^2.
__device__ __forceinline__ void model_closest_pair(const double *r, const double *pu, const double *pv, const double *qs,
                                                   const double *qt, double n0, double n1, double n2, double n3,
                                                   double hP, double hQ, double *a)
{
    const double sc4[4] = { hP, hP, -hQ, -hQ };
    const double *col[4] = { pu, pv, qs, qt };
    const double nrm[4] = { n0, n1, n2, n3 };
    double inv[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) { inv[i] = nrm[i] > 1e-300 ? rcp_pos(nrm[i]) * sc4[i] : 0.0; a[i] = 0.0; }
    double rho[3] = { r[0], r[1], r[2] };
#pragma unroll
    for (int sw = 0; sw < DC_CD_SWEEPS; ++sw)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const double *J = col[i];
            const double dot = J[0] * rho[0] + J[1] * rho[1] + J[2] * rho[2];      // (J_i . rho) / h_i
            double t = fma(-dot, inv[i], a[i]);
            t = dmax2(-1.0, dmin2(1.0, t));
            const double da = (t - a[i]) * sc4[i];
            rho[0] = fma(J[0], da, rho[0]); rho[1] = fma(J[1], da, rho[1]); rho[2] = fma(J[2], da, rho[2]);
            a[i] = t;
        }
}

struct NodeOut {
    double ub, lb; bool leaf, splitP;
    double x0[4];                                  // closest pair of the first-order model, local coordinates
};

// ROOT: the node is a whole patch pair (round 0 of the branch and bound, 97 % of the nodes at config 2): the centre is
// (0,0) and the half-widths are 1, so the centre values and first derivatives ARE coefficients (no evaluation) and the
// scalar ranges need no re-centring.
template <bool ROOT, class CP, class CQ>
__device__ __forceinline__ NodeOut bound_node(CP AP, CQ AQ, double KP, double KQ,
                                              double uc, double vc, double hP, double sc, double tc, double hQ,
                                              double theta2)
{
    double r[3], pu[3], pv[3], qs[3], qt[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double p, q;
        if (ROOT) {
            p = AP(9 * c); pu[c] = AP(9 * c + 1); pv[c] = AP(9 * c + 3);
            q = AQ(9 * c); qs[c] = AQ(9 * c + 1); qt[c] = AQ(9 * c + 3);
        } else {
            eval_d1([&](int m) { return AP(9 * c + m); }, uc, vc, p, pu[c], pv[c]);
            eval_d1([&](int m) { return AQ(9 * c + m); }, sc, tc, q, qs[c], qt[c]);
        }
        r[c] = p - q;
    }
    NodeOut o;
    const double d2c = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
    // subdivision rule (squared form)
    const double hP2 = hP * hP, hQ2 = hQ * hQ;
    const double npu = pu[0] * pu[0] + pu[1] * pu[1] + pu[2] * pu[2], npv = pv[0] * pv[0] + pv[1] * pv[1] + pv[2] * pv[2];
    const double nqs = qs[0] * qs[0] + qs[1] * qs[1] + qs[2] * qs[2], nqt = qt[0] * qt[0] + qt[1] * qt[1] + qt[2] * qt[2];
    {
        const double S1P = hP2 * dmax2(npu, npv), S1Q = hQ2 * dmax2(nqs, nqt);
        const double s2P = hP2 * KP, s2Q = hQ2 * KQ;
        const double M = dmax2(S1P, S1Q);
        const bool okP = !(S1P > 0.0) || s2P * s2P * M <= theta2 * S1P * S1P;
        const bool okQ = !(S1Q > 0.0) || s2Q * s2Q * M <= theta2 * S1Q * S1Q;
        o.leaf = okP && okQ;
        o.splitP = S1P >= S1Q;
    }
    // closest pair of the first-order model
    double a[4];
    model_closest_pair(r, pu, pv, qs, qt, hP2 * npu, hP2 * npv, hQ2 * nqs, hQ2 * nqt, hP, hQ, a);
#pragma unroll
    for (int i = 0; i < 4; ++i) o.x0[i] = a[i];
    // the true patches at x0
    const double u0 = fma(hP, a[0], uc), v0 = fma(hP, a[1], vc), s0 = fma(hQ, a[2], sc), t0 = fma(hQ, a[3], tc);
    double r0[3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
        r0[c] = eval_d0([&](int m) { return AP(9 * c + m); }, u0, v0) - eval_d0([&](int m) { return AQ(9 * c + m); }, s0, t0);
    const double d20 = r0[0] * r0[0] + r0[1] * r0[1] + r0[2] * r0[2];
    // direction of the bound: the closest pair's (the centre's if the patches touch there)
    const bool use0 = d20 > 0.0;
    const double dd = use0 ? d20 : d2c;
    const double inv = dd > 0.0 ? rsqrt(dd) : 0.0;
    const double n[3] = { (use0 ? r0[0] : r[0]) * inv, (use0 ? r0[1] : r[1]) * inv, (use0 ? r0[2] : r[2]) * inv };
    // attained distances, rounded up (sqrt of the smaller square)
    const double dmin = dmin2(d20, d2c);
    o.ub = sqrt(dmin) * (1.0 + 4e-16);
    double gP[9], gQ[9];
#pragma unroll
    for (int m = 1; m < 9; ++m) {
        gP[m] = fma(n[2], AP(18 + m), fma(n[1], AP(9 + m), n[0] * AP(m)));
        gQ[m] = fma(n[2], AQ(18 + m), fma(n[1], AQ(9 + m), n[0] * AQ(m)));
    }
    double loP, hiP, loQ, hiQ;
    scalar_range<ROOT>(gP, uc, vc, hP, loP, hiP);
    scalar_range<ROOT>(gQ, sc, tc, hQ, loQ, hiQ);
    o.lb = fma(n[2], r[2], fma(n[1], r[1], n[0] * r[0])) + loP - hiQ;
    return o;
}

} // namespace dcg
