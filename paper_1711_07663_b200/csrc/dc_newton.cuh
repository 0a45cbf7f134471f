// dc_newton.cuh -- one iteration of the projected Newton closest-point solve between two biquadratic
// patches, written so that a warp can run it in LOCKSTEP (every lane does exactly one evaluation of
// value + gradient + Hessian per call) and lanes that finish are refilled from a queue.
//
// The solve is the two-patch generalisation of PAPER.md Eq. 3-5 (L256-L270): minimise
//   f(x) = 1/2 |P(u,v) - Q(s,t)|^2,   x = (u,v,s,t) in the box [lo,hi]   (a leaf of the branch and bound),
// with the paper's clamp to the reference box (L272-L278) as a projected step: variables at a bound whose
// gradient pushes outward are held, the rest take a Newton step (LDL^T with repaired pivots), the trial
// point is clamped and accepted only if f does not increase.
//
// Both patches are evaluated straight from their ROOT monomial coefficients (no re-centring): the box
// bounds are dyadic and exactly representable, so clamped variables sit exactly on sub-patch borders.
// Coefficients are read through an accessor `cf(m)`: m = c*9 + i + 3j for P (c = x,y,z), 27 + ... for Q.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace dcn {

#define DCN_HD __device__ __forceinline__      /* device only: there is no host build of the solver */

// (compare-and-select min / max of finite doubles: see dc_geom.cuh)
DCN_HD double dmin2(double a, double b) { return a < b ? a : b; }
DCN_HD double dmax2(double a, double b) { return a > b ? a : b; }

// reciprocal of a normal-range double: hardware seed (20 bits) + two Newton steps, ~1 ulp, no slow path (the divide
// the compiler emits for 1.0 / x carries a range check and a call; the pivots it is used on are >= floor > 0)
DCN_HD double rcp_fast(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    y = fma(fma(-x, y, 1.0), y, y);
    y = fma(fma(-x, y, 1.0), y, y);
    return y;
}

#ifndef NW_MAXIT
#define NW_MAXIT 24                 /* evaluations per solve before it is declared unconverged */
#endif

// state of one lane's solve
struct NwState {
    double x[4];
    int iters;                      // evaluations done
    int ls;                         // rejected trial steps at the current point (0: none yet)
    int phase;                      // 0 idle, 1 iterating, 3 last evaluation of an unconverged solve
};

struct NwResult { double dist, cosv; int converged; };

// value + first + second derivatives of one coordinate of a biquadratic at (a,b); C(m) = coefficient of a^i b^j, m = i+3j
template <class CF>
DCN_HD void jet(CF C, double a, double b, double &p, double &pa, double &pb, double &paa, double &pab, double &pbb)
{
    const double c0 = C(0), c1 = C(1), c2 = C(2), c3 = C(3), c4 = C(4), c5 = C(5), c6 = C(6), c7 = C(7), c8 = C(8);
    const double a2 = a + a, b2 = b + b;
    const double r0 = fma(a, fma(a, c2, c1), c0);
    const double r1 = fma(a, fma(a, c5, c4), c3);
    const double r2 = fma(a, fma(a, c8, c7), c6);
    const double d0 = fma(a2, c2, c1);
    const double d1 = fma(a2, c5, c4);
    const double d2 = fma(a2, c8, c7);
    p = fma(b, fma(b, r2, r1), r0);
    pb = fma(b2, r2, r1);
    pbb = r2 + r2;
    pa = fma(b, fma(b, d2, d1), d0);
    pab = fma(b2, d2, d1);
    const double e = fma(b, fma(b, c8, c5), c2);
    paa = e + e;
}

template <class CF>
DCN_HD double value(CF C, double a, double b)
{
    const double r0 = fma(a, fma(a, C(2), C(1)), C(0));
    const double r1 = fma(a, fma(a, C(5), C(4)), C(3));
    const double r2 = fma(a, fma(a, C(8), C(7)), C(6));
    return fma(b, fma(b, r2, r1), r0);
}

// Modified LDL^T solve of H p = -g for the symmetric 4x4 H (upper triangle): a pivot d that is not safely
// positive is replaced by max(|d|, floor) (Gill-Murray style, one pass, no retries, no branches), which
// turns a direction of negative or vanishing curvature into a descent direction of curvature scale.
// Returns true if any pivot had to be modified (H was not positive definite).
DCN_HD bool ldl4_mod(double h00, double h01, double h02, double h03, double h11, double h12, double h13,
                     double h22, double h23, double h33, const double *g, double floor, double *p)
{
    bool mod = !(h00 > floor);
    const double d0 = mod ? dmax2(fabs(h00), floor) : h00;
    const double i0 = rcp_fast(d0);
    const double l10 = h01 * i0, l20 = h02 * i0, l30 = h03 * i0;
    double d1 = fma(-l10, h01, h11);
    if (!(d1 > floor)) { mod = true; d1 = dmax2(fabs(d1), floor); }
    const double i1 = rcp_fast(d1);
    const double t21 = fma(-l20, h01, h12), t31 = fma(-l30, h01, h13);
    const double l21 = t21 * i1, l31 = t31 * i1;
    double d2 = fma(-l21, t21, fma(-l20, h02, h22));
    if (!(d2 > floor)) { mod = true; d2 = dmax2(fabs(d2), floor); }
    const double i2 = rcp_fast(d2);
    const double t32 = fma(-l31, t21, fma(-l30, h02, h23));
    const double l32 = t32 * i2;
    double d3 = fma(-l32, t32, fma(-l31, t31, fma(-l30, h03, h33)));
    if (!(d3 > floor)) { mod = true; d3 = dmax2(fabs(d3), floor); }
    const double i3 = rcp_fast(d3);
    const double y0 = -g[0];
    const double y1 = fma(-l10, y0, -g[1]);
    const double y2 = fma(-l21, y1, fma(-l20, y0, -g[2]));
    const double y3 = fma(-l32, y2, fma(-l31, y1, fma(-l30, y0, -g[3])));
    p[3] = y3 * i3;
    p[2] = fma(-l32, p[3], y2 * i2);
    p[1] = fma(-l31, p[3], fma(-l21, p[2], y1 * i1));
    p[0] = fma(-l30, p[3], fma(-l20, p[2], fma(-l10, p[1], y0 * i0)));
    return mod;
}

// One lockstep iteration (tol_d2 = tol_d^2, tau_exit2 = tau_exit^2 or negative to disable).  Returns true when the solve is finished (R filled: the distance is attained
// at the point just evaluated, hence an upper bound of the minimum whether or not it converged).
template <class CF>
DCN_HD bool iterate(CF cf, NwState &s, const double *lo, const double *hi, double tol_d2, double tau_exit2, NwResult &R,
                    int maxit = NW_MAXIT)
{
    const double u = s.x[0], v = s.x[1], sq = s.x[2], tq = s.x[3];
    double rr = 0.0, g[4] = { 0.0, 0.0, 0.0, 0.0 };
    double h00 = 0.0, h01 = 0.0, h02 = 0.0, h03 = 0.0, h11 = 0.0, h12 = 0.0, h13 = 0.0, h22 = 0.0, h23 = 0.0, h33 = 0.0;
    double r[3], Qs[3], Qt[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double p, pa, pb, paa, pab, pbb, q, qa, qb, qaa, qab, qbb;
        jet([&](int m) { return cf(9 * c + m); }, u, v, p, pa, pb, paa, pab, pbb);
        jet([&](int m) { return cf(27 + 9 * c + m); }, sq, tq, q, qa, qb, qaa, qab, qbb);
        const double rc = p - q;
        r[c] = rc; Qs[c] = qa; Qt[c] = qb;
        rr = fma(rc, rc, rr);
        g[0] = fma(rc, pa, g[0]); g[1] = fma(rc, pb, g[1]); g[2] = fma(-rc, qa, g[2]); g[3] = fma(-rc, qb, g[3]);
        h00 = fma(pa, pa, fma(rc, paa, h00)); h01 = fma(pa, pb, fma(rc, pab, h01));
        h02 = fma(-pa, qa, h02); h03 = fma(-pa, qb, h03);
        h11 = fma(pb, pb, fma(rc, pbb, h11)); h12 = fma(-pb, qa, h12); h13 = fma(-pb, qb, h13);
        h22 = fma(qa, qa, fma(-rc, qaa, h22)); h23 = fma(qa, qb, fma(-rc, qab, h23));
        h33 = fma(qb, qb, fma(-rc, qbb, h33));
    }
    s.iters++;
    // active set (L272-L278): a variable at a bound whose gradient pushes outward is held
    bool fx[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) fx[i] = (s.x[i] <= lo[i] && g[i] > 0.0) || (s.x[i] >= hi[i] && g[i] < 0.0);
    const double tr = (fx[0] ? 0.0 : fabs(h00)) + (fx[1] ? 0.0 : fabs(h11)) + (fx[2] ? 0.0 : fabs(h22)) + (fx[3] ? 0.0 : fabs(h33));
    const double gg = (fx[0] ? 0.0 : g[0] * g[0]) + (fx[1] ? 0.0 : g[1] * g[1]) + (fx[2] ? 0.0 : g[2] * g[2]) + (fx[3] ? 0.0 : g[3] * g[3]);
    double rr_out = rr;
    bool finished = s.phase >= 2 || rr <= tau_exit2 || gg == 0.0 || !(tr > 0.0);
    int converged = s.phase != 3;
    if (!finished) {
        // plain projected Newton: the held variables are decoupled, the rest take the (pivot-repaired) Newton step
        if (fx[0]) { h01 = h02 = h03 = 0.0; h00 = tr; g[0] = 0.0; }
        if (fx[1]) { h01 = h12 = h13 = 0.0; h11 = tr; g[1] = 0.0; }
        if (fx[2]) { h02 = h12 = h23 = 0.0; h22 = tr; g[2] = 0.0; }
        if (fx[3]) { h03 = h13 = h23 = 0.0; h33 = tr; g[3] = 0.0; }
        // A free variable that sits ON a bound (its gradient points inward) can still be pushed outward by the coupled
        // Newton step; clamping it leaves the other components of a step that assumed it would move -- not a descent
        // direction, and the trial is rejected over and over (22 to 25 evaluations on the near-contact leaves that used
        // to end unconverged).  Such variables are held for THIS step and the rest is solved again on that face of the
        // box (6 or 7 evaluations on the same leaves).  The convergence test keeps the first solve's predicted decrease:
        // a held variable with an inward gradient is not a KKT point.
        double p[4], pred = 0.0;
        bool indefinite = false;
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            indefinite = ldl4_mod(h00, h01, h02, h03, h11, h12, h13, h22, h23, h33, g, 1e-10 * tr, p) || indefinite;
            if (pass == 1) break;
            pred = -0.5 * (g[0] * p[0] + g[1] * p[1] + g[2] * p[2] + g[3] * p[3]);
            bool o[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) o[i] = !fx[i] && ((s.x[i] >= hi[i] && p[i] > 0.0) || (s.x[i] <= lo[i] && p[i] < 0.0));
            if (!(o[0] || o[1] || o[2] || o[3])) break;
            if (o[0]) { h01 = h02 = h03 = 0.0; h00 = tr; g[0] = 0.0; }
            if (o[1]) { h01 = h12 = h13 = 0.0; h11 = tr; g[1] = 0.0; }
            if (o[2]) { h02 = h12 = h23 = 0.0; h22 = tr; g[2] = 0.0; }
            if (o[3]) { h03 = h13 = h23 = 0.0; h33 = tr; g[3] = 0.0; }
        }
        // Step length of THIS call's single trial (s.ls counts the rejected trials at this point).  With an
        // indefinite H the minimum along the valley sits on the box border: the first trial stretches the
        // step until the first free variable reaches its bound.  A rejected trial is retried by the NEXT call with a
        // shorter step (retrying inside the call with value-only evaluations was tried: fewer evaluations, but the
        // extra code spills and every evaluation gets slower: 1.261 against 1.240 ms per cut).
        double xn[4], fn = 0.0;
        bool dec = false;
        {
            double alpha = 1.0;
            if (indefinite || s.ls > 0) {
                // largest multiple of p that keeps every free variable inside its bounds
                // (the smallest ratio room/p is found by cross-multiplication: one division instead of four)
                double rn = 1.0, pd = 0.0;       // ahit = rn / pd; pd == 0: no bound in the way
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const double room = fabs((p[i] > 0.0 ? hi[i] : lo[i]) - s.x[i]), pa = fabs(p[i]);
                    // (a variable already on the bound it is pushed against just stays clamped)
                    if (pa != 0.0 && room != 0.0 && (pd == 0.0 || room * pd < rn * pa)) { rn = room; pd = pa; }
                }
                const double ahit = pd != 0.0 ? rn / pd : INFINITY;
                const bool stretch = indefinite && ahit > 1.0 && ahit < INFINITY;
                const double q = __longlong_as_double((long long)(1023 - 2 * (s.ls > 0 ? s.ls - 1 : 0)) << 52);   // 4^-(ls-1)
                if (s.ls == 0) alpha = stretch ? ahit : 1.0;
                // a rejected trial is followed by UNCLAMPED ones: up to the first bound (a clamped step is not a
                // descent step when the clamped variable is coupled to the others), then quarters of that
                else alpha = stretch ? q : (ahit < 1.0 ? ahit * q : 0.25 * q);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                // (a trial point within rounding of a bound is snapped onto it: the step to the first bound lands
                // an ulp short of it as often as not, and "on the bound" is tested exactly everywhere)
                const double t = fma(alpha, p[i], s.x[i]), w = 1e-14 * (hi[i] - lo[i]);
                xn[i] = t >= hi[i] - w ? hi[i] : (t <= lo[i] + w ? lo[i] : t);
            }
            fn = 0.0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double d = value([&](int m) { return cf(9 * c + m); }, xn[0], xn[1])
                               - value([&](int m) { return cf(27 + 9 * c + m); }, xn[2], xn[3]);
                fn = fma(d, d, fn);
            }
            dec = fn <= rr;
        }
        bool moved = false;              // (no division: 0 / width would take the slow path of the FP64 divide)
        if (dec) {
#pragma unroll
            for (int i = 0; i < 4; ++i) { moved = moved || fabs(xn[i] - s.x[i]) >= 1e-15 * (hi[i] - lo[i]); s.x[i] = xn[i]; }
            s.ls = 0;
        } else s.ls++;
        if (pred * pred <= tol_d2 * dmax2(rr, tol_d2)) {
            // predicted decrease of the DISTANCE below tolerance: converged.  The distance reported is the
            // one attained at the accepted trial point (value-only evaluation), the sign cosine the one here.
            finished = true;
            if (dec) rr_out = fn;
        } else if ((dec && !moved) || s.ls > 7) {
            finished = true; converged = 0;              // stalled at the point just evaluated
        } else if (s.iters >= maxit - 1) {
            s.phase = 3;                                  // one last evaluation
        }
    }
    if (finished) {
        const double nx = Qs[1] * Qt[2] - Qs[2] * Qt[1];
        const double ny = Qs[2] * Qt[0] - Qs[0] * Qt[2];
        const double nz = Qs[0] * Qt[1] - Qs[1] * Qt[0];
        const double nn = nx * nx + ny * ny + nz * nz;
        const double den2 = rr * nn;
        R.dist = sqrt(rr_out);
        // (the cosine only decides a sign and a 7-bit magnitude: reciprocal square root instead of sqrt and divide)
        R.cosv = den2 > 0.0 ? (r[0] * nx + r[1] * ny + r[2] * nz) * rsqrt(den2) : 0.0;
        R.converged = converged;
    }
    return finished;
}

} // namespace dcn
