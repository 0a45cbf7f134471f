/*
 * dc_oracle.c -- CPU ORACLE for the direct-cut hole-cutting pass.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, link, import or call this file.  It shares no code with the CUDA path
 * (paper_1711_07663_b200/csrc) and neither includes the other.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md):
 *   For every element e of a grid of 27-node quadratic hexahedra (tensor-product Lagrange map,
 *   PAPER.md Eq. 1, K = 2) and a closed, outward-oriented surface S of 9-node quadratic
 *   quadrilateral faces:
 *     d_e   = min over faces f and the 6 boundary patches k of e of
 *             min_{(u,v),(s,t) in [-1,1]^2} |P_{e,k}(u,v) - Q_f(s,t)|          (L163-L165: "all
 *             elements calculate the (signed) minimum distance to the boundary")
 *     label = CUT    if d_e <= tau_cut   (L151 "vector of length 0 means ... intersect";
 *                                         A.3 L719/L773-L777, A.4 L815-L837: D < tol => D = 0)
 *             HOLE   if (p* - q*) . n(q*) < 0 at the closest pair on the nearest face
 *             NORMAL otherwise            (L151, L215: dot of the minimal vector with the
 *                                          face's outward normal; ties: largest |cos|, L294)
 *     sdist = 0 (CUT), else +-min(d_e, d_band), + for NORMAL.
 *
 * How (deliberately plain, slow, single-threaded, no spatial index, no Newton solve): every
 * element is tested against EVERY face; the pair minimum is enclosed by branch and bound over
 * midpoint-subdivided Bezier sub-nets, using the paper's own geometric device -- linear
 * triangles and triangle-triangle shortest vectors (L159, L213-L215, A.3/A.4) -- as the lower
 * bound, made rigorous by a deviation bound delta of each sub-net from its two triangles.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): shape functions, Bezier conversion/split,
 * A.2 box distance hand cases, tri-tri distance vs brute force, PATCHPAIR vs closed forms and
 * dense sampling, whole oracle vs the closed-form box-vs-sphere test on config 0, invariants
 * (no HOLE next to NORMAL, coverage of inside centroids, face/element permutation, rigid
 * motion, orientation reversal, exact face refinement).
 * PARITY UNPINNED: nearest-face id and closest-point parameters (not unique: shared edges,
 * rings of minimisers) -- reported for debugging only, never compared.
 *
 * Plain C99.  Build: gcc -O2 -fPIC -shared -o liboracle_dc.so dc_oracle.c -lm   (no -ffast-math)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_HOLE 0
#define ORC_NORMAL 1
#define ORC_CUT 2

#define ORC_FLAG_AMBIGUOUS 1      /* enclosure of d_e meets [tau - 1e-9 L, tau + 1e-9 L] */
#define ORC_FLAG_SIGN_AMBIG 2     /* tie-list members disagree in sign */
#define ORC_FLAG_FAR 4            /* proved d_e > d_band; relaxed enclosure used */
#define ORC_FLAG_DEPTH 8          /* depth cap hit somewhere (must not happen) */

typedef struct {
    double tau_cut_rel;  /* default 1e-7  (x L_ref)   reading A3 */
    double d_band;       /* <= 0: auto = max element Bezier-box diagonal   reading A5 */
    double l_ref;        /* <= 0: auto = longest edge of the AABB of all surface nodes */
    double eps_rel;      /* enclosure width, default 1e-12 (x L_ref) */
    double eps_far_rel;  /* enclosure width once d_e > d_band is proved, default 1e-6 */
    double tie_rel;      /* tie slack, default 1e-9 (x L_ref) */
    int max_depth;       /* default 60 */
    int reserved;
} orc_params;

typedef struct {
    long long n_box_tests;      /* element-box vs face-box tests (N_e * N_f) */
    long long n_pair_tests;     /* (e,f) pairs that reached the patch level ("pair tests") */
    long long n_patchpair;      /* PATCHPAIR calls */
    long long n_subpairs;       /* sub-pairs bounded (4 tri-tri each) */
    long long n_depth_exceeded;
    long long n_cut, n_hole, n_normal, n_ambiguous, n_sign_ambiguous, n_far;
    double l_ref, tau_cut, d_band;
} orc_stats;

/* ------------------------------------------------------------------ small vector helpers */
static inline double dot3(const double *a, const double *b) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }
static inline void sub3(const double *a, const double *b, double *c) { c[0]=a[0]-b[0]; c[1]=a[1]-b[1]; c[2]=a[2]-b[2]; }
static inline void cross3(const double *a, const double *b, double *c) {
    c[0] = a[1]*b[2] - a[2]*b[1]; c[1] = a[2]*b[0] - a[0]*b[2]; c[2] = a[0]*b[1] - a[1]*b[0];
}
static inline double norm3(const double *a) { return sqrt(dot3(a, a)); }
static inline double clamp01(double x) { return x < 0.0 ? 0.0 : (x > 1.0 ? 1.0 : x); }

/* ------------------------------------------------------------------ shape functions (Eq. 1) */
/* Quadratic Lagrange basis on nodes {-1,0,+1} (Eq. 1 L241 with K = 2; reading A2). */
void orc_shape(double t, double *l, double *dl, double *ddl)
{
    l[0] = 0.5 * t * (t - 1.0); l[1] = 1.0 - t * t; l[2] = 0.5 * t * (t + 1.0);
    if (dl)  { dl[0] = t - 0.5; dl[1] = -2.0 * t; dl[2] = t + 0.5; }
    if (ddl) { ddl[0] = 1.0; ddl[1] = -2.0; ddl[2] = 1.0; }
}

/* Biquadratic patch of 9 nodes X[i+3j]: value and first derivatives at (u,v) (Eq. 1-2). */
void orc_patch_eval(const double *X /*[9][3]*/, double u, double v, double *P, double *Pu, double *Pv)
{
    double lu[3], du[3], lv[3], dv[3];
    orc_shape(u, lu, du, 0); orc_shape(v, lv, dv, 0);
    for (int c = 0; c < 3; ++c) {
        double p = 0, pu = 0, pv = 0;
        for (int j = 0; j < 3; ++j)
            for (int i = 0; i < 3; ++i) {
                double x = X[(i + 3*j)*3 + c];
                p  += lu[i] * lv[j] * x;
                pu += du[i] * lv[j] * x;
                pv += lu[i] * dv[j] * x;
            }
        P[c] = p; if (Pu) Pu[c] = pu; if (Pv) Pv[c] = pv;
    }
}

/* Triquadratic hex of 27 nodes X[i+3j+9k] (Eq. 1), value only (used by tests). */
void orc_hex_eval(const double *X /*[27][3]*/, double xi, double eta, double zeta, double *P)
{
    double a[3], b[3], g[3];
    orc_shape(xi, a, 0, 0); orc_shape(eta, b, 0, 0); orc_shape(zeta, g, 0, 0);
    for (int c = 0; c < 3; ++c) {
        double p = 0;
        for (int k = 0; k < 3; ++k) for (int j = 0; j < 3; ++j) for (int i = 0; i < 3; ++i)
            p += a[i] * b[j] * g[k] * X[(i + 3*j + 9*k)*3 + c];
        P[c] = p;
    }
}

/* ------------------------------------------------------------------ Bezier form */
/* 1-D: b0 = x0, b1 = 2 x1 - (x0+x2)/2, b2 = x2, applied along i then along j. */
void orc_lagrange_to_bezier(const double *X /*[9][3]*/, double *B /*[9][3]*/)
{
    double T[27];
    for (int j = 0; j < 3; ++j) for (int c = 0; c < 3; ++c) {
        double x0 = X[(0+3*j)*3+c], x1 = X[(1+3*j)*3+c], x2 = X[(2+3*j)*3+c];
        T[(0+3*j)*3+c] = x0; T[(1+3*j)*3+c] = 2.0*x1 - 0.5*(x0+x2); T[(2+3*j)*3+c] = x2;
    }
    for (int i = 0; i < 3; ++i) for (int c = 0; c < 3; ++c) {
        double x0 = T[(i+0)*3+c], x1 = T[(i+3)*3+c], x2 = T[(i+6)*3+c];
        B[(i+0)*3+c] = x0; B[(i+3)*3+c] = 2.0*x1 - 0.5*(x0+x2); B[(i+6)*3+c] = x2;
    }
}

/* de Casteljau evaluation of a biquadratic Bezier net at (a,b) in [0,1]^2 (tests: P1). */
void orc_bezier_eval(const double *B, double a, double b, double *P)
{
    for (int c = 0; c < 3; ++c) {
        double r[3];
        for (int j = 0; j < 3; ++j) {
            double b0 = B[(0+3*j)*3+c], b1 = B[(1+3*j)*3+c], b2 = B[(2+3*j)*3+c];
            double q0 = (1-a)*b0 + a*b1, q1 = (1-a)*b1 + a*b2;
            r[j] = (1-a)*q0 + a*q1;
        }
        double q0 = (1-b)*r[0] + b*r[1], q1 = (1-b)*r[1] + b*r[2];
        P[c] = (1-b)*q0 + b*q1;
    }
}

/* Midpoint split of (b0,b1,b2): left (b0,(b0+b1)/2,(b0+2b1+b2)/4), right ((b0+2b1+b2)/4,(b1+b2)/2,b2).
 * dir 0 splits along i (u), dir 1 along j (v).  Outputs lower-half and upper-half nets. */
void orc_bezier_split(const double *B, int dir, double *Lo, double *Hi)
{
    int si = dir == 0 ? 1 : 3, so = dir == 0 ? 3 : 1;
    for (int o = 0; o < 3; ++o) for (int c = 0; c < 3; ++c) {
        double b0 = B[(0*si + o*so)*3+c], b1 = B[(1*si + o*so)*3+c], b2 = B[(2*si + o*so)*3+c];
        double m = 0.25 * (b0 + 2.0*b1 + b2);
        Lo[(0*si + o*so)*3+c] = b0; Lo[(1*si + o*so)*3+c] = 0.5*(b0+b1); Lo[(2*si + o*so)*3+c] = m;
        Hi[(0*si + o*so)*3+c] = m;  Hi[(1*si + o*so)*3+c] = 0.5*(b1+b2); Hi[(2*si + o*so)*3+c] = b2;
    }
}

/* AABB [min xyz, max xyz] of n points. */
static void box_of(const double *P, int n, double *box)
{
    for (int c = 0; c < 3; ++c) { box[c] = P[c]; box[3+c] = P[c]; }
    for (int m = 1; m < n; ++m) for (int c = 0; c < 3; ++c) {
        double x = P[m*3+c];
        if (x < box[c]) box[c] = x;
        if (x > box[3+c]) box[3+c] = x;
    }
}

/* ------------------------------------------------------------------ Algorithm A.2 */
/* BOUNDINGBOXDIST (PAPER.md A.2, L689-L709; loop bound read as i in {0,1,2}, reading G1). */
double orc_box_dist(const double *B1, const double *B2)
{
    double D = 0.0;
    for (int i = 0; i < 3; ++i) {
        if (B1[i+3] < B2[i] || B2[i+3] < B1[i]) {
            double a = B2[i] - B1[i+3], b = B1[i] - B2[i+3];
            double d = a > b ? a : b;
            D += d * d;
        }
    }
    return sqrt(D);
}

/* ------------------------------------------------------------------ triangle-triangle distance */
/* Closest points of segments p1 + s d1 (s in [0,1]) and p2 + t d2 (t in [0,1]). */
static double seg_seg(const double *p1, const double *q1, const double *p2, const double *q2,
                      double *s_out, double *t_out)
{
    double d1[3], d2[3], r[3];
    sub3(q1, p1, d1); sub3(q2, p2, d2); sub3(p1, p2, r);
    double a = dot3(d1, d1), e = dot3(d2, d2), f = dot3(d2, r);
    double s, t;
    if (a <= 0.0 && e <= 0.0) { s = t = 0.0; }
    else if (a <= 0.0) { s = 0.0; t = clamp01(f / e); }
    else {
        double c = dot3(d1, r);
        if (e <= 0.0) { t = 0.0; s = clamp01(-c / a); }
        else {
            double b = dot3(d1, d2), den = a * e - b * b;
            s = den > 0.0 ? clamp01((b * f - c * e) / den) : 0.0;
            t = (b * s + f) / e;
            if (t < 0.0) { t = 0.0; s = clamp01(-c / a); }
            else if (t > 1.0) { t = 1.0; s = clamp01((b - c) / a); }
        }
    }
    double w[3];
    for (int k = 0; k < 3; ++k) w[k] = (p1[k] + s * d1[k]) - (p2[k] + t * d2[k]);
    *s_out = s; *t_out = t;
    return norm3(w);
}

/* Closest point of triangle (a,b,c) to point p; barycentrics w (p* = w0 a + w1 b + w2 c). */
static double pt_tri(const double *p, const double *a, const double *b, const double *c, double *w)
{
    double e0[3], e1[3], v[3];
    sub3(b, a, e0); sub3(c, a, e1); sub3(p, a, v);
    double a00 = dot3(e0, e0), a01 = dot3(e0, e1), a11 = dot3(e1, e1);
    double b0 = dot3(e0, v), b1 = dot3(e1, v);
    double det = a00 * a11 - a01 * a01;
    if (det > 1e-300 * (a00 * a11 + 1e-300)) {
        double x = (a11 * b0 - a01 * b1) / det, y = (a00 * b1 - a01 * b0) / det;
        if (x >= 0.0 && y >= 0.0 && x + y <= 1.0) {
            w[0] = 1.0 - x - y; w[1] = x; w[2] = y;
            double q[3];
            for (int k = 0; k < 3; ++k) q[k] = p[k] - (a[k] + x * e0[k] + y * e1[k]);
            return norm3(q);
        }
    }
    /* projection falls outside (or degenerate triangle): closest point is on an edge */
    double best = INFINITY;
    const double *V[3] = { a, b, c };
    for (int i = 0; i < 3; ++i) {
        const double *s0 = V[i], *s1 = V[(i+1)%3];
        double d[3], r[3]; sub3(s1, s0, d); sub3(p, s0, r);
        double dd = dot3(d, d), t = dd > 0.0 ? clamp01(dot3(d, r) / dd) : 0.0;
        double q[3];
        for (int k = 0; k < 3; ++k) q[k] = p[k] - (s0[k] + t * d[k]);
        double dist = norm3(q);
        if (dist < best) {
            best = dist; w[0] = w[1] = w[2] = 0.0;
            w[i] = 1.0 - t; w[(i+1)%3] = t;
        }
    }
    return best;
}

/* Does segment (p,q) pierce triangle (a,b,c)?  If yes: parameter t along the segment and
 * barycentrics w of the piercing point. */
static int seg_pierces_tri(const double *p, const double *q, const double *a, const double *b,
                           const double *c, double *t_out, double *w)
{
    double e0[3], e1[3], n[3], pa[3], qa[3];
    sub3(b, a, e0); sub3(c, a, e1); cross3(e0, e1, n);
    sub3(p, a, pa); sub3(q, a, qa);
    double sp = dot3(n, pa), sq = dot3(n, qa);
    if ((sp > 0.0 && sq > 0.0) || (sp < 0.0 && sq < 0.0)) return 0;
    double den = sp - sq;
    if (den == 0.0) return 0; /* coplanar: covered by the edge-edge / vertex-triangle cases */
    double t = sp / den;
    double x[3], v[3];
    for (int k = 0; k < 3; ++k) x[k] = p[k] + t * (q[k] - p[k]);
    sub3(x, a, v);
    double a00 = dot3(e0, e0), a01 = dot3(e0, e1), a11 = dot3(e1, e1);
    double b0 = dot3(e0, v), b1 = dot3(e1, v);
    double det = a00 * a11 - a01 * a01;
    if (!(det > 0.0)) return 0;
    double y0 = (a11 * b0 - a01 * b1) / det, y1 = (a00 * b1 - a01 * b0) / det;
    if (y0 < 0.0 || y1 < 0.0 || y0 + y1 > 1.0) return 0;
    *t_out = t; w[0] = 1.0 - y0 - y1; w[1] = y0; w[2] = y1;
    return 1;
}

/* Exact distance between triangles A and B (3 vertices x 3 coords each) with the barycentrics
 * of one closest pair: min over 9 edge-edge and 6 vertex-triangle cases, 0 if an edge of one
 * pierces the other (the shortest-vector computation the paper takes from Moller's tri-tri
 * routine, L213, A.3 L759, A.4 L813). */
double orc_tri_tri_dist(const double *A, const double *B, double *wa, double *wb)
{
    double best = INFINITY;
    double ta[3] = {1,0,0}, tb[3] = {1,0,0};
    /* piercing */
    for (int i = 0; i < 3; ++i) {
        double t, w[3];
        if (seg_pierces_tri(A + 3*i, A + 3*((i+1)%3), B, B+3, B+6, &t, w)) {
            wa[0] = wa[1] = wa[2] = 0.0; wa[i] = 1.0 - t; wa[(i+1)%3] = t;
            wb[0] = w[0]; wb[1] = w[1]; wb[2] = w[2];
            return 0.0;
        }
        if (seg_pierces_tri(B + 3*i, B + 3*((i+1)%3), A, A+3, A+6, &t, w)) {
            wb[0] = wb[1] = wb[2] = 0.0; wb[i] = 1.0 - t; wb[(i+1)%3] = t;
            wa[0] = w[0]; wa[1] = w[1]; wa[2] = w[2];
            return 0.0;
        }
    }
    /* vertex - triangle */
    for (int i = 0; i < 3; ++i) {
        double w[3];
        double d = pt_tri(A + 3*i, B, B+3, B+6, w);
        if (d < best) { best = d; ta[0]=ta[1]=ta[2]=0; ta[i]=1; tb[0]=w[0]; tb[1]=w[1]; tb[2]=w[2]; }
        d = pt_tri(B + 3*i, A, A+3, A+6, w);
        if (d < best) { best = d; tb[0]=tb[1]=tb[2]=0; tb[i]=1; ta[0]=w[0]; ta[1]=w[1]; ta[2]=w[2]; }
    }
    /* edge - edge */
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
        double s, t;
        double d = seg_seg(A + 3*i, A + 3*((i+1)%3), B + 3*j, B + 3*((j+1)%3), &s, &t);
        if (d < best) {
            best = d;
            ta[0]=ta[1]=ta[2]=0; ta[i] = 1.0 - s; ta[(i+1)%3] = s;
            tb[0]=tb[1]=tb[2]=0; tb[j] = 1.0 - t; tb[(j+1)%3] = t;
        }
    }
    for (int k = 0; k < 3; ++k) { wa[k] = ta[k]; wb[k] = tb[k]; }
    return best;
}

/* ------------------------------------------------------------------ PATCHPAIR */
typedef struct {
    double b[27];            /* Bezier sub-net, point m = i + 3j */
    double u0, u1, v0, v1;   /* reference-parameter rectangle it covers */
} subnet;

/* Deviation of a biquadratic Bezier sub-net from the two triangles (c00,c20,c22),(c00,c22,c02)
 * at equal parameters:
 *   delta = 1/4 ( max_j |b0j - 2 b1j + b2j| + max_{i in {0,2}} |bi0 - 2 bi1 + bi2|
 *                 + |b00 - b20 - b02 + b22| ). */
static double subnet_delta(const double *b)
{
    double m1 = 0.0, m2 = 0.0, w[3];
    for (int j = 0; j < 3; ++j) {
        for (int c = 0; c < 3; ++c) w[c] = b[(0+3*j)*3+c] - 2.0*b[(1+3*j)*3+c] + b[(2+3*j)*3+c];
        double n = norm3(w); if (n > m1) m1 = n;
    }
    for (int i = 0; i < 3; i += 2) {
        for (int c = 0; c < 3; ++c) w[c] = b[(i+0)*3+c] - 2.0*b[(i+3)*3+c] + b[(i+6)*3+c];
        double n = norm3(w); if (n > m2) m2 = n;
    }
    for (int c = 0; c < 3; ++c) w[c] = b[0*3+c] - b[2*3+c] - b[6*3+c] + b[8*3+c];
    return 0.25 * (m1 + m2 + norm3(w));
}

typedef struct {
    subnet P, Q;
    double lo;
    int depth;
} subpair;

typedef struct {
    double hi;               /* best attained distance of this pair (true patches) */
    double u, v, s, t;       /* attaining parameters */
    double r[3];             /* P(u,v) - Q(s,t) */
    double n[3];             /* Q_s x Q_t at (s,t) */
    int status;              /* 0 = enclosure [hi-eps,hi]; 1 = pruned (> cutoff); 2 = early exit hi <= tau_exit */
    int depth_exceeded;
    long long n_subpairs;
} pp_result;

typedef struct {
    const double *PX, *QX;   /* Lagrange nodes of the two root patches */
    double cutoff, eps, tau_exit;
    int max_depth;
    pp_result *res;
} pp_ctx;

/* Bound one sub-pair: returns lo; updates ctx->res->hi from the true patches at the mapped
 * closest points of the 4 triangle pairs. */
static double bound_subpair(pp_ctx *ctx, const subnet *P, const subnet *Q)
{
    double boxP[6], boxQ[6];
    box_of(P->b, 9, boxP); box_of(Q->b, 9, boxQ);
    double lo_box = orc_box_dist(boxP, boxQ);
    pp_result *R = ctx->res;
    double bound = R->hi - ctx->eps; if (ctx->cutoff < bound) bound = ctx->cutoff;
    if (lo_box > bound) return lo_box;
    R->n_subpairs++;
    /* triangles: T1 = (c00,c20,c22), T2 = (c00,c22,c02) with their parameter corners */
    const int ci[2][3] = { {0, 2, 8}, {0, 8, 6} };
    double TP[2][9], TQ[2][9], pu[2][3], pv[2][3], qs[2][3], qt[2][3];
    for (int k = 0; k < 2; ++k) for (int m = 0; m < 3; ++m) {
        int id = ci[k][m];
        for (int c = 0; c < 3; ++c) { TP[k][3*m+c] = P->b[id*3+c]; TQ[k][3*m+c] = Q->b[id*3+c]; }
        pu[k][m] = (id % 3 == 0) ? P->u0 : P->u1; pv[k][m] = (id / 3 == 0) ? P->v0 : P->v1;
        qs[k][m] = (id % 3 == 0) ? Q->u0 : Q->u1; qt[k][m] = (id / 3 == 0) ? Q->v0 : Q->v1;
    }
    double d_lin = INFINITY;
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) {
        double wa[3], wb[3];
        double d = orc_tri_tri_dist(TP[a], TQ[b], wa, wb);
        if (d < d_lin) d_lin = d;
        /* upper bound: the TRUE patches at the parameters of the triangle closest points */
        double u = wa[0]*pu[a][0] + wa[1]*pu[a][1] + wa[2]*pu[a][2];
        double v = wa[0]*pv[a][0] + wa[1]*pv[a][1] + wa[2]*pv[a][2];
        double s = wb[0]*qs[b][0] + wb[1]*qs[b][1] + wb[2]*qs[b][2];
        double t = wb[0]*qt[b][0] + wb[1]*qt[b][1] + wb[2]*qt[b][2];
        double Pp[3], Qp[3], Qs[3], Qt[3], r[3];
        orc_patch_eval(ctx->PX, u, v, Pp, 0, 0);
        orc_patch_eval(ctx->QX, s, t, Qp, Qs, Qt);
        sub3(Pp, Qp, r);
        double h = norm3(r);
        if (h < R->hi) {
            R->hi = h; R->u = u; R->v = v; R->s = s; R->t = t;
            R->r[0] = r[0]; R->r[1] = r[1]; R->r[2] = r[2];
            cross3(Qs, Qt, R->n);
        }
    }
    double lo = d_lin - subnet_delta(P->b) - subnet_delta(Q->b);
    if (lo_box > lo) lo = lo_box;
    if (lo < 0.0) lo = 0.0;
    return lo;
}

static void split4(const subnet *S, subnet *C /*[4]*/)
{
    double lo[27], hi[27];
    double um = 0.5 * (S->u0 + S->u1), vm = 0.5 * (S->v0 + S->v1);
    orc_bezier_split(S->b, 0, lo, hi);
    orc_bezier_split(lo, 1, C[0].b, C[2].b);
    orc_bezier_split(hi, 1, C[1].b, C[3].b);
    C[0].u0 = S->u0; C[0].u1 = um;    C[0].v0 = S->v0; C[0].v1 = vm;
    C[1].u0 = um;    C[1].u1 = S->u1; C[1].v0 = S->v0; C[1].v1 = vm;
    C[2].u0 = S->u0; C[2].u1 = um;    C[2].v0 = vm;    C[2].v1 = S->v1;
    C[3].u0 = um;    C[3].u1 = S->u1; C[3].v0 = vm;    C[3].v1 = S->v1;
}

static double box_diag(const double *b)
{
    double box[6]; box_of(b, 9, box);
    double d[3] = { box[3]-box[0], box[4]-box[1], box[5]-box[2] };
    return norm3(d);
}

/* PATCHPAIR(P, Q, cutoff): depth-first branch and bound over pairs of Bezier sub-nets
 * (SURVEY 8(c) step 4).  PX, QX: Lagrange nodes [9][3].  On return status 0 the pair minimum
 * lies in [hi - eps, hi]; status 1: it is > cutoff; status 2: hi <= tau_exit (certainly CUT). */
void orc_patch_pair(const double *PX, const double *QX, double cutoff, double eps,
                    double tau_exit, int max_depth, pp_result *R)
{
    pp_ctx ctx = { PX, QX, cutoff, eps, tau_exit, max_depth, R };
    R->hi = INFINITY; R->status = 1; R->depth_exceeded = 0; R->n_subpairs = 0;
    R->u = R->v = R->s = R->t = 0.0;
    R->r[0] = R->r[1] = R->r[2] = 0.0; R->n[0] = R->n[1] = R->n[2] = 0.0;

    int cap = 3 * (max_depth + 2) + 8;
    subpair *stack = (subpair *)malloc(sizeof(subpair) * (size_t)cap);
    int top = 0;
    subpair root;
    orc_lagrange_to_bezier(PX, root.P.b); orc_lagrange_to_bezier(QX, root.Q.b);
    root.P.u0 = root.P.v0 = root.Q.u0 = root.Q.v0 = -1.0;
    root.P.u1 = root.P.v1 = root.Q.u1 = root.Q.v1 = 1.0;
    root.depth = 0;
    root.lo = bound_subpair(&ctx, &root.P, &root.Q);
    stack[top++] = root;
    while (top > 0) {
        if (R->hi <= tau_exit) { R->status = 2; free(stack); return; }
        subpair cur = stack[--top];
        double bound = R->hi - eps; if (cutoff < bound) bound = cutoff;
        if (cur.lo > bound) continue;
        if (cur.depth >= max_depth) { R->depth_exceeded++; continue; }
        /* split the sub-net that deviates more from its triangles (tie: the larger one) */
        double dP = subnet_delta(cur.P.b), dQ = subnet_delta(cur.Q.b);
        int splitP = dP > dQ || (dP == dQ && box_diag(cur.P.b) >= box_diag(cur.Q.b));
        subnet C[4];
        subpair ch[4];
        split4(splitP ? &cur.P : &cur.Q, C);
        int nch = 0;
        for (int k = 0; k < 4; ++k) {
            subpair *c = &ch[nch];
            if (splitP) { c->P = C[k]; c->Q = cur.Q; } else { c->P = cur.P; c->Q = C[k]; }
            c->depth = cur.depth + 1;
            c->lo = bound_subpair(&ctx, &c->P, &c->Q);
            bound = R->hi - eps; if (cutoff < bound) bound = cutoff;
            if (c->lo > bound) continue;
            nch++;
        }
        /* push in descending lo so the most promising child is popped first */
        for (int a = 0; a < nch; ++a) for (int b = a + 1; b < nch; ++b)
            if (ch[b].lo > ch[a].lo) { subpair t = ch[a]; ch[a] = ch[b]; ch[b] = t; }
        for (int a = 0; a < nch; ++a) stack[top++] = ch[a];
    }
    if (R->hi <= tau_exit) R->status = 2;
    else if (R->hi <= cutoff) R->status = 0;
    else R->status = 1;
    free(stack);
}

/* Flat wrapper for tests: out = { hi, u, v, s, t, rx, ry, rz, nx, ny, nz, status, depth_exceeded, n_subpairs } */
void orc_patch_pair_flat(const double *PX, const double *QX, double cutoff, double eps,
                         double tau_exit, int max_depth, double *out)
{
    pp_result R;
    orc_patch_pair(PX, QX, cutoff, eps, tau_exit, max_depth, &R);
    out[0] = R.hi; out[1] = R.u; out[2] = R.v; out[3] = R.s; out[4] = R.t;
    out[5] = R.r[0]; out[6] = R.r[1]; out[7] = R.r[2];
    out[8] = R.n[0]; out[9] = R.n[1]; out[10] = R.n[2];
    out[11] = (double)R.status; out[12] = (double)R.depth_exceeded; out[13] = (double)R.n_subpairs;
}

/* ------------------------------------------------------------------ element boundary patches */
/* Local hex node ids (m = i + 3j + 9k) of the 9 nodes of boundary patch k, as a 3x3 quad
 * (a + 3b).  k = 0..5 <-> xi=-1, xi=+1, eta=-1, eta=+1, zeta=-1, zeta=+1 (reading A1). */
static void hex_face_nodes(int k, int *ids)
{
    for (int b = 0; b < 3; ++b) for (int a = 0; a < 3; ++a) {
        int i, j, l;
        switch (k) {
        case 0: i = 0; j = a; l = b; break;
        case 1: i = 2; j = a; l = b; break;
        case 2: j = 0; i = a; l = b; break;
        case 3: j = 2; i = a; l = b; break;
        case 4: l = 0; i = a; j = b; break;
        default: l = 2; i = a; j = b; break;
        }
        ids[a + 3*b] = i + 3*j + 9*l;
    }
}
void orc_hex_face_nodes(int k, int *ids) { hex_face_nodes(k, ids); }

typedef struct { double lb; int f; } cand;
static int cand_cmp(const void *a, const void *b)
{
    double x = ((const cand *)a)->lb, y = ((const cand *)b)->lb;
    if (x < y) return -1; if (x > y) return 1;
    return ((const cand *)a)->f - ((const cand *)b)->f;
}

typedef struct { double hi, cosv; int f; } tie_rec;

/* ------------------------------------------------------------------ the whole pass */
/*
 * Classify elements [e_begin, e_end) of the grid against ALL n_face faces (exhaustive).
 *   xyz [n_nodes][3], conn27 [n_elem][27] (m = i+3j+9k), faces [n_face][9][3] (m = i+3j).
 * Outputs are indexed by (e - e_begin); any of dmin/width/nearest/flags may be NULL.
 * Returns 0, or -1 on bad arguments / allocation failure.
 */
int orc_classify(long long n_nodes, const double *xyz, long long n_elem, const int *conn27,
                 long long n_face, const double *faces, const orc_params *prm,
                 long long e_begin, long long e_end,
                 signed char *labels, double *sdist, double *dmin, double *width,
                 int *nearest, unsigned char *flags, orc_stats *st)
{
    if (!xyz || !conn27 || !faces || !prm || !labels || !sdist || n_face <= 0 || n_elem <= 0) return -1;
    if (e_begin < 0) e_begin = 0;
    if (e_end > n_elem) e_end = n_elem;
    (void)n_nodes;
    orc_stats S; memset(&S, 0, sizeof S);

    /* step 1: pre-pass.  Face Bezier nets and boxes; L_ref; tau; d_band. */
    double *fbox = (double *)malloc(sizeof(double) * 6 * (size_t)n_face);
    if (!fbox) return -1;
    double smin[3] = { INFINITY, INFINITY, INFINITY }, smax[3] = { -INFINITY, -INFINITY, -INFINITY };
    for (long long f = 0; f < n_face; ++f) {
        double B[27];
        orc_lagrange_to_bezier(faces + 27*f, B);
        box_of(B, 9, fbox + 6*f);
        for (int m = 0; m < 9; ++m) for (int c = 0; c < 3; ++c) {
            double x = faces[27*f + 3*m + c];
            if (x < smin[c]) smin[c] = x;
            if (x > smax[c]) smax[c] = x;
        }
    }
    double L_ref = prm->l_ref;
    if (!(L_ref > 0.0)) {
        L_ref = 0.0;
        for (int c = 0; c < 3; ++c) if (smax[c] - smin[c] > L_ref) L_ref = smax[c] - smin[c];
    }
    double tau = (prm->tau_cut_rel > 0.0 ? prm->tau_cut_rel : 1e-7) * L_ref;
    double eps_near = (prm->eps_rel > 0.0 ? prm->eps_rel : 1e-12) * L_ref;
    double eps_far = (prm->eps_far_rel > 0.0 ? prm->eps_far_rel : 1e-6) * L_ref;
    double t_tie = (prm->tie_rel > 0.0 ? prm->tie_rel : 1e-9) * L_ref;
    double tau_exit = tau - 1e-9 * L_ref;
    int max_depth = prm->max_depth > 0 ? prm->max_depth : 60;

    int fid[6][9];
    for (int k = 0; k < 6; ++k) hex_face_nodes(k, fid[k]);

    double d_band = prm->d_band;
    if (!(d_band > 0.0)) {
        /* auto: max over ALL elements of the diagonal of the box of the 6 boundary Bezier nets */
        d_band = 0.0;
        for (long long e = 0; e < n_elem; ++e) {
            double eb[6] = { INFINITY, INFINITY, INFINITY, -INFINITY, -INFINITY, -INFINITY };
            for (int k = 0; k < 6; ++k) {
                double X[27], B[27], bx[6];
                for (int m = 0; m < 9; ++m) {
                    const double *p = xyz + 3 * (long long)conn27[27*e + fid[k][m]];
                    X[3*m] = p[0]; X[3*m+1] = p[1]; X[3*m+2] = p[2];
                }
                orc_lagrange_to_bezier(X, B); box_of(B, 9, bx);
                for (int c = 0; c < 3; ++c) {
                    if (bx[c] < eb[c]) eb[c] = bx[c];
                    if (bx[3+c] > eb[3+c]) eb[3+c] = bx[3+c];
                }
            }
            double d[3] = { eb[3]-eb[0], eb[4]-eb[1], eb[5]-eb[2] };
            double dg = norm3(d);
            if (dg > d_band) d_band = dg;
        }
    }
    S.l_ref = L_ref; S.tau_cut = tau; S.d_band = d_band;

    cand *cands = (cand *)malloc(sizeof(cand) * (size_t)n_face);
    double *lbs = (double *)malloc(sizeof(double) * (size_t)n_face);
    int tie_cap = 64, n_tie = 0;
    tie_rec *ties = (tie_rec *)malloc(sizeof(tie_rec) * (size_t)tie_cap);
    if (!cands || !lbs || !ties) { free(fbox); free(cands); free(lbs); free(ties); return -1; }

    for (long long e = e_begin; e < e_end; ++e) {
        long long o = e - e_begin;
        /* boundary patches of e: Lagrange nodes, Bezier boxes */
        double PX[6][27], pbox[6][6], ebox[6] = { INFINITY, INFINITY, INFINITY, -INFINITY, -INFINITY, -INFINITY };
        for (int k = 0; k < 6; ++k) {
            double B[27];
            for (int m = 0; m < 9; ++m) {
                const double *p = xyz + 3 * (long long)conn27[27*e + fid[k][m]];
                PX[k][3*m] = p[0]; PX[k][3*m+1] = p[1]; PX[k][3*m+2] = p[2];
            }
            orc_lagrange_to_bezier(PX[k], B); box_of(B, 9, pbox[k]);
            for (int c = 0; c < 3; ++c) {
                if (pbox[k][c] < ebox[c]) ebox[c] = pbox[k][c];
                if (pbox[k][3+c] > ebox[3+c]) ebox[3+c] = pbox[k][3+c];
            }
        }
        /* step 3a: box lower bound against EVERY face */
        double lb_min = INFINITY; long long f0 = 0;
        for (long long f = 0; f < n_face; ++f) {
            double lb = orc_box_dist(ebox, fbox + 6*f);
            lbs[f] = lb;
            if (lb < lb_min) { lb_min = lb; f0 = f; }
        }
        S.n_box_tests += n_face;
        /* step 2: upper bound from node pairs (nodes lie on the patches) with the min-lb face */
        double ub = INFINITY;
        for (int k = 0; k < 6; ++k) for (int m = 0; m < 9; ++m) for (int q = 0; q < 9; ++q) {
            double w[3]; sub3(&PX[k][3*m], faces + 27*f0 + 3*q, w);
            double d = norm3(w);
            if (d < ub) ub = d;
        }
        int far = lb_min > d_band + t_tie;
        double eps = far ? eps_far : eps_near;
        const double ub_nodes = ub;
        /* step 3b: every face whose box bound does not exceed the cutoff, nearest box first */
        long long nc = 0;
        for (long long f = 0; f < n_face; ++f)
            if (lbs[f] <= ub + t_tie) { cands[nc].lb = lbs[f]; cands[nc].f = (int)f; nc++; }
        qsort(cands, (size_t)nc, sizeof(cand), cand_cmp);
        int is_cut = 0, depth_hit = 0;
    redo:
        n_tie = 0;
        for (long long ci = 0; ci < nc && !is_cut; ++ci) {
            double c = ub + t_tie;
            if (cands[ci].lb > c) break;
            int f = cands[ci].f;
            S.n_pair_tests++;
            for (int k = 0; k < 6 && !is_cut; ++k) {
                c = ub + t_tie;
                if (orc_box_dist(pbox[k], fbox + 6*(long long)f) > c) continue;
                pp_result R;
                orc_patch_pair(PX[k], faces + 27*(long long)f, c, eps, tau_exit, max_depth, &R);
                S.n_patchpair++; S.n_subpairs += R.n_subpairs;
                if (R.depth_exceeded) { depth_hit = 1; S.n_depth_exceeded += R.depth_exceeded; }
                if (R.status == 2) { is_cut = 1; ub = R.hi; break; }
                if (R.status != 0) continue;
                double rn = norm3(R.r), nn = norm3(R.n);
                double cosv = (rn > 0.0 && nn > 0.0) ? dot3(R.r, R.n) / (rn * nn) : 0.0;
                if (R.hi < ub - t_tie) n_tie = 0;
                if (R.hi < ub) ub = R.hi;
                if (n_tie == tie_cap) {
                    tie_cap *= 2;
                    ties = (tie_rec *)realloc(ties, sizeof(tie_rec) * (size_t)tie_cap);
                    if (!ties) { free(fbox); free(cands); free(lbs); return -1; }
                }
                ties[n_tie].hi = R.hi; ties[n_tie].cosv = cosv; ties[n_tie].f = f; n_tie++;
            }
        }
        /* The relaxed enclosure of a far element (SURVEY 8(c) "Far elements") only certifies a pair's minimum to
         * eps_far, so PATCHPAIR may report "beyond the cutoff" for a pair whose minimum lies within eps_far below
         * it; when the node-pair bound `ub` happens to be that sharp for EVERY pair, no tie member is left and
         * step 5 would have no r.n to take a sign from.  The strict enclosure is the definition: redo the element
         * with it (then hi <= d* + eps_near < ub + t_tie for the nearest pair, so the list cannot be empty). */
        if (!is_cut && n_tie == 0 && eps != eps_near) { eps = eps_near; ub = ub_nodes; goto redo; }
        /* step 5: label */
        unsigned char fl = 0;
        if (far) { fl |= ORC_FLAG_FAR; S.n_far++; }
        if (depth_hit) fl |= ORC_FLAG_DEPTH;
        int lab; double sd; int near_f = -1;
        if (is_cut || ub <= tau) {
            lab = ORC_CUT; sd = 0.0;
            if (!is_cut && ub >= tau - 1e-9 * L_ref - eps) fl |= ORC_FLAG_AMBIGUOUS;
        } else {
            if (ub - eps <= tau + 1e-9 * L_ref) fl |= ORC_FLAG_AMBIGUOUS;
            double bestc = -1.0, sgn = 1.0; int npos = 0, nneg = 0;
            for (int i = 0; i < n_tie; ++i) {
                if (ties[i].hi > ub + t_tie) continue;
                if (ties[i].cosv < 0.0) nneg++; else npos++;
                double a = fabs(ties[i].cosv);
                if (a > bestc) { bestc = a; sgn = ties[i].cosv < 0.0 ? -1.0 : 1.0; near_f = ties[i].f; }
            }
            if (npos && nneg) fl |= ORC_FLAG_SIGN_AMBIG;
            lab = sgn < 0.0 ? ORC_HOLE : ORC_NORMAL;
            sd = sgn * (ub < d_band ? ub : d_band);
        }
        labels[o] = (signed char)lab; sdist[o] = sd;
        if (dmin) dmin[o] = ub;
        if (width) width[o] = eps;
        if (nearest) nearest[o] = near_f;
        if (flags) flags[o] = fl;
        if (lab == ORC_CUT) S.n_cut++; else if (lab == ORC_HOLE) S.n_hole++; else S.n_normal++;
        if (fl & ORC_FLAG_AMBIGUOUS) S.n_ambiguous++;
        if (fl & ORC_FLAG_SIGN_AMBIG) S.n_sign_ambiguous++;
    }
    free(fbox); free(cands); free(lbs); free(ties);
    if (st) *st = S;
    return 0;
}

/* Element Bezier box (tests compare the CUDA S2 boxes against this). out[6] = min xyz, max xyz. */
void orc_element_box(const double *xyz, const int *conn27_e, double *out)
{
    int ids[9];
    for (int c = 0; c < 3; ++c) { out[c] = INFINITY; out[3+c] = -INFINITY; }
    for (int k = 0; k < 6; ++k) {
        double X[27], B[27], bx[6];
        hex_face_nodes(k, ids);
        for (int m = 0; m < 9; ++m) {
            const double *p = xyz + 3 * (long long)conn27_e[ids[m]];
            X[3*m] = p[0]; X[3*m+1] = p[1]; X[3*m+2] = p[2];
        }
        orc_lagrange_to_bezier(X, B); box_of(B, 9, bx);
        for (int c = 0; c < 3; ++c) {
            if (bx[c] < out[c]) out[c] = bx[c];
            if (bx[3+c] > out[3+c]) out[3+c] = bx[3+c];
        }
    }
}
