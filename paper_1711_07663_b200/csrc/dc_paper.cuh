// dc_paper.cuh -- the paper's OWN approximate direct cut as a second path (DC_FLAG_PAPER_MODE):
// PAPER.md 4.2 L191-L215 and Appendix A (A.1 L672-L687, A.2 L689-L709, A.3 L711-L783, A.4 L785-L845), with its constants
// N_F^1 = 16 (L209), N_F^2 = 4 (L213), the nearest-corner 3-face shortcut (L213) and the normal averaging of L215.
// It replaces S5/S6 for the band elements (the candidate pairs of S4 stand in for the paper's hole-map and bounding-box
// filters, L177-L191; S7 labels the rest as in the exact mode), so that the heuristics can be compared with the exact
// result, element by element, and timed on the same machine.  Readings PM1-PM8 of DESIGN.md.
//
//   k_pm_rank    thread / band element : OBB of the 8 corner nodes (Jacobi on their covariance matrix), A.1 on every
//                                        candidate face, the 16 nearest kept (sorted by (distance, face id))
//   k_pm_pass1   thread / (element, j<16) : A.3 -- nearest corner, 3 element faces x 2 x 2 corner triangles
//   k_pm_select  thread / band element : the 4 nearest of the 16
//   k_pm_pass2   thread / (element, j<4, q<3) : A.4 -- one element face (8 triangles) against the face's 8 triangles
//   k_pm_decide  thread / band element : nearest face, averaged normals, label, signed distance
//
// TRITRIDISTANCE here is this file's own routine (segment-segment and point-triangle closest points, edge-triangle
// crossings); the oracle's (oracle/dc_oracle.c) is another implementation of the same textbook operation.
#pragma once

#define PM_NF1 16
#define PM_NF2 4

namespace dcp {

struct V3 { double x, y, z; };
__device__ __forceinline__ V3 v3(double x, double y, double z) { V3 r; r.x = x; r.y = y; r.z = z; return r; }
__device__ __forceinline__ V3 operator+(V3 a, V3 b) { return v3(a.x + b.x, a.y + b.y, a.z + b.z); }
__device__ __forceinline__ V3 operator-(V3 a, V3 b) { return v3(a.x - b.x, a.y - b.y, a.z - b.z); }
__device__ __forceinline__ V3 operator*(double s, V3 a) { return v3(s * a.x, s * a.y, s * a.z); }
__device__ __forceinline__ double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
__device__ __forceinline__ V3 cross(V3 a, V3 b) { return v3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x); }
__device__ __forceinline__ double clamp01(double t) { return t < 0.0 ? 0.0 : (t > 1.0 ? 1.0 : t); }
__device__ __forceinline__ V3 ldv(const double *p) { return v3(__ldg(p), __ldg(p + 1), __ldg(p + 2)); }

// (the OBB and Algorithm A.1 decide which 16 faces are kept: their arithmetic is written without FMA contraction, operation
// by operation as the oracle's C, so that both sides rank with the same numbers)
__device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double dot_nc(V3 a, V3 b) { return add(add(mul(a.x, b.x), mul(a.y, b.y)), mul(a.z, b.z)); }

struct Tri { V3 a, b, c; };

// closest points of the segments p1 + s d1 and p2 + t d2 (s, t in [0,1]): squared distance, vector (on 2) - (on 1)
__device__ __forceinline__ double seg_seg(V3 p1, V3 d1, V3 p2, V3 d2, V3 &w)
{
    const V3 r = p1 - p2;
    const double a = dot(d1, d1), e = dot(d2, d2), f = dot(d2, r);
    double s, t;
    if (a <= 0.0 && e <= 0.0) { s = t = 0.0; }
    else if (a <= 0.0) { s = 0.0; t = clamp01(f / e); }
    else {
        const double c = dot(d1, r);
        if (e <= 0.0) { t = 0.0; s = clamp01(-c / a); }
        else {
            const double b = dot(d1, d2), den = a * e - b * b;
            s = den > 0.0 ? clamp01((b * f - c * e) / den) : 0.0;
            t = (b * s + f) / e;
            if (t < 0.0) { t = 0.0; s = clamp01(-c / a); }
            else if (t > 1.0) { t = 1.0; s = clamp01((b - c) / a); }
        }
    }
    w = (p2 + t * d2) - (p1 + s * d1);
    return dot(w, w);
}

// closest point of triangle T to the point p (Voronoi regions of the triangle): vector (closest point) - p
__device__ __forceinline__ double pt_tri(V3 p, const Tri &T, V3 &w)
{
    const V3 ab = T.b - T.a, ac = T.c - T.a, ap = p - T.a;
    const double d1 = dot(ab, ap), d2 = dot(ac, ap);
    V3 q;
    if (d1 <= 0.0 && d2 <= 0.0) q = T.a;
    else {
        const V3 bp = p - T.b;
        const double d3 = dot(ab, bp), d4 = dot(ac, bp);
        if (d3 >= 0.0 && d4 <= d3) q = T.b;
        else {
            const double vc = d1 * d4 - d3 * d2;
            if (vc <= 0.0 && d1 >= 0.0 && d3 <= 0.0) q = T.a + (d1 / (d1 - d3)) * ab;
            else {
                const V3 cp = p - T.c;
                const double d5 = dot(ab, cp), d6 = dot(ac, cp);
                if (d6 >= 0.0 && d5 <= d6) q = T.c;
                else {
                    const double vb = d5 * d2 - d1 * d6;
                    if (vb <= 0.0 && d2 >= 0.0 && d6 <= 0.0) q = T.a + (d2 / (d2 - d6)) * ac;
                    else {
                        const double va = d3 * d6 - d5 * d4;
                        if (va <= 0.0 && (d4 - d3) >= 0.0 && (d5 - d6) >= 0.0) q = T.b + ((d4 - d3) / ((d4 - d3) + (d5 - d6))) * (T.c - T.b);
                        else {
                            const double den = 1.0 / (va + vb + vc);
                            q = T.a + (vb * den) * ab + (vc * den) * ac;
                        }
                    }
                }
            }
        }
    }
    w = q - p;
    return dot(w, w);
}

// does the segment p + t d (t in [0,1]) cross the triangle T?  (Moeller-Trumbore)
__device__ __forceinline__ bool seg_hits_tri(V3 p, V3 d, const Tri &T)
{
    const V3 e1 = T.b - T.a, e2 = T.c - T.a, h = cross(d, e2);
    const double det = dot(e1, h);
    if (det == 0.0) return false;                 // parallel (coplanar contact is found by the distances)
    const double inv = 1.0 / det;
    const V3 s = p - T.a;
    const double u = inv * dot(s, h);
    if (u < 0.0 || u > 1.0) return false;
    const V3 q = cross(s, e1);
    const double v = inv * dot(d, q);
    if (v < 0.0 || u + v > 1.0) return false;
    const double t = inv * dot(e2, q);
    return t >= 0.0 && t <= 1.0;
}

// TRITRIDISTANCE(TF, TC): shortest distance of two triangles (0 if they intersect) and the shortest vector
// dx = (point of TC) - (point of TF)
__device__ double tritri(const Tri &TF, const Tri &TC, V3 &dx)
{
    const V3 fv[3] = { TF.a, TF.b, TF.c }, cv[3] = { TC.a, TC.b, TC.c };
    double best = INFINITY;
    dx = v3(0.0, 0.0, 0.0);
    bool hit = false;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const V3 p1 = fv[i], d1 = fv[(i + 1) % 3] - fv[i];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            V3 w;
            const double d2 = seg_seg(p1, d1, cv[j], cv[(j + 1) % 3] - cv[j], w);
            if (d2 < best) { best = d2; dx = w; }
        }
        hit = hit || seg_hits_tri(p1, d1, TC);
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        V3 w;
        double d2 = pt_tri(fv[i], TC, w);                    // w = (on TC) - (vertex of TF)
        if (d2 < best) { best = d2; dx = w; }
        d2 = pt_tri(cv[i], TF, w);                           // w = (on TF) - (vertex of TC)
        if (d2 < best) { best = d2; dx = v3(-w.x, -w.y, -w.z); }
        hit = hit || seg_hits_tri(cv[i], cv[(i + 1) % 3] - cv[i], TF);
    }
    if (hit) { dx = v3(0.0, 0.0, 0.0); return 0.0; }
    return sqrt(best);
}

// corner triangles (i = 0, 1) of a 9-node patch given by its node pointers: (n0, n2, n8), (n0, n8, n6)
struct Patch { V3 n[9]; };
__device__ __forceinline__ Tri corner_tri(const Patch &P, int i) { Tri t; t.a = P.n[0]; t.b = i ? P.n[8] : P.n[2]; t.c = i ? P.n[6] : P.n[8]; return t; }
// triangle j of sub-quad (M, N) of the 2 x 2 grid (Fig. 11); index 2 (M + 2 N) + j
__device__ __forceinline__ Tri grid_tri(const Patch &P, int idx)
{
    const int j = idx & 1, M = (idx >> 1) & 1, N = idx >> 2;
    const V3 p00 = P.n[M + 3 * N], p10 = P.n[M + 1 + 3 * N], p11 = P.n[M + 1 + 3 * (N + 1)], p01 = P.n[M + 3 * (N + 1)];
    Tri t; t.a = p00; t.b = j ? p11 : p10; t.c = j ? p01 : p11;
    return t;
}

__device__ __forceinline__ void load_face(const double *face_nodes, int f, Patch &P)
{
    const double *X = face_nodes + (size_t)f * 27;
#pragma unroll
    for (int m = 0; m < 9; ++m) P.n[m] = ldv(X + 3 * m);
}
// boundary patch k of element e (node table of the narrow phase: base + sa a + sb b)
__device__ __forceinline__ void load_elem_patch(const double *xyz, const int *conn, int e, int k, Patch &P)
{
    const int nbase = k == 1 ? 2 : (k == 3 ? 6 : (k == 5 ? 18 : 0)), sa = k < 2 ? 3 : 1, sb = k < 4 ? 9 : 3;
    const int *cn = conn + (size_t)e * 27;
#pragma unroll
    for (int m = 0; m < 9; ++m) P.n[m] = ldv(xyz + (size_t)__ldg(cn + nbase + sa * (m % 3) + sb * (m / 3)) * 3);
}

} // namespace dcp

// per band element: 16 kept faces (original ids; -1 = none), their A.3 distance and corner; the 4 kept; A.4 results
struct PmWork {
    int *sel1;        // [max_band][16]
    double *d1;       // [max_band][16]   A.3 distance
    int *corner;      // [max_band][16]
    int *sel2;        // [max_band][4]    index j into sel1
    double *d2;       // [max_band][4][3] A.4 distance per element face q
    double *v2;       // [max_band][4][3][3] shortest vectors
};

__global__ void __launch_bounds__(128) k_pm_rank(const DcScalars *S, const double *__restrict__ xyz, const int *__restrict__ conn,
                                                 const int *__restrict__ band_elem, const long long *__restrict__ band_start,
                                                 const int *__restrict__ band_cnt, const int *__restrict__ pair_face,
                                                 const int *__restrict__ fperm, const double *__restrict__ face_nodes, PmWork W)
{
    pdl_start();
    if (S->status & DC_STATUS_INVALID) return;
    using namespace dcp;
    const int n_band = min(S->n_band, S->max_band);
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < n_band; b += gridDim.x * blockDim.x) {
        const int e = band_elem[b];
        // corner nodes c = i + 2 j + 4 k -> hex nodes 0, 2, 6, 8, 18, 20, 24, 26
        V3 X8[8];
        V3 m = v3(0.0, 0.0, 0.0);
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int node = 2 * (c & 1) + 6 * ((c >> 1) & 1) + 18 * (c >> 2);
            X8[c] = ldv(xyz + (size_t)__ldg(conn + (size_t)e * 27 + node) * 3);
            m = v3(add(m.x, X8[c].x), add(m.y, X8[c].y), add(m.z, X8[c].z));
        }
        m = v3(m.x / 8.0, m.y / 8.0, m.z / 8.0);
        // covariance matrix of the corner nodes and its eigenvectors: cyclic Jacobi, sweep order (0,1), (0,2), (1,2),
        // 8 sweeps from the identity (reading PM2)
        double A[3][3] = { { 0, 0, 0 }, { 0, 0, 0 }, { 0, 0, 0 } }, Vv[3][3] = { { 1, 0, 0 }, { 0, 1, 0 }, { 0, 0, 1 } };
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const double d[3] = { sub(X8[c].x, m.x), sub(X8[c].y, m.y), sub(X8[c].z, m.z) };
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int bb = 0; bb < 3; ++bb) A[a][bb] = add(A[a][bb], mul(d[a], d[bb]));
        }
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int bb = 0; bb < 3; ++bb) A[a][bb] = A[a][bb] / 8.0;
        for (int sweep = 0; sweep < 8; ++sweep)
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                const int p = r == 2 ? 1 : 0, q = r == 0 ? 1 : 2;
                if (A[p][q] == 0.0) continue;
                const double theta = __ddiv_rn(sub(A[q][q], A[p][p]), mul(2.0, A[p][q]));
                const double t = __ddiv_rn(theta >= 0.0 ? 1.0 : -1.0, add(fabs(theta), __dsqrt_rn(add(mul(theta, theta), 1.0))));
                const double c = __ddiv_rn(1.0, __dsqrt_rn(add(mul(t, t), 1.0))), s = mul(t, c);
#pragma unroll
                for (int k = 0; k < 3; ++k) { const double akp = A[k][p], akq = A[k][q]; A[k][p] = sub(mul(c, akp), mul(s, akq)); A[k][q] = add(mul(s, akp), mul(c, akq)); }
#pragma unroll
                for (int k = 0; k < 3; ++k) { const double apk = A[p][k], aqk = A[q][k]; A[p][k] = sub(mul(c, apk), mul(s, aqk)); A[q][k] = add(mul(s, apk), mul(c, aqk)); }
#pragma unroll
                for (int k = 0; k < 3; ++k) { const double vkp = Vv[k][p], vkq = Vv[k][q]; Vv[k][p] = sub(mul(c, vkp), mul(s, vkq)); Vv[k][q] = add(mul(s, vkp), mul(c, vkq)); }
            }
        V3 ax[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) ax[a] = v3(Vv[0][a], Vv[1][a], Vv[2][a]);
        double lo[3] = { INFINITY, INFINITY, INFINITY }, hi[3] = { -INFINITY, -INFINITY, -INFINITY };
#pragma unroll
        for (int c = 0; c < 8; ++c)
#pragma unroll
            for (int a = 0; a < 3; ++a) { const double y = dot_nc(ax[a], X8[c]); lo[a] = y < lo[a] ? y : lo[a]; hi[a] = y > hi[a] ? y : hi[a]; }
        // A.1 on every candidate, insertion into the 16 nearest (distance, then original face id)
        double kd[PM_NF1]; int kf[PM_NF1];
        int nk = 0;
        const long long p0 = band_start[b];
        const int np = band_cnt[b];
        for (int pl = 0; pl < np; ++pl) {
            const int f = __ldg(fperm + __ldg(pair_face + p0 + pl));
            const double *X = face_nodes + (size_t)f * 27;
            const V3 F4[4] = { ldv(X), ldv(X + 6), ldv(X + 24), ldv(X + 18) };
            double flo[3] = { INFINITY, INFINITY, INFINITY }, fhi[3] = { -INFINITY, -INFINITY, -INFINITY };
            V3 fcg = v3(0.0, 0.0, 0.0);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                fcg = v3(add(fcg.x, mul(0.25, F4[i].x)), add(fcg.y, mul(0.25, F4[i].y)), add(fcg.z, mul(0.25, F4[i].z)));
#pragma unroll
                for (int a = 0; a < 3; ++a) { const double y = dot_nc(ax[a], F4[i]); flo[a] = y < flo[a] ? y : flo[a]; fhi[a] = y > fhi[a] ? y : fhi[a]; }
            }
            const V3 dc = v3(sub(fcg.x, m.x), sub(fcg.y, m.y), sub(fcg.z, m.z));
            double D = 0.0;                                   // BOUNDINGBOXDIST (A.2)
#pragma unroll
            for (int a = 0; a < 3; ++a)
                if (fhi[a] < lo[a] || hi[a] < flo[a]) { const double g = fmax(sub(lo[a], fhi[a]), sub(flo[a], hi[a])); D = add(D, mul(g, g)); }
            const double dist = add(mul(0.01, __dsqrt_rn(dot_nc(dc, dc))), __dsqrt_rn(D));
            // insertion
            int pos = nk;
            while (pos > 0 && (dist < kd[pos - 1] || (dist == kd[pos - 1] && f < kf[pos - 1]))) --pos;
            if (pos < PM_NF1) {
                const int last = nk < PM_NF1 ? nk : PM_NF1 - 1;
                for (int i = last; i > pos; --i) { kd[i] = kd[i - 1]; kf[i] = kf[i - 1]; }
                kd[pos] = dist; kf[pos] = f;
                if (nk < PM_NF1) ++nk;
            }
        }
        for (int j = 0; j < PM_NF1; ++j) W.sel1[(size_t)b * PM_NF1 + j] = j < nk ? kf[j] : -1;
    }
}

__global__ void __launch_bounds__(128) k_pm_pass1(const DcScalars *S, const double *__restrict__ xyz, const int *__restrict__ conn,
                                                  const int *__restrict__ band_elem, const double *__restrict__ face_nodes, PmWork W)
{
    pdl_start();
    if (S->status & DC_STATUS_INVALID) return;
    using namespace dcp;
    const long long n = (long long)min(S->n_band, S->max_band) * PM_NF1;
    const double tol = S->tau;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(i / PM_NF1);
        const int f = W.sel1[i];
        if (f < 0) { W.d1[i] = INFINITY; W.corner[i] = 0; continue; }
        const int e = band_elem[b];
        Patch Q;
        load_face(face_nodes, f, Q);
        const V3 fcg = 0.25 * (Q.n[0] + Q.n[2] + Q.n[8] + Q.n[6]);
        double Dc = INFINITY; int c = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int node = 2 * (k & 1) + 6 * ((k >> 1) & 1) + 18 * (k >> 2);
            const V3 d = ldv(xyz + (size_t)__ldg(conn + (size_t)e * 27 + node) * 3) - fcg;
            const double D = sqrt(dot(d, d));
            if (D < Dc) { Dc = D; c = k; }
        }
        double Dmin = INFINITY;
        for (int q = 0; q < 3; ++q) {
            const int k = q == 0 ? (c & 1) : (q == 1 ? 2 + ((c >> 1) & 1) : 4 + ((c >> 2) & 1));
            Patch P;
            load_elem_patch(xyz, conn, e, k, P);
            for (int ii = 0; ii < 2; ++ii)
                for (int jj = 0; jj < 2; ++jj) {
                    V3 dx;
                    const double D = tritri(corner_tri(Q, jj), corner_tri(P, ii), dx);
                    if (D < Dmin) Dmin = D;
                }
        }
        if (Dmin < tol) Dmin = 0.0;
        W.d1[i] = Dmin; W.corner[i] = c;
    }
}

__global__ void __launch_bounds__(128) k_pm_select(const DcScalars *S, PmWork W)
{
    pdl_start();
    if (S->status & DC_STATUS_INVALID) return;
    const int n_band = min(S->n_band, S->max_band);
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < n_band; b += gridDim.x * blockDim.x) {
        double kd[PM_NF2]; int kf[PM_NF2], kj[PM_NF2];
        int nk = 0;
        for (int j = 0; j < PM_NF1; ++j) {
            const int f = W.sel1[(size_t)b * PM_NF1 + j];
            if (f < 0) break;
            const double d = W.d1[(size_t)b * PM_NF1 + j];
            int pos = nk;
            while (pos > 0 && (d < kd[pos - 1] || (d == kd[pos - 1] && f < kf[pos - 1]))) --pos;
            if (pos < PM_NF2) {
                const int last = nk < PM_NF2 ? nk : PM_NF2 - 1;
                for (int i = last; i > pos; --i) { kd[i] = kd[i - 1]; kf[i] = kf[i - 1]; kj[i] = kj[i - 1]; }
                kd[pos] = d; kf[pos] = f; kj[pos] = j;
                if (nk < PM_NF2) ++nk;
            }
        }
        for (int j = 0; j < PM_NF2; ++j) W.sel2[(size_t)b * PM_NF2 + j] = j < nk ? kj[j] : -1;
    }
}

__global__ void __launch_bounds__(128) k_pm_pass2(const DcScalars *S, const double *__restrict__ xyz, const int *__restrict__ conn,
                                                  const int *__restrict__ band_elem, const double *__restrict__ face_nodes, PmWork W)
{
    pdl_start();
    if (S->status & DC_STATUS_INVALID) return;
    using namespace dcp;
    const long long n = (long long)min(S->n_band, S->max_band) * PM_NF2 * 3;
    const double tol = S->tau;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(i / (PM_NF2 * 3)), j = (int)((i / 3) % PM_NF2), q = (int)(i % 3);
        const int j1 = W.sel2[(size_t)b * PM_NF2 + j];
        if (j1 < 0) { W.d2[i] = INFINITY; continue; }
        const int f = W.sel1[(size_t)b * PM_NF1 + j1], c = W.corner[(size_t)b * PM_NF1 + j1];
        const int e = band_elem[b];
        const int k = q == 0 ? (c & 1) : (q == 1 ? 2 + ((c >> 1) & 1) : 4 + ((c >> 2) & 1));
        Patch Q, P;
        load_face(face_nodes, f, Q);
        load_elem_patch(xyz, conn, e, k, P);
        double Dbest = INFINITY;
        V3 vbest = v3(0.0, 0.0, 0.0);
        for (int T = 0; T < 8; ++T) {
            const Tri TC = grid_tri(P, T);
            double Dmin = INFINITY;
            V3 dxmin = v3(0.0, 0.0, 0.0);
            for (int t = 0; t < 8; ++t) {
                V3 dx;
                const double D = tritri(grid_tri(Q, t), TC, dx);
                if (D < tol) { Dmin = 0.0; dxmin = v3(0.0, 0.0, 0.0); break; }
                if (D < Dmin) { Dmin = D; dxmin = dx; }
            }
            if (Dmin < Dbest) { Dbest = Dmin; vbest = dxmin; }
        }
        W.d2[i] = Dbest;
        W.v2[3 * i] = vbest.x; W.v2[3 * i + 1] = vbest.y; W.v2[3 * i + 2] = vbest.z;
    }
}

__global__ void __launch_bounds__(128) k_pm_decide(DcScalars *S, const int *__restrict__ band_elem, const double *__restrict__ face_nodes,
                                                   PmWork W, signed char *__restrict__ labels, double *__restrict__ sdist)
{
    pdl_start();
    if (S->status & DC_STATUS_INVALID) return;
    using namespace dcp;
    const int n_band = min(S->n_band, S->max_band);
    const double tol = S->tau, d_band = S->d_band;
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < n_band; b += gridDim.x * blockDim.x) {
        double DF[PM_NF2]; int FF[PM_NF2]; V3 VF[PM_NF2];
        int n2 = 0;
        for (int j = 0; j < PM_NF2; ++j) {
            const int j1 = W.sel2[(size_t)b * PM_NF2 + j];
            if (j1 < 0) break;
            double D = INFINITY; V3 v = v3(0.0, 0.0, 0.0);
            for (int q = 0; q < 3; ++q) {
                const size_t i = ((size_t)b * PM_NF2 + j) * 3 + q;
                if (W.d2[i] < D) { D = W.d2[i]; v = v3(W.v2[3 * i], W.v2[3 * i + 1], W.v2[3 * i + 2]); }
            }
            DF[n2] = D; FF[n2] = W.sel1[(size_t)b * PM_NF1 + j1]; VF[n2] = v; ++n2;
        }
        if (n2 == 0) continue;
        int jb = 0;
        for (int j = 1; j < n2; ++j) if (DF[j] < DF[jb] || (DF[j] == DF[jb] && FF[j] < FF[jb])) jb = j;
        const int e = band_elem[b];
        const double D = DF[jb];
        if (D <= 0.0) { labels[e] = DC_CUT; sdist[e] = 0.0; continue; }
        // L215: the normals of the faces at approximately the same distance (within tol) are averaged
        V3 navg = v3(0.0, 0.0, 0.0);
        for (int j = 0; j < n2; ++j)
            if (DF[j] <= D + tol) {
                const double *X = face_nodes + (size_t)FF[j] * 27;
                const V3 nrm = cross(ldv(X + 24) - ldv(X), ldv(X + 18) - ldv(X + 6));
                const double nn = sqrt(dot(nrm, nrm));
                if (nn > 0.0) navg = navg + (1.0 / nn) * nrm;
            }
        const bool hole = dot(VF[jb], navg) < 0.0;
        const double dd = D < d_band ? D : d_band;
        // (beyond the band the sign comes from the flood fill, as in the exact mode)
        if (D <= d_band) { labels[e] = hole ? DC_HOLE : DC_NORMAL; sdist[e] = hole ? -dd : dd; }
    }
}
