/* paper_oracle.c -- CPU ORACLE of the paper's own approximate direct cut (PAPER.md 4.2 L191-L215, Appendix A
 * L670-L845), SURVEY.md 8(f) NEXT-3.  TEST INFRASTRUCTURE ONLY (see dc_oracle.c): plain, slow, single-threaded,
 * one element after the other, in the paper's order and notation; shares no code with the CUDA path.
 *
 * What it computes, per element E with at least one candidate face (readings PM1-PM8 of DESIGN.md):
 *   preprocessing (L195-L197): OBB of the 8 CORNER nodes (axes = eigenvectors of their covariance matrix), corner-node
 *     centroids of the element and of every face;
 *   A.1 (L672-L687): Distance(E,F) = .01 |f_cg - e_cg| + BOUNDINGBOXDIST(AABB of the face's corner nodes in the OBB
 *     axes, OBB extents); keep the N_F^1 = 16 nearest faces (L209);
 *   A.3 (L711-L783): nearest corner c of E to f_cg; the 3 element faces touching c and the cutting face, each as two
 *     linear triangles of its corner nodes; D = min TRITRIDISTANCE, 0 below tol; keep the N_F^2 = 4 nearest (L213);
 *   A.4 (L785-L845): the same 3 element faces and the cutting face as 2 x 2 grids of linear quads of ALL their nodes,
 *     two triangles each (Fig. 11); per element triangle T the nearest of the face's 8 triangles, 0 below tol;
 *   final (L215): the nearest face; sign of the dot product of the shortest vector with the face's outward normal,
 *     the normals of faces at approximately the same distance averaged.
 * TRITRIDISTANCE is dc_oracle.c's orc_tri_tri_dist (pinned there, P3); BOUNDINGBOXDIST its orc_box_dist (A.2, P2).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

double orc_box_dist(const double *B1, const double *B2);
double orc_tri_tri_dist(const double *A, const double *B, double *wa, double *wb);
void orc_lagrange_to_bezier(const double *X, double *B);
void orc_hex_face_nodes(int k, int *ids);

#define PM_NF1 16
#define PM_NF2 4
#define PM_FLAG_FAR 4            /* no candidate face: not computed (label -1) */

static const int pm_corner_node[8] = { 0, 2, 6, 8, 18, 20, 24, 26 };   /* corner c = i + 2 j + 4 k */

/* Eigenvectors of the symmetric 3x3 matrix A by cyclic Jacobi (reading PM2: sweep order (0,1), (0,2), (1,2), 8
 * sweeps from the identity; a rotation is skipped when the off-diagonal entry is exactly 0).  R rows = axes. */
void orc_pm_eig3(const double *Ain /*[9]*/, double *R /*[9]*/)
{
    double A[3][3], V[3][3] = { {1,0,0}, {0,1,0}, {0,0,1} };
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) A[i][j] = Ain[3*i+j];
    const int P[3] = { 0, 0, 1 }, Q[3] = { 1, 2, 2 };
    for (int sweep = 0; sweep < 8; ++sweep)
        for (int r = 0; r < 3; ++r) {
            int p = P[r], q = Q[r];
            if (A[p][q] == 0.0) continue;
            double theta = (A[q][q] - A[p][p]) / (2.0 * A[p][q]);
            double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
            double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
            for (int k = 0; k < 3; ++k) {          /* A <- A J */
                double akp = A[k][p], akq = A[k][q];
                A[k][p] = c * akp - s * akq; A[k][q] = s * akp + c * akq;
            }
            for (int k = 0; k < 3; ++k) {          /* A <- J^T A */
                double apk = A[p][k], aqk = A[q][k];
                A[p][k] = c * apk - s * aqk; A[q][k] = s * apk + c * aqk;
            }
            for (int k = 0; k < 3; ++k) {          /* V <- V J */
                double vkp = V[k][p], vkq = V[k][q];
                V[k][p] = c * vkp - s * vkq; V[k][q] = s * vkp + c * vkq;
            }
        }
    for (int a = 0; a < 3; ++a) for (int k = 0; k < 3; ++k) R[3*a+k] = V[k][a];    /* axis a = column a of V */
}

/* OBB of the 8 corner nodes X8 [8][3] (L195): R rows = axes, ext = min/max of the corner nodes along them,
 * ecg = their centroid (L196). */
void orc_pm_obb(const double *X8, double *R, double *ext, double *ecg)
{
    double m[3] = { 0, 0, 0 }, Cv[9] = { 0 };
    for (int i = 0; i < 8; ++i) for (int k = 0; k < 3; ++k) m[k] += X8[3*i+k];
    for (int k = 0; k < 3; ++k) { m[k] /= 8.0; ecg[k] = m[k]; }
    for (int i = 0; i < 8; ++i)
        for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
            Cv[3*a+b] += (X8[3*i+a] - m[a]) * (X8[3*i+b] - m[b]);
    for (int a = 0; a < 9; ++a) Cv[a] /= 8.0;
    orc_pm_eig3(Cv, R);
    for (int a = 0; a < 3; ++a) { ext[a] = INFINITY; ext[3+a] = -INFINITY; }
    for (int i = 0; i < 8; ++i)
        for (int a = 0; a < 3; ++a) {
            double y = R[3*a] * X8[3*i] + R[3*a+1] * X8[3*i+1] + R[3*a+2] * X8[3*i+2];
            if (y < ext[a]) ext[a] = y;
            if (y > ext[3+a]) ext[3+a] = y;
        }
}

/* Algorithm A.1 (L672-L687).  F4: the face's 4 corner nodes [4][3]. */
double orc_pm_a1(const double *R, const double *ext, const double *ecg, const double *F4)
{
    double bf[6] = { INFINITY, INFINITY, INFINITY, -INFINITY, -INFINITY, -INFINITY }, fcg[3] = { 0, 0, 0 };
    for (int i = 0; i < 4; ++i) {
        for (int k = 0; k < 3; ++k) fcg[k] += 0.25 * F4[3*i+k];
        for (int a = 0; a < 3; ++a) {
            double y = R[3*a] * F4[3*i] + R[3*a+1] * F4[3*i+1] + R[3*a+2] * F4[3*i+2];
            if (y < bf[a]) bf[a] = y;
            if (y > bf[3+a]) bf[3+a] = y;
        }
    }
    double d[3] = { fcg[0] - ecg[0], fcg[1] - ecg[1], fcg[2] - ecg[2] };
    double dxc = sqrt(d[0]*d[0] + d[1]*d[1] + d[2]*d[2]);
    return 0.01 * dxc + orc_box_dist(bf, ext);
}

/* TRITRIDISTANCE with the shortest vector dx = (point of TC) - (point of TF) */
static double tritri(const double *TF, const double *TC, double *dx)
{
    double wf[3], wc[3];
    double D = orc_tri_tri_dist(TF, TC, wf, wc);
    for (int k = 0; k < 3; ++k)
        dx[k] = (wc[0]*TC[k] + wc[1]*TC[3+k] + wc[2]*TC[6+k]) - (wf[0]*TF[k] + wf[1]*TF[3+k] + wf[2]*TF[6+k]);
    return D;
}

/* the two triangles of the quad (p00, p10, p11, p01): (p00,p10,p11), (p00,p11,p01)  (reading PM5) */
static void quad_tris(const double *p00, const double *p10, const double *p11, const double *p01, double T[2][9])
{
    memcpy(T[0], p00, 24); memcpy(T[0] + 3, p10, 24); memcpy(T[0] + 6, p11, 24);
    memcpy(T[1], p00, 24); memcpy(T[1] + 3, p11, 24); memcpy(T[1] + 6, p01, 24);
}

/* 9-node patch X [9][3] (m = i + 3 j) -> its 2 corner triangles */
static void patch_corner_tris(const double *X, double T[2][9])
{
    quad_tris(X, X + 3*2, X + 3*8, X + 3*6, T);
}
/* 9-node patch -> the 8 triangles of its 2 x 2 grid of linear quads (Fig. 11), sub-quad (M,N), triangle j: index 2 (M + 2 N) + j */
static void patch_grid_tris(const double *X, double T[8][9])
{
    for (int N = 0; N < 2; ++N) for (int M = 0; M < 2; ++M) {
        const double *p00 = X + 3*(M + 3*N), *p10 = X + 3*(M + 1 + 3*N), *p11 = X + 3*(M + 1 + 3*(N + 1)), *p01 = X + 3*(M + 3*(N + 1));
        quad_tris(p00, p10, p11, p01, &T[2*(M + 2*N)]);
    }
}

typedef struct { double d; int f; } pm_rank;
static int pm_cmp(const void *a, const void *b)
{
    const pm_rank *x = (const pm_rank *)a, *y = (const pm_rank *)b;
    if (x->d < y->d) return -1;
    if (x->d > y->d) return 1;
    return (x->f > y->f) - (x->f < y->f);
}

typedef struct { long long n_a1, n_tritri, n_cut, n_hole, n_normal, n_far; double l_ref, tol, d_band; } pm_stats;

/* The paper's approximate cut for elements [e_begin, e_end).  d_band > 0 and l_ref > 0 are given by the caller (the
 * exact oracle's values).  Candidate faces of an element (reading PM1): Bezier box within d_band + 2 tol of the
 * element's Bezier box (the paper's hole-map / bounding-box filters, L177-L191, replaced by the exact pass's own).
 * labels -1 / flag PM_FLAG_FAR for elements without candidates.  nearest: face id of the minimum. */
int orc_paper_classify(long long n_nodes, const double *xyz, long long n_elem, const int *conn27,
                       long long n_face, const double *faces, double d_band, double l_ref,
                       long long e_begin, long long e_end,
                       signed char *labels, double *sdist, int *nearest, unsigned char *flags, pm_stats *st)
{
    (void)n_nodes; (void)n_elem;
    pm_stats S; memset(&S, 0, sizeof S);
    const double tol = 1e-7 * l_ref, reach = d_band + 2.0 * tol + 1e-9 * l_ref;
    S.l_ref = l_ref; S.tol = tol; S.d_band = d_band;
    double *fbox = (double *)malloc(sizeof(double) * 6 * (size_t)n_face);
    double *fcg = (double *)malloc(sizeof(double) * 3 * (size_t)n_face);
    double *fnrm = (double *)malloc(sizeof(double) * 3 * (size_t)n_face);
    pm_rank *rk = (pm_rank *)malloc(sizeof(pm_rank) * (size_t)n_face);
    if (!fbox || !fcg || !fnrm || !rk) { free(fbox); free(fcg); free(fnrm); free(rk); return -1; }
    for (long long f = 0; f < n_face; ++f) {
        const double *X = faces + 27*f;
        double B[27];
        orc_lagrange_to_bezier(X, B);
        for (int c = 0; c < 3; ++c) { fbox[6*f+c] = INFINITY; fbox[6*f+3+c] = -INFINITY; }
        for (int m = 0; m < 9; ++m) for (int c = 0; c < 3; ++c) {
            if (B[3*m+c] < fbox[6*f+c]) fbox[6*f+c] = B[3*m+c];
            if (B[3*m+c] > fbox[6*f+3+c]) fbox[6*f+3+c] = B[3*m+c];
        }
        const double *c00 = X, *c10 = X + 6, *c11 = X + 24, *c01 = X + 18;
        for (int k = 0; k < 3; ++k) fcg[3*f+k] = 0.25 * (c00[k] + c10[k] + c11[k] + c01[k]);
        /* outward normal from the corner nodes: (c11 - c00) x (c01 - c10), unit (reading PM7) */
        double a[3] = { c11[0]-c00[0], c11[1]-c00[1], c11[2]-c00[2] }, b[3] = { c01[0]-c10[0], c01[1]-c10[1], c01[2]-c10[2] };
        double n[3] = { a[1]*b[2]-a[2]*b[1], a[2]*b[0]-a[0]*b[2], a[0]*b[1]-a[1]*b[0] };
        double nn = sqrt(n[0]*n[0] + n[1]*n[1] + n[2]*n[2]);
        for (int k = 0; k < 3; ++k) fnrm[3*f+k] = nn > 0.0 ? n[k] / nn : 0.0;
    }
    int fid[6][9];
    for (int k = 0; k < 6; ++k) orc_hex_face_nodes(k, fid[k]);

    for (long long e = e_begin; e < e_end; ++e) {
        long long o = e - e_begin;
        double PX[6][27], ebox[6] = { INFINITY, INFINITY, INFINITY, -INFINITY, -INFINITY, -INFINITY }, X8[24];
        for (int k = 0; k < 6; ++k) {
            double B[27];
            for (int m = 0; m < 9; ++m) {
                const double *p = xyz + 3 * (long long)conn27[27*e + fid[k][m]];
                PX[k][3*m] = p[0]; PX[k][3*m+1] = p[1]; PX[k][3*m+2] = p[2];
            }
            orc_lagrange_to_bezier(PX[k], B);
            for (int m = 0; m < 9; ++m) for (int c = 0; c < 3; ++c) {
                if (B[3*m+c] < ebox[c]) ebox[c] = B[3*m+c];
                if (B[3*m+c] > ebox[3+c]) ebox[3+c] = B[3*m+c];
            }
        }
        for (int i = 0; i < 8; ++i) {
            const double *p = xyz + 3 * (long long)conn27[27*e + pm_corner_node[i]];
            X8[3*i] = p[0]; X8[3*i+1] = p[1]; X8[3*i+2] = p[2];
        }
        double R[9], ext[6], ecg[3];
        orc_pm_obb(X8, R, ext, ecg);
        /* A.1 over the candidates, keep the N_F^1 nearest */
        long long nc = 0;
        for (long long f = 0; f < n_face; ++f) {
            if (orc_box_dist(ebox, fbox + 6*f) > reach) continue;
            const double *X = faces + 27*f;
            double F4[12];
            memcpy(F4, X, 24); memcpy(F4 + 3, X + 6, 24); memcpy(F4 + 6, X + 24, 24); memcpy(F4 + 9, X + 18, 24);
            rk[nc].d = orc_pm_a1(R, ext, ecg, F4); rk[nc].f = (int)f; nc++;
            S.n_a1++;
        }
        labels[o] = -1; sdist[o] = 0.0; if (nearest) nearest[o] = -1; if (flags) flags[o] = 0;
        if (nc == 0) { if (flags) flags[o] = PM_FLAG_FAR; S.n_far++; continue; }
        qsort(rk, (size_t)nc, sizeof(pm_rank), pm_cmp);
        int n1 = nc < PM_NF1 ? (int)nc : PM_NF1;
        /* A.3: nearest corner, 3 faces x 2 x 2 corner triangles */
        pm_rank r2[PM_NF1]; int corner[PM_NF1];
        for (int j = 0; j < n1; ++j) {
            int f = rk[j].f;
            double Dc = INFINITY; int c = 0;
            for (int i = 0; i < 8; ++i) {
                double d[3] = { X8[3*i] - fcg[3*f], X8[3*i+1] - fcg[3*f+1], X8[3*i+2] - fcg[3*f+2] };
                double D = sqrt(d[0]*d[0] + d[1]*d[1] + d[2]*d[2]);
                if (D < Dc) { Dc = D; c = i; }
            }
            const int flist[3] = { (c & 1), 2 + ((c >> 1) & 1), 4 + ((c >> 2) & 1) };
            double TF[2][9], Dmin = INFINITY, dx[3];
            patch_corner_tris(faces + 27*(long long)f, TF);
            for (int q = 0; q < 3; ++q) {
                double TC[2][9];
                patch_corner_tris(PX[flist[q]], TC);
                for (int i = 0; i < 2; ++i) for (int jj = 0; jj < 2; ++jj) {
                    double D = tritri(TF[jj], TC[i], dx);
                    S.n_tritri++;
                    if (D < Dmin) Dmin = D;
                }
            }
            if (Dmin < tol) Dmin = 0.0;
            r2[j].d = Dmin; r2[j].f = f; corner[j] = c;
        }
        /* keep the N_F^2 nearest (the corner travels with its face) */
        int ord[PM_NF1];
        for (int j = 0; j < n1; ++j) ord[j] = j;
        for (int a = 0; a < n1; ++a) for (int b = a + 1; b < n1; ++b)
            if (pm_cmp(&r2[ord[b]], &r2[ord[a]]) < 0) { int t = ord[a]; ord[a] = ord[b]; ord[b] = t; }
        int n2 = n1 < PM_NF2 ? n1 : PM_NF2;
        /* A.4: 3 faces x 8 element triangles against the face's 8 triangles */
        double DF[PM_NF2], VF[PM_NF2][3]; int FF[PM_NF2];
        for (int j = 0; j < n2; ++j) {
            int f = r2[ord[j]].f, c = corner[ord[j]];
            const int flist[3] = { (c & 1), 2 + ((c >> 1) & 1), 4 + ((c >> 2) & 1) };
            double TF[8][9];
            patch_grid_tris(faces + 27*(long long)f, TF);
            double Dbest = INFINITY, vbest[3] = { 0, 0, 0 };
            for (int q = 0; q < 3; ++q) {
                double TC[8][9];
                patch_grid_tris(PX[flist[q]], TC);
                for (int T = 0; T < 8; ++T) {
                    double Dmin = INFINITY, dxmin[3] = { 0, 0, 0 };
                    for (int t = 0; t < 8; ++t) {
                        double dx[3];
                        double D = tritri(TF[t], TC[T], dx);
                        S.n_tritri++;
                        if (D < tol) { Dmin = 0.0; dxmin[0] = dxmin[1] = dxmin[2] = 0.0; break; }
                        if (D < Dmin) { Dmin = D; dxmin[0] = dx[0]; dxmin[1] = dx[1]; dxmin[2] = dx[2]; }
                    }
                    if (Dmin < Dbest) { Dbest = Dmin; vbest[0] = dxmin[0]; vbest[1] = dxmin[1]; vbest[2] = dxmin[2]; }
                }
            }
            DF[j] = Dbest; FF[j] = f; VF[j][0] = vbest[0]; VF[j][1] = vbest[1]; VF[j][2] = vbest[2];
        }
        /* final (L215): nearest face; normals of faces at approximately the same distance (within tol) averaged */
        int jb = 0;
        for (int j = 1; j < n2; ++j) if (DF[j] < DF[jb] || (DF[j] == DF[jb] && FF[j] < FF[jb])) jb = j;
        double D = DF[jb];
        if (nearest) nearest[o] = FF[jb];
        if (D <= 0.0) { labels[o] = 2; sdist[o] = 0.0; S.n_cut++; continue; }
        double navg[3] = { 0, 0, 0 };
        for (int j = 0; j < n2; ++j) if (DF[j] <= D + tol) for (int k = 0; k < 3; ++k) navg[k] += fnrm[3*FF[j]+k];
        double dot = VF[jb][0]*navg[0] + VF[jb][1]*navg[1] + VF[jb][2]*navg[2];
        int hole = dot < 0.0;
        labels[o] = hole ? 0 : 1;
        double dd = D < d_band ? D : d_band;
        sdist[o] = hole ? -dd : dd;
        if (hole) S.n_hole++; else S.n_normal++;
    }
    free(fbox); free(fcg); free(fnrm); free(rk);
    if (st) *st = S;
    return 0;
}
