/*
 * dc.h -- C ABI of libdc: the direct-cut hole-cutting pass on one NVIDIA B200 (sm_100a).
 *
 * What the library computes (PAPER.md = arxiv 1711.07663; line numbers of /root/reference/PAPER.md):
 *   "rather than searching for all elements which intersect a cutting boundary, we instead have
 *    all elements calculate the (signed) minimum distance to the boundary ... to directly
 *    determine whether each element is inside, outside, or intersecting with the boundary"
 *   (section 4.2).  For every element e of ONE grid of 27-node quadratic hexahedra
 *   (tensor-product Lagrange map, Eq. 1, K = 2) and ONE closed, outward-oriented cutting
 *   surface of 9-node quadratic quadrilateral faces (L171-L175, L215):
 *       d_e   = min over faces f, boundary patches k of e, and (u,v),(s,t) in [-1,1]^2 of
 *               |P_{e,k}(u,v) - Q_f(s,t)|
 *       label = DC_CUT    if d_e <= tau_cut     (L151; A.3 L719/L773-L777, A.4 L815-L837)
 *               DC_HOLE   if (p* - q*) . n(q*) < 0 at the closest pair, n = Q_s x Q_t  (L151, L215)
 *               DC_NORMAL otherwise
 *       sdist = 0 for CUT, else +-min(d_e, d_band), + for NORMAL.
 *   Elements farther than d_band from the surface take their label from a flood fill over the
 *   face adjacency of non-CUT elements (the classical paint-fill, L143, Fig. 5), seeded by the
 *   elements inside the band.
 *
 * Conventions (paper silent; readings A1/A2):
 *   hex node  m = i + 3 j + 9 k  (xi fastest), reference nodes {-1, 0, +1};  quad node m = i + 3 j;
 *   element faces k = 0..5 <-> xi=-1, xi=+1, eta=-1, eta=+1, zeta=-1, zeta=+1;
 *   adj6[e][k] = element across face k, or -1.
 *
 * Memory: every pointer marked "dev" is a CUDA device pointer OWNED BY THE CALLER (allocated
 * e.g. with torch); "host" pointers are host memory (pinned for asynchronous copies).  The
 * library never allocates device memory: all scratch lives in the caller's workspace.
 * The context borrows xyz / conn27 / adj6 / workspace until dc_destroy and the face buffer
 * until the next dc_set_cut_surface.
 *
 * Errors: every call returns 0 (DC_OK) or a negative code; no exceptions, no global state.
 * dc_set_cut_surface / dc_classify only enqueue work on `stream` (a cudaStream_t passed as
 * void*) and never synchronise; conditions found on the device (pair-list overflow, ...)
 * are latched into dc_stats.status and returned by dc_get_stats, which synchronises.
 */
#ifndef DC_H_
#define DC_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* labels (int8).  0/1 follow the usual iblank hole/field convention; the paper's hole map uses
 * the same three values (L169). */
#define DC_HOLE 0
#define DC_NORMAL 1
#define DC_CUT 2

/* return codes */
#define DC_OK 0
#define DC_ERR_ARG (-1)         /* NULL / negative / inconsistent argument */
#define DC_ERR_WORKSPACE (-2)   /* workspace too small, or a device-side list overflowed */
#define DC_ERR_UNSUPPORTED (-3) /* device is not sm_100, or input violates a documented precondition */
#define DC_ERR_CUDA (-4)        /* a CUDA runtime call failed */
#define DC_ERR_STATE (-5)       /* call order: dc_classify before dc_set_cut_surface, ... */
#define DC_ERR_RESULT (-6)      /* a device-side consistency check failed (DC_STATUS_FILL_CONFLICT,
                                   DC_STATUS_SEEDLESS_OVERFLOW): labels were written but are not to be trusted */

/* dc_stats.status bits (device-side conditions) */
#define DC_STATUS_PAIR_OVERFLOW 1   /* candidate pair list exceeded max_pairs: results invalid */
#define DC_STATUS_QUEUE_OVERFLOW 2  /* narrow-phase work queue spill area exhausted: results invalid */
#define DC_STATUS_FILL_CONFLICT 4   /* a flood-fill component has seeds of both signs */
#define DC_STATUS_SEEDLESS_OVERFLOW 8 /* more seedless components than the library resolves (1024): dc_get_stats
                                         returns DC_ERR_RESULT */
#define DC_STATUS_BAND_OVERFLOW 16  /* more elements with candidate pairs than the workspace holds (max_pairs / 8,
                                       at least 65 536): results invalid; dc_stats.band_needed says how many there
                                       were -- size max_pairs >= 8 * band_needed */
#define DC_STATUS_SURFACE_SMALL 32  /* the whole cutting surface is smaller than an element (longest edge of its box <
                                       max element box diagonal / sqrt 3): a surface component may lie strictly inside
                                       one element, where the distance to the element's BOUNDARY patches is not the
                                       distance to the element (reading A7); dc_get_stats returns DC_ERR_UNSUPPORTED.
                                       Labels and distances are still those of the boundary-patch definition. */

/* dc_params.flags */
#define DC_FLAG_RECOMPUTE_BOXES 1   /* redo step S2 (element boxes from raw nodes) inside dc_classify
                                       instead of using the boxes cached by dc_create_grid */
#define DC_FLAG_PAPER_MODE 2        /* the paper's own APPROXIMATE cut for the elements with candidate faces, in place of the
                                       exact narrow phase (S5, S6): Algorithms A.1, A.3, A.4 with N_F^1 = 16
                                       and N_F^2 = 4 nearest faces kept (L209, L213), the nearest-corner 3-face shortcut (L213),
                                       linear triangles (Fig. 11) and the normal averaging of L215.  Labels and distances are
                                       those of that method (its linearisation error included): for comparison with the exact
                                       mode, not for parity with the exact oracle.  S4 and S7 are unchanged. */

#define DC_FLAG_EXACT_FAR 4         /* exact distance EVERYWHERE (reading A5's alternative, "d_band = infinity"; SURVEY.md 8(f)
                                       NEXT-4): after the banded cut and the flood fill, every element still clamped at
                                       +-d_band gets sdist = +-d_e -- the magnitude from the same narrow phase (S5) run on the
                                       faces whose box is within an attained upper bound of the element (nearest-bin walk
                                       over an octree of the face bins, so no N_e x N_f pair list), the sign from S7.  Labels
                                       are unchanged.  Runs in passes sized to the workspace and SYNCHRONISES the stream
                                       after each; dc_get_pairs is not available afterwards.  Costs tens of banded cuts
                                       (most elements are far, and far from a round body a hundred
                                       faces are about as near as the nearest).  Ignored with DC_FLAG_PAPER_MODE.
                                       A pass holds max_pairs / 6 pairs: DC_ERR_WORKSPACE (dc_get_stats) when ONE element
                                       has more candidate faces than that (pairs_needed says what max_pairs would do). */

#define DC_FLAG_GRAPH 8             /* dc_cut / dc_classify_host only: capture the launch sequence of the cut into a CUDA graph
                                       the first time it is asked for with these arguments (surface address and face count,
                                       parameters, output addresses, stream) and replay it afterwards; up to 64 graphs are
                                       kept per context, the least recently used one goes.  The surface's contents may
                                       change between calls.  Needs a stream other than the legacy default stream (falls
                                       back to plain launches there, inside a caller's own capture, and with
                                       DC_FLAG_EXACT_FAR).  Results and the counters of dc_stats are those of the plain
                                       launches; the stage times (ms_stage, ms_kernel) are not recorded for a replayed
                                       cut and read 0. */

typedef struct dc_ctx dc_ctx;

typedef struct {
    double tau_cut_rel; /* CUT threshold / L_ref; <= 0: default 1e-7 (A.3 L719; reading A3) */
    double d_band;      /* exact-distance band; <= 0: auto = max element Bezier-box diagonal (A5) */
    double l_ref;       /* reference length; <= 0: auto = longest edge of the surface-node AABB */
    double theta_leaf;  /* subdivision stops when (patch size) x (curvature) <= theta; <= 0: 0.25 */
    int max_level;      /* subdivision bound per patch, 1..12; <= 0: default 12 */
    int flags;          /* DC_FLAG_* */
} dc_params;

typedef struct {
    long long n_elem, n_face;
    long long n_active;          /* elements that reached candidate generation (S4) */
    long long n_box_tests;       /* element-box vs face-box tests in S4 ("broad" pair tests) */
    long long n_pairs;           /* candidate (element, face) pairs = narrow-phase pair tests */
    long long n_bnb_nodes;       /* sub-pairs bounded in S5 */
    long long n_newton;          /* Newton solves in S5 */
    long long n_newton_iters;
    long long n_newton_fail;     /* solves that hit the iteration cap unconverged */
    long long n_depth_exceeded;  /* leaves forced by max_level */
    long long n_cut, n_hole, n_normal;
    long long n_ambiguous;       /* elements with |d_e - tau_cut| <= 1e-9 L_ref */
    long long n_sign_ambiguous;  /* elements whose tied nearest faces disagree in sign */
    long long n_seedless_components;
    long long n_fill_conflicts;
    long long pairs_needed;      /* pair slots S4 wanted (> max_pairs on overflow) */
    long long queue_peak;        /* max narrow-phase queue depth seen (items) */
    long long n_root_nodes;      /* (pair, patch) items of branch-and-bound round 0 (whole patch pairs) */
    long long band_needed;       /* elements with candidate pairs (> the band capacity on DC_STATUS_BAND_OVERFLOW) */
    long long queue_needed;      /* largest narrow-phase queue any round wanted (> the capacity max(2^20, max_pairs) on
                                    DC_STATUS_QUEUE_OVERFLOW: size max_pairs >= 1.25 queue_needed -- how many leaves are
                                    queued depends on the order in which the elements' bounds tighten and differs by a
                                    few per cent from run to run; the rounds after the one that overflowed are not run,
                                    so a second, larger need may show up on the next call) */
    long long n_far;             /* DC_FLAG_EXACT_FAR: elements the banded cut left clamped at +-d_band ... */
    long long n_far_done;        /* ... of which got their exact distance (= n_far unless the pass failed) */
    long long n_far_unresolved;  /* ... and for which the narrow phase solved no leaf (0; they keep the clamp) */
    long long far_pairs;         /* candidate pairs of the far pass, all chunks */
    long long far_passes;        /* passes the far pass ran in (each ends with a stream synchronisation) */
    double l_ref, tau_cut, d_band;
    float ms_stage[8];           /* 0 S1+S3 faces/bins, 1 S2 boxes, 2 S4 pairs, 3 S5+S6 narrow,
                                    4 S7 fill, 5 total dc_classify, 6 dc_set_cut_surface,
                                    7 every k_np_solve launch of S5 (seeds + leaf passes + overflow rounds, the latter
                                      with their two short k_np_bound passes) */
    float ms_kernel[8];          /* the kernels of S5/S6 one by one (CUDA events on the caller's stream):
                                    0 k_np_stage, 1 k_np_solve on the seeds, 2 k_np_roots, 3 k_np_bound (all rounds + tail),
                                    4 k_np_compact, 5 k_np_solve leaf passes 1-3, 6 overflow rounds (2 x bound + solve),
                                    7 k_np_decide */
    int status;                  /* DC_STATUS_* bits */
    int n_launches;              /* kernels launched by the last dc_set_cut_surface + dc_classify (far pass not counted) */
    float ms_far;                /* the exact far pass, host synchronisations included (CUDA events) */
    int reserved;
} dc_stats;

/* Bytes of device scratch dc_create_grid needs for a grid of this size, up to max_faces
 * surface faces and max_pairs candidate pairs.  Returns 0 on bad arguments. */
size_t dc_workspace_bytes(long long n_nodes, long long n_elem, long long max_faces, long long max_pairs);

/*
 * Register the element grid ("each partition contains a unique subset of a single
 * grid"; L233: structures that depend on the grid only are built once).  Runs S2 (conservative
 * element boxes from the Bezier control nets) and, if adj6_dev is NULL, derives the face
 * adjacency from shared face-centre nodes.
 *   xyz_dev    [n_nodes][3] f64 dev      node coordinates
 *   conn27_dev [n_elem][27] i32 dev      node ids, m = i + 3 j + 9 k
 *   adj6_dev   [n_elem][6]  i32 dev      or NULL
 *   workspace_dev, workspace_bytes       >= dc_workspace_bytes(...), 256-byte aligned
 * Enqueues on `stream`; the context is usable once the stream has drained (later calls on the
 * same stream are ordered correctly without a sync).
 */
int dc_create_grid(dc_ctx **out, int device,
                   long long n_nodes, const double *xyz_dev,
                   long long n_elem, const int *conn27_dev, const int *adj6_dev,
                   void *workspace_dev, size_t workspace_bytes,
                   long long max_faces, long long max_pairs, void *stream);

/*
 * Set the cutting surface (L171-L175: "each partition gathers all of its potential cutting
 * surfaces"; L215 "outward-oriented normal").  Runs S1 (face Bezier boxes, monomial
 * coefficients, surface AABB -> L_ref) and S3 (uniform face bins, a row of cells contiguous).
 *   face_nodes_dev [n_face][9][3] f64 dev, m = i + 3 j, normal x_s cross x_t points OUT of the body.
 */
int dc_set_cut_surface(dc_ctx *ctx, long long n_face, const double *face_nodes_dev, void *stream);

/*
 * One direct cut (S4 candidate pairs, S5 narrow phase, S6 decide, S7 flood fill; S2 too with
 * DC_FLAG_RECOMPUTE_BOXES).  params may be NULL (all defaults).
 *   labels_dev [n_elem] int8 dev  out    DC_HOLE / DC_NORMAL / DC_CUT   (L217 "blanking status ... saved to memory")
 *   sdist_dev  [n_elem] f64  dev  out    signed min distance, clamped to +-d_band (not clamped with
 *                                        DC_FLAG_EXACT_FAR), 0 for CUT
 * Asynchronous on `stream`, except with DC_FLAG_EXACT_FAR.
 */
int dc_classify(dc_ctx *ctx, const dc_params *params, signed char *labels_dev, double *sdist_dev,
                void *stream);

/*
 * dc_set_cut_surface + dc_classify in one call (same arguments, same results); with DC_FLAG_GRAPH in params->flags the
 * launch sequence is replayed from a CUDA graph (see the flag).  Asynchronous on `stream` except with DC_FLAG_EXACT_FAR.
 */
int dc_cut(dc_ctx *ctx, const dc_params *params, long long n_face, const double *face_nodes_dev,
           signed char *labels_dev, double *sdist_dev, void *stream);

/*
 * End-to-end variant with HOST buffers: copies the face nodes host->device, runs
 * dc_cut, copies labels and sdist device->host, and synchronises `stream` before returning.  Host buffers should be
 * pinned.  With DC_FLAG_GRAPH and pinned buffers the three copies are nodes of the cut's graph (keyed by the host
 * addresses too): the faces' upload then runs beside S2, which does not need them.
 */
int dc_classify_host(dc_ctx *ctx, const dc_params *params, long long n_face,
                     const double *face_nodes_host, signed char *labels_host, double *sdist_host,
                     void *stream);

/* Element boxes computed by S2: copies [n_elem][6] (min xyz, max xyz) to out_dev.  For tests. */
int dc_get_element_boxes(dc_ctx *ctx, double *out_dev, void *stream);

/* Face adjacency in use (given or derived): copies [n_elem][6] i32 to out_dev.  For tests. */
int dc_get_adjacency(dc_ctx *ctx, int *out_dev, void *stream);

/* Candidate pairs of the last dc_classify: element ids and ORIGINAL face ids, up to cap pairs.
 * Synchronises.  Returns the number of pairs (or a negative error).  For tests. */
long long dc_get_pairs(dc_ctx *ctx, int *elem_host, int *face_host, long long cap);

/* Synchronises the stream of the last call and fills *host_out (also when it returns an error).  Returns
 * DC_ERR_WORKSPACE on DC_STATUS_PAIR/QUEUE/BAND_OVERFLOW (pairs_needed / band_needed say what was wanted),
 * DC_ERR_RESULT on DC_STATUS_FILL_CONFLICT / DC_STATUS_SEEDLESS_OVERFLOW, DC_ERR_UNSUPPORTED on
 * DC_STATUS_SURFACE_SMALL, DC_OK otherwise. */
int dc_get_stats(dc_ctx *ctx, dc_stats *host_out);

void dc_destroy(dc_ctx *ctx);

const char *dc_error_string(int code);

/* ---- blanking logic that consumes direct cuts --------------------------------
 * Stateless device routines: plain device pointers owned by the caller, enqueued on `stream`, no host sync.
 * A blanking vector `iblank` is int8 per element: 1 = blanked ("hole cell"), 0 = field.  `cut_is_hole` != 0
 * counts DC_CUT elements as hole cells (the paper leaves the CUT elements of a wall cut to the caller). */
#define DC_MODE_WALL 0      /* body grid cut by solid wall surfaces (Algorithm 3.1 step 6) */
#define DC_MODE_OVERSET 1   /* background grid cut by overset boundary surfaces (step 7) */

/* Union of the hole cells of two cutting boundaries: out = HOLE if either is HOLE, else CUT if
 * either is CUT, else NORMAL.  out_dev may alias a_dev or b_dev.  All [n_elem] int8 dev. */
int dc_union_labels(long long n_elem, const signed char *a_dev, const signed char *b_dev,
                    signed char *out_dev, void *stream);

/* Algorithm 3.1 steps 6-7 for one grid.
 *   iblank_prev_dev [n_elem] int8 dev  in   I_{t-}: the blanking used for the previous time step (step 1)
 *   labels_t_dev, labels_tplus_dev      in   dc_classify labels of the cuts at t (step 5) and t + dt (step 3)
 *   iblank_out_dev  [n_elem] int8 dev  out  the blanking of this step: wall  -> hole at t OR at t + dt  (6.1),
 *                                           overset -> hole at t AND at t + dt (L112); may alias iblank_prev_dev
 *   unblank_list_dev [list_cap] i32 dev out elements that were blanked and must be unblanked now (6.2, 7.1)
 *   tohole_list_dev  [list_cap] i32 dev out elements newly blanked by this step (NULL: not wanted)
 *   counts_dev       [2] i64 dev        out number of must-unblank / to-hole elements (may exceed list_cap: the
 *                                           lists are then truncated; ids appear in no particular order)
 * Returns DC_ERR_ARG on NULL / negative arguments or an unknown mode. */
int dc_unblank(int mode, int cut_is_hole, long long n_elem, const signed char *iblank_prev_dev,
               const signed char *labels_t_dev, const signed char *labels_tplus_dev,
               signed char *iblank_out_dev, int *unblank_list_dev, int *tohole_list_dev, long long list_cap,
               long long *counts_dev, void *stream);

/* Artificial-boundary faces ("any face which has a hole cell on one side and a normal/field cell on
 * the other"): ab_mask_dev[e] gets bit k set iff e is a field cell and adj6[e][k] is a hole cell (each AB face is
 * reported on its field side); count_dev [1] i64 dev gets the number of AB faces (NULL: not wanted). */
int dc_ab_faces(long long n_elem, const signed char *iblank_dev, const int *adj6_dev,
                unsigned char *ab_mask_dev, long long *count_dev, void *stream);

/* ---- donor search for receptor points (PAPER.md 4.3 L229-L278; SURVEY.md 8(f) "(later)") ---------------------------
 * dc_adt_build: alternating digital tree over the element boxes of S2, built on the HOST (L233: once, during
 *   preprocessing; valid under rigid motion of the grid) into caller-owned device memory of dc_adt_bytes(n_elem)
 *   bytes, 16-byte aligned; synchronises `stream`.  Balanced (median splits), so the search needs a LIFO of
 *   height + 1 entries (L241-L247).
 * dc_find_donors: for each point x [n_pts][3] f64 dev -- given in the frame the grid has been MOVED to,
 *   x = R x_grid + o with rot9_host (row-major R, NULL = identity) and off3_host (NULL = 0) -- the element that
 *   contains it and its reference coordinates: stack-based tree search appending candidate elements (boxes that hold
 *   the point, at most 16 kept), then Newton on the isoparametric map of each candidate (Eq. 1-5, reference
 *   coordinates limited to [-1,1] + 1e-10, at most 10 iterations, L272-L278); converged = |x_p - x(X)| <= 1e-12 x
 *   element box diagonal.
 *     donor_dev [n_pts] i32 dev   out  element id, -1 if no element contains the point
 *     ref_dev   [n_pts][3] f64 dev out reference coordinates in the donor (0 if none)
 *     scratch_dev                      dc_donor_scratch_bytes(n_pts) bytes of device scratch
 *   A point on a face shared by two elements may be given either (both contain it).  Enqueued on `stream`. */
size_t dc_adt_bytes(long long n_elem);
size_t dc_donor_scratch_bytes(long long n_pts);
int dc_adt_build(dc_ctx *ctx, void *adt_dev, size_t adt_bytes, void *stream);
int dc_find_donors(dc_ctx *ctx, long long n_pts, const double *pts_dev, const double *rot9_host, const double *off3_host,
                   int *donor_dev, double *ref_dev, void *scratch_dev, size_t scratch_bytes, void *stream);

/*
 * dc_find_donors for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments minus the scratch, same kernels, same results.  The candidate lists
 * live in a fixed array inside the library (4 456 448 bytes of every GPU that loads libdc, until the process exits), so
 *   - n_pts <= DC_NOALLOC_MAX_POINTS, else DC_ERR_WORKSPACE (and a line on stderr that says so): split the batch;
 *   - the call allocates and frees nothing (no cudaMalloc / cudaFree, no allocating library routine); the first call on
 *     a device also asks the runtime for the array's address, once;
 *   - every call on a device shares the array: calls that OVERLAP on the GPU (different streams, no ordering between
 *     them) race on it and give wrong donors; calls ordered on one stream, or by events, are fine.
 */
#define DC_NOALLOC_MAX_POINTS 65536
int dc_find_donors_noalloc(dc_ctx *ctx, long long n_pts, const double *pts_dev, const double *rot9_host, const double *off3_host,
                           int *donor_dev, double *ref_dev, void *stream);

/* FP64 FMA peak microbenchmark (register-resident DFMA chains on every SM): returns measured
 * TFLOP/s (2 flop per FMA) or a negative error.  Used by bench.py for the "alu" roofline. */
double dc_measure_fp64_tflops(int device, int iters);

/* Library/ABI version. */
int dc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DC_H_ */
