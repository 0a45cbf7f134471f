"""-m gpu: the CUDA path (libdc.so through its C ABI) against the CPU oracle, element by element,
on the same seeded inputs.

Bar (BASELINE.json north_star): labels bit-exact except on elements the ORACLE flags ambiguous
(|d - tau_cut| <= 1e-9 L_ref; counted, and required to be zero on configs 0-1); per-element
signed distance within 1e-10 L_ref absolute.  Nearest-face id / closest parameters are not
compared (not unique, reading A12).

Reduced-size instances keep each config's structure, span several thread blocks / narrow-phase
batches and end in a ragged tail; the full-size cases (tests/test_gpu_fullsize.py) use sampled
elements and size-independent invariants.
"""
import numpy as np
import pytest

from oracle import dc_oracle as O
from workloads import make_config

pytestmark = pytest.mark.gpu

HOLE, NORMAL, CUT = 0, 1, 2
TOL_REL = 1e-10     # north_star: |sdist_gpu - sdist_oracle| <= 1e-10 L_ref


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_1711_07663_b200._build import build_lib
    build_lib()
    from paper_1711_07663_b200 import binding
    return binding


def gpu_cut(B, w, faces=None, adj="given", params=None, max_pairs=None, keep=False):
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6 if adj == "given" else None,
                       max_faces=w.n_face if faces is None else len(faces), max_pairs=max_pairs)
    dcut.set_cut_surface(w.faces if faces is None else faces)
    labels, sdist = dcut.classify(params)
    st = dcut.stats()
    out = labels.cpu().numpy().copy(), sdist.cpu().numpy().copy(), st
    if keep:
        return out + (dcut,)
    dcut.close()
    return out


def assert_parity(ref, labels, sdist, st, expect_zero_ambiguous=False, ids=None):
    if ids is not None:
        labels, sdist = labels[ids], sdist[ids]
    L = ref.stats["l_ref"]
    amb = (ref.flags & O.FLAG_AMBIGUOUS) != 0
    if expect_zero_ambiguous:
        assert amb.sum() == 0 and st.n_ambiguous == 0
    assert ref.stats["n_depth_exceeded"] == 0
    bad = (labels != ref.labels) & ~amb
    assert bad.sum() == 0, "label mismatches at %s: gpu %s oracle %s (oracle dmin %s)" % (
        np.nonzero(bad)[0][:10], labels[bad][:10], ref.labels[bad][:10], ref.dmin[bad][:10])
    err = np.abs(sdist - ref.sdist)
    assert err[~amb].max() <= TOL_REL * L, "max |dsdist| = %.3e at element %d (oracle %.12e gpu %.12e)" % (
        err[~amb].max(), int(np.argmax(np.where(amb, 0, err))), ref.sdist[np.argmax(np.where(amb, 0, err))],
        sdist[np.argmax(np.where(amb, 0, err))])
    assert abs(st.l_ref - L) <= 1e-15 * L
    assert abs(st.tau_cut - ref.stats["tau_cut"]) <= 1e-15 * L
    assert abs(st.d_band - ref.stats["d_band"]) <= 1e-14 * L
    assert st.status == 0 and st.n_fill_conflicts == 0
    assert st.n_cut + st.n_hole + st.n_normal == st.n_elem


# ------------------------------------------------------------------------------ config 0 (full size)
@pytest.fixture(scope="module")
def cfg0(nproc):
    w = make_config(0)
    return w, O.classify(w.xyz, w.conn27, w.faces, nproc=nproc)


def test_config0_full_parity_and_census(B, cfg0):
    w, ref = cfg0
    labels, sdist, st = gpu_cut(B, w)
    assert_parity(ref, labels, sdist, st, expect_zero_ambiguous=True)
    # closed-form census (tests/golden/config0_closed_form_census.txt)
    assert (st.n_hole, st.n_cut, st.n_normal) == (136, 296, 3664)
    assert st.n_sign_ambiguous == 0 and st.n_depth_exceeded == 0


def test_config0_derived_adjacency_and_recomputed_boxes(B, cfg0):
    w, ref = cfg0
    p = B.dc_params(); p.flags = B.DC_FLAG_RECOMPUTE_BOXES
    labels, sdist, st, dcut = gpu_cut(B, w, adj="derive", params=p, keep=True)
    assert_parity(ref, labels, sdist, st, expect_zero_ambiguous=True)
    assert np.array_equal(dcut.adjacency().cpu().numpy(), w.adj6)
    dcut.close()


def test_element_boxes_bit_exact(B):
    w = make_config(1, N=9, n=2)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
    got = dcut.element_boxes().cpu().numpy()
    dcut.close()
    want = np.stack([O.element_box(w.xyz, w.conn27[e]) for e in range(w.n_elem)])
    assert np.array_equal(got, want)


def test_candidate_pairs_equal_brute_force_box_test(B, cfg0):
    """S4 must emit exactly {(e,f): BOUNDINGBOXDIST(box_e, box_f) <= d_band + 2 tau + t_tie} (A.2)."""
    w, ref = cfg0
    labels, sdist, st, dcut = gpu_cut(B, w, keep=True)
    e, f = dcut.pairs()
    dcut.close()
    got = set(zip(e.tolist(), f.tolist()))
    assert len(got) == len(e) == st.n_pairs
    ebox = np.stack([O.element_box(w.xyz, w.conn27[i]) for i in range(w.n_elem)])
    fbox = np.empty((w.n_face, 6))
    for j in range(w.n_face):
        Bz = O.lagrange_to_bezier(w.faces[j])
        fbox[j, :3], fbox[j, 3:] = Bz.min(0), Bz.max(0)
    reach = st.d_band + 2 * st.tau_cut + 1e-9 * st.l_ref
    want = set()
    slack = set()
    for j in range(w.n_face):
        d = np.array([O.box_dist(ebox[i], fbox[j]) for i in range(w.n_elem)])
        want.update((int(i), j) for i in np.nonzero(d <= reach * (1 - 1e-12))[0])
        slack.update((int(i), j) for i in np.nonzero(d <= reach * (1 + 1e-12))[0])
    assert want <= got <= slack


# ------------------------------------------------------------------------------ reduced configs 1, 2, 4
@pytest.mark.parametrize("config,N,n", [(1, 21, 6), (2, 26, 10), (4, 30, 5)])
def test_reduced_config_parity(B, nproc, config, N, n):
    w = make_config(config, N=N, n=n)
    ref = O.classify(w.xyz, w.conn27, w.faces, nproc=nproc)
    labels, sdist, st = gpu_cut(B, w)
    assert_parity(ref, labels, sdist, st, expect_zero_ambiguous=(config == 1))
    assert st.n_cut > 50 and st.n_hole > 0
    # P7: no HOLE element face-adjacent to a NORMAL element
    for k in range(6):
        nb = w.adj6[:, k]; m = nb >= 0
        assert not ((labels[m] == HOLE) & (labels[nb[m]] == NORMAL)).any()
        assert not ((labels[m] == NORMAL) & (labels[nb[m]] == HOLE)).any()


def test_config3_spin_recut_same_context(B, nproc):
    """Config 3: re-cut of a fixed grid by the rotated surface, same dc_ctx (state reset between cuts)."""
    w = make_config(3, N=22, n=8)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
    for step in (1, 17, 32):
        faces = w.spin_faces(step)
        ref = O.classify(w.xyz, w.conn27, faces, nproc=nproc)
        dcut.set_cut_surface(faces)
        labels, sdist = dcut.classify()
        st = dcut.stats()
        assert_parity(ref, labels.cpu().numpy(), sdist.cpu().numpy(), st)
    dcut.close()


def test_host_buffer_entry_point_matches_device_one(B):
    import torch
    w = make_config(1, N=12, n=4)
    labels, sdist, st, dcut = gpu_cut(B, w, keep=True)
    fh = torch.from_numpy(w.faces).pin_memory()
    lh = torch.empty(w.n_elem, dtype=torch.int8).pin_memory()
    sh = torch.empty(w.n_elem, dtype=torch.float64).pin_memory()
    dcut.classify_host(fh, lh, sh)
    assert np.array_equal(lh.numpy(), labels) and np.array_equal(sh.numpy(), sdist)
    dcut.close()


# ------------------------------------------------------------------------------ invariances on the GPU path
def test_face_and_element_permutation(B):
    w = make_config(1, N=14, n=4)
    l0, s0, st0 = gpu_cut(B, w)
    rng = np.random.default_rng(6)
    pf = rng.permutation(w.n_face)
    l1, s1, st1 = gpu_cut(B, w, faces=w.faces[pf])
    assert np.array_equal(l0, l1)
    assert np.abs(s0 - s1).max() <= 1e-12 * st0.l_ref
    # run-to-run reproducibility (atomics change arrival order, not results)
    l2, s2, _ = gpu_cut(B, w)
    assert np.array_equal(l0, l2) and np.abs(s0 - s2).max() <= 1e-12 * st0.l_ref


def test_orientation_reversal_swaps_hole_and_normal(B):
    w = make_config(1, N=12, n=3)
    l0, s0, _ = gpu_cut(B, w)
    flipped = w.faces.reshape(-1, 3, 3, 3).transpose(0, 2, 1, 3).reshape(-1, 9, 3).copy()
    l1, s1, _ = gpu_cut(B, w, faces=flipped)
    swap = np.array([NORMAL, HOLE, CUT], np.int8)
    assert np.array_equal(l1, swap[l0])
    assert np.abs(s1 + s0).max() <= 1e-12


# ------------------------------------------------------------------------------ degenerate cases
def test_surface_outside_and_enclosing_the_grid(B):
    w = make_config(0, N=6, n=2)
    # surface far outside the grid: no candidate pairs at all, one seedless component -> NORMAL
    l, s, st = gpu_cut(B, w, faces=w.faces + np.array([10.0, 0, 0]))
    ref = O.classify(w.xyz, w.conn27, w.faces + np.array([10.0, 0, 0]))
    assert (l == NORMAL).all() and np.array_equal(l, ref.labels)
    assert np.abs(s - ref.sdist).max() <= 1e-14 and st.n_pairs == 0 and st.n_seedless_components == 1
    # surface enclosing the whole grid: everything HOLE
    l, s, st = gpu_cut(B, w, faces=w.faces * 10.0)
    ref = O.classify(w.xyz, w.conn27, w.faces * 10.0)
    assert (l == HOLE).all() and np.array_equal(l, ref.labels)
    assert np.abs(s - ref.sdist).max() <= 1e-14 and st.n_seedless_components == 1


def test_single_element_grid_is_reported_unsupported(B):
    """One hex [-1,1]^3 containing the whole sphere: the documented precondition (no surface component inside one
    element, reading A7 / SURVEY.md 8(a) note ii) is violated; dc_get_stats says DC_ERR_UNSUPPORTED
    (DC_STATUS_SURFACE_SMALL), and the labels / distances written are still those of the boundary-patch definition,
    which is what the oracle computes too."""
    w = make_config(0, N=1, n=2)
    ref = O.classify(w.xyz, w.conn27, w.faces)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
    dcut.set_cut_surface(w.faces)
    labels, sdist = dcut.classify()
    with pytest.raises(B.DcError) as ei:
        dcut.stats()
    assert ei.value.code == B.DC_ERR_UNSUPPORTED
    st = dcut.stats(allow_status=True)
    assert st.status == B.DC_STATUS_SURFACE_SMALL
    l, s = labels.cpu().numpy(), sdist.cpu().numpy()
    dcut.close()
    assert np.array_equal(l, ref.labels) and np.abs(s - ref.sdist).max() <= TOL_REL * st.l_ref


def test_many_seedless_components(B):
    """A grid of 216 hexes that are not connected to one another at all (adjacency all -1) and far from the surface:
    216 seedless components, each resolved by its own exhaustive nearest-face query (the library used to stop at 32)."""
    w = make_config(0, N=6, n=2)
    adj = np.full_like(w.adj6, -1)
    faces = w.faces * 0.25 + np.array([3.0, 0.0, 0.0])          # a small sphere outside the grid
    ref = O.classify(w.xyz, w.conn27, faces)
    dcut = B.DirectCut(w.xyz, w.conn27, adj, max_faces=len(faces))
    dcut.set_cut_surface(faces)
    labels, sdist = dcut.classify()
    st = dcut.stats(allow_status=True)
    l, s = labels.cpu().numpy(), sdist.cpu().numpy()
    dcut.close()
    assert st.n_pairs == 0 and st.n_seedless_components == w.n_elem
    assert (st.status & ~B.DC_STATUS_SURFACE_SMALL) == 0
    assert (l == NORMAL).all() and np.array_equal(l, ref.labels) and np.abs(s - ref.sdist).max() <= 1e-14


# ------------------------------------------------------------------------------ error behaviour (include/dc.h)
def test_error_codes(B):
    w = make_config(0, N=8, n=2)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face, max_pairs=64)
    with pytest.raises(B.DcError) as ei:           # classify before set_cut_surface
        dcut.classify()
    assert ei.value.code == B.DC_ERR_STATE
    with pytest.raises(B.DcError) as ei:           # more faces than max_faces
        dcut.set_cut_surface(np.concatenate([w.faces, w.faces]))
    assert ei.value.code == B.DC_ERR_WORKSPACE
    dcut.set_cut_surface(w.faces)
    dcut.classify()
    with pytest.raises(B.DcError) as ei:           # 64 pair slots are not enough: latched, reported
        dcut.stats()
    assert ei.value.code == B.DC_ERR_WORKSPACE
    st = dcut.stats(allow_status=True)
    assert st.status & B.DC_STATUS_PAIR_OVERFLOW and st.pairs_needed > 64
    dcut.close()
    assert B.dc_workspace_bytes(10, 10, 1 << 31, 100) == 0 and B.dc_workspace_bytes(10, 10, 100, 1 << 31) == 0
    # the reported size is sufficient
    l, s, st2 = gpu_cut(B, w, max_pairs=int(st.pairs_needed))
    assert st2.status == 0 and st2.n_pairs == st.pairs_needed


def test_band_overflow_is_reported_with_the_size_needed(B):
    """Few, large faces against a fine grid: many band elements with two or three pairs each, so the band arrays
    (capacity max_pairs / 8, at least 65 536) fill before the pair list does: DC_STATUS_BAND_OVERFLOW, and
    dc_stats.band_needed says what to ask for."""
    w = make_config(1, N=112, n=3)           # 1.4 M elements vs 54 faces
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face, max_pairs=400000)
    dcut.set_cut_surface(w.faces)
    dcut.classify()
    with pytest.raises(B.DcError) as ei:
        dcut.stats()
    assert ei.value.code == B.DC_ERR_WORKSPACE
    st = dcut.stats(allow_status=True)
    dcut.close()
    assert st.status & B.DC_STATUS_BAND_OVERFLOW and not (st.status & B.DC_STATUS_PAIR_OVERFLOW)
    assert st.band_needed > 65536 and st.pairs_needed <= 400000
    # following the sizes reported leads to a valid cut (this workload's whole faces make up to 6 root items per pair:
    # the queues, sized by max_pairs too, are the next thing to fill, and say so the same way; a queue that overflowed
    # hides what the later rounds would have wanted, hence the loop; the leaf queue's need depends on the order in which the
    # elements' bounds tighten and differs by a few per cent from run to run, hence the margin dc.h asks for)
    need = 8 * int(st.band_needed)
    for attempt in range(5):
        dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face, max_pairs=need)
        dcut.set_cut_surface(w.faces); dcut.classify()
        st1 = dcut.stats(allow_status=True)
        dcut.close()
        assert not (st1.status & (B.DC_STATUS_BAND_OVERFLOW | B.DC_STATUS_PAIR_OVERFLOW))
        if st1.status == 0:
            break
        assert st1.status & B.DC_STATUS_QUEUE_OVERFLOW and st1.queue_needed > max(need, 1 << 20)
        need = int(1.25 * st1.queue_needed)
    assert st1.status == 0 and st1.band_needed == st.band_needed and st1.n_cut > 1000


# ------------------------------------------------------------------------------ coarse grid, fine surface
def test_many_faces_per_element(B, nproc):
    """Large elements against a fine surface: hundreds of candidate faces per element, so k_pairs leaves its
    shared-memory stage (PR_CAP survivors) and re-walks the ranges, and the face bins span many cell blocks
    (the failure mode of box-only ranking in PAPER.md Fig. 10: exactness must not depend on a fixed K)."""
    w = make_config(1, N=5, n=14)           # 125 hexes of edge 0.4 vs 1176 faces of edge ~0.06
    ref = O.classify(w.xyz, w.conn27, w.faces, nproc=nproc)
    labels, sdist, st, dcut = gpu_cut(B, w, keep=True)
    e, f = dcut.pairs()
    dcut.close()
    assert np.bincount(e).max() > 224, "this case is meant to overflow the per-warp pair stage"
    assert_parity(ref, labels, sdist, st)
    assert st.n_cut > 20


def test_rigid_motion_of_grid_and_surface(B):
    """Metamorphic (the paper's edge-case sweep under rotation, L282): moving grid and surface
    together by one rigid motion leaves every label unchanged and every distance within rounding."""
    w = make_config(2, N=18, n=8)
    l0, s0, st0 = gpu_cut(B, w)
    rng = np.random.default_rng(11)
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    t = np.array([0.3, -0.2, 0.5])
    w2 = type(w)(**{**w.__dict__, "xyz": w.xyz @ q.T + t, "faces": w.faces @ q.T + t})
    l1, s1, st1 = gpu_cut(B, w2)
    # a rotated box is not the box of the rotated element, so d_band (the clamp of far distances) changes: compare inside the band
    band = min(st0.d_band, st1.d_band) * (1 - 1e-9)
    assert np.array_equal(l0, l1)
    near = (np.abs(s0) < band) & (np.abs(s1) < band)
    assert near.sum() > 100 and np.abs(s0 - s1)[near].max() <= 1e-11 * st0.l_ref


def test_parameters_theta_and_max_level_do_not_change_the_result(B):
    """The leaf rule (theta_leaf) and the subdivision bound (max_level) steer the work, not the answer."""
    w = make_config(2, N=16, n=8)
    l0, s0, st0 = gpu_cut(B, w)
    for theta, ml in ((0.03, 12), (0.125, 12), (0.5, 12), (0.25, 3)):
        p = B.dc_params(); p.theta_leaf = theta; p.max_level = ml
        l1, s1, st1 = gpu_cut(B, w, params=p)
        assert np.array_equal(l0, l1) and np.abs(s0 - s1).max() <= 1e-11 * st0.l_ref, (theta, ml)
    assert st0.n_newton > 0


def test_element_permutation(B):
    """Elements renumbered at random (adjacency remapped): neighbours no longer have nearby ids, so the tile-local
    union-find pass settles almost nothing and every edge goes through the global forest; the labels and distances
    must simply be permuted."""
    w = make_config(1, N=22, n=5)                    # 10 648 elements: 11 tiles of the fill, all of them mixed up
    l0, s0, st0 = gpu_cut(B, w)
    rng = np.random.default_rng(8)
    perm = rng.permutation(w.n_elem)                 # new element i is old element perm[i]
    inv = np.empty_like(perm); inv[perm] = np.arange(w.n_elem)
    adj = w.adj6[perm]
    adj = np.where(adj >= 0, inv[np.maximum(adj, 0)], -1).astype(np.int32)
    w2 = type(w)(**{**w.__dict__, "conn27": np.ascontiguousarray(w.conn27[perm]), "adj6": np.ascontiguousarray(adj)})
    l1, s1, st1 = gpu_cut(B, w2)
    assert np.array_equal(l1, l0[perm]) and np.abs(s1 - s0[perm]).max() <= 1e-12 * st0.l_ref
    # and with the adjacency derived by the library from the shared face-centre nodes
    l2, s2, _ = gpu_cut(B, w2, adj="derive")
    assert np.array_equal(l2, l1) and np.array_equal(s2, s1)


def test_whole_grid_inside_the_band(B, nproc):
    """d_band larger than the grid: every element gets its exact distance (no flood fill at all; the 'exact everywhere'
    option of reading A5), against the oracle with the same band."""
    w = make_config(1, N=9, n=3)
    p = B.dc_params(); p.d_band = 10.0
    ref = O.classify(w.xyz, w.conn27, w.faces, nproc=nproc, d_band=10.0)
    labels, sdist, st = gpu_cut(B, w, params=p, max_pairs=w.n_elem * w.n_face)
    assert st.n_pairs == w.n_elem * w.n_face
    assert_parity(ref, labels, sdist, st, expect_zero_ambiguous=True)
    assert np.abs(sdist).max() < 10.0 and np.abs(sdist).max() > 0.5
