"""-m gpu: DC_FLAG_EXACT_FAR (second half: "d_band = infinity", reading A5's alternative) against the
CPU oracle.

The oracle already computes the true d_e of EVERY element and clamps it only when it writes sdist (dc_oracle.c step 5);
called with a band wider than the domain it never relaxes its enclosure (no element is "far") and writes sdist = +-d_e.
The CUDA path runs its banded cut with the default band and then the far pass: labels bit-exact, sdist within
1e-10 L_ref on every element -- the same bar as the banded parity tests, now with no clamp to hide behind.
"""
import numpy as np
import pytest

from oracle import dc_oracle as O
from workloads import make_config

pytestmark = pytest.mark.gpu

TOL_REL = 1e-10
WIDE = 1e30          # "d_band = infinity" for the oracle


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_1711_07663_b200._build import build_lib
    build_lib()
    from paper_1711_07663_b200 import binding
    return binding


def exact_cut(B, w, max_pairs=None, flags=0):
    p = B.dc_params(); p.flags = B.DC_FLAG_EXACT_FAR | flags
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face, max_pairs=max_pairs)
    dcut.set_cut_surface(w.faces)
    labels, sdist = dcut.classify(p)
    st = dcut.stats()
    out = labels.cpu().numpy().copy(), sdist.cpu().numpy().copy(), st
    dcut.close()
    return out


def check(ref, labels, sdist, st, zero_ambiguous=True):
    L = ref.stats["l_ref"]
    amb = (ref.flags & O.FLAG_AMBIGUOUS) != 0
    if zero_ambiguous:
        assert amb.sum() == 0
    assert (ref.flags & O.FLAG_FAR).sum() == 0            # the oracle used its strict enclosure everywhere
    assert ref.stats["n_depth_exceeded"] == 0
    bad = (labels != ref.labels) & ~amb
    assert bad.sum() == 0, "label mismatches at %s" % np.nonzero(bad)[0][:10]
    err = np.abs(sdist - ref.sdist)
    worst = int(np.argmax(np.where(amb, 0, err)))
    assert err[~amb].max() <= TOL_REL * L, "max |dsdist| = %.3e at element %d (oracle %.15e gpu %.15e)" % (
        err[worst], worst, ref.sdist[worst], sdist[worst])
    assert st.status == 0 and st.n_far_unresolved == 0 and st.n_far_done == st.n_far
    # nothing is left on the clamp: every element beyond the band moved off +-d_band (its true distance is larger)
    far = (np.abs(ref.sdist) > st.d_band)
    assert st.n_far >= far.sum()
    assert (np.abs(sdist[far]) > st.d_band).all()
    return far


def test_config0_exact_everywhere(B, nproc):
    w = make_config(0)
    ref = O.classify(w.xyz, w.conn27, w.faces, nproc=nproc, d_band=WIDE)
    labels, sdist, st = exact_cut(B, w)
    far = check(ref, labels, sdist, st)
    assert far.sum() > w.n_elem // 2            # most of config 0 lies beyond the band: the pass did the bulk of the distances
    # the banded cut of the same context gives the same values inside the band and the clamp outside
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
    dcut.set_cut_surface(w.faces)
    lb, sb = dcut.classify()
    lb, sb = lb.cpu().numpy(), sb.cpu().numpy()
    dcut.close()
    assert np.array_equal(lb, labels)
    assert np.array_equal(sb[~far], sdist[~far])
    assert (np.abs(sb[far]) == st.d_band).all()


def test_config1_reduced_exact_everywhere_in_many_chunks(B, nproc):
    """A curved surface (config 1's sphere at reduced size) and a workspace so small that the far pass needs many chunks
    and defers elements from one chunk to the next: the result must not depend on the chunking."""
    w = make_config(1, N=14, n=6)
    ref = O.classify(w.xyz, w.conn27, w.faces, nproc=nproc, d_band=WIDE)
    labels, sdist, st = exact_cut(B, w)
    check(ref, labels, sdist, st)
    labels2, sdist2, st2 = exact_cut(B, w, max_pairs=32000)
    assert st2.far_passes > st.far_passes and st2.far_passes >= 3
    assert np.array_equal(labels2, labels)
    assert np.array_equal(sdist2, sdist)                 # bit for bit: chunk composition must not leak into the values
    assert st2.n_far == st.n_far and st2.far_pairs >= st.n_far


def test_exact_far_with_recomputed_boxes_and_element_inside_the_body(B, nproc):
    """Config 2's shape at reduced size: elements deep inside the closed surface (HOLE, far from every face, nearly
    equidistant from many of them) take the longest candidate lists."""
    w = make_config(2, N=12, n=8)
    ref = O.classify(w.xyz, w.conn27, w.faces, nproc=nproc, d_band=WIDE)
    labels, sdist, st = exact_cut(B, w, flags=B.DC_FLAG_RECOMPUTE_BOXES)
    check(ref, labels, sdist, st, zero_ambiguous=False)
    assert (labels == 0).sum() > 0 and (sdist[labels == 0] < 0).all()


def test_exact_far_between_several_bodies(B, nproc):
    """Config 4's eight ellipsoids at reduced size: between bodies the face with the nearest box is often on the wrong
    body (the second seed solve is for this case), and an element may be equally far from two bodies."""
    w = make_config(4, N=20, n=5)
    ref = O.classify(w.xyz, w.conn27, w.faces, nproc=nproc, d_band=WIDE)
    labels, sdist, st = exact_cut(B, w)
    far = check(ref, labels, sdist, st, zero_ambiguous=False)
    assert far.sum() > w.n_elem // 2
    # the smallest workspace the banded cut itself gets by with: more passes, same values
    small = max(int(1.3 * st.pairs_needed), 8 * int(st.band_needed))
    labels2, sdist2, st2 = exact_cut(B, w, max_pairs=small)
    assert st2.far_passes > st.far_passes, (st.far_passes, st2.far_passes, small, st.far_pairs)
    assert np.array_equal(labels2, labels) and np.array_equal(sdist2, sdist)


def test_one_element_with_more_candidates_than_a_chunk_reports_workspace(B):
    """max_pairs so small that a single far element's candidate faces exceed a chunk: DC_ERR_WORKSPACE, and pairs_needed
    large enough to succeed with."""
    w = make_config(1, N=10, n=8)
    p = B.dc_params(); p.flags = B.DC_FLAG_EXACT_FAR
    need = None
    for attempt in range(4):
        mp = 600 if need is None else need
        dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face, max_pairs=mp)
        dcut.set_cut_surface(w.faces)
        dcut.classify(p)
        st, rc = dcut.stats(allow_status=True, return_code=True)
        dcut.close()
        if rc == B.DC_OK:
            break
        assert rc == B.DC_ERR_WORKSPACE
        need = max(int(st.pairs_needed), int(st.queue_needed), 8 * int(st.band_needed), 2 * mp)
    assert rc == B.DC_OK and attempt >= 1
