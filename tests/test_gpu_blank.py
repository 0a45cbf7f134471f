"""-m gpu: the blanking kernels (dc_union_labels, dc_unblank, dc_ab_faces)
against oracle/blank_oracle.py, bit-exact (integer work; the id lists are compared as sets: their order is
whatever the atomics made it)."""
import numpy as np
import pytest

from oracle import blank_oracle as BO
from workloads import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_1711_07663_b200._build import build_lib
    build_lib()
    from paper_1711_07663_b200 import binding
    return binding


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("n", [1, 31, 32, 1000, 262147])
def test_union_and_unblank_random(B, n):
    rng = np.random.default_rng(n)
    a = rng.integers(0, 3, n).astype(np.int8); b = rng.integers(0, 3, n).astype(np.int8)
    prev = rng.integers(0, 2, n).astype(np.int8)
    assert np.array_equal(B.dc_union_labels(dev(a), dev(b)).cpu().numpy(), BO.union_labels(a, b))
    for mode in (B.DC_MODE_WALL, B.DC_MODE_OVERSET):
        for cih in (False, True):
            ib, unb, toh, counts = B.dc_unblank(mode, cih, dev(prev), dev(a), dev(b))
            rib, runb, rtoh = BO.unblank(mode, cih, prev, a, b)
            assert np.array_equal(ib.cpu().numpy(), rib)
            assert counts == [len(runb), len(rtoh)]
            assert np.array_equal(np.sort(unb.cpu().numpy()), runb) and np.array_equal(np.sort(toh.cpu().numpy()), rtoh)


def test_unblank_truncated_lists_and_errors(B):
    n = 5000
    prev = np.ones(n, np.int8); lab = np.ones(n, np.int8)            # everything was blanked, nothing is a hole now
    ib, unb, toh, counts = B.dc_unblank(B.DC_MODE_WALL, False, dev(prev), dev(lab), dev(lab), list_cap=100)
    assert counts == [n, 0] and unb.numel() == 100 and len(set(unb.cpu().tolist())) == 100 and not ib.any()
    with pytest.raises(B.DcError) as ei:
        B.dc_unblank(7, False, dev(prev), dev(lab), dev(lab))
    assert ei.value.code == B.DC_ERR_ARG


def test_ab_faces_after_a_real_cut(B):
    """Config-1-like cut: blank HOLE + CUT, tag the AB faces, compare with the oracle and with the closed count."""
    w = make_config(1, N=14, n=4)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
    dcut.set_cut_surface(w.faces)
    labels, _ = dcut.classify()
    lab = labels.cpu().numpy()
    ib, unb, toh, counts = B.dc_unblank(B.DC_MODE_WALL, True, dev(np.zeros(w.n_elem, np.int8)), labels, labels)
    rib, _, rtoh = BO.unblank(BO.MODE_WALL, True, np.zeros(w.n_elem, np.int8), lab, lab)
    assert np.array_equal(ib.cpu().numpy(), rib) and counts == [0, int(rib.sum())]
    mask, count = B.dc_ab_faces(ib, dev(w.adj6))
    rmask = BO.ab_faces(rib, w.adj6)
    assert np.array_equal(mask.cpu().numpy(), rmask)
    assert count == int(sum(bin(int(x)).count("1") for x in rmask)) and count > 0
    dcut.close()


def test_moving_body_unblank_matches_oracle(B):
    """Algorithm 3.1 on a body that moves by less than a cell per step (curved grid of config 1, sphere translated):
    cuts at t - dt, t and t + dt through dc_classify, then the wall-mode and overset-mode set logic."""
    w = make_config(1, N=20, n=6)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
    cuts = []
    for step in range(3):
        dcut.set_cut_surface(w.faces + np.array([0.06 * step, 0.0, 0.0]))
        labels, _ = dcut.classify()
        cuts.append(labels.clone())
    prev = (cuts[0] != 1).to(cuts[0].dtype)                           # I_{t-}: HOLE and CUT blanked
    for mode in (B.DC_MODE_WALL, B.DC_MODE_OVERSET):
        ib, unb, toh, counts = B.dc_unblank(mode, True, prev, cuts[1], cuts[2])
        rib, runb, rtoh = BO.unblank(mode, True, prev.cpu().numpy(), cuts[1].cpu().numpy(), cuts[2].cpu().numpy())
        assert np.array_equal(ib.cpu().numpy(), rib)
        assert np.array_equal(np.sort(unb.cpu().numpy()), runb) and np.array_equal(np.sort(toh.cpu().numpy()), rtoh)
        assert len(runb) > 0                                          # the body moves: some cells are left behind
    dcut.close()
