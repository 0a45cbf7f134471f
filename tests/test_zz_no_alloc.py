"""-m gpu, collected LAST (pytest runs files in name order; the suite runs with pytest -x): dc_find_donors_noalloc, the
donor search for callers that cannot allocate device memory, against the existing dc_find_donors on the same points.

The no-alloc entry point runs the same two kernels with the candidate lists in the library's built-in array instead of
caller-allocated scratch, so donors must be identical and the reference coordinates within the tolerance
tests/test_gpu_donor.py uses (in fact bit for bit).  Two calls in a row with different points check that the second is
not fooled by what the first left in the shared array; a third past the limit checks the refusal."""
import numpy as np
import pytest

from workloads import make_config

pytestmark = pytest.mark.gpu

TOL_REF = 1e-9          # reference coordinates, as in tests/test_gpu_donor.py


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_1711_07663_b200._build import build_lib
    build_lib()
    from paper_1711_07663_b200 import binding
    return binding


def test_noalloc_donor_search_equals_the_existing_path_on_two_calls_in_a_row(B):
    import torch
    w = make_config(1, N=12, n=4)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
    dcut.build_adt()
    rng = np.random.default_rng(20260711)
    lo, hi = w.xyz.min(axis=0), w.xyz.max(axis=0)
    # first call: a full-size batch (the limit itself); second: fewer, different points -- part of the array then still
    # holds the first call's lists
    batches = [lo + (hi - lo) * (rng.random((B.DC_NOALLOC_MAX_POINTS, 3)) * 1.1 - 0.05),
               lo + (hi - lo) * (rng.random((20011, 3)) * 1.1 - 0.05)]
    rot = np.array([[0.0, -1.0, 0.0], [1.0, 0.0, 0.0], [0.0, 0.0, 1.0]])
    off = np.array([0.3, -0.2, 0.1])
    for k, P in enumerate(batches):
        kw = dict(rot=rot, offset=off) if k == 1 else {}
        if k == 1:
            P = P @ rot.T + off                       # the grid has been moved: points in the moved frame
        pts = torch.from_numpy(np.ascontiguousarray(P)).cuda()
        donor_ref, ref_ref = dcut.find_donors(pts, **kw)         # existing path: caller-allocated scratch
        donor = torch.full((pts.shape[0],), -7, dtype=torch.int32, device="cuda")
        ref = torch.full((pts.shape[0], 3), 99.0, dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        dcut.find_donors_noalloc(pts, donor, ref, **kw)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before          # (nothing went through torch's allocator either)
        d0, d1 = donor_ref.cpu().numpy(), donor.cpu().numpy()
        r0, r1 = ref_ref.cpu().numpy(), ref.cpu().numpy()
        assert (d0 >= 0).sum() > len(d0) // 2 and (d0 < 0).sum() > 0      # points inside and outside the grid
        assert np.array_equal(d1, d0), "call %d: %d donors differ" % (k, int((d1 != d0).sum()))
        assert np.abs(r1 - r0).max() <= TOL_REF
        assert np.array_equal(r1, r0)
    # beyond the built-in scratch: refused, outputs untouched
    big = torch.zeros((B.DC_NOALLOC_MAX_POINTS + 1, 3), dtype=torch.float64, device="cuda")
    donor = torch.full((big.shape[0],), -7, dtype=torch.int32, device="cuda")
    ref = torch.full((big.shape[0], 3), 99.0, dtype=torch.float64, device="cuda")
    rc = dcut.find_donors_noalloc(big, donor, ref, return_code=True)
    torch.cuda.synchronize()
    assert rc == B.DC_ERR_WORKSPACE
    assert bool((donor == -7).all()) and bool((ref == 99.0).all())
    dcut.close()
