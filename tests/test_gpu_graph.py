"""-m gpu: dc_cut and DC_FLAG_GRAPH -- the cut's launch sequence replayed from a CUDA graph must give, bit for bit, what the
plain launches give (which tests/test_gpu_parity.py holds against the oracle), on every replay, for a surface that
changes in place between replays."""
import numpy as np
import pytest

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


def plain_cut(B, w, faces, flags=0):
    p = B.dc_params(); p.flags = flags
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
    dcut.set_cut_surface(faces)
    lab, sd = dcut.classify(p)
    st = dcut.stats()
    out = lab.cpu().numpy().copy(), sd.cpu().numpy().copy(), st
    dcut.close()
    return out


def test_graph_replay_equals_plain_launches_for_a_surface_moving_in_place(B):
    import torch
    w = make_config(3, N=20, n=8)
    steps = [w.spin_faces(s) for s in (0, 1, 2, 3, 2, 1)]
    want = [plain_cut(B, w, f, B.DC_FLAG_RECOMPUTE_BOXES) for f in steps]
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
        p = B.dc_params(); p.flags = B.DC_FLAG_RECOMPUTE_BOXES | B.DC_FLAG_GRAPH
        buf = torch.empty((w.n_face, 9, 3), dtype=torch.float64, device="cuda")
        for k, f in enumerate(steps):
            buf.copy_(torch.from_numpy(f))              # same address every step: one capture, then replays
            lab, sd = dcut.cut(buf, p)
            st = dcut.stats()
            assert st.status == 0
            assert np.array_equal(lab.cpu().numpy(), want[k][0]), "labels differ at step %d" % k
            assert np.array_equal(sd.cpu().numpy(), want[k][1]), "sdist differs at step %d" % k
            assert (st.n_cut, st.n_hole, st.n_normal, st.n_pairs) == (want[k][2].n_cut, want[k][2].n_hole, want[k][2].n_normal, want[k][2].n_pairs)
            # (no stage times for a replayed cut: the events are left out of the graph)
            assert st.ms_stage[5] == 0.0 and st.ms_kernel[3] == 0.0
            assert st.n_launches == want[k][2].n_launches
        dcut.close()


def test_dc_cut_without_the_flag_on_the_default_stream_and_with_other_parameters(B):
    import torch
    w = make_config(0)
    lab0, sd0, st0 = plain_cut(B, w, w.faces)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
    faces = torch.from_numpy(w.faces).cuda()
    # legacy default stream: the flag falls back to plain launches
    p = B.dc_params(); p.flags = B.DC_FLAG_GRAPH
    lab, sd = dcut.cut(faces, p)
    assert np.array_equal(lab.cpu().numpy(), lab0) and np.array_equal(sd.cpu().numpy(), sd0)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        # two parameter sets alternate: two graphs, each replayed
        q = B.dc_params(); q.flags = B.DC_FLAG_GRAPH; q.d_band = 2.0 * st0.d_band
        lab_q0, sd_q0, _ = None, None, None
        for rep in range(3):
            lab, sd = dcut.cut(faces, p)
            assert np.array_equal(lab.cpu().numpy(), lab0) and np.array_equal(sd.cpu().numpy(), sd0)
            labq, sdq = dcut.cut(faces, q)
            stq = dcut.stats()
            assert abs(stq.d_band - 2.0 * st0.d_band) < 1e-15
            if lab_q0 is None:
                lab_q0, sd_q0 = labq.cpu().numpy().copy(), sdq.cpu().numpy().copy()
            assert np.array_equal(labq.cpu().numpy(), lab_q0) and np.array_equal(sdq.cpu().numpy(), sd_q0)
        assert np.array_equal(lab_q0, lab0)                      # a wider band changes no label ...
        assert np.abs(sd_q0).max() > np.abs(sd0).max()           # ... but clamps later
        # exact far pass: not capturable (it reads counters back), runs as plain launches
        r = B.dc_params(); r.flags = B.DC_FLAG_GRAPH | B.DC_FLAG_EXACT_FAR
        labr, sdr = dcut.cut(faces, r)
        str_ = dcut.stats()
        assert str_.n_far > 0 and str_.n_far_done == str_.n_far
        assert np.array_equal(labr.cpu().numpy(), lab0)
    dcut.close()


def test_more_surfaces_than_the_graph_cache_holds(B):
    """70 distinct surface buffers through one context: the least recently used graphs are dropped and re-captured."""
    import torch
    w = make_config(0)
    lab0, sd0, _ = plain_cut(B, w, w.faces)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
        p = B.dc_params(); p.flags = B.DC_FLAG_GRAPH
        bufs = [torch.from_numpy(w.faces).cuda() for _ in range(70)]
        for rnd in range(2):
            for b in bufs:
                lab, sd = dcut.cut(b, p)
            assert np.array_equal(lab.cpu().numpy(), lab0) and np.array_equal(sd.cpu().numpy(), sd0)
        dcut.close()


def test_classify_host_with_the_copies_inside_the_graph(B):
    """dc_classify_host + DC_FLAG_GRAPH with pinned buffers: upload, cut and download are one graph (the upload beside S2);
    results must be those of the plain path for a surface that changes in place, and pageable buffers must still work."""
    import torch
    w = make_config(3, N=20, n=8)
    steps = [w.spin_faces(s) for s in (0, 5, 9)]
    want = [plain_cut(B, w, f, B.DC_FLAG_RECOMPUTE_BOXES) for f in steps]
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
        fh = torch.empty((w.n_face, 9, 3), dtype=torch.float64).pin_memory()
        lh = torch.empty(w.n_elem, dtype=torch.int8).pin_memory()
        sh = torch.empty(w.n_elem, dtype=torch.float64).pin_memory()
        for flags in (B.DC_FLAG_RECOMPUTE_BOXES | B.DC_FLAG_GRAPH, B.DC_FLAG_GRAPH):
            p = B.dc_params(); p.flags = flags
            for rep in range(2):
                for k, f in enumerate(steps):
                    fh.copy_(torch.from_numpy(f)); lh.fill_(-9); sh.fill_(99.0)
                    dcut.classify_host(fh, lh, sh, p)               # (synchronises)
                    assert np.array_equal(lh.numpy(), want[k][0]) and np.array_equal(sh.numpy(), want[k][1]), (flags, rep, k)
                    assert dcut.stats().status == 0
        # pageable host memory: the plain path (copies outside any graph)
        fp = torch.from_numpy(np.ascontiguousarray(steps[1])); lp = torch.empty(w.n_elem, dtype=torch.int8); sp = torch.empty(w.n_elem, dtype=torch.float64)
        p = B.dc_params(); p.flags = B.DC_FLAG_RECOMPUTE_BOXES | B.DC_FLAG_GRAPH
        dcut.classify_host(fp, lp, sp, p)
        assert np.array_equal(lp.numpy(), want[1][0]) and np.array_equal(sp.numpy(), want[1][1])
        dcut.close()


def test_cut_inside_the_callers_own_capture(B):
    """The caller captures the cut into a CUDA graph of its own (here torch's): the library must not start a capture of
    its own nor record its stage events, and the replayed graph must cut like the plain launches do."""
    import torch
    w = make_config(1, N=12, n=4)
    lab0, sd0, st0 = plain_cut(B, w, w.faces, B.DC_FLAG_RECOMPUTE_BOXES)
    dcut = B.DirectCut(w.xyz, w.conn27, w.adj6, max_faces=w.n_face)
    faces = torch.from_numpy(w.faces).cuda()
    p = B.dc_params(); p.flags = B.DC_FLAG_RECOMPUTE_BOXES | B.DC_FLAG_GRAPH     # (the flag is ignored under a capture)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        dcut.cut(faces, p); torch.cuda.synchronize()                             # (warm-up outside the capture)
        with torch.cuda.graph(g, stream=s):
            dcut.cut(faces, p)
    torch.cuda.synchronize()
    for rep in range(3):
        dcut.labels.fill_(-5); dcut.sdist.fill_(7.0)
        g.replay(); torch.cuda.synchronize()
        assert np.array_equal(dcut.labels.cpu().numpy(), lab0) and np.array_equal(dcut.sdist.cpu().numpy(), sd0), rep
        st = dcut.stats()
        assert st.status == 0 and (st.n_cut, st.n_hole, st.n_normal) == (st0.n_cut, st0.n_hole, st0.n_normal)
    dcut.close()
