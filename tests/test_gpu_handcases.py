"""-m gpu: the hand-built cases through the C ABI -- the tie rule (Fig. 6, Fig. 14), the
ambiguity band (BASELINE.json north_star) and the closest-point closed forms of SURVEY.md 8(c) P4 given to the CUDA
Newton IN ISOLATION (one element, one face), at the default theta_leaf.

Each case is checked against the geometry's closed form (written in tests/test_oracle_ties.py /
tests/test_oracle_handcases.py, where the oracle is pinned to it) AND against the oracle on the same input.
"""
import numpy as np
import pytest

from oracle import dc_oracle as O
from workloads import handcases as H

pytestmark = pytest.mark.gpu
HOLE, NORMAL, CUT = 0, 1, 2
D_BAND = 3.0
TOL_REL = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_1711_07663_b200._build import build_lib
    build_lib()
    from paper_1711_07663_b200 import binding
    return binding


def gpu(B, case, d_band=D_BAND, **pk):
    dcut = B.DirectCut(case.xyz, case.conn27, case.adj6, max_faces=case.n_face,
                       max_pairs=max(1 << 16, case.n_elem * case.n_face))
    p = B.dc_params()
    if d_band is not None:
        p.d_band = d_band
    for k, v in pk.items():
        setattr(p, k, v)
    dcut.set_cut_surface(case.faces)
    labels, sdist = dcut.classify(p)
    st = dcut.stats()
    out = labels.cpu().numpy().copy(), sdist.cpu().numpy().copy(), st
    dcut.close()
    return out


def both(B, case, d_band=D_BAND, tol_rel=TOL_REL, **okw):
    kw = dict(okw) if d_band is None else dict(okw, d_band=d_band)
    ref = O.classify(case.xyz, case.conn27, case.faces, **kw)
    lab, sd, st = gpu(B, case, d_band)
    L = ref.stats["l_ref"]
    amb = (ref.flags & O.FLAG_AMBIGUOUS) != 0
    assert np.array_equal(lab[~amb], ref.labels[~amb]), (lab, ref.labels)
    assert np.abs(sd - ref.sdist)[~amb].max(initial=0.0) <= tol_rel * L, (sd, ref.sdist)
    assert st.n_sign_ambiguous == ref.stats["n_sign_ambiguous"]
    assert st.n_ambiguous == ref.stats["n_ambiguous"]
    assert st.status == 0 and st.n_depth_exceeded == 0
    return lab, sd, st, ref


# ------------------------------------------------------------------------------------------- tie rule
ELEM_KNIFE = H.box_hex([1.0, 0.4, -0.2], [1.2, 0.6, -0.1])


@pytest.mark.parametrize("order", [(0, 1), (1, 0)])
def test_knife_edge_opposite_sign_tie(B, order):
    faces = H.knife_edge_faces()
    lab, sd, st, ref = both(B, H.assemble([ELEM_KNIFE], [faces[order[0]], faces[order[1]]]))
    assert lab[0] == NORMAL and abs(sd[0] - np.sqrt(1.01)) <= 1e-12 and st.n_sign_ambiguous == 1


def test_tie_window(B):
    for delta, want, tied in ((1e-6, HOLE, 0), (2e-10, NORMAL, 1), (-1e-6, NORMAL, 0)):
        lab, sd, st, ref = both(B, H.assemble([ELEM_KNIFE], H.knife_edge_faces(extend_a=delta)))
        assert lab[0] == want and st.n_sign_ambiguous == tied, delta


def test_plate_slot_and_corners(B):
    lab, sd, st, _ = both(B, H.assemble([H.box_hex([-0.2, -0.2, -0.1], [0.2, 0.2, 0.1])], H.plate_faces(0.5)))
    assert lab[0] == HOLE and abs(sd[0] + 0.4) <= 1e-12 and st.n_sign_ambiguous == 0
    hexes = [H.box_hex([-0.2, -0.2, -0.1], [0.2, 0.2, 0.1]), H.box_hex([0.3, 0.3, 0.05], [0.5, 0.5, 0.25])]
    lab, sd, st, _ = both(B, H.assemble(hexes, H.slot_faces(0.5)))
    assert list(lab) == [NORMAL, NORMAL] and np.abs(sd - [0.4, 0.25]).max() <= 1e-12 and st.n_sign_ambiguous == 0
    A, Bf = H.corner_faces()
    for faces in ([A, Bf], [Bf, A]):
        lab, sd, st, _ = both(B, H.assemble([H.box_hex([0.3, 0.4, 0.1], [0.5, 0.6, 0.2]),
                                             H.box_hex([0.2, 0.4, 0.2], [0.4, 0.6, 0.4])], faces))
        assert list(lab) == [NORMAL, NORMAL] and np.abs(sd - [np.sqrt(0.1), np.sqrt(0.08)]).max() <= 1e-12


def test_tie_rule_in_the_seedless_query(B):
    """With the default band (max element box diagonal, 0.3 here) the knife-edge element is OUTSIDE the band and has
    no neighbours: its sign comes from the exhaustive nearest-face query of a seedless component (k_seedless), which
    applies the same tie rule; sdist is the clamp +d_band."""
    faces = H.knife_edge_faces()
    case = H.assemble([ELEM_KNIFE], faces)
    ref = O.classify(case.xyz, case.conn27, case.faces)
    lab, sd, st = gpu(B, case, d_band=None)
    assert lab[0] == ref.labels[0] == NORMAL and st.n_pairs == 0 and st.n_seedless_components == 1
    assert abs(sd[0] - ref.sdist[0]) <= 1e-14 and abs(sd[0] - st.d_band) <= 1e-14


# ------------------------------------------------------------------------------------------- ambiguity band
def test_ambiguity_band_counts_agree(B):
    tau, a = 1e-7, 1e-9
    gaps = [tau - 0.5 * a, tau + 0.5 * a, tau - 5 * a, tau + 5 * a, tau - 1.5 * a, tau + 1.5 * a, 0.0, 0.05]
    hexes = [H.box_hex([0.05 + 0.1 * i, 0.4, g], [0.10 + 0.1 * i, 0.5, g + 0.05]) for i, g in enumerate(gaps)]
    case = H.assemble(hexes, [H.flat_quad([0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [0.0, 1.0, 0.0])])
    ref = O.classify(case.xyz, case.conn27, case.faces)
    lab, sd, st = gpu(B, case, d_band=None)
    assert ref.stats["n_ambiguous"] == 2 and st.n_ambiguous == 2
    assert np.array_equal(lab, [CUT, NORMAL, CUT, NORMAL, CUT, NORMAL, CUT, NORMAL])
    assert np.array_equal(lab, ref.labels) and np.abs(sd - ref.sdist).max() <= 1e-15


# ------------------------------------------------------------------------------------------- P4 in isolation
def test_p4_flat_vs_paraboloid(B):
    """(ii) flat element face z = -c under the paraboloid z = a (x^2 + y^2): interior-interior minimum c at the vertex."""
    for a, c in ((1.0, 0.25), (2.0, 0.05), (0.25, 1.0)):
        case = H.assemble([H.box_hex([-0.5, -0.5, -c - 0.5], [0.5, 0.5, -c])], [H.paraboloid_face(a)])
        lab, sd, st, _ = both(B, case)
        assert lab[0] == HOLE and abs(sd[0] + c) <= 1e-12


def ring_distance(a, z0):
    return np.sqrt(z0 / a - 1.0 / (4.0 * a * a))


@pytest.mark.parametrize("a,z0", [(1.0, 0.7), (1.0, 0.52), (2.0, 0.3), (0.75, 0.8), (4.0, 0.2)])
def test_p4_ring_of_minimisers_two_basins_in_a_leaf(B, a, z0):
    """(iii) a point on the axis of the bowl beyond its focal distance (z0 > 1/(2a)): the vertex below it is a local
    MAXIMUM of the distance, the minimisers form the ring rho^2 = z0/a - 1/(2a^2), d = sqrt(z0/a - 1/(4a^2)).
    The vertex is moved over a leaf centre, a leaf corner and a generic point, so that the ring crosses leaves of
    the subdivision in every way (two basins inside one leaf is what the theta rule has to survive)."""
    assert z0 > 1.0 / (2 * a)
    for i, (u0, v0) in enumerate(((0.0, 0.0), (0.0625, 0.0625), (0.125, 0.125), (0.03125, -0.21875), (0.3, 0.1234),
                                  (-0.5, 0.5), (0.015625, 0.046875))):
        case = H.assemble([H.point_hex([u0, v0, z0])], [H.paraboloid_face(a, u0, v0)])
        if i < 2:
            # (a curve of minimisers: the oracle's enclosure is affordable to 1e-7 L_ref only -- its upper end, the value
            # it reports, is in practice exact; the closed form below is the sharp check)
            lab, sd, st, ref = both(B, case, tol_rel=1.1e-7, eps_rel=1e-7)
            assert sd[0] <= ref.sdist[0] + 1e-12
        else:
            lab, sd, st = gpu(B, case)
            assert st.status == 0 and st.n_depth_exceeded == 0
        rho = np.sqrt(z0 / a - 1.0 / (2 * a * a))
        assert rho <= 1.0 - max(abs(u0), abs(v0))              # the whole ring lies on the patch
        assert abs(sd[0] - ring_distance(a, z0)) <= 1e-11, (u0, v0, sd[0] - ring_distance(a, z0))
        assert lab[0] == NORMAL


def test_p4_small_cube_above_the_bowl(B):
    """The same bowl under a small (non-degenerate) curved element: no closed form, the oracle is the reference."""
    rng = np.random.default_rng(5)
    for a, z0 in ((1.0, 0.7), (2.0, 0.4), (4.0, 0.3)):
        for _ in range(3):
            c = np.array([rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2), z0])
            X = H.box_hex(c - 0.02, c + 0.02)
            X = X + 0.004 * np.sin(40.0 * X[:, [1, 2, 0]])              # curved, still a valid hex
            both(B, H.assemble([X], [H.paraboloid_face(a, rng.uniform(-0.1, 0.1), rng.uniform(-0.1, 0.1))]))


def skew_edge_case(flip=False):
    """(iv) box edge {(x, 0, 0)} against the edge p2 + s d2 of a flat face; common perpendicular c = (0, 0.3, 0.4),
    |c| = 0.5; the face extends away from the box along w."""
    d2, w, p2 = np.array([1.0, 0.8, -0.6]), np.array([0.0, 1.0, 0.2]), np.array([0.0, 0.3, 0.4])
    face = H.flat_quad(p2 - 0.5 * d2, w, d2) if flip else H.flat_quad(p2 - 0.5 * d2, d2, w)
    return H.assemble([H.box_hex([-1.0, -1.0, -1.0], [1.0, 0.0, 0.0])], [face])


def test_p4_skew_straight_edges(B):
    lab, sd, st, _ = both(B, skew_edge_case())
    assert lab[0] == HOLE and abs(sd[0] + 0.5) <= 1e-12          # n = d2 x w = (0.76, -0.2, 1), r = -c: r.n < 0
    lab, sd, st, _ = both(B, skew_edge_case(flip=True))
    assert lab[0] == NORMAL and abs(sd[0] - 0.5) <= 1e-12


def test_p4_transversal_intersection(B):
    """(v) the bowl passes through the element: CUT, sdist = 0 (the enclosure collapses below tau)."""
    for a in (0.5, 2.0):
        case = H.assemble([H.box_hex([0.2, 0.1, -0.3], [0.6, 0.5, 0.9])], [H.paraboloid_face(a)])
        lab, sd, st, _ = both(B, case)
        assert lab[0] == CUT and sd[0] == 0.0


def test_p4_random_curved_pairs_vs_oracle(B):
    """Random curved single element / single face pairs at distances from touching to far: the CUDA solve alone
    (no neighbouring faces to hide a missed minimum) against the oracle's enclosure."""
    rng = np.random.default_rng(17)
    for trial in range(24):
        a = rng.uniform(-3.0, 3.0)
        F = H.quad_from(lambda s, t: [s + 0.1 * t * t, t - 0.1 * s * s, a * (s - 0.2) * (t + 0.1) + 0.3 * a * s * s])
        c = np.array([rng.uniform(-0.8, 0.8), rng.uniform(-0.8, 0.8), rng.uniform(-1.0, 1.0)])
        X = H.box_hex(c - 0.15, c + 0.15)
        X = X + 0.03 * np.sin(9.0 * X[:, [2, 0, 1]] + trial)
        both(B, H.assemble([X], [F]))
