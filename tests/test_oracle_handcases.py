"""Pins of the WHOLE oracle (orc_classify: boundary patches of an element, min over them, label, sign) against
closed forms exactly representable by quadratic geometry (SURVEY.md 8(c) P4 i-v, here with a real element on one
side).  -m "not gpu".  The same inputs go through the CUDA path in tests/test_gpu_handcases.py.
"""
import numpy as np
import pytest

from oracle import dc_oracle as O
from workloads import handcases as H

HOLE, NORMAL, CUT = 0, 1, 2
D_BAND = 3.0


def run(case, **kw):
    r = O.classify(case.xyz, case.conn27, case.faces, d_band=D_BAND, **kw)
    assert r.stats["n_depth_exceeded"] == 0
    return r


def test_flat_element_face_under_a_paraboloid():
    """Box with its top face at z = -c under z = a (x^2 + y^2) (outward normal +z at the vertex, the box is on the
    inner side): d = c at the vertex, interior-interior, r = (0,0,-c), cos = -1: HOLE, sdist = -c."""
    for a, c in ((1.0, 0.25), (2.0, 0.05), (0.25, 1.0)):
        r = run(H.assemble([H.box_hex([-0.5, -0.5, -c - 0.5], [0.5, 0.5, -c])], [H.paraboloid_face(a)]))
        assert r.labels[0] == HOLE and abs(r.sdist[0] + c) <= 1e-12


@pytest.mark.parametrize("a,z0", [(1.0, 0.52), (2.0, 0.3)])
def test_point_element_above_a_bowl_ring_of_minimisers(a, z0):
    """Degenerate element (all nodes at (u0, v0, z0)) on the axis of the bowl, z0 > 1/(2a): minimisers on the ring
    rho^2 = z0/a - 1/(2a^2), d^2 = rho^2 + (z0 - a rho^2)^2 = z0/a - 1/(4a^2); r.n = a rho^2 + z0 > 0: NORMAL.
    (Enclosure width 1e-7 L_ref: a CURVE of minimisers keeps O(ring length / size) sub-pairs alive per level, so the
    default 1e-12 is out of reach for the oracle here -- tests/test_oracle_patchpair.py does the same.)"""
    for u0, v0 in ((0.0, 0.0), (0.0625, 0.0625)):
        r = run(H.assemble([H.point_hex([u0, v0, z0])], [H.paraboloid_face(a, u0, v0)]), eps_rel=1e-7)
        rho = np.sqrt(z0 / a - 1.0 / (2 * a * a))
        assert rho <= 1.0 - max(abs(u0), abs(v0))
        d = np.sqrt(z0 / a - 1.0 / (4 * a * a))
        assert r.labels[0] == NORMAL and d - 1e-15 <= r.sdist[0] <= d + 1e-7 * r.stats["l_ref"]


def test_skew_straight_edges():
    """Box edge {(x,0,0), |x| <= 1} of the box [-1,1] x [-1,0] x [-1,0] against the edge p2 + s d2, |s| <= 1/2, of a
    flat face that extends away from the box along w: p2 = (0, .3, .4), d2 = (1, .8, -.6) (perpendicular to p2),
    w = (0, 1, .2).  Squared distance of the face point (s, t) to the box = (.3 + .8 s + t)^2 + (.4 - .6 s + .2 t)^2
    (convex; gradient at (0,0) = (0, .76), t >= 0): minimum 0.5 at s = t = 0 (textbook line-line distance
    |p2 . (e_x x d2)| / |e_x x d2| = 0.5).  n = d2 x w = (.76, -.2, 1); r = -p2; r.n = -0.34: HOLE; flipped: NORMAL."""
    d2, w, p2 = np.array([1.0, 0.8, -0.6]), np.array([0.0, 1.0, 0.2]), np.array([0.0, 0.3, 0.4])
    ex = np.array([1.0, 0.0, 0.0])
    assert abs(abs(p2 @ np.cross(ex, d2)) / np.linalg.norm(np.cross(ex, d2)) - 0.5) < 1e-15
    box = H.box_hex([-1.0, -1.0, -1.0], [1.0, 0.0, 0.0])
    r = run(H.assemble([box], [H.flat_quad(p2 - 0.5 * d2, d2, w)]))
    assert r.labels[0] == HOLE and abs(r.sdist[0] + 0.5) <= 1e-12
    r = run(H.assemble([box], [H.flat_quad(p2 - 0.5 * d2, w, d2)]))
    assert r.labels[0] == NORMAL and abs(r.sdist[0] - 0.5) <= 1e-12


def test_surface_through_the_element_is_cut():
    for a in (0.5, 2.0):
        r = run(H.assemble([H.box_hex([0.2, 0.1, -0.3], [0.6, 0.5, 0.9])], [H.paraboloid_face(a)]))
        assert r.labels[0] == CUT and r.sdist[0] == 0.0


def test_generator_structure_checks_on_every_config():
    """workloads' own structural checks on a reduced instance of every config: the wall
    surface is watertight (every patch edge's 3 nodes bit-identical in exactly two faces) and the background grid
    conforming (adj6 symmetric, neighbours share their 9 face nodes)."""
    from workloads import check_conforming, check_watertight, make_config
    for cfg, N, n in ((0, 6, 2), (1, 8, 3), (2, 8, 6), (3, 8, 4), (4, 10, 3)):
        w = make_config(cfg, N=N, n=n)
        if cfg == 4:
            per = w.n_face // 8
            assert all(check_watertight(w.faces[b * per:(b + 1) * per]) for b in range(8))
        else:
            assert check_watertight(w.faces)
        assert check_conforming(w.conn27, w.adj6)
        if cfg == 3:
            assert check_watertight(w.spin_faces(17))
