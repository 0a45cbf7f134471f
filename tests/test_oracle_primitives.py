"""Pins P1-P3 for the oracle's primitives.  -m "not gpu".

Each check is something the paper or the mathematics fixes, never the oracle re-typed:
partition of unity / nodal interpolation / finite differences for Eq. 1,
hand-computed cases for Algorithm A.2 (L689-L709), brute-force sampling for the
triangle-triangle shortest vector (L213).
"""
import os

import numpy as np
import pytest

from oracle import dc_oracle as O

RNG = np.random.default_rng(20171107)


# ----------------------------------------------------------------------------- P1
def test_shape_partition_of_unity_and_nodal():
    for t in np.linspace(-1, 1, 41):
        l, d, dd = O.shape(t)
        assert abs(l.sum() - 1) < 1e-15
        assert abs(d.sum()) < 1e-15
        assert abs(dd.sum()) < 1e-15
    nodes = [-1.0, 0.0, 1.0]
    for a, t in enumerate(nodes):
        l, _, _ = O.shape(t)
        e = np.zeros(3); e[a] = 1
        assert np.array_equal(l, e)


def test_shape_reproduces_quadratics_and_derivatives():
    # the basis must reproduce 1, t, t^2 exactly and its derivative must match d/dt
    for t in RNG.uniform(-1, 1, 20):
        l, d, dd = O.shape(t)
        x = np.array([-1.0, 0.0, 1.0])
        for p in range(3):
            assert abs(l @ x**p - t**p) < 1e-15
            assert abs(d @ x**p - (p * t**(p - 1) if p else 0.0)) < 1e-14
            assert abs(dd @ x**p - (2.0 if p == 2 else 0.0)) < 1e-14
        h = 1e-6
        lp, _, _ = O.shape(t + h); lm, _, _ = O.shape(t - h)
        assert np.allclose((lp - lm) / (2 * h), d, atol=1e-9)


def test_patch_eval_nodal_and_fd():
    X = RNG.normal(size=(9, 3))
    ref = [-1.0, 0.0, 1.0]
    for j in range(3):
        for i in range(3):
            P, _, _ = O.patch_eval(X, ref[i], ref[j])
            assert np.allclose(P, X[i + 3 * j], atol=1e-15)
    h = 1e-6
    for _ in range(10):
        u, v = RNG.uniform(-1, 1, 2)
        P, Pu, Pv = O.patch_eval(X, u, v)
        fu = (O.patch_eval(X, u + h, v)[0] - O.patch_eval(X, u - h, v)[0]) / (2 * h)
        fv = (O.patch_eval(X, u, v + h)[0] - O.patch_eval(X, u, v - h)[0]) / (2 * h)
        assert np.allclose(Pu, fu, atol=1e-8) and np.allclose(Pv, fv, atol=1e-8)


def test_patch_eval_reproduces_biquadratic_polynomial():
    # a polynomial surface of degree (2,2) sampled at the nodes is reproduced exactly
    def surf(u, v):
        return np.array([u + 0.3 * u * u * v, v - 0.2 * v * v + 0.1 * u * v, 0.5 * u * u * v * v + u - v])
    ref = [-1.0, 0.0, 1.0]
    X = np.array([surf(ref[i], ref[j]) for j in range(3) for i in range(3)])
    for _ in range(10):
        u, v = RNG.uniform(-1, 1, 2)
        assert np.allclose(O.patch_eval(X, u, v)[0], surf(u, v), atol=1e-14)


def test_bezier_conversion_matches_lagrange():
    X = RNG.normal(size=(9, 3))
    B = O.lagrange_to_bezier(X)
    # corner interpolation and convex-hull containment of samples
    for (m, _) in ((0, 0), (2, 0), (6, 0), (8, 0)):
        assert np.allclose(B[m], X[m], atol=1e-15)
    for _ in range(25):
        u, v = RNG.uniform(-1, 1, 2)
        P = O.patch_eval(X, u, v)[0]
        Q = O.bezier_eval(B, (u + 1) / 2, (v + 1) / 2)
        assert np.allclose(P, Q, atol=2e-15 * (1 + np.abs(X).max()))
        assert np.all(P >= B.min(0) - 1e-14) and np.all(P <= B.max(0) + 1e-14)


def test_lagrange_nodes_do_not_bound_patch_but_bezier_does():
    # H1 of SURVEY.md section 7: a quadratic with an overshoot beyond its node box
    X = np.zeros((9, 3))
    ref = [-1.0, 0.0, 1.0]
    for j in range(3):
        for i in range(3):
            X[i + 3 * j] = [ref[i], ref[j], [0.0, 1.0, 0.9][i]]   # z peaks beyond the node values
    zs = [O.patch_eval(X, u, 0.0)[0][2] for u in np.linspace(-1, 1, 201)]
    assert max(zs) > X[:, 2].max() + 1e-3
    B = O.lagrange_to_bezier(X)
    assert max(zs) <= B[:, 2].max() + 1e-15


def test_bezier_split_children_reproduce_parent():
    X = RNG.normal(size=(9, 3))
    B = O.lagrange_to_bezier(X)
    for direction in (0, 1):
        lo, hi = O.bezier_split(B, direction)
        for _ in range(10):
            a, b = RNG.uniform(0, 1, 2)
            if direction == 0:
                pl, ph = O.bezier_eval(B, a / 2, b), O.bezier_eval(B, 0.5 + a / 2, b)
            else:
                pl, ph = O.bezier_eval(B, a, b / 2), O.bezier_eval(B, a, 0.5 + b / 2)
            assert np.allclose(O.bezier_eval(lo, a, b), pl, atol=1e-14)
            assert np.allclose(O.bezier_eval(hi, a, b), ph, atol=1e-14)


def test_hex_face_nodes_are_the_hex_restricted_to_its_faces():
    X = RNG.normal(size=(27, 3))
    fixed = [(0, -1.0), (0, 1.0), (1, -1.0), (1, 1.0), (2, -1.0), (2, 1.0)]
    for k in range(6):
        ids = O.hex_face_nodes(k)
        assert len(set(ids.tolist())) == 9
        ax, val = fixed[k]
        for _ in range(5):
            a, b = RNG.uniform(-1, 1, 2)
            ref = [a, b]
            ref.insert(ax, val)
            assert np.allclose(O.patch_eval(X[ids], a, b)[0], O.hex_eval(X, *ref), atol=1e-14)
    # the centre node 13 is interior: on no boundary patch
    allb = set()
    for k in range(6):
        allb |= set(O.hex_face_nodes(k).tolist())
    assert allb == set(range(27)) - {13}


# ----------------------------------------------------------------------------- P2
def test_box_dist_hand_cases(golden_dir):
    rows = [l for l in open(os.path.join(golden_dir, "a2_box_dist_cases.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) >= 8
    for row in rows:
        v = [float(x) for x in row.split()]
        b1, b2, want = v[0:6], v[6:12], v[12]
        assert abs(O.box_dist(b1, b2) - want) < 1e-14
        assert abs(O.box_dist(b2, b1) - want) < 1e-14   # symmetric


def test_box_dist_is_a_lower_bound_on_point_distances():
    for _ in range(50):
        c1, c2 = RNG.uniform(-2, 2, 3), RNG.uniform(-2, 2, 3)
        h1, h2 = RNG.uniform(0, 1, 3), RNG.uniform(0, 1, 3)
        b1 = np.concatenate([c1 - h1, c1 + h1]); b2 = np.concatenate([c2 - h2, c2 + h2])
        p = c1 + RNG.uniform(-1, 1, (200, 3)) * h1
        q = c2 + RNG.uniform(-1, 1, (200, 3)) * h2
        dmin = np.linalg.norm(p[:, None] - q[None], axis=2).min()
        assert O.box_dist(b1, b2) <= dmin + 1e-14


# ----------------------------------------------------------------------------- P3
def _bary_grid(n):
    pts = []
    for i in range(n + 1):
        for j in range(n + 1 - i):
            pts.append((i / n, j / n, 1 - i / n - j / n))
    return np.array(pts)


def _brute_tri_tri(A, B, n=60):
    W = _bary_grid(n)
    PA, PB = W @ A, W @ B
    return np.sqrt(((PA[:, None] - PB[None]) ** 2).sum(2)).min()


def test_tri_tri_vs_brute_force_random():
    for it in range(60):
        A = RNG.normal(size=(3, 3)); B = RNG.normal(size=(3, 3)) + RNG.normal(size=3) * (it % 3)
        d, wa, wb = O.tri_tri_dist(A, B)
        assert abs(wa.sum() - 1) < 1e-12 and abs(wb.sum() - 1) < 1e-12
        assert (wa >= -1e-12).all() and (wb >= -1e-12).all()
        # the reported closest points really are at distance d
        assert abs(np.linalg.norm(wa @ A - wb @ B) - d) < 1e-12
        db = _brute_tri_tri(A, B)
        size = max(np.ptp(A, axis=0).max(), np.ptp(B, axis=0).max())
        assert d <= db + 1e-12            # exact min is below any sampled value
        assert db - d <= 2.5 * size / 60  # and within the sample spacing


def test_tri_tri_special_cases():
    A = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0]], float)
    # parallel, shifted in z
    d, _, _ = O.tri_tri_dist(A, A + [0, 0, 0.7]); assert abs(d - 0.7) < 1e-15
    # coplanar, disjoint: gap along x between vertex (1,0,0) and edge x=1.5
    B = np.array([[1.5, -1, 0], [1.5, 1, 0], [3, 0, 0]], float)
    d, _, _ = O.tri_tri_dist(A, B); assert abs(d - 0.5) < 1e-15
    # coplanar, one inside the other
    d, _, _ = O.tri_tri_dist(A * 4 - [1, 1, 0], A * 0.2 + [0.3, 0.3, 0]); assert d < 1e-15
    # piercing: segment through the interior
    B = np.array([[0.2, 0.2, -1], [0.2, 0.2, 1], [5, 5, 1]], float)
    d, wa, wb = O.tri_tri_dist(A, B); assert d == 0.0
    assert np.allclose(wa @ A, wb @ B, atol=1e-14)
    # vertex above the interior
    B = np.array([[0.25, 0.25, 0.3], [2, 2, 1], [2, 3, 2]], float)
    d, _, _ = O.tri_tri_dist(A, B); assert abs(d - 0.3) < 1e-15
    # skew edges: textbook segment-segment
    A2 = np.array([[0, 0, 0], [1, 0, 0], [0.5, -1, 0]], float)
    B2 = np.array([[0.5, 0.5, 0.4], [0.5, 1.5, 0.4], [0.5, 1.0, 3]], float)
    d, _, _ = O.tri_tri_dist(A2, B2); assert abs(d - np.hypot(0.5, 0.4)) < 1e-15
    # degenerate (zero-area) triangle = a segment
    B3 = np.array([[0.2, 0.2, 1.0], [0.2, 0.2, 1.0], [0.2, 0.2, 2.0]], float)
    d, _, _ = O.tri_tri_dist(A, B3); assert abs(d - 1.0) < 1e-15


def test_tri_tri_symmetry_and_rigid_motion():
    from workloads import random_rotation
    for _ in range(20):
        A = RNG.normal(size=(3, 3)); B = RNG.normal(size=(3, 3)) + [1.5, 0, 0]
        d1, _, _ = O.tri_tri_dist(A, B)
        d2, _, _ = O.tri_tri_dist(B, A)
        assert abs(d1 - d2) < 1e-13
        Rm = random_rotation(RNG); t = RNG.normal(size=3)
        d3, _, _ = O.tri_tri_dist(A @ Rm.T + t, B @ Rm.T + t)
        assert abs(d1 - d3) < 1e-12
        # vertex order must not matter
        d4, _, _ = O.tri_tri_dist(A[[2, 0, 1]], B[[1, 2, 0]])
        assert abs(d1 - d4) < 1e-13
