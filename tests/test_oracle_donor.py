"""Pins of the donor-search oracle (oracle/donor_oracle.py; PAPER.md 4.3 Eq. 1-5).  -m "not gpu".

* its map x(X) equals the C oracle's orc_hex_eval (itself pinned by P1: partition of unity, exact quadratics) and its
  Jacobian equals central differences;
* straight-sided box element: the inverse is the affine closed form;
* round trip on a curved grid: points made from known (element, X) come back with that element and X; a point on a
  shared face comes back with BOTH elements; a point outside the grid with none.
"""
import numpy as np

from oracle import dc_oracle as O
from oracle import donor_oracle as D
from workloads import make_config


def test_map_and_jacobian():
    w = make_config(1, N=4, n=2)
    rng = np.random.default_rng(0)
    for _ in range(20):
        e = rng.integers(w.n_elem); xi = rng.uniform(-1, 1, 3)
        X27 = w.xyz[w.conn27[e]]
        x, J = D.hex_map(X27, xi)
        assert np.abs(x - O.hex_eval(X27, *xi)).max() < 1e-15
        h = 1e-6
        for a in range(3):
            d = np.zeros(3); d[a] = h
            fd = (O.hex_eval(X27, *(xi + d)) - O.hex_eval(X27, *(xi - d))) / (2 * h)
            assert np.abs(J[:, a] - fd).max() < 1e-9


def test_affine_closed_form():
    w = make_config(0, N=2, n=2)                       # straight hexes of edge 1 on [-1,1]^3
    boxes = D.element_boxes(w.xyz, w.conn27)
    p = np.array([0.3, -0.45, 0.8])
    hits = D.find_donors(w.xyz, w.conn27, [p], boxes)[0]
    assert len(hits) == 1
    (e, xi), = hits.items()
    lo, hi = boxes[e, :3], boxes[e, 3:]
    assert np.all(lo <= p) and np.all(p <= hi)
    assert np.abs(xi - (2.0 * (p - lo) / (hi - lo) - 1.0)).max() < 1e-13


def test_round_trip_shared_face_and_outside():
    w = make_config(1, N=5, n=2)
    boxes = D.element_boxes(w.xyz, w.conn27)
    rng = np.random.default_rng(3)
    es = rng.integers(w.n_elem, size=25)
    xis = rng.uniform(-0.95, 0.95, (25, 3))
    pts = np.array([O.hex_eval(w.xyz[w.conn27[e]], *xi) for e, xi in zip(es, xis)])
    res = D.find_donors(w.xyz, w.conn27, pts, boxes)
    for e, xi, hits in zip(es, xis, res):
        assert list(hits) == [int(e)] and np.abs(hits[int(e)] - xi).max() < 1e-10
    # a point on the xi = +1 face of element 0 also lies on the xi = -1 face of its neighbour
    nb = int(w.adj6[0, 1])
    p = O.hex_eval(w.xyz[w.conn27[0]], 1.0, 0.3, -0.2)
    hits = D.find_donors(w.xyz, w.conn27, [p], boxes)[0]
    assert sorted(hits) == sorted([0, nb])
    assert np.abs(hits[0] - [1.0, 0.3, -0.2]).max() < 1e-9 and np.abs(hits[nb] - [-1.0, 0.3, -0.2]).max() < 1e-9
    assert D.find_donors(w.xyz, w.conn27, [[3.0, 0.0, 0.0]], boxes)[0] == {}
