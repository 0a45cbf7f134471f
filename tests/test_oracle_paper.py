"""Pins of the oracle of the paper's approximate mode (oracle/paper_oracle.c; Algorithms A.1-A.4, L670-L845;
SURVEY.md 8(f) NEXT-3).  -m "not gpu".

* OBB (L195): a rotated box with distinct edges gives back its own axes and half-extents; a cube gives the identity.
* A.1 (L672-L687): hand case on an axis-aligned unit cube.
* whole pass: where the geometry is LINEAR (straight-sided hexes, flat faces) the paper's linearisation is exact, so
  its distance and label must equal the closed form (and the exact oracle): parallel plates, edge-edge, corner-corner.
* config 0 (sphere): every label it computes equals the closed-form box-vs-sphere label of BASELINE.json's north star
  (tests/golden/config0_closed_form_census.txt: 136 HOLE / 296 CUT), distances within the linearisation error of a
  6 x 4 x 4 sphere.
"""
import numpy as np

from oracle import dc_oracle as O
from oracle import paper_oracle as P
from workloads import handcases as H
from workloads import make_config

HOLE, NORMAL, CUT = 0, 1, 2


def rot(axis, ang):
    axis = np.asarray(axis, float) / np.linalg.norm(axis)
    K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    return np.eye(3) + np.sin(ang) * K + (1 - np.cos(ang)) * K @ K


def corners(half):
    return np.array([[sx * half[0], sy * half[1], sz * half[2]] for sz in (-1, 1) for sy in (-1, 1) for sx in (-1, 1)], float)


def test_obb_of_a_rotated_box_is_the_box():
    half = np.array([0.5, 1.25, 2.0])
    Rm = rot([1.0, 2.0, -0.5], 0.83)
    c0 = np.array([0.3, -1.1, 2.2])
    X8 = corners(half) @ Rm.T + c0
    R, ext, ecg = P.obb(X8)
    assert np.abs(ecg - c0).max() < 1e-14
    assert np.abs(R @ R.T - np.eye(3)).max() < 1e-14                       # orthonormal axes
    # each axis is +- a column of Rm, and the extents along it are centre +- that column's half-length
    M = np.abs(R @ Rm)                                                      # |cos| between found axes and true axes
    perm = M.argmax(axis=1)
    assert sorted(perm) == [0, 1, 2] and np.abs(M[np.arange(3), perm] - 1.0).max() < 1e-12
    for a in range(3):
        mid, hw = 0.5 * (ext[a] + ext[3 + a]), 0.5 * (ext[3 + a] - ext[a])
        assert abs(hw - half[perm[a]]) < 1e-12 and abs(mid - R[a] @ c0) < 1e-12
    R, ext, ecg = P.obb(corners([1.0, 1.0, 1.0]))                           # cube: covariance = identity, no rotation at all
    assert np.array_equal(R, np.eye(3)) and np.array_equal(ext, [-1, -1, -1, 1, 1, 1])


def test_a1_hand_case():
    """Unit cube [0,1]^3 (axes = identity, extents [0,1]^3, centroid (.5,.5,.5)); face with corner nodes
    (2,0,0) (3,0,0) (3,1,0) (2,1,0): box gap 1 along x only, face centroid (2.5,.5,0): d_xc = sqrt(4 + .25):
    Distance = .01 sqrt(4.25) + 1 (Algorithm A.1 line 12)."""
    R, ext, ecg = np.eye(3), np.array([0, 0, 0, 1, 1, 1.0]), np.array([0.5, 0.5, 0.5])
    F4 = np.array([[2, 0, 0], [3, 0, 0], [3, 1, 0], [2, 1, 0]], float)
    assert abs(P.a1(R, ext, ecg, F4) - (0.01 * np.sqrt(4.25) + 1.0)) < 1e-15
    F4 = np.array([[2, 3, 0], [3, 3, 0], [3, 4, 0], [2, 4, 0]], float) + np.array([0, 0, -2.0])   # gaps 1, 2, 1 (z: 0 - (-2)... below)
    d_b = np.sqrt(1.0 + 4.0 + 4.0)                                          # x gap 1, y gap 2, z gap 2 (face at z = -2)
    d_xc = np.linalg.norm(np.array([2.5, 3.5, -2.0]) - ecg)
    assert abs(P.a1(R, ext, ecg, F4) - (0.01 * d_xc + d_b)) < 1e-15


def both(case):
    ex = O.classify(case.xyz, case.conn27, case.faces, d_band=3.0)
    pm = P.classify(case.xyz, case.conn27, case.faces, d_band=3.0, l_ref=ex.stats["l_ref"])
    return ex, pm


def test_linear_geometry_is_exact():
    # parallel plates: box under a flat face at gap 0.25 (face normal +z, box below: inside -> HOLE)
    case = H.assemble([H.box_hex([0.2, 0.2, -1.0], [0.6, 0.6, -0.25])], [H.flat_quad([0, 0, 0], [1, 0, 0], [0, 1, 0])])
    ex, pm = both(case)
    assert pm.labels[0] == ex.labels[0] == HOLE and abs(pm.sdist[0] + 0.25) < 1e-13 and abs(ex.sdist[0] + 0.25) < 1e-12
    # above the face: NORMAL, corner-to-interior
    case = H.assemble([H.box_hex([0.2, 0.2, 0.5], [0.6, 0.6, 0.9])], [H.flat_quad([0, 0, 0], [1, 0, 0], [0, 1, 0])])
    ex, pm = both(case)
    assert pm.labels[0] == NORMAL and abs(pm.sdist[0] - 0.5) < 1e-13
    # corner to corner: box [1.3,1.7]^2 x [0.4, 0.8] against the unit face: nearest points (1,1,0) and (1.3,1.3,0.4)
    case = H.assemble([H.box_hex([1.3, 1.3, 0.4], [1.7, 1.7, 0.8])], [H.flat_quad([0, 0, 0], [1, 0, 0], [0, 1, 0])])
    ex, pm = both(case)
    d = np.sqrt(0.09 + 0.09 + 0.16)
    assert pm.labels[0] == ex.labels[0] == NORMAL and abs(pm.sdist[0] - d) < 1e-13 and abs(ex.sdist[0] - d) < 1e-12
    # the face passes through the box: CUT
    case = H.assemble([H.box_hex([0.2, 0.2, -0.1], [0.6, 0.6, 0.3])], [H.flat_quad([0, 0, 0], [1, 0, 0], [0, 1, 0])])
    ex, pm = both(case)
    assert pm.labels[0] == ex.labels[0] == CUT and pm.sdist[0] == 0.0


def test_l215_normal_averaging_fails_inside_a_thin_plate():
    """The element midway between the two faces of a plate is at the same distance (0.4) from both; their normals are
    opposite.  L215 read literally ("the corresponding normals are averaged") gives a zero vector and no sign -- the
    case section 4.4 (L294) repairs ("same sign: never average"), which is the rule the exact mode uses (reading A6).
    The approximate mode keeps L215: the distance is right, the label is not."""
    ex, pm = both(H.assemble([H.box_hex([-0.2, -0.2, -0.1], [0.2, 0.2, 0.1])], H.plate_faces(0.5)))
    assert ex.labels[0] == HOLE and abs(ex.sdist[0] + 0.4) < 1e-12
    assert abs(abs(pm.sdist[0]) - 0.4) < 1e-13 and pm.labels[0] == NORMAL
    # off the mid-plane the nearest face alone decides and both modes agree
    ex, pm = both(H.assemble([H.box_hex([-0.2, -0.2, -0.05], [0.2, 0.2, 0.15])], H.plate_faces(0.5)))
    assert pm.labels[0] == ex.labels[0] == HOLE and abs(pm.sdist[0] - ex.sdist[0]) < 1e-12


def test_config0_labels_equal_the_closed_form():
    w = make_config(0)
    ex = O.classify(w.xyz, w.conn27, w.faces, nproc=4)
    pm = P.classify(w.xyz, w.conn27, w.faces, d_band=ex.stats["d_band"], l_ref=ex.stats["l_ref"], nproc=4)
    have = pm.labels >= 0
    # closed form (BASELINE.json north_star): box [lo,hi] against the sphere R = 0.5
    lo, hi = w.xyz[w.conn27[:, 0]], w.xyz[w.conn27[:, 26]]
    d_near = np.linalg.norm(np.clip(0.0, lo, hi), axis=1)
    d_far = np.linalg.norm(np.maximum(np.abs(lo), np.abs(hi)), axis=1)
    closed = np.where(d_far < 0.5, HOLE, np.where(d_near > 0.5, NORMAL, CUT))
    # the 24 elements that touch the sphere in one lattice node are CUT under reading A3 (tau > 0)
    touch = np.abs(d_near - 0.5) < 1e-12
    closed[touch] = CUT
    assert have.sum() == 1352 and (pm.flags[~have] == P.FLAG_FAR).all()
    assert np.array_equal(pm.labels[have], closed[have])
    assert (pm.labels == HOLE).sum() == 136 and (pm.labels == CUT).sum() == 296
    # distances: the linear triangles of a 6 x 4 x 4 sphere lie up to ~0.02 inside it
    assert np.abs(pm.sdist[have] - ex.sdist[have]).max() < 0.01
