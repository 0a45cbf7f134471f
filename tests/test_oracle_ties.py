"""Pins for steps 5 and 6 of the oracle's labelling rule:  -m "not gpu".

Step 5, the tie rule.  PAPER.md L151 (section 4.1): "In the case of an element being approximately equidistant
from multiple faces ... If one of the vector/normal combinations has a significantly larger dot product
magnitude, that dot product is used to determine the blanking status. ... If the dot products are of similar
magnitude and produce the same result however, averaging should not be used"; L294 (section 4.4, the slot of
Fig. 14): "with equidistant faces on both sides of these elements giving the same blanking status, the face
normals must not be averaged ...; instead, the face normal/minimum vector combination yielding the largest
magnitude dot product should be used."  Reading A6: among the faces within t_tie = 1e-9 L_ref of the
minimum the one with the largest |cos(r, n)| decides; opposite-sign ties are flagged (ORC_FLAG_SIGN_AMBIG).

Step 6, the ambiguity flag (BASELINE.json north_star): an element is ambiguous iff its distance enclosure meets
[tau - 1e-9 L_ref, tau + 1e-9 L_ref].

Every expected value below follows from the geometry alone (flat faces, box elements): the closest points, the
minimal vector r and the face normals are written out in the comments; a rule that took the SMALLEST |cos|, the
first or the last tied face, or the average of the tied normals fails at least one case.
"""
import numpy as np
import pytest

from oracle import dc_oracle as O
from workloads import handcases as H

HOLE, NORMAL, CUT = 0, 1, 2
D_BAND = 3.0          # every element of these cases is inside the band: the exact distance is reported


def run(case, **kw):
    kw.setdefault("d_band", D_BAND)
    return O.classify(case.xyz, case.conn27, case.faces, **kw)


def flag(r, bit):
    return (r.flags & bit) != 0


# ------------------------------------------------------------------------------------------- Fig. 6(a)
# Wedge body {z < 0, z > x/2, x < 0}; its edge is the y axis.  Element box x in [1, 1.2], y in [0.4, 0.6],
# z in [-0.2, -0.1]: OUTSIDE the body.  Its nearest edge {x = 1, z = -0.1} is parallel to the wedge's edge, so both
# faces tie at distance sqrt(1 + 0.01) with r = (1, 0, -0.1):
#   face A (top, n = +z):            cos = -0.1 / |r| = -0.0995   -> "inside"  (wrong: A's plane is seen from below)
#   face B (underside, n = (1,0,-2)/sqrt5): cos = (1 + 0.2) / (sqrt5 |r|) = +0.534 -> "outside" (right)
# The larger |cos| (the face that "sees" the element better) wins: NORMAL, and the disagreement is flagged.
ELEM_KNIFE = H.box_hex([1.0, 0.4, -0.2], [1.2, 0.6, -0.1])
D_KNIFE = np.sqrt(1.0 + 0.01)


@pytest.mark.parametrize("order", [(0, 1), (1, 0)])
def test_knife_edge_opposite_sign_tie_largest_cos_wins(order):
    faces = H.knife_edge_faces()
    case = H.assemble([ELEM_KNIFE], [faces[order[0]], faces[order[1]]])
    r = run(case)
    assert r.labels[0] == NORMAL
    assert abs(r.sdist[0] - D_KNIFE) <= 1e-12
    assert flag(r, O.FLAG_SIGN_AMBIG)[0] and r.stats["n_sign_ambiguous"] == 1
    assert r.nearest[0] == order.index(1)            # face B, wherever it sits in the list
    assert not flag(r, O.FLAG_AMBIGUOUS)[0]


def test_knife_edge_mirror_element_inside_the_body():
    """The same wedge, the element INSIDE it next to the underside: x in [-0.9,-0.8], z in [-0.35, -0.3]
    (the body at x = -0.8 spans z in (-0.4, 0)).  Nearest: face B alone (plane distance (x - 2z)/sqrt5 at the
    corner (-0.8, *, -0.35) = -0.1/sqrt5 ... inside), A is 0.3 away: no tie, HOLE, no flag."""
    case = H.assemble([H.box_hex([-0.9, 0.4, -0.35], [-0.8, 0.6, -0.3])], H.knife_edge_faces())
    r = run(case)
    # distance to the plane x - 2z = 0 from (-0.8, y, -0.35): |-0.8 + 0.7| / sqrt5
    assert r.labels[0] == HOLE and abs(r.sdist[0] + 0.1 / np.sqrt(5.0)) <= 1e-12
    assert not flag(r, O.FLAG_SIGN_AMBIG)[0] and r.nearest[0] == 1


def test_tie_window_is_t_tie():
    """Face A extended towards the element by delta makes it NEARER by ~delta: beyond t_tie = 1e-9 L_ref the
    nearest face alone decides (A: cos < 0 -> HOLE, no flag); within t_tie both count (B wins, flagged)."""
    # L_ref = 1 + delta (x extent of the surface nodes); |r| shrinks by delta / |r| to first order
    for delta, lab, tied in ((1e-6, HOLE, False), (2e-10, NORMAL, True), (-1e-6, NORMAL, False)):
        case = H.assemble([ELEM_KNIFE], H.knife_edge_faces(extend_a=delta))
        r = run(case)
        assert r.labels[0] == lab, delta
        assert bool(flag(r, O.FLAG_SIGN_AMBIG)[0]) == tied, delta
        dA = np.sqrt((1.0 - delta) ** 2 + 0.01)
        assert abs(abs(r.sdist[0]) - min(dA, D_KNIFE)) <= 1e-12, delta


# ------------------------------------------------------------------------------------------- Fig. 6(b) / Fig. 14
def test_plate_interior_element_same_sign_tie_is_not_averaged():
    """Solid plate |z| < 0.5, element centred in it (z in [-0.1, 0.1]): both walls 0.4 away, r = (0,0,-0.4) to the
    top wall (n = +z, cos = -1) and (0,0,+0.4) to the bottom wall (n = -z, cos = -1).  Both say HOLE; the AVERAGE of
    the two normals is the zero vector (Fig. 6(b): 'several normals can easily cancel out'), which would say
    nothing.  Expected: HOLE, sdist = -0.4, no sign ambiguity."""
    case = H.assemble([H.box_hex([-0.2, -0.2, -0.1], [0.2, 0.2, 0.1])], H.plate_faces(0.5))
    r = run(case)
    assert r.labels[0] == HOLE and abs(r.sdist[0] + 0.4) <= 1e-12
    assert not flag(r, O.FLAG_SIGN_AMBIG)[0]


def test_slot_centred_elements_are_field():
    """PAPER.md Fig. 14: elements 'directly centered in the slot' (fluid |z| < 0.5): both walls tie, both cos = +1:
    NORMAL, never HOLE, no flag; an element off the centre line is decided by the nearer wall alone."""
    hexes = [H.box_hex([-0.2, -0.2, -0.1], [0.2, 0.2, 0.1]),       # centred: 0.4 from both walls
             H.box_hex([0.3, 0.3, 0.05], [0.5, 0.5, 0.25])]        # off centre: 0.25 from the upper wall
    case = H.assemble(hexes, H.slot_faces(0.5))
    r = run(case)
    assert list(r.labels) == [NORMAL, NORMAL]
    assert np.abs(r.sdist - [0.4, 0.25]).max() <= 1e-12
    assert not flag(r, O.FLAG_SIGN_AMBIG).any()
    assert r.nearest[1] == 0


# ------------------------------------------------------------------------------------------- 90-degree corner
def test_convex_corner_same_sign_tie_with_different_cosines():
    """Body {x < 0, z < 0}, element in the opposite quadrant OFF the bisector: box x in [0.3, 0.5], z in [0.1, 0.2].
    Both faces tie on the shared edge (the y axis) at |r| = sqrt(0.09 + 0.01), r = (0.3, 0, 0.1):
    cos_A = 0.1/|r| = 0.316 (n = +z), cos_B = 0.3/|r| = 0.949 (n = +x).  Same sign: NORMAL, no flag, and the face
    with the larger cosine (B) is the one reported.  On the bisector the cosines are equal and either may be."""
    A, B = H.corner_faces()
    for faces, want in (([A, B], 1), ([B, A], 0)):
        case = H.assemble([H.box_hex([0.3, 0.4, 0.1], [0.5, 0.6, 0.2])], faces)
        r = run(case)
        assert r.labels[0] == NORMAL and abs(r.sdist[0] - np.sqrt(0.1)) <= 1e-12
        assert not flag(r, O.FLAG_SIGN_AMBIG)[0]
        assert r.nearest[0] == want
    case = H.assemble([H.box_hex([0.2, 0.4, 0.2], [0.4, 0.6, 0.4])], [A, B])     # on the bisector
    r = run(case)
    assert r.labels[0] == NORMAL and abs(r.sdist[0] - np.sqrt(0.08)) <= 1e-12


def test_concave_corner_bisector():
    """The same two planes seen from the concave side (orientation reversed: the body is everything EXCEPT the
    quadrant x < 0, z < 0; SURVEY.md section 4 'two flat patches at 90 degrees, element on the bisector').  An element
    on the bisector of the fluid quadrant is equidistant from both walls with perpendicular feet, cos = +1 each:
    NORMAL; off the bisector the nearer wall decides alone."""
    A, B = H.corner_faces()
    flip = lambda F: F.reshape(3, 3, 3).transpose(1, 0, 2).reshape(9, 3).copy()      # noqa: E731  swap s and t
    faces = [flip(A), flip(B)]                          # normals now -z and -x: into the quadrant x < 0, z < 0
    hexes = [H.box_hex([-0.5, 0.4, -0.5], [-0.3, 0.6, -0.3]),      # bisector: 0.3 from both
             H.box_hex([-0.5, 0.4, -0.3], [-0.3, 0.6, -0.1])]      # 0.1 from A (z = 0), 0.3 from B
    r = run(H.assemble(hexes, faces))
    assert list(r.labels) == [NORMAL, NORMAL]
    assert np.abs(r.sdist - [0.3, 0.1]).max() <= 1e-12
    assert not flag(r, O.FLAG_SIGN_AMBIG).any() and r.nearest[1] == 0


# ------------------------------------------------------------------------------------------- ambiguity flag
def ambiguity_case():
    """One flat face z = 0 over [0,1]^2 (normal +z, L_ref = 1, tau = 1e-7) and box elements hovering above it with
    their lower face parallel to it at the gaps below: the distance IS the gap."""
    tau, a = 1e-7, 1e-9
    gaps = [tau - 0.5 * a, tau + 0.5 * a, tau - 5 * a, tau + 5 * a, tau - 1.5 * a, tau + 1.5 * a, tau, 0.0, 0.05]
    hexes = [H.box_hex([0.05 + 0.1 * i, 0.4, g], [0.10 + 0.1 * i, 0.5, g + 0.05]) for i, g in enumerate(gaps)]
    face = H.flat_quad([0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [0.0, 1.0, 0.0])
    want_amb = [True, True, False, False, False, False, True, False, False]
    want_lab = [CUT, NORMAL, CUT, NORMAL, CUT, NORMAL, CUT, CUT, NORMAL]
    return H.assemble(hexes, [face]), np.array(gaps), np.array(want_amb), np.array(want_lab)


def test_ambiguity_flag_is_exactly_the_1e9_band_around_tau():
    case, gaps, want_amb, want_lab = ambiguity_case()
    r = O.classify(case.xyz, case.conn27, case.faces)
    assert r.stats["l_ref"] == 1.0 and r.stats["tau_cut"] == 1e-7
    assert np.array_equal(flag(r, O.FLAG_AMBIGUOUS), want_amb)
    assert r.stats["n_ambiguous"] == int(want_amb.sum())
    exact = gaps != 1e-7                 # (gap == tau sits ON the threshold: either label, and flagged as such)
    assert np.array_equal(r.labels[exact], want_lab[exact])
    notcut = (want_lab != CUT) & exact
    assert np.abs(r.sdist[notcut] - gaps[notcut]).max() <= 1e-15
    assert (r.sdist[(want_lab == CUT) & exact] == 0.0).all()
