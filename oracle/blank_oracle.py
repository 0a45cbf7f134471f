"""blank_oracle.py -- TEST INFRASTRUCTURE ONLY (imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg; the product path never imports it).

Plain numpy statement of the blanking logic that consumes direct cuts:

  * union of the hole cells of several cutting boundaries
  * Algorithm 3.1, steps 6 and 7 (the unblank procedure)
  * artificial-boundary (AB) faces

Conventions shared with include/dc.h: labels HOLE = 0, NORMAL = 1, CUT = 2; a blanking vector `iblank` is
int8 with 1 = blanked ("hole cell") and 0 = field.  `cut_is_hole` says whether an element the surface passes
through counts as a hole cell (the paper leaves that to the caller: DESIGN.md reading A9).

Everything is written element by element in the paper's words; no vector tricks beyond boolean masks.
"""
from __future__ import annotations

import numpy as np

HOLE, NORMAL, CUT = 0, 1, 2
MODE_WALL, MODE_OVERSET = 0, 1


def union_labels(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    """L217: "a separate function then takes the union of the hole cells created from each of the cutting
    boundaries".  Per element: HOLE if either cut says HOLE, else CUT if either says CUT, else NORMAL."""
    a = np.asarray(a, np.int8); b = np.asarray(b, np.int8)
    out = np.full(a.shape, NORMAL, np.int8)
    out[(a == CUT) | (b == CUT)] = CUT
    out[(a == HOLE) | (b == HOLE)] = HOLE
    return out


def is_hole_cell(labels: np.ndarray, cut_is_hole: bool) -> np.ndarray:
    labels = np.asarray(labels, np.int8)
    return (labels == HOLE) | ((labels == CUT) if cut_is_hole else np.zeros(labels.shape, bool))


def unblank(mode: int, cut_is_hole: bool, iblank_prev, labels_t, labels_tplus):
    """Algorithm 3.1 (L114-L133), steps 6 and 7, for one grid.

    I_{t-} = iblank_prev (step 1), I_t / I_{t+} = the hole cells of the cuts at t and t + dt (steps 3, 5).

    Step 6 (body grids cut by solid walls):
      6.1 "Any cell which becomes a hole cell in I_{t+} can be set to hole in I_t"     -> blank = I_t or I_{t+}
      6.2 "Any hole cell in I_{t-} which is no longer a hole cell in I_t and I_{t+} must be unblanked"
    Step 7 (background grids cut by overset boundaries):
      7.1 "Any hole cell in I_{t-} which is no longer a hole cell in I_t or I_{t+} must be unblanked";
      a cell stays blanked only while both cuts call it a hole ("we must not blank potential hole cells
      until we have ascertained we no longer need them", L112)                          -> blank = I_t and I_{t+}
    Returns (iblank_new int8, must_unblank ids, to_hole ids), ids ascending; to_hole = newly blanked cells.
    """
    prev = np.asarray(iblank_prev, np.int8) != 0
    ht = is_hole_cell(labels_t, cut_is_hole)
    hp = is_hole_cell(labels_tplus, cut_is_hole)
    n = prev.shape[0]
    blank = np.zeros(n, bool)
    unb = np.zeros(n, bool)
    for e in range(n):
        if mode == MODE_WALL:
            blank[e] = ht[e] or hp[e]
            unb[e] = prev[e] and (not ht[e]) and (not hp[e])
        else:
            blank[e] = ht[e] and hp[e]
            unb[e] = prev[e] and ((not ht[e]) or (not hp[e]))
    to_hole = blank & ~prev
    return blank.astype(np.int8), np.nonzero(unb)[0].astype(np.int32), np.nonzero(to_hole)[0].astype(np.int32)


def ab_faces(iblank, adj6) -> np.ndarray:
    """L217: "The artificial boundary faces are then determined to be any face which has a hole cell on one
    side and a normal/field cell on the other."  Returns a uint8 mask per element, bit k set iff the element is
    a field cell and its neighbour across face k is a hole cell (each AB face is reported on its field side)."""
    ib = np.asarray(iblank, np.int8) != 0
    adj6 = np.asarray(adj6)
    n = ib.shape[0]
    out = np.zeros(n, np.uint8)
    for e in range(n):
        if ib[e]:
            continue
        m = 0
        for k in range(6):
            nb = adj6[e, k]
            if nb >= 0 and ib[nb]:
                m |= 1 << k
        out[e] = m
    return out
