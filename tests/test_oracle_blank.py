"""-m "not gpu": pins of oracle/blank_oracle.py (union of holes, Algorithm 3.1 steps 6-7, AB faces) against
what the paper fixes: its sentences as a hand-written truth table (tests/golden/unblank_truth_table.txt),
set invariants that follow from them, and a closed-form moving-sphere scenario."""
import os

import numpy as np

from oracle import blank_oracle as BO
from workloads import make_config

HERE = os.path.dirname(os.path.abspath(__file__))
HOLE, NORMAL, CUT = 0, 1, 2


def truth_rows():
    rows = []
    for line in open(os.path.join(HERE, "golden", "unblank_truth_table.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        lhs, rhs = line.split("->")
        mode, prev, ht, hp = lhs.split()
        blank, unb = rhs.split()
        rows.append((mode, int(prev), int(ht), int(hp), int(blank), int(unb)))
    assert len(rows) == 16
    return rows


def test_unblank_truth_table():
    lab = {0: NORMAL, 1: HOLE}
    for mode, prev, ht, hp, blank, unb in truth_rows():
        m = BO.MODE_WALL if mode == "wall" else BO.MODE_OVERSET
        ib, u, th = BO.unblank(m, False, np.array([prev], np.int8), np.array([lab[ht]], np.int8), np.array([lab[hp]], np.int8))
        assert ib[0] == blank and (len(u) == 1) == bool(unb), (mode, prev, ht, hp)
        assert (len(th) == 1) == bool(blank and not prev)


def test_cut_counts_as_hole_only_when_asked():
    prev = np.zeros(3, np.int8)
    lt = np.array([CUT, HOLE, NORMAL], np.int8)
    ib, _, _ = BO.unblank(BO.MODE_WALL, False, prev, lt, lt)
    assert ib.tolist() == [0, 1, 0]
    ib, _, _ = BO.unblank(BO.MODE_WALL, True, prev, lt, lt)
    assert ib.tolist() == [1, 1, 0]


def test_unblank_invariants_random():
    rng = np.random.default_rng(3)
    n = 5000
    prev = rng.integers(0, 2, n).astype(np.int8)
    lt = rng.integers(0, 3, n).astype(np.int8); lp = rng.integers(0, 3, n).astype(np.int8)
    for mode in (BO.MODE_WALL, BO.MODE_OVERSET):
        for cih in (False, True):
            ib, u, th = BO.unblank(mode, cih, prev, lt, lp)
            ht, hp = BO.is_hole_cell(lt, cih), BO.is_hole_cell(lp, cih)
            assert not ib[u].any() and prev[u].all()               # unblanked cells were holes and are field now
            assert ib[th].all() and not prev[th].any()             # to-hole cells are new holes
            # every previously blanked cell is either still blanked or on the unblank list, never silently field
            assert np.array_equal(np.sort(np.concatenate([u, np.nonzero(prev & ib)[0]])), np.nonzero(prev)[0])
            if mode == BO.MODE_WALL:
                assert (ib[ht | hp] == 1).all()                    # no field cell inside the wall at t or t + dt
            else:
                assert (ib[~(ht & hp)] == 0).all()                 # nothing blanked that either position still needs
    # static grids: nothing to unblank, nothing new to blank once the blanking has settled
    ib0, _, _ = BO.unblank(BO.MODE_WALL, False, np.zeros(n, np.int8), lt, lt)
    ib1, u, th = BO.unblank(BO.MODE_WALL, False, ib0, lt, lt)
    assert np.array_equal(ib0, ib1) and len(u) == 0 and len(th) == 0


def test_union_labels():
    rng = np.random.default_rng(4)
    a = rng.integers(0, 3, 1000).astype(np.int8); b = rng.integers(0, 3, 1000).astype(np.int8)
    u = BO.union_labels(a, b)
    assert np.array_equal(u, BO.union_labels(b, a)) and np.array_equal(BO.union_labels(a, a), a)
    assert np.array_equal(u == HOLE, (a == HOLE) | (b == HOLE))                    # L217: union of the hole cells
    assert np.array_equal(u == NORMAL, (a == NORMAL) & (b == NORMAL))
    assert np.array_equal(BO.union_labels(a, np.full(1000, NORMAL, np.int8)), a)   # NORMAL is the neutral element


def test_ab_faces_chain_and_brute_force():
    # a 1-D chain of 5 cells along xi, cells 1 and 2 blanked: AB faces are (0, xi+) and (3, xi-)
    adj = -np.ones((5, 6), np.int64)
    for e in range(5):
        adj[e, 0] = e - 1 if e > 0 else -1
        adj[e, 1] = e + 1 if e < 4 else -1
    m = BO.ab_faces(np.array([0, 1, 1, 0, 0], np.int8), adj)
    assert m.tolist() == [0b10, 0, 0, 0b01, 0]
    # a 3-D grid: count the AB faces from the hole side instead (a different enumeration of the same set)
    w = make_config(0, N=6, n=2)
    rng = np.random.default_rng(5)
    ib = (rng.random(w.n_elem) < 0.3).astype(np.int8)
    m = BO.ab_faces(ib, w.adj6)
    from_hole_side = 0
    for e in np.nonzero(ib)[0]:
        for k in range(6):
            nb = w.adj6[e, k]
            if nb >= 0 and not ib[nb]:
                from_hole_side += 1
    assert int(sum(bin(int(x)).count("1") for x in m)) == from_hole_side
    assert (m[ib != 0] == 0).all()


def test_moving_sphere_scenario_closed_form():
    """A sphere of radius R moving by less than one cell per step through straight hexes (the closed-form
    box-vs-sphere labels of config 0): with wall-mode blanking no field cell is ever inside the body at t or t + dt,
    and every cell the body has left appears exactly once on an unblank list."""
    w = make_config(0, N=10, n=2)
    X = w.xyz[w.conn27]                                   # [n_elem, 27, 3]
    lo, hi = X.min(1), X.max(1)
    R, h = 0.35, 2.0 / 10

    def labels_at(cx):
        c = np.array([cx, 0.0, 0.0])
        near = np.linalg.norm(np.clip(c, lo, hi) - c, axis=1)
        far = np.linalg.norm(np.maximum(np.abs(lo - c), np.abs(hi - c)), axis=1)
        lab = np.full(w.n_elem, CUT, np.int8)
        lab[far < R] = HOLE
        lab[near > R] = NORMAL
        return lab

    xs = -0.3 + 0.5 * h * np.arange(8)
    ib = BO.is_hole_cell(labels_at(xs[0]), True).astype(np.int8)
    ever_unblanked = np.zeros(w.n_elem, int)
    for s in range(len(xs) - 1):
        lt, lp = labels_at(xs[s]), labels_at(xs[s + 1])
        ib_new, u, th = BO.unblank(BO.MODE_WALL, True, ib, lt, lp)
        inside_now = BO.is_hole_cell(lt, True) | BO.is_hole_cell(lp, True)
        assert (ib_new[inside_now] == 1).all()
        ever_unblanked[u] += 1
        ib = ib_new
    left_behind = BO.is_hole_cell(labels_at(xs[0]), True) & ~(ib != 0)
    assert left_behind.sum() > 0 and (ever_unblanked[left_behind] == 1).all()
    assert (ever_unblanked[~left_behind] == 0).all()
