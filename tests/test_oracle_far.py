"""Pin of the oracle's FAR branch (SURVEY.md 8(c) "Far elements": relaxed enclosure once d_e > d_band is proved).
-m "not gpu".

P8 (coverage, BASELINE.json north_star: "HOLE u CUT covers every element centroid inside the body") on the elements
where the relaxed enclosure once left the tie list EMPTY: the node-pair upper bound of step 2 was within eps_far of
the true minimum for every face, every PATCHPAIR answered "beyond the cutoff", and step 5 had no r.n to take the sign
from (it fell through to NORMAL for two elements 0.12 and 0.19 deep INSIDE the config-2 body, which the CUDA flood
fill labels HOLE).  The oracle now redoes such an element with the strict enclosure.  "Inside" here comes from the
ANALYTIC dimpled sphere of the generator, not from any distance computation.
"""
import numpy as np

from oracle import dc_oracle as O
from workloads import make_config

HOLE, NORMAL, CUT = 0, 1, 2


def test_far_elements_whose_node_pair_bound_is_sharp_take_a_sign():
    w = make_config(2)
    ids = np.array([778959, 842042, 1000000, 5])
    cen = w.xyz[w.conn27[ids, 13]]
    inside, margin = w.inside(cen), w.surf_margin(cen)
    assert list(inside) == [True, True, False, False] and (margin > 0.1).all()      # far from the surface, no doubt
    d_band = O.auto_d_band(w.xyz, w.conn27, w.faces)
    r = O.classify(w.xyz, w.conn27, w.faces, elem_ids=ids, nproc=1, d_band=d_band)
    assert (r.flags & O.FLAG_FAR).all() and r.stats["n_sign_ambiguous"] == 0
    assert list(r.labels) == [HOLE, HOLE, NORMAL, NORMAL]
    assert np.array_equal(r.sdist, np.where(inside, -d_band, d_band))
    assert (r.nearest >= 0).all()                                                   # a tie member decided each sign
    # the distances are enclosures of the true ones: the centroid margin less about half an element (h = 0.0156) and the dimple depth (0.005)
    assert (np.abs(r.dmin - margin) < 0.03).all()
