"""Pin P4: PATCHPAIR -- the oracle's global minimum distance between two
biquadratic patches with a rigorous enclosure -- against closed forms that ARE exactly
representable by biquadratic patches, and against dense sampling on small random inputs.
-m "not gpu".
"""
import numpy as np
import pytest

from oracle import dc_oracle as O

RNG = np.random.default_rng(4)
REF = [-1.0, 0.0, 1.0]


def patch_from(fn):
    """9 Lagrange nodes (m = i + 3j) of the map (u,v) -> fn(u,v)."""
    return np.array([fn(REF[i], REF[j]) for j in range(3) for i in range(3)], float)


def lag(t):
    return np.array([t * (t - 1) / 2, 1 - t * t, t * (t + 1) / 2])


def sample_patch(X, n):
    t = np.linspace(-1, 1, n)
    L = np.stack([lag(x) for x in t])            # [n,3]
    G = X.reshape(3, 3, 3)                        # [j,i,c]
    return np.einsum('ui,vj,jic->uvc', L, L, G).reshape(-1, 3)


def brute(PX, QX, n):
    A, B = sample_patch(PX, n), sample_patch(QX, n)
    best = np.inf
    for s in range(0, A.shape[0], 512):
        d = np.sqrt(((A[s:s + 512, None, :] - B[None, :, :]) ** 2).sum(2)).min()
        best = min(best, d)
    return best


def test_parallel_flat_squares():
    P = patch_from(lambda u, v: (u, v, 0.0))
    for g in (0.25, 1e-3, 3.0):
        Q = patch_from(lambda u, v: (0.5 * u + 0.2, 0.7 * v - 0.1, g))
        r = O.patch_pair(P, Q, eps=1e-13)
        assert r.status == 0 and abs(r.hi - g) < 1e-13


def test_flat_vs_paraboloid_interior_interior():
    a, c = 0.8, 0.37
    Q = patch_from(lambda u, v: (u, v, a * (u * u + v * v)))      # exact in the biquadratic space
    P = patch_from(lambda u, v: (0.9 * u + 0.05, 0.8 * v - 0.03, -c))
    r = O.patch_pair(P, Q, eps=1e-12)
    assert r.status == 0 and r.depth_exceeded == 0
    assert r.hi >= c - 1e-15 and r.hi - c <= 1e-12
    # closest point is the paraboloid's apex, below it on the plane
    assert abs(r.params[2]) < 1e-5 and abs(r.params[3]) < 1e-5


def test_point_above_paraboloid_ring_of_minimisers():
    # z0 > 1/(2a): the nearest points form a ring, distance sqrt(z0/a - 1/(4 a^2))
    a, z0 = 1.0, 0.9
    Q = patch_from(lambda u, v: (u, v, a * (u * u + v * v)))
    P = patch_from(lambda u, v: (1e-9 * u, 1e-9 * v, z0))
    want = np.sqrt(z0 / a - 1 / (4 * a * a))
    r = O.patch_pair(P, Q, eps=1e-7)
    assert r.status == 0 and r.depth_exceeded == 0
    assert abs(r.hi - want) < 2e-7 + 2e-9
    rho = np.hypot(r.params[2], r.params[3])
    assert abs(rho - np.sqrt(z0 / a - 1 / (2 * a * a))) < 1e-3


def test_point_inside_concave_bowl():
    # point on the axis BELOW the focal distance: unique nearest point = apex, distance z0
    a, z0 = 1.0, 0.3
    Q = patch_from(lambda u, v: (u, v, a * (u * u + v * v)))
    P = patch_from(lambda u, v: (1e-9 * u, 1e-9 * v, z0))
    r = O.patch_pair(P, Q, eps=1e-12)
    assert r.status == 0 and abs(r.hi - z0) < 1e-9


def test_skew_straight_edges():
    # nearest features are two skew straight edges: textbook segment-segment distance
    P = patch_from(lambda u, v: (u, 0.0, -1.0 + v))          # square in the plane y=0, top edge z=0
    Q = patch_from(lambda u, v: (0.3, 0.4 + (v + 1) * 0.5, 0.25 + (u + 1)))   # plane x=0.3, bottom edge z=0.25
    # top edge of P: {(x,0,0)}, nearest edge of Q: {(0.3, y>=0.4, z>=0.25)} corner (0.3,0.4,0.25)
    want = np.hypot(0.4, 0.25)
    r = O.patch_pair(P, Q, eps=1e-13)
    assert r.status == 0 and abs(r.hi - want) < 1e-13


def test_transversal_intersection_collapses():
    P = patch_from(lambda u, v: (u, v, 0.1 * u * v))
    Q = patch_from(lambda u, v: (0.2 + 0.1 * v * v, u, v))
    r = O.patch_pair(P, Q, eps=1e-12, tau_exit=1e-7 - 1e-9)
    assert r.status == 2 and r.hi <= 1e-7
    r = O.patch_pair(P, Q, eps=1e-12)
    assert r.status == 0 and r.hi < 1e-11


def test_cutoff_prunes_and_keeps():
    P = patch_from(lambda u, v: (u, v, 0.0))
    Q = patch_from(lambda u, v: (u, v, 0.5 + 0.1 * u * u))
    assert O.patch_pair(P, Q, cutoff=0.4).status == 1
    r = O.patch_pair(P, Q, cutoff=0.6)
    assert r.status == 0 and abs(r.hi - 0.5) < 1e-12


def test_sign_vector_and_normal():
    # r = P - Q points from the face to the element; n = Q_s x Q_t
    Q = patch_from(lambda u, v: (u, v, 0.0))                 # normal +z
    Pabove = patch_from(lambda u, v: (0.1 * u, 0.1 * v, 0.3))
    Pbelow = patch_from(lambda u, v: (0.1 * u, 0.1 * v, -0.2))
    r = O.patch_pair(Pabove, Q)
    assert np.allclose(r.n / np.linalg.norm(r.n), [0, 0, 1]) and r.r @ r.n > 0
    r = O.patch_pair(Pbelow, Q)
    assert r.r @ r.n < 0 and abs(r.hi - 0.2) < 1e-13


@pytest.mark.parametrize("seed", range(6))
def test_random_curved_patches_vs_dense_sampling(seed):
    rng = np.random.default_rng(100 + seed)
    def rnd(shift):
        c = rng.normal(size=(6, 3)) * 0.25
        return patch_from(lambda u, v: np.array([u, v, 0.0]) * [1, 1, 0] + shift
                          + c[0] * u * u + c[1] * v * v + c[2] * u * v + c[3] * u * u * v
                          + c[4] * u * v * v + c[5] * u * u * v * v)
    P = rnd(np.zeros(3)); Q = rnd(np.array([0.3 * seed % 2, 0.2, 0.6 + 0.15 * seed]))
    r = O.patch_pair(P, Q, eps=1e-11)
    assert r.depth_exceeded == 0
    n = 49
    ds = brute(P, Q, n)
    # sample spacing: patch extent ~ 2 (+ curvature) over n-1 intervals, both patches
    spacing = 2 * np.sqrt(2) * 1.6 / (n - 1)
    assert r.hi <= ds + 1e-12
    assert ds - r.hi <= spacing
    # the reported parameters attain hi on the TRUE patches (independent numpy evaluation)
    u, v, s, t = r.params
    p = np.einsum('i,j,jic->c', lag(u), lag(v), P.reshape(3, 3, 3))
    q = np.einsum('i,j,jic->c', lag(s), lag(t), Q.reshape(3, 3, 3))
    assert abs(np.linalg.norm(p - q) - r.hi) < 1e-13
    # first-order optimality at the reported pair: refine with a local polish and compare
    from scipy.optimize import minimize
    f = lambda x: np.linalg.norm(np.einsum('i,j,jic->c', lag(x[0]), lag(x[1]), P.reshape(3, 3, 3))
                                 - np.einsum('i,j,jic->c', lag(x[2]), lag(x[3]), Q.reshape(3, 3, 3)))
    best = min(minimize(f, x0, bounds=[(-1, 1)] * 4, method="L-BFGS-B", options=dict(ftol=1e-15, gtol=1e-12)).fun
               for x0 in ([u, v, s, t], [0, 0, 0, 0]))
    assert r.hi <= best + 1e-9     # nothing a local optimiser finds beats the enclosure
