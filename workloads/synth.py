"""Synthetic stand-ins for the paper's overset workloads (BASELINE.json configs).

The paper's meshes (golf ball L415-L422, TSTO L298, NACA L296, Taylor-Green L337 of
PAPER.md) are not available; these seeded recipes keep their structure: a closed,
outward-oriented wall surface of 9-node quadratic quadrilateral faces cutting a background
of 27-node quadratic hexahedra.

Conventions (DESIGN.md "Readings" A1/A2):
* hex node m = i + 3 j + 9 k   (xi fastest), reference nodes at {-1, 0, +1};
* quad node m = i + 3 j;
* element faces k = 0..5 <-> xi=-1, xi=+1, eta=-1, eta=+1, zeta=-1, zeta=+1;
* `adj6[e][k]` = neighbour across face k, or -1;
* face normal  x_s cross x_t  points OUT of the body.

Nothing in here computes a distance, a box, a Bezier net or a label.
"""
from __future__ import annotations

import dataclasses
from typing import Callable, Optional

import numpy as np

BASE_SEED = 171107663


# --------------------------------------------------------------------------------------
# background grid
# --------------------------------------------------------------------------------------
def background_grid(N: int, curved: bool, seed: int, amp: float = 0.04,
                    lo: float = -1.0, hi: float = 1.0, with_adj: bool = True):
    """N^3 27-node hexes tiling [lo,hi]^3 on a (2N+1)^3 lattice of shared nodes.

    Curved variant (BASELINE.json config 1): x' = x + amp sin(pi y + a) sin(pi z + b),
    y' = y + amp sin(pi z + b) sin(pi x + c), z' = z + amp sin(pi x + c) sin(pi y + a),
    sines evaluated at the unperturbed lattice point, (a,b,c) ~ U[0,2pi) from the seed.
    The element geometry IS the triquadratic interpolant of the moved nodes.

    Returns xyz [n_nodes,3] f64, conn27 [N^3,27] i32, adj6 [N^3,6] i32 (or None), phases (3,).
    """
    M = 2 * N + 1
    t = lo + (hi - lo) * (np.arange(M, dtype=np.float64) / (2 * N))
    # node id = I + M*(J + M*K)
    X = np.broadcast_to(t[None, None, :], (M, M, M))
    Y = np.broadcast_to(t[None, :, None], (M, M, M))
    Z = np.broadcast_to(t[:, None, None], (M, M, M))
    rng = np.random.default_rng(seed)
    phases = rng.uniform(0.0, 2.0 * np.pi, size=3)
    xyz = np.empty((M * M * M, 3), dtype=np.float64)
    if curved:
        a, b, c = phases
        sx = np.sin(np.pi * t + c)  # sin(pi x + c)
        sy = np.sin(np.pi * t + a)  # sin(pi y + a)
        sz = np.sin(np.pi * t + b)  # sin(pi z + b)
        SX = sx[None, None, :]
        SY = sy[None, :, None]
        SZ = sz[:, None, None]
        xyz[:, 0] = (X + amp * SY * SZ).reshape(-1)
        xyz[:, 1] = (Y + amp * SZ * SX).reshape(-1)
        xyz[:, 2] = (Z + amp * SX * SY).reshape(-1)
    else:
        xyz[:, 0] = X.reshape(-1)
        xyz[:, 1] = Y.reshape(-1)
        xyz[:, 2] = Z.reshape(-1)

    # connectivity: element (a,b,c), id = a + N (b + N c); node (i,j,k) -> lattice (2a+i, 2b+j, 2c+k)
    ea = np.arange(N, dtype=np.int64)
    A = np.broadcast_to(ea[None, None, :], (N, N, N)).reshape(-1)
    B = np.broadcast_to(ea[None, :, None], (N, N, N)).reshape(-1)
    C = np.broadcast_to(ea[:, None, None], (N, N, N)).reshape(-1)
    conn = np.empty((N * N * N, 27), dtype=np.int32)
    for k in range(3):
        for j in range(3):
            for i in range(3):
                conn[:, i + 3 * j + 9 * k] = ((2 * A + i) + M * ((2 * B + j) + M * (2 * C + k))).astype(np.int32)
    adj = None
    if with_adj:
        adj = np.full((N * N * N, 6), -1, dtype=np.int32)
        eid = (A + N * (B + N * C))
        adj[:, 0] = np.where(A > 0, eid - 1, -1)
        adj[:, 1] = np.where(A < N - 1, eid + 1, -1)
        adj[:, 2] = np.where(B > 0, eid - N, -1)
        adj[:, 3] = np.where(B < N - 1, eid + N, -1)
        adj[:, 4] = np.where(C > 0, eid - N * N, -1)
        adj[:, 5] = np.where(C < N - 1, eid + N * N, -1)
    return xyz, conn, adj, phases


# --------------------------------------------------------------------------------------
# cubed-sphere wall faces
# --------------------------------------------------------------------------------------
def cubed_sphere_dirs(n: int) -> np.ndarray:
    """Unit directions of the 9 nodes of each of the 6 n^2 faces: [6 n^2, 9, 3].

    Uniform-cube ("gnomonic") subdivision: cube point c = s e_a + y e_b + z e_c with
    y = -1 + (2p+i)/n, z = -1 + (2q+j)/n; direction d = c/|c|.  Node order (i + 3 j) is
    swapped on three of the six sides so that (x_s cross x_t) . d > 0 (outward).
    """
    out = np.empty((6, n, n, 3, 3, 3), dtype=np.float64)  # side, p, q, j, i, xyz
    g = -1.0 + np.arange(2 * n + 1, dtype=np.float64) / n
    side = 0
    for a in range(3):
        b, c = (a + 1) % 3, (a + 2) % 3
        for s in (+1.0, -1.0):
            for p in range(n):
                for q in range(n):
                    for j in range(3):
                        for i in range(3):
                            v = np.zeros(3)
                            v[a] = s
                            if s > 0:   # (e_b x e_c) = +e_a : natural order is outward
                                v[b] = g[2 * p + i]
                                v[c] = g[2 * q + j]
                            else:       # swap roles of i and j to flip the normal
                                v[b] = g[2 * p + j]
                                v[c] = g[2 * q + i]
                            out[side, p, q, j, i] = v / np.linalg.norm(v)
            side += 1
    return out.reshape(6 * n * n, 9, 3)


def cubed_sphere_faces(n: int, radius: float | Callable[[np.ndarray], np.ndarray] = 0.5) -> np.ndarray:
    """Faces [6 n^2, 9, 3]: node = rho(d) d with rho constant or a callable on unit directions."""
    D = cubed_sphere_dirs(n)
    if callable(radius):
        rho = radius(D.reshape(-1, 3)).reshape(D.shape[0], 9, 1)
    else:
        rho = float(radius)
    return np.ascontiguousarray(D * rho)


def random_rotation(rng: np.random.Generator) -> np.ndarray:
    """Uniform random rotation matrix (QR of a Gaussian matrix, sign-fixed, det=+1)."""
    Mx = rng.normal(size=(3, 3))
    Q, Rm = np.linalg.qr(Mx)
    Q = Q * np.sign(np.diag(Rm))[None, :]
    if np.linalg.det(Q) < 0:
        Q[:, 2] = -Q[:, 2]
    return Q


def dimple_centres(n_dimples: int, rot: np.ndarray) -> np.ndarray:
    """Fibonacci lattice z_k = 1-(2k+1)/n, phi_k = k pi (3 - sqrt 5), rotated by `rot`."""
    k = np.arange(n_dimples, dtype=np.float64)
    z = 1.0 - (2.0 * k + 1.0) / n_dimples
    ph = np.pi * (3.0 - np.sqrt(5.0)) * k
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    C = np.stack([s * np.cos(ph), s * np.sin(ph), z], axis=1)
    return C @ rot.T


def dimpled_radius(centres: np.ndarray, R: float = 0.5, depth_rel: float = 0.01,
                   sigma: float = 0.03) -> Callable[[np.ndarray], np.ndarray]:
    """r(d) = R - sum_k depth_rel R exp(-theta_k^2 / (2 sigma^2)), theta_k = angle(d, c_k)."""
    def rho(D: np.ndarray) -> np.ndarray:
        D = np.asarray(D, dtype=np.float64).reshape(-1, 3)
        out = np.empty(D.shape[0])
        chunk = 16384
        for s in range(0, D.shape[0], chunk):
            c = np.clip(D[s:s + chunk] @ centres.T, -1.0, 1.0)
            th = np.arccos(c)
            out[s:s + chunk] = R - (depth_rel * R) * np.exp(-th * th / (2.0 * sigma * sigma)).sum(axis=1)
        return out
    return rho


def spin_axis(seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    v = rng.normal(size=3)
    return v / np.linalg.norm(v)


def rotation_about_axis(axis: np.ndarray, angle_rad: float) -> np.ndarray:
    """Rodrigues rotation matrix."""
    x, y, z = axis
    K = np.array([[0, -z, y], [z, 0, -x], [-y, x, 0]], dtype=np.float64)
    return np.eye(3) + np.sin(angle_rad) * K + (1.0 - np.cos(angle_rad)) * (K @ K)


def ellipsoid_bodies(n_bodies: int, seed: int, amin: float = 0.08, amax: float = 0.2,
                     cmax: float = 0.7, gap: float = 0.05):
    """Sequential rejection: semi-axes U[amin,amax]^3, uniform rotation, centre U[-cmax,cmax]^3,
    rejected if closer to an earlier centre than max(axes_i)+max(axes_j)+gap."""
    rng = np.random.default_rng(seed)
    bodies = []
    while len(bodies) < n_bodies:
        ax = rng.uniform(amin, amax, size=3)
        rot = random_rotation(rng)
        ctr = rng.uniform(-cmax, cmax, size=3)
        ok = True
        for (ax2, _, ctr2) in bodies:
            if np.linalg.norm(ctr - ctr2) < ax.max() + ax2.max() + gap:
                ok = False
                break
        if ok:
            bodies.append((ax, rot, ctr))
    return bodies


# --------------------------------------------------------------------------------------
# configs
# --------------------------------------------------------------------------------------
@dataclasses.dataclass
class Workload:
    name: str
    config: int
    N: int
    xyz: np.ndarray          # [n_nodes,3] f64
    conn27: np.ndarray       # [n_elem,27] i32
    adj6: Optional[np.ndarray]   # [n_elem,6] i32
    faces: np.ndarray        # [n_face,9,3] f64
    inside: Callable[[np.ndarray], np.ndarray]       # analytic: points -> bool (strictly inside the body)
    surf_margin: Callable[[np.ndarray], np.ndarray]  # analytic: points -> |distance-like margin| to analytic surface
    meta: dict

    @property
    def n_elem(self) -> int:
        return int(self.conn27.shape[0])

    @property
    def n_face(self) -> int:
        return int(self.faces.shape[0])

    def spin_faces(self, step: int) -> np.ndarray:
        """Config 3: the surface nodes rotated about the seeded axis by `step` degrees
        (always from the unrotated nodes, no accumulation)."""
        axis = self.meta["spin_axis"]
        Rm = rotation_about_axis(axis, np.deg2rad(float(step)))
        return np.ascontiguousarray(self.faces @ Rm.T)


def _sphere_inside(R):
    def inside(P):
        return np.linalg.norm(P, axis=-1) < R

    def margin(P):
        return np.abs(np.linalg.norm(P, axis=-1) - R)
    return inside, margin


def make_config(config: int, *, N: Optional[int] = None, n: Optional[int] = None,
                seed: Optional[int] = None, with_adj: bool = True) -> Workload:
    """Build BASELINE.json config 0..4.  `N` (elements per edge) and `n` (faces per cube edge)
    may be overridden to get reduced-size instances with the same structure (for tests)."""
    if seed is None:
        seed = BASE_SEED + config
    R = 0.5
    if config == 0:
        N = 16 if N is None else N
        n = 4 if n is None else n
        xyz, conn, adj, ph = background_grid(N, curved=False, seed=seed, with_adj=with_adj)
        faces = cubed_sphere_faces(n, R)
        ins, mar = _sphere_inside(R)
        return Workload("sphere96_straight16", 0, N, xyz, conn, adj, faces, ins, mar,
                        dict(R=R, n=n, seed=seed, phases=ph))
    if config == 1:
        N = 64 if N is None else N
        n = 16 if n is None else n
        xyz, conn, adj, ph = background_grid(N, curved=True, seed=seed, with_adj=with_adj)
        faces = cubed_sphere_faces(n, R)
        ins, mar = _sphere_inside(R)
        return Workload("sphere1536_curved64", 1, N, xyz, conn, adj, faces, ins, mar,
                        dict(R=R, n=n, seed=seed, phases=ph))
    if config in (2, 3):
        N = 128 if N is None else N
        n = 64 if n is None else n
        # config 3 is config 2's geometry (same seed) plus the spin axis
        gseed = BASE_SEED + 2 if seed == BASE_SEED + config else seed
        xyz, conn, adj, ph = background_grid(N, curved=True, seed=gseed, with_adj=with_adj)
        rng = np.random.default_rng(gseed + 1000)
        rot = random_rotation(rng)
        cen = dimple_centres(336, rot)
        rho = dimpled_radius(cen, R=R, depth_rel=0.01, sigma=0.03)
        faces = cubed_sphere_faces(n, rho)

        def inside(P):
            P = np.asarray(P, dtype=np.float64).reshape(-1, 3)
            r = np.linalg.norm(P, axis=1)
            D = P / np.maximum(r, 1e-300)[:, None]
            return r < rho(D)

        def margin(P):
            P = np.asarray(P, dtype=np.float64).reshape(-1, 3)
            r = np.linalg.norm(P, axis=1)
            D = P / np.maximum(r, 1e-300)[:, None]
            return np.abs(r - rho(D))
        return Workload("dimpled24576_curved128" if config == 2 else "spin32_dimpled24576_curved128",
                        config, N, xyz, conn, adj, faces, inside, margin,
                        dict(R=R, n=n, seed=gseed, phases=ph, dimple_centres=cen,
                             spin_axis=spin_axis(BASE_SEED + 3 + 2000), spin_steps=32))
    if config == 4:
        N = 192 if N is None else N
        n = 32 if n is None else n
        xyz, conn, adj, ph = background_grid(N, curved=True, seed=seed, with_adj=with_adj)
        bodies = ellipsoid_bodies(8, seed + 1000)
        unit = cubed_sphere_dirs(n)
        parts = []
        for (ax, rot, ctr) in bodies:
            parts.append((unit * ax[None, None, :]) @ rot.T + ctr[None, None, :])
        faces = np.ascontiguousarray(np.concatenate(parts, axis=0))

        def _q(P):
            P = np.asarray(P, dtype=np.float64).reshape(-1, 3)
            qs = []
            for (ax, rot, ctr) in bodies:
                L = (P - ctr[None, :]) @ rot / ax[None, :]
                qs.append(np.sqrt((L * L).sum(axis=1)))
            return np.stack(qs, axis=1)  # [npts, nbodies], <1 inside

        def inside(P):
            return (_q(P) < 1.0).any(axis=1)

        def margin(P):
            q = _q(P)
            amin = min(b[0].min() for b in bodies)
            return np.abs(q - 1.0).min(axis=1) * amin
        return Workload("ellipsoids8x6144_curved192", 4, N, xyz, conn, adj, faces, inside, margin,
                        dict(n=n, seed=seed, phases=ph, bodies=bodies))
    raise ValueError("config must be 0..4")


# --------------------------------------------------------------------------------------
# structural checks on what the generator emits (no method arithmetic)
# --------------------------------------------------------------------------------------
def check_watertight(faces: np.ndarray) -> bool:
    """Every patch edge's 3 nodes occur bit-identically (in either direction) in exactly two faces."""
    F = faces.reshape(-1, 3, 3, 3)  # [f, j, i, xyz]
    edges = [F[:, 0, :, :], F[:, 2, :, :], F[:, :, 0, :], F[:, :, 2, :]]
    keys = {}
    for E in edges:
        for f in range(E.shape[0]):
            a = E[f].tobytes()
            b = E[f][::-1].copy().tobytes()
            k = min(a, b)
            keys[k] = keys.get(k, 0) + 1
    return all(v == 2 for v in keys.values())


def check_conforming(conn27: np.ndarray, adj6: np.ndarray) -> bool:
    """adj6 is symmetric and neighbours share the 9 face nodes (as a set)."""
    face_nodes = []
    idx = np.arange(27).reshape(3, 3, 3)  # [k, j, i]
    face_nodes.append(idx[:, :, 0].reshape(-1))
    face_nodes.append(idx[:, :, 2].reshape(-1))
    face_nodes.append(idx[:, 0, :].reshape(-1))
    face_nodes.append(idx[:, 2, :].reshape(-1))
    face_nodes.append(idx[0, :, :].reshape(-1))
    face_nodes.append(idx[2, :, :].reshape(-1))
    opp = [1, 0, 3, 2, 5, 4]
    ok = True
    for k in range(6):
        nb = adj6[:, k]
        m = nb >= 0
        e = np.nonzero(m)[0]
        ok &= bool(np.all(adj6[nb[m], opp[k]] == e))
        a = np.sort(conn27[e][:, face_nodes[k]], axis=1)
        b = np.sort(conn27[nb[m]][:, face_nodes[opp[k]]], axis=1)
        ok &= bool(np.array_equal(a, b))
    return ok
