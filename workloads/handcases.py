"""Hand-built inputs for the tie rule, the ambiguity flag and the closest-point closed forms
(section 4.1 Fig. 6, section 4.4 Fig. 14).

Input construction only: flat / paraboloid patches as 9 Lagrange nodes, box-shaped (or degenerate)
27-node hexes, and stand-alone elements assembled into a "grid" without shared nodes.  Nothing in here
computes a distance, a box test, a Bezier net or a label; the expected values live in the tests.
Served to both the oracle tests (-m "not gpu") and the CUDA parity tests (-m gpu).
"""
from __future__ import annotations

import dataclasses
from typing import Callable, Sequence

import numpy as np

REF = (-1.0, 0.0, 1.0)


def quad_from(fn: Callable[[float, float], Sequence[float]]) -> np.ndarray:
    """9 Lagrange nodes (m = i + 3 j) of the map (s,t) -> fn(s,t), (s,t) in {-1,0,1}^2.  A map that is
    (bi)quadratic in (s,t) is reproduced exactly.  Normal = x_s cross x_t."""
    return np.array([fn(REF[i], REF[j]) for j in range(3) for i in range(3)], dtype=np.float64)


def flat_quad(p0, eu, ev) -> np.ndarray:
    """Parallelogram p0 + a eu + b ev, (a,b) in [0,1]^2; normal eu x ev."""
    p0, eu, ev = (np.asarray(x, dtype=np.float64) for x in (p0, eu, ev))
    return quad_from(lambda s, t: p0 + 0.5 * (s + 1.0) * eu + 0.5 * (t + 1.0) * ev)


def hex_from(fn: Callable[[float, float, float], Sequence[float]]) -> np.ndarray:
    """27 Lagrange nodes (m = i + 3 j + 9 k) of (xi,eta,zeta) -> fn(xi,eta,zeta)."""
    return np.array([fn(REF[i], REF[j], REF[k]) for k in range(3) for j in range(3) for i in range(3)],
                    dtype=np.float64)


def box_hex(lo, hi) -> np.ndarray:
    """Axis-aligned straight-sided hex [lo, hi]."""
    lo, hi = np.asarray(lo, dtype=np.float64), np.asarray(hi, dtype=np.float64)
    c, h = 0.5 * (lo + hi), 0.5 * (hi - lo)
    return hex_from(lambda a, b, g: c + h * np.array([a, b, g]))


@dataclasses.dataclass
class HandCase:
    xyz: np.ndarray      # [27 n_elem, 3]  (no shared nodes)
    conn27: np.ndarray   # [n_elem, 27] i32
    adj6: np.ndarray     # [n_elem, 6] i32, all -1: every element is its own flood-fill component
    faces: np.ndarray    # [n_face, 9, 3]

    @property
    def n_elem(self) -> int:
        return int(self.conn27.shape[0])

    @property
    def n_face(self) -> int:
        return int(self.faces.shape[0])


def assemble(hexes: Sequence[np.ndarray], faces: Sequence[np.ndarray]) -> HandCase:
    n = len(hexes)
    xyz = np.ascontiguousarray(np.concatenate([np.asarray(h, dtype=np.float64).reshape(27, 3) for h in hexes]))
    conn = np.arange(27 * n, dtype=np.int32).reshape(n, 27)
    adj = np.full((n, 6), -1, dtype=np.int32)
    F = np.ascontiguousarray(np.stack([np.asarray(f, dtype=np.float64).reshape(9, 3) for f in faces]))
    return HandCase(xyz, conn, adj, F)


# ---------------------------------------------------------------------------------------------
# surfaces of the tie-rule cases
def knife_edge_faces(extend_a: float = 0.0) -> list:
    """PAPER.md Fig. 6(a): a thin wedge body {z < 0, z > x/2, x < 0} seen from beyond its edge (the y axis).
    Face A: the top z = 0, x in [-1, extend_a], outward normal +z.  Face B: the underside z = x / 2,
    x in [-1, 0], outward normal (1, 0, -2)/sqrt 5.  With extend_a = 0 they share the edge x = z = 0."""
    A = flat_quad([-1.0, 0.0, 0.0], [1.0 + extend_a, 0.0, 0.0], [0.0, 1.0, 0.0])          # eu x ev = +z
    B = flat_quad([-1.0, 0.0, -0.5], [0.0, 1.0, 0.0], [1.0, 0.0, 0.5])                    # eu x ev = (0.5, 0, -1)
    return [A, B]


def plate_faces(half: float = 0.5) -> list:
    """A plate body |z| < half (Fig. 6(b) / Fig. 14 seen from inside the solid): top face normal +z,
    bottom face normal -z; both span [-1,1]^2 in x, y."""
    top = flat_quad([-1.0, -1.0, half], [2.0, 0.0, 0.0], [0.0, 2.0, 0.0])
    bot = flat_quad([-1.0, -1.0, -half], [0.0, 2.0, 0.0], [2.0, 0.0, 0.0])
    return [top, bot]


def slot_faces(half: float = 0.5) -> list:
    """A straight-sided slot (Fig. 14): the FLUID is |z| < half, the solid lies above and below;
    upper wall z = +half with outward (into the fluid) normal -z, lower wall z = -half with normal +z."""
    up = flat_quad([-1.0, -1.0, half], [0.0, 2.0, 0.0], [2.0, 0.0, 0.0])
    low = flat_quad([-1.0, -1.0, -half], [2.0, 0.0, 0.0], [0.0, 2.0, 0.0])
    return [up, low]


def corner_faces() -> list:
    """Convex 90-degree edge of the body {x < 0, z < 0} along the y axis: face A z = 0 (x in [-1,0], normal +z),
    face B x = 0 (z in [-1,0], normal +x)."""
    A = flat_quad([-1.0, 0.0, 0.0], [1.0, 0.0, 0.0], [0.0, 1.0, 0.0])
    B = flat_quad([0.0, 0.0, -1.0], [0.0, 1.0, 0.0], [0.0, 0.0, 1.0])
    return [A, B]


def paraboloid_face(a: float, u0: float = 0.0, v0: float = 0.0, flip: bool = False) -> np.ndarray:
    """z = a ((x - u0)^2 + (y - v0)^2) over (x, y) in [-1,1]^2 with x = s, y = t: exactly biquadratic.
    Normal (x_s cross x_t) points to +z at the vertex (flip: swap s and t, normal to -z)."""
    if flip:
        return quad_from(lambda s, t: [t, s, a * ((t - u0) ** 2 + (s - v0) ** 2)])
    return quad_from(lambda s, t: [s, t, a * ((s - u0) ** 2 + (t - v0) ** 2)])


def point_hex(p) -> np.ndarray:
    """Degenerate element: all 27 nodes at p (every boundary patch is the point p)."""
    return np.tile(np.asarray(p, dtype=np.float64), (27, 1))
