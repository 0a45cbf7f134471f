"""CPU oracle of the donor search (PAPER.md 4.3, Eq. 1-5; SURVEY.md 8(f) "(later)").  TEST INFRASTRUCTURE ONLY.

Plain definition: the donor of a point p is an element e with reference coordinates X in [-1,1]^3 (within the paper's
small tolerance) such that x_e(X) = p, x_e the triquadratic Lagrange map of its 27 nodes (Eq. 1, K = 2).  Brute force:
EVERY element whose conservative box (oracle/dc_oracle.c orc_element_box) holds the point is tried, one after the
other, with the paper's Newton iteration (Eq. 3-5: Delta = p - x(X_n); X_{n+1} = X_n + J^-1 Delta; X limited to
[-1,1] + 1e-10; at most 10 iterations, L272-L278).  No tree, no shared code with the CUDA path.
"""
from __future__ import annotations

import numpy as np

from . import dc_oracle as O

MAXIT = 10
LIM = 1.0 + 1e-10


def lag(t):
    """Eq. 1, K = 2, nodes (-1, 0, 1): values and derivatives."""
    return (np.array([0.5 * t * (t - 1.0), 1.0 - t * t, 0.5 * t * (t + 1.0)]),
            np.array([t - 0.5, -2.0 * t, t + 0.5]))


def hex_map(X27, xi):
    """x(X) and J = dx/dX (Eq. 2, Eq. 5) of one element; X27 [27][3], node m = i + 3 j + 9 k."""
    lx, dx = lag(xi[0]); ly, dy = lag(xi[1]); lz, dz = lag(xi[2])
    N = np.einsum("k,j,i->kji", lz, ly, lx).reshape(27)
    Nx = np.einsum("k,j,i->kji", lz, ly, dx).reshape(27)
    Ny = np.einsum("k,j,i->kji", lz, dy, lx).reshape(27)
    Nz = np.einsum("k,j,i->kji", dz, ly, lx).reshape(27)
    return N @ X27, np.stack([Nx @ X27, Ny @ X27, Nz @ X27], axis=1)


def invert(X27, p, tol):
    """The paper's Newton iteration from the element centre; (converged, X)."""
    xi = np.zeros(3)
    for it in range(MAXIT + 1):
        x, J = hex_map(X27, xi)
        D = p - x
        if D @ D <= tol * tol:
            return True, xi
        if it == MAXIT:
            break
        try:
            step = np.linalg.solve(J, D)
        except np.linalg.LinAlgError:
            break
        xi = np.clip(xi + step, -LIM, LIM)
    return False, xi


def element_boxes(xyz, conn27):
    return np.array([O.element_box(xyz, conn27[e]) for e in range(conn27.shape[0])])


def find_donors(xyz, conn27, pts, boxes=None):
    """For each point: (sorted list of ALL elements that contain it, dict element -> X).  A point on a shared face has
    several donors; none = outside the grid."""
    xyz = np.asarray(xyz, float); pts = np.asarray(pts, float).reshape(-1, 3)
    boxes = element_boxes(xyz, conn27) if boxes is None else boxes
    out = []
    for p in pts:
        inside = np.all(boxes[:, :3] - 1e-12 <= p, axis=1) & np.all(p <= boxes[:, 3:] + 1e-12, axis=1)
        hits = {}
        for e in np.nonzero(inside)[0]:
            X27 = xyz[conn27[e]]
            diag = np.linalg.norm(boxes[e, 3:] - boxes[e, :3])
            ok, xi = invert(X27, p, 1e-12 * diag)
            if ok:
                hits[int(e)] = xi
        out.append(hits)
    return out
