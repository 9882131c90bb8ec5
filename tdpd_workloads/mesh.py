"""Triangulated red-blood-cell surface used as INPUT by both the CUDA path and the oracle.

This module only produces vertex coordinates and a triangle list.  It holds none of the
method's arithmetic (no bonds, dihedrals, rest lengths, areas, forces): the CUDA library and
the oracle each derive those from (verts, tris) on their own.

Recipe (SURVEY.md §8(c) "Mesh" pin; BASELINE config 3: "642-vertex membrane (level-3 subdivided
icosahedron mapped to the Evans–Fung biconcave shape, 7.82 um diameter; 1920 bonds, 1280
triangles)"):
  seed icosahedron = cyclic permutations of (0, +-1, +-phi) normalised; each level splits every
  triangle into 4 through edge midpoints projected back to the unit sphere; the unit sphere
  (x, y, z) is mapped to (D0 x/2, D0 y/2, D0 z [a0 + a1 s/4 + a2 s^2/16]), s = x^2 + y^2.
"""
from __future__ import annotations

import numpy as np

D0_RBC = 7.82
EF_A = (0.0518, 2.0026, -4.491)


def icosphere(level: int) -> tuple[np.ndarray, np.ndarray]:
    """Unit-sphere vertices [nv,3] float64 and triangles [nt,3] int32, CCW seen from outside."""
    phi = (1.0 + 5.0 ** 0.5) / 2.0
    v = []
    for a in (-1.0, 1.0):
        for b in (-phi, phi):
            v.append((0.0, a, b))
            v.append((a, b, 0.0))
            v.append((b, 0.0, a))
    verts = np.array(v, dtype=np.float64)
    verts /= np.linalg.norm(verts, axis=1, keepdims=True)
    # the 20 faces = all vertex triples that are mutually nearest neighbours
    d = np.linalg.norm(verts[:, None, :] - verts[None, :, :], axis=2)
    edge = d[d > 1e-9].min()
    adj = np.abs(d - edge) < 1e-9
    tris = []
    for i in range(12):
        for j in range(i + 1, 12):
            if not adj[i, j]:
                continue
            for k in range(j + 1, 12):
                if adj[i, k] and adj[j, k]:
                    tris.append((i, j, k))
    tris = np.array(tris, dtype=np.int64)
    assert tris.shape == (20, 3)
    tris = _orient_outward(verts, tris)
    for _ in range(level):
        verts, tris = _subdivide(verts, tris)
    return verts, tris.astype(np.int32)


def _orient_outward(verts: np.ndarray, tris: np.ndarray) -> np.ndarray:
    a, b, c = verts[tris[:, 0]], verts[tris[:, 1]], verts[tris[:, 2]]
    n = np.cross(b - a, c - a)
    flip = np.einsum("ij,ij->i", n, a + b + c) < 0.0
    tris = tris.copy()
    tris[flip] = tris[flip][:, [0, 2, 1]]
    return tris


def _subdivide(verts: np.ndarray, tris: np.ndarray) -> tuple[np.ndarray, np.ndarray]:
    verts = list(map(tuple, verts))
    mid: dict[tuple[int, int], int] = {}

    def midpoint(i: int, j: int) -> int:
        key = (i, j) if i < j else (j, i)
        if key not in mid:
            p = (np.array(verts[i]) + np.array(verts[j])) * 0.5
            p /= np.linalg.norm(p)
            mid[key] = len(verts)
            verts.append(tuple(p))
        return mid[key]

    out = []
    for a, b, c in tris:
        ab, bc, ca = midpoint(a, b), midpoint(b, c), midpoint(c, a)
        out += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
    return np.array(verts, dtype=np.float64), np.array(out, dtype=np.int64)


def evans_fung_map(unit_verts: np.ndarray, d0: float = D0_RBC) -> np.ndarray:
    """Map unit-sphere points onto the biconcave surface of diameter d0 (axis = z)."""
    x, y, z = unit_verts[:, 0], unit_verts[:, 1], unit_verts[:, 2]
    s = x * x + y * y
    a0, a1, a2 = EF_A
    out = np.empty_like(unit_verts)
    out[:, 0] = 0.5 * d0 * x
    out[:, 1] = 0.5 * d0 * y
    out[:, 2] = d0 * z * (a0 + a1 * s / 4.0 + a2 * s * s / 16.0)
    return out


def evans_fung_inside(p: np.ndarray, d0: float = D0_RBC) -> np.ndarray:
    """Boolean mask: is the point (cell frame, axis z) strictly inside the analytic surface."""
    r2 = p[:, 0] ** 2 + p[:, 1] ** 2
    t = r2 / (d0 * d0)
    a0, a1, a2 = EF_A
    inside_disc = t < 0.25
    root = np.sqrt(np.clip(1.0 - 4.0 * t, 0.0, None))
    half = d0 * root * (a0 + a1 * t + a2 * t * t)
    return inside_disc & (np.abs(p[:, 2]) < half)


def rbc_mesh(level: int = 3, d0: float = D0_RBC) -> tuple[np.ndarray, np.ndarray]:
    """(verts float64 [nv,3] in the cell frame, tris int32 [nt,3]); level 3 -> 642 / 1280."""
    u, tris = icosphere(level)
    return evans_fung_map(u, d0), tris


def random_rotations(rng: np.random.Generator, n: int) -> np.ndarray:
    """n uniform random rotation matrices from normalised 4-vectors of normals (unit quaternions)."""
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z)
    R[:, 0, 1] = 2 * (x * y - z * w)
    R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w)
    R[:, 1, 1] = 1 - 2 * (x * x + z * z)
    R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w)
    R[:, 2, 1] = 2 * (y * z + x * w)
    R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R
