"""Closed triangulated surfaces: icosphere and mesh sanity checks (no method arithmetic)."""
from __future__ import annotations

import numpy as np


def icosphere(radius: float, subdiv: int):
    """Icosahedron split 4-ways `subdiv` times, vertices re-projected on the sphere of
    `radius` (inscribed polyhedron), outward oriented (DESIGN R-21).
    Returns (verts float64 [nv][3], tris int32 [20*4^subdiv][3])."""
    t = (1.0 + 5.0 ** 0.5) / 2.0
    v = np.array([[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0],
                  [0, -1, t], [0, 1, t], [0, -1, -t], [0, 1, -t],
                  [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array([[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
                  [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
                  [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
                  [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]], dtype=np.int64)
    verts = [tuple(p) for p in v]
    for _ in range(subdiv):
        cache = {}
        new_f = []

        def mid(a, b):
            key = (a, b) if a < b else (b, a)
            if key not in cache:
                m = (np.array(verts[a]) + np.array(verts[b])) * 0.5
                m /= np.linalg.norm(m)
                verts.append(tuple(m))
                cache[key] = len(verts) - 1
            return cache[key]

        for a, b, c in f:
            ab, bc, ca = mid(a, b), mid(b, c), mid(c, a)
            new_f += [[a, ab, ca], [b, bc, ab], [c, ca, bc], [ab, bc, ca]]
        f = np.array(new_f, dtype=np.int64)
    verts = np.array(verts, dtype=np.float64) * radius
    tris = f.astype(np.int32)
    # outward orientation: n . c > 0
    a, b, c = verts[tris[:, 0]], verts[tris[:, 1]], verts[tris[:, 2]]
    n = np.cross(b - a, c - a)
    flip = np.einsum("ij,ij->i", n, a + b + c) < 0
    tris[flip] = tris[flip][:, [0, 2, 1]]
    return verts, tris


def check_closed_oriented(verts, tris):
    """True iff every undirected edge is shared by exactly two triangles, the two uses
    have opposite direction (consistent orientation), and the enclosed signed volume is
    positive (outward normals)."""
    tris = np.asarray(tris, dtype=np.int64)
    e = np.concatenate([tris[:, [0, 1]], tris[:, [1, 2]], tris[:, [2, 0]]])
    nv = int(tris.max()) + 1
    fwd = e[:, 0] * nv + e[:, 1]
    bwd = e[:, 1] * nv + e[:, 0]
    if np.unique(fwd).size != fwd.size:
        return False
    if not np.array_equal(np.sort(fwd), np.sort(bwd)):
        return False
    a, b, c = verts[tris[:, 0]], verts[tris[:, 1]], verts[tris[:, 2]]
    vol = np.einsum("ij,ij->i", a, np.cross(b, c)).sum() / 6.0
    return bool(vol > 0)


def mesh_stats(verts, tris):
    a, b, c = verts[tris[:, 0]], verts[tris[:, 1]], verts[tris[:, 2]]
    n = np.cross(b - a, c - a)
    area = 0.5 * np.linalg.norm(n, axis=1)
    e = np.stack([np.linalg.norm(b - a, axis=1), np.linalg.norm(c - b, axis=1), np.linalg.norm(a - c, axis=1)])
    return dict(panels=int(tris.shape[0]), vertices=int(verts.shape[0]), area=float(area.sum()),
                min_area=float(area.min()), max_area=float(area.max()),
                tri_per_A2=float(tris.shape[0] / area.sum()),
                max_aspect=float((e.max(axis=0) ** 2 / (area * 4 / 3 ** 0.5)).max()))
