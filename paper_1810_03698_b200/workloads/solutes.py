"""Synthetic solutes: AMOEBA-style site draws, a protein-like random-walk globule, and
its van-der-Waals-union surface triangulated on a grid (no method arithmetic).

Recipes: BASELINE.json configs[1..4] as read in DESIGN.md section 4."""
from __future__ import annotations

import numpy as np

from .meshes import check_closed_oriented


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def draw_multipoles(rng, n):
    """q ~ U[-0.5,0.5] e; dipole components ~ N(0,0.2) e*A; quadrupole symmetric with
    N(0,0.3) entries, trace removed (Eq. 7 convention needs a traceless tensor)."""
    q = rng.uniform(-0.5, 0.5, n)
    dip = rng.normal(0.0, 0.2, (n, 3))
    e = rng.normal(0.0, 0.3, (n, 6))  # xx,xy,xz,yy,yz,zz
    tr = (e[:, 0] + e[:, 3] + e[:, 5]) / 3.0
    e[:, 0] -= tr
    e[:, 3] -= tr
    e[:, 5] -= tr
    return q, dip, e


def draw_sites(seed, n, ball_radius, min_sep=1.0, alpha=1.0):
    """`n` sites uniform in the ball r < ball_radius with rejection for a minimum
    separation (BASELINE configs[1]; min_sep is a DESIGN reading), each its own
    polarization group."""
    rng = _rng(seed)
    pos = []
    while len(pos) < n:
        p = rng.uniform(-ball_radius, ball_radius, 3)
        if np.dot(p, p) >= ball_radius ** 2:
            continue
        if any(np.linalg.norm(p - o) < min_sep for o in pos):
            continue
        pos.append(p)
    pos = np.array(pos)
    q, dip, quad = draw_multipoles(rng, n)
    return dict(pos=pos, q=q, dip=dip, quad=quad, alpha=np.full(n, float(alpha)),
                group=np.arange(n, dtype=np.int32))


def random_chain_globule(seed, n_atoms, ball_radius=None, step=1.5, min_nonbonded=2.0,
                         group_size=4, alpha=1.0, n_try=32, max_stall=6):
    """Protein-like solute (BASELINE configs[2]): a seeded random-walk chain with
    `step`-Angstrom bonds, bond angle U[100,120] degrees, uniform torsion, radii
    U[1.2,2.0] A, confined to a ball (14 A at 1000 atoms, scaling with n^(1/3)) by
    rejecting steps that leave it or come within `min_nonbonded` of a non-bonded atom.
    On a dead end the walk backtracks a few atoms; after `max_stall` dead ends without
    progress the chain is broken and a new segment starts at a free spot of the ball (a
    multi-chain globule, like the paper's larger proteins), so the cost stays linear in
    n_atoms.  Sites sit on the atom centres with the configs[1] multipole distributions;
    polarization group = atom index // group_size.

    All candidate steps of one atom are tested at once against a dense cell grid (cell
    edge = min_nonbonded, up to 8 atoms per cell)."""
    rng = _rng(seed)
    if ball_radius is None:
        ball_radius = 14.0 * (n_atoms / 1000.0) ** (1.0 / 3.0)
    cell = float(min_nonbonded)
    ng = int(np.ceil(2.0 * ball_radius / cell)) + 4
    origin = -0.5 * ng * cell
    slots = 8
    cell_cnt = np.zeros((ng, ng, ng), dtype=np.int32)
    cell_atoms = -np.ones((ng, ng, ng, slots), dtype=np.int64)
    pos = np.zeros((n_atoms + 1, 3))                 # row n_atoms: a far-away dummy for empty slots
    pos[n_atoms] = 1e9
    nb = np.array([(dx, dy, dz) for dx in (-1, 0, 1) for dy in (-1, 0, 1) for dz in (-1, 0, 1)])
    r2min = min_nonbonded ** 2

    def cell_of(p):
        return np.floor((p - origin) / cell).astype(np.int64)

    def free_mask(cand, skip0, skip1):
        """cand [m][3] -> bool[m]: inside the ball and clear of every placed atom but the two skipped."""
        inside = np.einsum("ij,ij->i", cand, cand) <= ball_radius ** 2
        c = cell_of(cand)[:, None, :] + nb[None, :, :]                     # [m][27][3]
        ids = cell_atoms[c[..., 0], c[..., 1], c[..., 2]]                  # [m][27][slots]
        ids = ids.reshape(cand.shape[0], -1)
        ids = np.where((ids == skip0) | (ids == skip1) | (ids < 0), n_atoms, ids)
        d = pos[ids] - cand[:, None, :]
        clear = (np.einsum("ijk,ijk->ij", d, d) >= r2min).all(axis=1)
        return inside & clear

    def place(i, p):
        pos[i] = p
        c = cell_of(p)
        k = cell_cnt[c[0], c[1], c[2]]
        if k >= slots:
            raise RuntimeError("globule generator: cell overflow")
        cell_atoms[c[0], c[1], c[2], k] = i
        cell_cnt[c[0], c[1], c[2]] = k + 1

    def unplace(i):
        c = cell_of(pos[i])
        k = cell_cnt[c[0], c[1], c[2]]
        row = cell_atoms[c[0], c[1], c[2]]
        j = int(np.nonzero(row[:k] == i)[0][0])
        row[j] = row[k - 1]
        row[k - 1] = -1
        cell_cnt[c[0], c[1], c[2]] = k - 1

    def unit(v):
        return v / np.linalg.norm(v)

    def start_segment(i):
        """Atoms i and i+1 of a new chain segment at a free spot (i+1 may run past the end)."""
        for _ in range(10000):
            c = rng.uniform(-ball_radius, ball_radius, (64, 3))
            ok = np.nonzero(free_mask(c, -2, -2))[0]
            for k in ok:
                if i + 1 >= n_atoms:
                    place(i, c[k])
                    return
                d = rng.normal(size=(16, 3))
                d /= np.linalg.norm(d, axis=1)[:, None]
                c2 = c[k] + step * d
                ok2 = np.nonzero(free_mask(c2, -2, -2))[0]
                if ok2.size:
                    place(i, c[k])
                    place(i + 1, c2[ok2[0]])
                    return
        raise RuntimeError("globule generator: no free spot left in the ball")

    seg_start = 0
    seg_starts = [0]
    place(0, rng.normal(0, 0.5, 3))
    place(1, pos[0] + step * unit(rng.normal(size=3)))
    i = 2
    high = 2                                          # furthest atom index reached so far
    stall = 0
    n_segments = 1
    while i < n_atoms:
        prev = unit(pos[i - 1] - pos[i - 2])
        a = np.cross(prev, [1.0, 0.0, 0.0])
        if np.linalg.norm(a) < 1e-3:
            a = np.cross(prev, [0.0, 1.0, 0.0])
        a = unit(a)
        b = np.cross(prev, a)
        dev = np.pi - np.deg2rad(rng.uniform(100.0, 120.0, n_try))   # deviation of the new bond from the old direction
        tors = rng.uniform(0.0, 2.0 * np.pi, n_try)
        dirn = (np.cos(dev)[:, None] * prev[None, :]
                + np.sin(dev)[:, None] * (np.cos(tors)[:, None] * a[None, :] + np.sin(tors)[:, None] * b[None, :]))
        cand = pos[i - 1] + step * dirn
        ok = np.nonzero(free_mask(cand, i - 1, i - 2))[0]
        if ok.size:
            place(i, cand[ok[0]])
            i += 1
            if i > high:
                high = i
                stall = 0
            continue
        stall += 1
        if stall > max_stall:                         # trapped: break the chain here
            seg_start = i
            seg_starts.append(i)
            start_segment(i)
            n_segments += 1
            i = min(i + 2, n_atoms)
            high = max(high, i)
            stall = 0
            continue
        back = min(i - seg_start - 2, 1 + stall)
        for j in range(i - 1, i - 1 - back, -1):
            unplace(j)
        i -= back
    pos = pos[:n_atoms]
    radii = rng.uniform(1.2, 2.0, n_atoms)
    q, dip, quad = draw_multipoles(rng, n_atoms)
    return dict(pos=pos.copy(), radii=radii, q=q, dip=dip, quad=quad,
                alpha=np.full(n_atoms, float(alpha)),
                group=(np.arange(n_atoms) // group_size).astype(np.int32),
                ball_radius=float(ball_radius), n_segments=n_segments,
                seg_starts=np.array(seg_starts, dtype=np.int64))


# ---------------------------------------------------------------------------
# van der Waals union surface by "surface nets" on a regular grid


def _level_set(centres, radii, h, pad):
    lo = (centres - radii[:, None]).min(axis=0) - pad
    hi = (centres + radii[:, None]).max(axis=0) + pad
    n = np.ceil((hi - lo) / h).astype(int) + 1
    f = np.full(tuple(n), 10.0)
    ax = [lo[d] + h * np.arange(n[d]) for d in range(3)]
    for c, r in zip(centres, radii):
        reach = r + 1.5 * h
        i0 = np.maximum(np.floor((c - reach - lo) / h).astype(int), 0)
        i1 = np.minimum(np.ceil((c + reach - lo) / h).astype(int) + 1, n)
        gx = ax[0][i0[0]:i1[0]] - c[0]
        gy = ax[1][i0[1]:i1[1]] - c[1]
        gz = ax[2][i0[2]:i1[2]] - c[2]
        d = np.sqrt(gx[:, None, None] ** 2 + gy[None, :, None] ** 2 + gz[None, None, :] ** 2) - r
        blk = f[i0[0]:i1[0], i0[1]:i1[1], i0[2]:i1[2]]
        np.minimum(blk, d, out=blk)
    return f, lo


def _fix_topology(f):
    """Fill cavities (exterior = the outside component touching the grid boundary) and
    remove checkerboard faces (which would give edges shared by four quads)."""
    from scipy import ndimage
    outside = f >= 0
    lab, _ = ndimage.label(outside)
    ext = lab == lab[0, 0, 0]
    f = np.where(outside & ~ext, -1e-3, f)
    for _ in range(64):
        ins = f < 0
        changed = False
        for axis in range(3):
            sl = [slice(None)] * 3
            o1, o2 = [d for d in range(3) if d != axis]

            def sh(a, d1, d2):
                s = list(sl)
                s[o1] = slice(d1, a.shape[o1] - 1 + d1)
                s[o2] = slice(d2, a.shape[o2] - 1 + d2)
                return a[tuple(s)]

            a, b, c, d = sh(ins, 0, 0), sh(ins, 1, 0), sh(ins, 0, 1), sh(ins, 1, 1)
            bad = (a & d & ~b & ~c) | (b & c & ~a & ~d)
            if bad.any():
                changed = True
                for d1 in (0, 1):
                    for d2 in (0, 1):
                        s = list(sl)
                        s[o1] = slice(d1, f.shape[o1] - 1 + d1)
                        s[o2] = slice(d2, f.shape[o2] - 1 + d2)
                        view = f[tuple(s)]
                        view[bad & (view >= 0)] = -1e-3
        if not changed:
            break
    return f


def _surface_nets(f, lo, h, blend=0.7):
    ins = f < 0
    nx, ny, nz = f.shape
    # ---- one vertex per cell that the surface crosses ------------------------------
    cs = np.zeros((nx - 1, ny - 1, nz - 1), dtype=np.int8)
    for dx in (0, 1):
        for dy in (0, 1):
            for dz in (0, 1):
                cs += ins[dx:nx - 1 + dx, dy:ny - 1 + dy, dz:nz - 1 + dz]
    active = (cs > 0) & (cs < 8)
    cell_id = -np.ones(active.shape, dtype=np.int64)
    ai, aj, ak = np.nonzero(active)
    cell_id[ai, aj, ak] = np.arange(ai.size)
    acc = np.zeros((ai.size, 3))
    cnt = np.zeros(ai.size)
    # the 12 edges of a cell: (corner offset, axis)
    for axis in range(3):
        o1, o2 = [d for d in range(3) if d != axis]
        for d1 in (0, 1):
            for d2 in (0, 1):
                off = np.zeros(3, dtype=int)
                off[o1], off[o2] = d1, d2
                p0 = (ai + off[0], aj + off[1], ak + off[2])
                off2 = off.copy()
                off2[axis] = 1
                p1 = (ai + off2[0], aj + off2[1], ak + off2[2])
                f0, f1 = f[p0], f[p1]
                cross = (f0 < 0) != (f1 < 0)
                t = np.where(cross, f0 / np.where(cross, f0 - f1, 1.0), 0.0)
                pt = np.stack([off[0] + (t if axis == 0 else 0.0) * np.ones_like(t),
                               off[1] + (t if axis == 1 else 0.0) * np.ones_like(t),
                               off[2] + (t if axis == 2 else 0.0) * np.ones_like(t)], axis=1)
                acc += np.where(cross[:, None], pt, 0.0)
                cnt += cross
    mean = acc / cnt[:, None]
    local = 0.5 + blend * (mean - 0.5)              # pulled toward the cell centre: no tiny edges
    verts = lo[None, :] + h * (np.stack([ai, aj, ak], axis=1) + local)
    # ---- one quad per sign-changing grid edge ---------------------------------------
    tris = []
    for axis in range(3):
        o1, o2 = (axis + 1) % 3, (axis + 2) % 3     # cyclic: (y,z), (z,x), (x,y)
        s0 = [slice(None)] * 3
        s1 = [slice(None)] * 3
        s0[axis] = slice(0, f.shape[axis] - 1)
        s1[axis] = slice(1, f.shape[axis])
        a_in, b_in = ins[tuple(s0)], ins[tuple(s1)]
        cross = a_in != b_in
        ei = np.array(np.nonzero(cross))            # edge base node indices [3][ne]
        if ei.shape[1] == 0:
            continue
        if (ei[o1] < 1).any() or (ei[o2] < 1).any() or (ei[o1] > f.shape[o1] - 2).any() \
                or (ei[o2] > f.shape[o2] - 2).any():
            raise RuntimeError("surface touches the grid boundary; increase pad")

        def cell(d1, d2):
            idx = ei.copy()
            idx[o1] += d1
            idx[o2] += d2
            return cell_id[idx[0], idx[1], idx[2]]

        q0, q1, q2, q3 = cell(-1, -1), cell(0, -1), cell(0, 0), cell(-1, 0)
        a_inside = a_in[cross]                      # a inside, b outside -> normal +axis
        q = np.stack([q0, q1, q2, q3], axis=1)
        q[~a_inside] = q[~a_inside][:, ::-1]
        assert (q >= 0).all()
        p = verts[q]                                # [ne][4][3]
        d02 = np.linalg.norm(p[:, 0] - p[:, 2], axis=1)
        d13 = np.linalg.norm(p[:, 1] - p[:, 3], axis=1)
        use02 = d02 <= d13
        t1 = np.where(use02[:, None], q[:, [0, 1, 2]], q[:, [0, 1, 3]])
        t2 = np.where(use02[:, None], q[:, [0, 2, 3]], q[:, [1, 2, 3]])
        tris.append(t1)
        tris.append(t2)
    tris = np.concatenate(tris).astype(np.int32)
    return verts, tris


def vdw_surface(centres, radii, target_panels=None, h=None, tol=0.05, max_iter=6, pad=None, iso_shift=0.35):
    """Triangulate the boundary of the union of spheres (cavities dropped).  Either a grid
    spacing `h` is given or it is tuned so the panel count lands within `tol` of
    `target_panels` (the controlling quantity in BASELINE.json's configs).
    Returns (verts, tris, info)."""
    centres = np.asarray(centres, dtype=np.float64)
    radii = np.asarray(radii, dtype=np.float64)

    def run(hh):
        f, lo = _level_set(centres, radii, hh, pad if pad is not None else 3.0 * hh)
        # The smoothed net (vertices pulled toward cell centres) cuts up to ~0.5 h INSIDE the spheres
        # where they are convex, leaving atom centres far closer to the dielectric boundary than their
        # radius.  Meshing the level set at +iso_shift*h instead keeps the whole net outside the union
        # (measured: min over vertices and centroids of min_i(|x - c_i| - r_i) >= -0.05 A at h = 1.15).
        f = _fix_topology(f - iso_shift * hh)
        return _surface_nets(f, lo, hh)

    if h is None:
        h = 1.0
        verts = tris = None
        for _ in range(max_iter):
            verts, tris = run(h)
            n = tris.shape[0]
            if abs(n - target_panels) <= tol * target_panels:
                break
            h *= (n / target_panels) ** 0.5
    else:
        verts, tris = run(h)
    # drop unreferenced vertices (none expected) and verify
    used = np.unique(tris)
    remap = -np.ones(verts.shape[0], dtype=np.int64)
    remap[used] = np.arange(used.size)
    verts = verts[used]
    tris = remap[tris].astype(np.int32)
    ok = check_closed_oriented(verts, tris)
    return verts, tris, dict(h=float(h), closed_oriented=bool(ok))
