"""The five BASELINE.json configs (C0..C4) as seeded synthetic workloads.

Seeds: 181003698 + 1000*config + replica.  No method arithmetic."""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from .meshes import icosphere
from .solutes import draw_sites, random_chain_globule, vdw_surface

BASE_SEED = 181003698


def seed_for(config: int, replica: int = 0) -> int:
    return BASE_SEED + 1000 * config + replica


@dataclass
class Workload:
    name: str
    verts: np.ndarray
    tris: np.ndarray
    sites: dict                      # pos, q, dip, quad, alpha, group
    params: dict                     # eps_in, eps_out, kappa, K_far, theta, order_P, gmres_tol, scf_tol_debye, thole_a
    info: dict = field(default_factory=dict)


_COMMON = dict(eps_in=1.0, eps_out=80.0, kappa=0.125, thole_a=0.39, theta=0.5, order_P=6,
               scf_tol_debye=1e-7, gmres_tol=1e-6)


def _one_site(q=0.0, dip=(0, 0, 0), quad=(0, 0, 0, 0, 0, 0), alpha=0.0):
    return dict(pos=np.zeros((1, 3)), q=np.array([float(q)]), dip=np.array([dip], dtype=float),
                quad=np.array([quad], dtype=float), alpha=np.array([float(alpha)]),
                group=np.zeros(1, dtype=np.int32))


def config_c0(kind: str = "charge", subdiv: int = 2, radius: float = 4.0):
    """configs[0]: sphere R=4, icosphere subdiv 2 (320 panels), K=4, one centred site."""
    verts, tris = icosphere(radius, subdiv)
    site = {"charge": _one_site(q=1.0),
            "dipole": _one_site(dip=(0, 0, 1.0)),
            "quadrupole": _one_site(quad=(-0.5, 0, 0, -0.5, 0, 1.0)),
            "polarizable_dipole": _one_site(dip=(0, 0, 1.0), alpha=1.0)}[kind]
    prm = dict(_COMMON, K_far=4, gmres_tol=1e-10)
    return Workload(f"C0-{kind}", verts, tris, site, prm, dict(radius=radius, subdiv=subdiv))


def config_c1(subdiv: int = 4, radius: float = 6.0, n_sites: int = 12):
    """configs[1]: sphere R=6, subdiv 4 (5120 panels), K=7, 12 random polarizable sites in r<0.7R."""
    verts, tris = icosphere(radius, subdiv)
    sites = draw_sites(seed_for(1), n_sites, 0.7 * radius, min_sep=1.0, alpha=1.0)
    return Workload("C1", verts, tris, sites, dict(_COMMON, K_far=7), dict(radius=radius, subdiv=subdiv))


def _globule_workload(name, cfg, n_atoms, target_panels, replica=0, extra=None):
    g = random_chain_globule(seed_for(cfg, replica), n_atoms)
    pos, radii = g["pos"], g["radii"]
    if extra is not None:
        pos = np.concatenate([pos, extra["pos"]])
        radii = np.concatenate([radii, extra["radii"]])
    verts, tris, info = vdw_surface(pos, radii, target_panels=target_panels)
    sites = {k: g[k] for k in ("pos", "q", "dip", "quad", "alpha", "group")}
    if extra is not None:
        gmax = int(sites["group"].max()) + 1
        sites = {k: np.concatenate([sites[k], extra[k] + (gmax if k == "group" else 0)])
                 for k in sites}
        sites["group"] = sites["group"].astype(np.int32)
    info.update(n_atoms=int(pos.shape[0]), ball_radius=g["ball_radius"])
    return Workload(name, verts, tris, sites, dict(_COMMON, K_far=7), info), g


def config_c2(n_atoms: int = 1000, target_panels: int = 10_000):
    """configs[2]: 1,000-atom protein-like globule, ~10k panels (2 triangles/A^2)."""
    return _globule_workload("C2", 2, n_atoms, target_panels)[0]


def config_c3(which: str = "complex", n_receptor: int = 3000, n_ligand: int = 50,
              target_panels: int = 60_000):
    """configs[3]: binding triple.  Receptor and ligand draws are shared by the three
    solves; the ligand is translated to 3 A from the receptor surface."""
    rec = random_chain_globule(seed_for(3, 0), n_receptor)
    lig = random_chain_globule(seed_for(3, 1), n_ligand)
    rng = np.random.Generator(np.random.PCG64(seed_for(3, 2)))
    u = rng.normal(size=3)
    u /= np.linalg.norm(u)
    # push the ligand out along u until its atoms clear every receptor atom surface by 3 A
    lig_c = lig["pos"] - lig["pos"].mean(axis=0)
    t = rec["ball_radius"] * 0.5
    while True:
        p = lig_c + t * u
        d = np.linalg.norm(p[:, None, :] - rec["pos"][None, :, :], axis=2) - rec["radii"][None, :] - lig["radii"][:, None]
        if d.min() >= 3.0:
            break
        t += 0.25
    lig = dict(lig, pos=lig_c + t * u)
    dens = target_panels / (n_receptor + n_ligand)

    def surf(parts, tp):
        pos = np.concatenate([p["pos"] for p in parts])
        radii = np.concatenate([p["radii"] for p in parts])
        verts, tris, info = vdw_surface(pos, radii, target_panels=int(tp))
        sites = {k: np.concatenate([p[k] for p in parts]) for k in ("pos", "q", "dip", "quad", "alpha")}
        groups, base = [], 0
        for p in parts:
            groups.append(p["group"] + base)
            base += int(p["group"].max()) + 1
        sites["group"] = np.concatenate(groups).astype(np.int32)
        info.update(n_atoms=int(pos.shape[0]))
        return verts, tris, sites, info

    parts = {"complex": [rec, lig], "receptor": [rec], "ligand": [lig]}[which]
    tp = dens * sum(p["pos"].shape[0] for p in parts)
    if which == "ligand":
        tp = max(tp, 2000)
    verts, tris, sites, info = surf(parts, tp)
    return Workload(f"C3-{which}", verts, tris, sites, dict(_COMMON, K_far=7), info)


def config_c4(n_atoms: int = 20_000, target_panels: int = 1_000_000):
    """configs[4]: 20,000-atom globule, ~1M panels, K=7."""
    return _globule_workload("C4", 4, n_atoms, target_panels)[0]


CONFIGS = {
    "C0": config_c0, "C1": config_c1, "C2": config_c2, "C3": config_c3, "C4": config_c4,
}


def _cache_dir():
    """Generated globule workloads (C2-C4: 1-60 s of surface netting each) are kept as .npz files in a scratch
    directory outside the repository -- PB_WORKLOAD_CACHE, default /tmp/paper_1810_03698_b200_workloads; set it to
    an empty string to switch the cache off.  The file name carries a hash of the generator sources, the config and
    its arguments, so a changed recipe never reads a stale file; nothing depends on the cache being there."""
    import os
    d = os.environ.get("PB_WORKLOAD_CACHE", "/tmp/paper_1810_03698_b200_workloads")
    return d or None


def _cache_key(name, kw):
    import hashlib
    import os
    h = hashlib.sha256()
    here = os.path.dirname(os.path.abspath(__file__))
    for f in ("configs.py", "meshes.py", "solutes.py"):
        with open(os.path.join(here, f), "rb") as fh:
            h.update(fh.read())
    h.update(repr((name, sorted(kw.items()), np.__version__)).encode())
    return h.hexdigest()[:20]


def make_config(name: str, **kw) -> Workload:
    import os
    d = _cache_dir() if name in ("C2", "C3", "C4") else None
    path = os.path.join(d, f"{name}-{_cache_key(name, kw)}.npz") if d else None
    if path and os.path.exists(path):
        try:
            import json
            z = np.load(path, allow_pickle=False)
            meta = json.loads(str(z["meta"]))
            sites = {k[5:]: z[k] for k in z.files if k.startswith("site_")}
            return Workload(meta["name"], z["verts"], z["tris"], sites, meta["params"], meta["info"])
        except Exception:
            pass                                     # unreadable file: regenerate
    w = CONFIGS[name](**kw)
    if path:
        try:
            import json
            os.makedirs(d, exist_ok=True)
            info = {k: (v.item() if hasattr(v, "item") else v) for k, v in w.info.items()}
            meta = json.dumps(dict(name=w.name, params=w.params, info=info), default=float)
            tmp = f"{path}.{os.getpid()}.tmp.npz"
            np.savez(tmp, verts=w.verts, tris=w.tris, meta=np.array(meta), **{"site_" + k: v for k, v in w.sites.items()})
            os.replace(tmp, path)
        except Exception:
            pass                                     # read-only or full scratch space: the cache is optional
    return w
