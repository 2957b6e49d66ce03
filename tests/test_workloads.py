"""Seeded input generators: shapes, determinism, closed outward meshes, sites inside."""
import numpy as np
import pytest

from paper_1810_03698_b200.workloads import (check_closed_oriented, icosphere, make_config, mesh_stats,
                                             random_chain_globule, seed_for, vdw_surface)


@pytest.mark.parametrize("subdiv,panels", [(0, 20), (1, 80), (2, 320), (3, 1280)])
def test_icosphere(subdiv, panels):
    v, t = icosphere(4.0, subdiv)
    assert t.shape == (panels, 3) and t.dtype == np.int32
    assert v.shape[0] == panels // 2 + 2
    np.testing.assert_allclose(np.linalg.norm(v, axis=1), 4.0, rtol=1e-14)
    assert check_closed_oriented(v, t)
    assert not check_closed_oriented(v, t[:, [0, 2, 1]])          # inward orientation is rejected
    assert not check_closed_oriented(v, t[:-1])                   # a hole is rejected


def test_c0_and_c1_configs():
    w = make_config("C0", kind="quadrupole")
    assert w.tris.shape[0] == 320 and w.params["K_far"] == 4
    q = w.sites["quad"][0]
    assert abs(q[0] + q[3] + q[5]) < 1e-15 and q[5] == 1.0
    w1 = make_config("C1")
    w1b = make_config("C1")
    assert w1.tris.shape[0] == 5120 and w1.sites["pos"].shape == (12, 3)
    for k in w1.sites:
        np.testing.assert_array_equal(w1.sites[k], w1b.sites[k])         # seeded
    r = np.linalg.norm(w1.sites["pos"], axis=1)
    assert r.max() < 0.7 * 6.0
    d = np.linalg.norm(w1.sites["pos"][:, None] - w1.sites["pos"][None], axis=2) + 10 * np.eye(12)
    assert d.min() >= 1.0
    tr = w1.sites["quad"][:, 0] + w1.sites["quad"][:, 3] + w1.sites["quad"][:, 5]
    assert np.abs(tr).max() < 1e-15
    assert np.all(np.abs(w1.sites["q"]) <= 0.5) and np.all(w1.sites["alpha"] == 1.0)
    assert seed_for(1) == 181003698 + 1000


def _check_chain(g, n):
    p = g["pos"]
    seg = np.zeros(n, dtype=np.int64)
    seg[g["seg_starts"][1:]] = 1
    seg = np.cumsum(seg)                                   # segment id of every atom
    same1 = seg[1:] == seg[:-1]
    bonds = np.linalg.norm(p[1:] - p[:-1], axis=1)
    np.testing.assert_allclose(bonds[same1], 1.5, rtol=1e-12)
    same2 = seg[2:] == seg[:-2]
    a, b = p[:-2] - p[1:-1], p[2:] - p[1:-1]
    ang = np.degrees(np.arccos(np.einsum("ij,ij->i", a, b)[same2] / 2.25))
    assert ang.min() > 100 - 1e-6 and ang.max() < 120 + 1e-6
    assert np.linalg.norm(p, axis=1).max() <= g["ball_radius"] + 1e-9
    d = np.linalg.norm(p[:, None] - p[None], axis=2)
    i, j = np.triu_indices(n, 1)
    nonbonded = (j - i >= 3) | (seg[i] != seg[j])
    assert d[i, j][nonbonded].min() >= 2.0 - 1e-9
    assert g["radii"].min() >= 1.2 and g["radii"].max() <= 2.0
    assert np.diff(g["seg_starts"]).min(initial=2) >= 2      # no single-atom segments inside the chain


def test_globule_chain_geometry():
    g = random_chain_globule(seed_for(2), 300)
    _check_chain(g, 300)
    assert g["group"][7] == 1 and g["group"].dtype == np.int32
    g2 = random_chain_globule(seed_for(2), 300)
    np.testing.assert_array_equal(g["pos"], g2["pos"])          # seeded


def test_globule_chain_breaks_keep_the_cost_linear():
    """A ball this full traps the walk; the generator must break the chain (several segments)
    rather than thrash, and every segment must still obey the recipe."""
    import time
    t0 = time.perf_counter()
    g = random_chain_globule(seed_for(2), 2000)
    assert time.perf_counter() - t0 < 30.0
    assert g["n_segments"] == len(g["seg_starts"]) > 1
    _check_chain(g, 2000)


def test_vdw_surface_is_closed_and_hits_the_panel_count():
    g = random_chain_globule(seed_for(2), 120)
    v, t, info = vdw_surface(g["pos"], g["radii"], target_panels=2500)
    assert info["closed_oriented"]
    assert abs(t.shape[0] - 2500) <= 0.05 * 2500
    st = mesh_stats(v, t)
    assert st["min_area"] > 1e-4 and st["max_aspect"] < 30
    # every atom centre is inside: the solid angle of the surface seen from it is 4 pi
    c = v[t].mean(axis=1)
    n = np.cross(v[t[:, 1]] - v[t[:, 0]], v[t[:, 2]] - v[t[:, 0]]) / 2
    for x in g["pos"][::15]:
        d = c - x
        omega = np.sum(np.einsum("ij,ij->i", d, n) / np.linalg.norm(d, axis=1) ** 3)
        assert abs(omega - 4 * np.pi) < 1.0          # 1-point rule; outside would give 0
    # the net circumscribes the union: no vertex or centroid is inside an atom by more than 0.1 A,
    # so every site keeps (nearly) its atom's radius of clearance from the dielectric boundary
    for x in (v, c):
        f = (np.linalg.norm(x[:, None, :] - g["pos"][None], axis=2) - g["radii"][None]).min(axis=1)
        assert f.min() > -0.1 and f.mean() < 0.8       # (filled crevices and cavities lie further out)
    # two well-separated atoms give two closed components
    v2, t2, info2 = vdw_surface(np.array([[0.0, 0, 0], [8.0, 0, 0]]), np.array([1.5, 1.5]), h=0.4, iso_shift=0.0)
    assert info2["closed_oriented"]
    area = 0.5 * np.linalg.norm(np.cross(v2[t2[:, 1]] - v2[t2[:, 0]], v2[t2[:, 2]] - v2[t2[:, 0]]), axis=1).sum()
    assert abs(area - 2 * 4 * np.pi * 1.5 ** 2) < 0.08 * area
