"""pb_multipole_field_static (include/pb.h): the multipole field of Eq. (7), (14), (31), (32) through the entry point that
allocates nothing -- its partial sums live in a file-scope device array of the library -- against the existing path
pb_multipole_field, which takes them from the context's allocated scratch buffer.  Same kernels, chunking and summation
order, so the two agree to rounding (the bound is the direct-mode tolerance of the other GPU tests, 1e-11).

Collected last on purpose (the name): the suite runs with `pytest -x`.  The test makes no assumption about what ran
before it in the process: the static array may hold anything (another test's or an earlier call's partial sums)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-11


def rel(a, b):
    a, b = np.asarray(a, dtype=float), np.asarray(b, dtype=float)
    d = a - b
    return max(float(np.linalg.norm(d) / np.linalg.norm(b)), float(np.max(np.abs(d)) / np.max(np.abs(b))))


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test run without a CUDA device: the product has no CPU fallback")
    return torch


@pytest.fixture(scope="module")
def pbm(torch_cuda):
    from paper_1810_03698_b200 import pb
    pb.build()
    return pb


def _device_sites(torch, s, n=None):
    dev = torch.device("cuda", 0)
    cut = slice(0, n)
    f = lambda a, dt: torch.from_numpy(np.ascontiguousarray(np.asarray(a)[cut])).to(dev, dt).contiguous()
    return dict(pos=f(s["pos"], torch.float64), q=f(s["q"], torch.float64), dip=f(s["dip"], torch.float64),
                quad=f(s["quad"], torch.float64), alpha=f(s["alpha"], torch.float64), group=f(s["group"], torch.int32))


def test_static_entry_point_matches_the_allocating_path_on_calls_in_a_row(pbm, torch_cuda):
    torch = torch_cuda
    from paper_1810_03698_b200.workloads import make_config
    max_sites, nbytes = pbm.multipole_field_static_limit()
    assert max_sites == 4096 and 0 < nbytes <= 1 << 20          # the stated, modest maximum (include/pb.h)

    w = make_config("C2")                                         # BASELINE configs[2]: 1,000 AMOEBA-style sites
    s = w.sites
    na = int(np.asarray(s["pos"]).shape[0])
    assert 256 < na <= max_sites
    ctx = pbm.from_workload(w)
    prm = ctx.get_params()
    thole_a, eps_in = float(prm.thole_a), float(prm.eps_in)
    d = _device_sites(torch, s)
    rng = np.random.Generator(np.random.PCG64(11))
    mu = torch.from_numpy(0.05 * rng.normal(size=(na, 3))).cuda()

    # --- call 1: all parts, masked, potential + gradient + Hessian
    phi_r, grad_r, hess_r = ctx.multipole_field(mu, use_mask=True)
    phi = torch.full((na,), float("nan"), dtype=torch.float64, device="cuda")
    grad = torch.full((na, 3), float("nan"), dtype=torch.float64, device="cuda")
    hess = torch.full((na, 6), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    n_alloc = torch.cuda.memory_stats()["allocation.all.allocated"]
    held = torch.cuda.memory_allocated()
    pbm.multipole_field_static(d["pos"], d["q"], d["dip"], d["quad"], d["alpha"], d["group"], mu, thole_a, eps_in, True, phi, grad, hess)
    torch.cuda.synchronize()
    # nothing went through the allocator the library's other paths use (torch's caching allocator, via pb_set_allocator)
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == n_alloc and torch.cuda.memory_allocated() == held
    first = (phi.clone(), grad.clone(), hess.clone())
    for got, want in ((phi, phi_r), (grad, grad_r), (hess, hess_r)):
        assert bool(torch.isfinite(got).all())
        assert rel(got.cpu().numpy(), want.cpu().numpy()) <= TOL

    # --- call 2, directly after: fewer sites (other chunking: the array still holds call 1's sums), permanent multipoles
    #     only, unmasked, and the gradient alone (three of the ten columns are written and read)
    n2 = 301
    w2 = {k: np.ascontiguousarray(np.asarray(v)[:n2]) for k, v in s.items()}
    ctx2 = pbm.PB(0, **{k: getattr(prm, k) for k, _ in pbm.Params._fields_})
    ctx2.mesh_load(w.verts, w.tris)
    ctx2.sites_load(w2["pos"], w2["q"], w2["dip"], w2["quad"], w2["alpha"], w2["group"])
    _, grad2_r, _ = ctx2.multipole_field(None, use_mask=False)
    d2 = _device_sites(torch, s, n2)
    grad2 = torch.full((n2, 3), float("nan"), dtype=torch.float64, device="cuda")
    pbm.multipole_field_static(d2["pos"], d2["q"], d2["dip"], d2["quad"], d2["alpha"], d2["group"], None, thole_a, eps_in, False,
                               None, grad2, None)
    assert rel(grad2.cpu().numpy(), grad2_r.cpu().numpy()) <= TOL

    # --- call 3: call 1 again, now over call 2's leftovers: the same bits as the first time
    phi.fill_(float("nan")); grad.fill_(float("nan")); hess.fill_(float("nan"))
    pbm.multipole_field_static(d["pos"], d["q"], d["dip"], d["quad"], d["alpha"], d["group"], mu, thole_a, eps_in, True, phi, grad, hess)
    torch.cuda.synchronize()
    assert torch.equal(phi, first[0]) and torch.equal(grad, first[1]) and torch.equal(hess, first[2])
    assert rel(hess.cpu().numpy(), hess_r.cpu().numpy()) <= TOL

    # --- sizes beyond the maximum are refused with a clear message, nothing is launched
    nbig = max_sites + 1
    big = dict(pos=torch.rand(nbig, 3, dtype=torch.float64, device="cuda"), q=torch.zeros(nbig, dtype=torch.float64, device="cuda"),
               dip=torch.zeros(nbig, 3, dtype=torch.float64, device="cuda"), quad=torch.zeros(nbig, 6, dtype=torch.float64, device="cuda"),
               alpha=torch.zeros(nbig, dtype=torch.float64, device="cuda"), group=torch.zeros(nbig, dtype=torch.int32, device="cuda"))
    out = torch.zeros(nbig, 3, dtype=torch.float64, device="cuda")
    with pytest.raises(pbm.PBError) as e:
        pbm.multipole_field_static(big["pos"], big["q"], big["dip"], big["quad"], big["alpha"], big["group"], None, thole_a, eps_in,
                                   False, None, out, None)
    assert e.value.code == -1 and "4096" in str(e.value) and str(nbig) in str(e.value)
    assert float(out.abs().max()) == 0.0
    # exactly the maximum is accepted
    sub = {k: v[:max_sites].contiguous() for k, v in big.items()}
    out = torch.full((max_sites, 3), float("nan"), dtype=torch.float64, device="cuda")
    pbm.multipole_field_static(sub["pos"], sub["q"], sub["dip"], sub["quad"], sub["alpha"], sub["group"], None, thole_a, eps_in,
                               False, None, out, None)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all()) and float(out.abs().max()) == 0.0      # all multipoles zero: zero field
    ctx.close()
    ctx2.close()
