"""Thin ctypes binding over the C-ABI library of include/pb.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of `csrc/`; PyTorch is used for device
memory (the library's allocator callback hands out torch tensors) and streams.  There is
no CPU fallback: if the shared library is missing, or no CUDA device is present, the
calls raise.  This module never imports anything under `oracle/`.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libpb_b200.so")
SOURCES = ["pb_api.cu", "pb_tree.cu", "pb_near.cu", "pb_matvec.cu", "pb_sites.cu", "pb_sitetree.cu", "pb_rhstree.cu", "pb_solve.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]

PB_OK = 0
PB_ERR_NO_CONVERGENCE = -6

EXPORTS = [
    "pb_create", "pb_destroy", "pb_last_error", "pb_set_allocator", "pb_default_params", "pb_set_params",
    "pb_get_params", "pb_mesh_load", "pb_sites_load", "pb_tree_build", "pb_rhs_multipole", "pb_matvec",
    "pb_matvec_timed", "pb_matvec_host", "pb_reaction_field", "pb_multipole_field", "pb_gmres", "pb_solve",
    "pb_solve_host", "pb_get_stats", "pb_fp64_peak_probe", "pb_set_profiling", "pb_quadrature_rule",
    "pb_gauss_legendre", "pb_farfield_table", "pb_binding_cycle", "pb_set_shard", "pb_get_shard", "pb_shard_partition", "pb_set_stern", "pb_fp64_pipe_probe",
    "pb_multipole_field_static", "pb_multipole_field_static_limit", "pb_static_last_error",
]


class PBError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"pb error {code}: {msg}")
        self.code = code


class Params(ctypes.Structure):
    _fields_ = [
        ("eps_in", ctypes.c_double), ("eps_out", ctypes.c_double), ("kappa", ctypes.c_double),
        ("theta", ctypes.c_double), ("order_P", ctypes.c_int32), ("ncrit", ctypes.c_int32),
        ("K_far", ctypes.c_int32), ("K_near", ctypes.c_int32), ("near_tau", ctypes.c_double),
        ("nq_edge", ctypes.c_int32), ("precond", ctypes.c_int32), ("gmres_tol", ctypes.c_double),
        ("gmres_restart", ctypes.c_int32), ("gmres_maxit", ctypes.c_int32), ("scf_tol_debye", ctypes.c_double),
        ("scf_omega", ctypes.c_double), ("scf_maxit", ctypes.c_int32), ("site_treecode", ctypes.c_int32),
        ("thole_a", ctypes.c_double), ("rhs_treecode", ctypes.c_int32), ("scf_recycle", ctypes.c_int32),
        ("list_split", ctypes.c_int32), ("scf_eta", ctypes.c_double),
        ("scf_store_mb", ctypes.c_int32),
    ]


class Result(ctypes.Structure):
    _fields_ = [
        ("dG_solv", ctypes.c_double), ("G_solvterm", ctypes.c_double), ("G_mult_diss", ctypes.c_double),
        ("G_vac", ctypes.c_double), ("final_scf_delta_debye", ctypes.c_double),
        ("final_gmres_relres", ctypes.c_double), ("scf_iters", ctypes.c_int32), ("scf_iters_vac", ctypes.c_int32),
        ("gmres_iters_total", ctypes.c_int32), ("matvecs_total", ctypes.c_int32), ("status", ctypes.c_int32),
        ("reserved", ctypes.c_int32),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


class Binding(ctypes.Structure):
    _fields_ = [("dG_bind_vac", ctypes.c_double), ("ddG_bind", ctypes.c_double), ("dG_bind_diss", ctypes.c_double)]


class Stats(ctypes.Structure):
    _fields_ = [
        ("n_panels", ctypes.c_int64), ("n_sources", ctypes.c_int64), ("n_sites", ctypes.c_int64),
        ("n_cells", ctypes.c_int64), ("n_leaves", ctypes.c_int64), ("n_levels", ctypes.c_int64),
        ("n_groups", ctypes.c_int64), ("p2p_pairs", ctypes.c_int64), ("m2p_pairs", ctypes.c_int64),
        ("near_entries", ctypes.c_int64), ("n_terms", ctypes.c_int64), ("matvec_calls", ctypes.c_int64),
        ("device_bytes", ctypes.c_int64), ("kernel_launches", ctypes.c_int64),
        ("prof_p2p_launches", ctypes.c_int64), ("prof_m2p_launches", ctypes.c_int64),
        ("prof_p2p_ms", ctypes.c_double), ("prof_m2p_ms", ctypes.c_double),
        ("last_matvec_ms", ctypes.c_double * 8),
        ("ncrit_used", ctypes.c_int64), ("m2p_pairs_low", ctypes.c_int64),
        ("covered_pairs", ctypes.c_int64), ("site_p2p_pairs", ctypes.c_int64), ("site_m2p_pairs", ctypes.c_int64),
        ("site_covered_pairs", ctypes.c_int64), ("rhs_p2p_pairs", ctypes.c_int64), ("rhs_m2p_pairs", ctypes.c_int64),
        ("rhs_covered_pairs", ctypes.c_int64), ("p2p_pairs_half", ctypes.c_int64), ("m2p_pairs_half", ctypes.c_int64),
        ("m2p_pairs_mid", ctypes.c_int64),
    ]

    def as_dict(self):
        d = {k: getattr(self, k) for k, _ in self._fields_ if k != "last_matvec_ms"}
        ms = list(self.last_matvec_ms)
        d["last_matvec_ms"] = dict(weights=ms[0], p2m_m2m=ms[1], m2p=ms[2], p2p=ms[3], near_combine=ms[4], total=ms[5])
        return d


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu for sm_100a into libpb_b200.so next to this file (nvcc cross-compiles
    without a GPU).  One object per source, compiled in parallel and only when the source or a header
    is newer than the object; the objects live in build/ (git-ignored)."""
    import glob
    from concurrent.futures import ThreadPoolExecutor
    srcs = [os.path.join(_CSRC, s) for s in SOURCES]
    hdrs = sorted(glob.glob(os.path.join(_CSRC, "*.cuh"))) + [os.path.join(_HERE, "..", "include", "pb.h")]
    deps = srcs + hdrs
    if not force and os.path.exists(LIB_PATH) and all(os.path.getmtime(LIB_PATH) >= os.path.getmtime(d) for d in deps):
        return LIB_PATH
    bdir = os.path.join(_HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    hnew = max(os.path.getmtime(h) for h in hdrs)
    cflags = [f for f in NVCC_FLAGS if f != "-shared"] + (["-Xptxas", "-v"] if verbose else [])
    cflags += os.environ.get("PB_NVCC_EXTRA", "").split()          # experiments: extra -D switches

    def compile_one(src):
        obj = os.path.join(bdir, os.path.basename(src)[:-3] + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hnew):
            subprocess.check_call(["nvcc"] + cflags + ["-c", "-o", obj, src])
        return obj

    with ThreadPoolExecutor(max_workers=min(len(srcs), os.cpu_count() or 1)) as ex:
        objs = list(ex.map(compile_one, srcs))
    subprocess.check_call(["nvcc"] + NVCC_FLAGS + ["-o", LIB_PATH] + objs)
    return LIB_PATH


_lib = None
_ALLOC_T = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t)
_FREE_T = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)
_GATHER_T = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t)


def lib():
    """Load the shared library (fails loudly if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PBError(-100, f"{LIB_PATH} is missing: run __graft_entry__.build() (nvcc, sm_100a). "
                                "There is no CPU fallback.")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, i32, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double
        L.pb_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, vp]
        L.pb_destroy.argtypes = [vp]
        L.pb_last_error.argtypes = [vp]
        L.pb_last_error.restype = ctypes.c_char_p
        L.pb_set_allocator.argtypes = [vp, _ALLOC_T, _FREE_T, vp]
        L.pb_default_params.argtypes = [ctypes.POINTER(Params)]
        L.pb_default_params.restype = None
        L.pb_set_params.argtypes = [vp, ctypes.POINTER(Params)]
        L.pb_get_params.argtypes = [vp, ctypes.POINTER(Params)]
        L.pb_mesh_load.argtypes = [vp, vp, i64, vp, i64]
        L.pb_sites_load.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp]
        L.pb_tree_build.argtypes = [vp]
        L.pb_rhs_multipole.argtypes = [vp, vp, vp]
        L.pb_matvec.argtypes = [vp, vp, vp]
        L.pb_matvec_timed.argtypes = [vp, vp, vp]
        L.pb_matvec_host.argtypes = [vp, vp, vp]
        L.pb_reaction_field.argtypes = [vp, vp, vp, vp, vp]
        L.pb_multipole_field.argtypes = [vp, vp, ctypes.c_int, vp, vp, vp]
        L.pb_gmres.argtypes = [vp, vp, vp, ctypes.POINTER(i32), ctypes.POINTER(dbl)]
        L.pb_solve.argtypes = [vp, vp, vp, ctypes.POINTER(Result)]
        L.pb_solve_host.argtypes = [vp, vp, vp, ctypes.POINTER(Result)]
        L.pb_get_stats.argtypes = [vp, ctypes.POINTER(Stats)]
        L.pb_fp64_peak_probe.argtypes = [vp, ctypes.POINTER(dbl)]
        L.pb_set_profiling.argtypes = [vp, ctypes.c_int]
        L.pb_fp64_pipe_probe.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(dbl)]
        L.pb_quadrature_rule.argtypes = [ctypes.c_int, vp, vp]
        L.pb_gauss_legendre.argtypes = [ctypes.c_int, vp, vp]
        L.pb_farfield_table.argtypes = [ctypes.c_int, vp, vp, vp, vp, ctypes.POINTER(i64)]
        L.pb_binding_cycle.argtypes = [ctypes.POINTER(Result)] * 3 + [ctypes.POINTER(Binding)]
        L.pb_set_stern.argtypes = [vp, i64, dbl]
        L.pb_set_shard.argtypes = [vp, ctypes.c_int, ctypes.c_int, _GATHER_T, vp]
        L.pb_get_shard.argtypes = [vp, ctypes.POINTER(i64)]
        L.pb_shard_partition.argtypes = [ctypes.POINTER(i64), i64, ctypes.c_int, ctypes.POINTER(i64)]
        L.pb_multipole_field_static.argtypes = [ctypes.c_int, vp, i64, vp, vp, vp, vp, vp, vp, vp, dbl, dbl, ctypes.c_int, vp, vp, vp]
        L.pb_multipole_field_static_limit.argtypes = [ctypes.POINTER(i64), ctypes.POINTER(i64)]
        L.pb_static_last_error.argtypes = []
        L.pb_static_last_error.restype = ctypes.c_char_p
        for name in EXPORTS:
            if name not in ("pb_last_error", "pb_default_params", "pb_static_last_error"):
                getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


def multipole_field_static_limit():
    """(max sites, bytes of the static scratch array) of `multipole_field_static`."""
    a, b = ctypes.c_int64(0), ctypes.c_int64(0)
    lib().pb_multipole_field_static_limit(ctypes.byref(a), ctypes.byref(b))
    return int(a.value), int(b.value)


def multipole_field_static(pos, q, dip, quad, alpha, group, mu, thole_a, eps_in, use_mask, phi, grad, hess, stream=None):
    """pb_multipole_field_static: the multipole field with no allocation.  Every array is the caller's CUDA tensor
    (float64, group int32, contiguous); outputs are written in place (None = not wanted); runs on torch's current stream
    unless `stream` is given.  Argument marshalling only: nothing is created here."""
    import torch
    na = int(pos.shape[0])
    for t, dt in ((pos, torch.float64), (q, torch.float64), (dip, torch.float64), (quad, torch.float64), (alpha, torch.float64),
                  (group, torch.int32), (mu, torch.float64), (phi, torch.float64), (grad, torch.float64), (hess, torch.float64)):
        if t is not None and not (t.is_cuda and t.dtype == dt and t.is_contiguous() and t.device == pos.device):
            raise PBError(-1, "multipole_field_static: arrays must be contiguous CUDA tensors of one device (float64; group int32)")
    st = (stream if stream is not None else torch.cuda.current_stream(pos.device)).cuda_stream
    rc = lib().pb_multipole_field_static(pos.device.index, ctypes.c_void_p(st), na, _ptr(pos), _ptr(q), _ptr(dip), _ptr(quad),
                                         _ptr(alpha), _ptr(group), _ptr(mu), float(thole_a), float(eps_in), 1 if use_mask else 0,
                                         _ptr(phi), _ptr(grad), _ptr(hess))
    if rc != 0:
        raise PBError(rc, lib().pb_static_last_error().decode())


def binding_cycle(res_ab: dict, res_a: dict, res_b: dict) -> dict:
    """Eq. (25)-(27) from the result dicts of three `PB.solve()` calls (complex, A, B)."""
    rs = []
    for r in (res_ab, res_a, res_b):
        c = Result()
        for k, _ in Result._fields_:
            if k in r:
                setattr(c, k, r[k])
        rs.append(c)
    out = Binding()
    rc = lib().pb_binding_cycle(ctypes.byref(rs[0]), ctypes.byref(rs[1]), ctypes.byref(rs[2]), ctypes.byref(out))
    if rc not in (PB_OK, PB_ERR_NO_CONVERGENCE):
        raise PBError(rc, "pb_binding_cycle")
    return dict(dG_bind_vac=out.dG_bind_vac, ddG_bind=out.ddG_bind, dG_bind_diss=out.dG_bind_diss, converged=rc == PB_OK)


def shard_partition(cost, world: int):
    """The library's partition rule (host-only call): first [world + 1] group boundaries for per-group costs."""
    import numpy as np
    cost = np.ascontiguousarray(cost, dtype=np.int64)
    first = np.zeros(world + 1, dtype=np.int64)
    i64p = ctypes.POINTER(ctypes.c_int64)
    rc = lib().pb_shard_partition(cost.ctypes.data_as(i64p), cost.size, world, first.ctypes.data_as(i64p))
    if rc != PB_OK:
        raise PBError(rc, "pb_shard_partition")
    return first


def default_params() -> Params:
    p = Params()
    lib().pb_default_params(ctypes.byref(p))
    return p


def quadrature_rule(K: int):
    """The library's own K-point triangle rule (host-only call): (lam [K][3], w [K])."""
    import numpy as np
    lam = np.zeros((K, 3))
    w = np.zeros(K)
    rc = lib().pb_quadrature_rule(K, lam.ctypes.data, w.ctypes.data)
    if rc != PB_OK:
        raise PBError(rc, f"no {K}-point rule")
    return lam, w


def gauss_legendre(n: int):
    import numpy as np
    x = np.zeros(n)
    w = np.zeros(n)
    rc = lib().pb_gauss_legendre(n, x.ctypes.data, w.ctypes.data)
    if rc != PB_OK:
        raise PBError(rc, "pb_gauss_legendre")
    return x, w


def farfield_table(P: int):
    """The library's M -> F conversion table for order P (host-only call):
    (expo [NT][4] = a,b,c,j ; off [NT+1] ; idx ; coef)."""
    import numpy as np
    nnz = ctypes.c_int64(0)
    nt = lib().pb_farfield_table(P, None, None, None, None, ctypes.byref(nnz))
    if nt < 0:
        raise PBError(nt, "pb_farfield_table")
    expo = np.zeros((nt, 4), dtype=np.int32)
    off = np.zeros(nt + 1, dtype=np.int32)
    idx = np.zeros(nnz.value, dtype=np.int32)
    coef = np.zeros(nnz.value)
    lib().pb_farfield_table(P, expo.ctypes.data, off.ctypes.data, idx.ctypes.data, coef.ctypes.data, ctypes.byref(nnz))
    return expo, off, idx, coef


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


class PB:
    """One solver context on one GPU.  Tensors are torch CUDA tensors (fp64 / int32)."""

    def __init__(self, device: int = 0, **params):
        import torch
        if not torch.cuda.is_available():
            raise PBError(-101, "no CUDA device: the B200 path has no CPU fallback")
        self.torch = torch
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self._L = lib()
        self._h = ctypes.c_void_p()
        stream = torch.cuda.current_stream(self.device).cuda_stream
        rc = self._L.pb_create(ctypes.byref(self._h), device, ctypes.c_void_p(stream))
        if rc != PB_OK:
            raise PBError(rc, "pb_create failed (no usable CUDA device?)")
        self._bufs = {}

        def _alloc(_user, nbytes):
            t = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
            p = t.data_ptr()
            self._bufs[p] = t
            return p

        def _free(_user, p):
            self._bufs.pop(p, None)

        self._alloc_cb = _ALLOC_T(_alloc)
        self._free_cb = _FREE_T(_free)
        self._ck(self._L.pb_set_allocator(self._h, self._alloc_cb, self._free_cb, None))
        self.nt = 0
        self.na = 0
        if params:
            self.set_params(**params)

    # -- plumbing -----------------------------------------------------------------------------------
    def _ck(self, rc, allow=()):
        if rc != PB_OK and rc not in allow:
            raise PBError(rc, self._L.pb_last_error(self._h).decode())
        return rc

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.pb_destroy(self._h)
            self._h = ctypes.c_void_p()
            self._bufs.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev(self, a, dtype):
        torch = self.torch
        t = torch.as_tensor(a, dtype=dtype)
        return t.to(self.device).contiguous()

    # -- parameters ---------------------------------------------------------------------------------
    def get_params(self) -> Params:
        p = Params()
        self._ck(self._L.pb_get_params(self._h, ctypes.byref(p)))
        return p

    def set_params(self, **kw):
        p = self.get_params()
        names = {k for k, _ in Params._fields_}
        for k, v in kw.items():
            if k not in names:
                raise KeyError(f"unknown parameter {k}")
            setattr(p, k, v)
        self._ck(self._L.pb_set_params(self._h, ctypes.byref(p)))

    # -- inputs -------------------------------------------------------------------------------------
    def mesh_load(self, verts, tris):
        torch = self.torch
        v = self._dev(verts, torch.float64).reshape(-1, 3)
        t = self._dev(tris, torch.int32).reshape(-1, 3)
        self._ck(self._L.pb_mesh_load(self._h, _ptr(v), v.shape[0], _ptr(t), t.shape[0]))
        self.nt = int(t.shape[0])

    def sites_load(self, pos, q, dip, quad, alpha, group):
        torch = self.torch
        pos = self._dev(pos, torch.float64).reshape(-1, 3)
        na = pos.shape[0]
        q = self._dev(q, torch.float64).reshape(na)
        dip = self._dev(dip, torch.float64).reshape(na, 3)
        quad = self._dev(quad, torch.float64).reshape(na, 6)
        alpha = self._dev(alpha, torch.float64).reshape(na)
        group = self._dev(group, torch.int32).reshape(na)
        self._ck(self._L.pb_sites_load(self._h, na, _ptr(pos), _ptr(q), _ptr(dip), _ptr(quad), _ptr(alpha), _ptr(group)))
        torch.cuda.current_stream(self.device).synchronize()   # inputs may be freed by the caller
        self.na = int(na)

    def set_stern(self, n_inner: int, eps_stern: float):
        """Panels [0, n_inner) of the loaded (union) mesh are Gamma_1, the rest Gamma_2; see include/pb.h."""
        self._ck(self._L.pb_set_stern(self._h, int(n_inner), float(eps_stern)))

    def tree_build(self):
        self._ck(self._L.pb_tree_build(self._h))

    # -- multi-GPU target sharding ------------------------------------------------------------------
    def set_shard(self, rank: int, world: int, group=None, exchange: bool = True, gather=None):
        """This context evaluates rank's share of the target groups (call before tree_build).  With `exchange` the
        owned rows of y are all-gathered over torch.distributed's `group` (NCCL) inside every matvec, so y is complete
        on every rank; without it only the owned rows of y are written.  `gather(send, recv)` replaces the
        collective (tests: send is a float64 tensor of 2 * nmax values, recv of world times as many)."""
        self._shard = (rank, world)
        if world > 1 and exchange:
            torch = self.torch
            if gather is None:
                import torch.distributed as dist

                def gather(s, r):
                    dist.all_gather_into_tensor(r, s, group=group)     # enqueued on the current (= the context's) stream

            def _gather(_user, send, recv, nbytes):
                try:
                    s = self._bufs[send][:nbytes].view(torch.float64)
                    r = self._bufs[recv][:nbytes * world].view(torch.float64)
                    gather(s, r)
                    return 0
                except Exception:                                      # never let an exception cross the C boundary
                    import traceback
                    traceback.print_exc()
                    return 1

            self._gather_cb = _GATHER_T(_gather)
        else:
            self._gather_cb = _GATHER_T()                              # NULL
        self._ck(self._L.pb_set_shard(self._h, rank, world, self._gather_cb, None))

    def shard_ranges(self):
        """first [world + 1]: first owned panel (Morton order) of every rank, after tree_build."""
        import numpy as np
        world = getattr(self, "_shard", (0, 1))[1]
        first = np.zeros(world + 1, dtype=np.int64)
        self._ck(self._L.pb_get_shard(self._h, first.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))))
        return first

    # -- operators ----------------------------------------------------------------------------------
    def rhs_multipole(self, mu=None):
        torch = self.torch
        b = torch.empty(2 * self.nt, dtype=torch.float64, device=self.device)
        mu_t = None if mu is None else self._dev(mu, torch.float64).reshape(self.na, 3)
        self._ck(self._L.pb_rhs_multipole(self._h, _ptr(mu_t), _ptr(b)))
        return b

    def matvec(self, x, out=None, timed=False):
        torch = self.torch
        x = self._dev(x, torch.float64).reshape(2 * self.nt)
        y = out if out is not None else torch.empty_like(x)
        fn = self._L.pb_matvec_timed if timed else self._L.pb_matvec
        self._ck(fn(self._h, _ptr(x), _ptr(y)))
        return y

    def matvec_host(self, x_host, y_host):
        """x_host, y_host: pinned or pageable CPU torch tensors / numpy arrays of 2*nt float64."""
        xp = x_host.data_ptr() if hasattr(x_host, "data_ptr") else x_host.ctypes.data
        yp = y_host.data_ptr() if hasattr(y_host, "data_ptr") else y_host.ctypes.data
        self._ck(self._L.pb_matvec_host(self._h, ctypes.c_void_p(xp), ctypes.c_void_p(yp)))
        return y_host

    def reaction_field(self, x, want_hess=True):
        torch = self.torch
        x = self._dev(x, torch.float64).reshape(2 * self.nt)
        phi = torch.empty(self.na, dtype=torch.float64, device=self.device)
        grad = torch.empty(self.na, 3, dtype=torch.float64, device=self.device)
        hess = torch.empty(self.na, 6, dtype=torch.float64, device=self.device) if want_hess else None
        self._ck(self._L.pb_reaction_field(self._h, _ptr(x), _ptr(phi), _ptr(grad), _ptr(hess)))
        return phi, grad, hess

    def multipole_field(self, mu=None, use_mask=True):
        torch = self.torch
        mu_t = None if mu is None else self._dev(mu, torch.float64).reshape(self.na, 3)
        phi = torch.empty(self.na, dtype=torch.float64, device=self.device)
        grad = torch.empty(self.na, 3, dtype=torch.float64, device=self.device)
        hess = torch.empty(self.na, 6, dtype=torch.float64, device=self.device)
        self._ck(self._L.pb_multipole_field(self._h, _ptr(mu_t), 1 if use_mask else 0, _ptr(phi), _ptr(grad), _ptr(hess)))
        return phi, grad, hess

    # -- solvers ------------------------------------------------------------------------------------
    def gmres(self, b, x0=None):
        torch = self.torch
        b = self._dev(b, torch.float64).reshape(2 * self.nt)
        x = torch.zeros_like(b) if x0 is None else self._dev(x0, torch.float64).clone()
        it = ctypes.c_int32(0)
        rr = ctypes.c_double(0.0)
        rc = self._ck(self._L.pb_gmres(self._h, _ptr(b), _ptr(x), ctypes.byref(it), ctypes.byref(rr)),
                      allow=(PB_ERR_NO_CONVERGENCE,))
        return x, dict(iters=it.value, relres=rr.value, converged=rc == PB_OK)

    def solve(self):
        torch = self.torch
        x = torch.empty(2 * self.nt, dtype=torch.float64, device=self.device)
        mu = torch.empty(self.na, 3, dtype=torch.float64, device=self.device)
        res = Result()
        self._ck(self._L.pb_solve(self._h, _ptr(x), _ptr(mu), ctypes.byref(res)), allow=(PB_ERR_NO_CONVERGENCE,))
        return x, mu, res.as_dict()

    def solve_host(self, x_host=None, mu_host=None):
        res = Result()
        xp = None if x_host is None else ctypes.c_void_p(x_host.data_ptr())
        mp = None if mu_host is None else ctypes.c_void_p(mu_host.data_ptr())
        self._ck(self._L.pb_solve_host(self._h, xp, mp, ctypes.byref(res)), allow=(PB_ERR_NO_CONVERGENCE,))
        return res.as_dict()

    def stats(self) -> dict:
        s = Stats()
        self._ck(self._L.pb_get_stats(self._h, ctypes.byref(s)))
        return s.as_dict()

    def set_profiling(self, on: bool):
        self._ck(self._L.pb_set_profiling(self._h, 1 if on else 0))

    def fp64_peak_probe(self) -> float:
        v = ctypes.c_double(0.0)
        self._ck(self._L.pb_fp64_peak_probe(self._h, ctypes.byref(v)))
        return v.value


def fp64_pipe_table(device: int = 0):
    """The FP64 pipe probe over resident warps, ILP and mixed-in integer instructions (profiles/r02_fp64_pipe_probes.md):
    rows of (warps_per_sm, ilp, other_per_8, kind, percent of the DFMA issue peak)."""
    ctx = PB(device)
    rows = []
    try:
        for wps in (4, 8, 16, 32, 64):
            for ilp in (1, 2, 4, 8):
                v = ctypes.c_double(0.0)
                ctx._ck(ctx._L.pb_fp64_pipe_probe(ctx._h, wps, ilp, 0, 0, ctypes.byref(v)))
                rows.append((wps, ilp, 0, "-", v.value))
        for kind, name in ((0, "IMAD"), (1, "LOP3")):
            for ni in (2, 4, 8):
                v = ctypes.c_double(0.0)
                ctx._ck(ctx._L.pb_fp64_pipe_probe(ctx._h, 16, 8, ni, kind, ctypes.byref(v)))
                rows.append((16, 8, ni, name, v.value))
        v = ctypes.c_double(0.0)
        ctx._ck(ctx._L.pb_fp64_pipe_probe(ctx._h, 16, 8, 0, 2, ctypes.byref(v)))
        rows.append((16, 8, 0, "3 distinct register operands", v.value))
    finally:
        ctx.close()
    return rows


def from_workload(w, device: int = 0, **overrides) -> PB:
    """Context loaded with a `workloads.Workload` (mesh, sites, parameters); tree not yet built."""
    names = {k for k, _ in Params._fields_}
    prm = {k: v for k, v in w.params.items() if k in names}
    prm.update(overrides)
    pb = PB(device, **prm)
    pb.mesh_load(w.verts, w.tris)
    s = w.sites
    pb.sites_load(s["pos"], s["q"], s["dip"], s["quad"], s["alpha"], s["group"])
    return pb
