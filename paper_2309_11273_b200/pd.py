"""Thin Python binding over the C-ABI of include/pd.h (libpd.so): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch supplies device memory
(its caching allocator, through the pd_runtime callbacks) and the stream; nothing else.  There is
no CPU fallback: if libpd.so is missing or no CUDA device is present, this module raises.
Names mirror the header: Sim.create / step / get_u / get_v / get_damage / destroy (+ extensions).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.environ.get("PD_LIBPATH") or os.path.join(_HERE, "libpd.so")   # PD_LIBPATH: an alternative build (debugging)

PD_OK, PD_ERR_ARG, PD_ERR_ISOLATED, PD_ERR_ALLOC, PD_ERR_CUDA, PD_ERR_LIMIT = 0, -1, -2, -3, -4, -5
STATIC_MAX_DOUBLES = 1 << 20   # PD_STATIC_MAX_DOUBLES of include/pd.h: capacity of the static scratch of pd_get_u_static
EXPORTS = ["pd_create", "pd_step", "pd_get_u", "pd_get_v", "pd_get_damage", "pd_destroy", "pd_get_stats",
           "pd_get_bond_mask", "pd_get_node_fields", "pd_get_layout", "pd_step_timed", "pd_last_error", "pd_version",
           "pd_matrix_create", "pd_matrix_step", "pd_matrix_get", "pd_matrix_destroy", "pd_adr_step",
           "pd_gather_u", "pd_scatter_u", "pd_measure_fp64_rate", "pd_get_u_static",
           "pd_measure_pair_exchange"]


class PdMaterial(C.Structure):
    _fields_ = [("dim", C.c_int), ("mode", C.c_int), ("E", C.c_double), ("nu", C.c_double), ("rho", C.c_double),
                ("s_c", C.c_double), ("dt", C.c_double), ("ramp_time", C.c_double), ("extension", C.c_int)]


class PdBoundary(C.Structure):
    _fields_ = [("flags", C.c_void_p), ("value", C.c_void_p), ("precut", C.c_void_p), ("n_precut", C.c_int64),
                ("u0", C.c_void_p), ("v0", C.c_void_p)]


_ALLOC_T = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE_T = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class PdRuntime(C.Structure):
    _fields_ = [("alloc", _ALLOC_T), ("free", _FREE_T), ("ctx", C.c_void_p), ("stream", C.c_void_p)]


class PdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libpd error {code}: {msg}")
        self.code = code


_lib = None


def load():
    """dlopen libpd.so (built by paper_2309_11273_b200.build).  Raises if it is not there."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            raise ImportError(f"{_LIBPATH} not built: run `python -m paper_2309_11273_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(_LIBPATH)
        lib.pd_last_error.restype = C.c_char_p
        lib.pd_version.restype = C.c_char_p
        for name in EXPORTS:
            getattr(lib, name)  # AttributeError if a declared symbol is missing
        lib.pd_create.argtypes = [C.POINTER(C.c_void_p), C.c_int64, C.c_void_p, C.c_void_p, C.c_double,
                                  C.POINTER(PdMaterial), C.POINTER(PdBoundary), C.POINTER(PdRuntime)]
        lib.pd_step.argtypes = [C.c_void_p, C.c_int64]
        for name in ("pd_get_u", "pd_get_v", "pd_get_damage", "pd_get_u_static"):
            getattr(lib, name).argtypes = [C.c_void_p, C.c_void_p]
        lib.pd_destroy.argtypes = [C.c_void_p]
        lib.pd_get_stats.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        lib.pd_get_bond_mask.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.pd_get_node_fields.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        lib.pd_get_layout.argtypes = [C.c_void_p, C.c_void_p]
        lib.pd_step_timed.argtypes = [C.c_void_p, C.c_int64, C.c_void_p]
        lib.pd_matrix_create.argtypes = [C.POINTER(C.c_void_p), C.c_int64, C.c_void_p, C.c_void_p, C.POINTER(PdMaterial),
                                         C.POINTER(PdBoundary), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.pd_matrix_step.argtypes = [C.c_void_p, C.c_int64]
        lib.pd_adr_step.argtypes = [C.c_void_p, C.c_int64, C.c_double]
        lib.pd_gather_u.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        lib.pd_scatter_u.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        lib.pd_matrix_get.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.pd_matrix_destroy.argtypes = [C.c_void_p]
        _lib = lib
    return _lib


def measure_fp64_rate(reps: int = 5) -> float:
    """pd_measure_fp64_rate: FP64 fused multiply-adds per second the device sustains (8 independent chains per thread)."""
    lib = load()
    out = C.c_double(0.0)
    lib.pd_measure_fp64_rate.argtypes = [C.c_int, C.c_void_p, C.POINTER(C.c_double)]
    rc = lib.pd_measure_fp64_rate(int(reps), None, C.byref(out))
    if rc != 0:
        raise PdError(rc, lib.pd_last_error().decode())
    return float(out.value)


def measure_pair_exchange(reps: int = 5) -> dict:
    """pd_measure_pair_exchange: issue rates (per second, all threads) of FP64 FMAs, 64-bit lane shifts, groups of one lane
    shift + 5 dependent FMAs, and doubles through shared memory"""
    lib = load()
    out = (C.c_double * 4)()
    lib.pd_measure_pair_exchange.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
    rc = lib.pd_measure_pair_exchange(int(reps), None, C.addressof(out))
    if rc != 0:
        raise PdError(rc, lib.pd_last_error().decode())
    return dict(zip(("dfma_per_s", "shift64_per_s", "shift64_plus_5dfma_per_s", "smem_double_per_s"), map(float, out)))


def _ptr(a):
    """host numpy array, torch tensor (host or cuda) or None -> raw address"""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()  # torch tensor


class _TorchRuntime:
    """pd_runtime backed by torch's caching allocator and the stream that is current when the handle is created
    (the handle keeps that stream for its whole life: pd_runtime is read once, in pd_create)."""

    def __init__(self, device):
        import torch
        self.torch = torch
        self.device = device
        self.live = {}
        self.fail_allocs = False   # fault injection for the tests: every allocation fails (-> PD_ERR_ALLOC)
        self._alloc = _ALLOC_T(self._do_alloc)
        self._free = _FREE_T(self._do_free)
        self.struct = PdRuntime(self._alloc, self._free, None,
                                C.c_void_p(torch.cuda.current_stream(device).cuda_stream))

    def _do_alloc(self, nbytes, _ctx):
        if self.fail_allocs:
            return None
        try:
            t = self.torch.empty(max(int(nbytes), 1), dtype=self.torch.uint8, device=self.device)
        except Exception:  # out of memory -> NULL -> PD_ERR_ALLOC
            return None
        self.live[t.data_ptr()] = t
        return t.data_ptr()

    def _do_free(self, ptr, _ctx):
        self.live.pop(ptr, None)


class Sim:
    """One simulation handle (pd_sim*)."""

    def __init__(self, coords, volumes, horizon, *, dim, mode, E, nu, rho, dt, s_c=0.0, ramp_time=0.0, flags=None,
                 value=None, precut=None, u0=None, v0=None, device="cuda:0", use_torch_allocator=True,
                 extension="linearized"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: paper_2309_11273_b200 has no CPU path")
        self.lib = load()
        self.device = torch.device(device)
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        torch.cuda.set_device(self.device)
        self.dim = int(dim)
        keep = []

        def prep(a, dtype, shape=None):
            if a is None:
                return None
            if isinstance(a, np.ndarray) or not hasattr(a, "data_ptr"):
                a = np.ascontiguousarray(a, dtype=dtype)
                if shape is not None:
                    a = a.reshape(shape)
            else:
                assert a.is_contiguous()
            keep.append(a)
            return a

        coords = prep(coords, np.float64)
        self.n = int(coords.shape[0])
        volumes = prep(volumes, np.float64)
        flags = prep(flags, np.uint8)
        value = prep(value, np.float64)
        u0 = prep(u0, np.float64)
        v0 = prep(v0, np.float64)
        precut = prep(precut, np.int32)
        npre = 0 if precut is None else int(np.prod(precut.shape)) // 2
        mat = PdMaterial(dim, mode, E, nu, rho, s_c, dt, ramp_time, {"linearized": 0, "geometric": 1}[extension])
        bc = PdBoundary(_ptr(flags), _ptr(value), _ptr(precut) if npre else None, npre, _ptr(u0), _ptr(v0))
        self._rt = _TorchRuntime(self.device) if use_torch_allocator else None
        h = C.c_void_p()
        rc = self.lib.pd_create(C.byref(h), self.n, _ptr(coords), _ptr(volumes), float(horizon), C.byref(mat),
                                C.byref(bc), C.byref(self._rt.struct) if self._rt else None)
        if rc != PD_OK:
            raise PdError(rc, self.lib.pd_last_error().decode())
        self.h = h

    @classmethod
    def create(cls, *a, **kw):
        return cls(*a, **kw)

    @classmethod
    def from_workload(cls, wl, **kw):
        return cls(wl.coords, wl.volumes, wl.horizon, **wl.material_kwargs(), flags=wl.flags, value=wl.value,
                   precut=wl.precut, u0=wl.u0, v0=wl.v0, **kw)

    def _ck(self, rc):
        if rc != PD_OK:
            raise PdError(rc, self.lib.pd_last_error().decode())

    def step(self, nsteps=1):
        self._ck(self.lib.pd_step(self.h, int(nsteps)))

    def step_timed(self, nsteps=1):
        """(ms in the dilatation kernel, ms in the force+update kernel), summed over nsteps"""
        ms = (C.c_double * 2)()
        self._ck(self.lib.pd_step_timed(self.h, int(nsteps), C.addressof(ms)))
        return float(ms[0]), float(ms[1])

    def _get(self, fn, shape, out):
        if out is None:
            out = np.empty(shape, dtype=np.float64)
        else:   # the library writes prod(shape) doubles through the raw pointer: refuse anything else
            n = int(np.prod(shape))
            if isinstance(out, np.ndarray):
                ok = out.dtype == np.float64 and out.flags["C_CONTIGUOUS"] and out.size == n
            else:   # torch tensor: host, or on this handle's device
                import torch
                ok = (out.dtype == torch.float64 and out.is_contiguous() and out.numel() == n and
                      (not out.is_cuda or out.device == self.device))
            if not ok:
                raise ValueError(f"out must be a contiguous float64 array of {n} elements on the host or on {self.device}")
        self._ck(fn(self.h, _ptr(out)))
        return out

    def _dev_idx(self, idx):
        """device copy (int32) of an index list, cached per list object"""
        import torch
        cache = self.__dict__.setdefault("_idx_cache", {})
        key = id(idx)
        if key not in cache:
            cache[key] = (idx, torch.as_tensor(np.ascontiguousarray(idx, dtype=np.int32), device=self.device))
        return cache[key][1]

    def gather_u(self, idx):
        """rows idx (user indices) of u^n as a (len(idx), dim) float64 tensor on the handle's device (pd_gather_u)"""
        import torch
        di = self._dev_idx(idx)
        out = torch.empty((di.numel(), self.dim), dtype=torch.float64, device=self.device)
        self._ck(self.lib.pd_gather_u(self.h, di.data_ptr(), di.numel(), out.data_ptr()))
        return out

    def scatter_u(self, idx, values):
        """overwrite rows idx of u^n with values ((len(idx), dim), tensor on the device or array) (pd_scatter_u)"""
        import torch
        di = self._dev_idx(idx)
        v = torch.as_tensor(values, dtype=torch.float64, device=self.device).contiguous()
        assert v.numel() == di.numel() * self.dim
        self._ck(self.lib.pd_scatter_u(self.h, di.data_ptr(), di.numel(), v.data_ptr()))

    def adr_step(self, niter, lam):
        """niter iterations of adaptive dynamic relaxation (pd_adr_step); the handle must have rho = 1, dt = 1"""
        self._ck(self.lib.pd_adr_step(self.h, int(niter), float(lam)))

    def get_u(self, out=None):
        return self._get(self.lib.pd_get_u, (self.n, self.dim), out)

    def get_u_static(self, out=None):
        """pd_get_u_static: get_u through the library's static device scratch (no device allocation; dim*n <= STATIC_MAX_DOUBLES)"""
        return self._get(self.lib.pd_get_u_static, (self.n, self.dim), out)

    def get_v(self, out=None):
        return self._get(self.lib.pd_get_v, (self.n, self.dim), out)

    def get_damage(self, out=None):
        return self._get(self.lib.pd_get_damage, (self.n,), out)

    def get_stats(self):
        z, nb, ng, st = C.c_int64(), C.c_int64(), C.c_int64(), C.c_int64()
        md = C.c_double()
        self._ck(self.lib.pd_get_stats(self.h, C.addressof(z), C.addressof(nb), C.addressof(md), C.addressof(ng),
                                       C.addressof(st)))
        return dict(n_directed_bonds=z.value, n_broken_directed=nb.value, max_damage=md.value,
                    n_nodes_damage_ge_half=ng.value, step=st.value)

    def get_bond_mask(self, rows_only=False):
        rowptr = np.empty(self.n + 1, dtype=np.int64)
        if rows_only:
            self._ck(self.lib.pd_get_bond_mask(self.h, _ptr(rowptr), None, None))
            return rowptr
        self._ck(self.lib.pd_get_bond_mask(self.h, _ptr(rowptr), None, None))
        z = int(rowptr[-1])
        col = np.empty(z, dtype=np.int32)
        intact = np.empty(z, dtype=np.uint8)
        self._ck(self.lib.pd_get_bond_mask(self.h, _ptr(rowptr), _ptr(col), _ptr(intact)))
        return rowptr, col, intact

    def get_node_fields(self, want_m=True, want_theta=True):
        m = np.empty(self.n) if want_m else None
        th = np.empty(self.n) if want_theta else None
        self._ck(self.lib.pd_get_node_fields(self.h, _ptr(m), _ptr(th)))
        return m, th

    def get_layout(self):
        c = (C.c_int64 * 8)()
        self._ck(self.lib.pd_get_layout(self.h, C.addressof(c)))
        keys = ["n", "n_padded", "n_directed_bonds", "stored_slots", "step_launches", "device_bytes",
                "uniform_volume", "layout"]
        return dict(zip(keys, [int(x) for x in c]))

    def destroy(self):
        if getattr(self, "h", None):
            self.lib.pd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class MatrixScheme:
    """The paper's own 4-SpMV scheme (pd_matrix_* of include/pd.h) on the family of an existing Sim: the on-box
    comparison for the matrix-free path (no fracture).  Argument marshalling only."""

    def __init__(self, sim, coords, volumes, *, dim, mode, E, nu, rho, dt, s_c=0.0, ramp_time=0.0, flags=None, value=None,
                 u0=None, v0=None, **_ignored):
        import torch
        self.lib, self.n, self.dim = sim.lib, sim.n, int(dim)
        rowptr, col, _ = sim.get_bond_mask()
        m, _ = sim.get_node_fields(want_theta=False)
        keep = [np.ascontiguousarray(coords, np.float64), np.ascontiguousarray(volumes, np.float64), rowptr, col, m]
        opt = [None if a is None else np.ascontiguousarray(a, dt_) for a, dt_ in
               ((flags, np.uint8), (value, np.float64), (u0, np.float64), (v0, np.float64))]
        mat = PdMaterial(dim, mode, E, nu, rho, 0.0, dt, ramp_time, 0)
        bc = PdBoundary(_ptr(opt[0]), _ptr(opt[1]), None, 0, _ptr(opt[2]), _ptr(opt[3]))
        h = C.c_void_p()
        stream = C.c_void_p(torch.cuda.current_stream(sim.device).cuda_stream)
        rc = self.lib.pd_matrix_create(C.byref(h), self.n, _ptr(keep[0]), _ptr(keep[1]), C.byref(mat), C.byref(bc),
                                       _ptr(rowptr), _ptr(col), _ptr(m), stream)
        if rc != PD_OK:
            raise PdError(rc, self.lib.pd_last_error().decode())
        self.h = h

    @classmethod
    def from_workload(cls, sim, wl):
        return cls(sim, wl.coords, wl.volumes, **wl.material_kwargs(), flags=wl.flags, value=wl.value, u0=wl.u0, v0=wl.v0)

    def step(self, nsteps=1):
        rc = self.lib.pd_matrix_step(self.h, int(nsteps))
        if rc != PD_OK:
            raise PdError(rc, self.lib.pd_last_error().decode())

    def get(self):
        """(u, v, info) with info = dict(n, n_bonds, nnz_CE, nnz_CTH, nnz_KTH, nnz_KE, matrix_bytes, step)"""
        u, v = np.empty((self.n, self.dim)), np.empty((self.n, self.dim))
        info = (C.c_int64 * 8)()
        rc = self.lib.pd_matrix_get(self.h, _ptr(u), _ptr(v), C.addressof(info))
        if rc != PD_OK:
            raise PdError(rc, self.lib.pd_last_error().decode())
        keys = ["n", "n_bonds", "nnz_CE", "nnz_CTH", "nnz_KTH", "nnz_KE", "matrix_bytes", "step"]
        return u, v, dict(zip(keys, [int(x) for x in info]))

    def destroy(self):
        if getattr(self, "h", None):
            self.lib.pd_matrix_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
