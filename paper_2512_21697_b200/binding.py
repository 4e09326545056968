"""Thin ctypes binding over libtdde.so (include/tdde.h).  Argument marshalling only: every step of the hot path
runs in the library's CUDA kernels.  torch is used for device memory and streams, nothing else.

The names mirror the C ABI: ``Tdde.step / propagate / norm / apply / precond`` call ``tdde_step`` etc.
There is no CPU fallback: importing works without a GPU (so that the ABI can be inspected), but creating a
propagator without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("TDDE_LIB_PATH", os.path.join(_HERE, "libtdde.so"))

EXPORTS = [
    "tdde_create", "tdde_step", "tdde_propagate", "tdde_norm", "tdde_apply", "tdde_precond",
    "tdde_propagate_host", "tdde_step_forced", "tdde_apply_coupling", "tdde_time_kernel", "tdde_fp64_peak", "tdde_fp64_pipe_probe", "tdde_launch_count",
    "tdde_apply_path", "tdde_snorm_noalloc_setup", "tdde_snorm_noalloc", "tdde_iter_apply_kernel", "tdde_nccl_unique_id", "tdde_group_create", "tdde_group_propagate", "tdde_group_destroy", "tdde_set_eigenstates", "tdde_project", "tdde_eigensolve", "tdde_selftest_partition", "tdde_selftest_mma_frags", "tdde_paper_variant", "tdde_destroy", "tdde_strerror", "tdde_last_cuda_error", "tdde_version",
]

STATUS = {0: "TDDE_OK", -1: "TDDE_EINVAL", -2: "TDDE_ENOMEM", -3: "TDDE_ECUDA", -4: "TDDE_ESINGULAR",
          -5: "TDDE_EBREAKDOWN", -6: "TDDE_ENOCONV"}


class tdde_c64(C.Structure):
    _fields_ = [("re", C.c_double), ("im", C.c_double)]


class tdde_config(C.Structure):
    _fields_ = [("n_ang", C.c_int32), ("n_rad", C.c_int32), ("n_cls", C.c_int32), ("w0", C.c_int32),
                ("n_terms", C.c_int32), ("max_iter", C.c_int32), ("dt", C.c_double), ("rtol", C.c_double)]


class tdde_term(C.Structure):
    _fields_ = [("w", C.c_int32), ("reserved", C.c_int32), ("R_band", C.c_void_p), ("A_rowptr", C.c_void_p),
                ("A_col", C.c_void_p), ("A_val", C.c_void_p)]


class tdde_stats(C.Structure):
    _fields_ = [("steps", C.c_int64), ("half_iters", C.c_int64), ("applies", C.c_int64), ("preconds", C.c_int64),
                ("rel_res", C.c_double), ("status", C.c_int32), ("last_half_iters", C.c_int32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class tdde_shard(C.Structure):
    _fields_ = [("rank", C.c_int32), ("world", C.c_int32), ("own_lo", C.c_int32), ("own_hi", C.c_int32),
                ("n_recv", C.c_int32), ("recv_rank", C.c_void_p), ("recv_lo", C.c_void_p), ("recv_src_lo", C.c_void_p), ("recv_n", C.c_void_p),
                ("n_send", C.c_int32), ("send_rank", C.c_void_p), ("send_lo", C.c_void_p), ("send_n", C.c_void_p)]


class TddeError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        super().__init__(f"{where}: {STATUS.get(status, status)} ({detail})" if detail else f"{where}: {STATUS.get(status, status)}")


_lib = None


def load_library(path: Optional[str] = None) -> C.CDLL:
    """dlopen libtdde.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise RuntimeError(f"{p} is missing: build it with `python -m paper_2512_21697_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(p)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.tdde_create.argtypes = [C.POINTER(vp), C.POINTER(tdde_config), vp, vp, vp, C.POINTER(tdde_term), vp]
    lib.tdde_step.argtypes = [vp, vp, vp, C.POINTER(tdde_stats)]
    lib.tdde_propagate.argtypes = [vp, vp, i64, vp, C.POINTER(tdde_stats)]
    lib.tdde_propagate_host.argtypes = [vp, vp, i64, vp, C.POINTER(tdde_stats)]
    lib.tdde_norm.argtypes = [vp, vp, C.POINTER(dbl)]
    lib.tdde_apply.argtypes = [vp, tdde_c64, tdde_c64, vp, vp, vp]
    lib.tdde_precond.argtypes = [vp, vp, vp]
    lib.tdde_step_forced.argtypes = [vp, vp, vp, i32, vp]
    lib.tdde_time_kernel.argtypes = [vp, i32, i32, vp, C.POINTER(dbl)]
    lib.tdde_apply_coupling.argtypes = [vp, tdde_c64, vp, vp, vp, vp, vp, i32, vp]
    lib.tdde_apply_coupling.restype = C.c_int
    lib.tdde_fp64_peak.argtypes = [vp, C.POINTER(dbl)]
    lib.tdde_fp64_pipe_probe.argtypes = [vp, i32, C.POINTER(dbl)]
    lib.tdde_fp64_pipe_probe.restype = C.c_int
    lib.tdde_launch_count.argtypes = [vp]
    lib.tdde_launch_count.restype = i64
    lib.tdde_apply_path.argtypes = [vp]
    lib.tdde_iter_apply_kernel.argtypes = [vp]
    lib.tdde_iter_apply_kernel.restype = C.c_int
    lib.tdde_set_eigenstates.argtypes = [vp, i32, vp]
    lib.tdde_set_eigenstates.restype = C.c_int
    lib.tdde_project.argtypes = [vp, vp, vp]
    lib.tdde_project.restype = C.c_int
    lib.tdde_eigensolve.argtypes = [i32, i32, i32, vp, vp, vp, vp, vp]
    lib.tdde_eigensolve.restype = C.c_int
    lib.tdde_selftest_partition.argtypes = [i32, i32, i32, C.c_uint32, C.POINTER(dbl)]
    lib.tdde_selftest_partition.restype = C.c_int
    lib.tdde_selftest_mma_frags.argtypes = [i32, i32, i32, C.c_uint32, C.POINTER(dbl)]
    lib.tdde_selftest_mma_frags.restype = C.c_int
    lib.tdde_paper_variant.argtypes = [vp, vp, vp, vp, i32, C.POINTER(dbl), C.POINTER(dbl), C.POINTER(i64)]
    lib.tdde_paper_variant.restype = C.c_int
    lib.tdde_nccl_unique_id.argtypes = [vp]
    lib.tdde_nccl_unique_id.restype = C.c_int
    lib.tdde_group_create.argtypes = [C.POINTER(vp), i32, vp, vp, vp]
    lib.tdde_group_create.restype = C.c_int
    lib.tdde_group_propagate.argtypes = [vp, vp, i64, vp, C.POINTER(tdde_stats)]
    lib.tdde_group_propagate.restype = C.c_int
    lib.tdde_group_destroy.argtypes = [vp]
    lib.tdde_group_destroy.restype = None
    lib.tdde_snorm_noalloc_setup.argtypes = []
    lib.tdde_snorm_noalloc_setup.restype = C.c_int
    lib.tdde_snorm_noalloc.argtypes = [i32, i32, i32, i32, vp, vp, vp, vp, vp]
    lib.tdde_snorm_noalloc.restype = C.c_int
    lib.tdde_destroy.argtypes = [vp]
    lib.tdde_destroy.restype = None
    lib.tdde_strerror.argtypes = [C.c_int]
    lib.tdde_strerror.restype = C.c_char_p
    lib.tdde_last_cuda_error.restype = C.c_char_p
    for name in ("tdde_create", "tdde_step", "tdde_propagate", "tdde_propagate_host", "tdde_norm", "tdde_apply",
                 "tdde_precond", "tdde_step_forced", "tdde_time_kernel", "tdde_fp64_peak", "tdde_apply_path",
                 "tdde_version"):
        getattr(lib, name).restype = C.c_int
    if path is None:
        _lib = lib
    return lib


def _check(lib, rc: int, where: str):
    if rc != 0:
        detail = lib.tdde_last_cuda_error().decode() if rc == -3 else lib.tdde_strerror(rc).decode()
        raise TddeError(rc, where, detail)


def _np_ptr(a: np.ndarray) -> int:
    return a.ctypes.data


def _g_array(g, n_terms: int, rows: Optional[int] = None) -> np.ndarray:
    g = np.ascontiguousarray(np.asarray(g, dtype=np.float64))
    want = n_terms if rows is None else rows * n_terms
    if g.size != want:
        raise ValueError(f"g has {g.size} entries, expected {want}")
    return g


def eigensolve(S_band: np.ndarray, H0_band: np.ndarray, want_vectors: bool = True, stream=None):
    """All eigenpairs of the per-class pencils (H0_k, S_k) on the GPU (tdde_eigensolve): returns (E [n_cls, n_rad] ascending,
    V [n_cls, n_rad, n_rad] with V[k, e, :] the S-orthonormal eigenvector of E[k, e], or None)."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: the TDDE library has no CPU fallback")
    lib = load_library()
    S = np.ascontiguousarray(S_band, dtype=np.complex128)
    H = np.ascontiguousarray(H0_band, dtype=np.complex128)
    n_cls, n_rad, nd = S.shape
    E = np.empty((n_cls, n_rad), dtype=np.float64)
    V = np.empty((n_cls, n_rad, n_rad), dtype=np.complex128) if want_vectors else None
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = lib.tdde_eigensolve(n_cls, n_rad, (nd - 1) // 2, _np_ptr(S), _np_ptr(H), _np_ptr(E), _np_ptr(V) if want_vectors else None,
                             C.c_void_p(st.cuda_stream))
    _check(lib, rc, "tdde_eigensolve")
    return E, V


class Tdde:
    """One propagator handle (tdde_create ... tdde_destroy) for a tdde_inputs.Problem-like object."""

    def __init__(self, problem, dt: Optional[float] = None, rtol: Optional[float] = None,
                 max_iter: Optional[int] = None, stream=None, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the TDDE propagator has no CPU fallback")
        self.lib = load_library()
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.n_ang, self.n_rad, self.n_terms = problem.n_ang, problem.n_rad, problem.n_terms
        self.n = problem.n_ang * problem.n_rad
        cfg = tdde_config(problem.n_ang, problem.n_rad, problem.n_cls, problem.w0, problem.n_terms,
                          int(problem.max_iter if max_iter is None else max_iter),
                          float(problem.dt if dt is None else dt), float(problem.rtol if rtol is None else rtol))
        S = np.ascontiguousarray(problem.S_band, dtype=np.complex128)
        H0 = np.ascontiguousarray(problem.H0_band, dtype=np.complex128)
        cls = np.ascontiguousarray(problem.cls_of_chan, dtype=np.int32)
        keep = [S, H0, cls]
        terms = (tdde_term * max(1, problem.n_terms))()
        for L, t in enumerate(problem.terms):
            R = np.ascontiguousarray(t.R_band, dtype=np.complex128)
            rp = np.ascontiguousarray(t.A_rowptr, dtype=np.int32)
            col = np.ascontiguousarray(t.A_col, dtype=np.int32)
            val = np.ascontiguousarray(t.A_val, dtype=np.complex128)
            keep += [R, rp, col, val]
            terms[L] = tdde_term(int(t.w), 0, _np_ptr(R), _np_ptr(rp), _np_ptr(col), _np_ptr(val))
        h = C.c_void_p()
        rc = self.lib.tdde_create(C.byref(h), C.byref(cfg), _np_ptr(S), _np_ptr(H0), _np_ptr(cls), terms,
                                  C.c_void_p(self.stream.cuda_stream))
        _check(self.lib, rc, "tdde_create")
        self.h = h

    # -- helpers --
    def to_device(self, c: np.ndarray):
        t = self.torch.from_numpy(np.ascontiguousarray(c, dtype=np.complex128))
        return t.to(self.device)

    def _vec(self, t, name="vector"):
        if t.dtype != self.torch.complex128 or not t.is_cuda or not t.is_contiguous() or t.numel() != self.n:
            raise ValueError(f"{name} must be a contiguous CUDA complex128 tensor of {self.n} elements")
        return C.c_void_p(t.data_ptr())

    # -- C ABI mirrors --
    def step(self, c_dev, g_mid, want_stats: bool = True):
        g = _g_array(g_mid, self.n_terms)
        st = tdde_stats()
        rc = self.lib.tdde_step(self.h, self._vec(c_dev), _np_ptr(g), C.byref(st) if want_stats else None)
        _check(self.lib, rc, "tdde_step")
        return st.as_dict()

    def propagate(self, c_dev, g_table, n_steps: Optional[int] = None, check: bool = True):
        g = np.asarray(g_table, dtype=np.float64)
        n_steps = (g.shape[0] if g.ndim == 2 else 1) if n_steps is None else n_steps
        g = _g_array(g, self.n_terms, n_steps)
        st = tdde_stats()
        rc = self.lib.tdde_propagate(self.h, self._vec(c_dev), n_steps, _np_ptr(g), C.byref(st))
        if check:
            _check(self.lib, rc, "tdde_propagate")
        out = st.as_dict()
        out["rc"] = rc
        return out

    def propagate_host(self, c_host: np.ndarray, g_table, n_steps: int):
        if c_host.dtype != np.complex128 or not c_host.flags.c_contiguous or c_host.size != self.n:
            raise ValueError("c_host must be a contiguous complex128 array of n elements")
        g = _g_array(g_table, self.n_terms, n_steps)
        st = tdde_stats()
        rc = self.lib.tdde_propagate_host(self.h, _np_ptr(c_host), n_steps, _np_ptr(g), C.byref(st))
        _check(self.lib, rc, "tdde_propagate_host")
        return st.as_dict()

    def norm(self, c_dev) -> float:
        out = C.c_double()
        _check(self.lib, self.lib.tdde_norm(self.h, self._vec(c_dev), C.byref(out)), "tdde_norm")
        return out.value

    def apply(self, alpha: complex, beta: complex, g, x_dev, y_dev=None):
        g = _g_array(g, self.n_terms) if self.n_terms else np.zeros(1)
        y = self.torch.empty_like(x_dev) if y_dev is None else y_dev
        a, b = complex(alpha), complex(beta)
        rc = self.lib.tdde_apply(self.h, tdde_c64(a.real, a.imag), tdde_c64(b.real, b.imag), _np_ptr(g),
                                 self._vec(x_dev, "x"), self._vec(y, "y"))
        _check(self.lib, rc, "tdde_apply")
        return y

    def apply_coupling(self, beta: complex, g, x_dev, addv_dev, aux_dev=None, which: int = 0):
        """y = addv + beta sum_L g_L (A_L (x) R_L) x by the in-iteration kernel; returns (y, <aux,y>, ||y||^2)  (tdde_apply_coupling)."""
        g = _g_array(g, self.n_terms)
        y = self.torch.empty_like(x_dev)
        b = complex(beta)
        dots = np.zeros(3)
        rc = self.lib.tdde_apply_coupling(self.h, tdde_c64(b.real, b.imag), _np_ptr(g), self._vec(x_dev, "x"), self._vec(addv_dev, "addv"),
                                          self._vec(aux_dev, "aux") if aux_dev is not None else None, self._vec(y, "y"), int(which), _np_ptr(dots))
        _check(self.lib, rc, "tdde_apply_coupling")
        return y, complex(dots[0], dots[1]), float(dots[2])

    def precond(self, x_dev, y_dev=None):
        y = self.torch.empty_like(x_dev) if y_dev is None else y_dev
        _check(self.lib, self.lib.tdde_precond(self.h, self._vec(x_dev, "x"), self._vec(y, "y")), "tdde_precond")
        return y

    def step_forced(self, c_dev, g_mid, n_iters: int, trace: bool = True):
        g = _g_array(g_mid, self.n_terms)
        tr = self.torch.empty((n_iters, 8, self.n), dtype=self.torch.complex128, device=self.device) if trace else None
        rc = self.lib.tdde_step_forced(self.h, self._vec(c_dev), _np_ptr(g), n_iters,
                                       C.c_void_p(tr.data_ptr()) if trace else None)
        _check(self.lib, rc, "tdde_step_forced")
        return tr

    def set_eigenstates(self, V: np.ndarray):
        """V[k, e, :] = eigenvector e of the pencil (H0_k, S_k) of kappa-class k (tdde_set_eigenstates)."""
        V = np.ascontiguousarray(V, dtype=np.complex128)
        if V.ndim != 3 or V.shape[2] != self.n_rad:
            raise ValueError("V must have shape [n_cls, n_states, n_rad]")
        self._n_states = V.shape[1]
        _check(self.lib, self.lib.tdde_set_eigenstates(self.h, V.shape[1], _np_ptr(V)), "tdde_set_eigenstates")

    def project(self, c_dev) -> np.ndarray:
        """P[a, e] = |v_{k(a),e}^H S c_a|^2 (tdde_project; Eq. 33 before the sum over channels)."""
        out = np.empty((self.n_ang, self._n_states), dtype=np.float64)
        _check(self.lib, self.lib.tdde_project(self.h, self._vec(c_dev), _np_ptr(out)), "tdde_project")
        return out

    def time_kernel(self, which: int, reps: int, g=None) -> float:
        garr = _g_array(g, self.n_terms) if (g is not None and self.n_terms) else np.zeros(max(1, self.n_terms))
        out = C.c_double()
        _check(self.lib, self.lib.tdde_time_kernel(self.h, which, reps, _np_ptr(garr), C.byref(out)), "tdde_time_kernel")
        return out.value

    def paper_variant(self, g, x_dev, reps: int = 3):
        """The paper's formulation (CSR assembly + SpMV) as a comparator: returns (y, ms_assemble, ms_spmv, nnz)."""
        garr = _g_array(g, self.n_terms) if self.n_terms else np.zeros(1)
        y = self.torch.empty_like(x_dev)
        ta, ts, nnz = C.c_double(), C.c_double(), C.c_int64()
        rc = self.lib.tdde_paper_variant(self.h, _np_ptr(garr), self._vec(x_dev, "x"), self._vec(y, "y"), reps,
                                         C.byref(ta), C.byref(ts), C.byref(nnz))
        _check(self.lib, rc, "tdde_paper_variant")
        return y, ta.value, ts.value, nnz.value

    def fp64_pipe_probe(self, mode: int) -> float:
        """FLOP/s of the FP64 pipe: mode 0 DFMA, 1 DMMA, 2 DMMA + DFMA mixed (tdde_fp64_pipe_probe)."""
        out = C.c_double()
        _check(self.lib, self.lib.tdde_fp64_pipe_probe(C.c_void_p(self.stream.cuda_stream), mode, C.byref(out)), "tdde_fp64_pipe_probe")
        return out.value

    def fp64_peak(self) -> float:
        out = C.c_double()
        _check(self.lib, self.lib.tdde_fp64_peak(C.c_void_p(self.stream.cuda_stream), C.byref(out)), "tdde_fp64_peak")
        return out.value

    @property
    def launch_count(self) -> int:
        return int(self.lib.tdde_launch_count(self.h))

    @property
    def apply_path(self) -> str:
        return {1: "banded", 2: "staged", 0: "generic"}.get(self.lib.tdde_apply_path(self.h), "unknown")

    @property
    def iter_apply_kernel(self) -> str:
        """The kernel an iteration uses for v = A y (tdde_iter_apply_kernel)."""
        return {0: "k_apply_generic", 1: "k_apply_banded", 2: "k_apply_sparse", 3: "k_apply_mma"}.get(
            self.lib.tdde_iter_apply_kernel(self.h), "unknown")

    def close(self):
        if getattr(self, "h", None):
            self.lib.tdde_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def nccl_unique_id() -> bytes:
    """128-byte NCCL id (tdde_nccl_unique_id): rank 0 creates it, the launcher broadcasts it to the other ranks."""
    lib = load_library()
    buf = C.create_string_buffer(128)
    _check(lib, lib.tdde_nccl_unique_id(buf), "tdde_nccl_unique_id")
    return buf.raw


class TddeGroup:
    """The shards of one process driven in lock step (tdde_group_*).  `shards`: Tdde handles built from the
    rank-local problems; `specs`: one dict per shard with rank, world, own_lo, own_hi and the integer lists recv_rank, recv_lo,
    recv_src_lo, recv_n, send_rank, send_lo, send_n (paper_2512_21697_b200.sharding.shard_specs); `nccl_id`: 128 bytes for one shard
    per process over NCCL, None when every shard of the job is in this process."""

    def __init__(self, shards, specs, nccl_id: Optional[bytes] = None):
        self.lib = load_library()
        self.shards = list(shards)
        self._keep = []
        arr = (tdde_shard * len(specs))()

        def ptr(v):
            a = np.ascontiguousarray(v, dtype=np.int32)
            self._keep.append(a)
            return a.ctypes.data if a.size else None
        for k, sp in enumerate(specs):
            arr[k].rank, arr[k].world, arr[k].own_lo, arr[k].own_hi = sp["rank"], sp["world"], sp["own_lo"], sp["own_hi"]
            arr[k].n_recv, arr[k].n_send = len(sp["recv_n"]), len(sp["send_n"])
            arr[k].recv_rank, arr[k].recv_lo, arr[k].recv_src_lo, arr[k].recv_n = (ptr(sp[q]) for q in ("recv_rank", "recv_lo", "recv_src_lo", "recv_n"))
            arr[k].send_rank, arr[k].send_lo, arr[k].send_n = (ptr(sp[q]) for q in ("send_rank", "send_lo", "send_n"))
        hs = (C.c_void_p * len(self.shards))(*[sh.h for sh in self.shards])
        self.g = C.c_void_p()
        idbuf = C.create_string_buffer(nccl_id, 128) if nccl_id is not None else None
        _check(self.lib, self.lib.tdde_group_create(C.byref(self.g), len(self.shards), hs, arr, idbuf), "tdde_group_create")

    def propagate(self, c_devs, g_table, n_steps: Optional[int] = None):
        g = np.asarray(g_table, dtype=np.float64)
        n_steps = (g.shape[0] if g.ndim == 2 else 1) if n_steps is None else n_steps
        g = _g_array(g, self.shards[0].n_terms, n_steps)
        ptrs = (C.c_void_p * len(self.shards))(*[sh._vec(c).value for sh, c in zip(self.shards, c_devs)])
        st = tdde_stats()
        rc = self.lib.tdde_group_propagate(self.g, ptrs, n_steps, _np_ptr(g), C.byref(st))
        _check(self.lib, rc, "tdde_group_propagate")
        return st.as_dict()

    def close(self):
        if getattr(self, "g", None):
            self.lib.tdde_group_destroy(self.g)
            self.g = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


NOALLOC_MAX_N = 2048 * 8192      # TDDE_NOALLOC_MAX_N of include/tdde.h


def snorm_noalloc_setup():
    """Resolve the static scratch array's device address on the current device (tdde_snorm_noalloc_setup)."""
    lib = load_library()
    _check(lib, lib.tdde_snorm_noalloc_setup(), "tdde_snorm_noalloc_setup")


def snorm_noalloc(n_ang: int, n_rad: int, n_cls: int, w0: int, S_dev, cls_dev, c_dev, out_dev, stream=None, check: bool = True) -> int:
    """*out_dev = Re(c^H S c) without any allocation (tdde_snorm_noalloc).  S_dev: CUDA complex128 [n_cls, n_rad, 2 w0 + 1] (row band),
    cls_dev: CUDA int32 [n_ang], c_dev: CUDA complex128 [n_ang * n_rad], out_dev: CUDA float64 [1].  Argument marshalling only."""
    lib = load_library()
    st = C.c_void_p(stream.cuda_stream) if stream is not None else None
    rc = lib.tdde_snorm_noalloc(n_ang, n_rad, n_cls, w0, C.c_void_p(S_dev.data_ptr()), C.c_void_p(cls_dev.data_ptr()),
                                C.c_void_p(c_dev.data_ptr()), C.c_void_p(out_dev.data_ptr()), st)
    if check:
        _check(lib, rc, "tdde_snorm_noalloc")
    return rc
