"""ctypes binding of include/lgf.h (argument marshalling only; every step runs in the CUDA kernels)."""
from __future__ import annotations

import ctypes
import os
import re
from dataclasses import dataclass
from typing import Optional, Sequence

LGF_F32, LGF_F64 = 0, 1
LGF_REAL18, LGF_REAL12 = 18, 12
LGF_HOST, LGF_DEVICE = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
_HEADER = os.path.join(os.path.dirname(_HERE), "include", "lgf.h")
_lib: Optional[ctypes.CDLL] = None


class LgfError(RuntimeError):
    pass


class _Result(ctypes.Structure):
    _fields_ = [("iterations", ctypes.c_int64), ("theta", ctypes.c_double), ("F", ctypes.c_double),
                ("converged", ctypes.c_int32)]


@dataclass
class LgfResult:
    iterations: int
    theta: float
    F: float
    converged: bool


def library_path() -> str:
    # LGF_LIBRARY: developer override used to A/B kernel variants; the default is the in-tree build
    return os.environ.get("LGF_LIBRARY") or os.path.join(_HERE, "liblgf.so")


def declared_symbols() -> list:
    """Every function include/lgf.h declares (used by the CPU test that the library exports them)."""
    text = open(_HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lgf_[a-z_0-9]+)\s*\(", text)))


def load_library() -> ctypes.CDLL:
    """dlopen liblgf.so (no build here: `__graft_entry__.build()` / `_build.build()` compile it)."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path):
        raise LgfError(f"{path} is missing: run `python -m paper_1208_1186_b200._build` (there is no CPU fallback)")
    lib = ctypes.CDLL(path)
    i32p = ctypes.POINTER(ctypes.c_int32)
    rp = ctypes.POINTER(_Result)
    vp = ctypes.c_void_p
    lib.lgf_workspace_bytes.restype = ctypes.c_size_t
    lib.lgf_workspace_bytes.argtypes = [i32p, ctypes.c_int, ctypes.c_int]
    lib.lgf_create.argtypes = [i32p, ctypes.c_int, ctypes.c_int, vp, ctypes.c_size_t, vp, ctypes.POINTER(vp)]
    lib.lgf_create_simple.argtypes = [i32p, ctypes.c_int, ctypes.c_int, ctypes.POINTER(vp)]
    lib.lgf_workspace_bytes_batch.restype = ctypes.c_size_t
    lib.lgf_workspace_bytes_batch.argtypes = [i32p, ctypes.c_int, ctypes.c_int, ctypes.c_int32]
    lib.lgf_create_batch.argtypes = [i32p, ctypes.c_int, ctypes.c_int, ctypes.c_int32, vp, ctypes.c_size_t, vp, ctypes.POINTER(vp)]
    lib.lgf_batch_size.restype = ctypes.c_int32
    lib.lgf_batch_size.argtypes = [vp]
    lib.lgf_destroy.argtypes = [vp]
    lib.lgf_load.argtypes = [vp, vp, ctypes.c_int]
    lib.lgf_store.argtypes = [vp, vp, ctypes.c_int]
    lib.lgf_measure.argtypes = [vp, rp]
    lib.lgf_iterate.argtypes = [vp, ctypes.c_int64, ctypes.c_double, rp]
    lib.lgf_iterate_async.argtypes = [vp, ctypes.c_int64, ctypes.c_double]
    lib.lgf_wait.argtypes = [vp, rp]
    lib.lgf_fix.argtypes = [vp, ctypes.c_double, ctypes.c_double, ctypes.c_int64, rp]
    lib.lgf_profile_iterate.argtypes = [vp, ctypes.c_int64, ctypes.c_double, ctypes.POINTER(ctypes.c_double), rp]
    lib.lgf_debug_get_delta.argtypes = [vp, vp, ctypes.c_int]
    lib.lgf_wilson_lines.argtypes = [vp, vp, ctypes.c_int]
    lib.lgf_singlet_correlator.argtypes = [vp, vp, ctypes.c_int]
    lib.lgf_debug_fourier_accelerate.argtypes = [vp]
    lib.lgf_path_info.argtypes = [vp, i32p]
    lib.lgf_describe.argtypes = [vp, ctypes.c_char_p, ctypes.c_size_t]
    lib.lgf_launch_count.restype = ctypes.c_int64
    lib.lgf_launch_count.argtypes = [vp]
    lib.lgf_static_init.argtypes = []
    lib.lgf_measure_static.argtypes = [i32p, ctypes.c_int, vp, vp, vp]
    lib.lgf_static_scratch_bytes.restype = ctypes.c_size_t
    lib.lgf_static_scratch_bytes.argtypes = []
    lib.lgf_static_last_error.restype = ctypes.c_char_p
    lib.lgf_static_last_error.argtypes = []
    for f in (lib.lgf_strerror, lib.lgf_last_error, lib.lgf_version):
        f.restype = ctypes.c_char_p
    lib.lgf_strerror.argtypes = [ctypes.c_int]
    _lib = lib
    return lib


def _L(L: Sequence[int]):
    return (ctypes.c_int32 * 4)(*[int(v) for v in L])


def workspace_bytes(L: Sequence[int], precision: int, storage: int, nbatch: int = 1) -> int:
    return int(load_library().lgf_workspace_bytes_batch(_L(L), precision, storage, int(nbatch)))


def _check(rc: int, what: str) -> None:
    if rc != 0:
        lib = load_library()
        raise LgfError(f"{what}: {lib.lgf_strerror(rc).decode()} [{rc}] {lib.lgf_last_error().decode()}")


STATIC_MAX_SITES = 16777216   # LGF_STATIC_MAX_SITES of include/lgf.h (64^4)


def static_init() -> None:
    """lgf_static_init: resolve the static scratch array's address on the current CUDA device."""
    lib = load_library()
    rc = lib.lgf_static_init()
    if rc:
        raise LgfError(f"lgf_static_init: {lib.lgf_strerror(rc).decode()} [{rc}] {lib.lgf_static_last_error().decode()}")


def measure_static(L: Sequence[int], links, out=None, stream=None):
    """lgf_measure_static: theta and F of a DEVICE link tensor [V, 4, 3, 3, 2] (float32 / float64) without a context,
    a workspace or any allocation inside the library (its scratch is a 1 MiB static device array, at most
    STATIC_MAX_SITES sites; calls that overlap on the GPU race on it).  -> `out`, a device tensor of 2 float64
    {theta, F} (made here when not given -- pass one to keep the caller's side allocation-free too); the kernels are
    enqueued on `stream` (default: torch's current stream) and the call does not synchronise."""
    import torch
    lib = load_library()
    if not links.is_cuda or not links.is_contiguous() or links.dtype not in (torch.float32, torch.float64):
        raise LgfError("measure_static: links must be a contiguous CUDA tensor of float32 or float64")
    if out is None:
        out = torch.empty(2, dtype=torch.float64, device=links.device)
    if not out.is_cuda or out.dtype != torch.float64 or out.numel() < 2 or out.device != links.device:
        raise LgfError("measure_static: out must be a CUDA tensor of 2 float64 on the links' device")
    with torch.cuda.device(links.device):
        s = stream if stream is not None else torch.cuda.current_stream()
        rc = lib.lgf_measure_static(_L(L), LGF_F64 if links.dtype == torch.float64 else LGF_F32, links.data_ptr(),
                                    s.cuda_stream, out.data_ptr())
    if rc:
        raise LgfError(f"lgf_measure_static: {lib.lgf_strerror(rc).decode()} [{rc}] {lib.lgf_static_last_error().decode()}")
    return out


class GaugeFixer:
    """One lattice -- or `nbatch` independent lattices of one shape fixed by the same launches -- on one GPU.  Methods
    mirror the C ABI: load, store, measure, iterate, fix.  With nbatch > 1 link tensors carry a leading batch axis
    ([nbatch * V, 4, 3, 3, 2]) and every result is a list of nbatch LgfResult."""

    def __init__(self, L: Sequence[int], precision: int = LGF_F64, storage: int = LGF_REAL18,
                 device: str = "cuda:0", stream=None, nbatch: int = 1):
        import torch
        if not torch.cuda.is_available():
            raise LgfError("no CUDA device: the lgf library has no CPU fallback")
        self._torch = torch
        self.lib = load_library()
        self.L = tuple(int(v) for v in L)
        self.V = self.L[0] * self.L[1] * self.L[2] * self.L[3]
        self.precision, self.storage = precision, storage
        self.dtype = torch.float64 if precision == LGF_F64 else torch.float32
        self.device = torch.device(device)
        self.nbatch = int(nbatch)
        nbytes = self.lib.lgf_workspace_bytes_batch(_L(self.L), precision, storage, self.nbatch)
        if nbytes == 0:
            raise LgfError(f"unsupported lattice {self.L} x {self.nbatch} (extents must be 2^a 3^b >= 2, tiles must fit on chip)")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            ptr = (self.workspace.data_ptr() + 255) // 256 * 256
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = ctypes.c_void_p()
            _check(self.lib.lgf_create_batch(_L(self.L), precision, storage, self.nbatch, ctypes.c_void_p(ptr), nbytes,
                                             ctypes.c_void_p(self.stream.cuda_stream), ctypes.byref(h)), "lgf_create_batch")
        self._h = h

    def close(self) -> None:
        if getattr(self, "_h", None):
            self.lib.lgf_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- marshalling helpers
    def _ptr_space(self, t):
        assert t.dtype == self.dtype and t.is_contiguous(), (t.dtype, self.dtype)
        return ctypes.c_void_p(t.data_ptr()), (LGF_DEVICE if t.is_cuda else LGF_HOST)

    def load(self, links) -> None:
        """links: real tensor [V,4,3,3,2] (host or device) of the context precision."""
        assert links.numel() == self.nbatch * self.V * 72
        p, sp = self._ptr_space(links)
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_load(self._h, p, sp), "lgf_load")

    def store(self, out=None, device=None):
        torch = self._torch
        if out is None:
            out = torch.empty(self.nbatch * self.V, 4, 3, 3, 2, dtype=self.dtype, device=device or "cpu")
        p, sp = self._ptr_space(out)
        with torch.cuda.device(self.device):
            _check(self.lib.lgf_store(self._h, p, sp), "lgf_store")
        return out

    def _new_res(self):
        return (_Result * self.nbatch)()

    def _res(self, r):
        out = [LgfResult(int(x.iterations), float(x.theta), float(x.F), bool(x.converged)) for x in r]
        return out[0] if self.nbatch == 1 else out

    def measure(self) -> LgfResult:
        r = self._new_res()
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_measure(self._h, r), "lgf_measure")
        return self._res(r)

    def iterate(self, n: int, alpha: float) -> LgfResult:
        r = self._new_res()
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_iterate(self._h, int(n), float(alpha), r), "lgf_iterate")
        return self._res(r)

    def iterate_async(self, n: int, alpha: float) -> None:
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_iterate_async(self._h, int(n), float(alpha)), "lgf_iterate_async")

    def wait(self) -> LgfResult:
        r = self._new_res()
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_wait(self._h, r), "lgf_wait")
        return self._res(r)

    def fix(self, alpha: float, theta_tol: float, max_iter: int) -> LgfResult:
        r = self._new_res()
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_fix(self._h, float(alpha), float(theta_tol), int(max_iter), r), "lgf_fix")
        return self._res(r)

    KERNELS = ("K2_fft_xy_fwd", "K3_fft_zt_fwd_scale_inv", "K4_fft_xy_inv", "K5_gbuild_update", "K1_delta_theta_F")
    KERNELS_FUSED = ("K2_fft_xy_fwd", "K3_fft_zt_fwd_scale_inv", "K4_fft_xy_inv", "K51_update_delta_fused")

    def path_info(self) -> dict:
        """Which kernels the iteration runs: fft_path 0/1/2, fused K5+K1, site-kernel CTAs, launches per iteration."""
        info = (ctypes.c_int32 * 4)()
        _check(self.lib.lgf_path_info(self._h, info), "lgf_path_info")
        return {"fft_path": ("runtime-radix", "compile-time", "pipelined")[info[0]], "fused": bool(info[1]),
                "site_ctas": int(info[2]), "launches_per_iteration": int(info[3])}

    def describe(self) -> str:
        buf = ctypes.create_string_buffer(1024)
        _check(self.lib.lgf_describe(self._h, buf, 1024), "lgf_describe")
        return buf.value.decode()

    def profile_iterate(self, n: int, alpha: float):
        """-> (dict kernel name -> average ms per launch, LgfResult).  With the fused update kernel the
        dict has four entries (K5 and K1 are one kernel)."""
        ms = (ctypes.c_double * 5)()
        r = self._new_res()
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_profile_iterate(self._h, int(n), float(alpha), ms, r), "lgf_profile_iterate")
        names = self.KERNELS_FUSED if self.path_info()["fused"] else self.KERNELS
        return {k: float(ms[i]) for i, k in enumerate(names)}, self._res(r)

    def wilson_lines(self, device=None):
        """Temporal Wilson lines of the current links: real tensor [Vs, 3, 3, 2]."""
        out = self._torch.empty(self.V // self.L[3], 3, 3, 2, dtype=self.dtype, device=device or "cpu")
        p, sp = self._ptr_space(out)
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_wilson_lines(self._h, p, sp), "lgf_wilson_lines")
        return out

    def singlet_correlator(self, device=None):
        """C(r) = (1/(3 Vs)) sum_x Tr[W(x + r) W(x)^+] of the current links: real tensor [Vs, 2], r with x fastest."""
        out = self._torch.empty(self.V // self.L[3], 2, dtype=self.dtype, device=device or "cpu")
        p, sp = self._ptr_space(out)
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_singlet_correlator(self._h, p, sp), "lgf_singlet_correlator")
        return out

    def debug_delta(self):
        """Packed Delta field as a host tensor [V,4,2]."""
        out = self._torch.empty(self.V, 4, 2, dtype=self.dtype)
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_debug_get_delta(self._h, ctypes.c_void_p(out.data_ptr()), LGF_HOST), "lgf_debug_get_delta")
        return out

    def debug_fourier_accelerate(self) -> None:
        with self._torch.cuda.device(self.device):
            _check(self.lib.lgf_debug_fourier_accelerate(self._h), "lgf_debug_fourier_accelerate")

    def launch_count(self) -> int:
        return int(self.lib.lgf_launch_count(self._h))
