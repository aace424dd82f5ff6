"""Thin Python binding of the C-ABI in include/potts.h (same names, argument marshalling only).

Every step of the hot path runs in the CUDA kernels of ``csrc/``; this module only converts
arguments.  PyTorch supplies device memory (the lattice workspace is a ``torch.uint8`` CUDA
tensor handed to ``potts_create_ex``) and the stream (torch's current stream).  There is no CPU
fallback: if the shared library is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpotts_b200.so")

OK, ERR_ARG, ERR_UNSUPPORTED, ERR_NOMEM, ERR_CUDA = 0, 1, 2, 3, 4
INIT_ORDERED, INIT_RANDOM = 0, 1
LAYOUT_U8, LAYOUT_PACKED = 0, 1

_lib = None


class PottsError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"potts error {code}: {msg}")
        self.code = code


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_1101_0876_b200.build` "
            "(or __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, u64, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_uint64, ctypes.c_double
    P = ctypes.POINTER
    sigs = {
        "potts_create": ([P(vp), i32, i32, u64, i32], ctypes.c_int),
        "potts_create_ex": ([P(vp), i32, i32, u64, i32, i32, vp, ctypes.c_size_t, vp], ctypes.c_int),
        "potts_workspace_bytes": ([i32, i32, i32, P(ctypes.c_size_t)], ctypes.c_int),
        "potts_set_stream": ([vp, vp], ctypes.c_int),
        "potts_destroy": ([vp], None),
        "potts_sweep": ([vp, dbl, i64], ctypes.c_int),
        "potts_sweep_measured": ([vp, dbl, i64, i64, vp, vp], ctypes.c_int),
        "potts_sweep_measured_dev": ([vp, dbl, i64, i64, vp, vp], ctypes.c_int),
        "potts_sweep_delta": ([vp, dbl, i64, vp], ctypes.c_int),
        "potts_ladder": ([vp, vp, i32, i64, i64, i64, vp, vp], ctypes.c_int),
        "potts_batch_workspace_bytes": ([i32, i32, i32, P(ctypes.c_size_t)], ctypes.c_int),
        "potts_batch_create": ([P(vp), i32, i32, i32, vp, i32, vp, ctypes.c_size_t, vp], ctypes.c_int),
        "potts_batch_destroy": ([vp], None),
        "potts_batch_sweep_measured": ([vp, vp, i64, i64, vp, vp], ctypes.c_int),
        "potts_batch_download": ([vp, i32, vp], ctypes.c_int),
        "potts_batch_sweep_delta": ([vp, vp, i64, vp], ctypes.c_int),
        "potts_batch_sweep_measured_dev": ([vp, vp, i64, i64, vp, vp], ctypes.c_int),
        "potts_batch_ladder": ([vp, vp, i32, i64, i64, i64, vp, vp], ctypes.c_int),
        "potts_batch_sweep_count": ([vp, P(u64)], ctypes.c_int),
        "potts_batch_launch_count": ([vp, P(u64)], ctypes.c_int),
        "potts_set_stream_spec": ([vp, i32], ctypes.c_int),
        "potts_get_stream_spec": ([vp, P(i32)], ctypes.c_int),
        "potts_batch_set_stream_spec": ([vp, i32], ctypes.c_int),
        "potts_energy": ([vp, P(i64)], ctypes.c_int),
        "potts_histogram": ([vp, vp], ctypes.c_int),
        "potts_download": ([vp, vp], ctypes.c_int),
        "potts_upload": ([vp, vp], ctypes.c_int),
        "potts_sweep_count": ([vp, P(u64)], ctypes.c_int),
        "potts_set_sweep_count": ([vp, u64], ctypes.c_int),
        "potts_observables": ([vp, i64, i64, dbl, P(dbl), P(dbl), P(dbl)], ctypes.c_int),
        "potts_magnetisation": ([vp, i32, P(dbl)], ctypes.c_int),
        "potts_susceptibility": ([vp, i64, i32, dbl, P(dbl), P(dbl), P(dbl)], ctypes.c_int),
        "potts_launch_count": ([vp, P(u64)], ctypes.c_int),
        "potts_set_option": ([vp, ctypes.c_char_p, i64], ctypes.c_int),
        "potts_get_option": ([vp, ctypes.c_char_p, P(i64)], ctypes.c_int),
        "potts_create_strip": ([P(vp), i32, i32, u64, i32, i32, i32, vp], ctypes.c_int),
        "potts_strip_half_sweep": ([vp, dbl, i32, vp, vp], ctypes.c_int),
        "potts_strip_advance": ([vp], ctypes.c_int),
        "potts_strip_rows": ([vp, i32, P(vp), P(vp), P(vp), P(vp), P(ctypes.c_size_t)], ctypes.c_int),
        "potts3_create": ([P(vp), i32, i32, u64, i32, vp], ctypes.c_int),
        "potts3_destroy": ([vp], None),
        "potts3_sweep": ([vp, dbl, i64], ctypes.c_int),
        "potts3_sweep_measured": ([vp, dbl, i64, i64, vp, vp], ctypes.c_int),
        "potts3_energy": ([vp, P(i64)], ctypes.c_int),
        "potts3_histogram": ([vp, vp], ctypes.c_int),
        "potts3_download": ([vp, vp], ctypes.c_int),
        "potts3_upload": ([vp, vp], ctypes.c_int),
        "potts3_sweep_count": ([vp, P(u64)], ctypes.c_int),
        "potts3_set_sweep_count": ([vp, u64], ctypes.c_int),
        "potts3_launch_count": ([vp, P(u64)], ctypes.c_int),
        "potts3_set_option": ([vp, ctypes.c_char_p, i64], ctypes.c_int),
        "potts8_set_option": ([vp, ctypes.c_char_p, i64], ctypes.c_int),
        "potts_measure_noalloc": ([vp, i32, i32, vp, vp, vp], ctypes.c_int),
        "potts8_create": ([P(vp), i32, i32, u64, i32, vp], ctypes.c_int),
        "potts8_destroy": ([vp], None),
        "potts8_sweep": ([vp, dbl, i64], ctypes.c_int),
        "potts8_sweep_measured": ([vp, dbl, i64, i64, vp, vp], ctypes.c_int),
        "potts8_energy": ([vp, P(i64)], ctypes.c_int),
        "potts8_histogram": ([vp, vp], ctypes.c_int),
        "potts8_download": ([vp, vp], ctypes.c_int),
        "potts8_upload": ([vp, vp], ctypes.c_int),
        "potts8_sweep_count": ([vp, P(u64)], ctypes.c_int),
        "potts8_set_sweep_count": ([vp, u64], ctypes.c_int),
        "potts8_launch_count": ([vp, P(u64)], ctypes.c_int),
        "potts_last_error": ([], ctypes.c_char_p),
        "potts_version": ([], ctypes.c_char_p),
    }
    for name, (argtypes, restype) in sigs.items():
        fn = getattr(lib, name)          # AttributeError if the symbol is not exported
        fn.argtypes = argtypes
        fn.restype = restype
    _lib = lib
    return lib


EXPORTED_SYMBOLS = [
    "potts_create", "potts_create_ex", "potts_workspace_bytes", "potts_set_stream", "potts_destroy",
    "potts_sweep", "potts_sweep_measured", "potts_sweep_measured_dev", "potts_sweep_delta", "potts_ladder", "potts_energy", "potts_histogram",
    "potts_download", "potts_upload", "potts_sweep_count", "potts_set_sweep_count", "potts_observables",
    "potts_magnetisation", "potts_susceptibility", "potts_launch_count", "potts_set_option", "potts_get_option", "potts_last_error",
    "potts_version", "potts_batch_workspace_bytes", "potts_batch_create", "potts_batch_destroy",
    "potts_batch_sweep_measured", "potts_batch_sweep_measured_dev", "potts_batch_sweep_delta", "potts_batch_ladder", "potts_batch_download", "potts_batch_sweep_count", "potts_batch_launch_count",
    "potts_set_stream_spec", "potts_get_stream_spec", "potts_batch_set_stream_spec",
    "potts_create_strip", "potts_strip_half_sweep", "potts_strip_advance", "potts_strip_rows",
    "potts3_create", "potts3_destroy", "potts3_sweep", "potts3_sweep_measured", "potts3_energy", "potts3_histogram",
    "potts3_download", "potts3_upload", "potts3_sweep_count", "potts3_set_sweep_count", "potts3_launch_count", "potts3_set_option",
    "potts8_create", "potts8_destroy", "potts8_sweep", "potts8_sweep_measured", "potts8_energy", "potts8_histogram",
    "potts8_download", "potts8_upload", "potts8_sweep_count", "potts8_set_sweep_count", "potts8_launch_count", "potts8_set_option",
    "potts_measure_noalloc",
]


def _host_series(shape) -> np.ndarray:
    """int64 host array for a series the library copies from the device: page-locked (torch's caching host allocator, so
    repeated calls reuse the pages) once it is large enough for the copy to matter -- a pageable destination takes the
    driver's bounce-buffer path at a fraction of the PCIe rate.  Marshalling only; the contents come from the kernels."""
    n = int(np.prod(shape))
    if n * 8 >= (1 << 20):
        import torch
        return torch.empty(tuple(int(x) for x in shape), dtype=torch.int64, pin_memory=True).numpy()
    return np.zeros(shape, dtype=np.int64)


def _check(rc: int):
    if rc != OK:
        raise PottsError(rc, load_library().potts_last_error().decode())


def potts_version() -> str:
    return load_library().potts_version().decode()


def potts_workspace_bytes(L: int, q: int, layout: int = LAYOUT_U8) -> int:
    n = ctypes.c_size_t(0)
    _check(load_library().potts_workspace_bytes(L, q, layout, ctypes.byref(n)))
    return int(n.value)


def potts_observables(E_series, N: int, T: float):
    """-> (mean_e, c_v, binder) in double, computed by the library on the host."""
    E = np.ascontiguousarray(E_series, dtype=np.int64)
    a, b, c = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _check(load_library().potts_observables(E.ctypes.data, E.size, int(N), float(T),
                                            ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)))
    return a.value, b.value, c.value


NOALLOC_MAX_L = 2048     # POTTS_NOALLOC_MAX_L of include/potts.h


def potts_measure_noalloc(spins, q: int, E_out=None, hist_out=None, stream: int = 0):
    """Energy and histogram of a device lattice without any allocation (include/potts.h, potts_measure_noalloc).

    spins: uint8 CUDA tensor [L, L] (contiguous); E_out: int64 CUDA tensor of 1 element or None; hist_out: int64 CUDA
    tensor of q elements or None -- all caller-owned, on the current device.  Enqueues on `stream` (a raw CUDA stream
    handle, 0 = default) and returns without synchronising."""
    L = int(spins.shape[0])
    if tuple(spins.shape) != (L, L) or not spins.is_contiguous() or not spins.is_cuda or spins.element_size() != 1:
        raise PottsError(ERR_ARG, "spins must be a contiguous uint8 CUDA tensor of shape [L, L]")
    for t, n in ((E_out, 1), (hist_out, int(q))):
        if t is not None and (not t.is_cuda or t.element_size() != 8 or t.numel() != n or not t.is_contiguous()):
            raise PottsError(ERR_ARG, "E_out / hist_out must be contiguous int64 CUDA tensors of 1 / q elements")
    _check(load_library().potts_measure_noalloc(
        ctypes.c_void_p(spins.data_ptr()), L, int(q),
        ctypes.c_void_p(E_out.data_ptr()) if E_out is not None else None,
        ctypes.c_void_p(hist_out.data_ptr()) if hist_out is not None else None, ctypes.c_void_p(int(stream))))


def potts_magnetisation(counts, q: int) -> float:
    H = np.ascontiguousarray(counts, dtype=np.int64)
    m = ctypes.c_double()
    _check(load_library().potts_magnetisation(H.ctypes.data, int(q), ctypes.byref(m)))
    return m.value


def potts_susceptibility(hist_series, q: int, T: float):
    """-> (<m>, <m^2>, chi = N/T (<m^2> - <m>^2)) from a series of histograms, computed by the library on the host."""
    H = np.ascontiguousarray(hist_series, dtype=np.int64).reshape(-1, int(q))
    a, b, c = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _check(load_library().potts_susceptibility(H.ctypes.data, H.shape[0], int(q), float(T),
                                               ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)))
    return a.value, b.value, c.value


class Potts:
    """One lattice on the current CUDA device.  Methods mirror the C entry points one to one."""

    def __init__(self, L: int, q: int, seed: int, init: int = INIT_ORDERED, layout: int = LAYOUT_U8,
                 device: Optional[int] = None):
        import torch

        self._lib = load_library()
        if not torch.cuda.is_available():
            raise PottsError(ERR_CUDA, "no CUDA device: the Potts sweep has no CPU fallback")
        self._torch = torch
        self.device = torch.device("cuda", torch.cuda.current_device() if device is None else device)
        self.L, self.q, self.seed, self.layout = int(L), int(q), int(seed), int(layout)
        nbytes = potts_workspace_bytes(self.L, self.q, self.layout)
        with torch.cuda.device(self.device):
            # device memory from torch's caching allocator; the handle borrows it
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self._ws.data_ptr()
            off = (-base) % 256
            h = ctypes.c_void_p()
            _check(self._lib.potts_create_ex(ctypes.byref(h), self.L, self.q, self.seed, int(init), self.layout,
                                             ctypes.c_void_p(base + off), nbytes, self._stream_ptr()))
        self._h = h

    # -- plumbing ---------------------------------------------------------------------------
    def _stream_ptr(self):
        return ctypes.c_void_p(self._torch.cuda.current_stream(self.device).cuda_stream)

    def _sync_stream(self):
        _check(self._lib.potts_set_stream(self._h, self._stream_ptr()))

    def close(self):
        if getattr(self, "_h", None):
            self._torch.cuda.synchronize(self.device)
            self._lib.potts_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C-ABI, name for name -------------------------------------------------------------
    def potts_sweep(self, T: float, nsweeps: int):
        self._sync_stream()
        _check(self._lib.potts_sweep(self._h, float(T), int(nsweeps)))

    def potts_sweep_measured(self, T: float, nsweeps: int, every: int = 1, hist: bool = True):
        """-> (E_series int64[n/every], hist_series int64[n/every, q] or None) on the host."""
        self._sync_stream()
        ns = int(nsweeps) // int(every) if every >= 1 and nsweeps >= 0 else 0
        E = np.zeros(ns, dtype=np.int64)
        H = np.zeros((ns, self.q), dtype=np.int64) if hist else None
        _check(self._lib.potts_sweep_measured(self._h, float(T), int(nsweeps), int(every), E.ctypes.data,
                                              H.ctypes.data if hist else None))
        return E, H

    def potts_sweep_measured_dev(self, T: float, nsweeps: int, every: int, E_dev, hist_dev=None):
        """E_dev / hist_dev: torch.int64 CUDA tensors of nsweeps/every (x q) entries; no sync."""
        self._sync_stream()
        _check(self._lib.potts_sweep_measured_dev(
            self._h, float(T), int(nsweeps), int(every),
            ctypes.c_void_p(E_dev.data_ptr()) if E_dev is not None else None,
            ctypes.c_void_p(hist_dev.data_ptr()) if hist_dev is not None else None))

    def potts_sweep_delta(self, T: float, nsweeps: int) -> np.ndarray:
        """-> dE int64[nsweeps] on the host: the energy change of each sweep summed over its accepted moves."""
        self._sync_stream()
        dE = np.zeros(int(nsweeps), dtype=np.int64)
        _check(self._lib.potts_sweep_delta(self._h, float(T), int(nsweeps), dE.ctypes.data))
        return dE

    def potts_ladder(self, temperatures, t_tran: int, t_max: int, dt: int, hist: bool = True):
        """-> (E int64[nT, t_max/dt], hist int64[nT, t_max/dt, q] or None) on the host."""
        self._sync_stream()
        T = np.ascontiguousarray(temperatures, dtype=np.float64)
        per = int(t_max) // int(dt) if dt >= 1 and t_max >= 0 else 0
        E = np.zeros((T.size, per), dtype=np.int64)
        H = np.zeros((T.size, per, self.q), dtype=np.int64) if hist else None
        _check(self._lib.potts_ladder(self._h, T.ctypes.data, int(T.size), int(t_tran), int(t_max), int(dt),
                                      E.ctypes.data, H.ctypes.data if hist else None))
        return E, H

    def potts_energy(self) -> int:
        self._sync_stream()
        E = ctypes.c_int64()
        _check(self._lib.potts_energy(self._h, ctypes.byref(E)))
        return int(E.value)

    def potts_histogram(self) -> np.ndarray:
        self._sync_stream()
        H = np.zeros(self.q, dtype=np.int64)
        _check(self._lib.potts_histogram(self._h, H.ctypes.data))
        return H

    def potts_download(self, out: Optional[np.ndarray] = None) -> np.ndarray:
        self._sync_stream()
        if out is None:
            out = np.empty((self.L, self.L), dtype=np.uint8)
        assert out.dtype == np.uint8 and out.size == self.L * self.L and out.flags.c_contiguous
        _check(self._lib.potts_download(self._h, out.ctypes.data))
        return out

    def potts_upload(self, spins: np.ndarray):
        self._sync_stream()
        a = np.ascontiguousarray(spins, dtype=np.uint8)
        if a.size != self.L * self.L:
            raise PottsError(ERR_ARG, "upload needs L*L spins")
        _check(self._lib.potts_upload(self._h, a.ctypes.data))

    def potts_sweep_count(self) -> int:
        t = ctypes.c_uint64()
        _check(self._lib.potts_sweep_count(self._h, ctypes.byref(t)))
        return int(t.value)

    def potts_set_sweep_count(self, t: int):
        _check(self._lib.potts_set_sweep_count(self._h, int(t)))

    def potts_set_stream_spec(self, spec: int):
        _check(self._lib.potts_set_stream_spec(self._h, int(spec)))

    def potts_get_stream_spec(self) -> int:
        v = ctypes.c_int32()
        _check(self._lib.potts_get_stream_spec(self._h, ctypes.byref(v)))
        return int(v.value)

    def potts_launch_count(self) -> int:
        n = ctypes.c_uint64()
        _check(self._lib.potts_launch_count(self._h, ctypes.byref(n)))
        return int(n.value)

    def potts_set_option(self, key: str, value: int):
        _check(self._lib.potts_set_option(self._h, key.encode(), int(value)))

    def potts_get_option(self, key: str) -> int:
        v = ctypes.c_int64()
        _check(self._lib.potts_get_option(self._h, key.encode(), ctypes.byref(v)))
        return int(v.value)


class PottsBatch:
    """n independent lattices of the same (L, q) advanced by one launch per call (replica batch)."""

    def __init__(self, L: int, q: int, seeds, init: int = INIT_ORDERED, device: Optional[int] = None):
        import torch

        self._lib = load_library()
        if not torch.cuda.is_available():
            raise PottsError(ERR_CUDA, "no CUDA device: the Potts sweep has no CPU fallback")
        self._torch = torch
        self.device = torch.device("cuda", torch.cuda.current_device() if device is None else device)
        self._seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
        self.n, self.L, self.q = int(self._seeds.size), int(L), int(q)
        nb = ctypes.c_size_t(0)
        _check(self._lib.potts_batch_workspace_bytes(self.n, self.L, self.q, ctypes.byref(nb)))
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nb.value + 256, dtype=torch.uint8, device=self.device)
            base = self._ws.data_ptr()
            off = (-base) % 256
            h = ctypes.c_void_p()
            stream = ctypes.c_void_p(torch.cuda.current_stream(self.device).cuda_stream)
            _check(self._lib.potts_batch_create(ctypes.byref(h), self.n, self.L, self.q, self._seeds.ctypes.data, int(init),
                                                ctypes.c_void_p(base + off), nb.value, stream))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self._torch.cuda.synchronize(self.device)
            self._lib.potts_batch_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def potts_batch_sweep_measured(self, T, nsweeps: int, every: int = 1, energy: bool = True, hist: bool = True):
        """T: one temperature per lattice.  -> (E int64[n, ns] or None, hist int64[n, ns, q] or None)."""
        Ta = np.ascontiguousarray(np.broadcast_to(np.asarray(T, dtype=np.float64), (self.n,)))
        ns = int(nsweeps) // int(every) if every >= 1 and nsweeps >= 0 else 0
        E = _host_series((self.n, ns)) if energy else None
        H = _host_series((self.n, ns, self.q)) if hist else None
        _check(self._lib.potts_batch_sweep_measured(self._h, Ta.ctypes.data, int(nsweeps), int(every),
                                                    E.ctypes.data if energy else None, H.ctypes.data if hist else None))
        return E, H

    def potts_batch_sweep_measured_dev(self, T, nsweeps: int, every: int, E_dev, hist_dev=None):
        """E_dev / hist_dev: torch.int64 CUDA tensors [n, nsweeps/every] / [n, nsweeps/every, q]; no sync."""
        Ta = np.ascontiguousarray(np.broadcast_to(np.asarray(T, dtype=np.float64), (self.n,)))
        _check(self._lib.potts_batch_sweep_measured_dev(self._h, Ta.ctypes.data, int(nsweeps), int(every),
                                                        ctypes.c_void_p(E_dev.data_ptr()) if E_dev is not None else None,
                                                        ctypes.c_void_p(hist_dev.data_ptr()) if hist_dev is not None else None))

    def potts_batch_sweep_delta(self, T, nsweeps: int) -> np.ndarray:
        """-> dE int64[n, nsweeps]: energy change of every sweep of every lattice, from its accepted moves."""
        Ta = np.ascontiguousarray(np.broadcast_to(np.asarray(T, dtype=np.float64), (self.n,)))
        dE = _host_series((self.n, int(nsweeps)))
        _check(self._lib.potts_batch_sweep_delta(self._h, Ta.ctypes.data, int(nsweeps), dE.ctypes.data))
        return dE

    def potts_batch_ladder(self, T, t_tran: int, t_max: int, dt: int, energy: bool = True, hist: bool = True):
        """T: [n, nT] (or [nT], the same ladder for every lattice).  -> (E int64[n, nT, t_max/dt], hist [..., q])."""
        Ta = np.asarray(T, dtype=np.float64)
        if Ta.ndim == 1:
            Ta = np.broadcast_to(Ta, (self.n, Ta.shape[0]))
        Ta = np.ascontiguousarray(Ta)
        nT = Ta.shape[1]
        per = int(t_max) // int(dt) if dt >= 1 else 0
        E = _host_series((self.n, nT, per)) if energy else None
        H = _host_series((self.n, nT, per, self.q)) if hist else None
        _check(self._lib.potts_batch_ladder(self._h, Ta.ctypes.data, nT, int(t_tran), int(t_max), int(dt),
                                            E.ctypes.data if energy else None, H.ctypes.data if hist else None))
        return E, H

    def potts_batch_set_stream_spec(self, spec: int):
        _check(self._lib.potts_batch_set_stream_spec(self._h, int(spec)))

    def potts_batch_download(self, r: int) -> np.ndarray:
        out = np.empty((self.L, self.L), dtype=np.uint8)
        _check(self._lib.potts_batch_download(self._h, int(r), out.ctypes.data))
        return out

    def potts_batch_sweep_count(self) -> int:
        t = ctypes.c_uint64()
        _check(self._lib.potts_batch_sweep_count(self._h, ctypes.byref(t)))
        return int(t.value)

    def potts_batch_launch_count(self) -> int:
        n = ctypes.c_uint64()
        _check(self._lib.potts_batch_launch_count(self._h, ctypes.byref(n)))
        return int(n.value)


class Potts3D:
    """One L x L x L lattice on the current CUDA device.  Methods mirror the potts3_* entry points."""

    def __init__(self, L: int, q: int, seed: int, init: int = INIT_ORDERED):
        import torch
        if not torch.cuda.is_available():
            raise PottsError(ERR_CUDA, "no CUDA device: the product has no CPU fallback")
        self._lib = load_library()
        self.L, self.q, self.seed = int(L), int(q), int(seed)
        self._stream = torch.cuda.current_stream().cuda_stream
        h = ctypes.c_void_p()
        _check(self._lib.potts3_create(ctypes.byref(h), self.L, self.q, self.seed, int(init), ctypes.c_void_p(self._stream)))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self._lib.potts3_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def potts3_sweep(self, T: float, nsweeps: int):
        _check(self._lib.potts3_sweep(self._h, float(T), int(nsweeps)))

    def potts3_sweep_measured(self, T: float, nsweeps: int, every: int = 1, hist: bool = True):
        ns = int(nsweeps) // int(every) if every >= 1 and nsweeps >= 0 else 0
        E = np.zeros(ns, dtype=np.int64)
        H = np.zeros((ns, self.q), dtype=np.int64) if hist else None
        _check(self._lib.potts3_sweep_measured(self._h, float(T), int(nsweeps), int(every), E.ctypes.data,
                                               H.ctypes.data if hist else None))
        return E, H

    def potts3_energy(self) -> int:
        E = ctypes.c_int64()
        _check(self._lib.potts3_energy(self._h, ctypes.byref(E)))
        return int(E.value)

    def potts3_histogram(self) -> np.ndarray:
        out = np.zeros(self.q, dtype=np.int64)
        _check(self._lib.potts3_histogram(self._h, out.ctypes.data))
        return out

    def potts3_download(self) -> np.ndarray:
        out = np.empty((self.L, self.L, self.L), dtype=np.uint8)
        _check(self._lib.potts3_download(self._h, out.ctypes.data))
        return out

    def potts3_upload(self, spins):
        a = np.ascontiguousarray(spins, dtype=np.uint8)
        if a.shape != (self.L, self.L, self.L):
            raise ValueError("spins must be L x L x L")
        _check(self._lib.potts3_upload(self._h, a.ctypes.data))

    def potts3_sweep_count(self) -> int:
        t = ctypes.c_uint64()
        _check(self._lib.potts3_sweep_count(self._h, ctypes.byref(t)))
        return int(t.value)

    def potts3_set_sweep_count(self, t: int):
        _check(self._lib.potts3_set_sweep_count(self._h, int(t)))

    def potts3_launch_count(self) -> int:
        n = ctypes.c_uint64()
        _check(self._lib.potts3_launch_count(self._h, ctypes.byref(n)))
        return int(n.value)

    def potts3_set_option(self, key: str, value: int):
        _check(self._lib.potts3_set_option(self._h, key.encode(), int(value)))


class Potts8:
    """One L x L lattice with first and second neighbour interactions on the current CUDA device.  Methods mirror the potts8_* entry points."""

    def __init__(self, L: int, q: int, seed: int, init: int = INIT_ORDERED):
        import torch
        if not torch.cuda.is_available():
            raise PottsError(ERR_CUDA, "no CUDA device: the product has no CPU fallback")
        self._lib = load_library()
        self.L, self.q, self.seed = int(L), int(q), int(seed)
        self._stream = torch.cuda.current_stream().cuda_stream
        h = ctypes.c_void_p()
        _check(self._lib.potts8_create(ctypes.byref(h), self.L, self.q, self.seed, int(init), ctypes.c_void_p(self._stream)))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self._lib.potts8_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def potts8_sweep(self, T: float, nsweeps: int):
        _check(self._lib.potts8_sweep(self._h, float(T), int(nsweeps)))

    def potts8_sweep_measured(self, T: float, nsweeps: int, every: int = 1, hist: bool = True):
        ns = int(nsweeps) // int(every) if every >= 1 and nsweeps >= 0 else 0
        E = np.zeros(ns, dtype=np.int64)
        H = np.zeros((ns, self.q), dtype=np.int64) if hist else None
        _check(self._lib.potts8_sweep_measured(self._h, float(T), int(nsweeps), int(every), E.ctypes.data,
                                               H.ctypes.data if hist else None))
        return E, H

    def potts8_energy(self) -> int:
        E = ctypes.c_int64()
        _check(self._lib.potts8_energy(self._h, ctypes.byref(E)))
        return int(E.value)

    def potts8_histogram(self) -> np.ndarray:
        out = np.zeros(self.q, dtype=np.int64)
        _check(self._lib.potts8_histogram(self._h, out.ctypes.data))
        return out

    def potts8_download(self) -> np.ndarray:
        out = np.empty((self.L, self.L), dtype=np.uint8)
        _check(self._lib.potts8_download(self._h, out.ctypes.data))
        return out

    def potts8_upload(self, spins):
        a = np.ascontiguousarray(spins, dtype=np.uint8)
        if a.shape != (self.L, self.L):
            raise ValueError("spins must be L x L")
        _check(self._lib.potts8_upload(self._h, a.ctypes.data))

    def potts8_sweep_count(self) -> int:
        t = ctypes.c_uint64()
        _check(self._lib.potts8_sweep_count(self._h, ctypes.byref(t)))
        return int(t.value)

    def potts8_set_sweep_count(self, t: int):
        _check(self._lib.potts8_set_sweep_count(self._h, int(t)))

    def potts8_launch_count(self) -> int:
        n = ctypes.c_uint64()
        _check(self._lib.potts8_launch_count(self._h, ctypes.byref(n)))
        return int(n.value)

    def potts8_set_option(self, key: str, value: int):
        _check(self._lib.potts8_set_option(self._h, key.encode(), int(value)))
