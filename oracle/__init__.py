"""CPU oracle for the checkerboard Potts sweep of arXiv 1101.0876 -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_1101_0876_b200``) never does, and this package never imports the product.

``potts_oracle.c`` holds the method (Philox4x32-10, thresholds, red/black Metropolis sweep,
energy, histogram; PAPER.md:46 Eq. 1, :94, :145, :175).  This module only builds it with gcc
and marshals arguments through ctypes.  ``observables.py`` holds the host-side derived
quantities (PAPER.md:73 Eq. 7, :209 Eq. 9) in exact integer arithmetic.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "potts_oracle.c")
_SRC3 = os.path.join(_HERE, "potts3d_oracle.c")       # the 3D generalisation, same library
_SRC8 = os.path.join(_HERE, "potts8_oracle.c")        # first + second neighbours, nine sub-networks
_LIB = os.path.join(_HERE, "libpotts_oracle.so")
_lock = threading.Lock()
_lib = None

INIT_ORDERED = 0
INIT_RANDOM = 1


def build(force: bool = False) -> str:
    """Compile potts_oracle.c -> libpotts_oracle.so (plain -O2, OpenMP for the optional row-parallel mode)."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC3), os.path.getmtime(_SRC8)):
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.check_call(
                ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
                 "-o", tmp, _SRC, _SRC3, _SRC8, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u8p = ctypes.POINTER(ctypes.c_uint8)
        u32p = ctypes.POINTER(ctypes.c_uint32)
        i64p = ctypes.POINTER(ctypes.c_int64)
        vp = ctypes.c_void_p
        lib.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        lib.oracle_philox4x32_10.restype = None
        lib.oracle_thresholds.argtypes = [ctypes.c_double, u32p]
        lib.oracle_thresholds.restype = None
        lib.oracle_create.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_uint64, ctypes.c_int32]
        lib.oracle_create.restype = vp
        lib.oracle_destroy.argtypes = [vp]
        lib.oracle_destroy.restype = None
        lib.oracle_set_threads.argtypes = [vp, ctypes.c_int]
        lib.oracle_set_threads.restype = None
        lib.oracle_get_threads.argtypes = [vp]
        lib.oracle_get_threads.restype = ctypes.c_int
        lib.oracle_sweep.argtypes = [vp, ctypes.c_double, ctypes.c_int64]
        lib.oracle_sweep.restype = ctypes.c_int
        lib.oracle_sweep_measured.argtypes = [vp, ctypes.c_double, ctypes.c_int64, ctypes.c_int64, i64p, i64p]
        lib.oracle_sweep_measured.restype = ctypes.c_int
        lib.oracle_energy.argtypes = [vp]
        lib.oracle_energy.restype = ctypes.c_int64
        lib.oracle_energy_incremental.argtypes = [vp]
        lib.oracle_energy_incremental.restype = ctypes.c_int64
        lib.oracle_histogram.argtypes = [vp, i64p]
        lib.oracle_histogram.restype = None
        lib.oracle_spins.argtypes = [vp]
        lib.oracle_spins.restype = u8p
        lib.oracle_sweep_count.argtypes = [vp]
        lib.oracle_sweep_count.restype = ctypes.c_uint64
        lib.oracle_set_state.argtypes = [vp, u8p, ctypes.c_uint64]
        lib.oracle_set_state.restype = ctypes.c_int
        lib.oracle_update_site.argtypes = [ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32,
                                           ctypes.c_uint64, ctypes.c_uint32, ctypes.c_double, ctypes.c_uint8, u8p]
        lib.oracle_update_site.restype = ctypes.c_uint8
        lib.oracle_update_site_s.argtypes = lib.oracle_update_site.argtypes + [ctypes.c_int]
        lib.oracle_update_site_s.restype = ctypes.c_uint8
        lib.oracle_set_stream.argtypes = [vp, ctypes.c_int]
        lib.oracle_set_stream.restype = ctypes.c_int
        lib.oracle3_thresholds.argtypes = [ctypes.c_double, u32p]
        lib.oracle3_thresholds.restype = None
        lib.oracle3_create.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_uint64, ctypes.c_int32]
        lib.oracle3_create.restype = vp
        lib.oracle3_destroy.argtypes = [vp]
        lib.oracle3_destroy.restype = None
        lib.oracle3_set_threads.argtypes = [vp, ctypes.c_int]
        lib.oracle3_set_threads.restype = None
        lib.oracle3_sweep.argtypes = [vp, ctypes.c_double, ctypes.c_int64]
        lib.oracle3_sweep.restype = ctypes.c_int
        lib.oracle3_sweep_measured.argtypes = [vp, ctypes.c_double, ctypes.c_int64, ctypes.c_int64, i64p, i64p]
        lib.oracle3_sweep_measured.restype = ctypes.c_int
        lib.oracle3_energy.argtypes = [vp]
        lib.oracle3_energy.restype = ctypes.c_int64
        lib.oracle3_energy_incremental.argtypes = [vp]
        lib.oracle3_energy_incremental.restype = ctypes.c_int64
        lib.oracle3_histogram.argtypes = [vp, i64p]
        lib.oracle3_histogram.restype = None
        lib.oracle3_spins.argtypes = [vp]
        lib.oracle3_spins.restype = u8p
        lib.oracle3_sweep_count.argtypes = [vp]
        lib.oracle3_sweep_count.restype = ctypes.c_uint64
        lib.oracle3_set_state.argtypes = [vp, u8p, ctypes.c_uint64]
        lib.oracle3_set_state.restype = ctypes.c_int
        lib.oracle8_thresholds.argtypes = [ctypes.c_double, u32p]
        lib.oracle8_thresholds.restype = None
        lib.oracle8_create.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_uint64, ctypes.c_int32]
        lib.oracle8_create.restype = vp
        lib.oracle8_destroy.argtypes = [vp]
        lib.oracle8_destroy.restype = None
        lib.oracle8_set_threads.argtypes = [vp, ctypes.c_int]
        lib.oracle8_set_threads.restype = None
        lib.oracle8_sweep.argtypes = [vp, ctypes.c_double, ctypes.c_int64]
        lib.oracle8_sweep.restype = ctypes.c_int
        lib.oracle8_sweep_measured.argtypes = [vp, ctypes.c_double, ctypes.c_int64, ctypes.c_int64, i64p, i64p]
        lib.oracle8_sweep_measured.restype = ctypes.c_int
        lib.oracle8_energy.argtypes = [vp]
        lib.oracle8_energy.restype = ctypes.c_int64
        lib.oracle8_energy_incremental.argtypes = [vp]
        lib.oracle8_energy_incremental.restype = ctypes.c_int64
        lib.oracle8_histogram.argtypes = [vp, i64p]
        lib.oracle8_histogram.restype = None
        lib.oracle8_spins.argtypes = [vp]
        lib.oracle8_spins.restype = u8p
        lib.oracle8_sweep_count.argtypes = [vp]
        lib.oracle8_sweep_count.restype = ctypes.c_uint64
        lib.oracle8_set_state.argtypes = [vp, u8p, ctypes.c_uint64]
        lib.oracle8_set_state.restype = ctypes.c_int
        _lib = lib
    return _lib


def philox4x32_10(ctr, key):
    """Known-answer entry point: ctr = 4 uint32, key = 2 uint32 -> 4 uint32 (R3)."""
    lib = _load()
    c = (ctypes.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (ctypes.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (ctypes.c_uint32 * 4)()
    lib.oracle_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def thresholds(T: float):
    """[thr(1), thr(2), thr(3), thr(4)] = floor(2^32 exp(-d/T)) (R6)."""
    lib = _load()
    o = (ctypes.c_uint32 * 5)()
    lib.oracle_thresholds(float(T), o)
    return [int(o[d]) for d in range(1, 5)]


def update_site(i, j, t, colour, seed, q, T, s_old, nb, stream=1):
    """New spin of site (i,j) in half-sweep (t, colour) given its 4 neighbours (up, down, left, right)."""
    lib = _load()
    a = (ctypes.c_uint8 * 4)(*[int(x) for x in nb])
    return int(lib.oracle_update_site_s(int(i), int(j), int(t) & 0xFFFFFFFF, int(colour), int(seed), int(q),
                                        float(T), int(s_old), a, int(stream)))


class OraclePotts:
    """One lattice held by the C oracle.  Mirrors the call sequence of the product's C-ABI."""

    def __init__(self, L: int, q: int, seed: int, init: int, threads: int = 1, stream: int = 1):
        self._lib = _load()
        self._h = self._lib.oracle_create(int(L), int(q), int(seed), int(init))
        if not self._h:
            raise ValueError(f"oracle_create rejected L={L} q={q} init={init}")
        self.L, self.q, self.seed = int(L), int(q), int(seed)
        self._lib.oracle_set_threads(self._h, int(threads))
        self.stream = int(stream)
        if self._lib.oracle_set_stream(self._h, self.stream):
            raise ValueError(f"oracle_set_stream rejected stream={stream} for L={L}")

    def close(self):
        if self._h:
            self._lib.oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def threads(self) -> int:
        return int(self._lib.oracle_get_threads(self._h))

    def set_threads(self, n: int):
        self._lib.oracle_set_threads(self._h, int(n))

    @property
    def t(self) -> int:
        return int(self._lib.oracle_sweep_count(self._h))

    def sweep(self, T: float, nsweeps: int):
        rc = self._lib.oracle_sweep(self._h, float(T), int(nsweeps))
        if rc:
            raise ValueError(f"oracle_sweep rc={rc}")

    def sweep_measured(self, T: float, nsweeps: int, every: int = 1, hist: bool = True):
        """-> (E_series[n/every], hist_series[n/every, q] or None); raises if an invariant broke."""
        n = int(nsweeps) // int(every) if every >= 1 else 0
        E = np.zeros(n, dtype=np.int64)
        H = np.zeros((n, self.q), dtype=np.int64) if hist else None
        i64p = ctypes.POINTER(ctypes.c_int64)
        rc = self._lib.oracle_sweep_measured(
            self._h, float(T), int(nsweeps), int(every), E.ctypes.data_as(i64p),
            H.ctypes.data_as(i64p) if hist else None)
        if rc == 2:
            raise AssertionError("oracle bookkeeping invariant broke (E_inc != E or sum(hist) != L^2)")
        if rc:
            raise ValueError(f"oracle_sweep_measured rc={rc}")
        return E, H

    def energy(self) -> int:
        return int(self._lib.oracle_energy(self._h))

    def energy_incremental(self) -> int:
        return int(self._lib.oracle_energy_incremental(self._h))

    def histogram(self) -> np.ndarray:
        H = np.zeros(self.q, dtype=np.int64)
        self._lib.oracle_histogram(self._h, H.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)))
        return H

    def spins(self) -> np.ndarray:
        """Copy of the L x L uint8 configuration, row-major s[i, j]."""
        p = self._lib.oracle_spins(self._h)
        return np.ctypeslib.as_array(p, shape=(self.L, self.L)).copy()

    def set_state(self, spins: np.ndarray, t: int):
        a = np.ascontiguousarray(spins, dtype=np.uint8).reshape(self.L, self.L)
        rc = self._lib.oracle_set_state(self._h, a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)), int(t))
        if rc:
            raise ValueError("oracle_set_state rejected the configuration")


def thresholds3(T: float):
    """[thr(1) .. thr(6)] = floor(2^32 exp(-d/T)) for the 3D lattice (R6')."""
    lib = _load()
    o = (ctypes.c_uint32 * 7)()
    lib.oracle3_thresholds(float(T), o)
    return [int(o[d]) for d in range(1, 7)]


class OraclePotts3D:
    """The 3D (simple-cubic, 6 neighbours) checkerboard chain of potts3d_oracle.c; spins()[z, y, x]."""

    def __init__(self, L: int, q: int, seed: int, init: int, threads: int = 1):
        self._lib = _load()
        self.L, self.q, self.seed = int(L), int(q), int(seed)
        self._h = self._lib.oracle3_create(self.L, self.q, self.seed, int(init))
        if not self._h:
            raise ValueError(f"bad arguments L={L} q={q} init={init}")
        self._lib.oracle3_set_threads(self._h, int(threads))

    def close(self):
        if getattr(self, "_h", None):
            self._lib.oracle3_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def t(self) -> int:
        return int(self._lib.oracle3_sweep_count(self._h))

    def sweep(self, T: float, nsweeps: int):
        if self._lib.oracle3_sweep(self._h, float(T), int(nsweeps)):
            raise ValueError("bad arguments to sweep")

    def sweep_measured(self, T: float, nsweeps: int, every: int = 1, hist: bool = True):
        ns = int(nsweeps) // int(every)
        E = np.zeros(ns, dtype=np.int64)
        H = np.zeros((ns, self.q), dtype=np.int64) if hist else None
        i64p = ctypes.POINTER(ctypes.c_int64)
        rc = self._lib.oracle3_sweep_measured(self._h, float(T), int(nsweeps), int(every), E.ctypes.data_as(i64p),
                                              H.ctypes.data_as(i64p) if hist else None)
        if rc:
            raise ValueError("bad arguments to sweep_measured")
        return E, H

    def energy(self) -> int:
        return int(self._lib.oracle3_energy(self._h))

    def energy_incremental(self) -> int:
        return int(self._lib.oracle3_energy_incremental(self._h))

    def histogram(self) -> np.ndarray:
        out = np.zeros(self.q, dtype=np.int64)
        self._lib.oracle3_histogram(self._h, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)))
        return out

    def spins(self) -> np.ndarray:
        p = self._lib.oracle3_spins(self._h)
        return np.ctypeslib.as_array(p, shape=(self.L, self.L, self.L)).copy()

    def set_state(self, spins: np.ndarray, t: int):
        a = np.ascontiguousarray(spins, dtype=np.uint8)
        assert a.shape == (self.L, self.L, self.L)
        if self._lib.oracle3_set_state(self._h, a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)), int(t)):
            raise ValueError("spin value >= q")


def thresholds8(T: float):
    """[thr(1) .. thr(8)] = floor(2^32 exp(-d/T)) for the 8-neighbour model (R6")."""
    lib = _load()
    o = (ctypes.c_uint32 * 9)()
    lib.oracle8_thresholds(float(T), o)
    return [int(o[d]) for d in range(1, 9)]


class OraclePotts8(OraclePotts3D):
    """The 2D chain with first and second neighbours, nine sub-networks (potts8_oracle.c); spins()[i, j]."""

    def __init__(self, L: int, q: int, seed: int, init: int, threads: int = 1):
        self._lib = _Prefixed(_load(), "oracle8_")
        self.L, self.q, self.seed = int(L), int(q), int(seed)
        self._h = self._lib.oracle3_create(self.L, self.q, self.seed, int(init))
        if not self._h:
            raise ValueError(f"bad arguments L={L} q={q} init={init}")
        self._lib.oracle3_set_threads(self._h, int(threads))

    def spins(self) -> np.ndarray:
        p = self._lib.oracle3_spins(self._h)
        return np.ctypeslib.as_array(p, shape=(self.L, self.L)).copy()

    def set_state(self, spins: np.ndarray, t: int):
        a = np.ascontiguousarray(spins, dtype=np.uint8)
        assert a.shape == (self.L, self.L)
        if self._lib.oracle3_set_state(self._h, a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)), int(t)):
            raise ValueError("spin value >= q")


class _Prefixed:
    """Lets OraclePotts8 reuse OraclePotts3D's marshalling: oracle3_xyz -> oracle8_xyz of the same library."""

    def __init__(self, lib, prefix):
        self._lib, self._prefix = lib, prefix

    def __getattr__(self, name):
        return getattr(self._lib, name.replace("oracle3_", self._prefix))
