"""One lattice split into row strips over several GPUs: host-side driver of the potts_strip_* calls.

The random words are a pure function of the GLOBAL site (seed, t, colour, i, j), so n strips together follow exactly
the chain of one ``Potts`` handle whatever n is.  The only data that crosses strips are the two boundary rows of the
plane a half-sweep has just written: L/2 bytes to the strip above and L/2 bytes to the strip below, twice per sweep.

Two transports over the same exchange rule:

* ``LocalStrips``: n strips in ONE process on one GPU, rows copied device to device.  This is how the strip form of the
  kernels is parity-tested on the one-GPU box (no rank waits for another: one stream, launches in order).
* ``RankStrip``: one strip per rank of a ``torch.distributed`` group (NCCL between GPUs; any backend that can send and
  receive the tensors the compute side hands out).  Energy and histogram are all-reduced sums of per-strip parts.

The compute side is anything with the small interface of ``GpuStrip`` (half_sweep / advance / rows / ...); the CPU
tests drive the same exchange code with a stand-in built on the oracle, over gloo with world_size 2.
"""
from __future__ import annotations

import ctypes
from typing import List, Tuple

import numpy as np

from . import binding as _b


def partition(L: int, n: int) -> List[Tuple[int, int]]:
    """Rows [row0, row0 + rows) of strip r = 0..n-1: contiguous, both ends multiples of 32, sizes as even as that allows."""
    if L % 32 or n < 1 or n > L // 32:
        raise ValueError(f"cannot split L = {L} into {n} strips of whole 32-row tiles")
    tiles = L // 32
    out, row0 = [], 0
    for r in range(n):
        rows = 32 * (tiles // n + (1 if r < tiles % n else 0))
        out.append((row0, rows))
        row0 += rows
    return out


def neighbours(r: int, n: int) -> Tuple[int, int]:
    """(strip above, strip below) of strip r on the periodic lattice."""
    return (r - 1) % n, (r + 1) % n


class _DevBytes:
    """A device address range exposed through __cuda_array_interface__ so that torch can wrap it without a copy."""

    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (int(ptr), False), "version": 3}


class GpuStrip:
    """Rows [row0, row0 + rows) of an L x L lattice on the current CUDA device (potts_create_strip)."""

    def __init__(self, L: int, q: int, seed: int, init: int, row0: int, rows: int):
        import torch
        if not torch.cuda.is_available():
            raise _b.PottsError(_b.ERR_CUDA, "no CUDA device: the product has no CPU fallback")
        self._torch, self._lib = torch, _b.load_library()
        self.L, self.q, self.row0, self.nrows = int(L), int(q), int(row0), int(rows)
        h = ctypes.c_void_p()
        stream = torch.cuda.current_stream().cuda_stream
        _b._check(self._lib.potts_create_strip(ctypes.byref(h), self.L, self.q, int(seed), int(init), self.row0, self.nrows,
                                               ctypes.c_void_p(stream)))
        self._h = h
        self._acc = torch.zeros(1 + self.q, dtype=torch.int64, device="cuda")
        self._rows = [self._row_tensors(c) for c in (0, 1)]

    def _row_tensors(self, colour: int):
        p = [ctypes.c_void_p() for _ in range(4)]
        n = ctypes.c_size_t()
        _b._check(self._lib.potts_strip_rows(self._h, colour, *[ctypes.byref(x) for x in p], ctypes.byref(n)))
        return tuple(self._torch.as_tensor(_DevBytes(x.value, n.value), device="cuda") for x in p)

    def close(self):
        if getattr(self, "_h", None):
            self._torch.cuda.synchronize()
            self._lib.potts_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def rows(self, colour: int):
        """(first row, last row, halo above, halo below) of plane `colour`: uint8 tensors of L/2 bytes, views of the handle's memory."""
        return self._rows[colour]

    def half_sweep(self, T: float, colour: int, sample: bool = False):
        """One half-sweep; sample: add this strip's part of the energy (colour 1) and histogram to the accumulators."""
        E = ctypes.c_void_p(self._acc.data_ptr()) if (sample and colour == 1) else None
        H = ctypes.c_void_p(self._acc.data_ptr() + 8) if sample else None
        _b._check(self._lib.potts_strip_half_sweep(self._h, float(T), int(colour), E, H))

    def advance(self):
        _b._check(self._lib.potts_strip_advance(self._h))

    def take_sample(self):
        """-> int64 tensor [E_part, hist_part...] accumulated since the last call (device), accumulators zeroed."""
        out = self._acc.clone()
        self._acc.zero_()
        return out

    def energy_histogram_parts(self):
        """Standalone partial sums over the strip (the halos of plane 0 must be current): int64 tensor [E, hist...] on the device."""
        E = ctypes.c_int64()
        _b._check(self._lib.potts_energy(self._h, ctypes.byref(E)))
        H = np.zeros(self.q, dtype=np.int64)
        _b._check(self._lib.potts_histogram(self._h, H.ctypes.data))
        return self._torch.tensor([E.value] + [int(x) for x in H], dtype=self._torch.int64, device="cuda")

    def download(self) -> np.ndarray:
        out = np.empty((self.nrows, self.L), dtype=np.uint8)
        _b._check(self._lib.potts_download(self._h, out.ctypes.data))
        return out


# ---- the exchange rule, shared by both transports ---------------------------------------------------------------
def exchange_local(strips, colour: int):
    """After the half-sweep of `colour` on every strip of this process: boundary rows into the neighbours' halos."""
    n = len(strips)
    for r, s in enumerate(strips):
        first, last, _, _ = s.rows(colour)
        up, dn = neighbours(r, n)
        strips[up].rows(colour)[3].copy_(first)      # my first row is the row below the strip above
        strips[dn].rows(colour)[2].copy_(last)       # my last row is the row above the strip below


def exchange_ranks(strip, colour: int, dist, rank: int, world: int, group=None):
    """The same between ranks: two sends and two receives per rank (one of each if world == 2 merges nothing: the two
    neighbours are the same rank but the rows are different, so tags by direction keep them apart)."""
    first, last, halo_above, halo_below = strip.rows(colour)
    if world == 1:
        halo_below.copy_(first)
        halo_above.copy_(last)
        return
    up, dn = neighbours(rank, world)
    ops = [dist.P2POp(dist.isend, first, up, group=group, tag=0), dist.P2POp(dist.isend, last, dn, group=group, tag=1),
           dist.P2POp(dist.irecv, halo_below, dn, group=group, tag=0), dist.P2POp(dist.irecv, halo_above, up, group=group, tag=1)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()


class LocalStrips:
    """n strips of one lattice in this process; same results as one Potts handle."""

    def __init__(self, L: int, q: int, seed: int, init: int, n: int, make_strip=GpuStrip):
        self.L, self.q = int(L), int(q)
        self.strips = [make_strip(L, q, seed, init, row0, rows) for row0, rows in partition(L, n)]
        for c in (0, 1):
            exchange_local(self.strips, c)

    def sweep(self, T: float, nsweeps: int, every: int = 0):
        """-> (E int64[n/every], hist int64[n/every, q]) if every > 0 else None."""
        E, H = [], []
        for k in range(int(nsweeps)):
            sample = every > 0 and (k + 1) % every == 0
            for c in (0, 1):
                for s in self.strips:
                    s.half_sweep(T, c, sample)
                exchange_local(self.strips, c)
            for s in self.strips:
                s.advance()
            if sample:
                tot = sum(s.take_sample() for s in self.strips)
                E.append(int(tot[0])); H.append([int(x) for x in tot[1:]])
        if every > 0:
            return np.asarray(E, dtype=np.int64), np.asarray(H, dtype=np.int64).reshape(-1, self.q)
        return None

    def energy_histogram(self):
        tot = sum(s.energy_histogram_parts() for s in self.strips)
        return int(tot[0]), np.asarray([int(x) for x in tot[1:]], dtype=np.int64)

    def download(self) -> np.ndarray:
        return np.concatenate([s.download() for s in self.strips], axis=0)

    def close(self):
        for s in self.strips:
            s.close()


class RankStrip:
    """This rank's strip of a lattice split over a torch.distributed group; every rank calls the same methods."""

    def __init__(self, L: int, q: int, seed: int, init: int, dist, group=None, make_strip=GpuStrip):
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.L, self.q = int(L), int(q)
        row0, rows = partition(L, self.world)[self.rank]
        self.strip = make_strip(L, q, seed, init, row0, rows)
        for c in (0, 1):
            exchange_ranks(self.strip, c, dist, self.rank, self.world, group)

    def sweep(self, T: float, nsweeps: int, every: int = 0):
        E, H = [], []
        for k in range(int(nsweeps)):
            sample = every > 0 and (k + 1) % every == 0
            for c in (0, 1):
                self.strip.half_sweep(T, c, sample)
                exchange_ranks(self.strip, c, self.dist, self.rank, self.world, self.group)
            self.strip.advance()
            if sample:
                tot = self.strip.take_sample()
                self.dist.all_reduce(tot, group=self.group)          # energy and histogram are sums over the strips
                E.append(int(tot[0])); H.append([int(x) for x in tot[1:]])
        if every > 0:
            return np.asarray(E, dtype=np.int64), np.asarray(H, dtype=np.int64).reshape(-1, self.q)
        return None

    def energy_histogram(self):
        tot = self.strip.energy_histogram_parts()
        self.dist.all_reduce(tot, group=self.group)
        return int(tot[0]), np.asarray([int(x) for x in tot[1:]], dtype=np.int64)

    def download_strip(self) -> np.ndarray:
        return self.strip.download()

    def close(self):
        self.strip.close()
