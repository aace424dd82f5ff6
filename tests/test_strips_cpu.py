"""Host logic of the row-strip decomposition (paper_1101_0876_b200/strips.py) on CPU, -m "not gpu".

The product's exchange code (partition, neighbours, exchange_local, exchange_ranks, LocalStrips, RankStrip) is driven
here with a stand-in for the compute side built on the ORACLE's single-site rule (test infrastructure: the product
never sees it), so that what is tested is exactly what a multi-GPU run adds: which rows go where, in which order, and
the all-reduce of the partial sums.  Two strips / two gloo ranks must reproduce the single-lattice oracle bit for bit.
"""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import workloads
from paper_1101_0876_b200 import strips


class OracleStrip:
    """Rows [row0, row0 + rows) of the lattice plus one halo row above and below, advanced with oracle.update_site."""

    def __init__(self, L, q, seed, init, row0, rows):
        self.L, self.q, self.seed, self.row0, self.nrows, self.t = L, q, seed, row0, rows, 0
        full = oracle.OraclePotts(L, q, seed, init).spins()          # the start state is a pure function of the site
        self.s = np.zeros((rows + 2, L), dtype=np.uint8)
        self.s[1:-1] = full[row0:row0 + rows]
        # per colour: first row, last row, halo above, halo below (the sites of that colour only: L/2 bytes each)
        self.buf = [[torch.zeros(L // 2, dtype=torch.uint8) for _ in range(4)] for _ in (0, 1)]
        self.acc = torch.zeros(1 + q, dtype=torch.int64)
        for c in (0, 1):
            self._pack(c)

    def _cols(self, global_row, colour):
        return np.arange((global_row + colour) & 1, self.L, 2)

    def _pack(self, c):
        self.buf[c][0][:] = torch.from_numpy(self.s[1, self._cols(self.row0, c)].copy())
        self.buf[c][1][:] = torch.from_numpy(self.s[self.nrows, self._cols(self.row0 + self.nrows - 1, c)].copy())

    def _unpack_halos(self):
        for c in (0, 1):
            self.s[0, self._cols(self.row0 - 1, c)] = self.buf[c][2].numpy()
            self.s[self.nrows + 1, self._cols(self.row0 + self.nrows, c)] = self.buf[c][3].numpy()

    def rows(self, colour):
        return tuple(self.buf[colour])

    def half_sweep(self, T, colour, sample=False):
        self._unpack_halos()
        L, src = self.L, self.s.copy()
        for r in range(1, self.nrows + 1):
            i = self.row0 + r - 1
            for j in range((i + colour) & 1, L, 2):
                nb = [src[r - 1, j], src[r + 1, j], src[r, (j - 1) % L], src[r, (j + 1) % L]]
                self.s[r, j] = oracle.update_site(i, j, self.t, colour, self.seed, self.q, T, src[r, j], nb)
        self._pack(colour)
        if sample:
            own = np.concatenate([self.s[r, self._cols(self.row0 + r - 1, colour)] for r in range(1, self.nrows + 1)])
            self.acc[1:] += torch.from_numpy(np.bincount(own, minlength=self.q).astype(np.int64))
            if colour == 1:                                           # energy from the colour-1 sites (every bond joins the colours)
                e = 0
                for r in range(1, self.nrows + 1):
                    for j in self._cols(self.row0 + r - 1, 1):
                        v = self.s[r, j]
                        e += int(self.s[r - 1, j] == v) + int(self.s[r + 1, j] == v) + int(self.s[r, (j - 1) % L] == v) + int(self.s[r, (j + 1) % L] == v)
                self.acc[0] -= e

    def advance(self):
        self.t += 1

    def take_sample(self):
        out = self.acc.clone()
        self.acc.zero_()
        return out

    def download(self):
        return self.s[1:-1].copy()

    def close(self):
        pass


def test_partition_and_neighbours():
    assert strips.partition(128, 1) == [(0, 128)]
    assert strips.partition(128, 3) == [(0, 64), (64, 32), (96, 32)]
    assert strips.partition(32768, 8) == [(4096 * r, 4096) for r in range(8)]
    for L, n in ((96, 3), (4096, 7), (1024, 32)):
        p = strips.partition(L, n)
        assert p[0][0] == 0 and sum(r for _, r in p) == L and all(a % 32 == 0 and r % 32 == 0 and r > 0 for a, r in p)
        assert all(p[k][0] + p[k][1] == p[k + 1][0] for k in range(n - 1))
    with pytest.raises(ValueError):
        strips.partition(64, 3)
    assert strips.neighbours(0, 4) == (3, 1) and strips.neighbours(3, 4) == (2, 0) and strips.neighbours(0, 1) == (0, 0)


@pytest.mark.parametrize("n", [1, 2])
def test_local_strips_reproduce_the_single_lattice_chain(n):
    L, q, seed = 64, 5, 12
    T = 0.95 * workloads.t_c(q)
    o = oracle.OraclePotts(L, q, seed, workloads.INIT_RANDOM)
    run = strips.LocalStrips(L, q, seed, workloads.INIT_RANDOM, n, make_strip=OracleStrip)
    E, H = run.sweep(T, 3, every=1)
    Eo, Ho = o.sweep_measured(T, 3, 1, hist=True)
    assert (E == Eo).all() and (H == Ho).all()
    assert (run.download() == o.spins()).all()


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    L, qq, seed = 64, 4, 3
    T = 1.02 * workloads.t_c(qq)
    run = strips.RankStrip(L, qq, seed, workloads.INIT_RANDOM, dist, make_strip=OracleStrip)
    E, H = run.sweep(T, 3, every=1)
    q.put((rank, run.strip.row0, [int(x) for x in E], H.tolist(), run.download_strip().tolist()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_gloo_ranks_one_lattice():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=600) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    L, qq, seed = 64, 4, 3
    T = 1.02 * workloads.t_c(qq)
    o = oracle.OraclePotts(L, qq, seed, workloads.INIT_RANDOM)
    Eo, Ho = o.sweep_measured(T, 3, 1, hist=True)
    assert [r[1] for r in res] == [0, 32]
    for _, _, E, H, _ in res:                                         # every rank holds the all-reduced series
        assert E == [int(x) for x in Eo] and H == Ho.tolist()
    assert (np.concatenate([np.asarray(r[4], dtype=np.uint8) for r in res], axis=0) == o.spins()).all()
