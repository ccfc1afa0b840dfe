"""World-size-2 `gloo` test of the packet-sharding host logic (paper_1201_3588_b200/sharding.py,
SURVEY.md 8(e)) on CPU.  The engine behind the runner is the fp64 oracle (tests may use it);
on a GPU box the same runner drives mcrt.Context.  Integer tallies commute, so the sharded run
must equal the single-rank run over the same packet ids BIT FOR BIT (tallies, SED, counters,
temperatures)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1201_3588_b200 import workloads as W          # noqa: E402
from paper_1201_3588_b200.sharding import ShardedRunner, rank_range   # noqa: E402

BATCHES = [(0, 5001), (5001, 4000), (9001, 2999)]       # odd sizes: ragged split over 2 ranks


class OracleEngine:
    """Adapter with the binding's call names (run_batch / transport_batch_delta /
    accumulate_update / get_cell_energy).  Like the library after a sharded batch, it keeps the
    GLOBAL cumulative tally (`glob`): the oracle's own tally holds this rank's packets only."""

    def __init__(self, wl, pah=None):
        from oracle import oracle as O
        self.o = O.Oracle(wl)
        self.pah = pah is not None
        if self.pah:
            self.o.set_pah(pah.n_C, pah.mass_fraction, pah.kabs, pah.theta_K, pah.T_lo, pah.T_hi, pah.n_Tp)
            self.glob_pah = np.zeros((self.o.slots, self.o.nb), dtype=np.uint64)
        self.glob = np.zeros(self.o.slots, dtype=np.uint64)
        self.sharded = False

    def run_batch(self, seed, first, n, stream=None):
        self.o.run_batch(seed, first, n, 1)

    def transport_batch_delta(self, seed, first, n, stream=None):
        before = self.o.cell_energy()[0]
        before_pah = self.o.pah_absorbed()[0] if self.pah else None
        self.o.transport_batch(seed, first, n, 1)
        delta = self.o.cell_energy()[0] - before
        assert delta.max(initial=0) < 2 ** 31
        if self.pah:            # like mcrt_delta_words: the PAH's absorbed spectrum of every leaf behind the counts
            delta = np.concatenate([delta, (self.o.pah_absorbed()[0] - before_pah).ravel()])
        return torch.from_numpy(delta.astype(np.int32))

    def accumulate_update(self, delta_sum, n_cum, stream=None):
        self.sharded = True
        d = delta_sum.numpy().astype(np.uint64)
        self.glob += d[:self.o.slots]
        self.o.update_temperature(self.glob, n_cum)
        if self.pah:
            self.glob_pah += d[self.o.slots:].reshape(self.glob_pah.shape)
            self.o.pah_update(self.glob_pah, n_cum)

    def get_cell_energy(self, device=False):
        n, eps = self.o.cell_energy()
        return torch.from_numpy((self.glob if self.sharded else n).astype(np.int64)), eps


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _pah_case():
    wl = W.sphere(n_root=8, tau_v=2.0, gval=0.3, n_bins=24, n_packets=12_000, batch=4_000)
    pah = W.pah_share(wl, n_C=100, mass_fraction=0.04)
    pah.n_Tp = 24
    return wl, pah


def _worker(rank, world, port, out_dir, with_pah=False):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl, pah = _pah_case() if with_pah else (W.c0(), None)
        eng = OracleEngine(wl, pah)
        run = ShardedRunner(eng, dist)
        assert run.world == world and run.rank == rank
        mine = []
        for first, n in BATCHES:
            mine.append(run.run_batch(wl.seed, first, n))
        tally, _ = eng.get_cell_energy()                 # already the global tally on every rank
        sed = run.reduce_counts(torch.from_numpy(eng.o.sed().astype(np.int64)))
        c = eng.o.counters()
        cnt = run.reduce_counts(torch.tensor([c[k] for k in ("emitted", "escaped", "lost",
                                                             "absorptions", "scatterings",
                                                             "flights", "crossings")]))
        extra = dict(pah_abs=eng.glob_pah, pah_cdf=eng.o.pah_cdf()) if with_pah else {}
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), tally=tally.numpy(), sed=sed.numpy(),
                 cnt=cnt.numpy(), T=eng.o.cell_temperature(), mine=np.array(mine),
                 n_cum=run.n_cum, **extra)
    finally:
        dist.destroy_process_group()


def test_rank_range_tiles_the_batch():
    for first, n, world in [(0, 10, 3), (7, 0, 2), (5, 1, 4), (1 << 40, 1048577, 8), (3, 8, 8)]:
        parts = [rank_range(first, n, world, r) for r in range(world)]
        assert parts[0][0] == first
        for (f0, c0), (f1, _) in zip(parts, parts[1:]):
            assert f0 + c0 == f1
        assert parts[-1][0] + parts[-1][1] == first + n
        sizes = [c for _, c in parts]
        assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        rank_range(0, 4, 2, 2)


def test_two_rank_sharded_run_equals_single_rank(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    r = [np.load(tmp_path / f"r{k}.npz") for k in range(world)]
    # single-rank run of the same batches
    wl = W.c0()
    eng = OracleEngine(wl)
    one = ShardedRunner(eng, None)
    for first, n in BATCHES:
        one.run_batch(wl.seed, first, n)
    tally, _ = eng.get_cell_energy()
    c = eng.o.counters()
    cnt = np.array([c[k] for k in ("emitted", "escaped", "lost", "absorptions", "scatterings",
                                   "flights", "crossings")])
    for k in range(world):
        assert int(r[k]["n_cum"]) == sum(n for _, n in BATCHES)
        np.testing.assert_array_equal(r[k]["tally"], tally.numpy())
        np.testing.assert_array_equal(r[k]["sed"], eng.o.sed().astype(np.int64))
        np.testing.assert_array_equal(r[k]["cnt"], cnt)
        np.testing.assert_array_equal(r[k]["T"], eng.o.cell_temperature())     # bit-identical
    # the two ranks' ranges tile every batch
    for b, (first, n) in enumerate(BATCHES):
        (f0, c0), (f1, c1) = r[0]["mine"][b], r[1]["mine"][b]
        assert f0 == first and f0 + c0 == f1 and f1 + c1 == first + n
    assert cnt[0] == cnt[1] and cnt[2] == 0                                     # emitted = escaped


def test_two_rank_sharded_run_with_pah_equals_single_rank(tmp_path):
    """The same with a transiently heated PAH declared (row f2): the delta array the ranks all-reduce carries
    the PAH's absorbed spectrum of every leaf behind the equilibrium counts; P(T) and the PAH emission CDFs
    (which steer the re-emission of the following batches) come out bit-identical on both ranks."""
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path), True), nprocs=world, join=True)
    r = [np.load(tmp_path / f"r{k}.npz") for k in range(world)]
    wl, pah = _pah_case()
    eng = OracleEngine(wl, pah)
    one = ShardedRunner(eng, None)
    for first, n in BATCHES:
        one.run_batch(wl.seed, first, n)
    tally, _ = eng.get_cell_energy()
    pah_abs, total = eng.o.pah_absorbed()
    assert total > 200
    for k in range(world):
        np.testing.assert_array_equal(r[k]["tally"], tally.numpy())
        np.testing.assert_array_equal(r[k]["sed"], eng.o.sed().astype(np.int64))
        np.testing.assert_array_equal(r[k]["T"], eng.o.cell_temperature())
        np.testing.assert_array_equal(r[k]["pah_abs"], pah_abs)
        np.testing.assert_array_equal(r[k]["pah_cdf"], eng.o.pah_cdf())
