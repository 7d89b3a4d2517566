"""Source-sharded tracing, host logic on CPU: the partition of the sources, and -
with gloo at world size 2 - `sharded.trace_sharded` / `sharded.reduce_stats` driving an oracle-backed stand-in for the
device context (same three methods as `arc.Context`): the reduced accumulators, rates and tallies equal those of one
trace of all sources.  The CUDA kernels are not involved here; the GPU side of the same path is tests/test_gpu_sharded.py."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1807_07094_b200 import sharded, workloads as wl  # noqa: E402


@pytest.mark.parametrize("nsrc,world", [(0, 1), (1, 4), (7, 2), (16, 3), (1024, 8), (4096, 8)])
def test_partition_is_disjoint_complete_and_balanced(nsrc, world):
    shards = sharded.partition_sources(nsrc, world)
    assert len(shards) == world
    allidx = np.concatenate(shards) if nsrc else np.zeros(0, np.int64)
    assert sorted(allidx.tolist()) == list(range(nsrc))
    sizes = [len(s) for s in shards]
    assert max(sizes) - min(sizes) <= 1
    for s in shards:
        assert np.all(np.diff(s) > 0)
    again = sharded.partition_sources(nsrc, world)
    assert all(np.array_equal(a, b) for a, b in zip(shards, again))


def test_weighted_partition_balances_the_load():
    rng = np.random.default_rng(3)
    w = 10.0 ** rng.uniform(0, 2, 257)
    for world in (2, 4, 8):
        shards = sharded.partition_sources(len(w), world, w)
        assert sorted(np.concatenate(shards).tolist()) == list(range(len(w)))
        loads = np.array([w[s].sum() for s in shards])
        # longest-processing-time greedy: no rank exceeds the mean by more than the largest single weight
        assert loads.max() - loads.mean() <= w.max()
        assert loads.max() / loads.mean() < 1.05
    one_heavy = sharded.partition_sources(5, 2, [100.0, 1.0, 1.0, 1.0, 1.0])
    assert one_heavy[0].tolist() == [0] and one_heavy[1].tolist() == [1, 2, 3, 4]
    with pytest.raises(ValueError):
        sharded.partition_sources(3, 2, [1.0, -1.0, 1.0])
    with pytest.raises(ValueError):
        sharded.partition_sources(3, 0)


class _OracleShard:
    """stand-in for arc.Context on a box without a GPU: this rank's share of the sources traced by the oracle"""

    def __init__(self, w, idx):
        from oracle import oracle as orc
        self.orc, self.w, self.idx = orc, w, idx
        self.A = None
        self.st = None

    def trace_partial(self, step=0):
        A, self.st, _ = self.orc.trace(self.w, sources=self.idx)
        self.A = torch.from_numpy(np.ascontiguousarray(A))

    def accum_tensor(self):
        return self.A

    def finalize(self):
        return self.orc.finalize(self.w, self.A.numpy())

    def stats(self):
        s = dict(self.st)
        s["absorbed"] = self.A.numpy().sum(axis=0)         # as arc_finalize does: from the reduced accumulators
        return s


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = wl.tiny(N=12, nsrc=5, nb=3, seed=11)
        idx = sharded.partition_sources(w.nsrc, world, w.src_Ndot)[rank]
        sh = _OracleShard(w, idx)
        G, H, Ht = sharded.trace_sharded(sh, None)
        st = sharded.reduce_stats(sh.stats(), None)
        torch.save(dict(A=sh.A.clone(), G=G, H=H, Ht=Ht, st=st, idx=idx, own_segments=sh.st["segments"]), os.path.join(out, f"r{rank}.pt"))
    finally:
        dist.destroy_process_group()


def test_two_ranks_reduce_to_the_trace_of_all_sources(tmp_path):
    from oracle import oracle as orc
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = wl.tiny(N=12, nsrc=5, nb=3, seed=11)
    A, st, _ = orc.trace(w)
    G, H, Ht = orc.finalize(w, A)
    res = [torch.load(os.path.join(tmp_path, f"r{r}.pt"), weights_only=False) for r in range(world)]
    assert sorted(np.concatenate([r["idx"] for r in res]).tolist()) == list(range(w.nsrc))
    assert sum(r["own_segments"] for r in res) == st["segments"] and all(0 < r["own_segments"] < st["segments"] for r in res)
    for r in res:
        # every rank ends with the same, complete answer (sum over sources in another order: 1e-12)
        np.testing.assert_allclose(r["A"].numpy(), A, rtol=1e-12, atol=1e-12 * A.max())
        np.testing.assert_allclose(r["G"], G, rtol=1e-11, atol=1e-12 * G.max())
        np.testing.assert_allclose(r["Ht"], Ht, rtol=1e-11, atol=1e-12 * Ht.max())
        assert r["st"]["segments"] == st["segments"] and r["st"]["rays"] == st["rays"]
        assert r["st"]["splits"] == st["splits"].tolist() and r["st"]["ends"] == st["ends"].tolist()
        np.testing.assert_allclose(r["st"]["emitted"], st["emitted"], rtol=1e-14)
        np.testing.assert_allclose(r["st"]["escaped"], st["escaped"], rtol=1e-12)
        np.testing.assert_allclose(r["st"]["absorbed"], st["absorbed"], rtol=1e-12)
        e, a, x = (np.asarray(r["st"][k]) for k in ("emitted", "absorbed", "escaped"))
        assert np.all(np.abs(a + x - e) <= 1e-10 * e)                      # photon conservation of the whole job
    assert torch.equal(res[0]["A"], res[1]["A"])


def test_single_process_needs_no_group():
    w = wl.tiny(N=8, nsrc=2, nb=2, seed=5)
    sh = _OracleShard(w, np.arange(w.nsrc))
    G, H, Ht = sharded.trace_sharded(sh)
    from oracle import oracle as orc
    A, st, _ = orc.trace(w)
    assert np.array_equal(sh.A.numpy(), A)
    assert sharded.reduce_stats(sh.stats())["segments"] == st["segments"]
