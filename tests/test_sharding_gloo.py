"""N > 1 path on CPU: world_size-2 gloo processes exercise the sharding logic bench.py uses: per-rank
seeds, disjoint covering slices, MAX-over-ranks timing, whole-job throughput; and the oracle confirms that a batch cut
in rank slices gives exactly the unsharded result (no cross-sample coupling anywhere on the path)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as WL
from workloads import sharding as SH


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # weak scaling: own seed -> own parameters and offsets
        wl = WL.make_c2(batch=8, seed=SH.rank_seed(0xA3D30002, rank), strip_len=1 << 18)
        digest = torch.tensor([float(wl.params.sum()), float(wl.offsets.sum())], dtype=torch.float64)
        gathered = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(gathered, digest)
        # strong split of a global batch of 11 samples
        start, count = SH.shard_batch(11, world, rank)
        sl = torch.tensor([start, count], dtype=torch.int64)
        slices = [torch.zeros(2, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(slices, sl)
        # timing: rank r "measured" (1 + r) ms; everyone must see the max
        t_max = SH.max_over_ranks(1.0 + rank, dist)
        ret[rank] = {"digests": [g.tolist() for g in gathered], "slices": [s.tolist() for s in slices], "t_max": t_max,
                     "value": SH.aggregate_throughput(1000, world, t_max)}
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_sharding():
    world = 2
    port = _free_port()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, port, ret), nprocs=world, join=True)
    assert set(ret.keys()) == {0, 1}
    for r in range(world):
        out = ret[r]
        assert out["digests"][0] != out["digests"][1]            # different data on the two ranks
        assert out["slices"] == [[0, 6], [6, 5]]                  # disjoint, ordered, covering
        assert out["t_max"] == 2.0                                # MAX over ranks, seen by both
        assert out["value"] == pytest.approx(2 * 1000 / 2e-3)
    assert ret[0]["digests"] == ret[1]["digests"]


def test_shard_batch_properties():
    for b in (0, 1, 7, 2048):
        for w in (1, 2, 3, 8):
            parts = [SH.shard_batch(b, w, r) for r in range(w)]
            assert parts[0][0] == 0 and sum(c for _, c in parts) == b
            for (s0, c0), (s1, _) in zip(parts, parts[1:]):
                assert s0 + c0 == s1
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
    with pytest.raises(ValueError):
        SH.shard_batch(4, 2, 2)


def test_oracle_sharded_equals_unsharded():
    from oracle import project as OP, waveform as OW, whiten as OWH
    wl = WL.make_c0()
    f = np.arange(wl.n // 2 + 1) * wl.fs / wl.n
    psd = np.tile(WL.aligo_psd(f), (wl.n_det, 1))

    def run(rows):
        hp, hc, _ = OW.waveform_fd(wl.approximant, wl.params[rows], wl.n, wl.fs, wl.f_lo, wl.f_hi)
        h_det, _ = OP.project(hp, hc, wl.params[rows], wl.gmst, wl.det_ids, wl.n, wl.fs)
        return OWH.inject_whiten(wl.noise[rows].astype(np.float64), h_det, psd, wl.fs, wl.f_lo, wl.f_hi)

    full = run(slice(0, wl.batch))
    parts = []
    for r in range(2):
        s, c = SH.shard_batch(wl.batch, 2, r)
        parts.append(run(slice(s, s + c)))
    assert np.array_equal(np.concatenate(parts, axis=0), full)
