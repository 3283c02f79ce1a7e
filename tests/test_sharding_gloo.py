"""The N>1 path of bench.py on CPU: world_size-2 `gloo` processes (independent (b,h) units, replicas of the
single-GPU path, no collective on the data path; timing = max over ranks; value = all ranks' work / that time).

Each rank takes its own units (bench.rank_heads), evaluates them with the float64 oracle (the GPU kernels are not
available here; what is tested is the host logic: unit ownership, no overlap, no exchange needed, the timing reduction
and the whole-job aggregate), and the gathered per-rank results must equal the oracle run over the global batch."""
from __future__ import annotations

import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    import torch
    import torch.distributed as dist

    import bench
    import workloads as W
    from oracle.streamkl_oracle import attention_kl

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = W.shrink(W.CONFIGS[3], B=1, H=2, NQ=96, NK=160)
        heads = bench.rank_heads(cfg, rank)
        inp = bench.gen_inputs(cfg, rank)
        ref = attention_kl(*(W.widen_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")), cfg.c1, cfg.c2, cfg.causal,
                           g=inp["g"].astype(np.float64), teacher=False)
        # timing reduction: rank r pretends to have taken (r+1) ms
        step_ms = bench.max_over_ranks(float(rank + 1), world, device="cpu")
        # gather everything on rank 0 only to CHECK it; the data path itself exchanged nothing
        gathered = [None] * world
        dist.all_gather_object(gathered, {"heads": heads, "kl": ref["kl"], "dK2": ref["dK2"], "step_ms": step_ms})
        if rank == 0:
            q.put(gathered)
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_two_rank_replicas_partition_the_units_and_reduce_time():
    import torch.multiprocessing as mp

    import bench
    import workloads as W
    from oracle.streamkl_oracle import attention_kl

    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    gathered = q.get(timeout=150)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # unit ownership: disjoint, and together exactly the global batch of world*B batches
    cfg = W.shrink(W.CONFIGS[3], B=1, H=2, NQ=96, NK=160)
    all_heads = [h for g in gathered for h in g["heads"]]
    assert len(all_heads) == len(set(all_heads)) == world * cfg.BH
    assert sorted(all_heads) == [(b, h) for b in range(world * cfg.B) for h in range(cfg.H)]
    # max over ranks, seen identically by every rank
    assert [g["step_ms"] for g in gathered] == [float(world)] * world
    # whole-job aggregate: all ranks' work / slowest rank's time
    assert bench.whole_job_tflops(world, 3e12, 2.0) == pytest.approx(world * 3e12 / 2e-3 / 1e12)
    # the concatenation of the per-rank results IS the result on the global batch (no cross-unit term anywhere)
    gcfg = W.shrink(cfg, B=world * cfg.B)
    ginp = W.all_inputs(gcfg)
    gref = attention_kl(*(W.widen_f64(ginp[k]) for k in ("Q1", "K1", "Q2", "K2")), gcfg.c1, gcfg.c2, gcfg.causal,
                        g=ginp["g"].astype(np.float64), teacher=False)
    for r, g in enumerate(gathered):
        assert np.array_equal(g["kl"], gref["kl"][r * cfg.B:(r + 1) * cfg.B])
        assert np.array_equal(g["dK2"], gref["dK2"][r * cfg.B:(r + 1) * cfg.B])
