"""include/streamkl.h: "Thread-safe for concurrent calls on distinct streams".  Two HOST threads, each with its own stream, its own
forward plan and backward mode (both are per calling thread) and its own shapes -- different head-dim pairs, so the run-time-sized
kernels set different shared-memory sizes, and one thread on the persistent forward, whose scheduler slots are shared process
state -- call the library a few hundred times at once.  Every result must equal, bit for bit, what the same thread's calls give
when they run alone (SEPARATE backward: tile ownership, no atomics, so bit-reproducible)."""
from __future__ import annotations

import threading

import pytest

import workloads as W
from parity_util import to_torch

pytestmark = pytest.mark.gpu


def _problem(cfg):
    inp = W.all_inputs(cfg)
    return [to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2")] + [to_torch(inp["g"])]


def _worker(skl, torch, jobs, plan, stream, rounds, out, errors):
    try:
        skl.streamkl_set_fwd_plan(plan)                       # per-thread settings: must not leak into the other thread
        skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_SEPARATE)
        with torch.cuda.stream(stream):
            for r in range(rounds):
                for cfg, d in jobs:
                    f = skl.streamkl_fwd(*d[:4], cfg.c1, cfg.c2, cfg.causal, stream=stream)
                    b = skl.streamkl_bwd(*d[:4], cfg.c1, cfg.c2, cfg.causal, *f, d[4], teacher=True, stream=stream)
                    if r % 10 == 9 or r == rounds - 1:        # keep a sample of the results (all of them would not fit)
                        out.append((cfg.name, list(f) + list(b)))
        stream.synchronize()
    except BaseException as e:   # noqa: BLE001 -- reported by the main thread
        errors.append(e)


def test_two_host_threads_with_their_own_streams_plans_and_shapes():
    import torch

    import paper_2606_20005_b200 as skl

    jobs_a = [(c, _problem(c)) for c in (W.Config(140, "th-a1", 1, 40, 1024, 1024, 128, 64, "bf16", True),     # persistent forward
                                         W.Config(141, "th-a2", 1, 2, 300, 500, 192, 64, "bf16", False))]     # BLOCKED / wide kernels
    jobs_b = [(c, _problem(c)) for c in (W.Config(142, "th-b1", 2, 3, 457, 901, 64, 128, "bf16", False),
                                         W.Config(143, "th-b2", 1, 2, 260, 700, 256, 256, "bf16", True))]     # other wide head dims
    plans = (skl.STREAMKL_FWD_PERSISTENT, skl.STREAMKL_FWD_PER_TILE)
    rounds = 60                                                # 2 threads x 60 rounds x 2 problems x (fwd + bwd) = 480 calls
    # serial reference: each thread's job list run alone, with that thread's settings, from this thread
    want = {}
    for jobs, plan in ((jobs_a, plans[0]), (jobs_b, plans[1])):
        out, errors = [], []
        _worker(skl, torch, jobs, plan, torch.cuda.Stream(), 1, out, errors)
        assert not errors, errors
        want.update(dict(out))
    skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_AUTO)
    skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)
    torch.cuda.synchronize()
    outs, errors = ([], []), []
    threads = [threading.Thread(target=_worker, args=(skl, torch, jobs, plan, torch.cuda.Stream(), rounds, o, errors))
               for jobs, plan, o in ((jobs_a, plans[0], outs[0]), (jobs_b, plans[1], outs[1]))]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    torch.cuda.synchronize()
    assert not errors, errors
    for o in outs:
        assert len(o) == 2 * (rounds // 10)
        for name, tensors in o:
            for got, exp in zip(tensors, want[name]):
                assert torch.equal(got, exp), f"{name}: a concurrent call differs from the same call made alone"
    # the main thread's own settings were not touched by the workers
    cfg, d = jobs_b[0]
    f = skl.streamkl_fwd(*d[:4], cfg.c1, cfg.c2, cfg.causal)
    assert all(torch.equal(a, b) for a, b in zip(f, want[cfg.name][:3]))
