"""N > 1 path on CPU: world_size-2 gloo processes shard the frames (no data-path collective), the
concatenated shards equal the whole batch, and the step time is the max over ranks."""
import os
import socket

import numpy as np
import pytest

from paper_1501_03869_b200 import sharding


def test_split_and_ranges_cover_exactly():
    for n, w in [(0, 1), (1, 2), (5, 2), (64, 8), (7, 3)]:
        parts = sharding.split_frames(n, w)
        assert parts[0][0] == 0 and parts[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
        assert max(e - b for b, e in parts) - min(e - b for b, e in parts) <= 1
    assert sharding.rank_frame_range(1, 2, 4) == (4, 8)
    with pytest.raises(ValueError):
        sharding.rank_frame_range(2, 2, 4)
    assert sharding.max_over_ranks(3.5) == 3.5


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(7)                      # every rank builds the same seeded problem
    S, P, Nt, B = 5, 97, 48, 6
    tau = (rng.uniform(0.5, Nt - 2, size=(S, P)) / 20e6).astype(np.float32)
    tr = rng.standard_normal((B, S, Nt)).astype(np.float32)
    b, e = sharding.split_frames(B, world)[rank]
    mine = oracle.backproject(tau, tr[b:e], 20e6, 0.0, 1)      # the rank's own frames, no exchange
    ms = sharding.max_over_ranks(10.0 + rank, dist)            # slowest rank defines the step
    gathered = [None] * world
    dist.all_gather_object(gathered, (b, e, mine))             # test-only gather
    if rank == 0:
        whole = oracle.backproject(tau, tr, 20e6, 0.0, 1)
        cat = np.concatenate([g[2] for g in sorted(gathered, key=lambda g: g[0])], axis=0)
        out["ok"] = bool(np.array_equal(cat, whole)) and ms == 10.0 + world - 1
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_frame_sharding_with_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    mgr = ctx.Manager()
    out = mgr.dict()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert out.get("ok") is True


def _gpu_worker(rank, world, port, out):
    """One process per rank, each with its OWN plan (table copy) on its device and its own frames of the batch --
    the product path, not the oracle.  With fewer devices than ranks the ranks share device 0: no kernel of one rank
    ever waits for another rank (there is no data-path collective), so that is a valid stand-in for placement only."""
    import torch
    import torch.distributed as dist
    import workloads as W
    import paper_1501_03869_b200 as pat
    from _cases import prod_tau
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = rank % torch.cuda.device_count()
    torch.cuda.set_device(dev)
    geom = W.make_geometry(0)
    tau = prod_tau(geom)
    B = 6
    traces = W.make_traces(geom, tau, frames=range(B))             # every rank builds the same seeded batch
    b, e = sharding.split_frames(B, world)[rank]
    plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs,
                    geom.t0, max_batch=B)
    plan.set_travel_times(tau)
    img = torch.full((e - b, geom.npix), float("nan"), dtype=torch.float32, device="cuda:%d" % dev)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    plan.backproject(torch.from_numpy(np.ascontiguousarray(traces[b:e])).cuda(), img, e - b)
    ev1.record()
    torch.cuda.synchronize()
    ms = sharding.max_over_ranks(ev0.elapsed_time(ev1), dist)      # slowest rank defines the step (gloo: CPU tensor)
    gathered = [None] * world
    dist.all_gather_object(gathered, (b, e, img.cpu().numpy(), ev0.elapsed_time(ev1), plan.launches()))
    if rank == 0:
        whole = torch.full((B, geom.npix), float("nan"), dtype=torch.float32, device="cuda:%d" % dev)
        plan.backproject(torch.from_numpy(np.ascontiguousarray(traces)).cuda(), whole, B)
        torch.cuda.synchronize()
        cat = np.concatenate([g[2] for g in sorted(gathered, key=lambda g: g[0])], axis=0)
        ref = whole.cpu().numpy()
        # a frame's image does not depend on the batch it is in up to the fp32 order of the cross-CTA sums
        rel = np.linalg.norm(cat - ref) / np.linalg.norm(ref)
        out["rel"] = float(rel)
        out["ok"] = bool(np.isfinite(cat).all()) and rel <= 1e-5 and abs(ms - max(g[3] for g in gathered)) < 1e-9 \
            and all(g[4] >= 2 for g in gathered)
    plan.close()
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.gpu
def test_two_ranks_run_the_product_path_on_their_own_frames():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    mgr = ctx.Manager()
    out = mgr.dict()
    port = _free_port()
    procs = [ctx.Process(target=_gpu_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(300)
        assert p.exitcode == 0
    assert out.get("ok") is True, dict(out)
