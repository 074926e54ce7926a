"""world_size-2 gloo tests of the multi-GPU path's host logic, through the very functions
bench.py runs under torchrun: the library partitions the terms (hpsi_shard_terms), every rank fills and plans its own
shard (workloads.make_shard + hpsi_plan_ex; host-only plans here, the schedule executed by hpsi_debug_interpret), psi is
replicated, the partial results are all-gathered and added in rank order - compared element by element with the oracle on
the unsharded problem.  (The same shards run through the CUDA kernels in tests/test_gpu_parity.py.)"""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _spawn(worker, world=2, timeout=300):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=worker, args=(r, world, port, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    got = q.get(timeout=timeout)
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    return got


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import workloads
    import paper_2407_07411_b200 as H
    p, plan_kw, shard_flops = bench.shard_for_rank("small", rank, world)
    plan = H.plan_problem(p, flags=H.HPSI_PLAN_HOST_ONLY, **plan_kw)
    assert H.hpsi_query(plan, H.HPSI_Q_USEFUL_FLOPS) == shard_flops[rank]
    psi = workloads.make_psi(p)                       # replicated: same seed on every rank
    mine = torch.from_numpy(H.hpsi_debug_interpret(plan, p.a_data, p.b_data, psi))
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)                      # the exchange step; hpsi_sum_shards adds in rank order
    out = parts[0].clone()
    for r in range(1, world):
        out += parts[r]
    stats = torch.tensor([H.hpsi_query(plan, H.HPSI_Q_USEFUL_FLOPS), H.hpsi_query(plan, H.HPSI_Q_N_TASKS),
                          H.hpsi_query(plan, H.HPSI_Q_N_TERMS_PLANNED), p.a_len + p.b_len])
    dist.all_reduce(stats)
    if rank == 0:
        q.put((out.numpy(), stats.tolist(), [int(x) for x in shard_flops]))
    dist.barrier()
    dist.destroy_process_group()


def test_term_sharded_apply_world2():
    import oracle
    import workloads
    got, stats, shard_flops = _spawn(_worker)
    full = workloads.make_problem("small")
    ref = oracle.apply(full, workloads.make_psi(full))
    assert np.max(np.abs(got - ref)) <= 1e-13 * np.max(np.abs(ref))            # element by element
    flops, ntask = oracle.useful_flops(full)
    assert stats == [flops, ntask, full.n_terms, full.a_len + full.b_len]        # the shards partition tasks, terms and storage
    assert max(shard_flops) <= 1.01 * (flops / 2)                                # balanced by useful flops


def _worker_site_update(rank, world, port, q):
    """Site update under the same term sharding: the truncation is replicated (psi is), every rank updates the operator
    blocks of its own terms with the replicated isometries - no exchange step; every updated block of every shard must
    equal, element by element, the oracle's update of that block in the full operator set, and the flops must add up."""
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import workloads
    import paper_2407_07411_b200 as H
    from oracle import site_update as su
    half = 40
    p = workloads.make_problem("small", n_terms=2 * half, base_terms=np.arange(rank, half, world))
    full = workloads.make_problem("small", n_terms=2 * half)
    chi = workloads.proportional_chi(p.d_left, 0.25, zero_every=6)          # replicated: same on every rank
    ot = workloads.make_isometries(p.d_left, chi, seed=5)
    r = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, None, p.a_len, H.HPSI_PLAN_HOST_ONLY)
    out = H.hpsi_rotate_debug_interpret(r, p.a_data, workloads.pack_isometries(ot))
    desc = H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_BLOCKS)
    # the oracle on the FULL operator set; block (term, row, col) of the shard is block (global term, row, col) there
    gid = np.concatenate([p.base_term_ids, p.base_term_ids + half])
    where = {(int(e["term"]), int(e["row"]), int(e["col"])): i for i, e in enumerate(full.a_desc)}
    ref = su.rotate(full.d_left, chi, full.a_desc, full.a_data, ot)
    worst, nblk = 0.0, 0
    for e in desc:
        x = ref[where[(int(gid[e["term"]]), int(e["row"]), int(e["col"]))]]
        if e["offset"] < 0:
            assert x.size == 0
            continue
        blk = np.lib.stride_tricks.as_strided(out[int(e["offset"]):], shape=x.shape, strides=(int(e["ld"]) * 8, 8))
        worst = max(worst, float(np.max(np.abs(blk - x))) / max(float(np.max(np.abs(x))), 1e-300))
        nblk += 1
    stats = torch.tensor([float(H.hpsi_rotate_query(r, H.HPSI_RQ_USEFUL_FLOPS)), float(len(p.a_desc)), float(nblk)],
                         dtype=torch.float64)
    worst_t = torch.tensor([worst], dtype=torch.float64)
    dist.all_reduce(stats)
    dist.all_reduce(worst_t, op=dist.ReduceOp.MAX)
    if rank == 0:
        q.put((stats.tolist(), float(worst_t.item())))
    dist.barrier()
    dist.destroy_process_group()


def test_term_sharded_site_update_world2():
    import workloads
    from oracle import site_update as su
    (flops, nblk, nalive), worst = _spawn(_worker_site_update)
    full = workloads.make_problem("small", n_terms=80)
    chi = workloads.proportional_chi(full.d_left, 0.25, zero_every=6)
    assert worst <= 1e-13                                                         # every block, element by element
    assert int(nblk) == len(full.a_desc) and int(flops) == su.rotate_flops(full.d_left, chi, full.a_desc)
    alive = sum(1 for e in full.a_desc if chi[e["row"]] > 0 and chi[e["col"]] > 0)
    assert int(nalive) == alive                                                   # the shards partition the surviving blocks


def test_bench_withholds_stale_traffic(monkeypatch):
    """roofline.traffic comes from a committed ncu capture: bench.py reports it only while the digest of the kernel
    sources equals the one recorded with the capture (profiles/ncu_traffic.json.txt), and null otherwise."""
    import bench
    val, src = bench.ncu_traffic("cyp", "p1_kernel")
    assert src["capture_kernels_digest"] == src["kernels_digest"] == bench.kernel_sources_digest()
    assert isinstance(val, int) and val > 10 ** 10          # the committed capture describes the committed kernels
    monkeypatch.setattr(bench, "kernel_sources_digest", lambda: "0" * 16)
    val, src = bench.ncu_traffic("cyp", "p1_kernel")
    assert val is None and src["kernels_digest"] != src["capture_kernels_digest"]
