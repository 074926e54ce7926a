"""world_size-2 gloo test of the multi-GPU path's host logic: terms are sharded over ranks,
each rank plans its shard (host-only plan, schedule executed by hpsi_debug_interpret), psi is replicated and one
all-reduce(sum) of psi' gives the full result - compared with the oracle on the unsharded problem."""
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


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import workloads
    import paper_2407_07411_b200 as H
    half = workloads.config_params("small")["n_terms"] // 2
    p = workloads.make_problem("small", base_terms=np.arange(rank, half, world))
    plan = H.plan_problem(p, flags=H.HPSI_PLAN_HOST_ONLY)
    psi = workloads.make_psi(p)                       # replicated: same seed on every rank
    out = torch.from_numpy(H.hpsi_debug_interpret(plan, p.a_data, p.b_data, psi))
    stats = torch.tensor([H.hpsi_query(plan, H.HPSI_Q_USEFUL_FLOPS), H.hpsi_query(plan, H.HPSI_Q_N_TASKS)])
    dist.all_reduce(out)
    dist.all_reduce(stats)
    if rank == 0:
        q.put((out.numpy(), stats.tolist()))
    dist.barrier()
    dist.destroy_process_group()


def test_term_sharded_apply_world2():
    import oracle
    import workloads
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    got, stats = q.get(timeout=300)
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    full = workloads.make_problem("small")
    ref = oracle.apply(full, workloads.make_psi(full))
    assert np.linalg.norm(got - ref) <= 1e-13 * np.linalg.norm(ref)
    flops, ntask = oracle.useful_flops(full)
    assert stats == [flops, ntask]                    # the shards partition the tasks exactly


def _worker_site_update(rank, world, port, q):
    """Site update under the same term sharding: the truncation is replicated (psi is), every rank updates the operator
    blocks of its own terms with the replicated isometries - no exchange step; the union of the shards' results must be
    the update of the full operator set, and the flop counts must add up."""
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import workloads
    import paper_2407_07411_b200 as H
    from oracle import site_update as su
    half = 40
    p = workloads.make_problem("small", n_terms=2 * half, base_terms=np.arange(rank, half, world))
    chi = workloads.proportional_chi(p.d_left, 0.25, zero_every=6)          # replicated: same on every rank
    ot = workloads.make_isometries(p.d_left, chi, seed=5)
    r = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, None, p.a_len, H.HPSI_PLAN_HOST_ONLY)
    out = H.hpsi_rotate_debug_interpret(r, p.a_data, workloads.pack_isometries(ot))
    desc = H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_BLOCKS)
    # Frobenius norm^2 of this shard's updated blocks, and the same from the oracle on the shard
    mine = 0.0
    for e in desc:
        if e["offset"] >= 0:
            rr, cc = int(chi[e["row"]]), int(chi[e["col"]])
            blk = np.lib.stride_tricks.as_strided(out[int(e["offset"]):], shape=(rr, cc), strides=(int(e["ld"]) * 8, 8))
            mine += float(np.sum(blk ** 2))
    ref = sum(float(np.sum(x ** 2)) for x in su.rotate(p.d_left, chi, p.a_desc, p.a_data, ot))
    stats = torch.tensor([mine, ref, float(H.hpsi_rotate_query(r, H.HPSI_RQ_USEFUL_FLOPS)), float(len(p.a_desc))],
                         dtype=torch.float64)
    dist.all_reduce(stats)
    if rank == 0:
        q.put(stats.tolist())
    dist.barrier()
    dist.destroy_process_group()


def test_term_sharded_site_update_world2():
    import workloads
    from oracle import site_update as su
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker_site_update, args=(r, 2, port, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    mine, ref, flops, nblk = q.get(timeout=300)
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    full = workloads.make_problem("small", n_terms=80)
    chi = workloads.proportional_chi(full.d_left, 0.25, zero_every=6)
    ot = workloads.make_isometries(full.d_left, chi, seed=5)
    whole = sum(float(np.sum(x ** 2)) for x in su.rotate(full.d_left, chi, full.a_desc, full.a_data, ot))
    assert abs(mine - ref) <= 1e-12 * ref and abs(ref - whole) <= 1e-12 * whole      # shards partition the blocks
    assert int(nblk) == len(full.a_desc) and int(flops) == su.rotate_flops(full.d_left, chi, full.a_desc)
