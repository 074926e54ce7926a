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
