"""Smallest program that runs the hot path, for ncu captures (profiles/*.md name the command lines):

    python -m paper_2407_07411_b200.profile_apply --config cyp --applies 3 [--share-adjoint] [--site-update] [--n-vectors K]

Plans the named synthetic config, runs ``--applies`` hpsi_apply calls (or site updates) on cuda:0 and prints their
mean device time.  No calibration, no oracle: bench.py is the measurement, this is what gets profiled.
"""
import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    import numpy as np
    import torch
    import workloads
    import paper_2407_07411_b200 as H
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="cyp", choices=list(workloads.CONFIG_NAMES))
    ap.add_argument("--applies", type=int, default=3)
    ap.add_argument("--share-adjoint", action="store_true")
    ap.add_argument("--site-update", action="store_true")
    ap.add_argument("--n-vectors", type=int, default=1)
    ap.add_argument("--fused", action="store_true", help="HPSI_PLAN_FUSE_ALL: narrow groups through the one-CTA kernel")
    ap.add_argument("--D", type=int, default=None)
    args = ap.parse_args()
    assert torch.cuda.is_available(), "needs cuda:0 (there is no CPU fallback)"
    torch.cuda.set_device(0)
    p = workloads.make_problem(args.config, share_adjoint=args.share_adjoint, D=args.D)
    a, b = torch.from_numpy(p.a_data).cuda(), torch.from_numpy(p.b_data).cuda()
    st = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if args.site_update:
        small = workloads.make_problem(args.config, n_terms=2, D=args.D)
        plan = H.plan_problem(small, torch.from_numpy(small.a_data).cuda(), torch.from_numpy(small.b_data).cuda())
        psi = torch.from_numpy(workloads.make_psi(p)).cuda()
        ot = torch.zeros(H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY), dtype=torch.float64, device="cuda")
        chi, _, _ = H.hpsi_truncate(plan, psi, max(1, int(p.d_left.sum()) // 4), ot, st)
        rot = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, a, p.a_len)
        out = torch.empty(H.hpsi_rotate_query(rot, H.HPSI_RQ_OUT_LENGTH), dtype=torch.float64, device="cuda")
        e0.record(st)
        for _ in range(args.applies):
            H.hpsi_truncate(plan, psi, max(1, int(p.d_left.sum()) // 4), ot, st)
            H.hpsi_rotate_apply(rot, ot, out, st)
        e1.record(st)
        torch.cuda.synchronize()
        print(f"{args.config}: site update {e0.elapsed_time(e1) / args.applies:.3f} ms")
        return
    nv = max(1, args.n_vectors)
    plan = H.plan_problem(p, a, b, H.HPSI_PLAN_FUSE_ALL if args.fused else 0, n_vectors=nv if nv > 1 else 0)
    psi = torch.from_numpy(np.stack([workloads.make_psi(p, k) for k in range(nv)])).cuda()
    out = torch.empty_like(psi)
    e0.record(st)
    for _ in range(args.applies):
        if nv > 1:
            H.hpsi_apply_multi(plan, psi, out, nv, st)
        else:
            H.hpsi_apply(plan, psi[0], out[0], st)
    e1.record(st)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.applies
    print(f"{args.config}: {ms:.3f} ms per apply of {nv} vector(s), "
          f"{H.hpsi_query(plan, H.HPSI_Q_USEFUL_FLOPS) * nv / ms / 1e9:.2f} TFLOPS (first applies, cold)")


if __name__ == "__main__":
    main()
