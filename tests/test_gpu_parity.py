"""GPU parity: hpsi_apply / hpsi_diagonal / hpsi_davidson through the C ABI versus the CPU oracle, element by element
on the same seeded inputs.  Bar (BASELINE.json north_star): relative L2 error <= 1e-12 in FP64."""
import numpy as np
import pytest

import oracle
import workloads
from workloads.hubbard import hubbard_two_block_problem
from gpu_util import GpuProblem, assert_blockwise, fill_device_arenas, rel_l2, shard_sum
from test_oracle_pins import random_custom

pytestmark = pytest.mark.gpu
TOL = 1e-12      # north_star: "relative L2 error <= 1e-12 in FP64"


@pytest.fixture(scope="module")
def H():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2407_07411_b200 as H
    return H


FLAG_NAMES = ["min_flops", "order1", "order2", "fused", "fused_order1", "fused_order2"]


def plan_flags(H, name):
    """Contraction-order and fusion variants of the planner (fused = every narrow group runs both GEMMs in one CTA)."""
    return {"min_flops": 0, "order1": H.HPSI_PLAN_FIXED_ORDER1, "order2": H.HPSI_PLAN_FIXED_ORDER2,
            "fused": H.HPSI_PLAN_FUSE_ALL, "fused_order1": H.HPSI_PLAN_FUSE_ALL | H.HPSI_PLAN_FIXED_ORDER1,
            "fused_order2": H.HPSI_PLAN_FUSE_ALL | H.HPSI_PLAN_FIXED_ORDER2}[name]


@pytest.mark.parametrize("flags_name", FLAG_NAMES)
def test_toy_parity(H, toy, flags_name):
    flags = plan_flags(H, flags_name)
    g = GpuProblem(toy, flags)
    if flags_name.startswith("fused"):          # every toy dim is <= 6: all tasks fused, nothing through the workspace
        assert g.q(H.HPSI_Q_N_FUSED_TASKS) == g.q(H.HPSI_Q_N_TASKS) and g.q(H.HPSI_Q_N_P1_UNITS) == 0
        assert g.q(H.HPSI_Q_INTERMEDIATE_BYTES) == 0
    else:
        assert g.q(H.HPSI_Q_N_FUSED_TASKS) == 0
    for k in range(3):
        psi = workloads.make_psi(toy, k)
        assert rel_l2(g.apply(psi), oracle.apply(toy, psi)) <= TOL


@pytest.mark.parametrize("flags_name", FLAG_NAMES)
def test_small_parity(H, small, flags_name):
    flags = plan_flags(H, flags_name)
    g = GpuProblem(small, flags)
    if flags_name.startswith("fused"):          # dims 7..136: a mix of fused groups and groups through the workspace
        assert 0 < g.q(H.HPSI_Q_N_FUSED_TASKS) < g.q(H.HPSI_Q_N_TASKS)
    psi = workloads.make_psi(small)
    ref = oracle.apply(small, psi)
    got = g.apply(psi)
    assert rel_l2(got, ref) <= TOL
    # worst block, as a diagnostic with the same bar
    for (i, j, r, c, off) in small.psi_blocks():
        assert np.linalg.norm(got[off:off + r * c] - ref[off:off + r * c]) <= 1e-11 * np.linalg.norm(ref)


def test_small_unaligned_staging(H):
    """Dense (odd) leading dimensions and an 8-byte-aligned arena: the 8-byte cp.async variant of the kernels."""
    p = workloads.make_problem("small", pad_even=False, n_terms=60)
    g = GpuProblem(p, misalign=True)
    assert g.q(H.HPSI_Q_ALIGNED16) == 0
    psi = workloads.make_psi(p)
    assert rel_l2(g.apply(psi), oracle.apply(p, psi)) <= TOL
    g2 = GpuProblem(workloads.make_problem("small", pad_even=True, n_terms=60), misalign=True)
    assert g2.q(H.HPSI_Q_ALIGNED16) == 0
    assert rel_l2(g2.apply(psi), oracle.apply(g2.p, psi)) <= TOL


@pytest.mark.parametrize("seed", range(8))
def test_irregular_parity(H, seed):
    p = random_custom(seed, grid=(seed < 4))
    g = GpuProblem(p, H.HPSI_PLAN_FUSE_ALL if seed % 2 else 0)
    psi = np.random.default_rng(seed).standard_normal(p.psi_len)
    ref = oracle.apply(p, psi)
    assert np.linalg.norm(g.apply(psi) - ref) <= TOL * max(np.linalg.norm(ref), 1.0)


def test_multi_tile_ragged_split_k(H):
    """Output blocks spanning several 64x64 tiles with ragged tails (150x131, 70x9) and split-K partials."""
    rng = np.random.default_rng(5)
    dL, dR = [150, 70], [131, 9]
    terms = []
    for _ in range(40):
        ab = {(r, c): rng.standard_normal((dL[r], dL[c])) for r in range(2) for c in range(2)}
        bb = {(r, c): rng.standard_normal((dR[r], dR[c])) for r in range(2) for c in range(2)}
        terms.append((float(rng.standard_normal()), ab, bb))
    p = workloads.custom_problem([(0, 0), (1, 1)], dL, [(3, 1), (2, 0)], dR, (3, 1), terms, pad_even=True)
    g = GpuProblem(p)
    psi = rng.standard_normal(p.psi_len)
    assert rel_l2(g.apply(psi), oracle.apply(p, psi)) <= TOL


def test_single_block_equals_blas(H):
    """n_L = n_R = 1, one term, c = 1: the result is A @ psi @ B.T (LAPACK/BLAS DGEMM)."""
    rng = np.random.default_rng(11)
    A, B = rng.standard_normal((77, 77)), rng.standard_normal((45, 45))
    p = workloads.custom_problem([(1, 0)], [77], [(2, 0)], [45], (3, 0), [(1.0, {(0, 0): A}, {(0, 0): B})])
    psi = rng.standard_normal(77 * 45)
    ref = (A @ psi.reshape(77, 45) @ B.T).ravel()
    assert rel_l2(GpuProblem(p).apply(psi), ref) <= TOL


def test_empty_cases(H):
    import torch
    p = workloads.make_problem("toy", n_terms=0)
    g = GpuProblem(p)
    assert np.all(g.apply(workloads.make_psi(p)) == 0.0)            # overwrite semantics: zeros, not the NaN prefill
    # a destination block that no task writes is zero-filled
    q = workloads.custom_problem([(0, 0), (1, 0)], [3, 2], [(1, 0), (0, 0)], [2, 4], (1, 0),
                                 [(2.0, {(0, 0): np.ones((3, 3))}, {(0, 0): np.ones((2, 2))})])
    g = GpuProblem(q)
    psi = np.arange(1.0, 1.0 + q.psi_len)
    ref = oracle.apply(q, psi)
    out = g.apply(psi)
    assert rel_l2(out, ref) <= TOL and np.all(out[6:] == 0.0)
    with pytest.raises(H.HpsiError):
        x = torch.zeros(q.psi_len, dtype=torch.float64, device="cuda")
        H.hpsi_apply(g.plan, x, x)                                    # aliasing is rejected


def test_bitwise_determinism(H, small):
    g = GpuProblem(small)
    psi = workloads.make_psi(small, 1)
    a, b = g.apply(psi), g.apply(psi)
    assert np.array_equal(a, b)
    assert np.array_equal(a, GpuProblem(small).apply(psi))           # a fresh plan gives the same bits


def test_apply_host_and_graph_capture(H, small):
    import torch
    g = GpuProblem(small)
    psi = workloads.make_psi(small, 2)
    ref = g.apply(psi)
    out = np.empty_like(psi)
    H.hpsi_apply_host(g.plan, psi, out, torch.cuda.current_stream())
    assert np.array_equal(out, ref)
    # hpsi_apply only enqueues: it can be captured into a CUDA graph and replayed
    x = torch.from_numpy(psi).cuda()
    y = torch.zeros_like(x)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        H.hpsi_apply(g.plan, x, y, s)
        s.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            H.hpsi_apply(g.plan, x, y, s)
        y.zero_()
        graph.replay()
        s.synchronize()
    assert np.array_equal(y.cpu().numpy(), ref)


def test_hermiticity_on_gpu(H, small):
    g = GpuProblem(small)
    rng = np.random.default_rng(3)
    x, y = rng.standard_normal(small.psi_len), rng.standard_normal(small.psi_len)
    Hx, Hy = g.apply(x), g.apply(y)
    assert abs(x @ Hy - Hx @ y) <= 1e-12 * np.linalg.norm(x) * np.linalg.norm(Hy)


def test_diagonal(H, toy):
    import torch
    g = GpuProblem(toy)
    d = torch.empty(g.n, dtype=torch.float64, device="cuda")
    H.hpsi_diagonal(g.plan, d)
    torch.cuda.synchronize()
    ref = oracle.diagonal(toy)
    assert np.linalg.norm(d.cpu().numpy() - ref) <= 1e-13 * max(np.linalg.norm(ref), 1.0)
    assert np.allclose(ref, np.diag(oracle.dense_hamiltonian(toy)), atol=1e-13)


def _davidson(H, g, v0, **kw):
    import torch
    x = torch.from_numpy(np.ascontiguousarray(v0)).cuda()
    theta, info = H.hpsi_davidson(g.plan, x, **kw)
    return theta, x.cpu().numpy(), info


def test_davidson_toy_vs_dense(H, toy):
    g = GpuProblem(toy)
    ev = np.linalg.eigvalsh(oracle.dense_hamiltonian(toy))
    theta, x, info = _davidson(H, g, workloads.make_psi(toy), tol=1e-9, max_iter=400)
    assert info["converged"] and abs(theta - ev[0]) <= 1e-10
    assert np.linalg.norm(oracle.apply(toy, x) - theta * x) <= 1e-8
    th_o, _, nmv_o, _ = oracle.davidson(toy, workloads.make_psi(toy), tol=1e-9, max_iter=400)
    assert abs(theta - th_o) <= 1e-10
    theta2, _, info2 = _davidson(H, g, workloads.make_psi(toy), tol=1e-9, max_iter=400, precondition=False, m_max=8)
    assert info2["converged"] and abs(theta2 - ev[0]) <= 1e-10


def test_davidson_hubbard_closed_forms(H):
    """Textbook pins (tests/golden/hubbard_closed_forms.txt): dimer (U - sqrt(U^2+16t^2))/2, 4-site chain -2 sqrt(5) t."""
    dimer = hubbard_two_block_problem(1, 1, 1.0, 3.7, 2, 0)
    theta, _, info = _davidson(H, GpuProblem(dimer), np.ones(dimer.psi_len), tol=1e-10)
    assert info["converged"] and abs(theta - (3.7 - np.sqrt(3.7 ** 2 + 16.0)) / 2) <= 1e-10
    chain = hubbard_two_block_problem(2, 2, 1.0, 0.0, 4, 0)
    v0 = np.random.default_rng(0).standard_normal(chain.psi_len)
    theta, _, info = _davidson(H, GpuProblem(chain), v0, tol=1e-10, precondition=False)
    assert info["converged"] and abs(theta + 2 * np.sqrt(5.0)) <= 1e-9


def test_davidson_small(H, small):
    g = GpuProblem(small)
    theta, x, info = _davidson(H, g, workloads.make_psi(small), tol=1e-7, max_iter=300)
    assert info["converged"]
    assert np.linalg.norm(oracle.apply(small, x) - theta * x) <= 1e-6


def _nan_padded(p):
    """Copy of the arenas with every element that is not inside a block (ld padding, gaps) set to NaN."""
    a, b = np.full_like(p.a_data, np.nan), np.full_like(p.b_data, np.nan)
    for desc, src, dst, dims in ((p.a_desc, p.a_data, a, p.d_left), (p.b_desc, p.b_data, b, p.d_right)):
        for e in desc:
            r, c, ld, off = int(dims[e["row"]]), int(dims[e["col"]]), int(e["ld"]), int(e["offset"])
            for x in range(r):
                dst[off + x * ld: off + x * ld + c] = src[off + x * ld: off + x * ld + c]
    return a, b


@pytest.mark.parametrize("misalign", [False, True])
def test_padding_is_never_read_and_rebind(H, misalign):
    """TMA boxes (and the LDGSTS fallback) clip at the matrix edge: NaN in the ld padding must not reach the result.
    hpsi_bind to arenas at a new address re-encodes the tensor maps."""
    import torch
    p = workloads.make_problem("small", n_terms=40)
    g = GpuProblem(p, misalign=misalign)
    assert g.q(H.HPSI_Q_ALIGNED16) == (0 if misalign else 1)
    psi = workloads.make_psi(p)
    ref = oracle.apply(p, psi)
    assert rel_l2(g.apply(psi), ref) <= TOL
    a_nan, b_nan = _nan_padded(p)
    assert np.isnan(a_nan).any() and np.isnan(b_nan).any()
    a2 = torch.from_numpy(a_nan).cuda()
    b2 = torch.from_numpy(b_nan).cuda()
    H.hpsi_bind(g.plan, a2, b2)
    g.a.fill_(float("nan"))                      # the old arenas must not be read any more
    g.b.fill_(float("nan"))
    assert g.q(H.HPSI_Q_ALIGNED16) == 1
    out = g.apply(psi)
    assert np.isfinite(out).all() and rel_l2(out, ref) <= TOL


def test_warp_grid_shapes(H):
    """Blocks whose tiles make the planner pick each warp grid: 56x64 (7x8 fragments -> 1x4), 64x56 (-> 4x1),
    40x40 (5x5 -> 2x2), 8x64 and 64x8 (one fragment row / column), plus ragged 61x59."""
    rng = np.random.default_rng(21)
    dL, dR = [56, 64, 40, 8, 64, 61], [64, 56, 40, 64, 8, 59]
    n = len(dL)
    terms = []
    for _ in range(6):
        ab = {(r, c): rng.standard_normal((dL[r], dL[c])) for r in range(n) for c in range(n) if (r + c) % 2 == 0 or r == c}
        bb = {(r, c): rng.standard_normal((dR[r], dR[c])) for r in range(n) for c in range(n) if (r + c) % 2 == 0 or r == c}
        terms.append((float(rng.standard_normal()), ab, bb))
    qL = [(i, 0) for i in range(n)]
    qR = [(n - i, 0) for i in range(n)]
    p = workloads.custom_problem(qL, dL, qR, dR, (n, 0), terms, pad_even=True)
    psi = rng.standard_normal(p.psi_len)
    ref = oracle.apply(p, psi)
    for flags in (0, H.HPSI_PLAN_FIXED_ORDER1, H.HPSI_PLAN_FIXED_ORDER2):
        assert rel_l2(GpuProblem(p, flags).apply(psi), ref) <= TOL


def _samples(p, n, seed=7):
    rng = np.random.default_rng(seed)
    blocks = p.psi_blocks()
    bi = rng.integers(0, len(blocks), n)
    sl = np.array([blocks[b][0] for b in bi], np.int32)
    sx = np.array([rng.integers(0, blocks[b][2]) for b in bi], np.int32)
    sy = np.array([rng.integers(0, blocks[b][3]) for b in bi], np.int32)
    idx = np.array([blocks[b][4] + x * blocks[b][3] + y for b, x, y in zip(bi, sx, sy)], np.int64)
    return sl, sx, sy, idx


@pytest.mark.parametrize("cfg", ["cyp", "stress"])
def test_full_size_full_vector_parity(H, cfg):
    """BASELINE.json configs[2] / configs[4] at full size, in the launch configuration bench.py times: the WHOLE output
    vector against one full oracle apply (620 188 / 1 583 102 elements), block by block; Hermiticity of the GPU result
    against the oracle's; bitwise reproducibility; and the same operators cut into 8 term shards (hpsi_shard_terms +
    hpsi_plan_ex), every shard through the CUDA kernels, summed in rank order by hpsi_sum_shards."""
    import torch
    p = workloads.make_problem(cfg)
    g = GpuProblem(p)
    assert g.q(H.HPSI_Q_ALIGNED16) == 1
    psi = workloads.make_psi(p)
    out = g.apply(psi)
    ref = oracle.apply(p, psi)
    assert_blockwise(p, out, ref, TOL)
    y = workloads.make_psi(p, 1)
    Hy = g.apply(y)
    assert abs(psi @ Hy - ref @ y) <= 1e-12 * np.linalg.norm(psi) * np.linalg.norm(Hy)     # <x, H_gpu y> = <H_oracle x, y>
    assert np.array_equal(out, g.apply(psi))                       # bitwise reproducible at full size
    # term shards through the kernels (the multi-GPU path's compute, one shard after the other on this GPU)
    world, half = 8, p.n_terms // 2
    shard, fl = H.hpsi_shard_terms(p, world, np.arange(p.n_terms) % half)
    assert int(fl.sum()) == g.q(H.HPSI_Q_USEFUL_FLOPS) and fl.max() <= 1.02 * fl.mean()
    x = torch.from_numpy(psi).cuda()
    parts, ntask = [], 0
    for r in range(world):
        gs = GpuProblem(p, arenas=(g.a, g.b), shard_of_term=shard, shard_index=r)
        assert gs.q(H.HPSI_Q_USEFUL_FLOPS) == fl[r]
        ntask += gs.q(H.HPSI_Q_N_TASKS)
        parts.append(gs.apply_dev(x))
        del gs
    assert ntask == g.q(H.HPSI_Q_N_TASKS)
    assert_blockwise(p, shard_sum(H, torch, parts), ref, TOL)


def test_femoco_shaped_full_vector_parity(H):
    """BASELINE.json configs[3] (D = 8192, sector dims up to 555: ~9 tiles per block edge, K-stacks across several
    groups) with 120 of its 2900 terms, so that the operators are 3.3 GB instead of 80: the whole output vector against
    the oracle, block by block, for the planner's order choice and both forced orders."""
    p = workloads.make_problem("femoco", n_terms=120)
    assert p.d_left.sum() == 8192 and p.d_right.sum() == 8192 and max(p.d_left.max(), p.d_right.max()) > 500
    psi = workloads.make_psi(p)
    ref = oracle.apply(p, psi)
    g = GpuProblem(p)
    assert g.q(H.HPSI_Q_ALIGNED16) == 1
    out = g.apply(psi)
    assert_blockwise(p, out, ref, TOL)
    assert np.array_equal(out, g.apply(psi))
    for flags in (H.HPSI_PLAN_FIXED_ORDER1, H.HPSI_PLAN_FIXED_ORDER2):
        assert_blockwise(p, GpuProblem(p, flags, arenas=(g.a, g.b)).apply(psi), ref, TOL)
    sh = workloads.make_problem("femoco", n_terms=120, share_adjoint=True)      # the 40 GB storage mode of the full config
    assert_blockwise(p, GpuProblem(sh).apply(psi), ref, TOL)


def test_femoco_full_config_sampled_parity(H):
    """BASELINE.json configs[3] in full (2900 terms, 80 GB of operators resident, the launch configuration bench.py
    --config femoco times): device arenas filled chunk by chunk, the same chunks streamed through the oracle, which
    computes 48 sampled outputs one by one (a full oracle apply would take minutes: 5.7 TFLOP)."""
    import torch
    free, total = torch.cuda.mem_get_info()
    full = workloads.make_problem("femoco", fill=False)
    need = 8 * (full.a_len + full.b_len)
    assert total > need + 45e9, "the FeMoco-shaped config is sized for a 180 GB B200 (BASELINE.json configs[3])"
    psi = workloads.make_psi(full)
    sl, sx, sy, idx = _samples(full, 48)
    vals = np.zeros(len(sl))
    a, b = fill_device_arenas(torch, full, on_chunk=lambda sub: oracle.apply_samples(sub, psi, sl, sx, sy, vals=vals))
    g = GpuProblem(full, arenas=(a, b))
    assert g.q(H.HPSI_Q_N_TASKS) > 100000 and g.q(H.HPSI_Q_ALIGNED16) == 1
    out = g.apply(psi)
    assert np.linalg.norm(out[idx] - vals) <= TOL * np.linalg.norm(vals)
    assert np.max(np.abs(out[idx] - vals)) <= 10 * TOL * np.max(np.abs(vals))
    assert np.isfinite(out).all() and np.array_equal(out, g.apply(psi))


@pytest.mark.parametrize("world", [2, 8])
@pytest.mark.parametrize("share", [False, True])
def test_term_shards_through_the_kernels(H, small, world, share):
    """The multi-GPU apply on one GPU, rank after rank: hpsi_shard_terms partitions the terms, every rank's arenas hold
    its own terms only (workloads.make_shard), hpsi_plan_ex plans the shard, hpsi_apply runs it through the DMMA
    kernels, hpsi_sum_shards adds the partial results in rank order - against the oracle on the unsharded problem,
    element by element."""
    import torch
    psi = workloads.make_psi(small)
    ref = oracle.apply(small, psi)
    desc = workloads.make_problem("small", fill=False, share_adjoint=share)
    half = desc.n_terms // 2
    shard, fl = H.hpsi_shard_terms(desc, world, np.arange(desc.n_terms) % half)
    x = torch.from_numpy(psi).cuda()
    parts, flops, tasks = [], 0, 0
    for r in range(world):
        p = workloads.make_shard("small", shard, r, share_adjoint=share)
        g = GpuProblem(p, shard_of_term=shard, shard_index=r)
        assert g.q(H.HPSI_Q_N_TERMS_PLANNED) == int((shard == r).sum())
        flops += g.q(H.HPSI_Q_USEFUL_FLOPS); tasks += g.q(H.HPSI_Q_N_TASKS)
        parts.append(g.apply_dev(x))
    assert (flops, tasks) == oracle.useful_flops(small)
    got = shard_sum(H, torch, parts)
    assert_blockwise(small, got, ref, TOL)
    assert np.array_equal(got, shard_sum(H, torch, parts))
    # in place over shard 0 is allowed, any other overlap is refused
    buf = torch.cat(parts)
    H.hpsi_sum_shards(buf, world, buf[:small.psi_len], torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert np.array_equal(buf[:small.psi_len].cpu().numpy(), got)
    with pytest.raises(H.HpsiError):
        H.hpsi_sum_shards(buf, world, buf[1:small.psi_len + 1], torch.cuda.current_stream())


def test_term_sharded_site_update_on_gpu(H):
    """Operator update under term sharding (no exchange step): every rank rotates the blocks of its own terms with the
    replicated isometries through the DMMA kernels; every block against the oracle on the full operator set."""
    import torch
    from oracle import site_update as su
    half, world = 40, 2
    full = workloads.make_problem("small", n_terms=2 * half)
    chi = workloads.proportional_chi(full.d_left, 0.25, zero_every=6)
    ot = workloads.make_isometries(full.d_left, chi, seed=5)
    otd = torch.from_numpy(np.concatenate([workloads.pack_isometries(ot), np.zeros(1)])).cuda()
    ref = su.rotate(full.d_left, chi, full.a_desc, full.a_data, ot)
    where = {(int(e["term"]), int(e["row"]), int(e["col"])): i for i, e in enumerate(full.a_desc)}
    seen = flops = 0
    for rank in range(world):
        p = workloads.make_problem("small", n_terms=2 * half, base_terms=np.arange(rank, half, world))
        gid = np.concatenate([p.base_term_ids, p.base_term_ids + half])
        a = torch.from_numpy(p.a_data).cuda()
        r = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, a, p.a_len)
        out = torch.full((H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_LENGTH),), float("nan"), dtype=torch.float64, device="cuda")
        H.hpsi_rotate_apply(r, otd, out, torch.cuda.current_stream())
        torch.cuda.synchronize()
        outh = out.cpu().numpy()
        flops += H.hpsi_rotate_query(r, H.HPSI_RQ_USEFUL_FLOPS)
        for e in H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_BLOCKS):
            x = ref[where[(int(gid[e["term"]]), int(e["row"]), int(e["col"]))]]
            seen += 1
            if e["offset"] < 0:
                assert x.size == 0
                continue
            blk = np.lib.stride_tricks.as_strided(outh[int(e["offset"]):], shape=x.shape, strides=(int(e["ld"]) * 8, 8))
            assert np.max(np.abs(blk - x)) <= 1e-12 * max(np.max(np.abs(x)), 1e-300)
    assert seen == len(full.a_desc) and flops == su.rotate_flops(full.d_left, chi, full.a_desc)


def test_plan_options_on_gpu(H, small):
    """hpsi_plan_options_t schedule knobs re-cut the work; the result stays within the bar and HPSI_Q_TUNING reports them."""
    psi = workloads.make_psi(small)
    ref = oracle.apply(small, psi)
    base = GpuProblem(small)
    for kw in (dict(p1_stages_per_unit=5), dict(p2_waves=2), dict(p2_min_unit_dmma=100000, p1_stages_per_unit=400)):
        g = GpuProblem(small, arenas=(base.a, base.b), **kw)
        assert g.q(H.HPSI_Q_TUNING) != base.q(H.HPSI_Q_TUNING)
        assert_blockwise(small, g.apply(psi), ref, TOL)


def test_task_coefficients(H, toy):
    """hpsi_set_task_coefficients: per-(t, l, l', r, r') factors; checked against the oracle on the same operator
    written with one term per task; hpsi_diagonal follows."""
    import torch
    from test_planner_cpu import exploded_problem
    p = workloads.make_problem("small", n_terms=30)
    for prob in (toy, p):
        g = GpuProblem(prob)
        f = np.random.default_rng(9).standard_normal(g.q(H.HPSI_Q_N_TASKS))
        psi = workloads.make_psi(prob)
        # stream-ordered: an apply enqueued before the call sees the old coefficients, one enqueued after it the new ones
        s = torch.cuda.Stream()
        x = torch.from_numpy(psi).cuda()
        y0, y1 = torch.full_like(x, float("nan")), torch.full_like(x, float("nan"))
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            H.hpsi_apply(g.plan, x, y0, s)
            H.hpsi_set_task_coefficients(g.plan, f, s)
            H.hpsi_apply(g.plan, x, y1, s)
        s.synchronize()
        ex = exploded_problem(prob, g.plan, f)
        assert rel_l2(y0.cpu().numpy(), oracle.apply(prob, psi)) <= TOL
        assert rel_l2(y1.cpu().numpy(), oracle.apply(ex, psi)) <= TOL
        assert rel_l2(g.apply(psi), oracle.apply(ex, psi)) <= TOL
        d = torch.empty(g.n, dtype=torch.float64, device="cuda")
        H.hpsi_diagonal(g.plan, d)
        torch.cuda.synchronize()
        ref = oracle.diagonal(ex)
        assert np.linalg.norm(d.cpu().numpy() - ref) <= 1e-12 * max(np.linalg.norm(ref), 1.0)


def _lanczos(H, g, v0, **kw):
    import torch
    x = torch.from_numpy(np.ascontiguousarray(v0)).cuda()
    theta, info = H.hpsi_lanczos(g.plan, x, **kw)
    return theta, x.cpu().numpy(), info


def test_lanczos_toy_vs_dense_and_hubbard(H, toy):
    """hpsi_lanczos ("the Lanczos or Davidson method"): lowest eigenvalue against a dense eigensolver on
    the toy config, against the textbook Hubbard closed forms, and against hpsi_davidson."""
    g = GpuProblem(toy)
    ev = np.linalg.eigvalsh(oracle.dense_hamiltonian(toy))
    theta, x, info = _lanczos(H, g, workloads.make_psi(toy), tol=1e-9, max_iter=2000, m_max=32)
    assert info["converged"] and abs(theta - ev[0]) <= 1e-10, (theta, ev[0], info)
    assert abs(np.linalg.norm(x) - 1.0) <= 1e-12
    assert np.linalg.norm(oracle.apply(toy, x) - theta * x) <= 1e-7
    th_d, _, _ = _davidson(H, g, workloads.make_psi(toy), tol=1e-9, max_iter=400)
    assert abs(theta - th_d) <= 1e-9
    dimer = hubbard_two_block_problem(1, 1, 1.0, 3.7, 2, 0)
    theta, _, info = _lanczos(H, GpuProblem(dimer), np.ones(dimer.psi_len), tol=1e-10)
    assert info["converged"] and abs(theta - (3.7 - np.sqrt(3.7 ** 2 + 16.0)) / 2) <= 1e-10
    chain = hubbard_two_block_problem(2, 2, 1.0, 0.0, 4, 0)
    v0 = np.random.default_rng(0).standard_normal(chain.psi_len)
    theta, _, info = _lanczos(H, GpuProblem(chain), v0, tol=1e-10, max_iter=500, m_max=24)
    assert info["converged"] and abs(theta + 2 * np.sqrt(5.0)) <= 1e-9


def test_lanczos_small(H, small):
    g = GpuProblem(small)
    theta, x, info = _lanczos(H, g, workloads.make_psi(small), tol=1e-6, max_iter=600, m_max=32)
    assert info["residual"] <= 1e-4
    assert np.linalg.norm(oracle.apply(small, x) - theta * x) <= 2e-4
    th_d, _, info_d = _davidson(H, g, workloads.make_psi(small), tol=1e-7, max_iter=300)
    assert info_d["converged"] and abs(theta - th_d) <= 1e-6 * max(1.0, abs(th_d))


@pytest.mark.parametrize("misalign", [False, True])
def test_shared_adjoint_storage(H, toy, misalign):
    """hpsi_terms_t a_transposed / b_transposed: adjoint terms read their partner's blocks transposed (TMA 16x16 boxes,
    or the 8-byte LDGSTS variant when misaligned); the oracle sees the fully materialised problem."""
    import torch
    for name, kw in (("toy", {}), ("small", {"n_terms": 60})):
        full = workloads.make_problem(name, **kw)
        shared = workloads.make_problem(name, share_adjoint=True, **kw)
        psi = workloads.make_psi(full, 1)
        ref = oracle.apply(full, psi)
        for flags in (0, H.HPSI_PLAN_FIXED_ORDER1, H.HPSI_PLAN_FIXED_ORDER2):
            g = GpuProblem(shared, flags, misalign=misalign)
            assert g.q(H.HPSI_Q_ALIGNED16) == (0 if misalign else 1)
            out = g.apply(psi)
            assert rel_l2(out, ref) <= TOL, (name, flags, rel_l2(out, ref))
            assert np.array_equal(out, g.apply(psi))
        d = torch.empty(g.n, dtype=torch.float64, device="cuda")
        H.hpsi_diagonal(g.plan, d)
        torch.cuda.synchronize()
        dref = oracle.diagonal(full)
        assert np.linalg.norm(d.cpu().numpy() - dref) <= 1e-12 * max(np.linalg.norm(dref), 1.0)


def test_shared_adjoint_ragged_multi_tile(H):
    """Transposed blocks spanning several tiles with ragged tails, even-but-not-multiple-of-4 leading dimensions."""
    rng = np.random.default_rng(31)
    dL, dR = [150, 70, 9], [131, 9, 77]
    n = len(dL)
    terms_full, half = [], []
    for _ in range(5):
        ab = {(r, c): rng.standard_normal((dL[r], dL[c])) for r in range(n) for c in range(n) if (r + 2 * c) % 3 != 1}
        bb = {(r, c): rng.standard_normal((dR[r], dR[c])) for r in range(n) for c in range(n) if (r + 2 * c) % 3 != 1}
        half.append((float(rng.standard_normal()), ab, bb))
    adj = [(c, {(cc, r): a.T.copy() for (r, cc), a in ab.items()}, {(cc, r): b.T.copy() for (r, cc), b in bb.items()})
           for c, ab, bb in half]
    qL, qR = [(i, 0) for i in range(n)], [(n - i, 0) for i in range(n)]
    full = workloads.custom_problem(qL, dL, qR, dR, (n, 0), half + adj, pad_even=True)
    base = workloads.custom_problem(qL, dL, qR, dR, (n, 0), half, pad_even=True)
    # shared problem: the adjoint terms' descriptors point at the base blocks, flagged transposed
    import copy
    shared = copy.copy(full)
    def share(desc_full, desc_base, nterm):
        out = desc_full.copy()
        tr = np.zeros(out.shape[0], np.uint8)
        key = {(int(e["term"]), int(e["row"]), int(e["col"])): e for e in desc_base}
        for i, e in enumerate(out):
            if e["term"] >= nterm:
                b = key[(int(e["term"]) - nterm, int(e["col"]), int(e["row"]))]
                out[i]["offset"], out[i]["ld"], tr[i] = b["offset"], b["ld"], 1
        return out, tr
    shared.a_desc, shared.a_trans = share(full.a_desc, base.a_desc, len(half))
    shared.b_desc, shared.b_trans = share(full.b_desc, base.b_desc, len(half))
    shared.a_data, shared.b_data, shared.a_len, shared.b_len = base.a_data, base.b_data, base.a_len, base.b_len
    psi = rng.standard_normal(full.psi_len)
    ref = oracle.apply(full, psi)
    for misalign in (False, True):
        assert rel_l2(GpuProblem(shared, misalign=misalign).apply(psi), ref) <= TOL


@pytest.mark.parametrize("seed", range(6))
def test_mixed_storage_irregular(H, seed):
    """Plain and transposed blocks mixed at random inside one term, on irregular structures (dims 1 .. 4, partner-less
    sectors, odd or even leading dimensions, 16-byte or 8-byte aligned arenas) and on the multi-tile ragged blocks."""
    from gpu_util import store_randomly_transposed
    rng = np.random.default_rng(100 + seed)
    if seed < 4:
        p = random_custom(seed, grid=(seed < 2))
    else:
        dL, dR = [150, 70, 9], [131, 9, 77]
        terms = []
        for _ in range(6):
            ab = {(r, c): rng.standard_normal((dL[r], dL[c])) for r in range(3) for c in range(3) if rng.random() < 0.7}
            bb = {(r, c): rng.standard_normal((dR[r], dR[c])) for r in range(3) for c in range(3) if rng.random() < 0.7}
            terms.append((float(rng.standard_normal()), ab, bb))
        p = workloads.custom_problem([(i, 0) for i in range(3)], dL, [(3 - i, 0) for i in range(3)], dR, (3, 0), terms,
                                     pad_even=(seed == 4))
    psi = rng.standard_normal(p.psi_len)
    ref = oracle.apply(p, psi)
    for k in range(2):
        q = store_randomly_transposed(p, 10 * seed + k)
        assert q.a_trans.any() or q.b_trans.any()
        for misalign in (False, True):
            out = GpuProblem(q, misalign=misalign).apply(psi)
            assert np.linalg.norm(out - ref) <= TOL * max(np.linalg.norm(ref), 1.0), (seed, k, misalign)


def _tiny_eig_problems():
    """psi_length 1; H = 0; a diagonal H; one diagonal and one dense block (the preconditioned correction of a Ritz vector
    living in the diagonal block vanishes under Gram-Schmidt)."""
    rng = np.random.default_rng(12)
    one = workloads.custom_problem([(0, 0)], [1], [(1, 0)], [1], (1, 0), [(2.0, {(0, 0): np.array([[0.7]])}, {(0, 0): np.array([[-0.3]])})])
    zero = workloads.custom_problem([(0, 0)], [3], [(1, 0)], [2], (1, 0),
                                    [(1.0, {(0, 0): np.zeros((3, 3))}, {(0, 0): np.zeros((2, 2))})])
    dvals = np.array([-2.0, 1.0, 3.0, 0.5])
    diag = workloads.custom_problem([(0, 0)], [4], [(1, 0)], [1], (1, 0), [(1.0, {(0, 0): np.diag(dvals)}, {(0, 0): np.ones((1, 1))})])
    S = rng.standard_normal((3, 3))
    mixed = workloads.custom_problem([(0, 0), (1, 0)], [4, 3], [(1, 0), (0, 0)], [1, 1], (1, 0),
                                     [(1.0, {(0, 0): np.diag(dvals), (1, 1): S + S.T}, {(0, 0): np.ones((1, 1)), (1, 1): np.ones((1, 1))})])
    return one, zero, diag, mixed


def test_eigensolvers_exact_start_vector(H):
    """psi_length 1, H = 0 and a start vector that already is the eigenvector: the residual is exactly 0 after the first
    mat-vec, the correction vector vanishes with it, and the solvers must report convergence (not a breakdown)."""
    import torch
    one, zero, diag, _ = _tiny_eig_problems()
    for p, v0, want in ((one, np.array([3.0]), 2.0 * 0.7 * -0.3), (zero, np.arange(1.0, 7.0), 0.0),
                        (diag, np.array([2.0, 0.0, 0.0, 0.0]), -2.0)):
        g = GpuProblem(p)
        for pre in (True, False):
            x = torch.from_numpy(v0.copy()).cuda()
            th, info = H.hpsi_davidson(g.plan, x, tol=1e-10, max_iter=50, precondition=pre)
            assert info["converged"] and info["residual"] <= 1e-10 and abs(th - want) <= 1e-14, (p.psi_len, pre, th, info)
            assert info["n_matvec"] == 1 and np.allclose(x.cpu().numpy(), v0 / np.linalg.norm(v0), atol=1e-14)
        x = torch.from_numpy(v0.copy()).cuda()
        th, info = H.hpsi_lanczos(g.plan, x, tol=1e-10, max_iter=50)
        assert info["converged"] and abs(th - want) <= 1e-14, (p.psi_len, th, info)
        X = torch.from_numpy(v0.copy()[None, :]).cuda()
        thm, infom = H.hpsi_davidson_multi(g.plan, X, 1, tol=1e-10, max_iter=50)
        assert infom["converged"] and abs(thm[0] - want) <= 1e-14, (p.psi_len, thm, infom)


def test_davidson_vanished_correction_takes_the_residual(H):
    """Reading A21c through the kernels: on a diagonal operator (and one with a diagonal block) the preconditioned
    correction vanishes with |r| > tol; the solvers go on with the residual and reach LAPACK's eigenvalues with the
    oracle's mat-vec count."""
    import torch
    _, _, diag, mixed = _tiny_eig_problems()
    rng = np.random.default_rng(3)
    for p in (diag, mixed):
        ev = np.linalg.eigvalsh(oracle.dense_hamiltonian(p))
        g = GpuProblem(p)
        v0 = rng.standard_normal(p.psi_len)
        for pre in (True, False):
            x = torch.from_numpy(v0.copy()).cuda()
            th, info = H.hpsi_davidson(g.plan, x, tol=1e-10, max_iter=100, precondition=pre)
            th_o, x_o, nmv_o, rn_o = oracle.davidson(p, v0, tol=1e-10, max_iter=100, precondition=pre)
            assert info["converged"] and abs(th - ev[0]) <= 1e-12 and abs(th - th_o) <= 1e-12, (pre, th, ev[0], info)
            assert info["n_matvec"] == nmv_o, (pre, info, nmv_o)
            xv = x.cpu().numpy()
            assert min(np.linalg.norm(xv - x_o), np.linalg.norm(xv + x_o)) <= 1e-8
            V0 = rng.standard_normal((p.psi_len, 2))
            thm, X, infom = _davidson_multi(H, g, V0, tol=1e-10, max_iter=200, precondition=pre)
            thb, _, nb, _ = oracle.davidson_block(p, V0, tol=1e-10, max_iter=200, precondition=pre)
            assert infom["converged"] and np.max(np.abs(thm - ev[:2])) <= 1e-12, (pre, thm, ev[:2], infom)
            assert infom["n_matvec"] == nb, (pre, infom, nb)


class _EmulatedRanks:
    """The exchange hook of a term-sharded eigensolver with all ranks on one GPU (B200_PROFILING.md: emulate the ranks as
    kernels over all ranks' data, never as processes whose kernels wait on one another): the callback plays ranks 1 ..
    world-1 - it multiplies the same vectors by their shard plans - and adds the partial results in rank order with
    hpsi_sum_shards, which is what all-gather + hpsi_sum_shards leaves on every rank of a real run."""

    def __init__(self, H, torch, p, world, n_vectors=1):
        self.H, self.torch, self.world = H, torch, world
        shard, _ = H.hpsi_shard_terms(p, world)
        self.a, self.b = torch.from_numpy(p.a_data).cuda(), torch.from_numpy(p.b_data).cuda()
        self.plans = [H.plan_problem(p, self.a, self.b, shard_of_term=shard, shard_index=r, n_vectors=n_vectors)
                      for r in range(world)]
        self.n = H.hpsi_query(self.plans[0], H.HPSI_Q_PSI_LENGTH)
        self.buf = torch.empty((world, self.n), dtype=torch.float64, device="cuda")
        self.calls, self.diag_calls = 0, 0
        H.hpsi_set_exchange(self.plans[0], self)

    def __call__(self, v, w, n, nvec, ld, stream):
        H, torch = self.H, self.torch
        assert n == self.n and (stream or 0) == torch.cuda.current_stream().cuda_stream
        st = torch.cuda.current_stream()
        wt = H.device_tensor(w, (nvec, ld), torch)
        if v is None:
            self.diag_calls += 1
            assert nvec == 1
            self.buf[0].copy_(wt[0, :n])
            for r in range(1, self.world):
                H.hpsi_diagonal(self.plans[r], self.buf[r], st)
            H.hpsi_sum_shards(self.buf, self.world, wt[0, :n], st)
            return
        self.calls += 1
        vt = H.device_tensor(v, (nvec, ld), torch)
        for k in range(nvec):
            self.buf[0].copy_(wt[k, :n])
            for r in range(1, self.world):
                H.hpsi_apply(self.plans[r], vt[k, :n], self.buf[r], st)
            H.hpsi_sum_shards(self.buf, self.world, wt[k, :n], st)


def test_eigensolvers_on_term_shards_through_the_exchange_hook(H, toy):
    """hpsi_set_exchange: the solvers run on rank 0's shard plan, every product (and diag(H)) passes through the hook, and
    the result is the full operator's eigenpair - LAPACK on the dense toy H, and the single-plan solvers."""
    import torch
    ev = np.linalg.eigvalsh(oracle.dense_hamiltonian(toy))
    Hd = oracle.dense_hamiltonian(toy)
    v0 = workloads.make_psi(toy)
    full = GpuProblem(toy)
    for world in (2, 3):
        ranks = _EmulatedRanks(H, torch, toy, world)
        plan0 = ranks.plans[0]
        for pre in (True, False):
            ranks.calls = ranks.diag_calls = 0
            x = torch.from_numpy(v0.copy()).cuda()
            th, info = H.hpsi_davidson(plan0, x, tol=1e-9, max_iter=400, precondition=pre)
            th1, _, info1 = _davidson(H, full, v0, tol=1e-9, max_iter=400, precondition=pre)
            assert info["converged"] and abs(th - ev[0]) <= 1e-10 and abs(th - th1) <= 1e-10, (world, pre, th, ev[0], info)
            assert ranks.calls == info["n_matvec"] and ranks.diag_calls == (1 if pre else 0)
            assert abs(info["n_matvec"] - info1["n_matvec"]) <= 2                   # same method, sums in another order
            xv = x.cpu().numpy()
            assert np.linalg.norm(Hd @ xv - th * xv) <= 1e-8
        ranks.calls = 0
        x = torch.from_numpy(v0.copy()).cuda()
        th, info = H.hpsi_lanczos(plan0, x, tol=1e-9, max_iter=400)
        assert info["converged"] and abs(th - ev[0]) <= 1e-10 and ranks.calls == info["n_matvec"]
    # block Davidson on a batched shard plan: the hook receives several vectors per call
    ranks = _EmulatedRanks(H, torch, toy, 2, n_vectors=3)
    V0 = np.random.default_rng(3).standard_normal((toy.psi_len, 3))
    X = torch.from_numpy(np.ascontiguousarray(V0.T)).cuda()
    th, info = H.hpsi_davidson_multi(ranks.plans[0], X, 3, tol=1e-9, max_iter=800)
    assert info["converged"] and np.max(np.abs(th - ev[:3])) <= 1e-10, (th, ev[:3], info)
    assert ranks.diag_calls == 1 and 1 <= ranks.calls <= info["n_matvec"]
    # a failing hook stops the solver with ESTATE; removing the hook gives the shard's own (different) operator
    def boom(*_a):
        raise RuntimeError("link down")
    H.hpsi_set_exchange(ranks.plans[0], boom)
    with pytest.raises(H.HpsiError) as e:
        H.hpsi_davidson(ranks.plans[0], torch.from_numpy(v0.copy()).cuda(), tol=1e-9)
    assert e.value.code == H.HPSI_ESTATE and isinstance(ranks.plans[0].exchange_error, RuntimeError)
    H.hpsi_set_exchange(ranks.plans[0], None)
    th_s, info_s = H.hpsi_davidson(ranks.plans[0], torch.from_numpy(v0.copy()).cuda(), tol=1e-9, max_iter=400)
    assert abs(th_s - ev[0]) > 1e-6


def _small_eig_cases(n, seed=0):
    """Symmetric matrices of order 1 .. 32: dense Gaussian, diagonal, zero, a degenerate lowest eigenvalue, an arrowhead
    with 1e-9 coupling (a Davidson subspace matrix near convergence), scaled by 1e+150 / 1e-150, a lowest pair 1e-13
    apart, and a Lanczos tridiagonal whose lowest Ritz value has converged."""
    rng = np.random.default_rng(seed)
    for trial in range(n):
        j, kind = int(rng.integers(1, 33)), trial % 9
        if kind == 0:
            A = rng.standard_normal((j, j))
        elif kind == 1:
            A = np.diag(rng.standard_normal(j))
        elif kind == 2:
            A = np.zeros((j, j))
        elif kind in (3, 7):
            Q, _ = np.linalg.qr(rng.standard_normal((j, j)))
            lam = np.sort(rng.standard_normal(j))
            if kind == 3:
                lam[:min(3, j)] = lam[0]
            else:
                lam = np.concatenate([[-1.0, -1.0 + 1e-13], rng.random(max(j - 2, 0))])[:j]
            A = Q @ np.diag(lam) @ Q.T
        elif kind == 4:
            A = np.diag(np.sort(rng.standard_normal(j)) * 10)
            A[-1, :] = A[:, -1] = rng.standard_normal(j) * 1e-9
            A[-1, -1] = rng.standard_normal()
        elif kind in (5, 6):
            A = rng.standard_normal((j, j)) * (1e-150 if kind == 5 else 1e150)
        else:
            n_big = 200
            M = rng.standard_normal((n_big, n_big))
            M, q, qp, b, V, al, be = M + M.T, rng.standard_normal(n_big), np.zeros(n_big), 0.0, [], [], []
            q /= np.linalg.norm(q)
            for _ in range(j):
                w = M @ q - b * qp
                a = q @ w
                w -= a * q
                for u in V:
                    w -= u * (u @ w)
                V.append(q)
                al.append(a)
                b = np.linalg.norm(w)
                be.append(b)
                qp, q = q, w / b
            A = np.diag(al) + np.diag(be[:-1], 1) + np.diag(be[:-1], -1)
        yield kind, 0.5 * (A + A.T)


def test_subspace_eigensolver_vs_lapack(H):
    """hpsi_debug_small_eig: the drivers' subspace solver on its own.  k = 1 (tridiagonalisation, multisection on the Sturm
    count, inverse iteration): lowest eigenvalue against LAPACK, residual of the vector, and the solver must not have
    needed its Jacobi fallback; k = 3 (the Jacobi solver of hpsi_davidson_multi): the three lowest pairs."""
    for kind, A in _small_eig_cases(1500):
        j = A.shape[0]
        ev = np.linalg.eigvalsh(A)
        sc = max(np.abs(ev).max(), 1e-300)
        th, y, fell_back = H.hpsi_debug_small_eig(A, 1)
        assert abs(th[0] - ev[0]) <= 1e-13 * sc and not fell_back, (kind, j, th[0], ev[0], fell_back)
        assert np.linalg.norm(A @ y[0] - th[0] * y[0]) <= 1e-12 * sc and abs(np.linalg.norm(y[0]) - 1.0) <= 1e-12, (kind, j)
        if j >= 3 and kind in (0, 1, 3, 4, 8):           # (the Jacobi solver's thresholds are absolute: not for 1e+-150 scales)
            th3, y3, _ = H.hpsi_debug_small_eig(A, 3)
            assert np.max(np.abs(th3 - ev[:3])) <= 1e-12 * sc, (kind, j, th3, ev[:3])
            assert np.max(np.abs(y3 @ y3.T - np.eye(3))) <= 1e-12
            assert np.max(np.linalg.norm(A @ y3.T - y3.T * th3[None, :], axis=0)) <= 1e-11 * sc


def test_davidson_trajectory_matches_oracle(H, small):
    """Step-by-step parity of the driver: without the (ill-conditioned) diagonal preconditioner the Ritz value and
    the residual after k mat-vecs agree with the oracle's textbook Davidson (A21) to rounding."""
    g = GpuProblem(small)
    v0 = workloads.make_psi(small)
    for it in (3, 7, 18):                       # 18 > m_max = 16: goes through a restart
        theta, _, info = _davidson(H, g, v0, tol=1e-12, max_iter=it, precondition=False)
        th_o, _, _, rn_o = oracle.davidson(small, v0, tol=1e-12, max_iter=it, precondition=False)
        assert abs(theta - th_o) <= 1e-9 * abs(th_o), (it, theta, th_o)
        assert abs(info["residual"] - rn_o) <= 1e-7 * rn_o, (it, info, rn_o)


def test_streamed_operators(H, small):
    """hpsi_stream_*: operator arenas in pinned host memory, streamed through two staging windows; several window
    sizes (1 window ... one term per window) all reproduce the oracle, and repeated applies are bitwise equal."""
    import torch
    a_host = torch.from_numpy(small.a_data).pin_memory()
    b_host = torch.from_numpy(small.b_data).pin_memory()
    psi = workloads.make_psi(small, 3)
    ref = oracle.apply(small, psi)
    x = torch.from_numpy(psi).cuda()
    per_term = (small.a_len + small.b_len) // small.n_terms
    seen = set()
    for window in (small.a_len + small.b_len, 40 * per_term, 3 * per_term):
        sp = H.hpsi_stream_create(small, a_host, b_host, window)
        nwin = H.hpsi_stream_query(sp, H.HPSI_SQ_N_WINDOWS)
        seen.add(nwin)
        assert H.hpsi_stream_query(sp, H.HPSI_Q_PSI_LENGTH) == small.psi_len
        assert H.hpsi_stream_query(sp, H.HPSI_Q_USEFUL_FLOPS) == oracle.useful_flops(small)[0]
        assert H.hpsi_stream_query(sp, H.HPSI_SQ_STAGING_BYTES) <= 2 * 8 * window + 64
        y = torch.full_like(x, float("nan"))
        H.hpsi_stream_apply(sp, x, y, torch.cuda.current_stream())
        torch.cuda.synchronize()
        out = y.cpu().numpy()
        assert rel_l2(out, ref) <= TOL, (window, nwin)
        y2 = torch.full_like(x, float("nan"))
        for _ in range(2):                                  # back-to-back applies reuse the slots correctly
            H.hpsi_stream_apply(sp, x, y2, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert np.array_equal(y2.cpu().numpy(), out)
    assert min(seen) == 1 and max(seen) > 50
    with pytest.raises(H.HpsiError):
        H.hpsi_stream_create(small, a_host, b_host, 16)     # a term does not fit the window


# ------------------------------------------------------------ batched apply and multi-root Davidson
@pytest.mark.parametrize("flags_name", ["min_flops", "order1", "order2"])
def test_apply_multi_parity(H, small, flags_name):
    """hpsi_apply_multi: nv vectors through one pass over the operators; every vector against the oracle, block by block;
    a partial batch and a strided layout give the same bits; hpsi_apply on a batched plan is the nv = 1 case."""
    import torch
    nv = 4
    g = GpuProblem(small, plan_flags(H, flags_name), n_vectors=nv)
    assert g.q(H.HPSI_Q_N_VECTORS) == nv
    psis = np.stack([workloads.make_psi(small, k) for k in range(nv)])
    refs = [oracle.apply(small, psis[k]) for k in range(nv)]
    x = torch.from_numpy(psis).cuda()
    y = torch.full_like(x, float("nan"))
    H.hpsi_apply_multi(g.plan, x, y, nv, torch.cuda.current_stream())
    torch.cuda.synchronize()
    out = y.cpu().numpy()
    for k in range(nv):
        assert_blockwise(small, out[k], refs[k], TOL)
    # two of the four vectors, 7 doubles of slack between them
    n = small.psi_len
    xs = torch.zeros(2 * (n + 7), dtype=torch.float64, device="cuda")
    ys = torch.full_like(xs, float("nan"))
    xs[:n] = x[0]; xs[n + 7:2 * n + 7] = x[1]
    H.hpsi_apply_multi(g.plan, xs, ys, 2, torch.cuda.current_stream(), ld_psi=n + 7, ld_out=n + 7)
    torch.cuda.synchronize()
    ysh = ys.cpu().numpy()
    assert np.array_equal(ysh[:n], out[0]) and np.array_equal(ysh[n + 7:2 * n + 7], out[1]) and np.isnan(ysh[n:n + 7]).all()
    assert np.array_equal(g.apply(psis[2]), out[2])
    with pytest.raises(H.HpsiError):
        H.hpsi_apply_multi(g.plan, x, y, nv + 1, torch.cuda.current_stream())
    with pytest.raises(H.HpsiError):
        H.hpsi_apply_multi(g.plan, x, x[1:], 2, torch.cuda.current_stream())        # overlapping sets


def test_apply_multi_ragged_and_unaligned(H):
    """Batched plans on irregular structures (dims 1 .. 200, odd leading dimensions, misaligned arenas: the 8-byte staging
    kernels) and on the multi-tile ragged problem."""
    import torch
    for seed in range(4):
        p = random_custom(seed, grid=(seed < 2))
        g = GpuProblem(p, misalign=bool(seed % 2), n_vectors=3)
        rng = np.random.default_rng(seed)
        psis = rng.standard_normal((3, p.psi_len))
        x = torch.from_numpy(psis).cuda()
        y = torch.full_like(x, float("nan"))
        H.hpsi_apply_multi(g.plan, x, y, 3, torch.cuda.current_stream())
        torch.cuda.synchronize()
        for k in range(3):
            ref = oracle.apply(p, psis[k])
            assert np.linalg.norm(y[k].cpu().numpy() - ref) <= TOL * max(np.linalg.norm(ref), 1.0)


def _davidson_multi(H, g, V0, **kw):
    import torch
    x = torch.from_numpy(np.ascontiguousarray(V0.T)).cuda()          # [k, n]
    theta, info = H.hpsi_davidson_multi(g.plan, x, V0.shape[1], **kw)
    return theta, x.cpu().numpy().T, info


@pytest.mark.parametrize("nvec_plan", [1, 3])
def test_davidson_multi_vs_dense_and_oracle(H, toy, nvec_plan):
    """hpsi_davidson_multi: the k lowest eigenvalues against LAPACK on the dense toy Hamiltonian, Ritz vectors orthonormal
    eigenvectors, and - without the preconditioner - the same trajectory as the oracle's block Davidson (reading A21b).
    A plan laid out for one vector runs the same method with one mat-vec per new vector."""
    g = GpuProblem(toy, n_vectors=nvec_plan)
    Hd = oracle.dense_hamiltonian(toy)
    ev = np.linalg.eigvalsh(Hd)
    k = 3
    V0 = np.random.default_rng(k).standard_normal((toy.psi_len, k))
    theta, X, info = _davidson_multi(H, g, V0, tol=1e-9, max_iter=800)
    assert info["converged"] and np.max(np.abs(theta - ev[:k])) <= 1e-10, (theta, ev[:k], info)
    assert np.max(np.abs(X.T @ X - np.eye(k))) <= 1e-11
    assert np.max(np.linalg.norm(Hd @ X - X * theta[None, :], axis=0)) <= 1e-8
    for it in (9, 20, 41):                                             # 41 > m_max: through restarts
        th_g, _, info_g = _davidson_multi(H, g, V0, tol=1e-12, max_iter=it, precondition=False)
        th_o, _, nmv_o, rn_o = oracle.davidson_block(toy, V0, tol=1e-12, max_iter=it, precondition=False)
        assert info_g["n_matvec"] == nmv_o
        assert np.max(np.abs(th_g - th_o)) <= 1e-9 * np.max(np.abs(th_o)), (it, th_g, th_o)
        assert np.max(np.abs(info_g["residuals"] - rn_o)) <= 1e-6 * np.max(rn_o)


def test_davidson_multi_hubbard_and_small(H, small):
    """Two lowest levels of the Hubbard dimer sector (closed form, tests/golden/hubbard_closed_forms.txt) and of the
    four-site chain (dense spectrum); on the D = 1024 config two roots through batched mat-vecs, residuals against the
    oracle's H."""
    dimer = hubbard_two_block_problem(1, 1, 1.0, 3.7, 2, 0)
    theta, _, info = _davidson_multi(H, GpuProblem(dimer, n_vectors=2), np.eye(4)[:, :2] + 0.1, tol=1e-11, m_max=4)
    assert info["converged"] and np.max(np.abs(theta - [(3.7 - np.sqrt(3.7 ** 2 + 16.0)) / 2, 0.0])) <= 1e-10
    chain = hubbard_two_block_problem(2, 2, 1.0, 0.0, 4, 0)
    ev = np.linalg.eigvalsh(oracle.dense_hamiltonian(chain))
    V0 = np.random.default_rng(4).standard_normal((chain.psi_len, 2))
    theta, _, info = _davidson_multi(H, GpuProblem(chain, n_vectors=2), V0, tol=1e-10, precondition=False, max_iter=400)
    assert info["converged"] and np.max(np.abs(theta - ev[:2])) <= 1e-9
    g = GpuProblem(small, n_vectors=2)
    V0 = np.stack([workloads.make_psi(small, 0), workloads.make_psi(small, 1)], axis=1)
    theta, X, info = _davidson_multi(H, g, V0, tol=1e-6, max_iter=400)
    assert info["converged"] and theta[0] < theta[1]
    for r in range(2):
        assert np.linalg.norm(oracle.apply(small, X[:, r]) - theta[r] * X[:, r]) <= 1e-5
    th1, _, _ = _davidson(H, g, V0[:, 0].copy(), tol=1e-7, max_iter=300)
    assert abs(th1 - theta[0]) <= 1e-6 * abs(th1)


def test_streamed_operators_shared_adjoint(H, small):
    """Streaming with adjoint-pair storage sharing: a term and its adjoint land in the same window, so the bytes copied per
    apply are those of the base terms only - half of the materialised form - and the result is still H psi."""
    import torch
    shared = workloads.make_problem("small", share_adjoint=True)
    a_host = torch.from_numpy(shared.a_data).pin_memory()
    b_host = torch.from_numpy(shared.b_data).pin_memory()
    psi = workloads.make_psi(small, 3)
    ref = oracle.apply(small, psi)
    x = torch.from_numpy(psi).cuda()
    full_bytes = 8 * (small.a_len + small.b_len)
    per_pair = (shared.a_len + shared.b_len) // (shared.n_terms // 2)
    for window in (shared.a_len + shared.b_len, 25 * per_pair, 2 * per_pair):
        sp = H.hpsi_stream_create(shared, a_host, b_host, window)
        copied = H.hpsi_stream_query(sp, H.HPSI_Q_OPERATOR_BYTES)
        assert copied <= 0.52 * full_bytes, (copied, full_bytes)
        assert H.hpsi_stream_query(sp, H.HPSI_Q_USEFUL_FLOPS) == oracle.useful_flops(small)[0]
        y = torch.full_like(x, float("nan"))
        H.hpsi_stream_apply(sp, x, y, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert rel_l2(y.cpu().numpy(), ref) <= TOL, (window, H.hpsi_stream_query(sp, H.HPSI_SQ_N_WINDOWS))
