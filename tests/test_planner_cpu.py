"""CPU-only tests of the product's host side: the C-ABI library loads and exports every declared symbol, the planner
validates its input, and the *device schedule* (executed by hpsi_debug_interpret with naive loops) reproduces the
oracle.  No CUDA call is made here (plans are HPSI_PLAN_HOST_ONLY)."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
import workloads
import paper_2407_07411_b200 as H
from test_oracle_pins import random_custom

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def host_plan(p, flags=0):
    return H.plan_problem(p, flags=H.HPSI_PLAN_HOST_ONLY | flags)


def rel(x, ref):
    return np.linalg.norm(x - ref) / max(np.linalg.norm(ref), 1e-300)


# ------------------------------------------------------------------------------------------------ ABI
def _declared(header):
    hdr = open(os.path.join(ROOT, "include", header)).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return set(re.findall(r"\b(hpsi_[a-z0-9_]+)\s*\(", hdr))


def test_library_exports_every_declared_symbol():
    """Every include/*.h has its library, and each library exports exactly what its header declares."""
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["hpsi.h", "hpsi_bench.h"]
    names = _declared("hpsi.h")
    assert {"hpsi_plan", "hpsi_plan_ex", "hpsi_shard_terms", "hpsi_layout_blocks", "hpsi_apply", "hpsi_apply_host",
            "hpsi_bind", "hpsi_davidson", "hpsi_query", "hpsi_destroy", "hpsi_last_error", "hpsi_diagonal",
            "hpsi_debug_interpret", "hpsi_apply_profiled"} <= names
    L = H.lib()
    for n in names:
        assert hasattr(L, n), n
    bench_names = _declared("hpsi_bench.h")
    assert bench_names == {"hpsi_bench_fp64_pipe", "hpsi_bench_last_error"}
    LB = H.binding.bench_lib()
    for n in bench_names:
        assert hasattr(LB, n), n
        assert not hasattr(L, n), f"{n}: calibration probes do not belong in the product library"


def test_schedule_ignores_the_environment(small, monkeypatch):
    """A plan depends on its arguments only: no environment variable changes the schedule (the old tuning hooks)."""
    base = host_plan(small)
    want = [H.hpsi_query(base, w) for w in (H.HPSI_Q_N_P1_UNITS, H.HPSI_Q_N_P2_UNITS, H.HPSI_Q_N_FUSED_UNITS)]
    for k, v in (("HPSI_FUSE", "1"), ("HPSI_P1_STAGES", "7"), ("HPSI_P2_WAVES", "3"), ("HPSI_P2_MIN", "99999"), ("HPSI_DEBUG", "2")):
        monkeypatch.setenv(k, v)
    again = host_plan(small)
    assert [H.hpsi_query(again, w) for w in (H.HPSI_Q_N_P1_UNITS, H.HPSI_Q_N_P2_UNITS, H.HPSI_Q_N_FUSED_UNITS)] == want
    assert H.hpsi_query(again, H.HPSI_Q_TUNING) == H.hpsi_query(base, H.HPSI_Q_TUNING)


def test_plan_options_change_the_schedule_not_the_result(small):
    """hpsi_plan_options_t knobs are visible through HPSI_Q_TUNING and only re-cut the work."""
    psi = workloads.make_psi(small)
    ref = oracle.apply(small, psi)
    base = host_plan(small)
    t0 = H.hpsi_query(base, H.HPSI_Q_TUNING)
    assert 8 <= t0[1] <= 48 and t0[2] == 3072 and 12 <= t0[0] <= 96
    for kw in (dict(p1_stages_per_unit=7), dict(p2_waves=3), dict(p2_min_unit_dmma=200000), dict(p1_stages_per_unit=500, p2_waves=100)):
        plan = H.plan_problem(small, flags=H.HPSI_PLAN_HOST_ONLY, **kw)
        t = H.hpsi_query(plan, H.HPSI_Q_TUNING)
        assert t != t0
        for k, v in kw.items():
            assert t[("p1_stages_per_unit", "p2_waves", "p2_min_unit_dmma").index(k)] == v
        assert rel(H.hpsi_debug_interpret(plan, small.a_data, small.b_data, psi), ref) <= 1e-13
    with pytest.raises(H.HpsiError):
        H.plan_problem(small, flags=H.HPSI_PLAN_HOST_ONLY, p2_waves=-1)


def test_preferred_layout_query_and_layout_blocks(small):
    """SURVEY.md 8(b) "preferred ld / arena layout": the rule as a query, and hpsi_layout_blocks applying it - a caller
    can describe its blocks, let the library lay them out, fill the arenas and plan (arenas bound later)."""
    lay = H.hpsi_query(host_plan(small), H.HPSI_Q_PREFERRED_LAYOUT)
    assert lay == {"ld_multiple": 4, "offset_multiple": 4, "tma_ld_multiple": 2, "tma_offset_multiple": 2,
                   "arena_align_bytes": 16, "transposed_pad_rows": 8}
    dense = workloads.make_problem("small", n_terms=20, pad_even=False)           # odd lds, dense offsets
    a_desc, a_len = H.hpsi_layout_blocks(dense.d_left, dense.a_desc)
    b_desc, b_len = H.hpsi_layout_blocks(dense.d_right, dense.b_desc)
    for desc, dims, n in ((a_desc, dense.d_left, a_len), (b_desc, dense.d_right, b_len)):
        assert np.all(desc["ld"] % lay["ld_multiple"] == 0) and np.all(desc["offset"] % lay["offset_multiple"] == 0)
        assert np.all(desc["ld"] >= dims[desc["col"]]) and np.all(desc["ld"] < dims[desc["col"]] + 4)
        ends = desc["offset"] + dims[desc["row"]].astype(np.int64) * desc["ld"]
        assert np.all(desc["offset"][1:] >= ends[:-1]) and n >= ends[-1]          # no overlap, in the order given
    # the library's layout is the generator's preferred one (row_align = 4)
    pref = workloads.make_problem("small", n_terms=20)
    assert np.array_equal(a_desc, pref.a_desc) and np.array_equal(b_desc, pref.b_desc) and (a_len, b_len) == (pref.a_len, pref.b_len)
    # move the entries into that layout and plan: same operator
    import copy
    moved = copy.copy(dense)
    moved.a_desc, moved.b_desc, moved.a_len, moved.b_len = a_desc, b_desc, a_len, b_len
    moved.a_data, moved.b_data = np.full(a_len, np.nan), np.full(b_len, np.nan)
    for side, old, new, data, dims in (("a", dense.a_desc, a_desc, moved.a_data, dense.d_left), ("b", dense.b_desc, b_desc, moved.b_data, dense.d_right)):
        for i, e in enumerate(new):
            r, c = int(dims[e["row"]]), int(dims[e["col"]])
            np.lib.stride_tricks.as_strided(data[int(e["offset"]):], shape=(r, c), strides=(int(e["ld"]) * 8, 8))[...] = dense.block(side, i)
    plan = host_plan(moved)
    assert H.hpsi_query(plan, H.HPSI_Q_ALIGNED16) == 1 and H.hpsi_query(host_plan(dense), H.HPSI_Q_ALIGNED16) == 0
    psi = workloads.make_psi(dense)
    assert rel(H.hpsi_debug_interpret(plan, moved.a_data, moved.b_data, psi), oracle.apply(dense, psi)) <= 1e-13
    # transposed blocks store d[col] x d[row]; ld == -1 marks a descriptor that shares storage and is left alone
    sh = workloads.make_problem("toy", share_adjoint=True)
    probe = sh.a_desc.copy()
    probe["ld"][sh.a_trans == 1] = -1
    laid, n = H.hpsi_layout_blocks(sh.d_left, probe, sh.a_trans)
    own = sh.a_trans == 0
    assert np.array_equal(laid[own], sh.a_desc[own]) and np.all(laid["ld"][~own] == -1) and n == sh.a_len


def test_shard_terms_partition(small):
    """hpsi_shard_terms: deterministic, balanced by useful flops, bundles stay together, every term placed; the shards
    planned with hpsi_plan_ex partition the tasks and the flops."""
    T, half = small.n_terms, small.n_terms // 2
    flops, ntask = oracle.useful_flops(small)
    for world in (1, 2, 5, 8):
        shard, fl = H.hpsi_shard_terms(small, world, np.arange(T) % half)
        assert shard.min() >= 0 and shard.max() < world and np.array_equal(shard[:half], shard[half:])
        assert int(fl.sum()) == flops and fl.max() <= 1.02 * fl.mean()
        again, _ = H.hpsi_shard_terms(small, world, np.arange(T) % half)
        assert np.array_equal(shard, again)
        tot_tasks = tot_flops = tot_terms = 0
        for r in range(world):
            plan = H.plan_problem(small, flags=H.HPSI_PLAN_HOST_ONLY, shard_of_term=shard, shard_index=r)
            assert H.hpsi_query(plan, H.HPSI_Q_USEFUL_FLOPS) == fl[r]
            tasks = H.hpsi_query(plan, H.HPSI_Q_TASKS)
            assert np.all(shard[tasks["term"]] == r)
            tot_tasks += len(tasks); tot_flops += int(fl[r]); tot_terms += H.hpsi_query(plan, H.HPSI_Q_N_TERMS_PLANNED)
        assert (tot_tasks, tot_flops, tot_terms) == (ntask, flops, T)
    alone, fl = H.hpsi_shard_terms(small, 4)                        # no bundles: every term on its own
    assert int(fl.sum()) == flops and fl.max() <= 1.02 * fl.mean()
    with pytest.raises(H.HpsiError):
        H.hpsi_shard_terms(small, 0)


def test_shard_plan_never_reads_other_terms(small):
    """A shard's arenas hold only its own terms (workloads.make_shard gives the other descriptors offset -1): the plan
    must accept that, and the shards' results must add up to the oracle's H psi element by element."""
    T, half = small.n_terms, small.n_terms // 2
    psi = workloads.make_psi(small)
    ref = oracle.apply(small, psi)
    for share in (False, True):
        desc = workloads.make_problem("small", fill=False, share_adjoint=share)
        shard, fl = H.hpsi_shard_terms(desc, 3, np.arange(T) % half)
        tot, a_doubles = np.zeros_like(ref), 0
        for r in range(3):
            p = workloads.make_shard("small", shard, r, share_adjoint=share)
            assert np.all(p.a_desc["offset"][shard[p.a_desc["term"]] != r] == -1)
            a_doubles += p.a_len
            plan = H.plan_problem(p, flags=H.HPSI_PLAN_HOST_ONLY, shard_of_term=shard, shard_index=r)
            tot += H.hpsi_debug_interpret(plan, p.a_data, p.b_data, psi)
            with pytest.raises(H.HpsiError):                      # without the shard map the -1 offsets are rejected
                H.plan_problem(p, flags=H.HPSI_PLAN_HOST_ONLY)
        assert a_doubles == desc.a_len                            # the shards partition the operator storage
        assert rel(tot, ref) <= 1e-13


def test_opblock_layout_matches_header():
    assert workloads.OPBLOCK_DTYPE.itemsize == 24
    assert [workloads.OPBLOCK_DTYPE.fields[k][1] for k in ("term", "row", "col", "ld", "offset")] == [0, 4, 8, 12, 16]


def test_no_cpu_fallback(toy):
    """Compute entry points refuse to run without a device plan (no CPU fallback exists)."""
    plan = host_plan(toy)
    x = np.zeros(H.hpsi_query(plan, H.HPSI_Q_PSI_LENGTH))
    with pytest.raises(H.HpsiError) as e:
        H.hpsi_apply(plan, x.ctypes.data, x.ctypes.data + 8, None)
    assert e.value.code == H.HPSI_ESTATE
    with pytest.raises(H.HpsiError):
        H.hpsi_apply_host(plan, x, x.copy(), None)


# ------------------------------------------------------------------------------------------ psi table
def test_psi_blocks_match_oracle_table(toy, small):
    for p in (toy, small, random_custom(3), random_custom(6, grid=False)):
        plan = host_plan(p)
        blocks = H.hpsi_query(plan, H.HPSI_Q_PSI_BLOCKS)
        partner, offset, n = oracle.psi_table(p)
        assert H.hpsi_query(plan, H.HPSI_Q_PSI_LENGTH) == n
        want = [(i, int(partner[i]), int(p.d_left[i]), int(p.d_right[partner[i]]), int(offset[i]))
                for i in range(len(partner)) if partner[i] >= 0]
        got = [(int(b["left"]), int(b["right"]), int(b["rows"]), int(b["cols"]), int(b["offset"])) for b in blocks]
        assert got == want


# ------------------------------------------------------------------------- schedule == oracle (CPU)
@pytest.mark.parametrize("flags", [0, H.HPSI_PLAN_FIXED_ORDER1, H.HPSI_PLAN_FIXED_ORDER2, H.HPSI_PLAN_FUSE_ALL,
                                   H.HPSI_PLAN_FUSE_ALL | H.HPSI_PLAN_FIXED_ORDER1, H.HPSI_PLAN_FUSE_ALL | H.HPSI_PLAN_FIXED_ORDER2])
def test_schedule_interpreter_toy(toy, flags):
    plan = host_plan(toy, flags)
    for k in range(2):
        psi = workloads.make_psi(toy, k)
        assert rel(H.hpsi_debug_interpret(plan, toy.a_data, toy.b_data, psi), oracle.apply(toy, psi)) <= 1e-13


@pytest.mark.parametrize("flags", [0, H.HPSI_PLAN_FUSE_ALL])
def test_schedule_interpreter_small(small, flags):
    plan = host_plan(small, flags)
    psi = workloads.make_psi(small)
    assert rel(H.hpsi_debug_interpret(plan, small.a_data, small.b_data, psi), oracle.apply(small, psi)) <= 1e-13
    fused = H.hpsi_query(plan, H.HPSI_Q_N_FUSED_TASKS)
    if flags:      # the narrow groups go to fused units and write no intermediate; the others keep the two-launch path
        assert 0 < fused < H.hpsi_query(plan, H.HPSI_Q_N_TASKS) and H.hpsi_query(plan, H.HPSI_Q_N_FUSED_UNITS) > 0
        assert H.hpsi_query(plan, H.HPSI_Q_INTERMEDIATE_BYTES) < H.hpsi_query(host_plan(small), H.HPSI_Q_INTERMEDIATE_BYTES)
        assert H.hpsi_query(plan, H.HPSI_Q_LAUNCHES_PER_APPLY) == 5
        assert H.hpsi_query(host_plan(small, flags | H.HPSI_PLAN_NO_FUSION), H.HPSI_Q_N_FUSED_TASKS) == 0
    else:
        assert fused == 0 and H.hpsi_query(plan, H.HPSI_Q_LAUNCHES_PER_APPLY) == 4


@pytest.mark.parametrize("seed", range(8))
def test_schedule_interpreter_irregular(seed):
    """Partner-less sectors, non-shift block patterns, dense (odd) and padded leading dimensions."""
    p = random_custom(seed, grid=(seed < 4))
    plan = host_plan(p)
    psi = np.random.default_rng(seed).standard_normal(p.psi_len)
    ref = oracle.apply(p, psi)
    got = H.hpsi_debug_interpret(plan, p.a_data, p.b_data, psi)
    assert np.linalg.norm(got - ref) <= 1e-13 * max(np.linalg.norm(ref), 1.0)
    assert H.hpsi_query(plan, H.HPSI_Q_ALIGNED16) == (1 if seed % 2 else 0) or p.a_desc.size == 0


def test_schedule_split_k_and_multi_tile():
    """A problem whose output block spans several 64x64 tiles with a ragged tail and whose K is split."""
    rng = np.random.default_rng(5)
    dL, dR = [150, 70], [131, 9]
    qL, qR = [(0, 0), (1, 1)], [(3, 1), (2, 0)]
    terms = []
    for _ in range(40):
        ab = {(r, c): rng.standard_normal((dL[r], dL[c])) for r in range(2) for c in range(2)}
        bb = {(r, c): rng.standard_normal((dR[r], dR[c])) for r in range(2) for c in range(2)}
        terms.append((float(rng.standard_normal()), ab, bb))
    p = workloads.custom_problem(qL, dL, qR, dR, (3, 1), terms, pad_even=True)
    plan = host_plan(p)
    assert H.hpsi_query(plan, H.HPSI_Q_N_P2_UNITS) > 6
    psi = rng.standard_normal(p.psi_len)
    assert rel(H.hpsi_debug_interpret(plan, p.a_data, p.b_data, psi), oracle.apply(p, psi)) <= 1e-13


# ---------------------------------------------------------------------------------- counts and flops
def test_flop_and_task_counts(toy, small):
    for p in (toy, small):
        plan = host_plan(p)
        flops, ntask = oracle.useful_flops(p)
        assert H.hpsi_query(plan, H.HPSI_Q_N_TASKS) == ntask
        assert H.hpsi_query(plan, H.HPSI_Q_USEFUL_FLOPS) == flops
        assert H.hpsi_query(plan, H.HPSI_Q_ISSUED_FLOPS) >= flops
        assert H.hpsi_query(plan, H.HPSI_Q_OPERATOR_BYTES) <= p.operator_bytes()
        tasks = H.hpsi_query(plan, H.HPSI_Q_TASKS)
        assert len(tasks) == ntask and set(np.unique(tasks["order"])) <= {1, 2}


def test_order_choice_is_min_flops(small):
    """Per task the planner picks min(2mn'(k+n), 2kn(n'+m)); forcing either order can only cost more DMMA work."""
    free = H.hpsi_query(host_plan(small), H.HPSI_Q_USEFUL_FLOPS)
    plan = host_plan(small)
    partner = small.partner
    for t in H.hpsi_query(plan, H.HPSI_Q_TASKS):
        l, lp = int(t["dst_left"]), int(t["src_left"])
        m, k = int(small.d_left[l]), int(small.d_left[lp])
        n, n1 = int(small.d_right[partner[l]]), int(small.d_right[partner[lp]])
        f1, f2 = 2 * m * n1 * (k + n), 2 * k * n * (n1 + m)
        assert int(t["order"]) == (2 if f2 < f1 else 1)
    assert free == oracle.useful_flops(small)[0]


def test_useful_flops_scale_as_D_cubed():
    """PAPER.md:62 / :82 - cost O(D^3): doubling every sector dim multiplies the useful flops by exactly 8."""
    base = workloads.make_problem("toy", fill=False)
    dbl = workloads.make_problem("toy", fill=False)
    dbl.d_left = (2 * base.d_left).astype(np.int32)
    dbl.d_right = (2 * base.d_right).astype(np.int32)
    dbl.a_desc = dbl.a_desc.copy(); dbl.b_desc = dbl.b_desc.copy()
    dbl.a_desc["ld"] *= 2; dbl.b_desc["ld"] *= 2
    dbl.a_desc["offset"] *= 4; dbl.b_desc["offset"] *= 4
    dbl.a_len *= 4; dbl.b_len *= 4
    f1 = H.hpsi_query(host_plan(base), H.HPSI_Q_USEFUL_FLOPS)
    f2 = H.hpsi_query(host_plan(dbl), H.HPSI_Q_USEFUL_FLOPS)
    assert f2 == 8 * f1


# ----------------------------------------------------------------------------------------- validation
def _expect_einval(p, match):
    with pytest.raises(H.HpsiError) as e:
        host_plan(p)
    assert e.value.code == H.HPSI_EINVAL and match in str(e.value)


def test_validation_errors():
    p = workloads.make_problem("toy")
    bad = workloads.make_problem("toy"); bad.q_left = bad.q_left.copy(); bad.q_left[1] = bad.q_left[0]
    _expect_einval(bad, "duplicate")
    bad = workloads.make_problem("toy"); bad.d_right = bad.d_right.copy(); bad.d_right[2] = 0
    _expect_einval(bad, "dimension")
    bad = workloads.make_problem("toy"); bad.a_desc = bad.a_desc.copy(); bad.a_desc["ld"][0] = 0
    _expect_einval(bad, "ld")
    bad = workloads.make_problem("toy"); bad.b_desc = bad.b_desc.copy(); bad.b_desc["offset"][-1] = bad.b_len
    _expect_einval(bad, "arena")
    bad = workloads.make_problem("toy"); bad.a_desc = np.concatenate([bad.a_desc, bad.a_desc[:1]])
    _expect_einval(bad, "two blocks")
    bad = workloads.make_problem("toy"); bad.a_desc = bad.a_desc.copy(); bad.a_desc["term"][0] = p.n_terms
    _expect_einval(bad, "term")


def test_empty_problems():
    """No terms / no psi blocks are legal: the schedule is empty and the result is zeros."""
    p = workloads.make_problem("toy", n_terms=0)
    plan = host_plan(p)
    assert H.hpsi_query(plan, H.HPSI_Q_N_TASKS) == 0
    out = H.hpsi_debug_interpret(plan, p.a_data, p.b_data, workloads.make_psi(p))
    assert np.all(out == 0.0)
    q = workloads.custom_problem([(0, 0)], [2], [(5, 5)], [3], (1, 1), [(1.0, {(0, 0): np.eye(2)}, {(0, 0): np.eye(3)})])
    plan = host_plan(q)
    assert H.hpsi_query(plan, H.HPSI_Q_PSI_LENGTH) == 0 and H.hpsi_query(plan, H.HPSI_Q_N_TASKS) == 0


def test_struct_sizes():
    assert ctypes.sizeof(H.binding.hpsi_sectors_t) == 48
    assert ctypes.sizeof(H.binding.hpsi_terms_t) == 96      # + a_transposed, b_transposed
    assert ctypes.sizeof(H.binding.hpsi_plan_options_t) == 32 and ctypes.sizeof(H.binding.hpsi_layout_t) == 24
    assert H.binding.PSI_BLOCK_DTYPE.itemsize == 24 and H.binding.TASK_DTYPE.itemsize == 24


# --------------------------------------------------------------------------------- tile / warp-grid policy
def test_schedule_balance_on_cyp_shapes():
    """The planner's tile split (even fragment counts, at most one odd tile per dimension) and per-unit warp grid keep
    the heaviest warp of a CTA close to the mean: issued / critical-path DMMA flops >= 0.97 on the cyp-shaped config
    (it was 0.865 with an even split and a fixed 2x2 grid), and padding to 8x8x4 fragments costs < 7 %."""
    p = workloads.make_problem("cyp", fill=False)
    plan = host_plan(p)
    useful, issued = H.hpsi_query(plan, H.HPSI_Q_USEFUL_FLOPS), H.hpsi_query(plan, H.HPSI_Q_ISSUED_FLOPS)
    critical = H.hpsi_query(plan, H.HPSI_Q_CRITICAL_FLOPS)
    assert useful <= issued <= critical
    assert issued / critical >= 0.97
    assert useful / issued >= 0.93
    # ~32 waves of P2 units on 148 SMs x 4 slots, and P1 units that bundle several terms
    assert 148 * 4 * 16 <= H.hpsi_query(plan, H.HPSI_Q_N_P2_UNITS) <= 148 * 4 * 64
    assert H.hpsi_query(plan, H.HPSI_Q_N_P1_UNITS) < H.hpsi_query(plan, H.HPSI_Q_N_TASKS)


def test_interpreter_parity_with_uneven_tiles():
    """Dimensions whose fragment counts exercise every branch of the tile split (9, 10, 13, 15, 17 fragments) and of
    the warp-grid choice, through the host interpreter of the device schedule."""
    rng = np.random.default_rng(17)
    dL, dR = [72, 80, 104, 9], [120, 136, 65, 130]
    n = len(dL)
    terms = []
    for _ in range(3):
        ab = {(r, c): rng.standard_normal((dL[r], dL[c])) for r in range(n) for c in range(n) if (r + c) % 3 != 1}
        bb = {(r, c): rng.standard_normal((dR[r], dR[c])) for r in range(n) for c in range(n) if (r + c) % 3 != 1}
        terms.append((float(rng.standard_normal()), ab, bb))
    p = workloads.custom_problem([(i, 0) for i in range(n)], dL, [(n - i, 0) for i in range(n)], dR, (n, 0), terms,
                                 pad_even=True)
    psi = rng.standard_normal(p.psi_len)
    ref = oracle.apply(p, psi)
    for flags in (0, H.HPSI_PLAN_FIXED_ORDER1, H.HPSI_PLAN_FIXED_ORDER2):
        plan = host_plan(p, flags)
        assert rel(H.hpsi_debug_interpret(plan, p.a_data, p.b_data, psi), ref) <= 1e-13


# ------------------------------------------------------------------------------ per-task coefficients (8(f)-2)
def exploded_problem(p, plan, task_coef):
    """The same operator with every task turned into its own one-block term carrying the task's coefficient: what
    hpsi_set_task_coefficients must compute, expressed in the boundary's plain per-term form for the oracle."""
    tasks = H.hpsi_query(plan, H.HPSI_Q_TASKS)
    terms = []
    for t, f in zip(tasks, task_coef):
        ea, eb = p.a_desc[int(t["a_block"])], p.b_desc[int(t["b_block"])]
        terms.append((float(f), {(int(ea["row"]), int(ea["col"])): p.block("a", int(t["a_block"]))},
                      {(int(eb["row"]), int(eb["col"])): p.block("b", int(t["b_block"]))}))
    return workloads.custom_problem(p.q_left, p.d_left, p.q_right, p.d_right, p.target, terms)


def test_task_coefficients_interpreter(toy):
    plan = host_plan(toy)
    n_tasks = H.hpsi_query(plan, H.HPSI_Q_N_TASKS)
    f = np.random.default_rng(5).standard_normal(n_tasks)
    with pytest.raises(H.HpsiError):
        H.hpsi_set_task_coefficients(plan, f[:-1])
    H.hpsi_set_task_coefficients(plan, f)
    psi = workloads.make_psi(toy)
    ref = oracle.apply(exploded_problem(toy, plan, f), psi)
    assert rel(H.hpsi_debug_interpret(plan, toy.a_data, toy.b_data, psi), ref) <= 1e-13
    # back to the per-term coefficients
    tasks = H.hpsi_query(plan, H.HPSI_Q_TASKS)
    H.hpsi_set_task_coefficients(plan, toy.coef[tasks["term"]])
    assert rel(H.hpsi_debug_interpret(plan, toy.a_data, toy.b_data, psi), oracle.apply(toy, psi)) <= 1e-13


# ------------------------------------------------------------------- adjoint-pair storage sharing (8(f)-2)
@pytest.mark.parametrize("name,kw", [("toy", {}), ("small", {"n_terms": 40})])
def test_shared_adjoint_storage_interpreter(name, kw):
    """Adjoint terms that point at their partner's storage (blocks flagged transposed) give the same operator as the
    fully materialised problem the oracle sees; the arenas are half as long."""
    full = workloads.make_problem(name, **kw)
    shared = workloads.make_problem(name, share_adjoint=True, **kw)
    assert shared.a_len <= 0.51 * full.a_len and shared.b_len <= 0.51 * full.b_len
    assert int(shared.a_trans.sum()) == full.a_desc.shape[0] // 2
    psi = workloads.make_psi(full)
    ref = oracle.apply(full, psi)
    for flags in (0, H.HPSI_PLAN_FIXED_ORDER1, H.HPSI_PLAN_FIXED_ORDER2):
        plan = host_plan(shared, flags)
        assert H.hpsi_query(plan, H.HPSI_Q_N_TASKS) == H.hpsi_query(host_plan(full, flags), H.HPSI_Q_N_TASKS)
        assert rel(H.hpsi_debug_interpret(plan, shared.a_data, shared.b_data, psi), ref) <= 1e-13


@pytest.mark.parametrize("seed", range(6))
def test_mixed_storage_interpreter(seed):
    """Plain and transposed blocks mixed at random inside one term (irregular structures, odd and even leading dimensions,
    every order): the A and B flags of a task are independent, so neither GEMM may assume the other's layout boundary."""
    from gpu_util import store_randomly_transposed
    for grid in (True, False):
        p = random_custom(seed, grid=grid)
        psi = np.random.default_rng(seed).standard_normal(p.psi_len)
        ref = oracle.apply(p, psi)
        for k in range(3):
            q = store_randomly_transposed(p, 10 * seed + k)
            assert q.a_trans.any() or q.b_trans.any()
            for flags in (0, H.HPSI_PLAN_FIXED_ORDER1, H.HPSI_PLAN_FIXED_ORDER2):
                got = H.hpsi_debug_interpret(host_plan(q, flags), q.a_data, q.b_data, psi)
                assert np.linalg.norm(got - ref) <= 1e-13 * max(np.linalg.norm(ref), 1.0), (grid, k, flags)


def test_set_exchange_arguments(toy):
    """hpsi_set_exchange on a host-only plan: setting and clearing the hook are plain state changes; a null plan is EINVAL."""
    plan = host_plan(toy)
    H.hpsi_set_exchange(plan, lambda *a: None)
    H.hpsi_set_exchange(plan, None)
    assert H.lib().hpsi_set_exchange(None, None, None) == H.HPSI_EINVAL


def test_transposed_block_validation(toy):
    shared = workloads.make_problem("toy", share_adjoint=True)
    bad = shared.a_desc.copy()
    j = int(np.flatnonzero(shared.a_trans)[0])
    bad[j]["ld"] = 0                                            # ld < stored columns
    with pytest.raises(H.HpsiError) as e:
        H.hpsi_plan(shared.q_left, shared.q_right, shared.d_left, shared.d_right, shared.target, shared.coef, bad,
                    shared.b_desc, None, None, shared.a_len, shared.b_len, H.HPSI_PLAN_HOST_ONLY, shared.a_trans, shared.b_trans)
    assert e.value.code == H.HPSI_EINVAL


# --------------------------------------------------------------------------------- batched plans (n_vectors > 1)
@pytest.mark.parametrize("flags", [0, H.HPSI_PLAN_FIXED_ORDER1, H.HPSI_PLAN_FIXED_ORDER2])
def test_batched_schedule_interpreter(toy, flags):
    """hpsi_plan_options_t.n_vectors: the schedule of a batched apply (vectors side by side in the intermediate, one unit
    per tile and vector) executed by the host interpreter gives H psi_v for every vector; fewer vectors than planned are
    a prefix of the same work; flop / byte queries stay per vector; transposed blocks and the fused kernel are refused."""
    for p in (toy, workloads.make_problem("small", n_terms=40), random_custom(5)):
        single = host_plan(p, flags)
        plan = H.plan_problem(p, flags=H.HPSI_PLAN_HOST_ONLY | flags, n_vectors=3)
        assert H.hpsi_query(plan, H.HPSI_Q_N_VECTORS) == 3 and H.hpsi_query(single, H.HPSI_Q_N_VECTORS) == 1
        rng = np.random.default_rng(1)
        psis = rng.standard_normal((3, p.psi_len))
        out = H.hpsi_debug_interpret(plan, p.a_data, p.b_data, psis)
        for k in range(3):
            ref = oracle.apply(p, psis[k])
            assert np.linalg.norm(out[k] - ref) <= 1e-13 * max(np.linalg.norm(ref), 1.0)
        assert np.array_equal(H.hpsi_debug_interpret(plan, p.a_data, p.b_data, psis[:2]), out[:2])
        assert np.array_equal(H.hpsi_debug_interpret(plan, p.a_data, p.b_data, psis[0]), out[0])
        for w in (H.HPSI_Q_USEFUL_FLOPS, H.HPSI_Q_ISSUED_FLOPS, H.HPSI_Q_OPERATOR_BYTES, H.HPSI_Q_N_TASKS):
            assert H.hpsi_query(plan, w) == H.hpsi_query(single, w)
        assert H.hpsi_query(plan, H.HPSI_Q_N_P1_UNITS) == 3 * H.hpsi_query(single, H.HPSI_Q_N_P1_UNITS)
    with pytest.raises(H.HpsiError):
        H.plan_problem(workloads.make_problem("toy", share_adjoint=True), flags=H.HPSI_PLAN_HOST_ONLY, n_vectors=2)
    with pytest.raises(H.HpsiError):
        H.plan_problem(toy, flags=H.HPSI_PLAN_HOST_ONLY | H.HPSI_PLAN_FUSE_ALL, n_vectors=2)
    with pytest.raises(H.HpsiError):
        H.plan_problem(toy, flags=H.HPSI_PLAN_HOST_ONLY, n_vectors=65)


# --------------------------------------------------------------------- argument checks of the round-2 entry points
def test_new_entry_points_refuse_bad_arguments(toy):
    """No device is needed to be refused: host-only plans answer ESTATE to every compute call (no CPU fallback), bad
    arguments EINVAL, and hpsi_plan_options_t is versioned by its size."""
    plan = host_plan(toy)
    n = H.hpsi_query(plan, H.HPSI_Q_PSI_LENGTH)
    x = np.zeros(2 * n)
    L = H.lib()
    st = ctypes.c_void_p
    # batched apply on a single-vector plan / a host-only plan
    assert L.hpsi_apply_multi(plan.handle, x.ctypes.data, n, x.ctypes.data + 8 * n, n, 2, None) == H.HPSI_EINVAL
    plan2 = H.plan_problem(toy, flags=H.HPSI_PLAN_HOST_ONLY, n_vectors=2)
    y = np.zeros(2 * n)
    assert L.hpsi_apply_multi(plan2.handle, x.ctypes.data, n, y.ctypes.data, n, 2, None) == H.HPSI_ESTATE
    assert L.hpsi_apply_multi(plan2.handle, x.ctypes.data, n - 1, y.ctypes.data, n, 2, None) == H.HPSI_EINVAL     # stride < psi_length
    assert L.hpsi_apply_multi(plan2.handle, x.ctypes.data, n, x.ctypes.data + 8, n, 2, None) == H.HPSI_EINVAL     # overlap
    # eigensolvers
    eig = (ctypes.c_double * 4)()
    prm = H.binding.hpsi_davidson_params_t(1e-8, 10, 16, 1)
    assert L.hpsi_davidson_multi(plan2.handle, x.ctypes.data, n, 2, eig, None, ctypes.byref(prm), None, None) == H.HPSI_ESTATE
    assert L.hpsi_davidson_multi(None, x.ctypes.data, n, 2, eig, None, ctypes.byref(prm), None, None) == H.HPSI_EINVAL
    # hpsi_sum_shards: argument checks come before any CUDA call
    assert L.hpsi_sum_shards(x.ctypes.data, 0, n, y.ctypes.data, None) == H.HPSI_EINVAL
    assert L.hpsi_sum_shards(None, 2, n, y.ctypes.data, None) == H.HPSI_EINVAL
    assert L.hpsi_sum_shards(x.ctypes.data, 2, n, x.ctypes.data + 8, None) == H.HPSI_EINVAL                       # overlapping, not in place
    assert L.hpsi_sum_shards(x.ctypes.data, 2, 0, y.ctypes.data, None) == H.HPSI_OK                               # nothing to do
    # options struct smaller than the library's: refused, not misread
    sec, trm, keep = H.binding._marshal(toy.q_left, toy.q_right, toy.d_left, toy.d_right, toy.target, toy.coef, toy.a_desc,
                                        toy.b_desc, None, None, toy.a_len, toy.b_len, None, None)
    opt = H.binding.hpsi_plan_options_t(8, 0, None, 0, 0, 0, 0)
    out = ctypes.c_void_p()
    assert L.hpsi_plan_ex(ctypes.byref(sec), ctypes.byref(trm), H.HPSI_PLAN_HOST_ONLY, ctypes.byref(opt), ctypes.byref(out)) == H.HPSI_EINVAL
    assert out.value is None and b"struct_bytes" in L.hpsi_last_error()
    # layout helper
    bad = toy.a_desc.copy(); bad["row"][0] = 99
    with pytest.raises(H.HpsiError):
        H.hpsi_layout_blocks(toy.d_left, bad)
    del st
