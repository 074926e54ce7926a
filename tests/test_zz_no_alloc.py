"""hpsi_truncate_static: the truncation for callers that may not allocate device memory (its scratch is a static
__device__ array of HPSI_TRUNCATE_STATIC_BYTES inside the library).  Checked against hpsi_truncate - the existing path,
which keeps its buffers in a cudaMalloc block on the plan - on two calls in a row that share the array (different psi,
different side), against the oracle, for the size limit, and for "allocates nothing".

This file is named so that pytest collects it last: the suite runs with `pytest -x`, and a failure here must not hide
the other tests.  It passes alone in a fresh process and after the rest of the suite."""
import numpy as np
import pytest

import workloads
from oracle import site_update as su

pytestmark = pytest.mark.gpu

TOL = 1e-12            # the site-update tests' bar for singular values and discarded weight (relative to sigma_max / |psi|^2)


def _plan(H, torch, p):
    """device plan bound to resident arenas, as the other site-update tests build it (the arenas ride on the plan object)"""
    a, b = torch.from_numpy(p.a_data).cuda(), torch.from_numpy(p.b_data).cuda()
    plan = H.plan_problem(p, a, b)
    plan._arenas = (a, b)
    return plan


def _truncate_both(H, torch, plan, psi, chi_max, eps, side):
    """(existing path, static path) results for one input; separate output buffers, NaN-prefilled."""
    cap = H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY_RIGHT if side else H.HPSI_Q_ISO_CAPACITY)
    st = torch.cuda.current_stream()
    x = torch.from_numpy(psi).cuda()
    out = []
    for fn in (H.hpsi_truncate, H.hpsi_truncate_static):
        ot = torch.full((max(cap, 1),), float("nan"), dtype=torch.float64, device="cuda")
        chi, sigma, disc = fn(plan, x, chi_max, ot, st, eps, side)
        torch.cuda.synchronize()
        out.append((chi, sigma, disc, ot.cpu().numpy()))
    return out


def _assert_same(ref, got, dims):
    chi_r, sig_r, disc_r, ot_r = ref
    chi_g, sig_g, disc_g, ot_g = got
    assert np.array_equal(chi_g, chi_r)
    smax = max(float(sig_r.max()), 1e-300)
    np.testing.assert_allclose(sig_g, sig_r, rtol=0, atol=TOL * smax)
    assert abs(disc_g - disc_r) <= TOL
    n = int(np.sum(chi_r.astype(np.int64) * dims))
    np.testing.assert_allclose(ot_g[:n], ot_r[:n], rtol=0, atol=1e-11)       # unit-norm rows: absolute = relative
    assert np.isnan(ot_g[n:]).all()                                          # nothing written past the isometries


def test_truncate_static_matches_truncate_on_two_calls_in_a_row():
    import torch
    import paper_2407_07411_b200 as H
    small = workloads.make_problem("small", n_terms=8)
    toy = workloads.make_problem("toy")
    plan_s, plan_t = _plan(H, torch, small), _plan(H, torch, toy)
    psi1 = workloads.make_psi(small)
    psi1 /= np.linalg.norm(psi1)
    psi2 = workloads.make_psi(toy, 5)
    psi2 /= np.linalg.norm(psi2)
    psi3 = workloads.make_psi(small, 7)
    psi3 /= np.linalg.norm(psi3)
    # call 1: the D = 1024 config, left side, by count.  call 2 (right after, on the array call 1 left behind): a smaller
    # problem, right side, by discarded weight.  call 3: back to the large one with another psi.
    for plan, p, psi, chi_max, eps, side in ((plan_s, small, psi1, 256, -1.0, 0), (plan_t, toy, psi2, 10 ** 6, 1e-3, 1),
                                             (plan_s, small, psi3, 700, -1.0, 1)):
        ref, got = _truncate_both(H, torch, plan, psi, chi_max, eps, side)
        _assert_same(ref, got, p.d_right if side else p.d_left)
        chi_o, _, sig_o, disc_o = su.truncate(p, psi, chi_max, eps, "right" if side else "left")      # and the oracle
        assert np.array_equal(got[0], chi_o) and abs(got[2] - disc_o) <= TOL


def test_truncate_static_allocates_nothing_and_is_repeatable():
    """Free device memory (cudaMemGetInfo) is the same before and after a call; the same input twice gives the same bits."""
    import torch
    import paper_2407_07411_b200 as H
    p = workloads.make_problem("small", n_terms=8)
    plan = _plan(H, torch, p)
    psi = workloads.make_psi(p)
    psi /= np.linalg.norm(psi)
    x = torch.from_numpy(psi).cuda()
    st = torch.cuda.current_stream()
    ot = [torch.zeros(H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY), dtype=torch.float64, device="cuda") for _ in range(2)]
    H.hpsi_truncate_static(plan, x, 300, ot[0], st)           # first use on this device: module load, symbol address
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    res = [H.hpsi_truncate_static(plan, x, 300, ot[k], st) for k in range(2)]
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1]) and res[0][2] == res[1][2]
    assert torch.equal(ot[0], ot[1])


def test_truncate_static_rejects_what_does_not_fit():
    """One 1500 x 1500 psi block needs 1500 * 3008 * 8 = 36 MB of working matrix: more than the 32 MiB array."""
    import torch
    import paper_2407_07411_b200 as H
    d = 1500
    rng = np.random.default_rng(0)
    p = workloads.custom_problem([(0, 0)], [d], [(1, 0)], [d], (1, 0),
                                 [(1.0, {(0, 0): np.zeros((d, d))}, {(0, 0): np.zeros((d, d))})], pad_even=True)
    plan = _plan(H, torch, p)
    psi = rng.standard_normal(p.psi_len)
    psi /= np.linalg.norm(psi)
    x = torch.from_numpy(psi).cuda()
    ot = torch.zeros(H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY), dtype=torch.float64, device="cuda")
    with pytest.raises(H.HpsiError) as e:
        H.hpsi_truncate_static(plan, x, 100, ot, torch.cuda.current_stream())
    assert e.value.code == H.HPSI_EINVAL and "HPSI_TRUNCATE_STATIC_BYTES" in str(e.value) and str(H.HPSI_TRUNCATE_STATIC_BYTES) in str(e.value)
    chi, sigma, _ = H.hpsi_truncate(plan, x, 100, ot, torch.cuda.current_stream())         # the allocating path takes it
    assert int(chi.sum()) == 100
    sv = np.linalg.svd(psi.reshape(d, d), compute_uv=False)
    np.testing.assert_allclose(sigma[:100], sv[:100], rtol=0, atol=TOL * sv[0])
