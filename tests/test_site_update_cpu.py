"""Host logic of the site update without a GPU: the operator-update planner is verified by walking
its device tables with naive loops (hpsi_rotate_debug_interpret) against oracle/site_update.py; argument validation;
no-CPU-fallback behaviour."""
import numpy as np
import pytest

import workloads
import paper_2407_07411_b200 as H
from oracle import site_update as su


def out_blocks_as_arrays(r, out, chi):
    desc = H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_BLOCKS)
    res = []
    for e in desc:
        rr, cc = int(chi[e["row"]]), int(chi[e["col"]])
        if e["offset"] < 0:
            assert rr == 0 or cc == 0 and e["ld"] == 0
            res.append(np.zeros((rr, cc)))
            continue
        assert e["ld"] >= cc and e["ld"] % 4 == 0 and e["offset"] % 4 == 0
        res.append(np.lib.stride_tricks.as_strided(out[int(e["offset"]):], shape=(rr, cc), strides=(int(e["ld"]) * 8, 8)).copy())
    return res, desc


@pytest.mark.parametrize("name,keep,zero_every,pad_even", [("toy", 0.5, 0, True), ("toy", 0.7, 3, False),
                                                          ("small", 0.25, 5, True)])
def test_rotate_schedule_interpreted_matches_oracle(name, keep, zero_every, pad_even):
    p = workloads.make_problem(name, pad_even=pad_even, n_terms=40 if name == "small" else None)
    chi = workloads.proportional_chi(p.d_left, keep, zero_every)
    ot = workloads.make_isometries(p.d_left, chi, seed=21)
    r = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, None, p.a_len, H.HPSI_PLAN_HOST_ONLY)
    assert H.hpsi_rotate_query(r, H.HPSI_RQ_ISO_LENGTH) == int(np.sum(chi.astype(np.int64) * p.d_left))
    out = H.hpsi_rotate_debug_interpret(r, p.a_data, workloads.pack_isometries(ot))
    got, desc = out_blocks_as_arrays(r, out, chi)
    ref = su.rotate(p.d_left, chi, p.a_desc, p.a_data, ot)
    num = den = 0.0
    for g, x in zip(got, ref):
        assert g.shape == x.shape
        num += np.sum((g - x) ** 2); den += np.sum(x ** 2)
    assert np.sqrt(num / den) <= 1e-13
    # the descriptors keep term / row / col and do not overlap
    assert np.array_equal(desc["term"], p.a_desc["term"]) and np.array_equal(desc["row"], p.a_desc["row"])
    spans = sorted((int(e["offset"]), int(e["offset"]) + int(chi[e["row"]]) * int(e["ld"])) for e in desc if e["offset"] >= 0)
    assert all(a[1] <= b[0] for a, b in zip(spans, spans[1:]))
    assert spans[-1][1] <= H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_LENGTH)
    # flop / byte accounting against the oracle's independent count
    assert H.hpsi_rotate_query(r, H.HPSI_RQ_USEFUL_FLOPS) == su.rotate_flops(p.d_left, chi, p.a_desc)
    assert H.hpsi_rotate_query(r, H.HPSI_RQ_ALIGNED16) == (1 if pad_even else 0) or not pad_even


def test_rotate_everything_truncated_away_and_empty():
    p = workloads.make_problem("toy")
    chi = np.zeros_like(p.d_left)
    r = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, None, p.a_len, H.HPSI_PLAN_HOST_ONLY)
    assert H.hpsi_rotate_query(r, H.HPSI_RQ_USEFUL_FLOPS) == 0 and H.hpsi_rotate_query(r, H.HPSI_RQ_N_UNITS_1) == 0
    assert all(e["offset"] == -1 for e in H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_BLOCKS))
    r = H.hpsi_rotate_plan(p.d_left, p.d_left, p.a_desc[:0], None, 0, H.HPSI_PLAN_HOST_ONLY)
    assert H.hpsi_rotate_query(r, H.HPSI_RQ_N_UNITS_2) == 0


def test_rotate_validation_and_no_cpu_fallback():
    p = workloads.make_problem("toy")
    chi = workloads.proportional_chi(p.d_left, 0.5)
    bad = chi.copy(); bad[0] = p.d_left[0] + 1
    with pytest.raises(H.HpsiError) as e:
        H.hpsi_rotate_plan(p.d_left, bad, p.a_desc, None, p.a_len, H.HPSI_PLAN_HOST_ONLY)
    assert e.value.code == H.HPSI_EINVAL
    desc = p.a_desc.copy(); desc[3]["ld"] = 0
    with pytest.raises(H.HpsiError):
        H.hpsi_rotate_plan(p.d_left, chi, desc, None, p.a_len, H.HPSI_PLAN_HOST_ONLY)
    desc = np.concatenate([p.a_desc, p.a_desc[:1]])
    with pytest.raises(H.HpsiError):
        H.hpsi_rotate_plan(p.d_left, chi, desc, None, p.a_len, H.HPSI_PLAN_HOST_ONLY)
    desc = p.a_desc.copy(); desc[0]["offset"] = p.a_len
    with pytest.raises(H.HpsiError):
        H.hpsi_rotate_plan(p.d_left, chi, desc, None, p.a_len, H.HPSI_PLAN_HOST_ONLY)
    r = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, None, p.a_len, H.HPSI_PLAN_HOST_ONLY)
    with pytest.raises(H.HpsiError) as e:               # a host-only object refuses to compute: there is no CPU path
        H.hpsi_rotate_apply(r, 8, 8)
    assert e.value.code == H.HPSI_ESTATE
    plan = H.plan_problem(p, flags=H.HPSI_PLAN_HOST_ONLY)
    assert H.hpsi_query(plan, H.HPSI_Q_PSI_ROWS) == sum(r for (_, _, r, _, _) in p.psi_blocks())
    assert H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY) == sum(min(r, c) * r for (_, _, r, c, _) in p.psi_blocks())
    with pytest.raises(H.HpsiError) as e:
        H.hpsi_truncate(plan, 8, 4, 8)
    assert e.value.code == H.HPSI_ESTATE
