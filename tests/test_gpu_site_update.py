"""GPU parity of the site update against oracle/site_update.py, through the C ABI.

hpsi_rotate_apply: element by element (unique result; rel-L2 <= 1e-12 as for hpsi_apply).
hpsi_truncate: singular values and kept dimensions are unique and compared directly; singular vectors are unique only up
to sign (and rotation inside degenerate spaces), so the isometries are checked for validity (orthonormal rows, rows are
singular vectors with the right singular value) and through the projectors O O^T, which are unique when the cut falls in a gap."""
import numpy as np
import pytest

import workloads
from oracle import site_update as su

pytestmark = pytest.mark.gpu


def _gpu():
    import torch
    import paper_2407_07411_b200 as H
    assert torch.cuda.is_available()
    return torch, H


def run_rotate(p, chi, ot, misalign=False):
    torch, H = _gpu()
    if misalign:
        store = torch.empty(p.a_data.size + 1, dtype=torch.float64, device="cuda:0")
        a = store[1:]
        a.copy_(torch.from_numpy(p.a_data))
    else:
        a = torch.from_numpy(p.a_data).cuda()
    r = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, a, p.a_len)
    otd = torch.from_numpy(workloads.pack_isometries(ot)).cuda() if sum(o.size for o in ot) else torch.zeros(1, dtype=torch.float64, device="cuda:0")
    out = torch.full((H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_LENGTH),), float("nan"), dtype=torch.float64, device="cuda:0")
    H.hpsi_rotate_apply(r, otd, out, torch.cuda.current_stream())
    torch.cuda.synchronize()
    out2 = torch.full_like(out, float("nan"))
    H.hpsi_rotate_apply(r, otd, out2, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert torch.equal(torch.nan_to_num(out, nan=7.0), torch.nan_to_num(out2, nan=7.0))      # bitwise reproducible
    return r, out.cpu().numpy(), H


def compare_blocks(H, r, out, chi, ref):
    desc = H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_BLOCKS)
    num = den = 0.0
    for e, x in zip(desc, ref):
        rr, cc = int(chi[e["row"]]), int(chi[e["col"]])
        assert x.shape == (rr, cc)
        if e["offset"] < 0:
            assert rr == 0 or cc == 0
            continue
        g = np.lib.stride_tricks.as_strided(out[int(e["offset"]):], shape=(rr, cc), strides=(int(e["ld"]) * 8, 8))
        assert np.all(np.isfinite(g))
        num += np.sum((g - x) ** 2); den += np.sum(x ** 2)
    return float(np.sqrt(num / max(den, 1e-300)))


@pytest.mark.parametrize("name,keep,zero_every,pad_even,misalign", [
    ("toy", 0.5, 0, True, False), ("toy", 0.7, 3, False, False), ("toy", 1.0, 0, True, True),
    ("small", 0.25, 0, True, False), ("small", 0.4, 5, False, False), ("small", 0.25, 7, True, True)])
def test_rotate_matches_oracle(name, keep, zero_every, pad_even, misalign):
    p = workloads.make_problem(name, pad_even=pad_even)
    chi = workloads.proportional_chi(p.d_left, keep, zero_every)
    ot = workloads.make_isometries(p.d_left, chi, seed=31)
    r, out, H = run_rotate(p, chi, ot, misalign)
    assert H.hpsi_rotate_query(r, H.HPSI_RQ_ALIGNED16) == (1 if (pad_even and not misalign) else 0)
    err = compare_blocks(H, r, out, chi, su.rotate(p.d_left, chi, p.a_desc, p.a_data, ot))
    assert err <= 1e-12, err


def test_rotate_stress_shapes_sampled():
    """Heavy-tailed dims (1..1024): the oracle rotates a seeded sample of blocks one by one."""
    p = workloads.make_problem("stress", n_terms=24)
    chi = workloads.proportional_chi(p.d_left, 0.25, 9)
    ot = workloads.make_isometries(p.d_left, chi, seed=32)
    r, out, H = run_rotate(p, chi, ot)
    rng = np.random.default_rng(33)
    pick = np.sort(rng.choice(len(p.a_desc), size=min(150, len(p.a_desc)), replace=False))
    ref = su.rotate(p.d_left, chi, p.a_desc[pick], p.a_data, ot)
    desc = H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_BLOCKS)[pick]
    num = den = 0.0
    for e, x in zip(desc, ref):
        if e["offset"] < 0:
            continue
        g = np.lib.stride_tricks.as_strided(out[int(e["offset"]):], shape=x.shape, strides=(int(e["ld"]) * 8, 8))
        num += np.sum((g - x) ** 2); den += np.sum(x ** 2)
    assert np.sqrt(num / den) <= 1e-12


def test_rotate_right_operators_with_right_isometries():
    """A left-moving sweep: right isometries from hpsi_truncate(HPSI_SIDE_RIGHT) rotate the B blocks (the update is
    side-agnostic: sector dims, kept dims, descriptors, arena)."""
    torch, H = _gpu()
    p = workloads.make_problem("small", n_terms=40)
    psi = workloads.make_psi(p)
    a, b = torch.from_numpy(p.a_data).cuda(), torch.from_numpy(p.b_data).cuda()
    plan = H.plan_problem(p, a, b)
    ot = torch.zeros(H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY_RIGHT), dtype=torch.float64, device="cuda:0")
    chi, sigma, disc = H.hpsi_truncate(plan, torch.from_numpy(psi).cuda(), 300, ot, torch.cuda.current_stream(), -1.0, H.HPSI_SIDE_RIGHT)
    assert chi.shape[0] == p.q_right.shape[0] and int(chi.sum()) == 300
    r = H.hpsi_rotate_plan(p.d_right, chi, p.b_desc, b, p.b_len)
    out = torch.full((H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_LENGTH),), float("nan"), dtype=torch.float64, device="cuda:0")
    H.hpsi_rotate_apply(r, ot, out, torch.cuda.current_stream())
    torch.cuda.synchronize()
    oth, ots, o = ot.cpu().numpy(), [], 0
    for l in range(len(chi)):
        n = int(chi[l]) * int(p.d_right[l])
        ots.append(oth[o:o + n].reshape(int(chi[l]), int(p.d_right[l])))
        o += n
    err = compare_blocks(H, r, out.cpu().numpy(), chi, su.rotate(p.d_right, chi, p.b_desc, p.b_data, ots))
    assert err <= 1e-12, err


def test_rotate_apply_is_graph_capturable():
    """hpsi_rotate_apply only enqueues (no sync, no allocation): captured into a CUDA graph and replayed."""
    torch, H = _gpu()
    p = workloads.make_problem("small", n_terms=20)
    chi = workloads.proportional_chi(p.d_left, 0.3)
    ot = workloads.make_isometries(p.d_left, chi, seed=61)
    a = torch.from_numpy(p.a_data).cuda()
    r = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, a, p.a_len)
    otd = torch.from_numpy(workloads.pack_isometries(ot)).cuda()
    out = torch.zeros(H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_LENGTH), dtype=torch.float64, device="cuda:0")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        H.hpsi_rotate_apply(r, otd, out, s)                 # warm-up outside the capture
        s.synchronize()
        expect = out.clone()
        out.zero_()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            H.hpsi_rotate_apply(r, otd, out, s)
        assert float(out.abs().sum()) == 0.0                # capture enqueued nothing yet
        graph.replay()
        s.synchronize()
    assert torch.equal(out, expect)


def test_rotate_nothing_survives():
    torch, H = _gpu()
    p = workloads.make_problem("toy")
    a = torch.from_numpy(p.a_data).cuda()
    r = H.hpsi_rotate_plan(p.d_left, np.zeros_like(p.d_left), p.a_desc, a, p.a_len)
    out = torch.zeros(4, dtype=torch.float64, device="cuda:0")
    H.hpsi_rotate_apply(r, out, out, torch.cuda.current_stream())      # no-op, no launch
    torch.cuda.synchronize()


# ------------------------------------------------------------------------------------------ truncate
def run_truncate(p, psi, chi_max, eps=-1.0, side="left"):
    torch, H = _gpu()
    a = torch.from_numpy(p.a_data).cuda()
    b = torch.from_numpy(p.b_data).cuda()
    plan = H.plan_problem(p, a, b)
    x = torch.from_numpy(np.ascontiguousarray(psi)).cuda()
    cap = H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY_RIGHT if side == "right" else H.HPSI_Q_ISO_CAPACITY)
    ot = torch.full((max(cap, 1),), float("nan"), dtype=torch.float64, device="cuda:0")
    chi, sigma, disc = H.hpsi_truncate(plan, x, chi_max, ot, torch.cuda.current_stream(), eps,
                                       H.HPSI_SIDE_RIGHT if side == "right" else H.HPSI_SIDE_LEFT)
    assert np.array_equal(x.cpu().numpy(), psi)                          # psi is not modified
    return plan, chi, sigma, disc, ot.cpu().numpy(), H


def check_truncation(p, psi, chi_max, proj_tol=1e-9, eps=-1.0, side="left"):
    plan, chi, sigma, disc, ot, H = run_truncate(p, psi, chi_max, eps, side)
    chi_ref, ot_ref, sigma_ref, disc_ref = su.truncate(p, psi, chi_max, eps, side)
    assert np.array_equal(chi, chi_ref)
    smax = max(float(s[0]) for s in sigma_ref if s.size)
    row0 = 0
    blocks = p.psi_blocks()
    if side == "right":      # effective blocks psi_l^T, sector = the right one; isometries are laid out by ascending sector
        blocks = [(j, i, c, r, off) for (i, j, r, c, off) in blocks]
    iso_off, o = {}, 0
    for sec in sorted(b[0] for b in blocks):
        iso_off[sec] = o
        o += int(chi[sec]) * int((p.d_right if side == "right" else p.d_left)[sec])
    for (i, j, r, c, off) in blocks:
        iso0 = iso_off[i]
        s_gpu = sigma[row0:row0 + r]
        row0 += r
        k = min(r, c)
        np.testing.assert_allclose(s_gpu[:k], sigma_ref[i], rtol=0, atol=1e-12 * smax)
        assert np.all(s_gpu[k:] == 0.0)
        O = ot[iso0:iso0 + int(chi[i]) * r].reshape(int(chi[i]), r)
        blk = psi[off:off + r * c].reshape(c, r).T if side == "right" else psi[off:off + r * c].reshape(r, c)
        np.testing.assert_allclose(O @ O.T, np.eye(O.shape[0]), atol=1e-12)            # orthonormal rows
        # row a is a left singular vector with singular value sigma_a:  || O psi ||_row = sigma,  O psi psi^T = sigma^2 O
        np.testing.assert_allclose(np.linalg.norm(O @ blk, axis=1), sigma_ref[i][:O.shape[0]], atol=1e-12 * smax)
        np.testing.assert_allclose(O @ (blk @ blk.T), (sigma_ref[i][:O.shape[0]] ** 2)[:, None] * O, atol=1e-11 * smax ** 2)
        if proj_tol is not None:
            np.testing.assert_allclose(O.T @ O, ot_ref[i].T @ ot_ref[i], atol=proj_tol)     # same kept subspace
    assert abs(disc - disc_ref) <= 1e-12 * float(np.dot(psi, psi))
    return plan, H


@pytest.mark.parametrize("name,chi_max", [("toy", 12), ("toy", 1000), ("small", 256), ("small", 700)])
def test_truncate_matches_oracle(name, chi_max):
    p = workloads.make_problem(name, n_terms=8)
    check_truncation(p, workloads.make_psi(p), chi_max)


@pytest.mark.parametrize("eps,chi_max", [(1e-1, 10 ** 6), (1e-3, 10 ** 6), (1e-3, 300), (0.0, 10 ** 6)])
def test_truncate_by_discarded_weight_matches_oracle(eps, chi_max):
    p = workloads.make_problem("small", n_terms=8)
    check_truncation(p, workloads.make_psi(p), chi_max, eps=eps)


@pytest.mark.parametrize("name,chi_max,eps", [("toy", 12, -1.0), ("small", 256, -1.0), ("small", 10 ** 6, 1e-2)])
def test_truncate_right_side_matches_oracle(name, chi_max, eps):
    p = workloads.make_problem(name, n_terms=8)
    check_truncation(p, workloads.make_psi(p), chi_max, eps=eps, side="right")


def test_truncate_both_sides_on_one_plan():
    """The plan's SVD workspace is regrown when the other side needs more; results do not depend on call history."""
    torch, H = _gpu()
    p = workloads.make_problem("small", n_terms=8)
    psi = workloads.make_psi(p)
    plan = H.plan_problem(p, torch.from_numpy(p.a_data).cuda(), torch.from_numpy(p.b_data).cuda())
    x = torch.from_numpy(psi).cuda()
    otl = torch.zeros(H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY), dtype=torch.float64, device="cuda:0")
    otr = torch.zeros(H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY_RIGHT), dtype=torch.float64, device="cuda:0")
    st = torch.cuda.current_stream()
    c1, s1, d1 = H.hpsi_truncate(plan, x, 128, otl, st)
    first = otl.clone()
    cr, sr, dr = H.hpsi_truncate(plan, x, 128, otr, st, -1.0, H.HPSI_SIDE_RIGHT)
    c2, s2, d2 = H.hpsi_truncate(plan, x, 128, otl, st)
    assert np.array_equal(c1, c2) and np.array_equal(s1, s2) and d1 == d2 and torch.equal(first, otl)
    assert int(cr.sum()) == int(c1.sum()) == 128 and abs(dr - d1) <= 1e-13
    for (i, j, r, c, off) in p.psi_blocks():
        assert cr[j] == c1[i]


def test_truncate_cyp_sized_blocks_and_reproducible():
    """Full-size sector dims of the metric's config (blocks up to ~350 x 350: several chunk pairs, many rounds)."""
    p = workloads.make_problem("cyp", n_terms=2)
    psi = workloads.make_psi(p)
    plan, H = check_truncation(p, psi, 1024)
    assert 3 <= H.hpsi_query(plan, H.HPSI_Q_SVD_SWEEPS) <= 30
    _, chi1, sig1, d1, ot1, _ = run_truncate(p, psi, 1024)
    _, chi2, sig2, d2, ot2, _ = run_truncate(p, psi, 1024)
    n = int(np.sum(chi1.astype(np.int64) * p.d_left))
    assert np.array_equal(sig1, sig2) and np.array_equal(ot1[:n], ot2[:n]) and d1 == d2


def test_truncate_rank_deficient_wide_tall_and_single_row():
    # block 0: 5 x 2 (tall: three zero singular directions), block 1: 1 x 4 (single row), block 2: 3 x 6 of rank 1
    p = workloads.custom_problem([(0, 0), (1, 0), (2, 0), (9, 9)], [5, 1, 3, 2], [(2, 0), (1, 0), (0, 0)], [2, 4, 6], (2, 0), [])
    assert [(r, c) for (_, _, r, c, _) in p.psi_blocks()] == [(5, 2), (1, 4), (3, 6)]
    rng = np.random.default_rng(41)
    parts = [rng.standard_normal((5, 2)), rng.standard_normal((1, 4)), np.outer(rng.standard_normal(3), rng.standard_normal(6))]
    psi = np.concatenate([m.ravel() for m in parts])
    psi /= np.linalg.norm(psi)
    plan, chi, sigma, disc, ot, H = run_truncate(p, psi, 100)
    chi_ref, ot_ref, sigma_ref, disc_ref = su.truncate(p, psi, 100)
    assert chi.tolist() == chi_ref.tolist() == [2, 1, 1, 0]
    assert disc <= 1e-26
    check_truncation(p, psi, 100)
    check_truncation(p, psi, 2)


def test_site_update_pipeline_truncate_then_rotate():
    """The two steps chained on the device: isometries from hpsi_truncate feed hpsi_rotate_apply; the result must equal
    the oracle's rotation with the DEVICE isometries (sign conventions cancel in O^T A O only if the same O is used)."""
    torch, H = _gpu()
    p = workloads.make_problem("small", n_terms=40)
    psi = workloads.make_psi(p)
    a = torch.from_numpy(p.a_data).cuda()
    b = torch.from_numpy(p.b_data).cuda()
    plan = H.plan_problem(p, a, b)
    x = torch.from_numpy(psi).cuda()
    ot = torch.zeros(H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY), dtype=torch.float64, device="cuda:0")
    chi, sigma, disc = H.hpsi_truncate(plan, x, 256, ot, torch.cuda.current_stream())
    assert int(chi.sum()) == 256
    r = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, a, p.a_len)
    n_iso = H.hpsi_rotate_query(r, H.HPSI_RQ_ISO_LENGTH)
    out = torch.full((H.hpsi_rotate_query(r, H.HPSI_RQ_OUT_LENGTH),), float("nan"), dtype=torch.float64, device="cuda:0")
    H.hpsi_rotate_apply(r, ot, out, torch.cuda.current_stream())
    torch.cuda.synchronize()
    oth = ot.cpu().numpy()[:n_iso]
    ots, o = [], 0
    for l in range(len(chi)):
        n = int(chi[l]) * int(p.d_left[l])
        ots.append(oth[o:o + n].reshape(int(chi[l]), int(p.d_left[l])))
        o += n
    err = compare_blocks(H, r, out.cpu().numpy(), chi, su.rotate(p.d_left, chi, p.a_desc, p.a_data, ots))
    assert err <= 1e-12, err


def test_rotated_arena_feeds_the_next_plan():
    """The output arena + HPSI_RQ_OUT_BLOCKS of hpsi_rotate_apply are used, unchanged, as the A arena of a new hpsi_plan
    over the truncated left basis; applying it to phi must equal projecting the full apply:
    H' phi = (O^T (x) 1) H (O (x) 1) phi   (all three applies and the update on the device, isometries from hpsi_truncate)."""
    torch, H = _gpu()
    p = workloads.make_problem("small", n_terms=60)
    psi = workloads.make_psi(p)
    a, b = torch.from_numpy(p.a_data).cuda(), torch.from_numpy(p.b_data).cuda()
    plan = H.plan_problem(p, a, b)
    st = torch.cuda.current_stream()
    ot = torch.zeros(H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY), dtype=torch.float64, device="cuda:0")
    chi, _, _ = H.hpsi_truncate(plan, torch.from_numpy(psi).cuda(), 200, ot, st)
    rot = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, a, p.a_len)
    arena2 = torch.zeros(H.hpsi_rotate_query(rot, H.HPSI_RQ_OUT_LENGTH), dtype=torch.float64, device="cuda:0")
    H.hpsi_rotate_apply(rot, ot, arena2, st)
    desc2 = H.hpsi_rotate_query(rot, H.HPSI_RQ_OUT_BLOCKS)
    # new sector table: the left sectors that kept something, renumbered; right side unchanged
    keep = np.flatnonzero(chi > 0)
    renum = -np.ones(len(chi), np.int64); renum[keep] = np.arange(len(keep))
    d2 = desc2[desc2["offset"] >= 0].copy()
    d2["row"] = renum[d2["row"]]; d2["col"] = renum[d2["col"]]
    plan2 = H.hpsi_plan(p.q_left[keep], p.q_right, chi[keep], p.d_right, p.target, p.coef, d2, p.b_desc, arena2, b,
                        arena2.numel(), p.b_len)
    assert H.hpsi_query(plan2, H.HPSI_Q_ALIGNED16) == 1                       # the dictated layout takes the TMA path
    blocks2 = H.hpsi_query(plan2, H.HPSI_Q_PSI_BLOCKS)
    rng = np.random.default_rng(77)
    phi = rng.standard_normal(H.hpsi_query(plan2, H.HPSI_Q_PSI_LENGTH))
    oth, ots, o = ot.cpu().numpy(), {}, 0
    for l in range(len(chi)):
        n = int(chi[l]) * int(p.d_left[l])
        ots[l] = oth[o:o + n].reshape(int(chi[l]), int(p.d_left[l]))
        o += n
    full_blocks = {i: (r, c, off) for (i, j, r, c, off) in p.psi_blocks()}
    lifted = np.zeros(p.psi_len)
    for e in blocks2:
        l = int(keep[e["left"]])
        r, c, off = full_blocks[l]
        lifted[off:off + r * c] = (ots[l].T @ phi[int(e["offset"]):int(e["offset"]) + int(e["rows"]) * c].reshape(int(e["rows"]), c)).ravel()
    x = torch.from_numpy(lifted).cuda(); y = torch.empty_like(x)
    H.hpsi_apply(plan, x, y, st)
    x2 = torch.from_numpy(phi).cuda(); y2 = torch.empty_like(x2)
    H.hpsi_apply(plan2, x2, y2, st)
    torch.cuda.synchronize()
    hl, got = y.cpu().numpy(), y2.cpu().numpy()
    proj = np.zeros_like(phi)
    for e in blocks2:
        l = int(keep[e["left"]])
        r, c, off = full_blocks[l]
        proj[int(e["offset"]):int(e["offset"]) + int(e["rows"]) * c] = (ots[l] @ hl[off:off + r * c].reshape(r, c)).ravel()
    assert np.linalg.norm(got - proj) <= 1e-12 * np.linalg.norm(proj)
