"""Pins of oracle/site_update.py (truncation + renormalised-operator update) against what the mathematics fixes.
CPU only; nothing here touches the CUDA path.  Every check compares with something that is not the oracle: LAPACK's
symmetric eigensolver on psi psi^T, the Eckart-Young theorem, closed forms (tests/golden/site_update_closed_forms.txt),
a dense einsum embedding, algebraic invariants, and the (separately pinned) H_eff oracle."""
import os

import numpy as np
import pytest

import oracle
import workloads
from oracle import site_update as su

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "site_update_closed_forms.txt")


def golden():
    out = {}
    with open(GOLDEN) as f:
        for line in f:
            if line.startswith("#") or ":" not in line:
                continue
            key, val = line.split(":", 1)
            out[key.split()[0]] = val.split()
    return out


def one_block_problem(block):
    """A problem whose psi is the single block `block` (no operators needed for the truncation)."""
    r, c = block.shape
    return workloads.custom_problem([(0, 0)], [r], [(0, 0)], [c], (0, 0), [])


# ------------------------------------------------------------------------------------------- truncate
def test_truncate_closed_form_diagonal():
    g = golden()["diag321"]
    sig = np.array([float(g[1]), float(g[2]), float(g[3])])
    disc = float(g[5])
    psi = np.diag([3.0, 2.0, 1.0]) / np.sqrt(14.0)
    chi, ot, sigma, dw = su.truncate(one_block_problem(psi), psi.ravel(), 2)
    assert chi.tolist() == [2]
    np.testing.assert_allclose(sigma[0], sig, rtol=0, atol=1e-15)
    assert abs(dw - disc) <= 1e-15
    np.testing.assert_allclose(np.abs(ot[0]), np.eye(3)[:2], atol=1e-15)


def test_truncate_by_discarded_weight_closed_form():
    g = golden()["diag321_eps"]
    psi = np.diag([3.0, 2.0, 1.0]) / np.sqrt(14.0)
    for eps, kept in zip(g[0::2], g[1::2]):
        chi, ot, sigma, dw = su.truncate(one_block_problem(psi), psi.ravel(), 3, float(eps))
        assert chi.tolist() == [int(kept)] and dw <= float(eps)
    chi, _, _, _ = su.truncate(one_block_problem(psi), psi.ravel(), 1, 0.08)      # chi_max still caps it
    assert chi.tolist() == [1]


def test_truncate_by_discarded_weight_is_minimal(small):
    psi = workloads.make_psi(small)
    for eps in (1e-1, 1e-2, 1e-4):
        chi, ot, sigma, dw = su.truncate(small, psi, 10 ** 6, eps)
        allsig2 = np.sort(np.concatenate(sigma) ** 2)            # ascending
        n_drop = int(np.searchsorted(np.cumsum(allsig2), eps, side="right"))
        assert int(chi.sum()) == allsig2.size - n_drop and dw <= eps


def test_truncate_closed_form_rank_one():
    g = golden()["rank1"]
    u = np.array([float(x) for x in g[5:8]])
    v = np.array([3.0, 4.0]) / 5.0
    psi = np.outer(u, v)
    chi, ot, sigma, dw = su.truncate(one_block_problem(psi), psi.ravel(), 3)
    assert chi.tolist() == [int(g[3])]                       # the zero singular value is never kept (R3)
    assert abs(sigma[0][0] - float(g[1])) <= 1e-15 and abs(sigma[0][1]) <= 1e-15
    np.testing.assert_allclose(ot[0][0] * np.sign(ot[0][0, 0]), u, atol=1e-15)
    assert dw <= 1e-30


def test_truncate_global_selection_two_blocks():
    g = golden()["two_blocks"]
    # left sectors (0,0), (1,0) with dims 1, 2; their partners (target (1,0)) are right labels (1,0), (0,0): dims 1, 2
    p = workloads.custom_problem([(0, 0), (1, 0)], [1, 2], [(1, 0), (0, 0)], [1, 2], (1, 0), [])
    blocks = su.psi_block_list(p)
    assert [(r, c) for (_, _, r, c, _) in blocks] == [(1, 1), (2, 2)]
    psi = np.concatenate([[0.6], np.diag([0.7, np.sqrt(0.15)]).ravel()])
    assert abs(np.linalg.norm(psi) - 1.0) <= 1e-15
    chi, ot, sigma, dw = su.truncate(p, psi, 2)
    assert chi.tolist() == [int(g[1]), int(g[2])]
    assert abs(dw - float(g[4])) <= 1e-15


@pytest.mark.parametrize("name,chi_max", [("toy", 12), ("small", 256)])
def test_truncate_against_density_matrix_and_eckart_young(name, chi_max):
    p = workloads.make_problem(name)
    psi = workloads.make_psi(p)
    chi, ot, sigma, dw = su.truncate(p, psi, chi_max)
    assert int(chi.sum()) == chi_max
    allsig = np.concatenate(sigma)
    assert abs(np.sum(allsig ** 2) - 1.0) <= 1e-13                    # sum sigma^2 = ||psi||^2
    kept_sig = []
    proj_err2 = 0.0
    for (i, j, r, c, off) in p.psi_blocks():
        blk = psi[off:off + r * c].reshape(r, c)
        # singular values^2 = the min(r,c) largest eigenvalues of the reduced density matrix psi psi^T (LAPACK dsyevd)
        ev = np.sort(np.linalg.eigvalsh(blk @ blk.T))[::-1][:min(r, c)]
        np.testing.assert_allclose(sigma[i] ** 2, np.maximum(ev, 0), rtol=0, atol=1e-14)
        O = ot[i]
        np.testing.assert_allclose(O @ O.T, np.eye(O.shape[0]), atol=1e-13)      # isometry
        # rows of O^T are eigenvectors of psi psi^T with eigenvalue sigma^2
        np.testing.assert_allclose(O @ (blk @ blk.T), (sigma[i][:O.shape[0]] ** 2)[:, None] * O, atol=1e-13)
        kept_sig.extend(sigma[i][:O.shape[0]].tolist())
        proj_err2 += np.linalg.norm(blk - O.T @ (O @ blk)) ** 2
    # Eckart-Young: the error of the rank-chi projection is exactly the discarded weight ...
    assert abs(proj_err2 - dw) <= 1e-13
    # ... and the kept values are the chi_max largest of all
    assert min(kept_sig) >= np.sort(allsig)[::-1][chi_max - 1] - 1e-15
    assert abs(dw - np.sum(np.sort(allsig ** 2)[::-1][chi_max:])) <= 1e-13


def test_truncate_right_side(small):
    """Right basis: rows of O_r^T are eigenvectors of psi_l^T psi_l; the singular values - hence the kept total and the
    discarded weight - are those of the left-side truncation."""
    p = small
    psi = workloads.make_psi(p)
    chiL, _, sigL, dwL = su.truncate(p, psi, 200)
    chiR, otR, sigR, dwR = su.truncate(p, psi, 200, side="right")
    assert chiR.shape[0] == p.q_right.shape[0] and int(chiR.sum()) == int(chiL.sum()) == 200
    assert abs(dwL - dwR) <= 1e-14
    for (i, j, r, c, off) in p.psi_blocks():
        blk = psi[off:off + r * c].reshape(r, c)
        assert chiR[j] == chiL[i]
        np.testing.assert_allclose(sigR[j], sigL[i], atol=1e-14)
        O = otR[j]
        assert O.shape == (chiR[j], c)
        np.testing.assert_allclose(O @ O.T, np.eye(O.shape[0]), atol=1e-13)
        np.testing.assert_allclose(O @ (blk.T @ blk), (sigR[j][:O.shape[0]] ** 2)[:, None] * O, atol=1e-13)


def test_truncate_sector_without_block_and_wide_block():
    # left sector 1 has no partner; block of sector 0 is 2 x 5 (more columns than rows), of sector 2 is 4 x 2
    p = workloads.custom_problem([(0, 0), (7, 0), (1, 0)], [2, 3, 4], [(2, 0), (1, 0)], [5, 2], (2, 0), [])
    rng = np.random.default_rng(5)
    psi = rng.standard_normal(p.psi_len)
    chi, ot, sigma, dw = su.truncate(p, psi, 100)
    assert chi.tolist() == [2, 0, 2] and ot[1].shape == (0, 3)
    assert [s.shape[0] for s in sigma] == [2, 0, 2]
    assert dw <= 1e-28


# --------------------------------------------------------------------------------------------- rotate
def test_rotate_closed_form_2x2():
    val = float(golden()["rotate2x2"][0])
    c, s = np.cos(0.3), np.sin(0.3)
    blocks = np.array([(0, 0, 0, 2, 0)], dtype=workloads.OPBLOCK_DTYPE)
    out = su.rotate([2], [1], blocks, np.array([1.0, 2.0, 3.0, 4.0]), [np.array([[c, s]])])
    assert out[0].shape == (1, 1) and abs(out[0][0, 0] - val) <= 1e-15


@pytest.mark.parametrize("name", ["toy", "small"])
def test_rotate_against_dense_embedding(name):
    """O^T A O with block-diagonal dense O and the dense embedding of each term's A, by einsum over dense D x D arrays."""
    p = workloads.make_problem(name, n_terms=6 if name == "small" else None)
    chi = workloads.proportional_chi(p.d_left, 0.5, zero_every=4)
    ot = workloads.make_isometries(p.d_left, chi, seed=11)
    out = su.rotate(p.d_left, chi, p.a_desc, p.a_data, ot)
    oL = np.concatenate([[0], np.cumsum(p.d_left)]).astype(int)
    oC = np.concatenate([[0], np.cumsum(chi)]).astype(int)
    Od = np.zeros((oL[-1], oC[-1]))
    for l in range(len(chi)):
        Od[oL[l]:oL[l + 1], oC[l]:oC[l + 1]] = ot[l].T
    for t in range(p.n_terms):
        Ad = np.zeros((oL[-1], oL[-1]))
        idx = [i for i, e in enumerate(p.a_desc) if int(e["term"]) == t]
        for i in idx:
            e = p.a_desc[i]
            Ad[oL[e["row"]]:oL[e["row"] + 1], oL[e["col"]]:oL[e["col"] + 1]] = p.block("a", i)
        Ar = np.einsum("ay,yb->ab", np.einsum("xa,xy->ay", Od, Ad), Od)
        seen = np.zeros_like(Ar, bool)
        for i in idx:
            e = p.a_desc[i]
            ref = Ar[oC[e["row"]]:oC[e["row"] + 1], oC[e["col"]]:oC[e["col"] + 1]]
            seen[oC[e["row"]]:oC[e["row"] + 1], oC[e["col"]]:oC[e["col"] + 1]] = True
            assert out[i].shape == ref.shape
            np.testing.assert_allclose(out[i], ref, atol=1e-13)
        assert np.all(np.abs(Ar[~seen]) <= 1e-14)           # nothing leaks outside the term's block pattern


def test_rotate_identity_and_orthogonal_invariants(toy):
    p = toy
    d = p.d_left
    ident = [np.eye(int(x)) for x in d]
    out = su.rotate(d, d, p.a_desc, p.a_data, ident)
    for i in range(len(p.a_desc)):
        np.testing.assert_array_equal(out[i], p.block("a", i))          # O = 1: unchanged, exactly
    full = workloads.make_isometries(d, d, seed=3)                       # square orthogonal O: norms / traces kept
    out = su.rotate(d, d, p.a_desc, p.a_data, full)
    for i, e in enumerate(p.a_desc):
        A = p.block("a", i)
        assert abs(np.linalg.norm(out[i]) - np.linalg.norm(A)) <= 1e-13 * max(1.0, np.linalg.norm(A))
        if e["row"] == e["col"]:
            assert abs(np.trace(out[i]) - np.trace(A)) <= 1e-13 * max(1.0, abs(np.trace(A)))
    # composing two rotations = rotating by the product:  O2^T (O1^T A O1) O2 = (O1 O2)^T A (O1 O2)
    chi1 = workloads.proportional_chi(d, 0.8)
    chi2 = workloads.proportional_chi(chi1, 0.5)
    o1 = workloads.make_isometries(d, chi1, seed=4)
    o2 = workloads.make_isometries(chi1, chi2, seed=5)
    first = su.rotate(d, chi1, p.a_desc, p.a_data, o1)
    desc2 = p.a_desc.copy()
    chunks, off = [], 0
    for i, m in enumerate(first):
        desc2[i]["ld"], desc2[i]["offset"] = max(m.shape[1], 1), off
        chunks.append(m.ravel()); off += m.size
    second = su.rotate(chi1, chi2, desc2, np.concatenate(chunks + [np.zeros(1)]), o2)
    direct = su.rotate(d, chi2, p.a_desc, p.a_data, [b @ a for a, b in zip(o1, o2)])
    for x, y in zip(second, direct):
        np.testing.assert_allclose(x, y, atol=1e-13)


def test_rotated_operators_give_the_projected_hamiltonian(toy):
    """(O^T (x) 1) H (O (x) 1) phi  ==  sum_t c_t (O^T A_t O) phi B_t^T : ties ``rotate`` to the pinned ``oracle.apply``."""
    p = toy
    chi = workloads.proportional_chi(p.d_left, 0.6)
    ot = workloads.make_isometries(p.d_left, chi, seed=8)
    rot = su.rotate(p.d_left, chi, p.a_desc, p.a_data, ot)
    desc2 = p.a_desc.copy()
    chunks, off = [], 0
    for i, m in enumerate(rot):
        desc2[i]["ld"], desc2[i]["offset"] = m.shape[1], off
        chunks.append(m.ravel()); off += m.size
    import dataclasses
    p2 = dataclasses.replace(p, d_left=chi.astype(np.int32), a_desc=desc2, a_data=np.concatenate(chunks), a_len=off)
    rng = np.random.default_rng(9)
    phi = rng.standard_normal(p2.psi_len)
    # lift phi to the enlarged basis, apply H there, project back
    lifted = np.zeros(p.psi_len)
    small_blocks = {i: (r, c, off) for (i, j, r, c, off) in p2.psi_blocks()}
    for (i, j, r, c, off) in p.psi_blocks():
        rr, cc, o2 = small_blocks[i]
        lifted[off:off + r * c] = (ot[i].T @ phi[o2:o2 + rr * cc].reshape(rr, cc)).ravel()
    hl = oracle.apply(p, lifted)
    proj = np.zeros(p2.psi_len)
    for (i, j, r, c, off) in p.psi_blocks():
        rr, cc, o2 = small_blocks[i]
        proj[o2:o2 + rr * cc] = (ot[i] @ hl[off:off + r * c].reshape(r, c)).ravel()
    direct = oracle.apply(p2, phi)
    np.testing.assert_allclose(direct, proj, atol=1e-12 * np.linalg.norm(proj))


def test_rotate_flops_doubling_law(toy):
    d = toy.d_left.astype(np.int64)
    chi = workloads.proportional_chi(d, 0.5)
    f1 = su.rotate_flops(d, chi, toy.a_desc)
    f2 = su.rotate_flops(2 * d, 2 * chi, toy.a_desc)
    assert f2 == 8 * f1                                      # the O(D^3) law of PAPER.md:62


def test_rotate_flops_hand_count():
    """tests/golden/site_update_closed_forms.txt item 6: the counter against flops counted by hand, block by block - a
    wrong coefficient, a dropped GEMM or swapped row / column dims changes one of the five numbers."""
    line = [l for l in open(os.path.join(os.path.dirname(__file__), "golden", "site_update_closed_forms.txt")) if l.startswith("rotate_flops")][0]
    first, second = line.split(";")
    tok = first.split(":")[1].split()
    want = {tok[i]: int(tok[i + 1]) for i in range(0, len(tok), 2)}
    d = np.array([3, 2])
    desc = np.zeros(4, workloads.OPBLOCK_DTYPE)
    for i, (r, c) in enumerate([(0, 1), (1, 0), (0, 0), (1, 1)]):
        desc[i] = (i, r, c, d[c], 0)
        assert su.rotate_flops(d, np.array([2, 1]), desc[i:i + 1]) == want[f"{r}<-{c}"]
    assert su.rotate_flops(d, np.array([2, 1]), desc) == want["all"] == 24 + 32 + 60 + 12
    assert su.rotate_flops(d, np.array([2, 0]), desc) == int(second.split()[-1]) == 60
