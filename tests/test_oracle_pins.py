"""Pins of the CPU oracle against what the mathematics fixes (CPU only; no CUDA path involved).

Every test compares oracle/ with something that is *not* the oracle: a dense NumPy Kronecker expansion,
LAPACK's eigensolver, BLAS products, textbook closed forms (tests/golden/), or algebraic invariants.
"""
import os

import numpy as np
import pytest

import oracle
import workloads
from workloads.hubbard import hubbard_two_block_problem, monolithic_hubbard

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hubbard_closed_forms.txt")


# ------------------------------------------------------------------------------------------ helpers
def dense_embed(p):
    """Dense D_L x D_L / D_R x D_R embedding of every term's operators (NumPy only)."""
    oL = np.concatenate([[0], np.cumsum(p.d_left)]).astype(int)
    oR = np.concatenate([[0], np.cumsum(p.d_right)]).astype(int)
    DL, DR = int(oL[-1]), int(oR[-1])
    As = [np.zeros((DL, DL)) for _ in range(p.n_terms)]
    Bs = [np.zeros((DR, DR)) for _ in range(p.n_terms)]
    for i, e in enumerate(p.a_desc):
        r, c = int(e["row"]), int(e["col"])
        As[int(e["term"])][oL[r]:oL[r + 1], oL[c]:oL[c + 1]] += p.block("a", i)
    for i, e in enumerate(p.b_desc):
        r, c = int(e["row"]), int(e["col"])
        Bs[int(e["term"])][oR[r]:oR[r + 1], oR[c]:oR[c + 1]] += p.block("b", i)
    return As, Bs, oL, oR


def target_mask(p, oL, oR):
    """Boolean D_L x D_R mask of the target sector, straight from the label sum (no partner table)."""
    mask = np.zeros((int(oL[-1]), int(oR[-1])), bool)
    for i in range(p.q_left.shape[0]):
        for j in range(p.q_right.shape[0]):
            if np.array_equal(p.q_left[i] + p.q_right[j], p.target):
                mask[oL[i]:oL[i + 1], oR[j]:oR[j + 1]] = True
    return mask


def embed_psi(p, psi, oL, oR):
    M = np.zeros((int(oL[-1]), int(oR[-1])))
    for (i, j, r, c, off) in p.psi_blocks():
        M[oL[i]:oL[i + 1], oR[j]:oR[j + 1]] = psi[off:off + r * c].reshape(r, c)
    return M


def extract_psi(p, M, oL, oR):
    out = np.zeros(p.psi_len)
    for (i, j, r, c, off) in p.psi_blocks():
        out[off:off + r * c] = M[oL[i]:oL[i + 1], oR[j]:oR[j + 1]].ravel()
    return out


def kron_apply(p, psi, project=True):
    """H_full = sum_t c_t kron(A_t, B_t) acting on row-major vec(psi): vec(A psi B^T) = (A (x) B) vec(psi)."""
    As, Bs, oL, oR = dense_embed(p)
    H = sum(c * np.kron(A, B) for c, A, B in zip(p.coef, As, Bs))
    full = (H @ embed_psi(p, psi, oL, oR).ravel()).reshape(int(oL[-1]), int(oR[-1]))
    mask = target_mask(p, oL, oR)
    leak = np.abs(full[~mask]).max() if (~mask).any() else 0.0
    return extract_psi(p, full, oL, oR), leak


def random_custom(seed, n_left=5, n_right=6, n_terms=7, grid=True):
    """Irregular instance: random labels, partner-less sectors, random block patterns (not shift-structured)."""
    rng = np.random.default_rng(seed)
    if grid:
        qL = np.array([(a, 2 * b) for a in range(3) for b in range(2)], np.int32)[:n_left]
    else:
        qL = rng.permutation(np.array([(a, b) for a in range(-3, 4) for b in range(-2, 3)], np.int32))[:n_left]
    target = np.array([5, 1], np.int32)
    qR = [tuple(target - q) for q in qL[rng.permutation(n_left)[: n_left - 1]]]     # one left sector has no partner
    qR += [(99, 99 + i) for i in range(n_right - len(qR))]                          # right sectors with no partner
    qR = np.array(qR, np.int32)[rng.permutation(n_right)]
    dL = rng.integers(1, 5, n_left)
    dR = rng.integers(1, 5, n_right)
    terms = []
    for _ in range(n_terms):
        ab, bb = {}, {}
        for _k in range(rng.integers(1, 6)):
            r, c = int(rng.integers(n_left)), int(rng.integers(n_left))
            ab[(r, c)] = rng.standard_normal((dL[r], dL[c]))
        for _k in range(rng.integers(1, 7)):
            r, c = int(rng.integers(n_right)), int(rng.integers(n_right))
            bb[(r, c)] = rng.standard_normal((dR[r], dR[c]))
        terms.append((float(rng.standard_normal()), ab, bb))
    return workloads.custom_problem(qL, dL, qR, dR, target, terms, pad_even=bool(seed % 2))


# --------------------------------------------------------------------------------------- psi table
def test_psi_table_matches_construction(toy, small):
    for p in (toy, small, workloads.make_problem("stress", fill=False)):
        partner, offset, n = oracle.psi_table(p)
        assert n == p.psi_len
        assert np.array_equal(partner, p.partner)
        blocks = p.psi_blocks()
        assert [int(offset[i]) for (i, *_r) in blocks] == [b[4] for b in blocks]


def test_psi_table_partnerless_sectors():
    p = random_custom(3)
    partner, offset, n = oracle.psi_table(p)
    assert (partner < 0).sum() == 1 and n == p.psi_len
    for i, j in enumerate(partner):
        if j >= 0:
            assert np.array_equal(p.q_left[i] + p.q_right[j], p.target)
        else:
            assert not any(np.array_equal(p.q_left[i] + q, p.target) for q in p.q_right)


# ----------------------------------------------------------------------- brute-force Kronecker pins
def test_kronecker_toy(toy):
    """BASELINE.json north_star: 'brute-force Kronecker expansion on tiny inputs' (configs[0])."""
    for k in range(3):
        psi = workloads.make_psi(toy, k)
        ref, leak = kron_apply(toy, psi)
        got = oracle.apply(toy, psi)
        assert leak == 0.0                      # shifts conserve the total label: nothing leaves the target sector
        assert np.linalg.norm(got - ref) <= 1e-14 * np.linalg.norm(ref)


@pytest.mark.parametrize("seed", range(8))
def test_kronecker_irregular(seed):
    """Non-shift-structured blocks, partner-less sectors, non-grid labels, padded and dense ld:
    out = P (sum c A(x)B) P psi with P the target-sector projector."""
    p = random_custom(seed, grid=(seed < 4))
    rng = np.random.default_rng(100 + seed)
    psi = rng.standard_normal(p.psi_len)
    ref, _ = kron_apply(p, psi)
    got = oracle.apply(p, psi)
    assert np.linalg.norm(got - ref) <= 1e-14 * max(np.linalg.norm(ref), 1.0)


def test_transposed_B_would_fail():
    """The pin is sensitive to the index convention of B: with non-symmetric square blocks, using B instead of
    B^T (a plausible mistake) changes the answer by O(1)."""
    rng = np.random.default_rng(5)
    A, B, psi = rng.standard_normal((3, 3)), rng.standard_normal((4, 4)), rng.standard_normal((3, 4))
    p = workloads.custom_problem([(0, 0)], [3], [(1, 0)], [4], (1, 0), [(1.0, {(0, 0): A}, {(0, 0): B})])
    got = oracle.apply(p, psi.ravel()).reshape(3, 4)
    assert np.allclose(got, A @ psi @ B.T, rtol=0, atol=1e-14)
    assert not np.allclose(got, A @ psi @ B, atol=1e-3)
    assert not np.allclose(got, A.T @ psi @ B.T, atol=1e-3)


# ------------------------------------------------------------------------------------- invariants
def test_hermiticity(toy, small):
    """<x,Hy> = <Hx,y> when every term is paired with its adjoint (PAPER.md:62 'hermitian'; north_star)."""
    for p in (toy, small):
        rng = np.random.default_rng(7)
        x, y = rng.standard_normal(p.psi_len), rng.standard_normal(p.psi_len)
        Hy, Hx = oracle.apply(p, y), oracle.apply(p, x)
        assert abs(x @ Hy - Hx @ y) <= 1e-13 * np.linalg.norm(x) * np.linalg.norm(Hy)


def test_dense_h_symmetric_and_diagonal(toy):
    H = oracle.dense_hamiltonian(toy)
    assert np.abs(H - H.T).max() <= 1e-14 * np.abs(H).max()
    assert np.abs(np.diag(H) - oracle.diagonal(toy)).max() <= 1e-14 * np.abs(H).max()


def test_single_block_is_blas():
    """n_L = n_R = 1, one term, c = 1  ->  A @ psi @ B.T from BLAS."""
    rng = np.random.default_rng(11)
    for (m, n) in ((1, 1), (7, 5), (33, 65), (128, 17)):
        A, B, psi = rng.standard_normal((m, m)), rng.standard_normal((n, n)), rng.standard_normal((m, n))
        for pad in (False, True):
            p = workloads.custom_problem([(2, 0)], [m], [(3, 1)], [n], (5, 1),
                                         [(1.0, {(0, 0): A}, {(0, 0): B})], pad_even=pad)
            got = oracle.apply(p, psi.ravel()).reshape(m, n)
            ref = A @ psi @ B.T
            assert np.linalg.norm(got - ref) <= 1e-14 * np.linalg.norm(ref)


def test_rectangular_blocks_shift():
    """Two sectors per side with different dims: a shift term moves block (0,1') to block (1,0')."""
    rng = np.random.default_rng(12)
    dL, dR = [3, 5], [4, 2]
    qL, qR, target = [(0, 0), (1, 0)], [(1, 0), (0, 0)], (1, 0)     # partner(0)=0', partner(1)=1'
    A10 = rng.standard_normal((5, 3))      # left 0 -> 1
    B10 = rng.standard_normal((2, 4))      # right 0' -> 1'
    p = workloads.custom_problem(qL, dL, qR, dR, target, [(0.5, {(1, 0): A10}, {(1, 0): B10})])
    psi0, psi1 = rng.standard_normal((3, 4)), rng.standard_normal((5, 2))
    out = oracle.apply(p, np.concatenate([psi0.ravel(), psi1.ravel()]))
    assert np.allclose(out[:12], 0.0)
    assert np.allclose(out[12:].reshape(5, 2), 0.5 * A10 @ psi0 @ B10.T, rtol=0, atol=1e-14)


def test_closed_forms(toy):
    rng = np.random.default_rng(13)
    # (i) identities on every sector, all terms delta=0:  H psi = (sum c_t) psi exactly
    nL = toy.q_left.shape[0]
    cs = [0.5, -1.0, 2.0]     # partial sums 0.5, -0.5 are exact scalings, so only the last add rounds
    terms = [(c, {(i, i): np.eye(toy.d_left[i]) for i in range(nL)},
              {(j, j): np.eye(toy.d_right[j]) for j in range(nL)}) for c in cs]
    pid = workloads.custom_problem(toy.q_left, toy.d_left, toy.q_right, toy.d_right, toy.target, terms)
    psi = rng.standard_normal(pid.psi_len)
    assert np.array_equal(oracle.apply(pid, psi), sum(cs) * psi)
    # (ii) rank-1 blocks: c u (v^T psi z) w^T
    u, v, w, z = (rng.standard_normal(k) for k in (4, 4, 3, 3))
    p1 = workloads.custom_problem([(0, 0)], [4], [(0, 0)], [3], (0, 0),
                                  [(-0.7, {(0, 0): np.outer(u, v)}, {(0, 0): np.outer(w, z)})])
    ps = rng.standard_normal((4, 3))
    assert np.allclose(oracle.apply(p1, ps.ravel()).reshape(4, 3), -0.7 * (v @ ps @ z) * np.outer(u, w), atol=1e-14)
    # (iii) linearity
    x, y = rng.standard_normal(toy.psi_len), rng.standard_normal(toy.psi_len)
    lhs = oracle.apply(toy, 0.3 * x - 1.7 * y)
    rhs = 0.3 * oracle.apply(toy, x) - 1.7 * oracle.apply(toy, y)
    assert np.linalg.norm(lhs - rhs) <= 1e-14 * np.linalg.norm(rhs)
    # (v) scaling all c_t by a power of two scales the output exactly
    import copy
    p2 = copy.copy(toy)
    p2.coef = toy.coef * 4.0
    assert np.array_equal(oracle.apply(p2, x), 4.0 * oracle.apply(toy, x))


def test_term_permutation_and_padding(toy):
    """(iv) term order only changes rounding; padded vs dense leading dimension changes nothing."""
    psi = workloads.make_psi(toy)
    base = oracle.apply(toy, psi)
    dense = workloads.make_problem("toy", pad_even=False)
    assert np.array_equal(oracle.apply(dense, psi), base)
    # reverse the descriptor arrays (blocks 'may arrive in any order'); per-term scan order is preserved per term
    import copy
    rev = copy.copy(toy)
    rev.a_desc = toy.a_desc[::-1].copy()
    rev.b_desc = toy.b_desc[::-1].copy()
    assert np.linalg.norm(oracle.apply(rev, psi) - base) <= 1e-14 * np.linalg.norm(base)


def test_samples_match_full_apply(toy, small):
    for p, ns in ((toy, 40), (small, 25)):
        psi = workloads.make_psi(p)
        full = oracle.apply(p, psi)
        rng = np.random.default_rng(21)
        blocks = p.psi_blocks()
        pick = rng.integers(0, len(blocks), ns)
        sl = np.array([blocks[b][0] for b in pick], np.int32)
        sx = np.array([rng.integers(blocks[b][2]) for b in pick], np.int32)
        sy = np.array([rng.integers(blocks[b][3]) for b in pick], np.int32)
        vals = oracle.apply_samples(p, psi, sl, sx, sy)
        ref = np.array([full[blocks[b][4] + x * blocks[b][3] + y] for b, x, y in zip(pick, sx, sy)])
        assert np.abs(vals - ref).max() <= 1e-13 * np.abs(full).max()


def test_useful_flops_cubic_law():
    """Reading A18 + PAPER.md:62/82 (D^3): doubling every sector dim multiplies useful flops by exactly 8."""
    p1 = workloads.make_problem("toy", fill=False)
    f1, n1 = oracle.useful_flops(p1)
    p2 = workloads.make_problem("toy", fill=False)
    p2.d_left = p1.d_left * 2
    p2.d_right = p1.d_right * 2
    f2, n2 = oracle.useful_flops(p2)
    assert n1 == n2 and f2 == 8 * f1
    # hand count on one task: m=2,k=3,n'=4,n=5 -> min(2*2*4*(3+5), 2*3*5*(4+2)) = min(128,180)
    p = workloads.custom_problem([(0, 0), (1, 0)], [3, 2], [(1, 0), (0, 0)], [4, 5], (1, 0),
                                 [(1.0, {(1, 0): np.ones((2, 3))}, {(1, 0): np.ones((5, 4))})])
    assert oracle.useful_flops(p) == (128, 1)


# -------------------------------------------------------------------------- physics closed forms
def _golden():
    vals = {}
    for line in open(GOLDEN):
        if line.startswith("#") or ":" not in line:
            continue
        key, rest = line.split(":")
        vals[key.split()[0]] = [float(x) for x in rest.split()]
    return vals


def test_hubbard_two_block_equals_monolithic():
    """The generator's two-block form sum c A(x)B (parity folded into A, reading A5) is the Jordan-Wigner chain."""
    for (nl, nr, U) in ((1, 1, 3.7), (2, 2, 0.0), (1, 2, 1.3)):
        p = hubbard_two_block_problem(nl, nr, 1.0, U, nl + nr, 0)
        As, Bs, oL, oR = dense_embed(p)
        H = sum(c * np.kron(A, B) for c, A, B in zip(p.coef, As, Bs))
        # undo the sector sorting of each side to compare with the monolithic JW matrix
        from workloads.hubbard import _sectorize
        _, _, ordL = _sectorize(nl)
        _, _, ordR = _sectorize(nr)
        perm = (ordL[:, None] * 4 ** nr + ordR[None, :]).ravel()
        Href = monolithic_hubbard(nl + nr, 1.0, U)[np.ix_(perm, perm)]
        assert np.allclose(H, Href, atol=1e-14)


def test_hubbard_dimer_spectrum():
    g = _golden()["dimer"]
    p = hubbard_two_block_problem(1, 1, 1.0, 3.7, 2, 0)
    assert p.psi_len == 4
    ev = np.linalg.eigvalsh(oracle.dense_hamiltonian(p))
    assert np.allclose(ev, sorted(g), rtol=0, atol=1e-13)
    r = np.sqrt(3.7 ** 2 + 16.0)
    assert np.allclose(sorted(g), sorted([(3.7 - r) / 2, 0.0, 3.7, (3.7 + r) / 2]), atol=1e-15)   # fixture == formula
    theta, x, _, rn = oracle.davidson(p, np.ones(4), tol=1e-12)
    assert abs(theta - g[0]) <= 1e-12 and rn <= 1e-12


def test_hubbard_chain4():
    e0, dim = _golden()["chain4"]
    p = hubbard_two_block_problem(2, 2, 1.0, 0.0, 4, 0)
    assert p.psi_len == int(dim)
    assert sorted(p.d_left.tolist()) == sorted([1, 2, 2, 1, 4, 1, 2, 2, 1])
    H = oracle.dense_hamiltonian(p)
    assert abs(np.linalg.eigvalsh(H)[0] - e0) <= 1e-13
    rng = np.random.default_rng(3)
    theta, x, nmv, rn = oracle.davidson(p, rng.standard_normal(p.psi_len), tol=1e-10)
    assert abs(theta - e0) <= 1e-10 and rn <= 1e-10
    assert np.linalg.norm(oracle.apply(p, x) - theta * x) <= 1e-9


# ----------------------------------------------------------------------------------------- Davidson
@pytest.mark.parametrize("precondition", [True, False])
def test_davidson_vs_dense_eigensolver(toy, precondition):
    """north_star: 'agreement of Davidson's lowest eigenvalue with a dense eigensolver on tiny instances'."""
    H = oracle.dense_hamiltonian(toy)
    e0 = np.linalg.eigvalsh(H)[0]
    theta, x, nmv, rn = oracle.davidson(toy, workloads.make_psi(toy), tol=1e-9, max_iter=400,
                                        precondition=precondition)
    assert abs(theta - e0) <= 1e-10
    assert rn <= 1e-9 and np.linalg.norm(H @ x - theta * x) <= 1e-8
    assert abs(np.linalg.norm(x) - 1.0) <= 1e-12


# ----------------------------------------------------------------------------- block (multi-root) Davidson
@pytest.mark.parametrize("k", [2, 3])
@pytest.mark.parametrize("precondition", [True, False])
def test_davidson_block_vs_dense_eigensolver(toy, k, precondition):
    """Reading A21b: the k lowest Ritz values against LAPACK's eigenvalues of the dense toy Hamiltonian, the Ritz vectors
    orthonormal and each one an eigenvector to the tolerance."""
    H = oracle.dense_hamiltonian(toy)
    ev = np.linalg.eigvalsh(H)
    V0 = np.random.default_rng(k).standard_normal((toy.psi_len, k))
    theta, X, nmv, rn = oracle.davidson_block(toy, V0, tol=1e-9, max_iter=800, precondition=precondition)
    assert np.max(np.abs(theta - ev[:k])) <= 1e-10 and rn.max() <= 1e-9
    assert np.max(np.abs(X.T @ X - np.eye(k))) <= 1e-12
    assert np.max(np.linalg.norm(H @ X - X * theta[None, :], axis=0)) <= 1e-8
    assert k <= nmv <= 800


def test_davidson_diagonal_operator_needs_the_residual_fallback():
    """Reading A21c, pinned against LAPACK: for a diagonal H the preconditioned correction r/(diag - theta) is the Ritz
    vector itself, so it vanishes under Gram-Schmidt with |r| > tol; the residual is taken instead and the solver still
    reaches the lowest eigenvalue (a block-diagonal H with one diagonal and one dense block does the same in one block).
    An exact start vector (r = 0) is a converged run after one mat-vec."""
    rng = np.random.default_rng(12)
    dvals = np.array([-2.0, 1.0, 3.0, 0.5])
    diag = workloads.custom_problem([(0, 0)], [4], [(1, 0)], [1], (1, 0), [(1.0, {(0, 0): np.diag(dvals)}, {(0, 0): np.ones((1, 1))})])
    S = rng.standard_normal((3, 3))
    mixed = workloads.custom_problem([(0, 0), (1, 0)], [4, 3], [(1, 0), (0, 0)], [1, 1], (1, 0),
                                     [(1.0, {(0, 0): np.diag(dvals), (1, 1): S + S.T}, {(0, 0): np.ones((1, 1)), (1, 1): np.ones((1, 1))})])
    for p in (diag, mixed):
        ev = np.linalg.eigvalsh(oracle.dense_hamiltonian(p))
        v0 = rng.standard_normal(p.psi_len)
        for pre in (True, False):
            th, x, nmv, rn = oracle.davidson(p, v0, tol=1e-10, max_iter=100, precondition=pre)
            assert rn <= 1e-10 and abs(th - ev[0]) <= 1e-12, (pre, th, ev[0], nmv)
            thb, X, nb, rb = oracle.davidson_block(p, rng.standard_normal((p.psi_len, 2)), tol=1e-10, max_iter=200, precondition=pre)
            assert rb.max() <= 1e-10 and np.max(np.abs(thb - ev[:2])) <= 1e-12, (pre, thb, ev[:2])
    e0 = np.array([1.0, 0.0, 0.0, 0.0])
    th, x, nmv, rn = oracle.davidson(diag, 3.0 * e0, tol=1e-10)
    assert nmv == 1 and rn == 0.0 and th == -2.0 and np.array_equal(x, e0)


def test_davidson_block_single_root_is_davidson(toy):
    """k = 1 is the single-root method of reading A21, mat-vec for mat-vec."""
    v0 = workloads.make_psi(toy)
    for it in (5, 11, 30):
        th1, x1, n1, r1 = oracle.davidson(toy, v0, tol=1e-12, max_iter=it, precondition=False)
        thb, xb, nb, rb = oracle.davidson_block(toy, v0[:, None], tol=1e-12, max_iter=it, precondition=False)
        # (the single-root routine spends one more mat-vec on a correction vector it then never uses: max_iter bounds its
        # iterations, while the block routine - like hpsi_davidson - bounds the mat-vecs)
        assert nb == it and n1 == it + 1
        assert abs(thb[0] - th1) <= 1e-12 * abs(th1) and abs(rb[0] - r1) <= 1e-6 * r1


def test_davidson_block_hubbard_levels():
    """tests/golden/hubbard_closed_forms.txt: the two lowest levels of the dimer sector, (U - sqrt(U^2 + 16 t^2)) / 2 and
    0, and the lowest two of the four-site chain against the dense spectrum."""
    g = sorted(_golden()["dimer"])
    dimer = hubbard_two_block_problem(1, 1, 1.0, 3.7, 2, 0)
    theta, X, _, rn = oracle.davidson_block(dimer, np.eye(4)[:, :2] + 0.1, tol=1e-12, m_max=4)
    assert np.max(np.abs(theta - g[:2])) <= 1e-12 and rn.max() <= 1e-12
    chain = hubbard_two_block_problem(2, 2, 1.0, 0.0, 4, 0)
    ev = np.linalg.eigvalsh(oracle.dense_hamiltonian(chain))
    V0 = np.random.default_rng(4).standard_normal((chain.psi_len, 2))
    theta, X, _, rn = oracle.davidson_block(chain, V0, tol=1e-10, precondition=False, max_iter=400)
    assert abs(theta[0] - _golden()["chain4"][0]) <= 1e-10 and abs(theta[1] - ev[1]) <= 1e-9
