"""ORACLE - test infrastructure, not product code.

The two steps that follow the eigen-solve in a DMRG tensor update: the paper names "tensor
contraction and matrix factorization" as the two core operations of tensor-network algorithms and the
sweep as a "sequence of updates of all tensors", but writes out neither step; the readings are R1-R5 of
DESIGN.md section 9.

* ``truncate``  - the matrix factorisation: SVD of every psi block (LAPACK through numpy, a library primitive used as
                  one step), global selection of the ``chi_max`` largest singular values, left isometries O_l.
* ``rotate``    - the renormalised-operator update  A'_t[l,l'] = O_l^T A_t[l,l'] O_l'  by its plain definition.

Only tests/, ``__graft_entry__.smoke()`` and bench.py's cpu_baseline leg may import this module.  It imports nothing
from ``paper_2407_07411_b200`` and shares no code with it.

Pins: tests/test_oracle_site_pins.py (eigenvalues of psi psi^T, Eckart-Young discarded weight, rank-1 and diagonal
closed forms from tests/golden/site_update_closed_forms.txt, dense embedding O^T A O with einsum, identity and
orthogonal-invariance special cases,  (O^T (x) 1) H (O (x) 1)  against the pinned ``oracle.apply``, and ``rotate_flops``
against flops counted by hand block by block, golden item 6, plus the x8 doubling law).
"""
from __future__ import annotations

from typing import List, Tuple

import numpy as np

# singular values at or below SIGMA_FLOOR * (largest singular value of psi) are never kept (reading R3): their
# singular vectors are rounding noise and not unique
SIGMA_FLOOR = 1e-13


def psi_block_list(p) -> List[Tuple[int, int, int, int, int]]:
    """(left i, right j, rows, cols, offset) of every psi block, ascending i - derived from the label sum alone."""
    right = {(int(a), int(b)): j for j, (a, b) in enumerate(np.asarray(p.q_right))}
    out, off = [], 0
    for i, (a, b) in enumerate(np.asarray(p.q_left)):
        j = right.get((int(p.target[0]) - int(a), int(p.target[1]) - int(b)))
        if j is None:
            continue
        r, c = int(p.d_left[i]), int(p.d_right[j])
        out.append((i, j, r, c, off))
        off += r * c
    return out


def truncate(p, psi: np.ndarray, chi_max: int, eps_discard: float = -1.0, side: str = "left"):
    """Reading R1-R3: psi is block diagonal over (left sector, partner), so its SVD is the SVD of every block
    psi_l = U_l S_l V_l^T.  Keep the ``chi_max`` largest singular values over all blocks (ties: lower left sector, then
    lower index first; values <= SIGMA_FLOOR * sigma_max never kept).  O_l = the kept columns of U_l.
    Reading R6 (the paper quotes results by their "truncation error"): with ``eps_discard`` >= 0 only as
    many of those values are kept as it takes for the discarded weight to be <= eps_discard (never more than chi_max).
    ``side="right"``: the new RIGHT basis instead - every block is transposed first, sectors / dims are the right ones
    (O_r = kept right singular vectors of the block whose right sector is r); ties still go by psi-table order.

    Returns (chi[n_left], ot, sigma, discarded_weight):
      chi    int32 kept states per left sector (0 for a sector without a psi block);
      ot     list over left sectors of O_l^T as a (chi_l, d_l) array, rows in descending singular value;
      sigma  list over left sectors of ALL min(d_l, d_r) singular values, descending (empty without a block);
      discarded_weight = sum of sigma^2 over everything not kept."""
    psi = np.asarray(psi, np.float64)
    right = side == "right"
    nL = int(np.asarray(p.q_right if right else p.q_left).shape[0])
    dims = p.d_right if right else p.d_left
    U, S, pos = {}, {}, {}
    for n_blk, (i, j, r, c, off) in enumerate(psi_block_list(p)):
        blk = psi[off:off + r * c].reshape(r, c)
        u, s, _ = np.linalg.svd(blk.T if right else blk, full_matrices=False)
        sec = j if right else i
        U[sec], S[sec], pos[sec] = u, s, n_blk
    cand = [(-float(s), pos[i], k, i) for i in S for k, s in enumerate(S[i])]
    cand.sort()
    cand = [(ms, i, k) for (ms, _, k, i) in cand]
    smax = -cand[0][0] if cand else 0.0
    kept = {i: [] for i in S}
    limit = chi_max
    if eps_discard >= 0.0:
        # tail[n] = weight discarded when the n largest are kept, summed smallest first
        tail = np.concatenate([np.cumsum(np.array([c[0] for c in cand[::-1]]) ** 2)[::-1], [0.0]])
        limit = min(chi_max, int(np.argmax(tail <= eps_discard)))
    n = 0
    for (ms, i, k) in cand:
        if n >= limit or -ms <= SIGMA_FLOOR * smax:
            break
        kept[i].append(k)
        n += 1
    chi = np.zeros(nL, np.int32)
    ot, sigma = [], []
    disc = 0.0
    for i in range(nL):
        if i not in S:
            ot.append(np.zeros((0, int(dims[i]))))
            sigma.append(np.zeros(0))
            continue
        ks = kept[i]
        chi[i] = len(ks)
        ot.append(U[i][:, ks].T.copy())
        sigma.append(S[i].copy())
        mask = np.ones(S[i].shape[0], bool)
        mask[ks] = False
        disc += float(np.sum(S[i][mask] ** 2))
    return chi, ot, sigma, disc


def rotate(d, chi, blocks, a_data, ot) -> List[np.ndarray]:
    """Reading R4: A'[a,a'] = sum_{x,x'} O_l[x,a] A[x,x'] O_l'[x',a'] for every operator block (row sector l, column
    sector l'), with ``ot[l]`` = O_l^T as a (chi_l, d_l) array.  Returns one (chi_l, chi_l') array per input block
    (possibly with a zero dimension).  Written as the definition, the two sums being two matrix products."""
    out = []
    for e in blocks:
        l, lp, ld, off = int(e["row"]), int(e["col"]), int(e["ld"]), int(e["offset"])
        r, c = int(d[l]), int(d[lp])
        A = np.lib.stride_tricks.as_strided(a_data[off:], shape=(r, c), strides=(ld * 8, 8))
        Ol, Olp = np.asarray(ot[l]), np.asarray(ot[lp])
        assert Ol.shape == (int(chi[l]), r) and Olp.shape == (int(chi[lp]), c)
        # t[a,x'] = sum_x O_l[x,a] A[x,x']   then   A'[a,a'] = sum_x' t[a,x'] O_l'[x',a']   (two BLAS products, FP64)
        Ap = (Ol @ A) @ Olp.T
        out.append(Ap)
    return out


def rotate_flops(d, chi, blocks) -> int:
    """Useful flops of the update in the order the product takes (right index first, reading R5):
    2 d_l d_l' chi_l' + 2 chi_l d_l chi_l' per block; a block whose row or column sector keeps nothing has no result
    and counts nothing."""
    f = 0
    for e in blocks:
        l, lp = int(e["row"]), int(e["col"])
        if int(chi[l]) == 0 or int(chi[lp]) == 0:
            continue
        f += 2 * int(d[l]) * int(d[lp]) * int(chi[lp]) + 2 * int(chi[l]) * int(d[l]) * int(chi[lp])
    return f
