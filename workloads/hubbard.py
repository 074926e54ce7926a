"""Hubbard chains written in the two-block form  H = sum_t c_t A_t (x) B_t  (textbook pins).

Each side is a block of ``ns`` sites (modes ordered site-major, spin up then down) represented with
Jordan-Wigner matrices.  Sectors are labelled (N, 2Sz).  A fermionic operator on the right block
anticommutes past the left block's electrons; that sign is the left parity P, folded into A (reading A5).
Only operator *construction* lives here; nothing is contracted.
"""
from __future__ import annotations

import numpy as np

from .configs import Problem, custom_problem

_a = np.array([[0.0, 1.0], [0.0, 0.0]])      # annihilator on one mode, basis (|0>, |1>)
_Z = np.diag([1.0, -1.0])
_I = np.eye(2)


def _kron(*ms):
    out = np.eye(1)
    for m in ms:
        out = np.kron(out, m)
    return out


def block_operators(ns: int):
    """Annihilators c[mode], number operators n[mode] and parity P of an ns-site block (dense 4^ns)."""
    nm = 2 * ns
    c = [_kron(*([_Z] * j + [_a] + [_I] * (nm - j - 1))) for j in range(nm)]
    n = [x.T @ x for x in c]
    P = _kron(*([_Z] * nm))
    return c, n, P


def block_hamiltonian(ns: int, t: float, U: float) -> np.ndarray:
    c, n, _ = block_operators(ns)
    H = np.zeros((4 ** ns, 4 ** ns))
    for s in range(ns):
        H = H + U * n[2 * s] @ n[2 * s + 1]
    for s in range(ns - 1):
        for sp in (0, 1):
            H = H - t * (c[2 * s + sp].T @ c[2 * (s + 1) + sp] + c[2 * (s + 1) + sp].T @ c[2 * s + sp])
    return H


def _sectorize(ns: int):
    """Sort the 4^ns block states by (N, 2Sz).  Returns labels [n_sec,2], dims [n_sec], order (state perm)."""
    _, n, _ = block_operators(ns)
    Nn = np.rint(np.diag(sum(n))).astype(int)
    Sz = np.rint(np.diag(sum(n[0::2]) - sum(n[1::2]))).astype(int)
    labels = sorted(set(zip(Nn.tolist(), Sz.tolist())))
    order, dims = [], []
    for lab in labels:
        idx = [i for i in range(4 ** ns) if (Nn[i], Sz[i]) == lab]
        order += idx
        dims.append(len(idx))
    return np.array(labels, np.int32), np.array(dims, np.int32), np.array(order)


def _blocks_of(op: np.ndarray, order: np.ndarray, dims: np.ndarray):
    """Cut a dense block-basis operator into its nonzero (row sector, col sector) blocks."""
    M = op[np.ix_(order, order)]
    offs = np.concatenate([[0], np.cumsum(dims)])
    out = {}
    for r in range(len(dims)):
        for c in range(len(dims)):
            blk = M[offs[r]:offs[r + 1], offs[c]:offs[c + 1]]
            if np.any(blk != 0.0):
                out[(r, c)] = blk.copy()
    return out


def hubbard_two_block_problem(ns_left: int, ns_right: int, t: float, U: float, n_elec: int, two_sz: int,
                              pad_even: bool = False) -> Problem:
    """Open Hubbard chain of ns_left+ns_right sites as left block (x) right block, target sector (n_elec, two_sz)."""
    qL, dL, oL = _sectorize(ns_left)
    qR, dR, oR = _sectorize(ns_right)
    cL, _, PL = block_operators(ns_left)
    cR, _, _ = block_operators(ns_right)
    IL, IR = np.eye(4 ** ns_left), np.eye(4 ** ns_right)
    dense_terms = [(1.0, block_hamiltonian(ns_left, t, U), IR), (1.0, IL, block_hamiltonian(ns_right, t, U))]
    for sp in (0, 1):
        A = cL[2 * (ns_left - 1) + sp].T @ PL     # c^dagger on the last left site, times left parity
        B = cR[sp]                                 # annihilator on the first right site (block-local JW)
        dense_terms += [(-t, A, B), (-t, A.T, B.T)]
    terms = [(c, _blocks_of(A, oL, dL), _blocks_of(B, oR, dR)) for c, A, B in dense_terms]
    return custom_problem(qL, dL, qR, dR, (n_elec, two_sz), terms, pad_even=pad_even,
                          name=f"hubbard{ns_left}+{ns_right}")


def monolithic_hubbard(n_sites: int, t: float, U: float) -> np.ndarray:
    """Dense Jordan-Wigner Hamiltonian of the whole open chain (for checking the two-block construction)."""
    return block_hamiltonian(n_sites, t, U)
