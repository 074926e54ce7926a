"""ORACLE - test infrastructure, not product code.

Plain, slow, obviously-correct CPU implementation of what the hot path computes (BASELINE.json
`north_star`; PAPER.md:62 names the step, SURVEY.md 8(c) / DESIGN.md give the readings):

    psi'(l,r) = sum_t c_t A_t(l,l') psi(l',r') B_t(r,r')^T      and a textbook Davidson around it.

* ``apply``            - C loop (hpsi_oracle.c) over terms x A blocks x B blocks, always (A psi) B^T, FP64.
* ``apply_samples``    - single output elements, one by one (for sizes a whole apply cannot reach).
* ``psi_table``        - the psi block table (step 1).
* ``dense_hamiltonian``- H restricted to the target sector, column by column through ``apply``.
* ``diagonal``         - diag(H) from the terms whose A and B blocks are both sector-diagonal (reading A21).
* ``davidson``         - Davidson-Liu, single root, step by step as reading A21 states it.
* ``davidson_block``   - the same for the k lowest eigenpairs at once (block / multi-root variant, reading A21b).
* ``useful_flops``     - the flop convention of reading A18.

Only tests/, ``__graft_entry__.smoke()`` and bench.py's cpu_baseline / ``--impl reference`` legs may import
this package.  It imports nothing from ``paper_2407_07411_b200`` and shares no code with it.

Pins: tests/test_oracle_pins.py (Kronecker brute force, Hermiticity, A@psi@B.T, closed forms, Hubbard
dimer and 4-site chain energies, dense eigensolver; ``davidson_block``: the k lowest levels of the dense toy
Hamiltonian, the dimer's closed-form spectrum, and k = 1 reproducing ``davidson`` step for step).  Unpinned: SU(2) recoupling / real-molecule
energies (the paper's integrals are not available) - "parity unpinned", out of scope.
"""
from __future__ import annotations

import ctypes
from typing import Optional, Tuple

import numpy as np

from .build import build as _build

_lib = None

_I32P = ctypes.POINTER(ctypes.c_int32)
_I64P = ctypes.POINTER(ctypes.c_int64)
_F64P = ctypes.POINTER(ctypes.c_double)


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build())
        _lib.oracle_psi_table.restype = ctypes.c_int64
        _lib.oracle_apply.restype = ctypes.c_int
        _lib.oracle_apply_samples.restype = ctypes.c_int
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def _i32(a):
    a = np.ascontiguousarray(a, np.int32)
    return a, a.ctypes.data_as(_I32P)


def _f64(a):
    a = np.ascontiguousarray(a, np.float64)
    return a, a.ctypes.data_as(_F64P)


def _sector_args(p):
    keep = []
    args = [ctypes.c_int32(p.q_left.shape[0]), ctypes.c_int32(p.q_right.shape[0])]
    for arr in (p.q_left, p.q_right, p.d_left, p.d_right, p.target):
        a, ptr = _i32(arr)
        keep.append(a)
        args.append(ptr)
    return args, keep


def _term_args(p, a_desc=None, a_data=None, b_desc=None, b_data=None):
    a_desc = p.a_desc if a_desc is None else a_desc
    b_desc = p.b_desc if b_desc is None else b_desc
    a_data = p.a_data if a_data is None else a_data
    b_data = p.b_data if b_data is None else b_data
    assert a_desc.dtype.itemsize == 24 and b_desc.dtype.itemsize == 24
    a_desc = np.ascontiguousarray(a_desc)
    b_desc = np.ascontiguousarray(b_desc)
    coef, coef_p = _f64(p.coef)
    ad, ad_p = _f64(a_data)
    bd, bd_p = _f64(b_data)
    args = [ctypes.c_int32(coef.shape[0]), coef_p,
            ctypes.c_int64(a_desc.shape[0]), ctypes.c_void_p(a_desc.ctypes.data), ad_p,
            ctypes.c_int64(b_desc.shape[0]), ctypes.c_void_p(b_desc.ctypes.data), bd_p]
    return args, [coef, ad, bd, a_desc, b_desc]


def psi_table(p) -> Tuple[np.ndarray, np.ndarray, int]:
    """(partner[n_left], offset[n_left], psi_len) - step 1 of SURVEY.md 8(a)."""
    sargs, keep = _sector_args(p)
    partner = np.empty(p.q_left.shape[0], np.int32)
    offset = np.empty(p.q_left.shape[0], np.int64)
    n = lib().oracle_psi_table(*sargs, partner.ctypes.data_as(_I32P), offset.ctypes.data_as(_I64P))
    return partner, offset, int(n)


def apply(p, psi: np.ndarray) -> np.ndarray:
    """out = H psi by the plain definition (C loop)."""
    _, _, n = psi_table(p)
    psi_c, psi_p = _f64(psi)
    assert psi_c.shape == (n,), (psi_c.shape, n)
    out = np.empty(n, np.float64)
    sargs, k1 = _sector_args(p)
    targs, k2 = _term_args(p)
    rc = lib().oracle_apply(*sargs, *targs, psi_p, out.ctypes.data_as(_F64P))
    if rc != 0:
        raise MemoryError("oracle_apply failed")
    return out


def apply_samples(p, psi: np.ndarray, sample_left, sample_x, sample_y, vals: Optional[np.ndarray] = None,
                  a_desc=None, a_data=None, b_desc=None, b_data=None) -> np.ndarray:
    """vals[s] += (H psi)[block sample_left[s]][sample_x[s], sample_y[s]], element by element.
    Optional descriptor/arena overrides let a caller stream disjoint term subsets (offsets relative to the arenas passed)."""
    psi_c, psi_p = _f64(psi)
    sl, sl_p = _i32(sample_left)
    sx, sx_p = _i32(sample_x)
    sy, sy_p = _i32(sample_y)
    if vals is None:
        vals = np.zeros(sl.shape[0], np.float64)
    assert vals.dtype == np.float64 and vals.flags.c_contiguous
    sargs, k1 = _sector_args(p)
    targs, k2 = _term_args(p, a_desc, a_data, b_desc, b_data)
    rc = lib().oracle_apply_samples(*sargs, *targs, psi_p, ctypes.c_int32(sl.shape[0]), sl_p, sx_p, sy_p,
                                    vals.ctypes.data_as(_F64P))
    if rc != 0:
        raise MemoryError("oracle_apply_samples failed")
    return vals


def dense_hamiltonian(p) -> np.ndarray:
    """H restricted to the target sector (psi_len x psi_len), column j = apply(e_j).  Tiny problems only."""
    _, _, n = psi_table(p)
    H = np.empty((n, n))
    e = np.zeros(n)
    for j in range(n):
        e[j] = 1.0
        H[:, j] = apply(p, e)
        e[j] = 0.0
    return H


def _blk(data, e, dims):
    r, c, ld, off = int(dims[e["row"]]), int(dims[e["col"]]), int(e["ld"]), int(e["offset"])
    return np.lib.stride_tricks.as_strided(data[off:], shape=(r, c), strides=(ld * 8, 8))


def diagonal(p) -> np.ndarray:
    """diag(H) on the psi layout (reading A21): only tasks whose A block and B block are both sector-diagonal
    touch the diagonal,  diag[l][x,y] = sum_t c_t A_t[l,l][x,x] B_t[r,r][y,y],  r = partner(l)."""
    partner, offset, n = psi_table(p)
    d = np.zeros(n)
    for ea in p.a_desc:
        l = int(ea["row"])
        if int(ea["col"]) != l or partner[l] < 0:
            continue
        t = int(ea["term"])
        r = int(partner[l])
        for eb in p.b_desc:
            if int(eb["term"]) != t or int(eb["row"]) != r or int(eb["col"]) != r:
                continue
            da = np.diag(_blk(p.a_data, ea, p.d_left))
            db = np.diag(_blk(p.b_data, eb, p.d_right))
            m, nn = int(p.d_left[l]), int(p.d_right[r])
            d[offset[l]: offset[l] + m * nn] += p.coef[t] * np.outer(da, db).ravel()
    return d


def useful_flops(p) -> Tuple[int, int]:
    """(useful_flops, n_tasks) under reading A18: per task min(2 m n'(k+n), 2 k n (n'+m)), 2MNK per GEMM."""
    partner, _, _ = psi_table(p)
    flops = 0
    ntask = 0
    b_by_term = {}
    for eb in p.b_desc:
        b_by_term.setdefault(int(eb["term"]), []).append((int(eb["row"]), int(eb["col"])))
    for ea in p.a_desc:
        l, lp, t = int(ea["row"]), int(ea["col"]), int(ea["term"])
        if partner[l] < 0 or partner[lp] < 0:
            continue
        for (r, rp) in b_by_term.get(t, ()):
            if r != partner[l] or rp != partner[lp]:
                continue
            m, k, n1, n = int(p.d_left[l]), int(p.d_left[lp]), int(p.d_right[rp]), int(p.d_right[r])
            flops += min(2 * m * n1 * (k + n), 2 * k * n * (n1 + m))
            ntask += 1
    return flops, ntask


def davidson(p, v0: np.ndarray, tol: float = 1e-8, max_iter: int = 200, m_max: int = 16,
             precondition: bool = True, matvec=None):
    """Davidson-Liu for the lowest eigenpair, single root, exactly as reading A21 lists it.

    V=[v0/|v0|]; loop: W=H V (one new column per iteration), G=V^T W, smallest Ritz pair (theta,y), x=V y,
    r=W y - theta x; stop if |r|<=tol; s=r/(diag(H)-theta) with small-denominator guard (or s=r); orthogonalise
    s against V twice (classical Gram-Schmidt, applied twice); if the preconditioned s vanishes (|s| < 1e-14) retry with
    s=r (reading A21c); append; when dim V == m_max restart with V=[x].
    Returns (theta, x, n_matvec, residual_norm)."""
    mv = (lambda x: apply(p, x)) if matvec is None else matvec
    d = diagonal(p) if precondition else None
    v = np.asarray(v0, np.float64)
    V = [v / np.linalg.norm(v)]
    Wc = [mv(V[0])]
    nmv = 1
    theta, x, rn = 0.0, V[0], np.inf
    for _ in range(max_iter):
        Vm = np.stack(V, axis=1)
        Wm = np.stack(Wc, axis=1)
        G = Vm.T @ Wm
        G = 0.5 * (G + G.T)
        ev, Y = np.linalg.eigh(G)
        theta, y = float(ev[0]), Y[:, 0]
        x = Vm @ y
        r = Wm @ y - theta * x
        rn = float(np.linalg.norm(r))
        if rn <= tol:
            break
        if d is not None:
            den = d - theta
            den = np.where(np.abs(den) < 1e-8, np.where(den < 0, -1e-8, 1e-8), den)
            s = r / den
        else:
            s = r.copy()
        if len(V) >= m_max:
            xn = x / np.linalg.norm(x)
            V = [xn]
            Wc = [Wm @ y / np.linalg.norm(x)]
            Vm = np.stack(V, axis=1)
        for _pass in range(2):
            s = s - Vm @ (Vm.T @ s)
        ns = np.linalg.norm(s)
        if ns < 1e-14 and d is not None:
            # reading A21c: the preconditioned correction lies in span(V) (e.g. H diagonal, where r/(diag - theta) is the
            # Ritz vector itself) although |r| > tol: take the residual itself as the new direction
            s = r.copy()
            for _pass in range(2):
                s = s - Vm @ (Vm.T @ s)
            ns = np.linalg.norm(s)
        if ns < 1e-14:
            break
        s = s / ns
        V.append(s)
        Wc.append(mv(s))
        nmv += 1
    return theta, x / np.linalg.norm(x), nmv, rn


def davidson_block(p, V0: np.ndarray, tol: float = 1e-8, max_iter: int = 200, m_max: int = 16,
                   precondition: bool = True, matvec=None):
    """Block Davidson-Liu for the k lowest eigenpairs (k = number of columns of V0), reading A21b of DESIGN.md - the
    "multi-root" companion of ``davidson`` (PAPER.md:62 only names "the Lanczos or Davidson method"):

    V = the k start vectors orthonormalised one after the other (classical Gram-Schmidt applied twice); W = H V.  Loop:
    G = V^T W (symmetrised), its k lowest Ritz pairs (theta_i, y_i), x_i = V y_i, r_i = W y_i - theta_i x_i; stop when
    every |r_i| <= tol or ``max_iter`` mat-vecs are spent.  For every root with |r_i| > tol, in ascending i:
    s = r_i / (diag(H) - theta_i) with the small-denominator guard (or s = r_i), orthogonalised twice against the current
    V (which includes the vectors appended before it in this iteration), dropped if |s| < 1e-14, else normalised and
    appended.  If appending would exceed m_max columns, V is first replaced by [x_1 .. x_k] (and W by [W y_1 .. W y_k]).
    One mat-vec per appended vector.  Returns (theta[k], X[n, k], n_matvec, residual_norms[k])."""
    mv = (lambda x: apply(p, x)) if matvec is None else matvec
    d = diagonal(p) if precondition else None
    V0 = np.asarray(V0, np.float64)
    k = V0.shape[1]
    assert 1 <= k <= m_max // 2, "m_max must hold the k Ritz vectors and k corrections"
    V = []
    for i in range(k):
        v = V0[:, i].copy()
        for _pass in range(2):
            for u in V:
                v = v - u * (u @ v)
        V.append(v / np.linalg.norm(v))
    Wc = [mv(v) for v in V]
    nmv = k
    theta, X, rn = np.zeros(k), np.stack(V, axis=1), np.full(k, np.inf)
    while True:
        Vm, Wm = np.stack(V, axis=1), np.stack(Wc, axis=1)
        G = Vm.T @ Wm
        G = 0.5 * (G + G.T)
        ev, Y = np.linalg.eigh(G)
        theta, Yk = ev[:k].copy(), Y[:, :k]
        X = Vm @ Yk
        WY = Wm @ Yk
        Rm = WY - X * theta[None, :]
        rn = np.linalg.norm(Rm, axis=0)
        todo = [i for i in range(k) if rn[i] > tol]
        if not todo or nmv >= max_iter:
            break
        if len(V) + len(todo) > m_max:                 # restart from the Ritz vectors
            V = [X[:, i].copy() for i in range(k)]
            Wc = [WY[:, i].copy() for i in range(k)]
        new = []
        for i in todo:
            if nmv + len(new) >= max_iter:
                break
            r = Rm[:, i]
            if d is not None:
                den = d - theta[i]
                den = np.where(np.abs(den) < 1e-8, np.where(den < 0, -1e-8, 1e-8), den)
                s = r / den
            else:
                s = r.copy()
            for _pass in range(2):
                Vm = np.stack(V, axis=1)
                s = s - Vm @ (Vm.T @ s)
            ns = np.linalg.norm(s)
            if ns < 1e-14 and d is not None:             # reading A21c: fall back to the residual itself
                s = r.copy()
                for _pass in range(2):
                    Vm = np.stack(V, axis=1)
                    s = s - Vm @ (Vm.T @ s)
                ns = np.linalg.norm(s)
            if ns < 1e-14:
                continue
            V.append(s / ns)
            new.append(V[-1])
        if not new:
            break
        for v in new:
            Wc.append(mv(v))
        nmv += len(new)
    return theta, X, nmv, rn
