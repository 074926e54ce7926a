"""Seeded inputs for the site-update steps: kept dimensions and isometries to rotate with.

Input drawing only - no SVD of a wavefunction, no operator rotation (those are the method's arithmetic and live in
oracle/ and in the CUDA library).  Orthonormal rows are drawn as the Q factor of a Gaussian matrix."""
from __future__ import annotations

from typing import List

import numpy as np


def proportional_chi(d, keep: float = 0.25, zero_every: int = 0) -> np.ndarray:
    """Kept dimension per sector: round(keep * d), at least 1; every ``zero_every``-th sector (if > 0) keeps nothing
    (a sector the truncation dropped altogether).  keep = 1/4 mirrors the site dimension 4 of PAPER.md:51-53."""
    d = np.asarray(d, np.int64)
    chi = np.maximum(1, np.rint(keep * d)).astype(np.int32)
    chi = np.minimum(chi, d.astype(np.int32))
    if zero_every > 0:
        chi[zero_every - 1::zero_every] = 0
    return chi


def make_isometries(d, chi, seed: int) -> List[np.ndarray]:
    """ot[l] = O_l^T, a (chi_l, d_l) array with orthonormal rows (Q factor of a seeded Gaussian d_l x chi_l matrix)."""
    out = []
    for l, (dl, cl) in enumerate(zip(np.asarray(d), np.asarray(chi))):
        rng = np.random.default_rng([seed, 505, l])
        g = rng.standard_normal((int(dl), int(cl)))
        if cl == 0:
            out.append(np.zeros((0, int(dl))))
            continue
        q, _ = np.linalg.qr(g)
        out.append(np.ascontiguousarray(q.T))
    return out


def pack_isometries(ot) -> np.ndarray:
    """Boundary layout of include/hpsi.h: O_l^T (chi_l x d_l, dense row-major) concatenated by ascending sector."""
    if not ot:
        return np.zeros(0)
    return np.concatenate([np.ascontiguousarray(o, np.float64).ravel() for o in ot] + [np.zeros(0)])
