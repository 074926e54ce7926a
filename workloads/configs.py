"""Seeded generators for the five BASELINE.json configs.

Everything here is input *drawing* only.  A ``Problem`` is exactly what crosses the C-ABI boundary of
``include/hpsi.h`` (host sector table, host block descriptors, operator arenas, coefficients) plus the
by-construction psi block table the generator itself knows (so tests can cross-check the table that the
oracle and the planner each derive on their own).

Readings of BASELINE.json used here (DESIGN.md lists them, A6-A16 of SURVEY.md 8(c)):
  * labels are an abstract integer grid, N step 1 and 2Sz step 2, no parity constraint (A7);
  * right labels are Q* - q_left, stored in a seeded random permutation (8(d) "Label grids");
  * A_t maps left sector q -> q+delta_t, B_t maps right sector q -> q-delta_t (A6);
  * A_t / B_t carry a block for *every* sector whose shifted label exists on that side (A8);
  * the second half of the term list holds the adjoints (same c_t, -delta, transposed blocks) (A9);
  * base-term block entries are N(0,1)/sqrt(#columns of the block) (A10); psi is N(0,1), ||psi||=1 (A11).
"""
from __future__ import annotations

import dataclasses
from typing import Dict, List, Optional, Tuple

import numpy as np

# Mirrors ``hpsi_opblock_t`` in include/hpsi.h (24 bytes, natural alignment).
OPBLOCK_DTYPE = np.dtype([("term", "<i4"), ("row", "<i4"), ("col", "<i4"), ("ld", "<i4"),
                          ("offset", "<i8")], align=True)
assert OPBLOCK_DTYPE.itemsize == 24

CONFIG_NAMES = ("toy", "small", "cyp", "femoco", "stress")

# (n_sectors, grid (gN, gS), D, n_terms, dims recipe)
_PARAMS = {
    "toy":    dict(index=0, grid=(5, 2), D=None, n_terms=48,   dims="uniform16"),
    "small":  dict(index=1, grid=(6, 4), D=1024, n_terms=400,  dims="gauss"),
    "cyp":    dict(index=2, grid=(8, 5), D=4096, n_terms=1700, dims="gauss"),
    "femoco": dict(index=3, grid=(8, 6), D=8192, n_terms=2900, dims="gauss"),
    "stress": dict(index=4, grid=(8, 8), D=4096, n_terms=1200, dims="pareto_mix"),
}

SHIFTS = [(dn, ds) for dn in (-2, -1, 0, 1, 2) for ds in (-2, 0, 2)]   # the 15 (dN, d2Sz) values


def config_params(name: str) -> dict:
    return dict(_PARAMS[name])


@dataclasses.dataclass
class Problem:
    """One H_eff*psi instance in boundary form (host numpy arrays)."""
    name: str
    seed: int
    q_left: np.ndarray          # [n_left, 2] int32  (N, 2Sz)
    q_right: np.ndarray         # [n_right, 2] int32
    d_left: np.ndarray          # [n_left] int32
    d_right: np.ndarray         # [n_right] int32
    target: np.ndarray          # [2] int32  Q*
    coef: np.ndarray            # [n_terms] float64
    a_desc: np.ndarray          # [n_a] OPBLOCK_DTYPE
    b_desc: np.ndarray          # [n_b] OPBLOCK_DTYPE
    a_len: int                  # doubles in the A arena
    b_len: int
    a_data: Optional[np.ndarray] = None   # float64 arenas (None until filled)
    b_data: Optional[np.ndarray] = None
    a_trans: Optional[np.ndarray] = None  # [n_a] uint8: 1 = the arena holds this block transposed (adjoint-pair sharing)
    b_trans: Optional[np.ndarray] = None
    # generator-side bookkeeping (not part of the boundary)
    shifts: Optional[np.ndarray] = None   # [n_terms, 2]
    partner: Optional[np.ndarray] = None  # [n_left] right index paired with left i by construction, -1 if none
    term_a_range: Optional[np.ndarray] = None   # [n_terms, 2] descriptor index range of each term in a_desc
    term_b_range: Optional[np.ndarray] = None
    entry_seed: Optional[Tuple[int, ...]] = None
    base_term_ids: Optional[np.ndarray] = None  # [n_terms/2] index of each base term in the full config (term shards)

    @property
    def n_terms(self) -> int:
        return int(self.coef.shape[0])

    @property
    def psi_len(self) -> int:
        tot = 0
        for i, j in enumerate(self.partner):
            if j >= 0:
                tot += int(self.d_left[i]) * int(self.d_right[j])
        return tot

    def psi_blocks(self) -> List[Tuple[int, int, int, int, int]]:
        """By-construction psi block table: (left i, right j, rows, cols, offset), ascending i, dense row-major."""
        out, off = [], 0
        for i, j in enumerate(self.partner):
            if j >= 0:
                r, c = int(self.d_left[i]), int(self.d_right[j])
                out.append((i, int(j), r, c, off))
                off += r * c
        return out

    def operator_bytes(self) -> int:
        """Bytes of operator entries proper (rows*cols*8 per block, padding excluded)."""
        tot = 0
        for desc, d in ((self.a_desc, self.d_left), (self.b_desc, self.d_right)):
            tot += int(np.sum(d[desc["row"]].astype(np.int64) * d[desc["col"]].astype(np.int64))) * 8
        return tot

    def block(self, side: str, idx: int) -> np.ndarray:
        """View of operator block ``idx`` of side 'a' or 'b' as a (rows, cols) array."""
        desc, data, d = ((self.a_desc, self.a_data, self.d_left) if side == "a"
                         else (self.b_desc, self.b_data, self.d_right))
        return _block_view(data, desc[idx], d)


# ----------------------------------------------------------------------------------------------- dims
def _round_to_sum(w: np.ndarray, total: int) -> np.ndarray:
    """Largest-remainder rounding of positive weights to integers >= 1 summing exactly to total (A13)."""
    n = w.size
    assert total >= n
    x = w / w.sum() * (total - n)          # every sector gets 1, distribute the rest
    base = np.floor(x).astype(np.int64)
    rem = int(total - n - base.sum())
    order = np.argsort(-(x - base), kind="stable")
    base[order[:rem]] += 1
    out = base + 1
    assert out.sum() == total and out.min() >= 1
    return out.astype(np.int32)


def _gauss_dims(rng: np.random.Generator, gN: int, gS: int, D: int) -> np.ndarray:
    """Discretised Gaussian over the label grid, centred on the grid middle, +-2 sigma spans it, with a
    log-normal(0.25) jitter (A14).  Returned in grid order a*gS+b."""
    a = np.arange(gN)[:, None]
    b = np.arange(gS)[None, :]
    cN, cS = (gN - 1) / 2.0, (gS - 1) / 2.0
    sN, sS = gN / 4.0, gS / 4.0
    w = np.exp(-0.5 * (((a - cN) / sN) ** 2 + ((b - cS) / sS) ** 2))
    w = w * np.exp(0.25 * rng.standard_normal(w.shape))
    return _round_to_sum(w.ravel(), D)


def _pareto_mix_dims(rng: np.random.Generator, n: int, D: int) -> np.ndarray:
    """A16 mixture: 3/4 of the sectors uniform 1..8, 1/4 Pareto(alpha=1.5) scaled so the side totals D exactly,
    each clipped at 1024.  Returned sorted descending (placement is done by the caller)."""
    n_big = n // 4
    n_small = n - n_big
    small = rng.integers(1, 9, size=n_small)
    raw = 1.0 + rng.pareto(1.5, size=n_big)
    want = D - int(small.sum())
    lo, hi = 1e-6, 1e6
    for _ in range(200):                       # bisection on the scale so that sum(clip(round)) ~ want
        mid = np.sqrt(lo * hi)
        s = np.minimum(np.maximum(np.rint(raw * mid), 1), 1024).sum()
        if s < want:
            lo = mid
        else:
            hi = mid
    big = np.minimum(np.maximum(np.rint(raw * hi), 1), 1024).astype(np.int64)
    # fix the residual on unclipped entries, largest first
    diff = int(want - big.sum())
    order = np.argsort(-big, kind="stable")
    k = 0
    while diff != 0:
        i = order[k % n_big]
        step = 1 if diff > 0 else -1
        if 1 <= big[i] + step <= 1024:
            big[i] += step
            diff -= step
        k += 1
    dims = np.concatenate([big, small]).astype(np.int32)
    assert dims.sum() == D
    return np.sort(dims)[::-1].copy()


# ------------------------------------------------------------------------------------- sector tables
def _sector_tables(name: str, seed: int, D: Optional[int] = None):
    p = dict(_PARAMS[name])
    if D is not None:                       # bond-dimension sweep (Fig. 1 / Fig. 2 plot against D): same grid,
        assert p["D"] is not None           # same profile and jitter, dims rounded to the new total
        p["D"] = int(D)
    gN, gS = p["grid"]
    rng = np.random.default_rng([seed, 101])
    n = gN * gS
    if name == "toy":
        target = np.array([8, 0], np.int32)
        Ns = np.arange(2, 2 + gN)
        Ss = np.array([0, 2])
    else:
        n0 = 10
        target = np.array([2 * n0 + gN - 1, 0], np.int32)
        Ns = np.arange(n0, n0 + gN)
        Ss = -(gS - 1) + 2 * np.arange(gS)
    q_left = np.array([(N, S) for N in Ns for S in Ss], np.int32)          # grid order a*gS+b
    if p["dims"] == "uniform16":
        rng0 = np.random.default_rng(seed)                                 # A12: default_rng(0).integers(1,7)
        d_left = rng0.integers(1, 7, size=n).astype(np.int32)
        d_right_by_partner = rng0.integers(1, 7, size=n).astype(np.int32)
    elif p["dims"] == "gauss":
        d_left = _gauss_dims(rng, gN, gS, p["D"])
        d_right_by_partner = _gauss_dims(rng, gN, gS, p["D"])              # same profile (mirror grid), own jitter
    else:
        big_l = _pareto_mix_dims(rng, n, p["D"])
        big_r = _pareto_mix_dims(rng, n, p["D"])
        place = rng.permutation(n)                                         # seeded placement on the grid
        d_left = np.empty(n, np.int32)
        d_right_by_partner = np.empty(n, np.int32)
        d_left[place] = big_l                                              # rank-matched: k-th largest left pairs
        d_right_by_partner[place] = big_r                                  # with k-th largest right
    # right side: label Q*-q_left[i], stored at position perm[i]
    perm = rng.permutation(n)
    q_right = np.empty_like(q_left)
    d_right = np.empty(n, np.int32)
    q_right[perm] = target[None, :] - q_left
    d_right[perm] = d_right_by_partner
    partner = perm.astype(np.int32)
    return q_left, q_right, d_left, d_right, target, partner


def _label_index(q: np.ndarray) -> Dict[Tuple[int, int], int]:
    return {(int(a), int(b)): i for i, (a, b) in enumerate(q)}


def _round_up(x: int, a: int) -> int:
    return (x + a - 1) // a * a


# -------------------------------------------------------------------------------------------- builder
def _build_descriptors(q_left, q_right, d_left, d_right, shifts, row_align: int):
    """Descriptor tables for all terms.  Arena layout: term-major, within a term blocks by ascending source
    (column) sector; ld = #cols and block offsets rounded up to a multiple of ``row_align`` doubles (4: every row
    starts on a 32-byte L2 sector, the library's preferred layout; 2: 16-byte rows; 1: dense, 8-byte rows)."""
    n_terms = shifts.shape[0]
    li, ri = _label_index(q_left), _label_index(q_right)
    a_rows, b_rows = [], []
    ta = np.zeros((n_terms, 2), np.int64)
    tb = np.zeros((n_terms, 2), np.int64)
    a_off = b_off = 0
    for t in range(n_terms):
        dn, ds = int(shifts[t, 0]), int(shifts[t, 1])
        ta[t, 0] = len(a_rows)
        for c in range(q_left.shape[0]):
            r = li.get((int(q_left[c, 0]) + dn, int(q_left[c, 1]) + ds))
            if r is None:
                continue
            ld = _round_up(int(d_left[c]), row_align)
            a_rows.append((t, r, c, ld, a_off))
            a_off = _round_up(a_off + int(d_left[r]) * ld, row_align)
        ta[t, 1] = len(a_rows)
        tb[t, 0] = len(b_rows)
        for c in range(q_right.shape[0]):
            r = ri.get((int(q_right[c, 0]) - dn, int(q_right[c, 1]) - ds))
            if r is None:
                continue
            ld = _round_up(int(d_right[c]), row_align)
            b_rows.append((t, r, c, ld, b_off))
            b_off = _round_up(b_off + int(d_right[r]) * ld, row_align)
        tb[t, 1] = len(b_rows)
    a_desc = np.array(a_rows, dtype=OPBLOCK_DTYPE) if a_rows else np.zeros(0, OPBLOCK_DTYPE)
    b_desc = np.array(b_rows, dtype=OPBLOCK_DTYPE) if b_rows else np.zeros(0, OPBLOCK_DTYPE)
    return a_desc, b_desc, a_off, b_off, ta, tb


def _block_view(data, desc_entry, dims):
    r, c = int(dims[desc_entry["row"]]), int(dims[desc_entry["col"]])
    ld, off = int(desc_entry["ld"]), int(desc_entry["offset"])
    return np.lib.stride_tricks.as_strided(data[off:], shape=(r, c), strides=(ld * 8, 8))


def fill_term(p: Problem, t: int, a_data: np.ndarray, b_data: np.ndarray,
              a_base: int = 0, b_base: int = 0) -> None:
    """Draw the entries of base term t (t < T/2) *and* its adjoint t+T/2 into the arenas.

    ``a_base``/``b_base`` are subtracted from descriptor offsets, which lets a caller stream a window of
    terms through a small staging buffer (used for the D=8192 config).  Entries: N(0,1)/sqrt(#cols) (A10);
    adjoint blocks are exact transposes (A9).  The stream of term t depends only on (entry_seed, t)."""
    half = p.n_terms // 2
    assert 0 <= t < half
    gid = int(p.base_term_ids[t]) if p.base_term_ids is not None else t      # stream of the term in the full config
    rng = np.random.default_rng(list(p.entry_seed) + [gid])
    for desc, rng_tab, data, base, dims in ((p.a_desc, p.term_a_range, a_data, a_base, p.d_left),
                                            (p.b_desc, p.term_b_range, b_data, b_base, p.d_right)):
        lo, hi = rng_tab[t]
        alo, ahi = rng_tab[t + half]
        adj = {(int(desc[i]["row"]), int(desc[i]["col"])): i for i in range(alo, ahi)}
        for i in range(lo, hi):
            e = desc[i]
            r, c = int(dims[e["row"]]), int(dims[e["col"]])
            blk = rng.standard_normal((r, c)) / np.sqrt(c)
            off = int(e["offset"]) - base
            ld = int(e["ld"])
            np.lib.stride_tricks.as_strided(data[off:], shape=(r, c), strides=(ld * 8, 8))[...] = blk
            if p.a_trans is not None:          # adjoint terms share the base term's storage (read transposed)
                continue
            j = adj[(int(e["col"]), int(e["row"]))]
            ea = desc[j]
            offa, lda = int(ea["offset"]) - base, int(ea["ld"])
            np.lib.stride_tricks.as_strided(data[offa:], shape=(c, r), strides=(lda * 8, 8))[...] = blk.T


def _share_adjoint(desc: np.ndarray, ranges: np.ndarray, half: int):
    """Point every block of adjoint term t+half at the storage of its partner block of base term t (same offset and
    ld, flagged transposed).  Returns (new descriptors, transposed flags, arena length that is still needed)."""
    desc = desc.copy()
    trans = np.zeros(desc.shape[0], np.uint8)
    for t in range(half):
        lo, hi = ranges[t]
        alo, ahi = ranges[t + half]
        base = {(int(desc[i]["row"]), int(desc[i]["col"])): i for i in range(lo, hi)}
        for j in range(alo, ahi):
            i = base[(int(desc[j]["col"]), int(desc[j]["row"]))]
            desc[j]["offset"] = desc[i]["offset"]
            desc[j]["ld"] = desc[i]["ld"]
            trans[j] = 1
    return desc, trans


def make_problem(name: str, seed: Optional[int] = None, fill: bool = True, pad_even: bool = True,
                 n_terms: Optional[int] = None, base_terms=None, row_align: Optional[int] = None,
                 share_adjoint: bool = False, D: Optional[int] = None) -> Problem:
    """Build config ``name`` (seed defaults to the config index).  ``fill=False`` returns descriptors only
    (arenas can then be streamed with ``fill_term``).  ``n_terms`` overrides the term count (tests).
    ``base_terms`` (indices into the T/2 base terms) keeps only those terms and their adjoints, with the same
    coefficients, shifts and entries they have in the full config (term shards for multi-GPU runs, bounded
    samples for the timed CPU baseline); arenas are compacted to the kept terms.  ``D`` overrides the total bond
    dimension per side of a Gaussian / Pareto config (sweeps over D as in PAPER.md Fig. 1-2; not one of the five configs)."""
    par = _PARAMS[name]
    seed = par["index"] if seed is None else seed
    q_left, q_right, d_left, d_right, target, partner = _sector_tables(name, seed, D)
    T = par["n_terms"] if n_terms is None else n_terms
    assert T % 2 == 0
    rng = np.random.default_rng([seed, 202])
    half = T // 2
    pick = rng.integers(0, len(SHIFTS), size=half)
    base_shift = np.array([SHIFTS[i] for i in pick], np.int32).reshape(half, 2)
    shifts = np.concatenate([base_shift, -base_shift], axis=0)
    c = rng.standard_normal(half)
    ids = None
    if base_terms is not None:
        ids = np.asarray(base_terms, np.int64)
        assert ids.ndim == 1 and (ids.size == 0 or (ids.min() >= 0 and ids.max() < half))
        base_shift = base_shift[ids].reshape(-1, 2)
        shifts = np.concatenate([base_shift, -base_shift], axis=0)
        c = c[ids]
        half = ids.size
    coef = np.concatenate([c, c])
    if row_align is None:
        row_align = 4 if pad_even else 1
    a_desc, b_desc, a_len, b_len, ta, tb = _build_descriptors(q_left, q_right, d_left, d_right, shifts, row_align)
    a_trans = b_trans = None
    if share_adjoint:
        # the arenas are term-major with the base terms first: keep that prefix, drop the materialised adjoint copies
        if half > 0 and ta[half, 0] < a_desc.shape[0]:
            a_len = int(a_desc["offset"][ta[half, 0]])
        if half > 0 and tb[half, 0] < b_desc.shape[0]:
            b_len = int(b_desc["offset"][tb[half, 0]])
        a_desc, a_trans = _share_adjoint(a_desc, ta, half)
        b_desc, b_trans = _share_adjoint(b_desc, tb, half)
    p = Problem(name=name, seed=seed, q_left=q_left, q_right=q_right, d_left=d_left, d_right=d_right,
                target=target, coef=coef, a_desc=a_desc, b_desc=b_desc, a_len=int(a_len), b_len=int(b_len),
                shifts=shifts, partner=partner, term_a_range=ta, term_b_range=tb, entry_seed=(seed, 303),
                base_term_ids=ids, a_trans=a_trans, b_trans=b_trans)
    if fill:
        p.a_data = np.zeros(max(p.a_len, 1), np.float64)
        p.b_data = np.zeros(max(p.b_len, 1), np.float64)
        for t in range(half):
            fill_term(p, t, p.a_data, p.b_data)
    return p


def make_shard(name: str, shard_of_term, shard_index: int, seed: Optional[int] = None, fill: bool = True,
               share_adjoint: bool = False, D: Optional[int] = None) -> Problem:
    """One rank's part of config ``name`` under a term partition (``shard_of_term[t] == shard_index`` keeps term t), in
    the term numbering of the FULL config: the sector table, the coefficients and the descriptor tables are the full
    config's, but the arenas hold the kept terms only (their blocks moved up, same alignment) and the descriptors of
    every other term get offset -1 - they must not be read, which is what hpsi_plan_ex with the same ``shard_of_term``
    promises.  A base term and its adjoint must be kept together (their entries are drawn together)."""
    p = make_problem(name, seed=seed, fill=False, share_adjoint=share_adjoint, D=D)
    half = p.n_terms // 2
    keep = np.asarray(shard_of_term) == shard_index
    assert keep.shape == (p.n_terms,) and np.array_equal(keep[:half], keep[half:]), "adjoint pairs must stay together"
    for side in ("a", "b"):
        desc = (p.a_desc if side == "a" else p.b_desc).copy()
        rng_tab = p.term_a_range if side == "a" else p.term_b_range
        total = p.a_len if side == "a" else p.b_len
        n_own = half if share_adjoint else p.n_terms             # terms that own storage (term-major arena)
        starts = [int(desc["offset"][rng_tab[t, 0]]) if rng_tab[t, 0] < rng_tab[t, 1] else None for t in range(n_own)]
        ends, nxt = [0] * n_own, total                            # a term's range ends where the next non-empty one starts
        for t in range(n_own - 1, -1, -1):
            ends[t] = nxt
            if starts[t] is not None:
                nxt = starts[t]
        shift, run = np.zeros(p.n_terms, np.int64), 0
        for t in range(n_own):
            if keep[t] and starts[t] is not None:
                shift[t] = starts[t] - run
                run += ends[t] - starts[t]
        if share_adjoint:
            shift[half:] = shift[:half]
        for t in range(p.n_terms):
            lo, hi = rng_tab[t]
            if keep[t]:
                desc["offset"][lo:hi] -= shift[t]
            else:
                desc["offset"][lo:hi] = -1
        if side == "a":
            p.a_desc, p.a_len = desc, int(run)
        else:
            p.b_desc, p.b_len = desc, int(run)
    if fill:
        p.a_data = np.zeros(max(p.a_len, 1), np.float64)
        p.b_data = np.zeros(max(p.b_len, 1), np.float64)
        for t in range(half):
            if keep[t]:
                fill_term(p, t, p.a_data, p.b_data)
    return p


def term_chunk(full: Problem, lo: int, hi: int, D: Optional[int] = None):
    """Base terms [lo, hi) of config ``full.name`` and their adjoints as a filled sub-problem, plus where its arenas sit in
    the arenas of the full config: ``full`` = make_problem(name, fill=False) (descriptors only), the result is
    (sub, [(side, src_lo, src_hi, dst_lo), ...]) with sub = make_problem(name, base_terms=arange(lo, hi)).  Lets a caller
    fill device arenas of the D = 8192 config (80 GB) without ever holding them on the host, and lets the oracle stream
    the same terms (oracle.apply_samples accumulates over disjoint term subsets)."""
    assert full.a_trans is None, "chunks are cut from the fully materialised layout"
    half = full.n_terms // 2
    sub = make_problem(full.name, seed=full.seed, base_terms=np.arange(lo, hi), D=D)
    n = hi - lo
    place = []
    for side, fdesc, frng, ftot, sdesc, srng, stot in (("a", full.a_desc, full.term_a_range, full.a_len, sub.a_desc, sub.term_a_range, sub.a_len),
                                                       ("b", full.b_desc, full.term_b_range, full.b_len, sub.b_desc, sub.term_b_range, sub.b_len)):
        def start(desc, rng_tab, total, t):           # arena offset where term t's range starts (term-major arenas)
            while t < rng_tab.shape[0] and rng_tab[t, 0] == rng_tab[t, 1]:
                t += 1
            return int(desc["offset"][rng_tab[t, 0]]) if t < rng_tab.shape[0] else int(total)
        for part, (f0, f1, s0, s1) in enumerate(((lo, hi, 0, n), (half + lo, half + hi, n, 2 * n))):
            src_lo, src_hi = start(sdesc, srng, stot, s0), start(sdesc, srng, stot, s1)
            dst_lo = start(fdesc, frng, ftot, f0)
            # same blocks, same relative layout
            a0, a1 = srng[s0, 0], srng[s1 - 1, 1]
            b0 = frng[f0, 0]
            assert np.array_equal(sdesc["offset"][a0:a1] - src_lo, fdesc["offset"][b0:b0 + (a1 - a0)] - dst_lo)
            assert np.array_equal(sdesc["ld"][a0:a1], fdesc["ld"][b0:b0 + (a1 - a0)])
            place.append((side, src_lo, src_hi, dst_lo))
    return sub, place


def make_psi(p: Problem, k: int = 0) -> np.ndarray:
    """k-th seeded wavefunction for problem p: N(0,1) entries on the psi blocks, global 2-norm 1 (A11, A17)."""
    rng = np.random.default_rng([p.seed, 404, k])
    v = rng.standard_normal(p.psi_len)
    return v / np.linalg.norm(v)


def custom_problem(q_left, d_left, q_right, d_right, target, terms, pad_even: bool = False,
                   name: str = "custom") -> Problem:
    """Assemble a Problem from explicit blocks (unit tests, Hubbard pins).

    ``terms`` is a list of (c, a_blocks, b_blocks) with a_blocks = {(row_sector, col_sector): 2-D array}."""
    q_left = np.asarray(q_left, np.int32).reshape(-1, 2)
    q_right = np.asarray(q_right, np.int32).reshape(-1, 2)
    d_left = np.asarray(d_left, np.int32)
    d_right = np.asarray(d_right, np.int32)
    target = np.asarray(target, np.int32)
    a_rows, b_rows, a_chunks, b_chunks = [], [], [], []
    a_off = b_off = 0
    ta, tb = [], []
    for t, (c, ab, bb) in enumerate(terms):
        lo = len(a_rows)
        for (r, cc), arr in ab.items():
            arr = np.asarray(arr, np.float64)
            assert arr.shape == (d_left[r], d_left[cc]), (arr.shape, r, cc)
            ld = _round_up(arr.shape[1], 2) if pad_even else arr.shape[1]
            buf = np.zeros((arr.shape[0], ld))
            buf[:, :arr.shape[1]] = arr
            a_rows.append((t, r, cc, ld, a_off))
            a_chunks.append(buf.ravel())
            a_off += buf.size
        ta.append((lo, len(a_rows)))
        lo = len(b_rows)
        for (r, cc), arr in bb.items():
            arr = np.asarray(arr, np.float64)
            assert arr.shape == (d_right[r], d_right[cc]), (arr.shape, r, cc)
            ld = _round_up(arr.shape[1], 2) if pad_even else arr.shape[1]
            buf = np.zeros((arr.shape[0], ld))
            buf[:, :arr.shape[1]] = arr
            b_rows.append((t, r, cc, ld, b_off))
            b_chunks.append(buf.ravel())
            b_off += buf.size
        tb.append((lo, len(b_rows)))
    li = _label_index(q_left)
    ri = _label_index(q_right)
    partner = np.full(q_left.shape[0], -1, np.int32)
    for i, (a, b) in enumerate(q_left):
        j = ri.get((int(target[0]) - int(a), int(target[1]) - int(b)))
        if j is not None:
            partner[i] = j
    del li
    return Problem(
        name=name, seed=-1, q_left=q_left, q_right=q_right, d_left=d_left, d_right=d_right, target=target,
        coef=np.array([c for c, _, _ in terms], np.float64),
        a_desc=np.array(a_rows, dtype=OPBLOCK_DTYPE) if a_rows else np.zeros(0, OPBLOCK_DTYPE),
        b_desc=np.array(b_rows, dtype=OPBLOCK_DTYPE) if b_rows else np.zeros(0, OPBLOCK_DTYPE),
        a_len=int(a_off), b_len=int(b_off),
        a_data=np.concatenate(a_chunks) if a_chunks else np.zeros(1),
        b_data=np.concatenate(b_chunks) if b_chunks else np.zeros(1),
        partner=partner, term_a_range=np.array(ta, np.int64).reshape(-1, 2),
        term_b_range=np.array(tb, np.int64).reshape(-1, 2))
