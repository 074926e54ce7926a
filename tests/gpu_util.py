"""Helpers shared by the GPU parity tests: upload a workloads.Problem, plan it through the C ABI, apply."""
import numpy as np


def rel_l2(x, ref):
    return float(np.linalg.norm(x - ref) / max(np.linalg.norm(ref), 1e-300))


class GpuProblem:
    """A Problem with its operator arenas resident on cuda:0 and an hpsi plan bound to them."""

    def __init__(self, p, flags=0, misalign=False, arenas=None, **plan_options):
        import torch
        import paper_2407_07411_b200 as H
        self.H, self.torch, self.p = H, torch, p
        dev = torch.device("cuda:0")
        if arenas is not None:        # device arenas that are already resident (several plans over one copy of the operators)
            self.a, self.b = arenas
            self.plan = H.plan_problem(p, self.a, self.b, flags, **plan_options)
            self.n = H.hpsi_query(self.plan, H.HPSI_Q_PSI_LENGTH)
            return
        if misalign:          # arena base only 8-byte aligned: forces the 8-byte staging kernels
            self._a_store = torch.empty(p.a_data.size + 1, dtype=torch.float64, device=dev)
            self._b_store = torch.empty(p.b_data.size + 1, dtype=torch.float64, device=dev)
            self.a = self._a_store[1:]
            self.b = self._b_store[1:]
            self.a.copy_(torch.from_numpy(p.a_data))
            self.b.copy_(torch.from_numpy(p.b_data))
        else:
            self.a = torch.from_numpy(p.a_data).to(dev)
            self.b = torch.from_numpy(p.b_data).to(dev)
        self.plan = H.plan_problem(p, self.a, self.b, flags, **plan_options)
        self.n = H.hpsi_query(self.plan, H.HPSI_Q_PSI_LENGTH)

    def apply_dev(self, x):
        """device tensor in, device tensor out (NaN-prefilled before the apply)"""
        torch = self.torch
        y = torch.full_like(x, float("nan"))
        self.H.hpsi_apply(self.plan, x, y, torch.cuda.current_stream())
        return y

    def apply(self, psi: np.ndarray) -> np.ndarray:
        torch = self.torch
        x = torch.from_numpy(np.ascontiguousarray(psi, np.float64)).to("cuda:0")
        y = torch.full_like(x, float("nan"))
        self.H.hpsi_apply(self.plan, x, y, torch.cuda.current_stream())
        torch.cuda.synchronize()
        return y.cpu().numpy()

    def q(self, what):
        return self.H.hpsi_query(self.plan, what)


def assert_blockwise(p, got, ref, tol=1e-12):
    """north_star's bar on the whole vector, and the same bar block by block (a wrong ragged edge in one tile of one rare
    block shape must not hide in the norm of a 600 000-element vector)."""
    assert rel_l2(got, ref) <= tol, rel_l2(got, ref)
    nref = np.linalg.norm(ref)
    for (i, j, r, c, off) in p.psi_blocks():
        d = np.linalg.norm(got[off:off + r * c] - ref[off:off + r * c])
        assert d <= 10 * tol * nref and d <= 100 * tol * max(np.linalg.norm(ref[off:off + r * c]), 1e-300), (i, j, r, c, d)


def shard_sum(H, torch, parts):
    """hpsi_sum_shards over a list of equally long device vectors (rank order)."""
    n = parts[0].numel()
    buf = torch.cat(parts)
    out = torch.full((n,), float("nan"), dtype=torch.float64, device=buf.device)
    H.hpsi_sum_shards(buf, len(parts), out, torch.cuda.current_stream())
    torch.cuda.synchronize()
    return out.cpu().numpy()


def fill_device_arenas(torch, full, chunk_terms=48, workers=6, on_chunk=None):
    """Device arenas of config ``full.name`` (``full`` = descriptors only) filled chunk by chunk through
    workloads.term_chunk, so that the host never holds more than a few chunks (the D = 8192 config is 80 GB).
    ``on_chunk(sub)`` is called with every filled sub-problem (e.g. to stream the same terms through the oracle)."""
    import concurrent.futures as cf
    import workloads
    a = torch.empty(max(full.a_len, 1), dtype=torch.float64, device="cuda:0")
    b = torch.empty(max(full.b_len, 1), dtype=torch.float64, device="cuda:0")
    half = full.n_terms // 2
    cuts = [(lo, min(half, lo + chunk_terms)) for lo in range(0, half, chunk_terms)]
    with cf.ThreadPoolExecutor(max_workers=workers) as ex:
        pending = []
        it = iter(cuts)
        for _ in range(workers):
            c = next(it, None)
            if c is not None:
                pending.append(ex.submit(workloads.term_chunk, full, c[0], c[1]))
        while pending:
            sub, place = pending.pop(0).result()
            c = next(it, None)
            if c is not None:
                pending.append(ex.submit(workloads.term_chunk, full, c[0], c[1]))
            for side, s0, s1, d0 in place:
                src = sub.a_data if side == "a" else sub.b_data
                (a if side == "a" else b)[d0:d0 + (s1 - s0)].copy_(torch.from_numpy(src[s0:s1]))
            if on_chunk is not None:
                on_chunk(sub)
            del sub
    torch.cuda.synchronize()
    return a, b


def store_randomly_transposed(p, seed, prob=0.5):
    """A copy of Problem ``p`` (materialised arenas) whose operator blocks are re-stored, each with probability ``prob``
    as its transpose (d[col] x d[row], flagged in a_trans / b_trans).  Even leading dimensions are kept when ``p`` has
    them.  The values of every block are unchanged, so the oracle's result for ``p`` is the expected one."""
    import copy
    rng = np.random.default_rng(seed)
    q = copy.copy(p)

    def restore(desc, data, d):
        even = all(int(e["ld"]) % 2 == 0 for e in desc)
        out, tr, chunks, off = desc.copy(), np.zeros(desc.shape[0], np.uint8), [], 0
        for i, e in enumerate(desc):
            r, c, ld, o = int(d[e["row"]]), int(d[e["col"]]), int(e["ld"]), int(e["offset"])
            blk = data[o:o + r * ld].reshape(r, ld)[:, :c]
            if rng.random() < prob:
                blk, tr[i] = blk.T, 1
            nld = blk.shape[1] + (blk.shape[1] % 2 if even else 0)
            buf = np.zeros((blk.shape[0], nld))
            buf[:, :blk.shape[1]] = blk
            out[i]["ld"], out[i]["offset"] = nld, off
            chunks.append(buf.ravel())
            off += buf.size
        return out, tr, (np.concatenate(chunks) if chunks else np.zeros(1)), off

    q.a_desc, q.a_trans, q.a_data, q.a_len = restore(p.a_desc, p.a_data, p.d_left)
    q.b_desc, q.b_trans, q.b_data, q.b_len = restore(p.b_desc, p.b_data, p.d_right)
    return q
