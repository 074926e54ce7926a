"""Helpers shared by the GPU parity tests: upload a workloads.Problem, plan it through the C ABI, apply."""
import numpy as np


def rel_l2(x, ref):
    return float(np.linalg.norm(x - ref) / max(np.linalg.norm(ref), 1e-300))


class GpuProblem:
    """A Problem with its operator arenas resident on cuda:0 and an hpsi plan bound to them."""

    def __init__(self, p, flags=0, misalign=False):
        import torch
        import paper_2407_07411_b200 as H
        self.H, self.torch, self.p = H, torch, p
        dev = torch.device("cuda:0")
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
        self.plan = H.plan_problem(p, self.a, self.b, flags)
        self.n = H.hpsi_query(self.plan, H.HPSI_Q_PSI_LENGTH)

    def apply(self, psi: np.ndarray) -> np.ndarray:
        torch = self.torch
        x = torch.from_numpy(np.ascontiguousarray(psi, np.float64)).to("cuda:0")
        y = torch.full_like(x, float("nan"))
        self.H.hpsi_apply(self.plan, x, y, torch.cuda.current_stream())
        torch.cuda.synchronize()
        return y.cpu().numpy()

    def q(self, what):
        return self.H.hpsi_query(self.plan, what)
