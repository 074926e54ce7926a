"""B200-native H_eff*psi for two-site QC-DMRG (arXiv:2407.07411 hot path): C-ABI library + thin binding.

``paper_2407_07411_b200.csrc``  - host planner (C++) and sm_100a kernels (CUDA, FP64 DMMA) behind include/hpsi.h
``paper_2407_07411_b200.binding`` - ctypes marshalling with the C names (hpsi_plan, hpsi_apply, ...)
"""
from .binding import *  # noqa: F401,F403
from .binding import (HpsiError, Plan, hpsi_apply, hpsi_apply_host, hpsi_apply_profiled, hpsi_bench_fp64_pipe, hpsi_bind,  # noqa: F401
                      hpsi_davidson, hpsi_lanczos, hpsi_debug_interpret, hpsi_diagonal, hpsi_plan, hpsi_query, hpsi_set_task_coefficients, hpsi_stream_apply, hpsi_stream_create,
                      hpsi_stream_query, lib, hpsi_debug_small_eig, hpsi_set_exchange, device_tensor, hpsi_truncate, hpsi_truncate_static, hpsi_rotate_plan, hpsi_rotate_apply, hpsi_rotate_apply_profiled,
                      hpsi_rotate_query, hpsi_rotate_debug_interpret, RotatePlan,
                      plan_problem)
