"""Thin ctypes binding of include/hpsi.h: same names, argument marshalling only (every step of the path runs in
libhpsi.so's kernels).  Device buffers are passed as torch CUDA tensors (or raw integer addresses); PyTorch is used
for device memory and streams only.  There is no CPU fallback: if libhpsi.so is missing or CUDA is unavailable
the calls raise."""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

from .build import BENCH_LIB, LIB, build, build_bench

HPSI_OK, HPSI_EINVAL, HPSI_ENOMEM, HPSI_ECUDA, HPSI_ESTATE = 0, -1, -2, -3, -4
HPSI_PLAN_HOST_ONLY = 1 << 0
HPSI_PLAN_FIXED_ORDER1 = 1 << 1
HPSI_PLAN_FIXED_ORDER2 = 1 << 2
HPSI_PLAN_NO_FUSION = 1 << 3
HPSI_PLAN_FUSE_ALL = 1 << 4

(HPSI_Q_PSI_LENGTH, HPSI_Q_N_PSI_BLOCKS, HPSI_Q_PSI_BLOCKS, HPSI_Q_N_TASKS, HPSI_Q_USEFUL_FLOPS, HPSI_Q_ISSUED_FLOPS,
 HPSI_Q_OPERATOR_BYTES, HPSI_Q_WORKSPACE_BYTES, HPSI_Q_N_GROUPS, HPSI_Q_N_P1_UNITS, HPSI_Q_N_P2_UNITS,
 HPSI_Q_N_ORDER1_TASKS, HPSI_Q_LAUNCHES_PER_APPLY, HPSI_Q_ALIGNED16, HPSI_Q_INTERMEDIATE_BYTES,
 HPSI_Q_ISSUED_FLOPS_P1, HPSI_Q_TASKS, HPSI_Q_USEFUL_FLOPS_P1, HPSI_Q_CRITICAL_FLOPS, HPSI_Q_PSI_ROWS,
 HPSI_Q_ISO_CAPACITY, HPSI_Q_SVD_SWEEPS, HPSI_Q_SVD_LAUNCHES, HPSI_Q_PSI_COLS, HPSI_Q_ISO_CAPACITY_RIGHT,
 HPSI_Q_N_FUSED_UNITS, HPSI_Q_N_FUSED_TASKS, HPSI_Q_TUNING, HPSI_Q_PREFERRED_LAYOUT, HPSI_Q_N_TERMS_PLANNED,
 HPSI_Q_N_VECTORS) = range(31)
HPSI_SIDE_LEFT, HPSI_SIDE_RIGHT = 0, 1
(HPSI_RQ_OUT_LENGTH, HPSI_RQ_OUT_BLOCKS, HPSI_RQ_ISO_LENGTH, HPSI_RQ_USEFUL_FLOPS, HPSI_RQ_ALGO_BYTES,
 HPSI_RQ_WORKSPACE_BYTES, HPSI_RQ_N_UNITS_1, HPSI_RQ_N_UNITS_2, HPSI_RQ_ALIGNED16, HPSI_RQ_INTERMEDIATE_BYTES) = range(10)
OPBLOCK_DTYPE = np.dtype([("term", "<i4"), ("row", "<i4"), ("col", "<i4"), ("ld", "<i4"), ("offset", "<i8")], align=True)

PSI_BLOCK_DTYPE = np.dtype([("left", "<i4"), ("right", "<i4"), ("rows", "<i4"), ("cols", "<i4"), ("offset", "<i8")],
                           align=True)
TASK_DTYPE = np.dtype([("term", "<i4"), ("a_block", "<i4"), ("b_block", "<i4"), ("src_left", "<i4"),
                       ("dst_left", "<i4"), ("order", "<i4")], align=True)


class hpsi_sectors_t(ctypes.Structure):
    _fields_ = [("n_left", ctypes.c_int32), ("n_right", ctypes.c_int32),
                ("q_left", ctypes.c_void_p), ("q_right", ctypes.c_void_p),
                ("d_left", ctypes.c_void_p), ("d_right", ctypes.c_void_p),
                ("target", ctypes.c_int32 * 2)]


class hpsi_terms_t(ctypes.Structure):
    _fields_ = [("n_terms", ctypes.c_int32), ("coef", ctypes.c_void_p),
                ("n_a", ctypes.c_int64), ("a_blocks", ctypes.c_void_p),
                ("n_b", ctypes.c_int64), ("b_blocks", ctypes.c_void_p),
                ("a_data", ctypes.c_void_p), ("b_data", ctypes.c_void_p),
                ("a_len", ctypes.c_int64), ("b_len", ctypes.c_int64),
                ("a_transposed", ctypes.c_void_p), ("b_transposed", ctypes.c_void_p)]


class hpsi_plan_options_t(ctypes.Structure):
    _fields_ = [("struct_bytes", ctypes.c_uint32), ("shard_index", ctypes.c_int32), ("shard_of_term", ctypes.c_void_p),
                ("p1_stages_per_unit", ctypes.c_int32), ("p2_waves", ctypes.c_int32),
                ("p2_min_unit_dmma", ctypes.c_int32), ("n_vectors", ctypes.c_int32)]


class hpsi_layout_t(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("ld_multiple", "offset_multiple", "tma_ld_multiple", "tma_offset_multiple",
                                              "arena_align_bytes", "transposed_pad_rows")]


class hpsi_davidson_params_t(ctypes.Structure):
    _fields_ = [("tol", ctypes.c_double), ("max_iter", ctypes.c_int32), ("m_max", ctypes.c_int32),
                ("precondition", ctypes.c_int32)]


class hpsi_davidson_info_t(ctypes.Structure):
    _fields_ = [("n_matvec", ctypes.c_int32), ("converged", ctypes.c_int32), ("residual", ctypes.c_double)]


class HpsiError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"hpsi error {code}: {msg}")
        self.code = code


_lib = None


def lib() -> ctypes.CDLL:
    """Load libhpsi.so (building it in-tree with nvcc if it is missing or stale).  Raises if that fails."""
    global _lib
    if _lib is None:
        path = build() if not os.environ.get("HPSI_NO_BUILD") else LIB
        L = ctypes.CDLL(path)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        L.hpsi_plan.argtypes = [ctypes.POINTER(hpsi_sectors_t), ctypes.POINTER(hpsi_terms_t), ctypes.c_uint32,
                                ctypes.POINTER(vp)]
        L.hpsi_plan_ex.argtypes = [ctypes.POINTER(hpsi_sectors_t), ctypes.POINTER(hpsi_terms_t), ctypes.c_uint32,
                                   ctypes.POINTER(hpsi_plan_options_t), ctypes.POINTER(vp)]
        L.hpsi_shard_terms.argtypes = [ctypes.POINTER(hpsi_sectors_t), ctypes.POINTER(hpsi_terms_t), vp, i32, vp, vp]
        L.hpsi_layout_blocks.argtypes = [i32, vp, i64, vp, vp, ctypes.POINTER(i64)]
        L.hpsi_bind.argtypes = [vp, vp, vp]
        L.hpsi_set_task_coefficients.argtypes = [vp, vp, i64, vp]
        L.hpsi_apply.argtypes = [vp, vp, vp, vp]
        L.hpsi_apply_host.argtypes = [vp, vp, vp, vp]
        L.hpsi_apply_multi.argtypes = [vp, vp, i64, vp, i64, i32, vp]
        L.hpsi_apply_multi.restype = ctypes.c_int
        L.hpsi_debug_interpret_multi.argtypes = [vp, vp, vp, vp, vp, i32]
        L.hpsi_debug_interpret_multi.restype = ctypes.c_int
        L.hpsi_sum_shards.argtypes = [vp, i32, i64, vp, vp]
        L.hpsi_sum_shards.restype = ctypes.c_int
        L.hpsi_apply_profiled.argtypes = [vp, vp, vp, vp, ctypes.POINTER(ctypes.c_float)]
        L.hpsi_diagonal.argtypes = [vp, vp, vp]
        L.hpsi_davidson.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(hpsi_davidson_params_t),
                                    ctypes.POINTER(hpsi_davidson_info_t), vp]
        L.hpsi_lanczos.argtypes = L.hpsi_davidson.argtypes
        L.hpsi_davidson_multi.argtypes = [vp, vp, i64, i32, vp, vp, ctypes.POINTER(hpsi_davidson_params_t),
                                          ctypes.POINTER(hpsi_davidson_info_t), vp]
        L.hpsi_davidson_multi.restype = ctypes.c_int
        L.hpsi_query.argtypes = [vp, ctypes.c_int, vp, ctypes.c_size_t]
        L.hpsi_stream_create.argtypes = [ctypes.POINTER(hpsi_sectors_t), ctypes.POINTER(hpsi_terms_t), i64, ctypes.c_uint32,
                                         ctypes.POINTER(vp)]
        L.hpsi_stream_apply.argtypes = [vp, vp, vp, vp]
        L.hpsi_stream_query.argtypes = [vp, ctypes.c_int, vp, ctypes.c_size_t]
        L.hpsi_stream_destroy.argtypes = [vp]
        L.hpsi_stream_destroy.restype = None
        for name in ("hpsi_stream_create", "hpsi_stream_apply", "hpsi_stream_query"):
            getattr(L, name).restype = ctypes.c_int
        L.hpsi_destroy.argtypes = [vp]
        L.hpsi_destroy.restype = None
        L.hpsi_last_error.restype = ctypes.c_char_p
        L.hpsi_debug_interpret.argtypes = [vp, vp, vp, vp, vp]
        L.hpsi_set_exchange.argtypes = [vp, vp, vp]
        L.hpsi_set_exchange.restype = ctypes.c_int
        L.hpsi_truncate.argtypes = [vp, vp, ctypes.c_int32, ctypes.c_int32, ctypes.c_double, vp, vp, vp, vp, vp]
        L.hpsi_truncate_static.argtypes = L.hpsi_truncate.argtypes
        L.hpsi_rotate_plan.argtypes = [ctypes.c_int32, vp, vp, i64, vp, vp, i64, ctypes.c_uint32, ctypes.POINTER(vp)]
        L.hpsi_rotate_apply.argtypes = [vp, vp, vp, vp]
        L.hpsi_rotate_apply_profiled.argtypes = [vp, vp, vp, vp, ctypes.POINTER(ctypes.c_float)]
        L.hpsi_rotate_query.argtypes = [vp, ctypes.c_int, vp, ctypes.c_size_t]
        L.hpsi_rotate_debug_interpret.argtypes = [vp, vp, vp, vp]
        L.hpsi_rotate_destroy.argtypes = [vp]
        L.hpsi_rotate_destroy.restype = None
        for name in ("hpsi_truncate", "hpsi_truncate_static", "hpsi_rotate_plan", "hpsi_rotate_apply", "hpsi_rotate_apply_profiled",
                     "hpsi_rotate_query", "hpsi_rotate_debug_interpret"):
            getattr(L, name).restype = ctypes.c_int
        for name in ("hpsi_plan", "hpsi_plan_ex", "hpsi_shard_terms", "hpsi_layout_blocks", "hpsi_bind",
                     "hpsi_set_task_coefficients", "hpsi_apply", "hpsi_apply_host", "hpsi_apply_profiled", "hpsi_diagonal",
                     "hpsi_davidson", "hpsi_lanczos", "hpsi_query", "hpsi_debug_interpret"):
            getattr(L, name).restype = ctypes.c_int
        del i32, i64
        _lib = L
    return _lib


def _check(rc: int) -> None:
    if rc != HPSI_OK:
        raise HpsiError(rc, lib().hpsi_last_error().decode())


def _ptr(x) -> Optional[int]:
    """Address of a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        assert x.flags.c_contiguous
        return x.ctypes.data
    assert x.is_contiguous()
    return x.data_ptr()


def _stream(stream) -> Optional[int]:
    if stream is None:
        return None
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None


class Plan:
    """Opaque hpsi_plan_t* plus the host arrays whose lifetime the caller would otherwise have to manage."""

    def __init__(self, handle: int, keep):
        self.handle = handle
        self._keep = keep

    def __del__(self):
        if getattr(self, "handle", None):
            lib().hpsi_destroy(self.handle)
            self.handle = None


def _marshal(q_left, q_right, d_left, d_right, target, coef, a_blocks, b_blocks, a_data, b_data, a_len, b_len,
             a_transposed, b_transposed):
    """(hpsi_sectors_t, hpsi_terms_t, arrays to keep alive) from numpy / torch arguments."""
    q_left = np.ascontiguousarray(q_left, np.int32).reshape(-1, 2)
    q_right = np.ascontiguousarray(q_right, np.int32).reshape(-1, 2)
    d_left = np.ascontiguousarray(d_left, np.int32)
    d_right = np.ascontiguousarray(d_right, np.int32)
    coef = np.ascontiguousarray(coef, np.float64)
    a_blocks = np.ascontiguousarray(a_blocks)
    b_blocks = np.ascontiguousarray(b_blocks)
    assert a_blocks.dtype.itemsize == 24 and b_blocks.dtype.itemsize == 24
    sec = hpsi_sectors_t(q_left.shape[0], q_right.shape[0], q_left.ctypes.data, q_right.ctypes.data,
                         d_left.ctypes.data, d_right.ctypes.data, (ctypes.c_int32 * 2)(int(target[0]), int(target[1])))
    if a_transposed is not None:
        a_transposed = np.ascontiguousarray(a_transposed, np.uint8)
        assert a_transposed.shape[0] == a_blocks.shape[0]
    if b_transposed is not None:
        b_transposed = np.ascontiguousarray(b_transposed, np.uint8)
        assert b_transposed.shape[0] == b_blocks.shape[0]
    trm = hpsi_terms_t(coef.shape[0], coef.ctypes.data, a_blocks.shape[0], a_blocks.ctypes.data,
                       b_blocks.shape[0], b_blocks.ctypes.data, _ptr(a_data), _ptr(b_data), int(a_len), int(b_len),
                       _ptr(a_transposed), _ptr(b_transposed))
    return sec, trm, (q_left, q_right, d_left, d_right, coef, a_blocks, b_blocks, a_transposed, b_transposed)


def hpsi_plan(q_left, q_right, d_left, d_right, target, coef, a_blocks, b_blocks, a_data=None, b_data=None,
              a_len: int = 0, b_len: int = 0, flags: int = 0, a_transposed=None, b_transposed=None,
              shard_of_term=None, shard_index: int = 0, p1_stages_per_unit: int = 0, p2_waves: int = 0,
              p2_min_unit_dmma: int = 0, n_vectors: int = 0) -> Plan:
    """hpsi_plan / hpsi_plan_ex(sector table, term list).  Host arrays: numpy; a_blocks/b_blocks: numpy arrays with the
    24-byte hpsi_opblock_t layout; a_data/b_data: torch CUDA float64 tensors (or None, to hpsi_bind later).  Any of the
    keyword options of hpsi_plan_options_t (term shard, schedule knobs) routes the call through hpsi_plan_ex."""
    sec, trm, keep = _marshal(q_left, q_right, d_left, d_right, target, coef, a_blocks, b_blocks, a_data, b_data,
                              a_len, b_len, a_transposed, b_transposed)
    out = ctypes.c_void_p()
    if shard_of_term is not None or p1_stages_per_unit or p2_waves or p2_min_unit_dmma or n_vectors:
        sot = None
        if shard_of_term is not None:
            sot = np.ascontiguousarray(shard_of_term, np.int32)
            assert sot.shape[0] == trm.n_terms
        opt = hpsi_plan_options_t(ctypes.sizeof(hpsi_plan_options_t), int(shard_index), _ptr(sot),
                                  int(p1_stages_per_unit), int(p2_waves), int(p2_min_unit_dmma), int(n_vectors))
        _check(lib().hpsi_plan_ex(ctypes.byref(sec), ctypes.byref(trm), flags, ctypes.byref(opt), ctypes.byref(out)))
    else:
        _check(lib().hpsi_plan(ctypes.byref(sec), ctypes.byref(trm), flags, ctypes.byref(out)))
    pl = Plan(out.value, (a_data, b_data))
    pl.n_left, pl.n_right = sec.n_left, sec.n_right
    return pl


def hpsi_shard_terms(p, shard_count: int, bundle_of_term=None):
    """Balanced term partition of a ``workloads.Problem``-like object: (shard_of_term int32[n_terms], shard_flops
    int64[shard_count])."""
    sec, trm, keep = _marshal(p.q_left, p.q_right, p.d_left, p.d_right, p.target, p.coef, p.a_desc, p.b_desc, None, None,
                              0, 0, None, None)
    bundle = None if bundle_of_term is None else np.ascontiguousarray(bundle_of_term, np.int32)
    shard = np.zeros(max(trm.n_terms, 1), np.int32)
    fl = np.zeros(int(shard_count), np.int64)
    _check(lib().hpsi_shard_terms(ctypes.byref(sec), ctypes.byref(trm), _ptr(bundle), int(shard_count), shard.ctypes.data,
                                  fl.ctypes.data))
    return shard[:trm.n_terms], fl


def hpsi_layout_blocks(d, blocks, transposed=None):
    """Write the preferred ld / offset into a copy of the descriptors; returns (blocks, arena_len)."""
    d = np.ascontiguousarray(d, np.int32)
    blocks = np.array(blocks, copy=True)
    assert blocks.dtype.itemsize == 24
    tr = None if transposed is None else np.ascontiguousarray(transposed, np.uint8)
    n = ctypes.c_int64()
    _check(lib().hpsi_layout_blocks(d.shape[0], d.ctypes.data, blocks.shape[0], blocks.ctypes.data, _ptr(tr), ctypes.byref(n)))
    return blocks, n.value


def hpsi_bind(plan: Plan, a_data, b_data) -> None:
    _check(lib().hpsi_bind(plan.handle, _ptr(a_data), _ptr(b_data)))
    plan._keep = (a_data, b_data)


def hpsi_set_task_coefficients(plan: Plan, coef, stream=None) -> None:
    """Per-task coefficients (numpy float64, HPSI_Q_TASKS order) replacing c_term; ordered on ``stream``."""
    coef = np.ascontiguousarray(coef, np.float64)
    _check(lib().hpsi_set_task_coefficients(plan.handle, coef.ctypes.data, coef.shape[0], _stream(stream)))


def hpsi_apply(plan: Plan, psi, out, stream=None) -> None:
    """out = H psi; psi/out: torch CUDA float64 tensors of psi_length; stream: torch.cuda.Stream or None."""
    _check(lib().hpsi_apply(plan.handle, _ptr(psi), _ptr(out), _stream(stream)))


def hpsi_apply_multi(plan: Plan, psi, out, n_vectors: int, stream=None, ld_psi: int = 0, ld_out: int = 0) -> None:
    """out_v = H psi_v for v < n_vectors; psi/out: torch CUDA float64 tensors holding the vectors ld_* doubles apart
    (default: psi_length, i.e. a contiguous [n_vectors, psi_length] array)."""
    n = hpsi_query(plan, HPSI_Q_PSI_LENGTH)
    _check(lib().hpsi_apply_multi(plan.handle, _ptr(psi), int(ld_psi or n), _ptr(out), int(ld_out or n), int(n_vectors),
                                  _stream(stream)))


def hpsi_sum_shards(parts, n_parts: int, out, stream=None) -> None:
    """out = sum over r of parts[r*n:(r+1)*n] in rank order (parts: torch CUDA tensor of n_parts * n doubles)."""
    _check(lib().hpsi_sum_shards(_ptr(parts), int(n_parts), int(out.numel()), _ptr(out), _stream(stream)))


def hpsi_apply_profiled(plan: Plan, psi, out, stream=None):
    """hpsi_apply with per-kernel device times: returns [prep, first GEMM, second GEMM, reduce] in milliseconds."""
    ms = (ctypes.c_float * 4)()
    _check(lib().hpsi_apply_profiled(plan.handle, _ptr(psi), _ptr(out), _stream(stream), ms))
    return list(ms)


def hpsi_apply_host(plan: Plan, psi_host, out_host, stream=None) -> None:
    """Same through HOST buffers (numpy arrays or pinned torch CPU tensors)."""
    _check(lib().hpsi_apply_host(plan.handle, _ptr(psi_host), _ptr(out_host), _stream(stream)))


def hpsi_diagonal(plan: Plan, diag, stream=None) -> None:
    _check(lib().hpsi_diagonal(plan.handle, _ptr(diag), _stream(stream)))


def hpsi_davidson(plan: Plan, psi_inout, tol: float = 1e-8, max_iter: int = 200, m_max: int = 16,
                  precondition: bool = True, stream=None):
    """Returns (theta, info dict); psi_inout (torch CUDA tensor) is overwritten with the Ritz vector."""
    prm = hpsi_davidson_params_t(tol, max_iter, m_max, 1 if precondition else 0)
    info = hpsi_davidson_info_t()
    eig = ctypes.c_double()
    _check(lib().hpsi_davidson(plan.handle, _ptr(psi_inout), ctypes.byref(eig), ctypes.byref(prm),
                               ctypes.byref(info), _stream(stream)))
    return eig.value, {"n_matvec": info.n_matvec, "converged": bool(info.converged), "residual": info.residual}


def hpsi_davidson_multi(plan: Plan, psi_inout, n_roots: int, tol: float = 1e-8, max_iter: int = 200, m_max: int = 16,
                        precondition: bool = True, stream=None):
    """Block Davidson for the n_roots lowest eigenpairs.  psi_inout: torch CUDA float64 tensor [n_roots, psi_length]
    (start vectors in, Ritz vectors out).  Returns (theta[n_roots], info dict with per-root residuals)."""
    prm = hpsi_davidson_params_t(tol, max_iter, m_max, 1 if precondition else 0)
    info = hpsi_davidson_info_t()
    eig = np.zeros(n_roots)
    res = np.zeros(n_roots)
    assert psi_inout.dim() == 2 and psi_inout.shape[0] == n_roots and psi_inout.is_contiguous()
    _check(lib().hpsi_davidson_multi(plan.handle, _ptr(psi_inout), int(psi_inout.shape[1]), int(n_roots), eig.ctypes.data,
                                     res.ctypes.data, ctypes.byref(prm), ctypes.byref(info), _stream(stream)))
    return eig, {"n_matvec": info.n_matvec, "converged": bool(info.converged), "residual": info.residual, "residuals": res}


EXCHANGE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
                               ctypes.c_int32, ctypes.c_int64, ctypes.c_void_p)


def device_tensor(ptr: int, shape, torch_module):
    """A float64 torch view of device memory the library owns (row-major ``shape``, no copy, no allocation): what an
    exchange callback wraps its pointers in to hand them to torch.distributed."""
    class _View:
        __cuda_array_interface__ = {"shape": tuple(int(x) for x in shape), "typestr": "<f8", "data": (int(ptr), False),
                                    "version": 3, "strides": None}
    return torch_module.as_tensor(_View(), device="cuda")


def hpsi_set_exchange(plan: Plan, fn) -> None:
    """fn(v_ptr | None, w_ptr, n, n_vectors, ld, stream_ptr) is called by hpsi_davidson / hpsi_davidson_multi /
    hpsi_lanczos after every mat-vec (and once for diag(H), v_ptr None) on a term-sharded plan; it enqueues the sum over
    ranks into w.  fn = None removes the hook.  A Python exception inside fn makes the solver fail with HPSI_ESTATE; the
    exception is kept in ``plan.exchange_error``."""
    if fn is None:
        _check(lib().hpsi_set_exchange(plan.handle, None, None))
        plan._exchange_cb = None
        return
    plan.exchange_error = None

    def trampoline(_user, v, w, n, nvec, ld, stream):
        try:
            fn(v, w, int(n), int(nvec), int(ld), stream)
            return 0
        except BaseException as e:                       # never unwind through the C frames
            plan.exchange_error = e
            return 1
    cb = EXCHANGE_FN(trampoline)
    _check(lib().hpsi_set_exchange(plan.handle, ctypes.cast(cb, ctypes.c_void_p), None))
    plan._exchange_cb = cb                               # keeps the thunk alive as long as the plan


def hpsi_lanczos(plan: Plan, psi_inout, tol: float = 1e-8, max_iter: int = 200, m_max: int = 16, stream=None):
    """Restarted Lanczos; returns (theta, info dict); psi_inout (torch CUDA tensor) is overwritten with the Ritz vector."""
    prm = hpsi_davidson_params_t(tol, max_iter, m_max, 0)
    info = hpsi_davidson_info_t()
    eig = ctypes.c_double()
    _check(lib().hpsi_lanczos(plan.handle, _ptr(psi_inout), ctypes.byref(eig), ctypes.byref(prm),
                              ctypes.byref(info), _stream(stream)))
    return eig.value, {"n_matvec": info.n_matvec, "converged": bool(info.converged), "residual": info.residual}


HPSI_SQ_N_WINDOWS, HPSI_SQ_STAGING_BYTES = 100, 101


class StreamPlan:
    """Opaque hpsi_stream_t* (operators streamed from pinned host arenas) plus the host arrays it borrows."""

    def __init__(self, handle: int, keep):
        self.handle = handle
        self._keep = keep

    def __del__(self):
        if getattr(self, "handle", None):
            lib().hpsi_stream_destroy(self.handle)
            self.handle = None


def hpsi_stream_create(p, a_host, b_host, window_doubles: int, flags: int = 0) -> StreamPlan:
    """p: a ``workloads.Problem``-like object; a_host / b_host: pinned torch CPU float64 tensors holding the arenas."""
    q_left = np.ascontiguousarray(p.q_left, np.int32).reshape(-1, 2)
    q_right = np.ascontiguousarray(p.q_right, np.int32).reshape(-1, 2)
    d_left = np.ascontiguousarray(p.d_left, np.int32)
    d_right = np.ascontiguousarray(p.d_right, np.int32)
    coef = np.ascontiguousarray(p.coef, np.float64)
    a_blocks, b_blocks = np.ascontiguousarray(p.a_desc), np.ascontiguousarray(p.b_desc)
    sec = hpsi_sectors_t(q_left.shape[0], q_right.shape[0], q_left.ctypes.data, q_right.ctypes.data,
                         d_left.ctypes.data, d_right.ctypes.data, (ctypes.c_int32 * 2)(int(p.target[0]), int(p.target[1])))
    trm = hpsi_terms_t(coef.shape[0], coef.ctypes.data, a_blocks.shape[0], a_blocks.ctypes.data,
                       b_blocks.shape[0], b_blocks.ctypes.data, _ptr(a_host), _ptr(b_host), int(p.a_len), int(p.b_len),
                       None, None)
    a_tr, b_tr = getattr(p, "a_trans", None), getattr(p, "b_trans", None)
    if a_tr is not None:
        a_tr = np.ascontiguousarray(a_tr, np.uint8)
        trm.a_transposed = a_tr.ctypes.data
    if b_tr is not None:
        b_tr = np.ascontiguousarray(b_tr, np.uint8)
        trm.b_transposed = b_tr.ctypes.data
    out = ctypes.c_void_p()
    _check(lib().hpsi_stream_create(ctypes.byref(sec), ctypes.byref(trm), int(window_doubles), flags, ctypes.byref(out)))
    return StreamPlan(out.value, (a_host, b_host))


def hpsi_stream_apply(sp: StreamPlan, psi, out, stream=None) -> None:
    _check(lib().hpsi_stream_apply(sp.handle, _ptr(psi), _ptr(out), _stream(stream)))


def hpsi_stream_query(sp: StreamPlan, what: int) -> int:
    v = ctypes.c_int64()
    _check(lib().hpsi_stream_query(sp.handle, what, ctypes.addressof(v), 8))
    return v.value


def hpsi_query(plan: Plan, what: int):
    """Scalar items return int; HPSI_Q_PSI_BLOCKS / HPSI_Q_TASKS return structured numpy arrays."""
    if what == HPSI_Q_TUNING:
        arr = np.zeros(3, np.int64)
        _check(lib().hpsi_query(plan.handle, what, arr.ctypes.data, arr.nbytes))
        return [int(v) for v in arr]
    if what == HPSI_Q_PREFERRED_LAYOUT:
        lay = hpsi_layout_t()
        _check(lib().hpsi_query(plan.handle, what, ctypes.addressof(lay), ctypes.sizeof(lay)))
        return {n: getattr(lay, n) for n, _ in hpsi_layout_t._fields_}
    if what in (HPSI_Q_PSI_BLOCKS, HPSI_Q_TASKS):
        n = hpsi_query(plan, HPSI_Q_N_PSI_BLOCKS if what == HPSI_Q_PSI_BLOCKS else HPSI_Q_N_TASKS)
        arr = np.zeros(max(n, 1), PSI_BLOCK_DTYPE if what == HPSI_Q_PSI_BLOCKS else TASK_DTYPE)
        _check(lib().hpsi_query(plan.handle, what, arr.ctypes.data, arr.nbytes))
        return arr[:n]
    v = ctypes.c_int64()
    _check(lib().hpsi_query(plan.handle, what, ctypes.addressof(v), 8))
    return v.value


_bench_lib = None


def bench_lib() -> ctypes.CDLL:
    """libhpsi_bench.so (include/hpsi_bench.h): calibration probes, loaded by bench.py only."""
    global _bench_lib
    if _bench_lib is None:
        L = ctypes.CDLL(build_bench() if not os.environ.get("HPSI_NO_BUILD") else BENCH_LIB)
        L.hpsi_bench_fp64_pipe.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                           ctypes.POINTER(ctypes.c_double)]
        L.hpsi_bench_fp64_pipe.restype = ctypes.c_int
        L.hpsi_bench_last_error.restype = ctypes.c_char_p
        _bench_lib = L
    return _bench_lib


def hpsi_bench_fp64_pipe(kind: int, iters: int):
    """(milliseconds, flops) of the register-resident FP64 pipe probe (0 DMMA, 1 DFMA, 2 both)."""
    ms, fl = ctypes.c_double(), ctypes.c_double()
    rc = bench_lib().hpsi_bench_fp64_pipe(kind, iters, ctypes.byref(ms), ctypes.byref(fl))
    if rc != 0:
        raise HpsiError(rc, bench_lib().hpsi_bench_last_error().decode())
    return ms.value, fl.value


def hpsi_debug_interpret(plan: Plan, a_host: np.ndarray, b_host: np.ndarray, psi_host: np.ndarray) -> np.ndarray:
    """Run the device schedule with naive loops on the CPU (planner verification; tests only).  psi_host of shape
    [psi_length] or, for a batched plan, [n_vectors, psi_length]."""
    psi_host = np.ascontiguousarray(psi_host, np.float64)
    out = np.empty_like(psi_host)
    nvec = 1 if psi_host.ndim == 1 else psi_host.shape[0]
    _check(lib().hpsi_debug_interpret_multi(plan.handle, _ptr(np.ascontiguousarray(a_host, np.float64)),
                                            _ptr(np.ascontiguousarray(b_host, np.float64)), _ptr(psi_host), _ptr(out), nvec))
    return out


# ------------------------------------------------------------------------ site update
HPSI_TRUNCATE_STATIC_BYTES = 32 << 20


def hpsi_debug_small_eig(g: np.ndarray, k: int = 1):
    """The drivers' subspace eigensolver on one symmetric matrix: (theta[k], y[k, j], fell_back)."""
    g = np.ascontiguousarray(g, np.float64)
    j = g.shape[0]
    theta, y, fb = np.zeros(k), np.zeros((k, j)), ctypes.c_int32()
    L = lib()
    L.hpsi_debug_small_eig.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_void_p, ctypes.c_void_p,
                                       ctypes.c_void_p]
    L.hpsi_debug_small_eig.restype = ctypes.c_int
    _check(L.hpsi_debug_small_eig(g.ctypes.data, j, int(k), theta.ctypes.data, y.ctypes.data, ctypes.addressof(fb)))
    return theta, y, bool(fb.value)


def hpsi_truncate(plan: Plan, psi, chi_max: int, ot, stream=None, eps_discard: float = -1.0, side: int = 0,
                  static_scratch: bool = False):
    """SVD truncation of psi (torch CUDA tensor).  ot: torch CUDA float64 tensor of >= HPSI_Q_ISO_CAPACITY doubles that
    receives the isometries; eps_discard >= 0 keeps only as many states as the discarded weight <= eps_discard needs.
    Returns (chi int32[n_left], sigma float64[HPSI_Q_PSI_ROWS], discarded_weight).
    static_scratch=True calls hpsi_truncate_static (no device allocation; scratch limited to HPSI_TRUNCATE_STATIC_BYTES)."""
    chi = np.zeros(int(plan.n_right if side == HPSI_SIDE_RIGHT else plan.n_left), np.int32)
    n_sig = hpsi_query(plan, HPSI_Q_PSI_COLS if side == HPSI_SIDE_RIGHT else HPSI_Q_PSI_ROWS)
    sigma = np.zeros(max(n_sig, 1), np.float64)
    disc = ctypes.c_double()
    fn = lib().hpsi_truncate_static if static_scratch else lib().hpsi_truncate
    _check(fn(plan.handle, _ptr(psi), int(side), int(chi_max), float(eps_discard), _ptr(ot), chi.ctypes.data, sigma.ctypes.data,
              ctypes.addressof(disc), _stream(stream)))
    return chi, sigma[:n_sig], disc.value


def hpsi_truncate_static(plan: Plan, psi, chi_max: int, ot, stream=None, eps_discard: float = -1.0, side: int = 0):
    """hpsi_truncate with its device buffers in the library's static scratch array: allocates nothing on the device."""
    return hpsi_truncate(plan, psi, chi_max, ot, stream, eps_discard, side, static_scratch=True)


class RotatePlan:
    """Opaque hpsi_rotate_t* plus the arena it borrows."""

    def __init__(self, handle: int, keep, n_blocks: int):
        self.handle = handle
        self._keep = keep
        self.n_blocks = n_blocks

    def __del__(self):
        if getattr(self, "handle", None):
            lib().hpsi_rotate_destroy(self.handle)
            self.handle = None


def hpsi_rotate_plan(d, chi, blocks, a_data=None, a_len: int = 0, flags: int = 0) -> RotatePlan:
    """d / chi: int32 arrays per sector; blocks: numpy array with the hpsi_opblock_t layout; a_data: torch CUDA tensor."""
    d = np.ascontiguousarray(d, np.int32)
    chi = np.ascontiguousarray(chi, np.int32)
    blocks = np.ascontiguousarray(blocks)
    assert blocks.dtype.itemsize == 24 and d.shape == chi.shape
    out = ctypes.c_void_p()
    _check(lib().hpsi_rotate_plan(d.shape[0], d.ctypes.data, chi.ctypes.data, blocks.shape[0], blocks.ctypes.data,
                                  _ptr(a_data), int(a_len), flags, ctypes.byref(out)))
    return RotatePlan(out.value, a_data, blocks.shape[0])


def hpsi_rotate_apply(r: RotatePlan, ot, out, stream=None) -> None:
    _check(lib().hpsi_rotate_apply(r.handle, _ptr(ot), _ptr(out), _stream(stream)))


def hpsi_rotate_apply_profiled(r: RotatePlan, ot, out, stream=None):
    """Returns [isometry copy, first GEMM, second GEMM] device milliseconds."""
    ms = (ctypes.c_float * 3)()
    _check(lib().hpsi_rotate_apply_profiled(r.handle, _ptr(ot), _ptr(out), _stream(stream), ms))
    return list(ms)


def hpsi_rotate_query(r: RotatePlan, what: int):
    if what == HPSI_RQ_OUT_BLOCKS:
        arr = np.zeros(max(r.n_blocks, 1), OPBLOCK_DTYPE)
        _check(lib().hpsi_rotate_query(r.handle, what, arr.ctypes.data, arr.nbytes))
        return arr[:r.n_blocks]
    v = ctypes.c_int64()
    _check(lib().hpsi_rotate_query(r.handle, what, ctypes.addressof(v), 8))
    return v.value


def hpsi_rotate_debug_interpret(r: RotatePlan, a_host: np.ndarray, ot_host: np.ndarray) -> np.ndarray:
    out = np.full(hpsi_rotate_query(r, HPSI_RQ_OUT_LENGTH), np.nan)
    _check(lib().hpsi_rotate_debug_interpret(r.handle, _ptr(np.ascontiguousarray(a_host, np.float64)),
                                             _ptr(np.ascontiguousarray(ot_host, np.float64)), _ptr(out)))
    return out


def plan_problem(p, a_data=None, b_data=None, flags: int = 0, **options) -> Plan:
    """Marshal a ``workloads.Problem`` (any object with the boundary's fields) into hpsi_plan / hpsi_plan_ex."""
    return hpsi_plan(p.q_left, p.q_right, p.d_left, p.d_right, p.target, p.coef, p.a_desc, p.b_desc,
                     a_data, b_data, p.a_len, p.b_len, flags, getattr(p, "a_trans", None), getattr(p, "b_trans", None),
                     **options)
