"""Thin ctypes binding of ``liblp_b200.so`` (include/lp_collectives.h): same names, argument marshalling only.

Device buffers are ``torch`` CUDA tensors (float32, contiguous); ``stream`` is a ``torch.cuda.Stream`` (default:
the current stream).  PyTorch only owns memory and streams -- every step of the path runs in the library's
kernels.  There is NO fallback: a missing library or a non-zero status raises.
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

# enums of include/lp_collectives.h
LP_OK, LP_ERR_INVALID_ARG, LP_ERR_UNSUPPORTED, LP_ERR_CUDA = 0, 1, 2, 3
LP_MAX_P = 32
OP_BROADCAST, OP_REDUCE, OP_ALLREDUCE, OP_BSP_SGD, OP_BSP_SGD_MOM = 0, 1, 2, 3, 4
VARIANT_PIPELINE, VARIANT_DIRECT, VARIANT_CLUSTER, VARIANT_COPY_ENGINE, VARIANT_AUTO = 0, 1, 2, 3, 4
MODEL_STAGE, MODEL_LINK, MODEL_LINK_RING = 0, 1, 2
TUNE_TILE_ELEMS, TUNE_STAGES, TUNE_OUT_STAGES, TUNE_CTAS_PER_SM, TUNE_CE_STREAMS, TUNE_L2_HINT, TUNE_STORE_WAIT, \
    TUNE_SCHED, TUNE_GRID_LIMIT, TUNE_NO_PDL, TUNE_GRANULE_DIV, TUNE_CLAIM_SLOTS, TUNE_PREFETCH, \
    TUNE_CLUSTER_TILE, TUNE_CHAIN, TUNE_DIRECT_OCC = range(16)
TUNE_COUNT = 16
REDUCE_SUM, REDUCE_PROD = 0, 1
DT_F32, DT_F16, DT_BF16, DT_F64 = 0, 1, 2, 3
DEFAULT_BLOCK = 65536
VARIANT_NAMES = {0: "pipeline", 1: "direct", 2: "cluster", 3: "copy_engine"}


class LpError(RuntimeError):
    def __init__(self, status, what):
        self.status = status
        super().__init__(f"{what}: status {status} ({status_string(status)})")


class PlanInfo(ctypes.Structure):
    _fields_ = [("nb", ctypes.c_uint64), ("n_tiles", ctypes.c_uint64), ("tile_elems", ctypes.c_uint32),
                ("grid", ctypes.c_uint32), ("threads", ctypes.c_uint32), ("smem_bytes", ctypes.c_uint32),
                ("stages", ctypes.c_uint32), ("out_stages", ctypes.c_uint32), ("variant", ctypes.c_uint32),
                ("sm_count", ctypes.c_uint32), ("block", ctypes.c_uint64), ("granule_elems", ctypes.c_uint32),
                ("claim_granules", ctypes.c_uint32)]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


class ChainRole(ctypes.Structure):
    _fields_ = [(k, ctypes.c_int) for k in ("position", "up", "down", "f_active", "f_load", "f_recv", "f_send_up", "f_store",
                                            "f_send_down", "f_update", "r_active", "r_store", "r_send_down")]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


class PlanDesc(ctypes.Structure):
    _fields_ = [("op", ctypes.c_int), ("reduce_op", ctypes.c_int), ("P", ctypes.c_int), ("root", ctypes.c_int),
                ("n", ctypes.c_size_t), ("block", ctypes.c_size_t), ("variant", ctypes.c_int),
                ("tuning", ctypes.c_int * 16), ("dtype", ctypes.c_int)]


_lib = None


def lib() -> ctypes.CDLL:
    """Load liblp_b200.so (building it in-tree with nvcc if sources are newer). Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    so = _build.SO
    if _build.needs_build():
        if os.path.exists(_build.NVCC):
            so = _build.build()
        elif not os.path.exists(so):
            raise RuntimeError("liblp_b200.so is missing and nvcc is not available: the CUDA library is the "
                               "product, there is no fallback")
    L = ctypes.CDLL(so)
    pp = ctypes.POINTER(ctypes.c_void_p)
    sz, i32, u64, f32, vp = ctypes.c_size_t, ctypes.c_int, ctypes.c_uint64, ctypes.c_float, ctypes.c_void_p
    L.lp_broadcast.argtypes = [pp, i32, sz, sz, i32, vp]
    L.lp_reduce.argtypes = [pp, i32, sz, sz, i32, vp]
    L.lp_allreduce.argtypes = [pp, i32, sz, sz, vp]
    L.lp_bsp_sgd_step.argtypes = [pp, pp, i32, sz, sz, i32, f32, vp]
    psz = ctypes.POINTER(sz)
    L.lp_broadcast_segments.argtypes = [pp, i32, sz, psz, psz, i32, sz, i32, vp]
    L.lp_reduce_segments.argtypes = [pp, i32, sz, psz, psz, i32, sz, i32, vp]
    L.lp_allreduce_segments.argtypes = [pp, i32, sz, psz, psz, i32, sz, vp]
    L.lp_bsp_sgd_step_segments.argtypes = [pp, pp, i32, sz, psz, psz, i32, sz, i32, f32, vp]
    L.lp_comm_create.argtypes = [ctypes.POINTER(vp)]
    L.lp_comm_destroy.argtypes = [vp]
    L.lp_comm_stream.argtypes = [vp]
    L.lp_comm_stream.restype = vp
    L.lp_comm_after.argtypes = [vp, vp]
    L.lp_comm_wait.argtypes = [vp, vp]
    L.lp_comm_test.argtypes = [vp, ctypes.POINTER(i32)]
    L.lp_bsp_sgd_momentum_step.argtypes = [pp, pp, vp, i32, sz, sz, i32, f32, f32, vp]
    L.lp_bsp_sgd_alg2_step.argtypes = [pp, pp, vp, i32, sz, sz, i32, f32, f32, vp]
    for name in ("lp_mst_broadcast", "lp_mst_reduce", "lp_be_broadcast", "lp_be_reduce"):
        getattr(L, name).argtypes = [pp, i32, sz, i32, vp]
    for name in ("lp_mst_allreduce", "lp_be_allreduce"):
        getattr(L, name).argtypes = [pp, i32, sz, vp]
    L.lp_stream_fence.argtypes = [vp]
    L.lp_mst_reduce_static.argtypes = [pp, i32, sz, i32, vp]
    L.lp_mst_reduce_static_max_n.argtypes = [i32]
    L.lp_mst_reduce_static_max_n.restype = sz
    L.lp_static_scratch_bytes.restype = sz
    L.lp_static_last_error.restype = ctypes.c_char_p
    L.lp_reduce_op.argtypes = [pp, i32, sz, sz, i32, i32, vp]
    L.lp_allreduce_op.argtypes = [pp, i32, sz, sz, i32, vp]
    for name in ("lp_mst_reduce_op", "lp_be_reduce_op"):
        getattr(L, name).argtypes = [pp, i32, sz, i32, i32, vp]
    for name in ("lp_mst_allreduce_op", "lp_be_allreduce_op"):
        getattr(L, name).argtypes = [pp, i32, sz, i32, vp]
    L.lp_broadcast_dt.argtypes = [pp, i32, sz, sz, i32, i32, vp]
    L.lp_reduce_dt.argtypes = [pp, i32, sz, sz, i32, i32, i32, vp]
    L.lp_allreduce_dt.argtypes = [pp, i32, sz, sz, i32, i32, vp]
    L.lp_broadcast_segments_dt.argtypes = [pp, i32, sz, psz, psz, i32, sz, i32, i32, vp]
    L.lp_reduce_segments_dt.argtypes = [pp, i32, sz, psz, psz, i32, sz, i32, i32, i32, vp]
    L.lp_allreduce_segments_dt.argtypes = [pp, i32, sz, psz, psz, i32, sz, i32, i32, vp]
    L.lp_dtype_size.argtypes = [i32]
    L.lp_dtype_size.restype = sz
    L.lp_chain_plan.argtypes = [i32, i32, i32, i32, ctypes.POINTER(ChainRole)]
    L.lp_chain_endpoint_bytes.argtypes = [i32, i32, i32]
    L.lp_chain_endpoint_bytes.restype = sz
    L.lp_chain_create.argtypes = [i32, i32, i32, i32, i32, ctypes.POINTER(vp)]
    L.lp_chain_get_handle.argtypes = [vp, ctypes.c_char_p]
    L.lp_chain_connect.argtypes = [vp, ctypes.c_char_p]
    L.lp_chain_connect_ptrs.argtypes = [vp, vp, vp]
    L.lp_chain_set_timeout.argtypes = [vp, ctypes.c_ulonglong]
    L.lp_chain_set_kernel.argtypes = [i32]
    L.lp_chain_auto_block.argtypes = [sz, i32, i32, i32]
    L.lp_chain_auto_block.restype = sz
    L.lp_chain_fitted_constants.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.lp_chain_fitted_constants.restype = None
    L.lp_chain_endpoint.argtypes = [vp]
    L.lp_chain_endpoint.restype = vp
    L.lp_chain_run.argtypes = [vp, i32, vp, sz, sz, i32, i32, vp]
    L.lp_chain_run_dt.argtypes = [vp, i32, vp, sz, sz, i32, i32, i32, vp]
    L.lp_chain_bsp_sgd_step.argtypes = [vp, vp, vp, sz, sz, f32, vp]
    L.lp_chain_emulate_dt.argtypes = [i32, pp, i32, sz, sz, i32, i32, i32, i32, i32, i32, vp]
    L.lp_chain_emulate_bsp_sgd_step.argtypes = [pp, pp, i32, sz, sz, f32, i32, i32, i32, vp]
    L.lp_chain_bsp_sgd_momentum_step.argtypes = [vp, vp, vp, vp, sz, sz, f32, f32, vp]
    L.lp_chain_emulate_bsp_sgd_momentum_step.argtypes = [pp, pp, vp, i32, sz, sz, f32, f32, i32, i32, i32, vp]
    L.lp_chain_bsp_sgd_alg2_step.argtypes = [vp, vp, vp, vp, sz, sz, i32, f32, f32, vp]
    L.lp_chain_emulate_bsp_sgd_alg2_step.argtypes = [pp, pp, vp, i32, sz, sz, i32, f32, f32, i32, i32, i32, vp]
    L.lp_chain_error.argtypes = [vp, ctypes.POINTER(i32)]
    L.lp_chain_destroy.argtypes = [vp]
    L.lp_chain_disconnect.argtypes = [vp]
    L.lp_chain_emulate.argtypes = [i32, pp, i32, sz, sz, i32, i32, i32, i32, i32, vp]
    L.lp_chain_emulate_channels.argtypes = [i32, i32]
    L.lp_chain_emulate_error.argtypes = [i32, i32, i32, i32, ctypes.POINTER(i32)]
    L.lp_plan_desc_init.argtypes = [ctypes.POINTER(PlanDesc)]
    L.lp_plan_create.argtypes = [ctypes.POINTER(PlanDesc), ctypes.POINTER(vp)]
    L.lp_plan_destroy.argtypes = [vp]
    L.lp_plan_run.argtypes = [vp, pp, pp, vp, f32, f32, vp]
    L.lp_plan_run_segments.argtypes = [vp, pp, pp, psz, psz, i32, f32, vp]
    L.lp_plan_get_info.argtypes = [vp, ctypes.POINTER(PlanInfo)]
    L.lp_hbm_probe.argtypes = [pp, i32, i32, sz, vp]
    L.lp_auto_block.argtypes = [i32, i32, sz, i32]
    L.lp_auto_block.restype = sz
    L.lp_fitted_constants.argtypes = [i32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.lp_fitted_constants.restype = None
    L.lp_allreduce_host.argtypes = [pp, i32, sz, sz]
    L.lp_bsp_sgd_step_host.argtypes = [pp, pp, i32, sz, sz, i32, f32]
    L.lp_num_blocks.argtypes = [sz, sz]
    L.lp_num_blocks.restype = u64
    L.lp_stage_block.argtypes = [i32, u64, u64, i32]
    L.lp_stage_block.restype = ctypes.c_int64
    L.lp_schedule_steps.argtypes = [i32, sz, sz, i32, i32, ctypes.POINTER(u64)]
    L.lp_mst_levels.argtypes = [i32]
    f64 = ctypes.c_double
    L.lp_cost_model.argtypes = [i32, i32, f64, f64, f64, f64, f64, f64]
    L.lp_cost_model.restype = f64
    L.lp_optimal_block.argtypes = [i32, f64, f64, f64, f64, f64]
    L.lp_optimal_block.restype = f64
    L.lp_plan_query.argtypes = [i32, i32, sz, sz, ctypes.POINTER(PlanInfo)]
    L.lp_min_bytes.argtypes = [i32, i32, sz]
    L.lp_min_bytes.restype = u64
    L.lp_set_variant.argtypes = [i32]
    L.lp_set_tuning.argtypes = [i32, i32]
    L.lp_get_tuning.argtypes = [i32]
    L.lp_launch_count.restype = u64
    L.lp_status_string.argtypes = [i32]
    L.lp_status_string.restype = ctypes.c_char_p
    _lib = L
    return L


ALGO_LP, ALGO_MST, ALGO_BE = 0, 1, 2


def lp_cost_model(algo, op, p, n_bytes, b_bytes, alpha, beta, gamma=0.0) -> float:
    return float(lib().lp_cost_model(algo, op, p, n_bytes, b_bytes, alpha, beta, gamma))


def lp_optimal_block(op, p, n_bytes, alpha, beta, gamma=0.0) -> float:
    return float(lib().lp_optimal_block(op, p, n_bytes, alpha, beta, gamma))


def lp_stream_fence(stream=None):
    """LP_TUNE_CHAIN = 1 / 3 only: other work went into `stream`; the next library launch there waits for it first."""
    _check(lib().lp_stream_fence(_stream_ptr(stream)), "lp_stream_fence")


def status_string(status: int) -> str:
    return lib().lp_status_string(status).decode()


def _check(rc, what):
    if rc != LP_OK:
        raise LpError(rc, what)


class Ranks:
    """P device vectors registered once.  Caches the host array of device pointers, so a collective on them is
    one ctypes call (~2 us) instead of P tensor checks per call; accepted wherever a list of tensors is."""

    def __init__(self, bufs):
        self.bufs = list(bufs)
        self.arr, self.n = _dev_ptrs(self.bufs)

    def __len__(self):
        return len(self.bufs)

    def __iter__(self):
        return iter(self.bufs)

    def __getitem__(self, i):
        return self.bufs[i]


def _dev_ptrs(bufs):
    """Host array of device pointers from a list of CUDA float32 tensors (checks dtype / contiguity / length)."""
    if isinstance(bufs, Ranks):
        return bufs.arr, bufs.n
    import torch
    n = bufs[0].numel() if len(bufs) else 0
    for b in bufs:
        if not (isinstance(b, torch.Tensor) and b.is_cuda and b.dtype == torch.float32 and b.is_contiguous()):
            raise TypeError("buffers must be contiguous float32 CUDA tensors")
        if b.numel() != n:
            raise ValueError("all ranks must hold vectors of the same length")
    return (ctypes.c_void_p * len(bufs))(*[b.data_ptr() for b in bufs]), n


def _host_ptrs(arrs):
    """Host array of host pointers from numpy float32 arrays or CPU torch tensors (pinned for full speed)."""
    ptrs, n = [], None
    for a in arrs:
        if hasattr(a, "data_ptr"):
            if a.is_cuda or str(a.dtype) != "torch.float32" or not a.is_contiguous():
                raise TypeError("host buffers must be contiguous float32 CPU tensors / numpy arrays")
            p, m = a.data_ptr(), a.numel()
        else:
            if str(a.dtype) != "float32" or not a.flags.c_contiguous:
                raise TypeError("host buffers must be contiguous float32 CPU tensors / numpy arrays")
            p, m = a.ctypes.data, a.size
        if n is not None and m != n:
            raise ValueError("all ranks must hold vectors of the same length")
        n = m
        ptrs.append(p)
    return (ctypes.c_void_p * len(ptrs))(*ptrs), (n or 0)


def _stream_ptr(stream):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return ctypes.c_void_p(s.cuda_stream)


# ---- LP collectives ------------------------------------------------------------------------------------
def lp_broadcast(bufs, block, root=0, stream=None):
    arr, n = _dev_ptrs(bufs)
    _check(lib().lp_broadcast(arr, len(bufs), n, block, root, _stream_ptr(stream)), "lp_broadcast")


def lp_reduce(bufs, block, root=0, stream=None):
    arr, n = _dev_ptrs(bufs)
    _check(lib().lp_reduce(arr, len(bufs), n, block, root, _stream_ptr(stream)), "lp_reduce")


def lp_allreduce(bufs, block, stream=None):
    arr, n = _dev_ptrs(bufs)
    _check(lib().lp_allreduce(arr, len(bufs), n, block, _stream_ptr(stream)), "lp_allreduce")


def lp_bsp_sgd_step(grads, weights, block, root=0, lr=0.01, stream=None):
    ga, n = _dev_ptrs(grads)
    wa, nw = _dev_ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    _check(lib().lp_bsp_sgd_step(ga, wa, len(grads), n, block, root, ctypes.c_float(lr), _stream_ptr(stream)),
           "lp_bsp_sgd_step")


def lp_reduce_op(bufs, block, reduce_op, root=0, stream=None):
    arr, n = _dev_ptrs(bufs)
    _check(lib().lp_reduce_op(arr, len(bufs), n, block, root, reduce_op, _stream_ptr(stream)), "lp_reduce_op")


def lp_allreduce_op(bufs, block, reduce_op, stream=None):
    arr, n = _dev_ptrs(bufs)
    _check(lib().lp_allreduce_op(arr, len(bufs), n, block, reduce_op, _stream_ptr(stream)), "lp_allreduce_op")


# ---- element types other than fp32 (U21) ------------------------------------------------------------------
def _torch_dt():
    import torch
    return {torch.float32: DT_F32, torch.float16: DT_F16, torch.bfloat16: DT_BF16, torch.float64: DT_F64}


def _dev_ptrs_dt(bufs, dtype=None):
    """Host array of device pointers from CUDA tensors of one element type; returns (array, n, LP_DT_*).  `dtype`
    overrides the tensors' own type for tensors that only carry bit patterns (int16 / uint16 holding f16 or bf16)."""
    import torch
    n = bufs[0].numel() if len(bufs) else 0
    table = _torch_dt()
    dt = dtype
    for b in bufs:
        if not (isinstance(b, torch.Tensor) and b.is_cuda and b.is_contiguous()):
            raise TypeError("buffers must be contiguous CUDA tensors")
        if b.numel() != n:
            raise ValueError("all ranks must hold vectors of the same length")
        if dtype is None:
            if b.dtype not in table:
                raise TypeError(f"no LP element type for {b.dtype}")
            if dt is not None and table[b.dtype] != dt:
                raise TypeError("all ranks must hold the same element type")
            dt = table[b.dtype]
        elif b.element_size() != int(lib().lp_dtype_size(dtype)):
            raise TypeError("tensor element size does not match the LP element type")
    return (ctypes.c_void_p * len(bufs))(*[b.data_ptr() for b in bufs]), n, (DT_F32 if dt is None else dt)


def lp_broadcast_dt(bufs, block, root=0, dtype=None, stream=None):
    arr, n, dt = _dev_ptrs_dt(bufs, dtype)
    _check(lib().lp_broadcast_dt(arr, len(bufs), n, block, root, dt, _stream_ptr(stream)), "lp_broadcast_dt")


def lp_reduce_dt(bufs, block, root=0, dtype=None, reduce_op=REDUCE_SUM, stream=None):
    arr, n, dt = _dev_ptrs_dt(bufs, dtype)
    _check(lib().lp_reduce_dt(arr, len(bufs), n, block, root, dt, reduce_op, _stream_ptr(stream)), "lp_reduce_dt")


def lp_allreduce_dt(bufs, block, dtype=None, reduce_op=REDUCE_SUM, stream=None):
    arr, n, dt = _dev_ptrs_dt(bufs, dtype)
    _check(lib().lp_allreduce_dt(arr, len(bufs), n, block, dt, reduce_op, _stream_ptr(stream)), "lp_allreduce_dt")


def lp_dtype_size(dtype) -> int:
    return int(lib().lp_dtype_size(dtype))


# ---- the chain over real GPUs (one rank per GPU) and its one-GPU emulation ---------------------------------------
CHAIN_HANDLE_BYTES = 64
CHAIN_KERNEL_DEFAULT, CHAIN_KERNEL_REGISTER, CHAIN_KERNEL_TMA = 0, 1, 2


def lp_chain_auto_block(n, P, channels=0, tile=0) -> int:
    return int(lib().lp_chain_auto_block(n, P, channels, tile))


def lp_chain_fitted_constants():
    a, b = ctypes.c_double(0), ctypes.c_double(0)
    lib().lp_chain_fitted_constants(ctypes.byref(a), ctypes.byref(b))
    return a.value, b.value


def lp_chain_set_kernel(kernel):
    _check(lib().lp_chain_set_kernel(kernel), "lp_chain_set_kernel")



def lp_chain_plan(op, P, root, rank) -> dict:
    """Host only: what `rank` does in collective `op` over P ranks (ring neighbours, forward / return steps)."""
    role = ChainRole()
    _check(lib().lp_chain_plan(op, P, root, rank, ctypes.byref(role)), "lp_chain_plan")
    return role.as_dict()


def lp_chain_emulate(op, bufs, block=0, root=0, reduce_op=REDUCE_SUM, channels=0, slots=0, tile=0, stream=None):
    """All P ranks of the multi-GPU chain on this GPU in one cooperative launch (the same per-rank device code)."""
    arr, n = _dev_ptrs(bufs)
    _check(lib().lp_chain_emulate(op, arr, len(bufs), n, block, root, reduce_op, channels, slots, tile, _stream_ptr(stream)),
           "lp_chain_emulate")


def lp_chain_emulate_dt(op, bufs, block=0, root=0, dtype=None, reduce_op=REDUCE_SUM, channels=0, slots=0, tile=0, stream=None):
    arr, n, dt = _dev_ptrs_dt(bufs, dtype)
    _check(lib().lp_chain_emulate_dt(op, arr, len(bufs), n, block, root, dt, reduce_op, channels, slots, tile,
                                     _stream_ptr(stream)), "lp_chain_emulate_dt")


def lp_chain_emulate_bsp_sgd_step(grads, weights, block=0, lr=0.01, channels=0, slots=0, tile=0, stream=None):
    """Alg. 3's step over the emulated chain; equals lp_bsp_sgd_step with root = P - 1."""
    ga, n = _dev_ptrs(grads)
    wa, nw = _dev_ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    _check(lib().lp_chain_emulate_bsp_sgd_step(ga, wa, len(grads), n, block, ctypes.c_float(lr), channels, slots, tile,
                                               _stream_ptr(stream)), "lp_chain_emulate_bsp_sgd_step")


def lp_chain_emulate_bsp_sgd_momentum_step(grads, weights, velocity, block=0, lr=0.01, mu=0.9, channels=0, slots=0, tile=0,
                                           stream=None):
    """Alg. 3's step with momentum over the emulated chain; equals lp_bsp_sgd_momentum_step with root = P - 1."""
    ga, n = _dev_ptrs(grads)
    wa, nw = _dev_ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    _check(lib().lp_chain_emulate_bsp_sgd_momentum_step(ga, wa, _velocity_ptr(velocity, n), len(grads), n, block,
                                                        ctypes.c_float(lr), ctypes.c_float(mu), channels, slots, tile,
                                                        _stream_ptr(stream)), "lp_chain_emulate_bsp_sgd_momentum_step")


def lp_chain_emulate_bsp_sgd_alg2_step(grads, weights, velocity=None, block=0, root=0, lr=0.01, mu=0.0, channels=0, slots=0,
                                       tile=0, stream=None):
    """Alg. 2 over the emulated chain: reduce to root, root update, broadcast."""
    ga, n = _dev_ptrs(grads)
    wa, nw = _dev_ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    _check(lib().lp_chain_emulate_bsp_sgd_alg2_step(ga, wa, _velocity_ptr(velocity, n), len(grads), n, block, root,
                                                    ctypes.c_float(lr), ctypes.c_float(mu), channels, slots, tile,
                                                    _stream_ptr(stream)), "lp_chain_emulate_bsp_sgd_alg2_step")


def lp_chain_emulate_error(P, channels=0, slots=0, tile=0) -> int:
    e = ctypes.c_int(0)
    _check(lib().lp_chain_emulate_error(P, channels, slots, tile, ctypes.byref(e)), "lp_chain_emulate_error")
    return int(e.value)


def lp_chain_emulate_channels(P, tile=0) -> int:
    return int(lib().lp_chain_emulate_channels(P, tile))


class Chain:
    """One rank's endpoint of the chain over real GPUs (lp_chain_*): create on the rank's device, exchange `handle()`
    with all ranks (any transport; chain.py uses torch.distributed), `connect(handles)`, then `run(op, buf, ...)`."""

    def __init__(self, rank, P, channels=0, slots=0, tile=0):
        h = ctypes.c_void_p()
        _check(lib().lp_chain_create(rank, P, channels, slots, tile, ctypes.byref(h)), "lp_chain_create")
        self.h, self.rank, self.P = h, rank, P

    def handle(self) -> bytes:
        buf = ctypes.create_string_buffer(CHAIN_HANDLE_BYTES)
        _check(lib().lp_chain_get_handle(self.h, buf), "lp_chain_get_handle")
        return buf.raw

    def endpoint(self) -> int:
        return int(lib().lp_chain_endpoint(self.h) or 0)

    def set_timeout(self, polls: int):
        _check(lib().lp_chain_set_timeout(self.h, polls), "lp_chain_set_timeout")

    def connect(self, handles):
        blob = b"".join(handles)
        if len(blob) != self.P * CHAIN_HANDLE_BYTES:
            raise ValueError("need one handle per rank, in rank order")
        _check(lib().lp_chain_connect(self.h, blob), "lp_chain_connect")

    def connect_ptrs(self, up_endpoint, down_endpoint):
        _check(lib().lp_chain_connect_ptrs(self.h, ctypes.c_void_p(up_endpoint), ctypes.c_void_p(down_endpoint)),
               "lp_chain_connect_ptrs")

    def run(self, op, buf, block=0, root=0, reduce_op=REDUCE_SUM, stream=None):
        import torch
        if not (isinstance(buf, torch.Tensor) and buf.is_cuda and buf.dtype == torch.float32 and buf.is_contiguous()):
            raise TypeError("buf must be a contiguous float32 CUDA tensor")
        _check(lib().lp_chain_run(self.h, op, ctypes.c_void_p(buf.data_ptr()), buf.numel(), block, root, reduce_op,
                                  _stream_ptr(stream)), "lp_chain_run")

    def run_dt(self, op, buf, block=0, root=0, reduce_op=REDUCE_SUM, dtype=None, stream=None):
        _, n, dt = _dev_ptrs_dt([buf], dtype)
        _check(lib().lp_chain_run_dt(self.h, op, ctypes.c_void_p(buf.data_ptr()), n, block, root, dt, reduce_op,
                                     _stream_ptr(stream)), "lp_chain_run_dt")

    def bsp_sgd_step(self, grad, weight, block=0, lr=0.01, stream=None):
        import torch
        for t in (grad, weight):
            if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
                raise TypeError("grad and weight must be contiguous float32 CUDA tensors")
        if grad.numel() != weight.numel():
            raise ValueError("grad and weight must have the same length")
        _check(lib().lp_chain_bsp_sgd_step(self.h, ctypes.c_void_p(grad.data_ptr()), ctypes.c_void_p(weight.data_ptr()),
                                           grad.numel(), block, ctypes.c_float(lr), _stream_ptr(stream)),
               "lp_chain_bsp_sgd_step")

    def bsp_sgd_momentum_step(self, grad, weight, velocity=None, block=0, lr=0.01, mu=0.9, stream=None):
        """`velocity`: the last rank's vector (the update is computed there); None on every other rank."""
        vp_ = ctypes.c_void_p(velocity.data_ptr()) if velocity is not None else None
        _check(lib().lp_chain_bsp_sgd_momentum_step(self.h, ctypes.c_void_p(grad.data_ptr()), ctypes.c_void_p(weight.data_ptr()),
                                                    vp_, grad.numel(), block, ctypes.c_float(lr), ctypes.c_float(mu),
                                                    _stream_ptr(stream)), "lp_chain_bsp_sgd_momentum_step")

    def bsp_sgd_alg2_step(self, grad, weight, velocity=None, block=0, root=0, lr=0.01, mu=0.0, stream=None):
        vp_ = ctypes.c_void_p(velocity.data_ptr()) if velocity is not None else None
        _check(lib().lp_chain_bsp_sgd_alg2_step(self.h, ctypes.c_void_p(grad.data_ptr()), ctypes.c_void_p(weight.data_ptr()), vp_,
                                                grad.numel(), block, root, ctypes.c_float(lr), ctypes.c_float(mu),
                                                _stream_ptr(stream)), "lp_chain_bsp_sgd_alg2_step")

    def error(self) -> int:
        e = ctypes.c_int(0)
        _check(lib().lp_chain_error(self.h, ctypes.byref(e)), "lp_chain_error")
        return int(e.value)

    def disconnect(self):
        """Unmap the neighbours' endpoints (step 2 of the tear-down in lp_collectives.h); synchronises the device."""
        if self.h:
            _check(lib().lp_chain_disconnect(self.h), "lp_chain_disconnect")

    def destroy(self):
        if self.h:
            lib().lp_chain_destroy(self.h)
            self.h = None


# ---- plans: per-call settings (variant, tuning) instead of the process-wide defaults -----------------------
class Plan:
    """lp_plan handle: `Plan(op, P, n, block=0, root=0, reduce_op=REDUCE_SUM, variant=VARIANT_AUTO, tuning={key: value})`;
    `run(bufs, ...)` enqueues it on a stream.  Immutable; usable from several threads at once."""

    def __init__(self, op, P, n, block=0, root=0, reduce_op=REDUCE_SUM, variant=VARIANT_AUTO, tuning=None, dtype=DT_F32):
        d = PlanDesc()
        _check(lib().lp_plan_desc_init(ctypes.byref(d)), "lp_plan_desc_init")
        d.op, d.reduce_op, d.P, d.root, d.n, d.block, d.variant = op, reduce_op, P, root, n, block, variant
        d.dtype = dtype
        for k, v in (tuning or {}).items():
            d.tuning[k] = v
        h = ctypes.c_void_p()
        _check(lib().lp_plan_create(ctypes.byref(d), ctypes.byref(h)), "lp_plan_create")
        self.handle, self.op, self.P, self.n, self.dtype = h, op, P, n, dtype

    def _ranks(self, bufs):
        if self.dtype != DT_F32:
            arr, n, _ = _dev_ptrs_dt(bufs, self.dtype)
        else:
            arr, n = _dev_ptrs(bufs)
        if n != self.n or len(bufs) != self.P:
            raise ValueError("buffers do not match the plan's P and n")
        return arr

    def run(self, bufs, weights=None, velocity=None, lr=0.0, mu=0.0, stream=None):
        ba = self._ranks(bufs)
        wa = self._ranks(weights) if weights is not None else None
        _check(lib().lp_plan_run(self.handle, ba, wa, _velocity_ptr(velocity, self.n), ctypes.c_float(lr),
                                 ctypes.c_float(mu), _stream_ptr(stream)), "lp_plan_run")

    def run_segments(self, bufs, segments, weights=None, lr=0.0, stream=None):
        ba = self._ranks(bufs)
        wa = self._ranks(weights) if weights is not None else None
        sg = _segments(segments)
        _check(lib().lp_plan_run_segments(self.handle, ba, wa, sg.off, sg.len, sg.k, ctypes.c_float(lr),
                                          _stream_ptr(stream)), "lp_plan_run_segments")

    def info(self) -> dict:
        info = PlanInfo()
        _check(lib().lp_plan_get_info(self.handle, ctypes.byref(info)), "lp_plan_get_info")
        return info.as_dict()

    def close(self):
        if self.handle is not None:
            _check(lib().lp_plan_destroy(self.handle), "lp_plan_destroy")
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lp_hbm_probe(read_bufs, write_bufs, stream=None):
    """HBM ceiling probe: stream len(read_bufs) reads and len(write_bufs) writes of n floats each (no schedule, no fold)."""
    arr, n = _dev_ptrs(list(read_bufs) + list(write_bufs))
    _check(lib().lp_hbm_probe(arr, len(read_bufs), len(write_bufs), n, _stream_ptr(stream)), "lp_hbm_probe")


def lp_auto_block(op, P, n, variant=VARIANT_AUTO) -> int:
    return lib().lp_auto_block(op, P, n, variant)


def lp_fitted_constants(P=6):
    a, b = ctypes.c_double(0), ctypes.c_double(0)
    lib().lp_fitted_constants(P, ctypes.byref(a), ctypes.byref(b))
    return a.value, b.value


# ---- layer-wise collectives (Alg. 1): one LP message per (offset, length) slice, one launch --------------
class Segments:
    """A list of (offset, length) slices marshalled once into the two host arrays the C ABI takes."""

    def __init__(self, segments):
        self.k = len(segments)
        self.off = (ctypes.c_size_t * max(self.k, 1))(*[int(o) for o, _ in segments])
        self.len = (ctypes.c_size_t * max(self.k, 1))(*[int(l) for _, l in segments])


def _segments(segments):
    return segments if isinstance(segments, Segments) else Segments(segments)


def lp_broadcast_segments(bufs, segments, block, root=0, stream=None):
    arr, n = _dev_ptrs(bufs)
    sg = _segments(segments)
    _check(lib().lp_broadcast_segments(arr, len(bufs), n, sg.off, sg.len, sg.k, block, root, _stream_ptr(stream)),
           "lp_broadcast_segments")


def lp_reduce_segments(bufs, segments, block, root=0, stream=None):
    arr, n = _dev_ptrs(bufs)
    sg = _segments(segments)
    _check(lib().lp_reduce_segments(arr, len(bufs), n, sg.off, sg.len, sg.k, block, root, _stream_ptr(stream)),
           "lp_reduce_segments")


def lp_allreduce_segments(bufs, segments, block, stream=None):
    arr, n = _dev_ptrs(bufs)
    sg = _segments(segments)
    _check(lib().lp_allreduce_segments(arr, len(bufs), n, sg.off, sg.len, sg.k, block, _stream_ptr(stream)),
           "lp_allreduce_segments")


def lp_broadcast_segments_dt(bufs, segments, block, root=0, dtype=None, stream=None):
    arr, n, dt = _dev_ptrs_dt(bufs, dtype)
    sg = _segments(segments)
    _check(lib().lp_broadcast_segments_dt(arr, len(bufs), n, sg.off, sg.len, sg.k, block, root, dt, _stream_ptr(stream)),
           "lp_broadcast_segments_dt")


def lp_reduce_segments_dt(bufs, segments, block, root=0, dtype=None, reduce_op=REDUCE_SUM, stream=None):
    arr, n, dt = _dev_ptrs_dt(bufs, dtype)
    sg = _segments(segments)
    _check(lib().lp_reduce_segments_dt(arr, len(bufs), n, sg.off, sg.len, sg.k, block, root, dt, reduce_op,
                                       _stream_ptr(stream)), "lp_reduce_segments_dt")


def lp_allreduce_segments_dt(bufs, segments, block, dtype=None, reduce_op=REDUCE_SUM, stream=None):
    arr, n, dt = _dev_ptrs_dt(bufs, dtype)
    sg = _segments(segments)
    _check(lib().lp_allreduce_segments_dt(arr, len(bufs), n, sg.off, sg.len, sg.k, block, dt, reduce_op,
                                          _stream_ptr(stream)), "lp_allreduce_segments_dt")


# ---- lp_comm: Alg. 1's non-blocking collectives (a library-owned high-priority stream) --------------------
class Comm:
    """lp_comm handle.  `comm.stream` is a torch ExternalStream over the library's comm stream: pass it as
    `stream=` to any collective; `after(s)` / `wait(s)` tie it to a compute stream (default: the current one)."""

    def __init__(self):
        import torch
        h = ctypes.c_void_p()
        _check(lib().lp_comm_create(ctypes.byref(h)), "lp_comm_create")
        self.handle = h
        self.stream = torch.cuda.ExternalStream(lib().lp_comm_stream(h))

    def after(self, stream=None):
        _check(lib().lp_comm_after(self.handle, _stream_ptr(stream)), "lp_comm_after")

    def wait(self, stream=None):
        _check(lib().lp_comm_wait(self.handle, _stream_ptr(stream)), "lp_comm_wait")

    def test(self) -> bool:
        done = ctypes.c_int(0)
        _check(lib().lp_comm_test(self.handle, ctypes.byref(done)), "lp_comm_test")
        return bool(done.value)

    def close(self):
        if self.handle is not None:
            _check(lib().lp_comm_destroy(self.handle), "lp_comm_destroy")
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lp_bsp_sgd_step_segments(grads, weights, segments, block, root=0, lr=0.01, stream=None):
    ga, n = _dev_ptrs(grads)
    wa, nw = _dev_ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    sg = _segments(segments)
    _check(lib().lp_bsp_sgd_step_segments(ga, wa, len(grads), n, sg.off, sg.len, sg.k, block, root, ctypes.c_float(lr),
                                          _stream_ptr(stream)), "lp_bsp_sgd_step_segments")


def _velocity_ptr(velocity, n):
    if velocity is None:
        return None
    import torch
    if not (isinstance(velocity, torch.Tensor) and velocity.is_cuda and velocity.dtype == torch.float32
            and velocity.is_contiguous() and velocity.numel() == n):
        raise TypeError("velocity must be a contiguous CUDA float32 tensor of n elements")
    return ctypes.c_void_p(velocity.data_ptr())


def lp_bsp_sgd_momentum_step(grads, weights, velocity, block, root=0, lr=0.01, mu=0.9, stream=None):
    ga, n = _dev_ptrs(grads)
    wa, nw = _dev_ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    _check(lib().lp_bsp_sgd_momentum_step(ga, wa, _velocity_ptr(velocity, n), len(grads), n, block, root,
                                          ctypes.c_float(lr), ctypes.c_float(mu), _stream_ptr(stream)),
           "lp_bsp_sgd_momentum_step")


def lp_bsp_sgd_alg2_step(grads, weights, block, velocity=None, root=0, lr=0.01, mu=0.0, stream=None):
    ga, n = _dev_ptrs(grads)
    wa, nw = _dev_ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    _check(lib().lp_bsp_sgd_alg2_step(ga, wa, _velocity_ptr(velocity, n), len(grads), n, block, root,
                                      ctypes.c_float(lr), ctypes.c_float(mu), _stream_ptr(stream)),
           "lp_bsp_sgd_alg2_step")


# ---- MST / BE baselines --------------------------------------------------------------------------------
def _baseline(name, bufs, root, stream, reduce_op=None):
    arr, n = _dev_ptrs(bufs)
    f = getattr(lib(), name)
    args = [arr, len(bufs), n] + ([] if root is None else [root]) + ([] if reduce_op is None else [reduce_op])
    _check(f(*args, _stream_ptr(stream)), name)


def lp_mst_reduce_op(bufs, reduce_op, root=0, stream=None):
    _baseline("lp_mst_reduce_op", bufs, root, stream, reduce_op)


def lp_mst_allreduce_op(bufs, reduce_op, stream=None):
    _baseline("lp_mst_allreduce_op", bufs, None, stream, reduce_op)


def lp_be_reduce_op(bufs, reduce_op, root=0, stream=None):
    _baseline("lp_be_reduce_op", bufs, root, stream, reduce_op)


def lp_be_allreduce_op(bufs, reduce_op, stream=None):
    _baseline("lp_be_allreduce_op", bufs, None, stream, reduce_op)


def lp_mst_broadcast(bufs, root=0, stream=None):
    _baseline("lp_mst_broadcast", bufs, root, stream)


def lp_mst_reduce(bufs, root=0, stream=None):
    _baseline("lp_mst_reduce", bufs, root, stream)


def lp_mst_allreduce(bufs, stream=None):
    _baseline("lp_mst_allreduce", bufs, None, stream)


def lp_mst_reduce_static(bufs, root=0, stream=None):
    """lp_mst_reduce for callers that must not allocate device memory (a framework pool owns all of HBM, a loop that
    cannot take cudaFree's device-wide sync, a thread beside a global-mode stream capture): same tree, same values, the
    non-root ranks' partial sums in a fixed 16 MiB array inside the library instead of cudaMalloc'ed scratch.  Raises
    LpError (LP_ERR_UNSUPPORTED) when n exceeds lp_mst_reduce_static_max_n(P).  One call at a time per GPU: calls
    that overlap on the device share the array and race.  First call on a device: before any stream capture."""
    arr, n = _dev_ptrs(bufs)
    rc = lib().lp_mst_reduce_static(arr, len(bufs), n, root, _stream_ptr(stream))
    if rc != LP_OK:
        raise LpError(rc, "lp_mst_reduce_static: " + lib().lp_static_last_error().decode())


def lp_mst_reduce_static_max_n(P: int) -> int:
    return int(lib().lp_mst_reduce_static_max_n(P))


def lp_static_scratch_bytes() -> int:
    return int(lib().lp_static_scratch_bytes())


def lp_be_broadcast(bufs, root=0, stream=None):
    _baseline("lp_be_broadcast", bufs, root, stream)


def lp_be_reduce(bufs, root=0, stream=None):
    _baseline("lp_be_reduce", bufs, root, stream)


def lp_be_allreduce(bufs, stream=None):
    _baseline("lp_be_allreduce", bufs, None, stream)


# ---- host-buffer entry points ----------------------------------------------------------------------------
def lp_allreduce_host(host_bufs, block):
    arr, n = _host_ptrs(host_bufs)
    _check(lib().lp_allreduce_host(arr, len(host_bufs), n, block), "lp_allreduce_host")


def lp_bsp_sgd_step_host(host_grads, host_weights, block, root=0, lr=0.01):
    ga, n = _host_ptrs(host_grads)
    wa, nw = _host_ptrs(host_weights)
    if n != nw or len(host_grads) != len(host_weights):
        raise ValueError("grads and weights must match in P and n")
    _check(lib().lp_bsp_sgd_step_host(ga, wa, len(host_grads), n, block, root, ctypes.c_float(lr)),
           "lp_bsp_sgd_step_host")


# ---- schedule engine (host only) ---------------------------------------------------------------------------
def lp_num_blocks(n, block) -> int:
    return lib().lp_num_blocks(n, block)


def lp_stage_block(P, nb, t, r) -> int:
    return lib().lp_stage_block(P, nb, t, r)


def lp_schedule_steps(P, n, block, op, model=MODEL_STAGE) -> int:
    out = ctypes.c_uint64(0)
    _check(lib().lp_schedule_steps(P, n, block, op, model, ctypes.byref(out)), "lp_schedule_steps")
    return out.value


def lp_mst_levels(P) -> int:
    return lib().lp_mst_levels(P)


def lp_plan_query(op, P, n, block) -> dict:
    info = PlanInfo()
    _check(lib().lp_plan_query(op, P, n, block, ctypes.byref(info)), "lp_plan_query")
    return info.as_dict()


def lp_min_bytes(op, P, n) -> int:
    return lib().lp_min_bytes(op, P, n)


# ---- control ---------------------------------------------------------------------------------------------
def lp_set_variant(variant):
    _check(lib().lp_set_variant(variant), "lp_set_variant")


def lp_get_variant() -> int:
    return lib().lp_get_variant()


def lp_set_tuning(key, value):
    _check(lib().lp_set_tuning(key, value), "lp_set_tuning")


def lp_get_tuning(key) -> int:
    return lib().lp_get_tuning(key)


def lp_launch_count() -> int:
    return lib().lp_launch_count()


def lp_shutdown():
    _check(lib().lp_shutdown(), "lp_shutdown")


def lp_version() -> int:
    return lib().lp_version()
