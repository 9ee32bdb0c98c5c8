"""ctypes binding of the CPU oracle (oracle/lpo_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / ``--impl reference`` legs may import this module.  It
imports nothing from paper_1611_04255_b200 and the CUDA path imports nothing
from here.

All functions take a list of P contiguous float32 numpy arrays of equal length
(the P virtual ranks' vectors) and work in place, like the C functions they
call.  Citations live in lpo_oracle.c next to each function.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lpo_oracle.c")
_SO = os.path.join(_HERE, "liblpo.so")

GCC_FLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
             "-fPIC", "-shared"]

OP_BROADCAST, OP_REDUCE, OP_ALLREDUCE = 0, 1, 2
RED_SUM, RED_PROD = 0, 1  # PAPER.md:59 "summations and multiplications"
ALGO_LP, ALGO_MST, ALGO_BE = 0, 1, 2
READING_A_REVERSE, READING_B_RING = 0, 1
# element types (lpo_oracle.c section 7, U21); f16 vectors are numpy float16 arrays, bf16 vectors are numpy
# uint16 arrays of bit patterns (numpy has no bfloat16), f64 / f32 the native types
DT_F32, DT_F16, DT_BF16, DT_F64 = 0, 1, 2, 3
NP_OF_DT = {DT_F32: np.float32, DT_F16: np.float16, DT_BF16: np.uint16, DT_F64: np.float64}


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no CUDA involved). Returns the .so path."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= os.path.getmtime(_SRC)):
        return _SO
    cmd = ["gcc", *GCC_FLAGS, _SRC, "-o", _SO, "-lm"]
    subprocess.run(cmd, check=True)
    return _SO


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_SO)
        pp = ctypes.POINTER(ctypes.c_void_p)
        sz, i32, u64, f32 = ctypes.c_size_t, ctypes.c_int, ctypes.c_uint64, ctypes.c_float
        pu64 = ctypes.POINTER(u64)
        L.lpo_chain_sum.argtypes = [pp, i32, sz, ctypes.c_void_p]
        L.lpo_chain_sum.restype = None
        for name in ("lpo_broadcast", "lpo_reduce", "lpo_mst_broadcast", "lpo_mst_reduce",
                     "lpo_be_broadcast", "lpo_be_reduce"):
            getattr(L, name).argtypes = [pp, i32, sz, i32]
        for name in ("lpo_allreduce", "lpo_allreduce_omp", "lpo_mst_allreduce",
                     "lpo_be_allreduce"):
            getattr(L, name).argtypes = [pp, i32, sz]
        for name in ("lpo_bsp_sgd_step", "lpo_bsp_sgd_step_omp"):
            getattr(L, name).argtypes = [pp, pp, i32, sz, i32, f32]
        for name in ("lpo_bsp_sgd_momentum_step", "lpo_bsp_sgd_alg2_step"):
            getattr(L, name).argtypes = [pp, pp, ctypes.c_void_p, i32, sz, i32, f32, f32]
        L.lpo_collective_segments.argtypes = [i32, pp, i32, sz, ctypes.POINTER(sz), ctypes.POINTER(sz), i32, i32]
        L.lpo_bsp_sgd_step_segments.argtypes = [pp, pp, i32, sz, ctypes.POINTER(sz), ctypes.POINTER(sz), i32, i32, f32]
        L.lpo_chain_fold.argtypes = [pp, i32, sz, i32, ctypes.c_void_p]
        for name in ("lpo_reduce_op", "lpo_mst_reduce_op", "lpo_be_reduce_op"):
            getattr(L, name).argtypes = [pp, i32, sz, i32, i32]
        for name in ("lpo_allreduce_op", "lpo_mst_allreduce_op", "lpo_be_allreduce_op"):
            getattr(L, name).argtypes = [pp, i32, sz, i32]
        L.lpo_collective_segments_op.argtypes = [i32, i32, pp, i32, sz, ctypes.POINTER(sz), ctypes.POINTER(sz), i32, i32]
        L.lpo_chain_fold_dt.argtypes = [pp, i32, sz, i32, i32, ctypes.c_void_p]
        L.lpo_broadcast_dt.argtypes = [pp, i32, sz, i32, i32]
        L.lpo_reduce_dt.argtypes = [pp, i32, sz, i32, i32, i32]
        L.lpo_allreduce_dt.argtypes = [pp, i32, sz, i32, i32]
        for name in ("lpo_f16_from_f64", "lpo_bf16_from_f64"):
            getattr(L, name).argtypes = [ctypes.c_double]
            getattr(L, name).restype = ctypes.c_uint16
        for name in ("lpo_f16_to_f64", "lpo_bf16_to_f64"):
            getattr(L, name).argtypes = [ctypes.c_uint16]
            getattr(L, name).restype = ctypes.c_double
        L.lpo_lp_blocked.argtypes = [pp, i32, sz, sz, i32, i32, pu64]
        L.lpo_num_blocks.argtypes = [sz, sz]
        L.lpo_num_blocks.restype = u64
        L.lpo_stage_block.argtypes = [i32, u64, u64, i32]
        L.lpo_stage_block.restype = ctypes.c_int64
        L.lpo_stage_ticks.argtypes = [i32, u64]
        L.lpo_stage_ticks.restype = u64
        L.lpo_link_sim.argtypes = [i32, u64, i32, i32, pu64, pu64]
        L.lpo_link_sim_reduce_ready.argtypes = [i32, u64, pu64]
        L.lpo_mst_levels.argtypes = [i32]
        L.lpo_cost.argtypes = [i32, i32] + [ctypes.c_double] * 6
        L.lpo_cost.restype = ctypes.c_double
        L.lpo_num_threads.restype = i32
        _lib = L
    return _lib


def _ptrs(bufs):
    for b in bufs:
        if not (isinstance(b, np.ndarray) and b.dtype == np.float32 and b.flags.c_contiguous
                and b.flags.writeable):
            raise TypeError("oracle buffers must be writable C-contiguous float32 numpy arrays")
    n = bufs[0].size if bufs else 0
    if any(b.size != n for b in bufs):
        raise ValueError("all ranks must hold vectors of the same length")
    arr = (ctypes.c_void_p * len(bufs))(*[b.ctypes.data for b in bufs])
    return arr, n


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with status {rc}")


def chain_sum(bufs) -> np.ndarray:
    arr, n = _ptrs(bufs)
    out = np.empty(n, dtype=np.float32)
    lib().lpo_chain_sum(arr, len(bufs), n, out.ctypes.data)
    return out


def broadcast(bufs, root=0, algo=ALGO_LP):
    arr, n = _ptrs(bufs)
    f = {ALGO_LP: "lpo_broadcast", ALGO_MST: "lpo_mst_broadcast", ALGO_BE: "lpo_be_broadcast"}[algo]
    _check(getattr(lib(), f)(arr, len(bufs), n, root), f)


def reduce(bufs, root=0, algo=ALGO_LP):
    arr, n = _ptrs(bufs)
    f = {ALGO_LP: "lpo_reduce", ALGO_MST: "lpo_mst_reduce", ALGO_BE: "lpo_be_reduce"}[algo]
    _check(getattr(lib(), f)(arr, len(bufs), n, root), f)


def allreduce(bufs, algo=ALGO_LP, omp=False):
    arr, n = _ptrs(bufs)
    f = {ALGO_LP: "lpo_allreduce_omp" if omp else "lpo_allreduce",
         ALGO_MST: "lpo_mst_allreduce", ALGO_BE: "lpo_be_allreduce"}[algo]
    _check(getattr(lib(), f)(arr, len(bufs), n), f)


def chain_fold(bufs, red=RED_SUM) -> np.ndarray:
    """Left fold in rank order with the reduce operator `red`."""
    arr, n = _ptrs(bufs)
    out = np.empty(n, dtype=np.float32)
    _check(lib().lpo_chain_fold(arr, len(bufs), n, red, out.ctypes.data), "lpo_chain_fold")
    return out


def reduce_op(bufs, red, root=0, algo=ALGO_LP):
    arr, n = _ptrs(bufs)
    f = {ALGO_LP: "lpo_reduce_op", ALGO_MST: "lpo_mst_reduce_op", ALGO_BE: "lpo_be_reduce_op"}[algo]
    _check(getattr(lib(), f)(arr, len(bufs), n, root, red), f)


def allreduce_op(bufs, red, algo=ALGO_LP):
    arr, n = _ptrs(bufs)
    f = {ALGO_LP: "lpo_allreduce_op", ALGO_MST: "lpo_mst_allreduce_op", ALGO_BE: "lpo_be_allreduce_op"}[algo]
    _check(getattr(lib(), f)(arr, len(bufs), n, red), f)


def _ptrs_dt(bufs, dt):
    want = np.dtype(NP_OF_DT[dt])
    for b in bufs:
        if not (isinstance(b, np.ndarray) and b.dtype == want and b.flags.c_contiguous and b.flags.writeable):
            raise TypeError(f"oracle buffers of element type {dt} must be writable C-contiguous {want} numpy arrays")
    n = bufs[0].size if bufs else 0
    if any(b.size != n for b in bufs):
        raise ValueError("all ranks must hold vectors of the same length")
    return (ctypes.c_void_p * len(bufs))(*[b.ctypes.data for b in bufs]), n


def chain_fold_dt(bufs, dt, red=RED_SUM) -> np.ndarray:
    """Left fold in rank order, one RN operation in the element type per combine (U21)."""
    arr, n = _ptrs_dt(bufs, dt)
    out = np.empty(n, dtype=NP_OF_DT[dt])
    _check(lib().lpo_chain_fold_dt(arr, len(bufs), n, dt, red, out.ctypes.data), "lpo_chain_fold_dt")
    return out


def broadcast_dt(bufs, dt, root=0):
    arr, n = _ptrs_dt(bufs, dt)
    _check(lib().lpo_broadcast_dt(arr, len(bufs), n, dt, root), "lpo_broadcast_dt")


def reduce_dt(bufs, dt, red=RED_SUM, root=0):
    arr, n = _ptrs_dt(bufs, dt)
    _check(lib().lpo_reduce_dt(arr, len(bufs), n, dt, root, red), "lpo_reduce_dt")


def allreduce_dt(bufs, dt, red=RED_SUM):
    arr, n = _ptrs_dt(bufs, dt)
    _check(lib().lpo_allreduce_dt(arr, len(bufs), n, dt, red), "lpo_allreduce_dt")


def f16_from_f64(x: float) -> int:
    return int(lib().lpo_f16_from_f64(float(x)))


def bf16_from_f64(x: float) -> int:
    return int(lib().lpo_bf16_from_f64(float(x)))


def f16_to_f64(bits: int) -> float:
    return float(lib().lpo_f16_to_f64(int(bits)))


def bf16_to_f64(bits: int) -> float:
    return float(lib().lpo_bf16_to_f64(int(bits)))


def collective_segments_op(op, red, bufs, segments, root=0):
    """Layer-wise reduce (op 1) / allreduce (op 2) with operator `red` on every (offset, length) slice."""
    arr, n = _ptrs(bufs)
    k = len(segments)
    off = (ctypes.c_size_t * max(k, 1))(*[int(o) for o, _ in segments])
    ln = (ctypes.c_size_t * max(k, 1))(*[int(l) for _, l in segments])
    _check(lib().lpo_collective_segments_op(op, red, arr, len(bufs), n, off, ln, k, root),
           "lpo_collective_segments_op")


def bsp_sgd_step(grads, weights, root=0, lr=0.01, omp=False):
    ga, n = _ptrs(grads)
    wa, nw = _ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    f = "lpo_bsp_sgd_step_omp" if omp else "lpo_bsp_sgd_step"
    _check(getattr(lib(), f)(ga, wa, len(grads), n, root, ctypes.c_float(lr)), f)


def _velocity_ptr(velocity, n):
    if velocity is None:
        return None
    if not (isinstance(velocity, np.ndarray) and velocity.dtype == np.float32 and velocity.flags.c_contiguous
            and velocity.flags.writeable and velocity.size == n):
        raise TypeError("velocity must be a writable C-contiguous float32 numpy array of n elements")
    return ctypes.c_void_p(velocity.ctypes.data)


def bsp_sgd_momentum_step(grads, weights, velocity, root=0, lr=0.01, mu=0.9):
    """Alg. 3 step with Caffe-style momentum (reading U18); velocity is one vector of n floats."""
    ga, n = _ptrs(grads)
    wa, nw = _ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    _check(lib().lpo_bsp_sgd_momentum_step(ga, wa, _velocity_ptr(velocity, n), len(grads), n, root,
                                           ctypes.c_float(lr), ctypes.c_float(mu)), "lpo_bsp_sgd_momentum_step")


def bsp_sgd_alg2_step(grads, weights, velocity=None, root=0, lr=0.01, mu=0.0):
    """Alg. 2 step: reduce to root (grads[root] <- S), root update, broadcast; velocity None = plain SGD."""
    ga, n = _ptrs(grads)
    wa, nw = _ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    _check(lib().lpo_bsp_sgd_alg2_step(ga, wa, _velocity_ptr(velocity, n), len(grads), n, root,
                                       ctypes.c_float(lr), ctypes.c_float(mu)), "lpo_bsp_sgd_alg2_step")


def collective_segments(op, bufs, segments, root=0):
    """Layer-wise collective (Alg. 1): `op` (0 broadcast, 1 reduce, 2 allreduce) on every (offset, length) slice."""
    arr, n = _ptrs(bufs)
    k = len(segments)
    off = (ctypes.c_size_t * max(k, 1))(*[int(o) for o, _ in segments])
    ln = (ctypes.c_size_t * max(k, 1))(*[int(l) for _, l in segments])
    _check(lib().lpo_collective_segments(op, arr, len(bufs), n, off, ln, k, root), "lpo_collective_segments")


def bsp_sgd_step_segments(grads, weights, segments, root=0, lr=0.01):
    """Layer-wise fused BSP-SGD step: bsp_sgd_step on every (offset, length) slice."""
    ga, n = _ptrs(grads)
    wa, nw = _ptrs(weights)
    if n != nw or len(grads) != len(weights):
        raise ValueError("grads and weights must match in P and n")
    k = len(segments)
    off = (ctypes.c_size_t * max(k, 1))(*[int(o) for o, _ in segments])
    ln = (ctypes.c_size_t * max(k, 1))(*[int(l) for _, l in segments])
    _check(lib().lpo_bsp_sgd_step_segments(ga, wa, len(grads), n, off, ln, k, root, ctypes.c_float(lr)),
           "lpo_bsp_sgd_step_segments")


def lp_blocked(bufs, block, op, root=0) -> int:
    """Tick-by-tick LP pipeline (stage model). Returns the tick count."""
    arr, n = _ptrs(bufs)
    ticks = ctypes.c_uint64(0)
    _check(lib().lpo_lp_blocked(arr, len(bufs), n, block, root, op, ctypes.byref(ticks)),
           "lpo_lp_blocked")
    return ticks.value


def num_blocks(n, block) -> int:
    return lib().lpo_num_blocks(n, block)


def stage_block(P, nb, t, r) -> int:
    return lib().lpo_stage_block(P, nb, t, r)


def stage_ticks(P, nb) -> int:
    return lib().lpo_stage_ticks(P, nb)


def link_sim(P, nb, op, reading=READING_A_REVERSE, per_block=False):
    steps = ctypes.c_uint64(0)
    done = (ctypes.c_uint64 * max(nb, 1))()
    _check(lib().lpo_link_sim(P, nb, op, reading, ctypes.byref(steps), done), "lpo_link_sim")
    if per_block:
        return steps.value, [done[k] for k in range(nb)]
    return steps.value


def link_sim_reduce_ready(P, nb):
    done = (ctypes.c_uint64 * max(nb, 1))()
    _check(lib().lpo_link_sim_reduce_ready(P, nb, done), "lpo_link_sim_reduce_ready")
    return [done[k] for k in range(nb)]


def mst_levels(P) -> int:
    return lib().lpo_mst_levels(P)


def cost(algo, op, p, n, b, alpha, beta, gamma) -> float:
    return lib().lpo_cost(algo, op, float(p), float(n), float(b), float(alpha), float(beta),
                          float(gamma))


def num_threads() -> int:
    return lib().lpo_num_threads()
