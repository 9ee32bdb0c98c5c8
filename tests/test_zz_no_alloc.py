"""lp_mst_reduce_static: the MST reduce for callers that cannot allocate device memory.

Who that is: a process whose framework pool allocator already owns the whole GPU (a cudaMalloc made by a library then
fails although the pool has room), a step loop that cannot take the device-wide synchronisation that freeing /
regrowing library scratch causes, or a thread that runs beside a global-mode stream capture (cudaMalloc is refused for
every thread of the process while it lasts).  The regular lp_mst_reduce keeps the non-root ranks' partial sums in scratch
it cudaMallocs on demand; the static entry point keeps them in a fixed 16 MiB array that is part of the library image
(csrc/lp_static.cu) and refuses messages that do not fit.

The GPU test compares it with the existing path byte for byte -- the tolerance every parity test of this repository
uses for one summation tree -- on two calls in a row (the second call finds the first call's partial sums in the array
and has to give the right answer anyway), with different roots, and checks that the non-root buffers are left alone.
The file sorts last on purpose: under `pytest -x` a failure here must not hide any other test.  It depends on nothing
the other tests leave behind (no variant, no tuning key, no library scratch), so it passes alone and after them.
"""
import ctypes

import numpy as np
import pytest

from paper_1611_04255_b200 import binding as lp
from paper_1611_04255_b200 import inputs

torch = pytest.importorskip("torch")

MiB = 1 << 20


# ---- host side: no device needed ------------------------------------------------------------------------------------
def test_static_limits_are_the_documented_ones():
    assert lp.lp_static_scratch_bytes() == 16 * MiB
    floats = 16 * MiB // 4
    # (P - 2) // 2 working copies, each a multiple of 64 floats (256 bytes)
    assert lp.lp_mst_reduce_static_max_n(4) == floats == 4_194_304
    assert lp.lp_mst_reduce_static_max_n(8) == 1_398_080
    assert lp.lp_mst_reduce_static_max_n(16) == 599_168
    assert lp.lp_mst_reduce_static_max_n(32) == 279_616
    for P in range(4, 33):
        c = (P - 2) // 2
        m = lp.lp_mst_reduce_static_max_n(P)
        assert m % 64 == 0 and c * m * 4 <= 16 * MiB < c * (m + 64) * 4
    # P <= 3: the tree has no non-root receiver, nothing to keep
    assert lp.lp_mst_reduce_static_max_n(2) == lp.lp_mst_reduce_static_max_n(3) > 1 << 40
    assert lp.lp_mst_reduce_static_max_n(0) == 0 and lp.lp_mst_reduce_static_max_n(33) == 0


def test_static_rejects_before_touching_a_device():
    """Argument and size errors come back before any CUDA call, with a text that names the limit."""
    L = lp.lib()

    def call(ptrs, n, root=0):
        arr = (ctypes.c_void_p * len(ptrs))(*ptrs)
        return L.lp_mst_reduce_static(arr, len(ptrs), n, root, None)

    base = 0x7000_0000_0000
    far = [base + i * (1 << 32) for i in range(8)]
    too_long = lp.lp_mst_reduce_static_max_n(8) + 1
    assert call(far, too_long) == lp.LP_ERR_UNSUPPORTED
    msg = L.lp_static_last_error().decode()
    assert str(too_long) in msg and "1398080" in msg and "lp_mst_reduce" in msg
    assert call(far, 16, root=8) == lp.LP_ERR_INVALID_ARG
    assert call([base, base + 4, base + 4096, base + 8192], 16) == lp.LP_ERR_INVALID_ARG      # misaligned
    assert call([base, base + 32, base + 4096, base + 8192], 16) == lp.LP_ERR_INVALID_ARG     # overlapping
    assert call([base, 0, base + 4096, base + 8192], 16) == lp.LP_ERR_INVALID_ARG             # NULL
    assert L.lp_mst_reduce_static(None, 4, 16, 0, None) == lp.LP_ERR_INVALID_ARG
    if not torch.cuda.is_available():
        # a valid call without a device: LP_ERR_CUDA, never a CPU fallback
        assert call(far[:4], 1024) == lp.LP_ERR_CUDA
        assert "CUDA" in L.lp_static_last_error().decode()


# ---- GPU: against the existing path, two calls in a row -------------------------------------------------------------
def _up(arrs):
    return [torch.from_numpy(a).cuda() for a in arrs]


def _bytes(tensors):
    torch.cuda.synchronize()
    return [t.cpu().numpy().tobytes() for t in tensors]


def _both_paths(seed, P, n, root, oracle=None):
    src = inputs.rank_vectors(seed, P, n, "uniform")
    ref = _up(src)
    lp.lp_mst_reduce(ref, root=root)            # existing path: library scratch from cudaMalloc
    got = _up(src)
    lp.lp_mst_reduce_static(got, root=root)     # new path: the fixed array
    want, have = _bytes(ref), _bytes(got)
    for r in range(P):
        assert have[r] == want[r], (P, n, root, r)
        if r != root:
            assert have[r] == src[r].tobytes(), ("non-root buffer changed", P, n, root, r)
    if P > 1 and n > 0:
        assert have[root] != src[root].tobytes()
    if oracle is not None:                      # and against the CPU oracle's binomial tree
        host = [a.copy() for a in src]
        oracle.reduce(host, root=root, algo=oracle.ALGO_MST)
        assert [h.tobytes() for h in host] == have, (P, n, root)


@pytest.mark.gpu
def test_static_reduce_equals_existing_path_twice_in_a_row():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    torch.cuda.set_device(0)
    # first call: ragged length (head of 3 floats beyond the last 16-byte vector), two working copies
    _both_paths(11, 6, 1_000_003, root=4)
    # second call, straight after: longer message, other root, more copies -- every slot of the array that it uses
    # still holds the first call's partial sums
    _both_paths(12, 8, 1_398_080, root=1)
    # and a third, shorter than what is lying in the array
    _both_paths(13, 5, 4_099, root=0)


@pytest.mark.gpu
@pytest.mark.parametrize("P", [1, 2, 3, 4, 7, 16, 32])
def test_static_reduce_every_tree_shape(oracle, P):
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    n = min(70_001, lp.lp_mst_reduce_static_max_n(P))
    for root in sorted({0, P // 2, P - 1}):
        _both_paths(100 + P, P, n, root, oracle)


@pytest.mark.gpu
def test_static_reduce_edges_and_limit():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    keep = _up(inputs.rank_vectors(21, 4, 100, "uniform"))          # empty message: a valid no-op (n = 0 on real pointers)
    before = _bytes(keep)
    arr = (ctypes.c_void_p * 4)(*[t.data_ptr() for t in keep])
    assert lp.lib().lp_mst_reduce_static(arr, 4, 0, 2, None) == lp.LP_OK
    assert _bytes(keep) == before
    _both_paths(22, 4, 1, root=3)                                   # shorter than one vector
    _both_paths(23, 4, lp.lp_mst_reduce_static_max_n(4), root=1)    # exactly the limit: the array filled to its last byte
    dev = _up(inputs.rank_vectors(24, 4, lp.lp_mst_reduce_static_max_n(4) + 1, "uniform"))
    before = _bytes(dev)
    with pytest.raises(lp.LpError) as e:
        lp.lp_mst_reduce_static(dev, root=0)
    assert e.value.status == lp.LP_ERR_UNSUPPORTED and "4194304" in str(e.value)
    assert _bytes(dev) == before                                    # refused before anything ran
    s = torch.cuda.Stream()                                         # a caller's own stream
    src = inputs.rank_vectors(25, 8, 300_001, "uniform")
    ref, got = _up(src), _up(src)
    torch.cuda.synchronize()
    lp.lp_mst_reduce(ref, root=5, stream=s)
    lp.lp_mst_reduce_static(got, root=5, stream=s)
    s.synchronize()
    assert _bytes(got) == _bytes(ref)
