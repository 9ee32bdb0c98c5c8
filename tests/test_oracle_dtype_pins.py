"""Pins of the oracle's element-type section (oracle/lpo_oracle.c section 7, U21): f16, bf16 and f64
vectors, one round-to-nearest-even operation IN THE ELEMENT TYPE per combine, left fold in rank order.

Independent references: numpy's float16 (its own half <-> float conversions and arithmetic), torch's bfloat16 CPU
tensors (its own float <-> bfloat16 rounding), numpy float64, the textbook integer formula for RNE truncation of an
fp32 pattern to bf16, exact small-integer arithmetic, order separators built from ties, and an fp64 error bound."""
import math

import numpy as np
import pytest

from paper_1611_04255_b200 import inputs

torch = pytest.importorskip("torch")

F32, F16, BF16, F64 = inputs.DT_F32, inputs.DT_F16, inputs.DT_BF16, inputs.DT_F64
SUM, PROD = 0, 1


def bf16_bits_to_f32(bits):
    return (bits.astype(np.uint32) << 16).view(np.float32)


def bf16_bits_to_torch(bits):
    return torch.from_numpy(bits.view(np.int16).copy()).view(torch.bfloat16)


def torch_to_bf16_bits(t):
    return t.view(torch.int16).numpy().view(np.uint16)


def same_bits_or_both_nan(got, want, dt):
    """Bit equality, except that any NaN matches any NaN (payload and sign of a NaN are not part of the definition)."""
    if dt == F16:
        g, w = got.view(np.uint16), want.view(np.uint16)
        gn, wn = np.isnan(got), np.isnan(want)
    elif dt == BF16:
        g, w = got, want
        gn, wn = np.isnan(bf16_bits_to_f32(got)), np.isnan(bf16_bits_to_f32(want))
    else:
        g, w = got.view(np.uint64 if dt == F64 else np.uint32), want.view(np.uint64 if dt == F64 else np.uint32)
        gn, wn = np.isnan(got), np.isnan(want)
    return bool(np.all((g == w) | (gn & wn)))


# ---- conversions ---------------------------------------------------------------------------------------------
def test_f16_widening_and_roundtrip_exhaustive(oracle):
    bits = np.arange(1 << 16, dtype=np.uint16)
    want = bits.view(np.float16).astype(np.float64)              # numpy's own half -> double
    for b, w in zip(bits.tolist(), want.tolist()):
        v = oracle.f16_to_f64(b)
        if math.isnan(w):
            assert math.isnan(v)
            continue
        assert v == w and math.copysign(1.0, v) == math.copysign(1.0, w), b
        assert oracle.f16_from_f64(v) == b                       # every f16 value survives the round trip


def test_bf16_widening_and_roundtrip_exhaustive(oracle):
    bits = np.arange(1 << 16, dtype=np.uint16)
    want = bf16_bits_to_f32(bits).astype(np.float64)             # a bf16 is the top half of an fp32 pattern
    for b, w in zip(bits.tolist(), want.tolist()):
        v = oracle.bf16_to_f64(b)
        if math.isnan(w):
            assert math.isnan(v)
            continue
        assert v == w and math.copysign(1.0, v) == math.copysign(1.0, w), b
        assert oracle.bf16_from_f64(v) == b


def test_f16_rounding_ties_neighbours_and_random_doubles_against_numpy(oracle):
    # every midpoint between two adjacent non-negative f16 values (exact in double) must go to the even neighbour,
    # and a hair to either side of it to the nearer one; numpy's double -> half conversion is the reference
    bits = np.arange(0, 0x7c00, dtype=np.uint16)                  # 0 .. largest finite
    lo = bits.view(np.float16).astype(np.float64)
    hi = (bits + 1).astype(np.uint16).view(np.float16).astype(np.float64)
    hi[-1] = 65536.0                                              # the value after the largest finite one, were the exponent unbounded
    mid = (lo + hi) / 2
    cases = np.concatenate([mid, np.nextafter(mid, 0.0), np.nextafter(mid, np.inf), -mid])
    rng = np.random.default_rng(7)
    rnd = np.concatenate([rng.standard_normal(20000) * 10.0 ** rng.integers(-9, 6, 20000),
                          [0.0, -0.0, np.inf, -np.inf, 65504.0, 65519.999, 65520.0, 1e9, 2.0 ** -25, 2.0 ** -24 * 1.5]])
    x = np.concatenate([cases, rnd])
    with np.errstate(over="ignore"):
        want = x.astype(np.float16).view(np.uint16)
    got = np.array([oracle.f16_from_f64(v) for v in x.tolist()], dtype=np.uint16)
    assert np.array_equal(got, want)
    assert oracle.f16_from_f64(2049.0) == np.float16(2048.0).view(np.uint16)   # tie -> even (2048), by hand
    assert oracle.f16_from_f64(2051.0) == np.float16(2052.0).view(np.uint16)   # tie -> even (2052)
    assert math.isnan(np.uint16(oracle.f16_from_f64(float("nan"))).view(np.float16))


def test_bf16_rounding_against_the_integer_formula_and_torch(oracle):
    # fp32-representable inputs (so that torch's float -> bfloat16 is a single rounding): all midpoints between adjacent
    # bf16 values of a few binades, their fp32 neighbours, random fp32 values, specials
    rng = np.random.default_rng(11)
    pats = np.concatenate([
        (np.arange(0x3f00, 0x4100, dtype=np.uint32) << 16) | 0x8000,          # exact midpoints around 0.5 .. 8
        (np.arange(0x3f00, 0x4100, dtype=np.uint32) << 16) | 0x7fff,
        (np.arange(0x3f00, 0x4100, dtype=np.uint32) << 16) | 0x8001,
        (np.arange(0x0000, 0x0100, dtype=np.uint32) << 16) | 0x8000,          # subnormal bf16 range
        np.array([0x7f7f8000, 0x7f7f7fff, 0x7f7fffff, 0x00000001, 0x80000000, 0x7f800000, 0xff800000], dtype=np.uint32),
        rng.integers(0, 1 << 32, 30000, dtype=np.uint64).astype(np.uint32),
    ])
    x32 = pats.view(np.float32)
    finite = np.isfinite(x32)
    # textbook RNE truncation of an fp32 pattern to its top 16 bits
    formula = ((pats.astype(np.uint64) + 0x7fff + ((pats >> 16) & 1)) >> 16).astype(np.uint16)
    tor = torch_to_bf16_bits(torch.from_numpy(x32.copy()).to(torch.bfloat16))
    got = np.array([oracle.bf16_from_f64(float(v)) for v in x32.astype(np.float64).tolist()], dtype=np.uint16)
    nan = np.isnan(x32)
    assert np.array_equal(got[~nan], tor[~nan])
    assert np.array_equal(got[finite], formula[finite])
    assert np.all(np.isnan(bf16_bits_to_f32(got[nan])))
    assert oracle.bf16_from_f64(257.0) == 0x4380 and oracle.bf16_from_f64(259.0) == 0x4382    # ties -> even: 256, 260


# ---- the fold -------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("red", [SUM, PROD])
@pytest.mark.parametrize("P", [2, 3, 6, 16])
@pytest.mark.parametrize("kind", ["sum", "prod", "wide"])
def test_f16_fold_equals_numpy_half_left_fold(oracle, P, red, kind):
    src = inputs.typed_rank_vectors([40, P], P, 4099, F16, kind)
    got = oracle.chain_fold_dt(src, F16, red)
    with np.errstate(all="ignore"):
        s = src[0].copy()
        for r in range(1, P):
            s = (s * src[r]) if red == PROD else (s + src[r])     # numpy half arithmetic, one rounding per operation
    assert s.dtype == np.float16
    assert same_bits_or_both_nan(got, s, F16)


@pytest.mark.parametrize("red", [SUM, PROD])
@pytest.mark.parametrize("P", [2, 3, 6, 16])
@pytest.mark.parametrize("kind", ["sum", "prod", "wide"])
def test_bf16_fold_equals_torch_bfloat16_left_fold(oracle, P, red, kind):
    src = inputs.typed_rank_vectors([41, P], P, 4099, BF16, kind)
    got = oracle.chain_fold_dt(src, BF16, red)
    s = bf16_bits_to_torch(src[0])
    for r in range(1, P):
        x = bf16_bits_to_torch(src[r])
        s = (s * x) if red == PROD else (s + x)                   # torch CPU bfloat16 arithmetic
    assert s.dtype == torch.bfloat16
    assert same_bits_or_both_nan(got, torch_to_bf16_bits(s), BF16)


@pytest.mark.parametrize("red", [SUM, PROD])
@pytest.mark.parametrize("P", [2, 5, 16])
def test_f64_and_f32_folds(oracle, P, red):
    src = inputs.typed_rank_vectors([42, P], P, 3001, F64, "prod" if red == PROD else "sum")
    got = oracle.chain_fold_dt(src, F64, red)
    s = src[0].copy()
    for r in range(1, P):
        s = (s * src[r]) if red == PROD else (s + src[r])
    assert same_bits_or_both_nan(got, s, F64)
    # f32 through the typed entry point = the fp32 fold pinned in test_oracle_pins / test_oracle_op_pins
    src32 = inputs.typed_rank_vectors([42, P], P, 3001, F32, "prod" if red == PROD else "sum")
    assert same_bits_or_both_nan(oracle.chain_fold_dt(src32, F32, red), oracle.chain_fold(src32, red), F32)


def test_order_separators_and_no_wide_accumulator(oracle):
    # f16: 2048 + 1 is a tie that goes to 2048; a fold that is not left-to-right, or that accumulates in a wider type and
    # rounds once at the end (2050), gives another value.  bf16: the same with 256 (spacing 2 above 256).
    col16 = lambda *v: [np.array([x], dtype=np.float16) for x in v]
    assert oracle.chain_fold_dt(col16(2048, 1, 1), F16, SUM)[0] == np.float16(2048)
    assert oracle.chain_fold_dt(col16(1, 1, 2048), F16, SUM)[0] == np.float16(2050)
    assert oracle.chain_fold_dt(col16(60000, 2, 0.25), F16, PROD)[0] == np.float16(np.inf)       # (60000 * 2) overflows first
    assert oracle.chain_fold_dt(col16(2, 0.25, 60000), F16, PROD)[0] == np.float16(30000)
    colb = lambda *v: [np.array([oracle.bf16_from_f64(x)], dtype=np.uint16) for x in v]
    assert oracle.bf16_to_f64(int(oracle.chain_fold_dt(colb(256, 1, 1), BF16, SUM)[0])) == 256.0
    assert oracle.bf16_to_f64(int(oracle.chain_fold_dt(colb(1, 1, 256), BF16, SUM)[0])) == 258.0
    # products (spacing 2^-6 in [2, 4), 2^-7 in [1, 2)): 3 x 1.0078125 = 3.0234375 is a tie -> 3.03125 (even), x 1.0078125 =
    # 3.0549... -> 3.0625; the other way round 1.0078125^2 = 1.01568... -> 1.015625, x 3 = 3.046875 exactly
    assert oracle.bf16_to_f64(int(oracle.chain_fold_dt(colb(3, 1.0078125, 1.0078125), BF16, PROD)[0])) == 3.0625
    assert oracle.bf16_to_f64(int(oracle.chain_fold_dt(colb(1.0078125, 1.0078125, 3), BF16, PROD)[0])) == 3.046875
    # f64: (1e308 * 10) overflows before the 0.01 arrives
    col64 = lambda *v: [np.array([x], dtype=np.float64) for x in v]
    assert oracle.chain_fold_dt(col64(1e308, 10.0, 0.01), F64, PROD)[0] == np.inf
    assert oracle.chain_fold_dt(col64(1.0, 2.0 ** -53, 2.0 ** -53), F64, SUM)[0] == 1.0         # each tie goes back to 1.0
    assert oracle.chain_fold_dt(col64(2.0 ** -53, 2.0 ** -53, 1.0), F64, SUM)[0] == 1.0 + 2.0 ** -52


@pytest.mark.parametrize("dt,limit", [(F16, 2048), (BF16, 256), (F64, 1 << 40)])
def test_small_integers_are_exact_in_any_order(oracle, dt, limit):
    rng = np.random.default_rng([43, dt])
    P, n = 7, 513
    ints = rng.integers(-(limit // (2 * P)), limit // (2 * P) + 1, size=(P, n))
    if dt == F16:
        src = [ints[r].astype(np.float16) for r in range(P)]
        back = lambda a: a.astype(np.int64)
    elif dt == BF16:
        src = [np.array([oracle.bf16_from_f64(float(v)) for v in ints[r]], dtype=np.uint16) for r in range(P)]
        back = lambda a: bf16_bits_to_f32(a).astype(np.int64)
    else:
        src = [ints[r].astype(np.float64) for r in range(P)]
        back = lambda a: a.astype(np.int64)
    assert np.array_equal(back(src[3]), ints[3])                  # the inputs themselves are exact
    assert np.array_equal(back(oracle.chain_fold_dt(src, dt, SUM)), ints.sum(axis=0))
    assert np.array_equal(back(oracle.chain_fold_dt(src[::-1], dt, SUM)), ints.sum(axis=0))


@pytest.mark.parametrize("dt,u", [(F16, 2.0 ** -11), (BF16, 2.0 ** -8), (F64, 2.0 ** -53)])
def test_fold_within_the_rounding_error_bound_of_the_exact_sum(oracle, dt, u):
    P, n = 16, 2000
    src = inputs.typed_rank_vectors([44, P], P, n, dt, "sum")
    if dt == F16:
        wide = [s.astype(np.float64) for s in src]
        out = oracle.chain_fold_dt(src, dt, SUM).astype(np.float64)
    elif dt == BF16:
        wide = [bf16_bits_to_f32(s).astype(np.float64) for s in src]
        out = bf16_bits_to_f32(oracle.chain_fold_dt(src, dt, SUM)).astype(np.float64)
    else:
        wide = src
        out = oracle.chain_fold_dt(src, dt, SUM)
    exact = np.array([math.fsum(w[i] for w in wide) for i in range(n)])
    mag = np.sum(np.abs(np.array(wide)), axis=0)
    g = (P - 1) * u / (1 - (P - 1) * u)
    assert np.all(np.abs(out - exact) <= g * mag)
    if dt != F64:   # and the 16-bit folds are NOT what a wide accumulator rounded once would give (some element differs)
        once = exact.astype(np.float16).astype(np.float64) if dt == F16 else None
        if once is not None:
            assert np.any(once != out)


# ---- the collectives ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dt", [F16, BF16, F64, F32])
@pytest.mark.parametrize("red", [SUM, PROD])
def test_typed_collectives_semantics(oracle, dt, red):
    P, n = 5, 1031
    src = inputs.typed_rank_vectors([45, P], P, n, dt, "prod" if red == PROD else "sum")
    want = oracle.chain_fold_dt(src, dt, red)
    for root in range(P):
        bufs = [s.copy() for s in src]
        oracle.reduce_dt(bufs, dt, red, root)
        assert bufs[root].tobytes() == want.tobytes()             # root-invariant chain order (U4)
        assert all(bufs[r].tobytes() == src[r].tobytes() for r in range(P) if r != root)   # U5
        oracle.broadcast_dt(bufs, dt, root)
        assert all(b.tobytes() == want.tobytes() for b in bufs)
    bufs = [s.copy() for s in src]
    oracle.allreduce_dt(bufs, dt, red)
    assert all(b.tobytes() == want.tobytes() for b in bufs)       # allreduce = broadcast o reduce
    one = [src[2].copy()]
    oracle.allreduce_dt(one, dt, red)
    assert one[0].tobytes() == src[2].tobytes()                   # P = 1: identity
    bufs = [s.copy() for s in src]
    oracle.broadcast_dt(bufs, dt, 3)
    assert all(b.tobytes() == src[3].tobytes() for b in bufs)     # broadcast moves bytes, no arithmetic


def test_typed_bad_arguments(oracle):
    src = inputs.typed_rank_vectors(46, 2, 8, F16)
    with pytest.raises(RuntimeError):
        oracle.chain_fold_dt(src, F16, 2)
    with pytest.raises(RuntimeError):
        oracle.reduce_dt([s.copy() for s in src], F16, SUM, root=2)
    with pytest.raises(TypeError):
        oracle.allreduce_dt([s.astype(np.float32) for s in src], F16, SUM)
    with pytest.raises((RuntimeError, KeyError)):
        oracle.lib().lpo_allreduce_dt  # symbol exists
        oracle.allreduce_dt([s.copy() for s in src], 9, SUM)
