"""Pins for the CPU oracle (oracle/oracle_mlp.c) -- CPU only.

The oracle is pinned to things other than itself: hand-worked values
(tests/golden/), exact-rational brute force, closed forms, special cases that
reduce to a library routine, the analytic rounding bound against float64, and
invariants.  Each test names the plausible mistake it would catch.
"""
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest
import torch

import oracle
from paper_2607_07862_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
ACT = {"none": oracle.ACT_NONE, "relu": oracle.ACT_RELU, "gelu": oracle.ACT_GELU_TANH}


def bf16_bits(a) -> np.ndarray:
    """float array (exactly bf16-representable or not) -> bf16 bits via torch's cast."""
    return inputs.as_u16(torch.tensor(np.asarray(a, dtype=np.float32)).to(torch.bfloat16))


def bits_to_f32(a: np.ndarray) -> np.ndarray:
    return (a.astype(np.uint32) << 16).view(np.float32)


# ---------------------------------------------------------------- bf16 RNE
def test_bf16_rne_golden_ties():
    """catches: truncation instead of rounding, ties-away instead of ties-even."""
    with open(os.path.join(GOLDEN, "bf16_rne.json")) as f:
        cases = json.load(f)["cases"]
    for c in cases:
        got = oracle.bf16_rne(float(np.float32(c["value"])))
        assert got == int(c["bf16_hex"], 16), c


def test_bf16_roundtrip_all_patterns():
    """every finite bf16 pattern survives bf16 -> f32 -> bf16 unchanged."""
    for h in range(0, 1 << 16, 1):
        if (h & 0x7F80) == 0x7F80:
            continue
        assert oracle.bf16_rne(oracle.bf16_to_f32(h)) == h
    assert oracle.bf16_to_f32(0x3F80) == 1.0 and oracle.bf16_to_f32(0xC020) == -2.5


def test_bf16_rne_matches_library_cast():
    """torch's own fp32->bf16 cast (a library routine) on random and near-tie floats."""
    rng = np.random.default_rng(7)
    x = np.concatenate([
        rng.standard_normal(20000).astype(np.float32) * np.float32(10.0) ** rng.integers(-6, 6, 20000).astype(np.float32),
        (1.0 + rng.integers(0, 1 << 16, 5000) * 2.0 ** -16).astype(np.float32),   # dense around ties
        np.array([0.0, -0.0, 3.3895314e38, 1e-40, -1e-40], dtype=np.float32),
    ])
    want = bf16_bits(x)
    got = np.array([oracle.bf16_rne(float(v)) for v in x], dtype=np.uint16)
    assert np.array_equal(got, want)


def test_brute_rounding_helpers_against_numpy():
    """pins the brute-force helper itself (it pins the oracle, so it needs a pin too)."""
    rng = np.random.default_rng(3)
    for _ in range(300):
        a, b = np.float32(rng.standard_normal()), np.float32(rng.standard_normal() * 1e-3)
        want = np.float32(a + b)                      # IEEE fp32 add
        got = oracle.brute_round_f32(Fraction(float(a)) + Fraction(float(b)))
        assert Fraction(float(want)) == got
    for h in [0x3F80, 0x4380, 0xC020, 0x0001, 0x8000 | 0x0080, 0x7F7F]:
        assert oracle.brute_bf16_bits(oracle.brute_bf16_value(h)) == h


# ---------------------------------------------------------------- GeLU
def test_gelu_identities():
    """g(0)=0, g(x)-g(-x)=x, g(x)->x for large x, g(x)->0 for very negative x."""
    assert oracle.gelu_tanh(0.0) == 0.0
    for x in [0.1, 0.5, 1.0, 2.0, 3.5]:
        assert abs((oracle.gelu_tanh(x) - oracle.gelu_tanh(-x)) - x) <= 2e-7 * max(1.0, x)
    for x in [6.0, 10.0, 50.0]:
        assert oracle.gelu_tanh(x) == pytest.approx(x, rel=1e-7)
        assert abs(oracle.gelu_tanh(-x)) < 1e-7


def test_gelu_matches_library_float64():
    """torch.nn.functional.gelu(approximate='tanh') in float64: pins the constants
    0.7978845608 = sqrt(2/pi) and 0.044715 (catches a wrong constant, erf-form, sign)."""
    xs = np.linspace(-8, 8, 4001).astype(np.float32)
    want = torch.nn.functional.gelu(torch.tensor(xs, dtype=torch.float64), approximate="tanh").numpy()
    got = np.array([oracle.gelu_tanh(float(x)) for x in xs], dtype=np.float64)
    assert np.max(np.abs(got - want)) <= 1e-6
    assert abs(math.sqrt(2.0 / math.pi) - 0.7978845608028654) < 1e-15
    # the erf form differs by up to ~5e-4 (max near |x| ~ 2): make sure we are not that one
    erf = torch.nn.functional.gelu(torch.tensor(xs, dtype=torch.float64)).numpy()
    assert np.max(np.abs(got - erf)) > 1e-4


def test_relu_and_none():
    assert oracle.act_f32(-3.0, oracle.ACT_RELU) == 0.0
    assert oracle.act_f32(2.5, oracle.ACT_RELU) == 2.5
    assert oracle.act_f32(-3.0, oracle.ACT_NONE) == -3.0
    assert math.copysign(1.0, oracle.act_f32(-0.0, oracle.ACT_RELU)) == 1.0


# ---------------------------------------------------------------- hand-worked
def test_handworked_golden():
    """catches: transposed operand, dropped activation, act on the last layer,
    missing bf16 rounding of H."""
    with open(os.path.join(GOLDEN, "handworked_chain.json")) as f:
        cases = json.load(f)["cases"]
    for c in cases:
        X = bf16_bits(c["X"])
        W1 = bf16_bits(np.array(c["W1_kn"], dtype=np.float32).T)   # boundary layout [N x K]
        W2 = bf16_bits(np.array(c["W2_kn"], dtype=np.float32).T)
        outs, _ = oracle.mlp_chain(X, [W1, W2], ACT[c["act"]])
        assert np.array_equal(bits_to_f32(outs[0]), np.array(c["H"], dtype=np.float32)), c["name"]
        assert np.array_equal(bits_to_f32(outs[1]), np.array(c["Y"], dtype=np.float32)), c["name"]


# ---------------------------------------------------------------- brute force
@pytest.mark.parametrize("shape,act,seed", [
    ((3, 5, 4, 2), "relu", 0), ((2, 8, 8, 8), "none", 1), ((1, 7, 3, 5), "relu", 2), ((4, 6, 2, 3), "none", 3),
])
def test_brute_force_tiny_random(shape, act, seed):
    """exact-rational triple loop with explicit fp32 / bf16 roundings vs the C oracle,
    on random (non-integer) bf16 inputs and non-square shapes: catches a wrong index,
    a transposed operand, a wrong rounding point or accumulation precision."""
    M, K, N1, N2 = shape
    rng = np.random.default_rng(seed)
    X = bf16_bits(rng.standard_normal((M, K)))
    W1 = bf16_bits(rng.standard_normal((N1, K)))
    W2 = bf16_bits(rng.standard_normal((N2, N1)))
    outs, _ = oracle.mlp_chain(X, [W1, W2], ACT[act])
    want = oracle.brute_mlp(X.tolist(), [W1.tolist(), W2.tolist()], ACT[act])
    assert outs[0].tolist() == want[0]
    assert outs[1].tolist() == want[1]


def test_brute_force_three_layers_act_placement():
    """L=3: activation after layers 1 and 2, none after layer 3 (reading c2)."""
    rng = np.random.default_rng(11)
    X = bf16_bits(rng.integers(-2, 3, (2, 4)))
    Ws = [bf16_bits(rng.integers(-2, 3, s)) for s in [(3, 4), (5, 3), (2, 5)]]
    outs, _ = oracle.mlp_chain(X, Ws, oracle.ACT_RELU)
    want = oracle.brute_mlp(X.tolist(), [w.tolist() for w in Ws], oracle.ACT_RELU)
    for o, w in zip(outs, want):
        assert o.tolist() == w
    assert (bits_to_f32(outs[0]) >= 0).all() and (bits_to_f32(outs[1]) >= 0).all()
    assert (bits_to_f32(outs[2]) < 0).any(), "last layer must not be activated"


def test_ascending_k_order_is_observable():
    """fp32 addition is not associative: 2^24 + 1 + 1 (ascending) = 2^24, while
    1 + 1 + 2^24 = 2^24 + 2.  Pins the summation order of the accumulator."""
    big = 2.0 ** 12
    X = bf16_bits([[big, 1.0, 1.0]])
    W = bf16_bits([[big, 1.0, 1.0]])                    # N=1, K=3
    _, acc, _ = oracle.gemm_layer(X, W, oracle.ACT_NONE, want_acc=True)
    assert acc[0, 0] == np.float32(2.0 ** 24)
    X2 = bf16_bits([[1.0, 1.0, big]])
    W2 = bf16_bits([[1.0, 1.0, big]])
    _, acc2, _ = oracle.gemm_layer(X2, W2, oracle.ACT_NONE, want_acc=True)
    assert acc2[0, 0] == np.float32(2.0 ** 24 + 2.0)


# ---------------------------------------------------------------- closed forms / special cases
def test_all_ones_closed_form_cfg0():
    """cfg 0 with all-ones inputs, ReLU: acc1 = 512, H = 512, acc2 = 2048*512 = 2^20."""
    M, K, N1, N2 = 64, 512, 2048, 512
    one = np.full((1,), 0x3F80, dtype=np.uint16)
    X = np.broadcast_to(one, (M, K)).copy()
    W1 = np.broadcast_to(one, (N1, K)).copy()
    W2 = np.broadcast_to(one, (N2, N1)).copy()
    outs, _ = oracle.mlp_chain(X, [W1, W2], oracle.ACT_RELU)
    assert (bits_to_f32(outs[0]) == 512.0).all()
    assert (bits_to_f32(outs[1]) == 2.0 ** 20).all()


def test_zero_input_gives_zero():
    rng = np.random.default_rng(5)
    X = np.zeros((3, 16), dtype=np.uint16)
    W1, W2 = bf16_bits(rng.standard_normal((8, 16))), bf16_bits(rng.standard_normal((4, 8)))
    for act in ACT.values():
        outs, _ = oracle.mlp_chain(X, [W1, W2], act)
        assert not outs[1].any()


def test_identity_special_cases():
    """W1 = I, ReLU: H = ReLU(X) bit-exactly, so Y = ReLU(X).W2 is ONE textbook GEMM,
    checked against numpy float64 (exact for these integer inputs).  W2 = I too: Y = ReLU(X)."""
    rng = np.random.default_rng(9)
    M, K, N2 = 5, 12, 7
    Xf = rng.integers(-2, 3, (M, K)).astype(np.float32) * 0.5
    X = bf16_bits(Xf)
    eye = bf16_bits(np.eye(K))
    W2f = rng.integers(-2, 3, (N2, K)).astype(np.float32)
    outs, _ = oracle.mlp_chain(X, [eye, bf16_bits(W2f)], oracle.ACT_RELU)
    assert np.array_equal(bits_to_f32(outs[0]), np.maximum(Xf, 0))
    want = np.maximum(Xf, 0).astype(np.float64) @ W2f.astype(np.float64).T
    assert np.array_equal(bits_to_f32(outs[1]).astype(np.float64), want)
    outs, _ = oracle.mlp_chain(X, [eye, eye], oracle.ACT_RELU)
    assert np.array_equal(bits_to_f32(outs[1]), np.maximum(Xf, 0))


def test_against_float64_library_matmul_within_rounding_bound():
    """act = NONE, single layer: |acc_fp32 - acc_f64| <= K * 2^-24 * sum_k |a_k||w_k|
    (standard forward bound for recursive summation; products are exact), and the
    bf16 output is within half a bf16 ulp of the fp32 accumulator."""
    cfg = inputs.get_config(0)
    X, Ws = inputs.make_inputs(cfg)
    Xu, Wu = inputs.as_u16(X), inputs.as_u16(Ws[0])
    out, acc, _ = oracle.gemm_layer(Xu, Wu, oracle.ACT_NONE, want_acc=True)
    X64, W64 = X.to(torch.float64), Ws[0].to(torch.float64)
    ref = (X64 @ W64.T).numpy()
    bound = cfg.widths[0] * 2.0 ** -24 * (X64.abs() @ W64.abs().T).numpy()
    assert (np.abs(acc.astype(np.float64) - ref) <= bound + 1e-300).all()
    assert np.abs(acc.astype(np.float64) - ref).max() > 0, "fp32 accumulation must be visible"
    o = bits_to_f32(out).astype(np.float64)
    assert (np.abs(o - acc) <= np.abs(acc) * 2.0 ** -8 + 1e-38).all()


def test_two_layer_against_float64_chain():
    """whole cfg-0 chain, act NONE: Y within the propagated bound of float64 X@W1@W2."""
    cfg = inputs.get_config(0)
    X, Ws = inputs.make_inputs(cfg)
    outs, _ = oracle.mlp_chain(inputs.as_u16(X), [inputs.as_u16(w) for w in Ws], oracle.ACT_NONE)
    X64, A64, B64 = X.to(torch.float64), Ws[0].to(torch.float64), Ws[1].to(torch.float64)
    H64 = X64 @ A64.T
    Y64 = (H64 @ B64.T).numpy()
    # H carries a relative error <= (K 2^-24 + 2^-9) on sum|x||a|; propagate through |B|.
    eH = (512 * 2.0 ** -24 + 2.0 ** -9) * (X64.abs() @ A64.abs().T)
    Hhat = H64.abs() + eH
    bound = (eH @ B64.abs().T + (2048 * 2.0 ** -24 + 2.0 ** -9) * (Hhat @ B64.abs().T)).numpy()
    got = bits_to_f32(outs[1]).astype(np.float64)
    assert (np.abs(got - Y64) <= bound).all()
    rel = oracle.rel_err(outs[1], inputs.as_u16(torch.tensor(Y64).to(torch.bfloat16)))
    assert rel["err"] < 2e-2


# ---------------------------------------------------------------- exact mode
def test_exact_mode_certificate_cfg0():
    """integer inputs in {-2..2}: every fp32 partial sum is an integer < 2^24, so
    fp32 accumulation equals int64 accumulation (reading c7) and equals numpy int64."""
    cfg = inputs.get_config(0, "exact")
    X, Ws = inputs.make_inputs(cfg)
    Xu, Wu = inputs.as_u16(X), [inputs.as_u16(w) for w in Ws]
    outs, certs = oracle.mlp_chain(Xu, Wu, oracle.ACT_RELU, want_cert=True)
    for mx, bad, nonint in certs:
        assert bad == 0 and nonint == 0 and mx < 2 ** 24
    Xi, W1i, W2i = (t.to(torch.float64).numpy().astype(np.int64) for t in (X, Ws[0], Ws[1]))
    assert set(np.unique(Xi)) <= {-2, -1, 0, 1, 2}
    acc1 = Xi @ W1i.T
    H = np.maximum(acc1, 0)
    Hb = bits_to_f32(bf16_bits(H.astype(np.float32))).astype(np.int64)    # library cast to bf16
    assert np.array_equal(bits_to_f32(outs[0]).astype(np.int64), Hb)
    acc2 = Hb @ W2i.T
    assert np.abs(acc2).max() < 2 ** 24
    assert np.array_equal(outs[1], bf16_bits(acc2.astype(np.float32)))
    # the final bf16 rounding really matters on this instance (most |Y| > 256)
    assert (bits_to_f32(outs[1]).astype(np.int64) != acc2).mean() > 0.3


def test_exact_mode_hidden_unit_permutation_invariance():
    """permuting W1 rows (hidden units) and W2 columns together leaves Y unchanged
    bit-for-bit in exact mode (every summation order is exact)."""
    cfg = inputs.get_config(0, "exact")
    X, Ws = inputs.make_inputs(cfg)
    Xu, W1, W2 = inputs.as_u16(X), inputs.as_u16(Ws[0]), inputs.as_u16(Ws[1])
    perm = np.random.default_rng(1).permutation(W1.shape[0])
    a, _ = oracle.mlp_chain(Xu, [W1, W2], oracle.ACT_RELU)
    b, _ = oracle.mlp_chain(Xu, [W1[perm].copy(), W2[:, perm].copy()], oracle.ACT_RELU)
    assert np.array_equal(a[1], b[1])
    assert np.array_equal(a[0][:, perm], b[0])


# ---------------------------------------------------------------- invariants
def test_row_independence_and_thread_independence():
    """Y row m depends only on X row m (this is MICROBATCH's parity), and the result
    does not depend on the OpenMP thread count."""
    cfg = inputs.get_config(0)
    X, Ws = inputs.make_inputs(cfg)
    Xu, Wu = inputs.as_u16(X), [inputs.as_u16(w) for w in Ws]
    full, _ = oracle.mlp_chain(Xu, Wu, oracle.ACT_GELU_TANH)
    one, _ = oracle.mlp_chain(Xu, Wu, oracle.ACT_GELU_TANH, threads=1)
    assert np.array_equal(full[1], one[1]) and np.array_equal(full[0], one[0])
    for r0, r1 in [(0, 16), (16, 17), (40, 64)]:
        part, _ = oracle.mlp_chain(Xu[r0:r1].copy(), Wu, oracle.ACT_GELU_TANH)
        assert np.array_equal(part[1], full[1][r0:r1])


def test_relu_power_of_two_homogeneity():
    """Y(2X) = 2 Y(X) bit-exactly for ReLU (scaling by 2 commutes with every rounding)."""
    cfg = inputs.get_config(0)
    X, Ws = inputs.make_inputs(cfg)
    Wu = [inputs.as_u16(w) for w in Ws]
    y1, _ = oracle.mlp_chain(inputs.as_u16(X), Wu, oracle.ACT_RELU)
    y2, _ = oracle.mlp_chain(inputs.as_u16((X.float() * 2).to(torch.bfloat16)), Wu, oracle.ACT_RELU)
    assert np.array_equal(bits_to_f32(y2[1]), 2 * bits_to_f32(y1[1]))


def test_rel_err_metric():
    """reading c3: err = max |Yg - Yo| / max(|Yo_ij|, rms(Yo))."""
    ref = bf16_bits([[1.0, -2.0, 0.0, 4.0]])
    got = bf16_bits([[1.0, -2.0, 0.03125, 4.0]])
    rms = math.sqrt((1 + 4 + 0 + 16) / 4)
    assert oracle.rel_err(got, ref)["err"] == pytest.approx(0.03125 / rms)
    assert oracle.rel_err(ref, ref)["err"] == 0.0
    nan = ref.copy()
    nan[0, 1] = 0x7FC0
    assert oracle.rel_err(nan, ref)["nan"] == 1


def test_inputs_are_seeded_and_shaped():
    """generator: deterministic, right shapes/layout, row prefix stable under M."""
    cfg = inputs.get_config(1)
    X, Ws = inputs.make_inputs(cfg, M=4)
    X2, _ = inputs.make_inputs(cfg, M=2)
    assert torch.equal(X[:2], X2)
    assert X.shape == (4, 4096) and Ws[0].shape == (14336, 4096) and Ws[1].shape == (4096, 14336)
    assert abs(float(Ws[0].float().std()) - 1 / 64.0) < 1e-3
    e = inputs.make_inputs(inputs.get_config(0, "exact"))[0]
    assert set(np.unique(e.float().numpy())) == {-2.0, -1.0, 0.0, 1.0, 2.0}
    assert inputs.CONFIGS[2].flops == 2 * 256 * 4096 * 14336 * 2
    assert inputs.CONFIGS[1].algorithmic_bytes == 2 * (2 * 4096 * 14336 + 16 * 4096 + 2 * 16 * 14336 + 16 * 4096)
