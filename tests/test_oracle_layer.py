"""Pins of the oracle's layer glue (FORMAT R8-R10; §4.1 "the butterfly folds into the preceding
LayerNorm"): bf16 rounding against torch's cast, RMSNorm and SiLU·mul against their float64
definitions, the canonical exponential against libm's double exp."""
import math

import numpy as np
import torch

from oracle import hqo


def _bf16_t(x):
    return torch.from_numpy(np.ascontiguousarray(x, np.float32)).to(torch.bfloat16).to(torch.float32).numpy()


def test_bf16_round_equals_torch_cast():
    rng = np.random.default_rng(0)
    x = np.concatenate([rng.standard_normal(50000).astype(np.float32) * 10.0 ** rng.integers(-20, 20, 50000),
                        # exact ties (low half-word 0x8000) on even and odd mantissas, zeros, tiny values
                        np.array([1.00390625, 1.01171875, -1.00390625, 0.0, -0.0, 1e-40, 3.3895e38], np.float32)]).astype(np.float32)
    bits = x.view(np.uint32).copy()
    bits[:2000] = (bits[:2000] & 0xffff0000) | 0x8000          # force ties
    x = bits.view(np.float32)
    assert np.array_equal(hqo.bf16_round(x).view(np.uint32), _bf16_t(x).view(np.uint32))


def test_exp_c_against_double_exp():
    t = np.concatenate([np.linspace(-87, 88, 20001), np.linspace(-1, 1, 4001), [0.0, -87.0, 88.0]]).astype(np.float32)
    got = hqo.exp_c(t).astype(np.float64)
    ref = np.exp(t.astype(np.float64))
    assert np.max(np.abs(got / ref - 1.0)) <= 2.5e-7
    assert hqo.exp_c([0.0])[0] == 1.0
    # clamped outside the range
    assert hqo.exp_c([-200.0])[0] == hqo.exp_c([-87.0])[0] and hqo.exp_c([200.0])[0] == hqo.exp_c([88.0])[0]


def test_rmsnorm_against_float64_definition():
    rng = np.random.default_rng(1)
    for n in (256, 4096, 14336):
        h = _bf16_t(rng.standard_normal(n) * 3.0)
        g = _bf16_t(1.0 + 0.1 * rng.standard_normal(n))
        eps = 1e-5
        x = hqo.rmsnorm_bf16(h, g, eps)
        h64, g64 = h.astype(np.float64), g.astype(np.float64)
        ref = h64 * g64 / math.sqrt(np.mean(h64 * h64) + eps)
        want = _bf16_t(ref.astype(np.float32))
        # fp32 evaluation may differ from the exact value by one rounding: at most one bf16 step, almost always equal
        ulp = np.maximum(np.abs(want), 1e-30) * 2.0 ** -7
        assert np.all(np.abs(x - want) <= ulp)
        assert np.mean(x == want) > 0.99
        assert np.array_equal(x, hqo.bf16_round(x))            # the result is a bf16 value
    # closed form: a constant vector c with unit gain gives c / sqrt(c^2 + eps) everywhere
    h = np.full(512, 2.0, np.float32)
    x = hqo.rmsnorm_bf16(h, np.ones(512, np.float32), 0.25)
    assert np.all(x == _bf16_t(np.float32(2.0 / math.sqrt(4.25))))
    # eps matters (a dropped eps fails): zero vector stays zero, not NaN
    assert np.all(hqo.rmsnorm_bf16(np.zeros(128, np.float32), np.ones(128, np.float32), 1e-6) == 0.0)


def test_silu_mul_against_float64_definition():
    rng = np.random.default_rng(2)
    a = _bf16_t(rng.standard_normal(20000) * 4.0)
    b = _bf16_t(rng.standard_normal(20000))
    x = hqo.silu_mul_bf16(a, b)
    a64, b64 = a.astype(np.float64), b.astype(np.float64)
    ref = a64 / (1.0 + np.exp(-a64)) * b64
    want = _bf16_t(ref.astype(np.float32))
    ulp = np.maximum(np.abs(want), 1e-30) * 2.0 ** -7
    assert np.all(np.abs(x - want) <= ulp)
    assert np.mean(x == want) > 0.99
    # special values: silu(0) = 0; large negative gate -> 0 (no NaN); large positive gate -> a * b
    x = hqo.silu_mul_bf16(np.array([0.0, -100.0, 100.0], np.float32), np.array([3.0, 3.0, 0.5], np.float32))
    assert x[0] == 0.0 and abs(x[1]) < 1e-30 and x[2] == 50.0
