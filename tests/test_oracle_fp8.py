"""Pins of the oracle's FP8-E4M3 cast (FORMAT R12; §4.8, L433-448 §6.3): the conversion against torch's
float8_e4m3fn cast, the activation cast against its definition, the FP8 linear against the INT8 one (the paper's Table 7
puts the two within 0.1 PPL: the FP8 result must sit close to, and be noisier than, the INT8 result)."""
import numpy as np
import torch

import hq_synth
from oracle import hqo

SNR = float(np.float32(22.68))


def test_e4m3_round_equals_torch_cast_inside_the_finite_range():
    rng = np.random.default_rng(0)
    x = np.concatenate([rng.uniform(-448, 448, 40000), rng.standard_normal(20000) * 0.01, rng.standard_normal(20000) * 1e-3,
                        np.arange(-127, 128), [0.0, 2.0 ** -9, 2.0 ** -10, 3 * 2.0 ** -10, 448.0, -448.0, 17.0, 19.0, 18.0]]).astype(np.float32)
    got = hqo.e4m3_round(x)
    ref = torch.from_numpy(x).to(torch.float8_e4m3fn).to(torch.float32).numpy()
    assert np.array_equal(got, ref)
    # every integer code up to 16 is exact, beyond that the grid is 2, 4, 8 wide (FORMAT R12)
    c = np.arange(-127, 128).astype(np.float32)
    r = hqo.e4m3_round(c)
    assert np.array_equal(r[np.abs(c) <= 16], c[np.abs(c) <= 16])
    assert np.max(np.abs(r - c)) == 4.0                                 # half of the widest step
    # saturation (cvt.rn.satfinite): anything that would round above 448 is 448
    assert list(hqo.e4m3_round(np.array([449.0, 464.0, 1e6, -1e9], np.float32))) == [448.0, 448.0, 448.0, -448.0]


def test_act_quant_fp8_definition():
    x = hq_synth.activations(3, 512, seed=2)
    q8, sx = hqo.act_quant_fp8(x, 128, 7)
    _, _, u = hqo.act_quant(x, hqo.E8, 128, 7, want_u=True)          # the same RHT output (R1), pinned elsewhere
    for b in range(3):
        for kt in range(4):
            ut = u[b, 128 * kt:128 * kt + 128]
            amax = np.float32(np.abs(ut).max())
            inv = np.float32(448.0) / amax
            want = torch.from_numpy((ut * inv).astype(np.float32)).to(torch.float8_e4m3fn).float().numpy()
            assert np.array_equal(q8[b, 128 * kt:128 * kt + 128], want)
            assert sx[b, kt] == amax / np.float32(448.0)
    assert np.abs(q8).max() == 448.0
    q0, s0 = hqo.act_quant_fp8(np.zeros((1, 128), np.float32), 128, 7)
    assert not q0.any() and s0[0, 0] == 0.0


def test_linear_fp8_close_to_int8_and_to_the_dense_product():
    W = hq_synth.gaussian_weight(96, 512, seed=11)
    x = hq_synth.activations(4, 512, seed=12)
    enc = hqo.encode_weights(W, hqo.E8, 128, SNR, 3)
    q, sx = hqo.act_quant(x, hqo.E8, 128, 3)
    _, y_i8 = hqo.linear(enc["codes"], enc["norms"], hqo.E8, 128, SNR, q, sx, want_acc=False)
    q8, sx8 = hqo.act_quant_fp8(x, 128, 3)
    y_f8 = hqo.linear_fp8(enc["codes"], enc["norms"], hqo.E8, 128, SNR, q8, sx8)
    y = x.astype(np.float64) @ W.astype(np.float64).T
    rms = np.sqrt((y ** 2).mean())
    e_i8 = np.sqrt(((y_i8 - y) ** 2).mean()) / rms
    e_f8 = np.sqrt(((y_f8 - y) ** 2).mean()) / rms
    assert e_i8 < 0.09 and e_f8 < 0.12          # both dominated by the 22.7 dB weight quantization (7.3 %)
    assert e_f8 > e_i8                          # FP8's 3 mantissa bits are coarser than INT8's 127 levels (§6.3 "INT8 wins")
    # by hand on one output: the operands are exactly the E4M3 roundings
    c8 = hqo.e4m3_round(enc["codes"][5].astype(np.float32)).astype(np.float64)
    A = hqo.lib().hqo_alpha(hqo.E8, SNR) * np.sqrt(128.0)
    want = 0.0
    for kt in range(4):
        rho = float(np.array([enc["norms"][5, kt]], np.uint16).view(np.float16)[0])
        want += rho / A * float(sx8[2, kt]) * float(c8[128 * kt:128 * kt + 128] @ q8[2, 128 * kt:128 * kt + 128].astype(np.float64))
    assert abs(y_f8[2, 5] - want) <= 1e-12 * max(1.0, abs(want))
