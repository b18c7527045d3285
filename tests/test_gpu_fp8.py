"""GPU parity of the FP8-E4M3 MMA cast (include/hq.h hq_linear_cast; §4.8, §6.3; SURVEY §8(f)2;
FORMAT R12) against the oracle: y within 1e-3 (G16) of the oracle's FP8 linear (E4M3 operands, double accumulation).
A wrong rounding of either operand, a swapped byte in a packed conversion or a wrong scale shows up at the 1e-2 level
(one E4M3 step is 6 % of a value), far above the bar."""
import numpy as np
import pytest

import hq_synth
from oracle import hqo

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

SNR = float(np.float32(22.68))


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23406_b200 as hq
    c = hq.Context(0)
    yield c
    c.close()


def _dev(a, dtype=torch.bfloat16):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda().to(dtype)


def _rel_err(y, ref, floor=1e-3):
    ref = np.asarray(ref, np.float64)
    rms = np.sqrt((ref ** 2).mean())
    return np.max(np.abs(np.asarray(y, np.float64) - ref) / np.maximum(np.abs(ref), floor * rms + 1e-30))


@pytest.mark.parametrize("B,m,n_in,n_tile,k", [
    (64, 128, 512, 128, (2, 2)),
    (300, 200, 1024, 128, (-1, -1)),      # ragged rows and batch, several batch tiles
    (257, 384, 1024, 256, (2, 2)),        # RHT tile 256: two operand chunks per accumulator drain
    (600, 130, 2048, 256, (1, 1)),
])
def test_linear_fp8_matches_oracle(ctx, B, m, n_in, n_tile, k):
    import paper_2606_23406_b200 as hq
    seed = 9
    W = hq_synth.gaussian_weight(m, n_in, seed=60 + m, outliers=True)
    x = hq_synth.activations(B, n_in, seed=61)
    x[3] = 0.0                                                   # a zero row: s_x = 0
    x[5, :n_tile] *= 50.0                                        # a tile whose amax is an outlier
    x = hq_synth.to_bf16_f32(x)                                  # both sides see the same bf16 values
    w = ctx.encode_weights(_dev(W), 8, n_tile, SNR, seed, k)
    enc = hqo.encode_weights(W, hqo.E8, n_tile, SNR, seed, k)
    assert (w.decode_int8()[0].cpu().numpy() == enc["codes"]).all()
    y, y32, acc = w.linear_cast(_dev(x), hq.CAST_FP8_E4M3, want_f32=True, want_acc=True)
    q8, sx8 = hqo.act_quant_fp8(x, n_tile, seed)
    ref, acc_ref, acc_abs = hqo.linear_fp8(enc["codes"], enc["norms"], hqo.E8, n_tile, SNR, q8, sx8, want_acc=True)
    assert _rel_err(y32.cpu().numpy(), ref) < 1e-3
    # The fp32 tensor-core accumulators of every (tile, activation row, weight row) against the exact sums of the E4M3
    # products: fp32 summation of n_tile terms in any order errs by < n_tile * 2^-24 * sum|t| (1.5e-5 at 256); ONE operand
    # that differs by one E4M3 step moves a sum by ~ (1/16) * sum|t| / n_tile = 2.4e-4 sum|t|.  So this bar pins both
    # operands' E4M3 codes, element by element, through the production kernels.
    err = np.abs(acc.cpu().numpy().astype(np.float64) - acc_ref)
    assert (err <= 2e-5 * acc_abs + 1e-30).all(), float((err / (acc_abs + 1e-30)).max())
    ref_bf16 = hq_synth.to_bf16_f32(ref.astype(np.float32))
    tol = np.abs(ref_bf16) * 2.0 ** -7 + 1e-3 * np.sqrt((ref ** 2).mean())
    assert (np.abs(y.float().cpu().numpy() - ref_bf16) <= tol).all()
    # the INT8 cast through the same entry point is hq_linear, bit for bit
    y_i8 = w.linear_cast(_dev(x), hq.CAST_INT8)
    assert torch.equal(y_i8, w.linear(_dev(x)))
    # and the two casts differ (FP8's grid is coarser) but agree to a few per cent of the output scale
    d = (y.float() - y_i8.float()).cpu().numpy()
    rms = np.sqrt((ref ** 2).mean())
    assert 1e-4 < np.sqrt((d ** 2).mean()) / rms < 0.1
    w.free()


def test_linear_fp8_rejects_what_it_cannot_run(ctx):
    import paper_2606_23406_b200 as hq
    W = hq_synth.gaussian_weight(128, 512, seed=3)
    w = ctx.encode_weights(_dev(W), 8, 128, SNR, 1, (2, 2))
    with pytest.raises(hq.HQError):
        w.linear_cast(_dev(hq_synth.activations(8, 512, seed=1)), hq.CAST_FP8_E4M3)          # batch < 64
    wd4 = ctx.encode_weights(_dev(W), 4, 128, float(np.float32(22.5)), 1, (-1, -1))
    with pytest.raises(hq.HQError):
        wd4.linear_cast(_dev(hq_synth.activations(64, 512, seed=1)), hq.CAST_FP8_E4M3)       # not E8
    with pytest.raises(hq.HQError):
        w.linear_cast(_dev(hq_synth.activations(64, 512, seed=1)), 7)                        # no such cast
    w.free(); wd4.free()


def test_linear_fp8_config5_full_size_sampled_outputs(ctx):
    """BASELINE config 5's first GEMM at full size (8192 tokens x 4096 -> 16384, E8 4 bps, RHT tile 256) with the FP8 cast,
    the call bench.py times as roofline.large_m.fp8_e4m3: 64 sampled weight rows x 64 sampled tokens (a row's code, a
    token's activation cast and each output are independent of the rest)."""
    import paper_2606_23406_b200 as hq
    m, n_in, B, seed = 16384, 4096, 8192, 5
    rng = np.random.default_rng(9)
    W = hq_synth.gaussian_weight(m, n_in, seed=5)
    x = hq_synth.activations(B, n_in, seed=6)
    w = ctx.encode_weights(_dev(W), 8, 256, SNR, seed, (2, 2))
    y, y32 = w.linear_cast(_dev(x), hq.CAST_FP8_E4M3, want_f32=True)
    rows = np.sort(np.concatenate([rng.choice(m, 58, replace=False), [0, 127, 128, 255, m - 129, m - 1]]))
    toks = np.sort(np.concatenate([rng.choice(B, 58, replace=False), [0, 255, 256, 511, B - 257, B - 1]]))
    enc = hqo.encode_weights(W[rows], hqo.E8, 256, SNR, seed, (2, 2))
    q8, sx8 = hqo.act_quant_fp8(x[toks], 256, seed)
    ref = hqo.linear_fp8(enc["codes"], enc["norms"], hqo.E8, 256, SNR, q8, sx8)
    got = y32.cpu().numpy()[np.ix_(toks, rows)]
    assert _rel_err(got, ref) < 1e-3
    w.free()
