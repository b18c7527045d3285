"""GPU parity of the decoder-layer folds (include/hq.h hq_linear_group_fold, hq_layer_decode; §4.1
"the butterfly folds into the preceding LayerNorm", Table 10's decode shape L496-511; FORMAT R8-R10)
against the oracle.

The folds decide the INT8 activation codes, so they are checked two ways: (i) the folded call must be BIT-IDENTICAL to
the same kernel fed with the bf16 vector the oracle's RMSNorm / SiLU.mul produced (one differing activation code would
change the fp32 output), and (ii) outputs against the oracle's linear at 1e-3 / one bf16 ulp (G16).  The layer is checked
stage by stage, each oracle stage fed with the GPU's own inputs of that stage, plus one loose end-to-end comparison."""
import numpy as np
import pytest

import hq_synth
from oracle import hqo

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

SNR = float(np.float32(22.68))
SNR_KV = float(np.float32(9.68))
SEED = 11


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23406_b200 as hq
    c = hq.Context(0)
    yield c
    c.close()


def _dev(a, dtype=torch.bfloat16):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda().to(dtype)


def _host(t):
    return t.float().cpu().numpy()


def _enc(ctx, W):
    """the weight on both sides, explicit Rice k so that the weights of a group share a launch"""
    w = ctx.encode_weights(_dev(W), 8, 128, SNR, SEED, (2, 2))
    e = hqo.encode_weights(W, hqo.E8, 128, SNR, SEED, (2, 2))
    return w, e


def _oracle_linear(e, x):
    q, sx = hqo.act_quant(x[None], hqo.E8, 128, SEED)
    _, y = hqo.linear(e["codes"], e["norms"], hqo.E8, 128, SNR, q, sx, want_acc=False)
    return y[0]


def _oracle_linear_seed(e, x, seed):
    q, sx = hqo.act_quant(x[None], hqo.E8, 128, seed)
    _, y = hqo.linear(e["codes"], e["norms"], hqo.E8, 128, SNR, q, sx, want_acc=False)
    return y[0]


def _rel_err(y, ref, floor=1e-3):
    ref = np.asarray(ref, np.float64)
    rms = np.sqrt((ref ** 2).mean())
    return np.max(np.abs(np.asarray(y, np.float64) - ref) / np.maximum(np.abs(ref), floor * rms + 1e-30))


def _assert_bf16_close(y, ref, floor=1e-3):
    ref = np.asarray(ref, np.float64)
    ref_bf16 = hq_synth.to_bf16_f32(ref.astype(np.float32))
    tol = np.abs(ref_bf16) * 2.0 ** -7 + floor * np.sqrt((ref ** 2).mean())
    assert (np.abs(np.asarray(y, np.float64) - ref_bf16) <= tol).all()


@pytest.mark.parametrize("n_in,ms", [(512, (256, 128)), (4096, (384, 256, 128)), (14336, (256,))])
def test_fold_rmsnorm_bit_identical_to_unfused_and_close_to_oracle(ctx, n_in, ms):
    import paper_2606_23406_b200 as hq
    rng = np.random.default_rng(n_in)
    h = hq_synth.to_bf16_f32(rng.standard_normal(n_in, dtype=np.float32) * 2.5)
    g = hq_synth.to_bf16_f32(1.0 + 0.2 * rng.standard_normal(n_in, dtype=np.float32))
    eps = 1e-5
    pairs = [_enc(ctx, hq_synth.gaussian_weight(m, n_in, seed=30 + i, outliers=True)) for i, m in enumerate(ms)]
    ws = [p[0] for p in pairs]
    ys, y32 = ctx.linear_group_fold(ws, _dev(h), hq.FOLD_RMSNORM, aux=_dev(g), eps=eps, want_f32=True)
    x = hqo.rmsnorm_bf16(h, g, eps)                      # the oracle's normalised bf16 vector
    ys_u, y32_u = ctx.linear_group_fold(ws, _dev(x), hq.FOLD_NONE, want_f32=True)   # same kernel, same partition, plain x
    for i, (w, e) in enumerate(pairs):
        assert torch.equal(y32[i], y32_u[i]) and torch.equal(ys[i], ys_u[i])
        ref = _oracle_linear(e, x)
        assert _rel_err(_host(y32[i]), ref) < 1e-3
        _assert_bf16_close(_host(ys[i]), ref)
    for w in ws:
        w.free()


@pytest.mark.parametrize("n_in,m", [(1024, 256), (14336, 384)])
def test_fold_silu_mul_and_residual(ctx, n_in, m):
    import paper_2606_23406_b200 as hq
    rng = np.random.default_rng(n_in + 1)
    a = hq_synth.to_bf16_f32(rng.standard_normal(n_in, dtype=np.float32) * 3.0)
    b = hq_synth.to_bf16_f32(rng.standard_normal(n_in, dtype=np.float32))
    res = hq_synth.to_bf16_f32(rng.standard_normal(m, dtype=np.float32))
    w, e = _enc(ctx, hq_synth.gaussian_weight(m, n_in, seed=40, outliers=True))
    res_d = _dev(res)
    ys, y32 = ctx.linear_group_fold([w], _dev(a), hq.FOLD_SILU_MUL, aux=_dev(b), residuals=[res_d], want_f32=True)
    x = hqo.silu_mul_bf16(a, b)
    ys_u, y32_u = ctx.linear_group_fold([w], _dev(x), hq.FOLD_NONE, residuals=[res_d], want_f32=True)
    assert torch.equal(y32[0], y32_u[0]) and torch.equal(ys[0], ys_u[0])
    ref = _oracle_linear(e, x) + res.astype(np.float64)          # R10
    assert _rel_err(_host(y32[0]), ref) < 1e-3
    _assert_bf16_close(_host(ys[0]), ref)
    # without the residual the plain call equals hq_linear's own result
    y_plain = w.linear(_dev(x)[None])
    ys_n = ctx.linear_group_fold([w], _dev(x), hq.FOLD_NONE)
    assert torch.equal(ys_n[0], y_plain[0])
    # in place: the residual may alias the output
    out = res_d.clone()
    ctx.linear_group_fold([w], _dev(a), hq.FOLD_SILU_MUL, aux=_dev(b), residuals=[out], ys=[out])
    assert torch.equal(out, ys[0])
    w.free()


def test_fold_rejects_what_it_cannot_run(ctx):
    import paper_2606_23406_b200 as hq
    W = hq_synth.gaussian_weight(128, 512, seed=3)
    wd4 = ctx.encode_weights(_dev(W), 4, 128, float(np.float32(22.5)), SEED, (-1, -1))
    x = _dev(hq_synth.activations(1, 512, seed=1)[0])
    with pytest.raises(hq.HQError):
        ctx.linear_group_fold([wd4], x, hq.FOLD_RMSNORM, aux=x, eps=1e-5)      # not an E8 / 128 weight: no unfused fallback
    w, _ = _enc(ctx, W)
    with pytest.raises(hq.HQError):
        ctx.linear_group_fold([w], x, hq.FOLD_RMSNORM, aux=None)                # the fold needs its gain
    y = ctx.linear_group_fold([w], x, hq.FOLD_NONE)                             # the context still works
    assert torch.isfinite(y[0].float()).all()
    wd4.free(); w.free()


@pytest.mark.parametrize("hidden,q_heads,kv_heads,ffn,T0", [(512, 4, 2, 1024, 200), (1024, 8, 2, 3584, 333)])
def test_layer_decode_stage_by_stage(ctx, hidden, q_heads, kv_heads, ffn, T0):
    d, window, eps = 128, 32, 1e-5
    rng = np.random.default_rng(hidden)
    shapes = [(q_heads * d, hidden), (kv_heads * d, hidden), (kv_heads * d, hidden), (hidden, q_heads * d),
              (ffn, hidden), (ffn, hidden), (hidden, ffn)]
    # weight scale ~ 1/sqrt(n_in) keeps every stage's activations O(1), like a trained layer
    pairs = [_enc(ctx, hq_synth.gaussian_weight(m, n, seed=50 + i, outliers=True, std=1.0 / np.sqrt(n)))
             for i, (m, n) in enumerate(shapes)]
    ws = [p[0] for p in pairs]
    eq, ek, ev, eo, eg, eu, ed = [p[1] for p in pairs]
    g1 = hq_synth.to_bf16_f32(1.0 + 0.1 * rng.standard_normal(hidden, dtype=np.float32))
    g2 = hq_synth.to_bf16_f32(1.0 + 0.1 * rng.standard_normal(hidden, dtype=np.float32))
    h = hq_synth.to_bf16_f32(rng.standard_normal(hidden, dtype=np.float32) * 1.5)
    K0 = hq_synth.kv_tokens(T0, kv_heads, d, seed=4)
    V0 = hq_synth.kv_tokens(T0, kv_heads, d, seed=5)
    kv = ctx.kv_create(kv_heads, d, 512, 8, SNR_KV, (0, 0), SEED, rotation=1, dither=1, window=window)
    kv.append(_dev(K0), _dev(V0))
    g1_d, g2_d = _dev(g1), _dev(g2)
    layer = ctx.layer(*ws, g1_d, g2_d, eps, kv, q_heads)
    h_out = _host(layer.decode(_dev(h)))
    torch.cuda.synchronize()
    got = {n: _host(layer.scratch_tensor(n)) for n in ("q", "k", "v", "a", "h2", "gate", "up")}

    # stage 1: q, k, v = W RMSNorm(h)
    x1 = hqo.rmsnorm_bf16(h, g1, eps)
    for name, e in (("q", eq), ("k", ek), ("v", ev)):
        _assert_bf16_close(got[name], _oracle_linear(e, x1))
    # stage 2: the cache took the GPU's k, v as token T0 (codes bit-exact), attention over T0 + 1 tokens for the GPU's q
    K = np.concatenate([K0, got["k"].reshape(1, kv_heads, d)]); V = np.concatenate([V0, got["v"].reshape(1, kv_heads, d)])
    ck, nk, _ = hqo.kv_quantize(K, 0, 0, hqo.E8, SNR_KV, 1, 1, SEED)
    cv, nv, _ = hqo.kv_quantize(V, 0, 1, hqo.E8, SNR_KV, 1, 1, SEED)
    assert (kv.decode_int8(0, T0, 1).cpu().numpy() == ck[T0:]).all()
    assert (kv.decode_int8(1, T0, 1).cpu().numpy() == cv[T0:]).all()
    Kh = hqo.kv_reconstruct(ck, nk, 0, 0, hqo.E8, SNR_KV, 1, 1, SEED)
    Vh = hqo.kv_reconstruct(cv, nv, 0, 1, hqo.E8, SNR_KV, 1, 1, SEED)
    a_ref = hqo.attend(Kh, Vh, K, V, window=window, q=got["q"].reshape(q_heads, d))
    _assert_bf16_close(got["a"], a_ref.reshape(-1), floor=2e-2)          # attention floor: DESIGN.md G16
    # stage 3: h2 = h + W_o a
    _assert_bf16_close(got["h2"], _oracle_linear(eo, got["a"]) + h.astype(np.float64))
    # stage 4: gate, up = W RMSNorm(h2)
    x2 = hqo.rmsnorm_bf16(got["h2"], g2, eps)
    _assert_bf16_close(got["gate"], _oracle_linear(eg, x2))
    _assert_bf16_close(got["up"], _oracle_linear(eu, x2))
    # stage 5: h_out = h2 + W_down (silu(gate) * up)
    z = hqo.silu_mul_bf16(got["gate"], got["up"])
    _assert_bf16_close(h_out, _oracle_linear(ed, z) + got["h2"].astype(np.float64))

    # end to end, the oracle on its own intermediates (bf16 at every stage boundary): loose, rounding differences propagate
    qo, ko, vo = [hq_synth.to_bf16_f32(_oracle_linear(e, x1).astype(np.float32)) for e in (eq, ek, ev)]
    K2 = np.concatenate([K0, ko.reshape(1, kv_heads, d)]); V2 = np.concatenate([V0, vo.reshape(1, kv_heads, d)])
    ck2, nk2, _ = hqo.kv_quantize(K2, 0, 0, hqo.E8, SNR_KV, 1, 1, SEED)
    cv2, nv2, _ = hqo.kv_quantize(V2, 0, 1, hqo.E8, SNR_KV, 1, 1, SEED)
    ao = hqo.attend(hqo.kv_reconstruct(ck2, nk2, 0, 0, hqo.E8, SNR_KV, 1, 1, SEED),
                    hqo.kv_reconstruct(cv2, nv2, 0, 1, hqo.E8, SNR_KV, 1, 1, SEED), K2, V2, window=window,
                    q=qo.reshape(q_heads, d))
    ao = hq_synth.to_bf16_f32(ao.reshape(-1).astype(np.float32))
    h2o = hq_synth.to_bf16_f32((_oracle_linear(eo, ao) + h).astype(np.float32))
    x2o = hqo.rmsnorm_bf16(h2o, g2, eps)
    go, uo = [hq_synth.to_bf16_f32(_oracle_linear(e, x2o).astype(np.float32)) for e in (eg, eu)]
    ho = _oracle_linear(ed, hqo.silu_mul_bf16(go, uo)) + h2o
    assert np.sqrt(np.mean((h_out - ho) ** 2)) / np.sqrt(np.mean(ho ** 2)) < 2e-2

    # a second step advances the cache position
    layer.decode(_dev(h))
    assert kv.export()["n_tokens"] == T0 + 2
    kv.free()
    for w in ws:
        w.free()


def test_layer_decode_full_size_llama_shapes_sampled_rows(ctx):
    """The configuration bench.py's roofline.layer_step times (Llama-3.1-8B-shaped layer: hidden 4096, 32 query / 8 KV
    heads of 128, FFN 14336; E8 4 bps weights, E8 2 bps cache with signs rotation, dither and a 32-token window), one
    decode step after a 2048-token prefill, stage by stage.  The linears are checked on 96 sampled rows each (a row's
    code and output are independent of the other rows, so the oracle encodes and contracts only those), attention in
    full."""
    hidden, q_heads, kv_heads, ffn, d, T0, window, eps, seed = 4096, 32, 8, 14336, 128, 2048, 32, 1e-5, 3
    rng = np.random.default_rng(77)
    names = ["q", "k", "v", "o", "gate", "up", "down"]
    Ws = {n: hq_synth.llama_weight(1, n) for n in names}
    ws = {n: ctx.encode_weights(_dev(Ws[n]), 8, 128, SNR, seed, (2, 2)) for n in names}
    g1 = hq_synth.to_bf16_f32(1.0 + 0.1 * rng.standard_normal(hidden, dtype=np.float32))
    g2 = hq_synth.to_bf16_f32(1.0 + 0.1 * rng.standard_normal(hidden, dtype=np.float32))
    h = hq_synth.to_bf16_f32(rng.standard_normal(hidden, dtype=np.float32))
    K0 = hq_synth.kv_tokens(T0, kv_heads, d, seed=4); V0 = hq_synth.kv_tokens(T0, kv_heads, d, seed=5)
    kv = ctx.kv_create(kv_heads, d, T0 + 64, 8, SNR_KV, (0, 0), seed, rotation=1, dither=1, window=window)
    kv.append(_dev(K0), _dev(V0))
    layer = ctx.layer(*[ws[n] for n in names], _dev(g1), _dev(g2), eps, kv, q_heads)
    h_out = _host(layer.decode(_dev(h)))
    torch.cuda.synchronize()
    got = {n: _host(layer.scratch_tensor(n)) for n in ("q", "k", "v", "a", "h2", "gate", "up")}

    def check_rows(name, x, out, res=None):
        W = Ws[name]; m = W.shape[0]
        rows = np.sort(np.concatenate([rng.choice(m, 90, replace=False), [0, 1, 127, 128, m - 2, m - 1]]))
        e = hqo.encode_weights(W[rows], hqo.E8, 128, SNR, seed, (2, 2))
        ref = _oracle_linear_seed(e, x, seed)
        if res is not None:
            ref = ref + res[rows].astype(np.float64)
        ref_bf16 = hq_synth.to_bf16_f32(ref.astype(np.float32))
        tol = np.abs(ref_bf16) * 2.0 ** -7 + 1e-3 * np.sqrt((ref ** 2).mean())
        assert (np.abs(out[rows].astype(np.float64) - ref_bf16) <= tol).all(), name

    x1 = hqo.rmsnorm_bf16(h, g1, eps)
    for n in ("q", "k", "v"):
        check_rows(n, x1, got[n])
    K = np.concatenate([K0, got["k"].reshape(1, kv_heads, d)]); V = np.concatenate([V0, got["v"].reshape(1, kv_heads, d)])
    ck, nk, _ = hqo.kv_quantize(K, 0, 0, hqo.E8, SNR_KV, 1, 1, seed)
    cv, nv, _ = hqo.kv_quantize(V, 0, 1, hqo.E8, SNR_KV, 1, 1, seed)
    assert (kv.decode_int8(0, T0, 1).cpu().numpy() == ck[T0:]).all() and (kv.decode_int8(1, T0, 1).cpu().numpy() == cv[T0:]).all()
    a_ref = hqo.attend(hqo.kv_reconstruct(ck, nk, 0, 0, hqo.E8, SNR_KV, 1, 1, seed),
                       hqo.kv_reconstruct(cv, nv, 0, 1, hqo.E8, SNR_KV, 1, 1, seed), K, V, window=window,
                       q=got["q"].reshape(q_heads, d))
    _assert_bf16_close(got["a"], a_ref.reshape(-1), floor=2e-2)
    check_rows("o", got["a"], got["h2"], res=h)
    x2 = hqo.rmsnorm_bf16(got["h2"], g2, eps)
    check_rows("gate", x2, got["gate"]); check_rows("up", x2, got["up"])
    check_rows("down", hqo.silu_mul_bf16(got["gate"], got["up"]), h_out, res=got["h2"])
    kv.free()
    for w in ws.values():
        w.free()


def test_fold_edge_cases(ctx):
    """Degenerate inputs of the folds: an all-zero residual stream (RMSNorm must give zeros, not NaN: eps), gates far outside
    the exponential's clamp (+-100: silu -> 0 or the identity), a zero second factor, and a vector with one huge element
    (the tree sum of squares and the bf16 rounding of tiny normalised values)."""
    import paper_2606_23406_b200 as hq
    n_in, m = 1024, 256
    w, e = _enc(ctx, hq_synth.gaussian_weight(m, n_in, seed=41, outliers=True))
    g = hq_synth.to_bf16_f32(np.linspace(0.5, 1.5, n_in).astype(np.float32))
    # zero vector
    ys, y32 = ctx.linear_group_fold([w], _dev(np.zeros(n_in, np.float32)), hq.FOLD_RMSNORM, aux=_dev(g), eps=1e-5, want_f32=True)
    assert (y32[0] == 0).all() and torch.isfinite(ys[0].float()).all()
    # one huge element
    h = hq_synth.to_bf16_f32(np.random.default_rng(5).standard_normal(n_in, dtype=np.float32) * 1e-2)
    h[77] = 3.0e4
    h = hq_synth.to_bf16_f32(h)                                   # both sides see the same bf16 values
    ys, y32 = ctx.linear_group_fold([w], _dev(h), hq.FOLD_RMSNORM, aux=_dev(g), eps=1e-6, want_f32=True)
    x = hqo.rmsnorm_bf16(h, g, 1e-6)
    _, y32_u = ctx.linear_group_fold([w], _dev(x), hq.FOLD_NONE, want_f32=True)
    assert torch.equal(y32[0], y32_u[0])
    assert _rel_err(_host(y32[0]), _oracle_linear(e, x)) < 1e-3
    # gates beyond the clamp, zero factors
    a = hq_synth.to_bf16_f32(np.random.default_rng(6).standard_normal(n_in, dtype=np.float32) * 3.0)
    b = hq_synth.to_bf16_f32(np.random.default_rng(7).standard_normal(n_in, dtype=np.float32))
    a[:8] = [100.0, -100.0, 88.0, -88.0, 87.5, -87.5, 0.0, -0.0]
    b[8:16] = 0.0
    a, b = hq_synth.to_bf16_f32(a), hq_synth.to_bf16_f32(b)
    ys, y32 = ctx.linear_group_fold([w], _dev(a), hq.FOLD_SILU_MUL, aux=_dev(b), want_f32=True)
    x = hqo.silu_mul_bf16(a, b)
    assert np.isfinite(x).all()
    _, y32_u = ctx.linear_group_fold([w], _dev(x), hq.FOLD_NONE, want_f32=True)
    assert torch.equal(y32[0], y32_u[0])
    assert _rel_err(_host(y32[0]), _oracle_linear(e, x)) < 1e-3
    w.free()
