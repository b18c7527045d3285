"""GPU parity: libhq.so (through the C ABI / Python binding) against the oracle, element by element.

Bars (BASELINE.json north_star): bit-exact bitstreams, lattice indices, INT8 points, INT32
accumulators; fp32 RHT outputs within 1e-5; fp32 outputs within 1e-3 (G16) and bf16 within one bf16 ulp.
"""
import numpy as np
import pytest

import hq_synth
from oracle import hqo

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

def f32(v):
    """hq_codec_config.snr_db is a C float: hand both sides the same representable value."""
    return float(np.float32(v))


SNR_4BPS = {hqo.E8: f32(22.68), hqo.D4: f32(22.5), hqo.A2: f32(22.2), hqo.Z: f32(21.9)}


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23406_b200 as hq
    c = hq.Context(0)
    yield c
    c.close()


def _dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t.to(dtype) if dtype is not None else t


def _rel_err(y, ref, floor=1e-3):
    """max |y - ref| / max(|ref|, floor * rms(ref)) (G16).  Linear outputs: floor 1e-3.  Attention outputs:
    floor 2e-2 - an element of a softmax-weighted sum over T cached vectors that cancels to |ref| << rms still carries
    the absolute fp32 rounding error of the whole sum (measured 2e-5 rms at T = 32768)."""
    ref = np.asarray(ref, np.float64)
    rms = np.sqrt((ref ** 2).mean())
    return np.max(np.abs(np.asarray(y, np.float64) - ref) / np.maximum(np.abs(ref), floor * rms + 1e-30))


def _assert_bf16_close(y, ref):
    """bf16 output within one bf16 ulp of bf16(ref), plus the fp32 tolerance near zero (G16)."""
    ref = np.asarray(ref, np.float64)
    ref_bf16 = torch.from_numpy(ref.astype(np.float32)).to(torch.bfloat16).float().numpy()
    tol = np.abs(ref_bf16) * 2.0 ** -7 + 1e-3 * np.sqrt((ref ** 2).mean())
    assert (np.abs(y.float().cpu().numpy() - ref_bf16) <= tol).all()


def _check_weight_bitstream(ctx, W, lattice, n_tile, snr, seed, k=(-1, -1), bf16=False):
    snr = f32(snr)
    enc = hqo.encode_weights(W, lattice, n_tile, snr, seed, k)
    w = ctx.encode_weights(_dev(W, torch.bfloat16 if bf16 else None), lattice, n_tile, snr, seed, k)
    assert tuple(w.k) == tuple(int(v) for v in enc["k"])
    blob, goff = w.export()
    assert (goff == enc["group_off"]).all()
    assert blob.size == enc["blob"].size
    if not (blob == enc["blob"]).all():
        bad = np.flatnonzero(blob != enc["blob"])
        raise AssertionError(f"bitstream differs at {bad.size} bytes, first {bad[:8]}")
    codes, norms = w.decode_int8()
    assert (codes.cpu().numpy() == enc["codes"]).all()
    assert (norms.cpu().numpy().view(np.uint16) == enc["norms"]).all()
    assert w.info.payload_bits == enc["payload_bits"] and w.info.clamp_count == enc["clamps"]
    return w, enc


def test_config1_bitstream_codes_linear(ctx):
    """BASELINE config 1: W 256x256 fp32 N(0,0.02^2) seed 0, tile 64, E8 at 4 bps, x fp32 N(0,1)."""
    W, x = hq_synth.c1_weight()
    snr, seed = SNR_4BPS[hqo.E8], 1234
    w, enc = _check_weight_bitstream(ctx, W, hqo.E8, 64, snr, seed)
    q_o, sx_o, u_o = hqo.act_quant(x, hqo.E8, 64, seed, want_u=True)
    q, s_x, u = w.act_quant(_dev(x), want_u=True)
    assert (q.cpu().numpy() == q_o).all() and (s_x.cpu().numpy() == sx_o).all()
    assert (u.cpu().numpy() == u_o).all()                       # canonical butterfly: identical bits
    d = hqo.signs(seed, 1, 256)
    for kt in range(4):                                          # fp32 RHT output within 1e-5 of the definition
        ref = hqo.rht_dense_f64(x[0, kt * 64:(kt + 1) * 64].astype(np.float64), d[kt * 64:(kt + 1) * 64])
        assert np.max(np.abs(u.cpu().numpy()[0, kt * 64:(kt + 1) * 64] - ref)) < 1e-5 * np.abs(ref).max()
    acc_o, y_o = hqo.linear(enc["codes"], enc["norms"], hqo.E8, 64, snr, q_o, sx_o)
    y, y32, acc = w.linear(_dev(x), want_f32=True, want_acc=True)
    assert (acc.cpu().numpy() == acc_o).all()
    assert _rel_err(y32.cpu().numpy(), y_o) < 1e-3
    _assert_bf16_close(y, y_o)
    w.free()


@pytest.mark.parametrize("lattice", [hqo.E8, hqo.D4, hqo.A2, hqo.Z])
@pytest.mark.parametrize("n_tile,m,bps_snr", [(64, 200, 16.5), (128, 384, 22.7), (256, 130, 28.7)])
def test_bitstream_all_lattices_tiles_ragged_rows(ctx, lattice, n_tile, m, bps_snr):
    W = hq_synth.gaussian_weight(m, 1024, seed=11 * lattice + m, outliers=True)
    w, enc = _check_weight_bitstream(ctx, W, lattice, n_tile, bps_snr, seed=77, bf16=True)
    w.free()


def test_explicit_k_and_degenerate_tiles(ctx):
    W = hq_synth.gaussian_weight(256, 512, seed=5)
    W[3] = 0.0                                  # zero rows -> rho = 0 (G18)
    W[:, 128:256] = 0.0                         # a zero K-tile for every row
    d = hqo.signs(3, 1, 512)[256:384].astype(np.float32)      # a row whose RHT is n*e_5: all energy in one
    had = np.array([(-1.0) ** bin(i & 5).count("1") for i in range(128)], np.float32)
    W[7, :] = 0.0; W[7, 256:384] = d * had * 0.5                # coordinate -> INT8 pre-clamp (G8)
    for k in ((0, 0), (3, 3)):
        w, enc = _check_weight_bitstream(ctx, W, hqo.E8, 128, 28.7, seed=3, k=k)
        assert enc["clamps"] > 0
        w.free()
    w, enc = _check_weight_bitstream(ctx, W, hqo.D4, 64, 28.7, seed=3, k=(2, 1))   # partial R chunks
    w.free()


@pytest.mark.parametrize("lattice,n_tile", [(hqo.E8, 128), (hqo.E8, 256), (hqo.D4, 128), (hqo.A2, 64), (hqo.Z, 128)])
@pytest.mark.parametrize("B", [1, 16, 40, 130])
def test_linear_acc_exact_and_outputs(ctx, lattice, n_tile, B):
    m, n_in, snr, seed = 300, 1024, SNR_4BPS[lattice], 21
    W = hq_synth.gaussian_weight(m, n_in, seed=lattice + 100, outliers=True)
    x = hq_synth.activations(B, n_in, seed=B + 7)
    enc = hqo.encode_weights(W, lattice, n_tile, snr, seed)
    w = ctx.encode_weights(_dev(W, torch.bfloat16), lattice, n_tile, snr, seed)
    q_o, sx_o = hqo.act_quant(x, lattice, n_tile, seed)
    acc_o, y_o = hqo.linear(enc["codes"], enc["norms"], lattice, n_tile, snr, q_o, sx_o)
    y, y32, acc = w.linear(_dev(x, torch.bfloat16), want_f32=True, want_acc=True)
    assert (acc.cpu().numpy() == acc_o).all()
    assert _rel_err(y32.cpu().numpy(), y_o) < 1e-3
    _assert_bf16_close(y, y_o)
    w.free()


def test_e8_fast_kernel_falls_back_on_long_quotients_and_ragged_blocks(ctx):
    """E8 / tile 128 runs the SWAR decoder; rows with a unary quotient >= 16 or more U words than it holds in
    registers must come out identical through its generic fallback.  k = 0 at 5 bps makes such rows the rule;
    the clamp row (all energy in one coordinate, G8) has a quotient near 250; m = 200 leaves absent rows."""
    m, n_in, snr, seed = 200, 512, f32(28.73), 3
    W = hq_synth.gaussian_weight(m, n_in, seed=5)
    W[3] = 0.0
    d = hqo.signs(seed, 1, n_in)[256:384].astype(np.float32)
    had = np.array([(-1.0) ** bin(i & 5).count("1") for i in range(128)], np.float32)
    W[7, :] = 0.0; W[7, 256:384] = d * had * 0.5
    for k in ((0, 0), (1, 1), (3, 3)):
        enc = hqo.encode_weights(W, hqo.E8, 128, snr, seed, k)
        w = ctx.encode_weights(_dev(W), hqo.E8, 128, snr, seed, k)
        for B in (1, 5):
            x = hq_synth.activations(B, n_in, seed=40 + B)
            q_o, sx_o = hqo.act_quant(x, hqo.E8, 128, seed)
            acc_o, y_o = hqo.linear(enc["codes"], enc["norms"], hqo.E8, 128, snr, q_o, sx_o)
            y, y32, acc = w.linear(_dev(x, torch.bfloat16), want_f32=True, want_acc=True)
            assert (acc.cpu().numpy() == acc_o).all()
            assert _rel_err(y32.cpu().numpy(), y_o) < 1e-3
        w.free()


@pytest.mark.parametrize("n_tile", [128, 256])
@pytest.mark.parametrize("B,m,k", [(600, 300, (-1, -1)), (512, 200, (0, 0)), (1030, 130, (3, 3))])
def test_linear_large_m_path(ctx, B, m, k, n_tile):
    """From 512 activation rows hq_linear decodes the weights once into an operand-layout scratch copy and runs the
    warp-specialised GEMM (hq_linear_large.cuh), at RHT tiles of 128 and 256 (two operand chunks per accumulator
    drain): ragged row block, ragged batch tile, several tiles per CTA, rows that
    take the decoder's generic fallback (k = 0 at 5 bps; a clamp row), an absent row; and the weights of a group."""
    n_in, seed = 1024, 17
    snr = f32(28.73) if k == (0, 0) else SNR_4BPS[hqo.E8]
    W = hq_synth.gaussian_weight(m, n_in, seed=m, outliers=True)
    W[3] = 0.0
    d = hqo.signs(seed, 1, n_in)[256:384].astype(np.float32)
    had = np.array([(-1.0) ** bin(i & 5).count("1") for i in range(128)], np.float32)
    W[7, :] = 0.0; W[7, 256:384] = d * had * 0.5               # at tile 128 this row is n * e_5 after the RHT (clamp, G8)
    x = hq_synth.activations(B, n_in, seed=B)
    enc = hqo.encode_weights(W, hqo.E8, n_tile, snr, seed, k)
    w = ctx.encode_weights(_dev(W), hqo.E8, n_tile, snr, seed, k)
    q_o, sx_o = hqo.act_quant(x, hqo.E8, n_tile, seed)
    acc_o, y_o = hqo.linear(enc["codes"], enc["norms"], hqo.E8, n_tile, snr, q_o, sx_o)
    xd = _dev(x, torch.bfloat16)
    y, y32, _ = w.linear(xd, want_f32=True)
    assert _rel_err(y32.cpu().numpy(), y_o) < 1e-3
    _assert_bf16_close(y, y_o)
    # the INT32 accumulators of THIS path (every K-tile's TMEM tile as the epilogue drains it), bit for bit
    y_f, y32_f, acc = w.linear(xd, want_f32=True, want_acc=True)
    assert (acc.cpu().numpy() == acc_o).all()
    assert torch.equal(y32_f, y32) and torch.equal(y_f, y)
    ys, y32s = ctx.linear_group([w, w], xd, want_f32=True)
    assert torch.equal(y32s[0], y32) and torch.equal(y32s[1], y32) and torch.equal(ys[1], y)
    w.free()


def test_linear_group_is_bit_identical_to_separate_calls(ctx):
    """hq_linear_group (q/k/v-style: several weights, one x, one fused launch) against hq_linear per weight and
    against the oracle for the first weight."""
    n_in, snr, seed = 1024, SNR_4BPS[hqo.E8], 11
    shapes = [384, 130, 256]
    Ws = [hq_synth.gaussian_weight(m, n_in, seed=70 + i, outliers=True) for i, m in enumerate(shapes)]
    ws = [ctx.encode_weights(_dev(W, torch.bfloat16), hqo.E8, 128, snr, seed, (2, 2)) for W in Ws]
    for B in (1, 16, 33, 130):
        x = _dev(hq_synth.activations(B, n_in, seed=B), torch.bfloat16)
        ys, y32s = ctx.linear_group(ws, x, want_f32=True)
        ys2, y32s2 = ctx.linear_group(ws, x, want_f32=True)
        for w, y, y32, y_again in zip(ws, ys, y32s, y32s2):
            assert torch.equal(y32, y_again)                               # deterministic: a fixed summation order
            y1, y1_32, _ = w.linear(x, want_f32=True)
            if B == 1:   # the batch-1 kernel cuts K where the launch's flat tile partition falls: equal to fp32 rounding
                assert _rel_err(y32.cpu().numpy(), y1_32.cpu().numpy().astype(np.float64)) < 1e-5
            else:
                assert torch.equal(y, y1) and torch.equal(y32, y1_32)
    enc = hqo.encode_weights(Ws[0], hqo.E8, 128, snr, seed, (2, 2))
    xh = hq_synth.activations(4, n_in, seed=3)
    q_o, sx_o = hqo.act_quant(xh, hqo.E8, 128, seed)
    _, y_o = hqo.linear(enc["codes"], enc["norms"], hqo.E8, 128, snr, q_o, sx_o)
    ys, y32s = ctx.linear_group(ws, _dev(xh, torch.bfloat16), want_f32=True)
    assert _rel_err(y32s[0].cpu().numpy(), y_o) < 1e-3
    # weights that cannot share a launch (different seed -> different RHT signs) still give the right answers
    w_other = ctx.encode_weights(_dev(Ws[1], torch.bfloat16), hqo.E8, 128, snr, seed + 1, (2, 2))
    ys = ctx.linear_group([ws[0], w_other], _dev(xh, torch.bfloat16))
    assert torch.equal(ys[1], w_other.linear(_dev(xh, torch.bfloat16)))
    for w in ws + [w_other]:
        w.free()


# ------------------------------------------------------------------------------------------ KV
def _oracle_kv_container(K, V, lattice, snr, k, rotation, dither, seed, chunks):
    """Oracle-side container for tokens appended in `chunks` (list of token counts)."""
    T, H, d = K.shape
    Rbits = hqo.rbits(lattice, d, k)
    rem = np.zeros((2, H, T * Rbits // 32 + 8), np.uint32)
    una = np.zeros((2, H, T * d * 16 // 32 + 64), np.uint32)             # room for any rate the tests use
    ulen = np.zeros((2, H, T), np.uint16); norm = np.zeros((2, H, T), np.uint16)
    codes_all = np.zeros((2, T, H, d), np.int8)
    upos = np.zeros((2, H), np.int64)
    t0 = 0
    for n in chunks:
        for role, X in enumerate((K, V)):
            codes, norms, _ = hqo.kv_quantize(X[t0:t0 + n], t0, role, lattice, snr, rotation, dither, seed)
            codes_all[role, t0:t0 + n] = codes
            norm[role, :, t0:t0 + n] = norms.T
            for h in range(H):
                pos, ul = hqo.kv_pack_head(codes, h, lattice, k, rem[role, h], una[role, h], int(upos[role, h]), t0=t0)
                ulen[role, h, t0:t0 + n] = ul
                upos[role, h] = pos
        t0 += n
    return dict(rem=rem, una=una, ulen=ulen, norm=norm, codes=codes_all, upos=upos)


@pytest.mark.parametrize("lattice,snr,k,dither,rotation", [
    (hqo.E8, 9.68, (0, 0), 1, 1),      # config 4: E8 at 2 bps, signs rotation, dither on
    (hqo.E8, 22.68, (2, 2), 0, 0),
    (hqo.D4, 16.3, (1, 0), 1, 1),
    (hqo.A2, 16.0, (1, 1), 1, 0),
    (hqo.Z, 15.7, (1, 1), 1, 1),
])
def test_kv_append_container_exact(ctx, lattice, snr, k, dither, rotation):
    T, H, d, seed, snr = 300, 2, 128, 99, f32(snr)
    K = hq_synth.kv_tokens(T, H, d, seed=4); V = hq_synth.kv_tokens(T, H, d, seed=5)
    chunks = [257, 1, 1, 41]                                       # bulk prefill, single-token steps, ragged
    ora = _oracle_kv_container(K, V, lattice, snr, k, rotation, dither, seed, chunks)
    kv = ctx.kv_create(H, d, 512, lattice, snr, k, seed, rotation=rotation, dither=dither, window=32)
    t0 = 0
    for n in chunks:
        kv.append(_dev(K[t0:t0 + n], torch.bfloat16), _dev(V[t0:t0 + n], torch.bfloat16))
        t0 += n
    ex = kv.export()
    assert ex["n_tokens"] == T
    assert (ex["ulen"][:, :, :T] == ora["ulen"]).all()
    assert (ex["norm"][:, :, :T] == ora["norm"]).all()
    assert (ex["upos"] == ora["upos"]).all()
    nr = min(ex["rem"].shape[2], ora["rem"].shape[2]); nu = min(ex["una"].shape[2], ora["una"].shape[2])
    assert (ex["rem"][:, :, :nr] == ora["rem"][:, :, :nr]).all()
    assert (ex["una"][:, :, :nu] == ora["una"][:, :, :nu]).all()
    for role in range(2):
        for h in range(H):                                         # block offsets = prefix sums of ulen
            cs = np.concatenate([[0], np.cumsum(ora["ulen"][role, h].astype(np.int64))])
            for b in range((T + 127) // 128):
                assert ex["blk_off"][role, h, b] == cs[128 * b]
        codes = kv.decode_int8(role, 0, T).cpu().numpy()
        assert (codes == ora["codes"][role]).all()
    kv.free()


@pytest.mark.parametrize("lattice,snr,k,dither,T,window", [
    (hqo.E8, 9.68, (0, 0), 1, 700, 32),
    (hqo.E8, 22.68, (2, 2), 0, 200, 0),
    (hqo.A2, 16.0, (1, 1), 1, 130, 32),
    (hqo.E8, 9.68, (0, 0), 1, 20, 32),       # everything inside the window: exact bf16 attention (G15)
])
def test_attend_matches_oracle_long_way(ctx, lattice, snr, k, dither, T, window):
    H, d, QH, seed, rotation, snr = 2, 128, 8, 5, 1, f32(snr)
    K = hq_synth.kv_tokens(T, H, d, seed=14); V = hq_synth.kv_tokens(T, H, d, seed=15)
    q = hq_synth.activations(QH, d, seed=16)
    kv = ctx.kv_create(H, d, 1024, lattice, snr, k, seed, rotation=rotation, dither=dither, window=window)
    kv.append(_dev(K, torch.bfloat16), _dev(V, torch.bfloat16))
    out, o32 = kv.attend(_dev(q, torch.bfloat16), want_f32=True)
    ck, nk, _ = hqo.kv_quantize(K, 0, 0, lattice, snr, rotation, dither, seed)
    cv, nv, _ = hqo.kv_quantize(V, 0, 1, lattice, snr, rotation, dither, seed)
    Kh = hqo.kv_reconstruct(ck, nk, 0, 0, lattice, snr, rotation, dither, seed)
    Vh = hqo.kv_reconstruct(cv, nv, 0, 1, lattice, snr, rotation, dither, seed)
    ref = hqo.attend(Kh, Vh, K, V, window=window, q=q)
    assert _rel_err(o32.cpu().numpy(), ref, floor=2e-2) < 1e-3
    _assert_bf16_close(out, ref)
    kv.free()


def test_attend_several_blocks_per_split_matches_oracle(ctx):
    """64 KV heads leave 148*4/64 = 9 splits per head: 3600 tokens = 28 blocks of 128 -> 4 blocks per split, so the
    running-max rescale INSIDE a split (online softmax, L178) is compared with the oracle's long way round."""
    T, H, d, QH, seed, snr = 3600, 64, 128, 64, 6, f32(9.68)
    K = hq_synth.kv_tokens(T, H, d, seed=24); V = hq_synth.kv_tokens(T, H, d, seed=25)
    K[1500:1510] *= 3.0                                            # a late block raises the running max
    K = hq_synth.to_bf16_f32(K)
    q = hq_synth.activations(QH, d, seed=26)
    kv = ctx.kv_create(H, d, 4096, hqo.E8, snr, (0, 0), seed, rotation=1, dither=1, window=32)
    kv.append(_dev(K, torch.bfloat16), _dev(V, torch.bfloat16))
    out, o32 = kv.attend(_dev(q, torch.bfloat16), want_f32=True)
    ck, nk, _ = hqo.kv_quantize(K, 0, 0, hqo.E8, snr, 1, 1, seed)
    cv, nv, _ = hqo.kv_quantize(V, 0, 1, hqo.E8, snr, 1, 1, seed)
    Kh = hqo.kv_reconstruct(ck, nk, 0, 0, hqo.E8, snr, 1, 1, seed)
    Vh = hqo.kv_reconstruct(cv, nv, 0, 1, hqo.E8, snr, 1, 1, seed)
    ref = hqo.attend(Kh, Vh, K, V, window=32, q=q)
    assert _rel_err(o32.cpu().numpy(), ref, floor=2e-2) < 1e-3
    _assert_bf16_close(out, ref)
    kv.free()


def test_kv_u_stream_overflow_is_detected_never_written_and_sticky(ctx):
    """a legal config whose unary bits outrun the U stream.  E8 at 22.68 dB with k = (0, 0) costs ~6.4 unary
    bits per scalar.  (i) the default capacity holds a full cache of it, container bit-exact; (ii) with a small
    caller-given capacity the vectors that do not fit are not written (the neighbouring head's stream and the words
    past the stream stay as the oracle has them), and the cache turns HQ_ERR_FORMAT on the next call and stays so."""
    import paper_2606_23406_b200 as hq
    T, H, d, seed, snr, k = 256, 2, 128, 31, f32(22.68), (0, 0)
    K = hq_synth.kv_tokens(T, H, d, seed=4); V = hq_synth.kv_tokens(T, H, d, seed=5)
    ora = _oracle_kv_container(K, V, hqo.E8, snr, k, 1, 1, seed, [T])
    assert ora["upos"].min() > 5.0 * T * d                          # really more than the old 4 bits / scalar
    kv = ctx.kv_create(H, d, T, hqo.E8, snr, k, seed, rotation=1, dither=1, window=0)
    kv.append(_dev(K, torch.bfloat16), _dev(V, torch.bfloat16))
    ex = kv.export()
    assert (ex["upos"] == ora["upos"]).all()
    nu = min(ex["una"].shape[2], ora["una"].shape[2])
    assert (ex["una"][:, :, :nu] == ora["una"][:, :, :nu]).all()
    kv.free()
    cap = int(ora["upos"].min()) // 2 // 32 * 32                    # room for about half of the tokens
    for chunks in ([T], [1] * 200):                                 # the bulk kernels and the one-token kernel
        kv = ctx.kv_create(H, d, T, hqo.E8, snr, k, seed, rotation=1, dither=1, window=0, una_capacity_bits=cap)
        t0, raised = 0, False
        try:
            for n in chunks:
                kv.append(_dev(K[t0:t0 + n], torch.bfloat16), _dev(V[t0:t0 + n], torch.bfloat16))
                t0 += n
                torch.cuda.synchronize()
        except hq.HQError:
            raised = True
        torch.cuda.synchronize()
        if not raised:                                              # the bulk call itself is asynchronous: the NEXT call reports
            with pytest.raises(hq.HQError):
                kv.attend(_dev(hq_synth.activations(8, d, seed=1), torch.bfloat16))
        with pytest.raises(hq.HQError):                             # sticky
            kv.append(_dev(K[:1], torch.bfloat16), _dev(V[:1], torch.bfloat16))
        with pytest.raises(hq.HQError):
            kv.export()
        # nothing was written outside [0, cap) of any stream: compare raw memory with the oracle's prefix
        una_words = cap // 32 + 4
        raw = None                                                  # the cache's `una` allocation, found by its size
        for obj in list(ctx._live.values()):
            if obj.numel() == 2 * H * una_words * 4:
                raw = obj.cpu().numpy().view(np.uint32).reshape(2, H, una_words)
        assert raw is not None
        for role in range(2):
            for h in range(H):
                cs = np.concatenate([[0], np.cumsum(ora["ulen"][role, h].astype(np.int64))])
                n_fit = int(np.searchsorted(cs, cap - 64, side="right")) - 1      # tokens whose U-section ends inside
                full_words = int(cs[n_fit]) // 32
                assert (raw[role, h, :full_words] == ora["una"][role, h, :full_words]).all()
                assert (raw[role, h, (cap - 64) // 32 + 1:] == 0).all()          # the guard zone is untouched
        kv.free()


def test_weight_export_host_import_round_trip_and_layout_checks(ctx):
    """SURVEY §5 checkpoint: the encoded weight leaves the process as host data and comes back; the imported handle
    is bit-identical in hq_linear / hq_decode_int8; a blob that fails the layout checks is HQ_ERR_FORMAT."""
    import paper_2606_23406_b200 as hq
    for lattice, n_tile, m in ((hqo.E8, 128, 300), (hqo.D4, 64, 130)):
        snr, seed = SNR_4BPS[lattice], 9
        W = hq_synth.gaussian_weight(m, 512, seed=m, outliers=True)
        w, enc = _check_weight_bitstream(ctx, W, lattice, n_tile, snr, seed)
        hd, blob, goff = w.export_host()
        assert (blob == enc["blob"]).all() and (goff == enc["group_off"]).all()
        assert hd.payload_bits == enc["payload_bits"] and (hd.rice_k[0], hd.rice_k[1]) == tuple(int(v) for v in enc["k"])
        w2 = ctx.import_weight(hd, blob.copy(), goff.copy())
        c1, n1 = w.decode_int8(); c2, n2 = w2.decode_int8()
        assert torch.equal(c1, c2) and torch.equal(n1, n2)
        for B in (1, 16, 70):
            x = _dev(hq_synth.activations(B, 512, seed=B), torch.bfloat16)
            a = w.linear(x, want_f32=True, want_acc=True); b = w2.linear(x, want_f32=True, want_acc=True)
            assert all(torch.equal(u, v) for u, v in zip(a, b))
        st1, st2 = w.stats(), w2.stats()
        tb = [hqo.tile_bits(lattice, enc["codes"][r, t * n_tile:(t + 1) * n_tile], enc["k"])
              for r in range(m) for t in range(512 // n_tile)]
        for st in (st1, st2):
            assert (st.tile_bits_min, st.tile_bits_max) == (min(tb), max(tb))
            assert st.payload_bits == sum(tb) and st.n_tiles == len(tb) and st.clamp_count == enc["clamps"]
            assert st.padding_bits == 8 * blob.size - st.payload_bits - 32 * len(tb) and st.padding_bits >= 0
        bad = goff.copy(); bad[3] += 1
        with pytest.raises(hq.HQError):
            ctx.import_weight(hd, blob, bad)
        bad = blob.copy(); bad[int(goff[2]) * 16] ^= 0x40           # a ulen that no longer matches its sub-group's size
        with pytest.raises(hq.HQError):
            ctx.import_weight(hd, bad, goff)
        hd2 = hq.WeightHeader.from_buffer_copy(hd); hd2.n_tile = 96
        with pytest.raises(hq.HQError):
            ctx.import_weight(hd2, blob, goff)
        w.free(); w2.free()


def test_snr_for_bps_operating_points_realize_their_rate_on_the_gpu_encoder(ctx):
    """§5.4: target bps -> table SNR -> the GPU encoder on iid Gaussian tiles realizes the rate within
    ~0.01 bps of the target (L295, L381)."""
    import paper_2606_23406_b200 as hq
    tiles = hq_synth.calib_tiles(4096, 128, seed=43)                # fresh tiles, not the table's
    W = _dev(tiles.reshape(512, 1024).copy())
    for lat in (hqo.E8, hqo.D4, hqo.A2, hqo.Z):
        for bps in (3.0, 4.0, 5.0):
            snr, k = hq.snr_for_bps(lat, bps)
            w = ctx.encode_weights(W, lat, 128, snr, seed=1)
            assert abs(w.stats().bits_per_scalar_payload - bps) < 0.015, (lat, bps)
            w.free()


def test_empty_and_out_of_range_arguments_fail_loudly_and_leave_the_context_usable(ctx):
    """include/hq.h error behaviour: empty batches, ragged K, an empty or overfull cache are HQ_ERR_SHAPE, never a
    silent no-op; the next valid call on the same context is still bit-exact against the oracle."""
    import paper_2606_23406_b200 as hq
    snr = SNR_4BPS[hqo.E8]
    W = hq_synth.gaussian_weight(64, 256, seed=21)
    with pytest.raises(hq.HQError):                                # n_in not a multiple of the RHT tile
        ctx.encode_weights(_dev(W[:, :200].copy()), hqo.E8, 128, snr, 1)
    w, enc = _check_weight_bitstream(ctx, W, hqo.E8, 128, snr, 1)
    with pytest.raises(hq.HQError):                                # empty batch
        w.linear(torch.empty((0, 256), dtype=torch.bfloat16, device="cuda"))
    with pytest.raises(hq.HQError):
        ctx.linear_group([w], torch.empty((0, 256), dtype=torch.bfloat16, device="cuda"))
    kv = ctx.kv_create(1, 128, 4, hqo.E8, f32(9.68), (0, 0), 5)
    q = _dev(hq_synth.kv_tokens(1, 2, 128, seed=8)[0], torch.bfloat16)
    with pytest.raises(hq.HQError):                                # attend on an empty cache
        kv.attend(q)
    K = _dev(hq_synth.kv_tokens(5, 1, 128, seed=6), torch.bfloat16)
    with pytest.raises(hq.HQError):                                # 5 tokens into a cache of 4
        kv.append(K, K)
    with pytest.raises(hq.HQError):                                # zero tokens
        kv.append(K[:0], K[:0])
    kv.append(K[:4], K[:4])
    assert kv.export()["n_tokens"] == 4
    with pytest.raises(hq.HQError):                                # full
        kv.append(K[:1], K[:1])
    kv.free()
    # the context still computes: accumulators bit-exact after the failed calls
    x = hq_synth.activations(3, 256, seed=22)
    q_o, sx_o = hqo.act_quant(x, hqo.E8, 128, 1)
    acc_o, _ = hqo.linear(enc["codes"], enc["norms"], hqo.E8, 128, snr, q_o, sx_o)
    _, _, acc = w.linear(_dev(x, torch.bfloat16), want_acc=True)
    assert (acc.cpu().numpy() == acc_o).all()
    w.free()
