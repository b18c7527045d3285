"""GPU parity of the qjl (dense Haar) KV rotation (include/hq.h hq_kv_config.qjl_dev; §3.4 eq.(2),
Table 4 L327 - the paper's default KV rotation at >= 2 bps; FORMAT R11) against the oracle:
lattice codes and norms bit-exact through bulk and single-token appends, attention against the oracle's long way
round (decode -> c - U -> un-normalize -> S^T -> inverse RHT -> textbook softmax in double) at 1e-3 (G16)."""
import numpy as np
import pytest

import hq_synth
from oracle import hqo

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def f32(v):
    return float(np.float32(v))


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23406_b200 as hq
    c = hq.Context(0)
    yield c
    c.close()


def _dev(a, dtype=torch.bfloat16):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda().to(dtype)


def _rel_err(y, ref, floor):
    ref = np.asarray(ref, np.float64)
    rms = np.sqrt((ref ** 2).mean())
    return np.max(np.abs(np.asarray(y, np.float64) - ref) / np.maximum(np.abs(ref), floor * rms + 1e-30))


@pytest.mark.parametrize("lattice,snr,k,dither,d", [
    (hqo.E8, 9.68, (0, 0), 1, 128),      # config 4's operating point with the paper's default rotation
    (hqo.E8, 22.68, (2, 2), 0, 128),
    (hqo.D4, 16.0, (1, 0), 1, 64),
    (hqo.Z, 21.9, (2, 2), 1, 256),
])
def test_qjl_codes_and_norms_bit_exact(ctx, lattice, snr, k, dither, d):
    T, H, seed, snr = 300, 2, 21, f32(snr)
    Q = hq_synth.haar_matrix(d, seed=d)
    K = hq_synth.kv_tokens(T, H, d, seed=4); V = hq_synth.kv_tokens(T, H, d, seed=5)
    kv = ctx.kv_create(H, d, 512, lattice, snr, k, seed, rotation=2, dither=dither, window=32, qjl=_dev(Q, torch.float32))
    t0 = 0
    for n in (257, 1, 1, 41):                                            # bulk prefill, decode steps, ragged tail
        kv.append(_dev(K[t0:t0 + n]), _dev(V[t0:t0 + n]))
        t0 += n
    ex = kv.export()
    assert ex["n_tokens"] == T
    for role, X in ((0, K), (1, V)):
        c, nrm, _ = hqo.kv_quantize(X, 0, role, lattice, snr, 2, dither, seed, qjl=Q)
        assert (kv.decode_int8(role, 0, T).cpu().numpy() == c).all()
        assert (ex["norm"][role, :, :T] == nrm.T).all()
    kv.free()


@pytest.mark.parametrize("lattice,snr,k,dither,T,window,H,QH", [
    (hqo.E8, 9.68, (0, 0), 1, 700, 32, 2, 8),
    (hqo.E8, 9.68, (0, 0), 0, 333, 0, 2, 4),        # qjl without dither: the paper's PPL winner at 2 bps (Table 6)
    (hqo.E8, 22.68, (2, 2), 1, 200, 32, 1, 8),
])
def test_qjl_attend_matches_oracle_long_way(ctx, lattice, snr, k, dither, T, window, H, QH):
    d, seed, snr = 128, 5, f32(snr)
    Q = hq_synth.haar_matrix(d, seed=77)
    K = hq_synth.kv_tokens(T, H, d, seed=14); V = hq_synth.kv_tokens(T, H, d, seed=15)
    q = hq_synth.activations(QH, d, seed=16)
    kv = ctx.kv_create(H, d, 1024, lattice, snr, k, seed, rotation=2, dither=dither, window=window, qjl=_dev(Q, torch.float32))
    kv.append(_dev(K), _dev(V))
    out, o32 = kv.attend(_dev(q), want_f32=True)
    ck, nk, _ = hqo.kv_quantize(K, 0, 0, lattice, snr, 2, dither, seed, qjl=Q)
    cv, nv, _ = hqo.kv_quantize(V, 0, 1, lattice, snr, 2, dither, seed, qjl=Q)
    Kh = hqo.kv_reconstruct(ck, nk, 0, 0, lattice, snr, 2, dither, seed, qjl=Q)
    Vh = hqo.kv_reconstruct(cv, nv, 0, 1, lattice, snr, 2, dither, seed, qjl=Q)
    ref = hqo.attend(Kh, Vh, K, V, window=window, q=q)
    assert _rel_err(o32.cpu().numpy(), ref, floor=2e-2) < 1e-3           # attention floor: DESIGN.md G16
    ref_bf16 = hq_synth.to_bf16_f32(ref.astype(np.float32))
    tol = np.abs(ref_bf16) * 2.0 ** -7 + 1e-3 * np.sqrt((ref ** 2).mean())
    assert (np.abs(out.float().cpu().numpy() - ref_bf16) <= tol).all()
    kv.free()


def test_qjl_argument_checks(ctx):
    import paper_2606_23406_b200 as hq
    Q = _dev(hq_synth.haar_matrix(128, 1), torch.float32)
    with pytest.raises(hq.HQError):
        ctx.kv_create(2, 128, 64, hqo.E8, f32(9.68), (0, 0), 1, rotation=2, dither=1, window=0)            # qjl without a matrix
    with pytest.raises(hq.HQError):
        ctx.kv_create(2, 128, 64, hqo.E8, f32(9.68), (0, 0), 1, rotation=1, dither=1, window=0, qjl=Q)     # a matrix without qjl


def test_qjl_attend_config4_shape_8192_tokens(ctx):
    """Config 4's shape (8 KV heads x 128, 32 query heads, E8 2 bps, dither, 32-token window) with the paper's default
    rotation at this rate (qjl, Table 4) over 8192 cached tokens: all 32 x 128 outputs against the long way round."""
    T, H, d, QH, seed, snr = 8192, 8, 128, 32, 4, f32(9.68)
    Q = hq_synth.haar_matrix(d, seed=123)
    K = hq_synth.kv_tokens(T, H, d, seed=4); V = hq_synth.kv_tokens(T, H, d, seed=5)
    q = hq_synth.activations(QH, d, seed=6)
    kv = ctx.kv_create(H, d, T + 64, hqo.E8, snr, (0, 0), seed, rotation=2, dither=1, window=32, qjl=_dev(Q, torch.float32))
    kv.append(_dev(K), _dev(V))
    out, o32 = kv.attend(_dev(q), want_f32=True)
    ck, nk, _ = hqo.kv_quantize(K, 0, 0, hqo.E8, snr, 2, 1, seed, qjl=Q)
    cv, nv, _ = hqo.kv_quantize(V, 0, 1, hqo.E8, snr, 2, 1, seed, qjl=Q)
    rng = np.random.default_rng(1)
    for role, c in ((0, ck), (1, cv)):                                   # sampled tokens of the cache: codes bit-exact
        for t in rng.choice(T, 24, replace=False):
            assert (kv.decode_int8(role, int(t), 1).cpu().numpy()[0] == c[t]).all()
    ref = hqo.attend(hqo.kv_reconstruct(ck, nk, 0, 0, hqo.E8, snr, 2, 1, seed, qjl=Q),
                     hqo.kv_reconstruct(cv, nv, 0, 1, hqo.E8, snr, 2, 1, seed, qjl=Q), K, V, window=32, q=q)
    assert _rel_err(o32.cpu().numpy(), ref, floor=2e-2) < 1e-3
    kv.free()
