"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times, on sampled outputs the oracle
computes one by one (the per-(row, tile) encode and the per-output contraction are independent, so a sample of rows /
tokens is an exact check of those outputs).  Explicit Rice parameters make a sampled row's code independent of the
rest of the tensor (auto-k is a tensor-wide argmin, covered at small sizes in test_gpu_parity.py).
"""
import numpy as np
import pytest

import hq_synth
from oracle import hqo

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

SNR = float(np.float32(22.68))      # E8 at 4.0 bps


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


def _oracle_rows(W, rows, seed, B_x):
    """Oracle codes / norms / y for the sampled rows of W (explicit k = 2) and the activations B_x."""
    enc = hqo.encode_weights(W[rows], hqo.E8, 128, SNR, seed, (2, 2))
    q_o, sx_o = hqo.act_quant(B_x, hqo.E8, 128, seed)
    acc_o, y_o = hqo.linear(enc["codes"], enc["norms"], hqo.E8, 128, SNR, q_o, sx_o)
    return enc, acc_o, y_o


def test_config2_grouped_layer_full_size_sampled_rows(ctx):
    """BASELINE config 2 at full size, batch 1 and 16: q+k+v and gate+up through hq_linear_group (what bench.py times),
    down through hq_linear; 96 sampled rows per matrix: INT8 codes, fp16 norms and INT32 accumulators bit-exact, y to 1e-3."""
    rng = np.random.default_rng(123)
    seed = 3
    for names in (["q", "k", "v"], ["gate", "up"], ["down"]):
        Ws = [hq_synth.llama_weight(0, n) for n in names]
        ws = [ctx.encode_weights(_dev(W, torch.bfloat16), hqo.E8, 128, SNR, seed, (2, 2)) for W in Ws]
        n_in = Ws[0].shape[1]
        for B in (1, 16):
            x = hq_synth.activations(B, n_in, seed=50 + B)
            xd = _dev(x, torch.bfloat16)
            ys, y32s = ctx.linear_group(ws, xd, want_f32=True)
            for W, w, y32 in zip(Ws, ws, y32s):
                m = W.shape[0]
                rows = np.sort(np.concatenate([rng.choice(m, 90, replace=False), [0, 1, 127, 128, m - 2, m - 1]]))
                enc, acc_o, y_o = _oracle_rows(W, rows, seed, x)
                assert _rel_err(y32.cpu().numpy()[:, rows], y_o) < 1e-3
                if B == 1:
                    codes, norms = w.decode_int8()
                    assert (codes.cpu().numpy()[rows] == enc["codes"]).all()
                    assert (norms.cpu().numpy().view(np.uint16)[rows] == enc["norms"]).all()
                    _, _, acc = w.linear(xd, want_f32=True, want_acc=True)     # the single-weight launch exposes acc
                    assert (acc.cpu().numpy()[:, :, rows] == acc_o).all()
        for w in ws:
            w.free()


def test_config5_large_m_full_size_sampled_outputs(ctx):
    """BASELINE config 5 at full size (8192 tokens x 4096 -> 16384): 64 sampled tokens x 64 sampled rows."""
    rng = np.random.default_rng(5)
    seed, m, n_in, T = 5, 16384, 4096, 8192
    W = hq_synth.gaussian_weight(m, n_in, seed=5)
    X = hq_synth.activations(T, n_in, seed=6)
    w = ctx.encode_weights(_dev(W, torch.bfloat16), hqo.E8, 128, SNR, seed, (2, 2))
    y = torch.empty((T, m), dtype=torch.bfloat16, device="cuda")
    w.linear(_dev(X, torch.bfloat16), y=y)
    rows = np.sort(rng.choice(m, 64, replace=False)); toks = np.sort(rng.choice(T, 64, replace=False))
    enc, acc_o, y_o = _oracle_rows(W, rows, seed, X[toks])
    got = y[_dev(toks)][:, _dev(rows)].float().cpu().numpy()
    ref_bf16 = torch.from_numpy(y_o.astype(np.float32)).to(torch.bfloat16).float().numpy()
    tol = np.abs(ref_bf16) * 2.0 ** -7 + 1e-3 * np.sqrt((y_o ** 2).mean())
    assert (np.abs(got - ref_bf16) <= tol).all()
    # the INT32 accumulators of the same launch configuration (every K-tile, full 8192 x 16384 extent: 17 GB) would not
    # fit beside y: they are compared on a 2048-token slice (4.3 GB of accumulators) that keeps the full weight
    Xs = X[:2048]
    del y
    ys, y32s, acc = w.linear(_dev(Xs, torch.bfloat16), want_f32=True, want_acc=True)
    tk = toks[toks < 2048]
    sel = acc[:, _dev(tk)][:, :, _dev(rows)].cpu().numpy()
    pos = np.searchsorted(toks, tk)
    assert (sel == acc_o[:, pos, :]).all()
    assert _rel_err(y32s[_dev(tk)][:, _dev(rows)].cpu().numpy(), y_o[pos]) < 1e-3
    w.free()


def test_config4_kv_full_size_sampled_tokens(ctx):
    """BASELINE config 4 at full size (8 heads x 128, 32768 tokens, E8 2 bps, signs rotation, dither): the cache is
    filled by one bulk append plus single-token appends (as bench.py does); sampled tokens must decode to the
    oracle's codes (the dither is keyed by the token index)."""
    T, H, d, seed = 32768, 8, 128, 4
    snr = float(np.float32(9.68))
    K = hq_synth.kv_tokens(T + 4, H, d, seed=4); V = hq_synth.kv_tokens(T + 4, H, d, seed=5)
    kv = ctx.kv_create(H, d, T + 64, hqo.E8, snr, (0, 0), seed, rotation=1, dither=1, window=32)
    kv.append(_dev(K[:T], torch.bfloat16), _dev(V[:T], torch.bfloat16))
    for i in range(4):
        kv.append(_dev(K[T + i:T + i + 1], torch.bfloat16), _dev(V[T + i:T + i + 1], torch.bfloat16))
    rng = np.random.default_rng(9)
    toks = np.concatenate([[0, 127, 128, 4095, 4096, T - 1, T, T + 3], rng.choice(T, 56, replace=False)])
    for role, X in enumerate((K, V)):
        for t in toks:
            ref, nrm, _ = hqo.kv_quantize(X[t:t + 1], int(t), role, hqo.E8, snr, 1, 1, seed)
            got = kv.decode_int8(role, int(t), 1).cpu().numpy()
            assert (got == ref).all(), (role, t)
    # attend over the whole cache against the oracle's long way round (un-dither, un-normalize, S^T, inverse RHT,
    # softmax in double, L178): all 32 x 128 outputs; the launch is the one bench.py times (3.5 blocks per split)
    q = hq_synth.activations(32, d, seed=6)
    out, o32 = kv.attend(_dev(q, torch.bfloat16), want_f32=True)
    Tn = T + 4
    ck, nk, _ = hqo.kv_quantize(K[:Tn], 0, 0, hqo.E8, snr, 1, 1, seed)
    cv, nv, _ = hqo.kv_quantize(V[:Tn], 0, 1, hqo.E8, snr, 1, 1, seed)
    assert (kv.decode_int8(1, Tn - 300, 300).cpu().numpy() == cv[Tn - 300:]).all()
    Kh = hqo.kv_reconstruct(ck, nk, 0, 0, hqo.E8, snr, 1, 1, seed)
    Vh = hqo.kv_reconstruct(cv, nv, 0, 1, hqo.E8, snr, 1, 1, seed)
    ref = hqo.attend(Kh, Vh, K[:Tn], V[:Tn], window=32, q=q)
    assert _rel_err(o32.cpu().numpy(), ref, floor=2e-2) < 1e-3
    ref_bf16 = torch.from_numpy(ref.astype(np.float32)).to(torch.bfloat16).float().numpy()
    tol = np.abs(ref_bf16) * 2.0 ** -7 + 1e-3 * np.sqrt((ref ** 2).mean())
    assert (np.abs(out.float().cpu().numpy() - ref_bf16) <= tol).all()
    kv.free()


@pytest.mark.parametrize("lattice,n_tile,snr,k", [
    (hqo.D4, 128, 22.5, (2, 1)), (hqo.A2, 128, 22.21, (2, 2)), (hqo.Z, 128, 21.9, (2, 2)),
    (hqo.E8, 64, 22.68, (2, 2)), (hqo.E8, 256, 22.68, (2, 2)), (hqo.D4, 256, 16.4, (1, 0)), (hqo.Z, 64, 27.9, (3, 3)),
])
def test_config3_full_size_other_lattices_and_tiles_sampled_rows(ctx, lattice, n_tile, snr, k):
    """BASELINE config 3 at full size (14336 x 4096) for the lattices / tiles that do not take the E8/128 kernel:
    96 sampled rows: INT8 codes, fp16 norms, INT32 accumulators bit-exact and y to 1e-3, at batch 1 (the launch and the
    K-split bench.py's sweep times) and batch 16."""
    rng = np.random.default_rng(33)
    seed, m, n_in = 3, 14336, 4096
    snr = float(np.float32(snr))
    W = hq_synth.gaussian_weight(m, n_in, seed=3)
    w = ctx.encode_weights(_dev(W, torch.bfloat16), lattice, n_tile, snr, seed, k)
    rows = np.sort(np.concatenate([rng.choice(m, 90, replace=False), [0, 1, 127, 128, m - 2, m - 1]]))
    enc = hqo.encode_weights(W[rows], lattice, n_tile, snr, seed, k)
    codes, norms = w.decode_int8()
    assert (codes.cpu().numpy()[rows] == enc["codes"]).all()
    assert (norms.cpu().numpy().view(np.uint16)[rows] == enc["norms"]).all()
    for B in (1, 16):
        x = hq_synth.activations(B, n_in, seed=60 + B)
        q_o, sx_o = hqo.act_quant(x, lattice, n_tile, seed)
        acc_o, y_o = hqo.linear(enc["codes"], enc["norms"], lattice, n_tile, snr, q_o, sx_o)
        y, y32, acc = w.linear(_dev(x, torch.bfloat16), want_f32=True, want_acc=True)
        assert (acc.cpu().numpy()[:, :, rows] == acc_o).all()
        assert _rel_err(y32.cpu().numpy()[:, rows], y_o) < 1e-3
        y1, y1_32, _ = w.linear(_dev(x, torch.bfloat16), want_f32=True)     # the launch without the debug output
        assert torch.equal(y1_32, y32) and torch.equal(y1, y)
    w.free()
