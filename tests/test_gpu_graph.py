"""A whole decoder layer under ONE CUDA graph (Table 10's decode shape L496-511): with a
device_position cache (include/hq.h) every replay of the captured hq_layer_decode is the next token.  The replayed
graph is compared bit for bit with eager hq_layer_decode calls on a twin cache whose position is host state - the same
kernels, so outputs, lattice codes, norms and stream lengths must be identical - and the eager path is the one
tests/test_gpu_layer.py checks against the oracle."""
import numpy as np
import pytest

import hq_synth

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


def _layer(ctx, hidden, q_heads, kv_heads, ffn, kv):
    d = 128
    shapes = [(q_heads * d, hidden), (kv_heads * d, hidden), (kv_heads * d, hidden), (hidden, q_heads * d),
              (ffn, hidden), (ffn, hidden), (hidden, ffn)]
    ws = [ctx.encode_weights(_dev(hq_synth.gaussian_weight(m, n, seed=50 + i, outliers=True, std=1.0 / np.sqrt(n))),
                             8, 128, SNR, SEED, (2, 2)) for i, (m, n) in enumerate(shapes)]
    g = _dev(hq_synth.to_bf16_f32(1.0 + 0.1 * np.random.default_rng(1).standard_normal(hidden).astype(np.float32)))
    return ctx.layer(*ws, g, g, 1e-5, kv, q_heads), ws


@pytest.mark.parametrize("T0,steps,window", [(100, 40, 32), (0, 5, 0), (250, 10, 32)])   # crosses a 128-token block; starts empty
def test_layer_graph_replay_equals_eager_steps(ctx, T0, steps, window):
    hidden, q_heads, kv_heads, ffn, d = 512, 4, 2, 1024, 128
    K0 = hq_synth.kv_tokens(max(T0, 1), kv_heads, d, seed=4); V0 = hq_synth.kv_tokens(max(T0, 1), kv_heads, d, seed=5)
    kvs = [ctx.kv_create(kv_heads, d, 512, 8, SNR_KV, (0, 0), SEED, rotation=1, dither=1, window=window, device_position=dp)
           for dp in (False, True)]
    if T0:
        for kv in kvs:
            kv.append(_dev(K0), _dev(V0))
    (eager, ws_e), (graphed, ws_g) = [_layer(ctx, hidden, q_heads, kv_heads, ffn, kv) for kv in kvs]
    hs = [_dev(hq_synth.activations(1, hidden, seed=200 + i)[0] * 1.5) for i in range(steps + 1)]
    # step 0 eagerly on both (sizes the library's workspaces before the capture)
    out_e = [eager.decode(hs[0]).clone()]
    h_buf, o_buf = hs[0].clone(), torch.empty_like(hs[0])
    graphed.decode(h_buf, o_buf)
    out_g = [o_buf.clone()]
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        h_buf.copy_(hs[1])
        with torch.cuda.graph(g, stream=st):
            graphed.decode(h_buf, o_buf)            # capture only: nothing runs
        for i in range(1, steps + 1):
            h_buf.copy_(hs[i])
            g.replay()
            out_g.append(o_buf.clone())
    st.synchronize()
    for i in range(1, steps + 1):
        out_e.append(eager.decode(hs[i]).clone())
    torch.cuda.synchronize()
    for i in range(steps + 1):
        assert torch.equal(out_e[i], out_g[i]), f"step {i}"
    T = T0 + steps + 1
    assert kvs[1].sync_position() == T and kvs[0].sync_position() == T
    ex_e, ex_g = kvs[0].export(), kvs[1].export()
    assert ex_g["n_tokens"] == T
    for key in ("ulen", "norm", "upos", "blk_off", "rem", "una"):
        assert (ex_e[key] == ex_g[key]).all(), key
    for role in range(2):
        assert torch.equal(kvs[0].decode_int8(role, 0, T), kvs[1].decode_int8(role, 0, T))
    for kv in kvs:
        kv.free()
    for w in ws_e + ws_g:
        w.free()


def test_replay_past_capacity_writes_nothing_and_turns_sticky(ctx):
    import paper_2606_23406_b200 as hq
    H, d = 2, 128
    kv = ctx.kv_create(H, d, 4, 8, SNR_KV, (0, 0), SEED, rotation=1, dither=1, window=0, device_position=True)
    k = _dev(hq_synth.kv_tokens(1, H, d, seed=4)); v = _dev(hq_synth.kv_tokens(1, H, d, seed=5))
    kv.append(k, v)
    g = torch.cuda.CUDAGraph()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        with torch.cuda.graph(g, stream=st):
            kv.append(k, v)
        for _ in range(5):                           # positions 1, 2, 3, then two replays past max_tokens = 4
            g.replay()
    st.synchronize()
    with pytest.raises(hq.HQError):
        kv.sync_position()                           # sticky HQ_ERR_FORMAT
    kv.free()


def test_attend_on_an_empty_device_position_cache_gives_zeros(ctx):
    """A host-position cache rejects attend on an empty cache; a device-position cache cannot know (the count is on the
    device): it must return zeros, not NaN."""
    kv = ctx.kv_create(2, 128, 64, 8, SNR_KV, (0, 0), SEED, rotation=1, dither=1, window=32, device_position=True)
    out = kv.attend(_dev(hq_synth.activations(4, 128, seed=1)))
    torch.cuda.synchronize()
    assert (out.float() == 0).all()
    kv.free()
