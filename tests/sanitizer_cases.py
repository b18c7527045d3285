"""Small invocations of every kernel family of libhq.so, sized for compute-sanitizer (memcheck / racecheck / synccheck /
initcheck).  Not a pytest module: run as

    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py

(profiles/r02_sanitizers.md records the runs).  Every result is still compared with the oracle.
"""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import hq_synth  # noqa: E402
import paper_2606_23406_b200 as hq  # noqa: E402
from oracle import hqo  # noqa: E402


def dev(a, dt=None):
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t.to(dt) if dt is not None else t


def main():
    ctx = hq.Context(0)
    snr = float(np.float32(22.68))
    # config 1 (tile 64: the generic kernel) and an E8 / tile 128 weight (batch 1: k_gemv_e8; 16: k_linear_e8; 70: large-M)
    W1, x1 = hq_synth.c1_weight()
    w1 = ctx.encode_weights(dev(W1), hqo.E8, 64, snr, 1234)
    enc1 = hqo.encode_weights(W1, hqo.E8, 64, snr, 1234)
    q_o, sx_o = hqo.act_quant(x1, hqo.E8, 64, 1234)
    acc_o, _ = hqo.linear(enc1["codes"], enc1["norms"], hqo.E8, 64, snr, q_o, sx_o)
    _, _, acc = w1.linear(dev(x1), want_f32=True, want_acc=True)
    assert (acc.cpu().numpy() == acc_o).all()
    W = hq_synth.gaussian_weight(300, 1024, seed=3, outliers=True)
    ws = [ctx.encode_weights(dev(W, torch.bfloat16), hqo.E8, 128, snr, 7, (2, 2)) for _ in range(2)]
    enc = hqo.encode_weights(W, hqo.E8, 128, snr, 7, (2, 2))
    blob, goff = ws[0].export()
    assert (blob == enc["blob"]).all()
    for B in (1, 16, 70):
        x = hq_synth.activations(B, 1024, seed=B)
        q_o, sx_o = hqo.act_quant(x, hqo.E8, 128, 7)
        acc_o, y_o = hqo.linear(enc["codes"], enc["norms"], hqo.E8, 128, snr, q_o, sx_o)
        _, y32, acc = ws[0].linear(dev(x, torch.bfloat16), want_f32=True, want_acc=True)
        assert (acc.cpu().numpy() == acc_o).all()
        ys, y32s = ctx.linear_group(ws, dev(x, torch.bfloat16), want_f32=True)     # grouped launch
        assert np.abs(y32s[1].cpu().numpy() - y_o).max() < 1e-3 * np.sqrt((y_o ** 2).mean()) * 10
    # KV: bulk + single-token appends (bit concatenation with atomicOr), attend
    T, H, d, QH = 300, 2, 128, 8
    snr_kv = float(np.float32(9.68))
    K = hq_synth.kv_tokens(T, H, d, seed=4); V = hq_synth.kv_tokens(T, H, d, seed=5)
    kv = ctx.kv_create(H, d, 512, hqo.E8, snr_kv, (0, 0), 5, rotation=1, dither=1, window=32)
    kv.append(dev(K[:290], torch.bfloat16), dev(V[:290], torch.bfloat16))
    for t in range(290, T):
        kv.append(dev(K[t:t + 1], torch.bfloat16), dev(V[t:t + 1], torch.bfloat16))
    ck, _, _ = hqo.kv_quantize(K, 0, 0, hqo.E8, snr_kv, 1, 1, 5)
    assert (kv.decode_int8(0, 0, T).cpu().numpy() == ck).all()
    out = kv.attend(dev(hq_synth.activations(QH, d, seed=6), torch.bfloat16))
    assert torch.isfinite(out.float()).all()
    torch.cuda.synchronize()
    kv.free()
    for w in ws + [w1]:
        w.free()
    ctx.close()
    print("sanitizer cases ok")


if __name__ == "__main__":
    main()
