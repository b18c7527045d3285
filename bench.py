#!/usr/bin/env python
"""bench.py — HyperQuant hot path on B200: fused Rice-decode + tcgen05 INT8 GEMV over one Llama-3.1-8B-shaped
decoder layer's linears (BASELINE.json configs[1]: E8, 4 bps, RHT tile 128, batch 1), seeded synthetic weights.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--layers L] [--impl reference]

A step = the seven linears (q,k,v,o,gate,up,down) of one layer at batch 1 through hq_linear_group: matrices that share an
input share ONE launch of the fused kernel (activation RHT + INT8 cast, Rice decode, tcgen05 INT8 MMA, split-K reduction
all inside k_gemv_e8), so a step is exactly four kernel launches.  L distinct layers (L x ~116 MB compressed > the 126 MB L2) are
cycled so no step re-reads its weights from L2.  One JSON line on stdout (rank 0).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import hq_synth  # noqa: E402

METRIC = "fused decode+INT8 GEMV % of HBM roofline; large-M INT8 TOPS vs peak"
UNIT = "GB/s of compressed weight bytes (batch-1 GEMV, whole layer)"
SNR_E8_4BPS = float(np.float32(22.68))   # E8 at 4.0 bps on iid Gaussian tiles (B.1 L857)
NAMES = list(hq_synth.LLAMA_SHAPES)
# ncu-derived figures (DRAM bytes and warp instructions of the four fused launches of one step) are NOT typed in here:
# they are read from profiles/r02_ncu_step.json, which the ncu pass of a named commit wrote (see the .md beside it)
NCU_STEP_JSON = os.path.join(ROOT, "profiles", "r02_ncu_step.json")
LARGE_M_TILE = 256   # RHT tile of the config-5 weights (the tile is chosen on kernel grounds)
WORKLOAD = "llama3.1-8b decoder-layer linears q/k/v/o/gate/up/down, E8 4 bps, RHT tile 128, batch 1 (BASELINE configs[1])"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    def __init__(self, index=0):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.rows = index, False, []

    def run(self):
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
            "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i",
                                      str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            time.sleep(0.05)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(int(r[0]) for r in self.rows if r[0].isdigit())
        mx = max(int(r[1]) for r in self.rows if r[1].isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": mx, "reasons": reasons, "samples": len(sm)}


def base_config(layers):
    """The `config` both arms print (same keys: the driver compares them)."""
    return {"workload": WORKLOAD, "lattice": "E8", "snr_db": SNR_E8_4BPS, "n_tile": 128, "batch": 1,
            "layers_cycled": layers, "l2_policy": "inputs larger than L2 (layers cycled)",
            "launch": "one CUDA graph per layer: hq_linear_group x 4 (q+k+v, o, gate+up, down) = 4 launches of k_gemv_e8",
            "scalars_per_step": sum(m * n for m, n in hq_synth.LLAMA_SHAPES.values()), "parallelism": "replicas only"}


def oracle_sample(threads_note=True):
    """The oracle (as it stands) on a bounded sample of the workload: the 'k' projection (1024 x 4096) of
    layer 0 — decode the container (O2) + activation cast + INT8 contraction (O3) at batch 1."""
    from oracle import hqo
    W = hq_synth.llama_weight(0, "k")
    x = hq_synth.activations(1, W.shape[1], seed=1000)
    enc = hqo.encode_weights(W, hqo.E8, 128, SNR_E8_4BPS, seed=0)          # untimed: building the sample
    nbytes = (enc["payload_bits"] + 32 * enc["norms"].size) / 8.0

    def one_pass():
        codes, norms = hqo.unpack_weights(enc["blob"], enc["group_off"], W.shape[0], W.shape[1], hqo.E8, 128, enc["k"])
        q, s_x = hqo.act_quant(x, hqo.E8, 128, seed=0)
        hqo.linear(codes, norms, hqo.E8, 128, SNR_E8_4BPS, q, s_x, want_acc=False)

    return one_pass, nbytes, "oracle decode (O2) + act cast + INT8 contraction (O3) on layer-0 'k' 1024x4096, batch 1"


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/unit/config, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    one_pass, nbytes, sample = oracle_sample()
    for _ in range(max(1, min(args.warmup, 2))):
        one_pass()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        one_pass()
    dt = time.perf_counter() - t0
    val = nbytes * args.steps / dt / 1e9
    cores = len(os.sched_getaffinity(0))
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int8", "data": "synthetic",
            "config": base_config(args.layers),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def max_over_ranks(value, device=None):
    """Replicas only: the job's time is the slowest rank's.  No-op without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(bytes_per_step_per_rank, ms_per_step_max, world):
    """Whole-job throughput of N independent replicas (weak scaling): all ranks' bytes over the slowest rank's time."""
    return world * bytes_per_step_per_rank / (ms_per_step_max * 1e-3) / 1e9


def _time_cuda(fn, reps, warm=1):
    import torch
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def measure_large_m(ctx, hq, dev, reps=10):
    """BASELINE config 5, both GEMMs of the DiT-scale MLP (8192 tokens: 4096 -> 16384 and 16384 -> 4096), E8 4 bps,
    whole hq_linear call (activation operand + weight decode + warp-specialised tcgen05 GEMM), >= 10 repetitions each;
    peak = torch._int_mm 8192^3 measured in the same run (a plain library INT8 GEMM)."""
    import torch
    res = {"bound": "tensor", "unit": "TOPS", "reps": reps, "gemms": []}
    a = torch.randint(-127, 127, (8192, 8192), dtype=torch.int8, device=dev)
    b = torch.randint(-127, 127, (8192, 8192), dtype=torch.int8, device=dev)
    ms_mm = _time_cuda(lambda: torch._int_mm(a, b), reps=10, warm=3)
    peak = 2.0 * 8192 ** 3 / (ms_mm * 1e-3) / 1e12
    del a, b
    res["peak"], res["peak_source"] = peak, "torch._int_mm 8192^3 INT8, measured in this run"
    res["peak_nominal_dense_int8"] = 4500.0
    tot_ops, tot_ms, fp8_ms = 0.0, 0.0, []
    for m, n_in, seed in ((16384, 4096, 5), (4096, 16384, 7)):
        W = torch.from_numpy(hq_synth.gaussian_weight(m, n_in, seed=seed)).to(dev).to(torch.bfloat16)
        w = ctx.encode_weights(W, hq.Lattice.E8, LARGE_M_TILE, SNR_E8_4BPS, seed=seed)
        del W
        X = torch.from_numpy(hq_synth.activations(8192, n_in, seed=6)).to(dev).to(torch.bfloat16)
        y = torch.empty((8192, m), dtype=torch.bfloat16, device=dev)
        ms = _time_cuda(lambda: w.linear(X, y=y), reps=reps, warm=2)
        ops = 2.0 * 8192 * m * n_in
        res["gemms"].append({"shape": f"8192 tokens x {n_in} -> {m}", "ms": ms, "TOPS": ops / (ms * 1e-3) / 1e12,
                             "frac": ops / (ms * 1e-3) / 1e12 / peak})
        tot_ops += ops; tot_ms += ms
        # the same GEMM with the FP8-E4M3 cast of PAPER.md §4.8 (hq_linear_cast: kind::f8f6f4, fp32 accumulator)
        ms8 = _time_cuda(lambda: w.linear_cast(X, hq.CAST_FP8_E4M3, y=y), reps=reps, warm=2)
        fp8_ms.append(ms8)
        w.free(); del X, y
    res["achieved"] = tot_ops / (tot_ms * 1e-3) / 1e12
    res["frac"] = res["achieved"] / peak
    fp8_tops = tot_ops / (sum(fp8_ms) * 1e-3) / 1e12
    res["fp8_e4m3"] = {"ms": fp8_ms, "achieved": fp8_tops, "peak": peak, "frac": fp8_tops / peak,
                       "peak_source": "the in-run INT8 peak x 1.0 (B200's nominal dense FP8 : INT8 ratio)",
                       "what": "hq_linear_cast(HQ_CAST_FP8_E4M3) on the same two GEMMs (SURVEY §8(f)2)"}
    res["n_tile"] = LARGE_M_TILE
    res["workload"] = "BASELINE configs[4]: 8192 tokens x (4096 -> 16384, 16384 -> 4096), E8 4 bps, bf16 activations through the per-tile RHT"
    return res


def measure_attend(ctx, hq, dev, peak_gbs):
    """BASELINE config 4: 8 KV heads x 128, 32768 tokens, E8 2 bps, signs rotation, dither, window 32; 32 query heads."""
    import torch
    T, H, d, QH = 32768, 8, 128, 32
    snr_kv = float(np.float32(9.68))
    K = torch.from_numpy(hq_synth.kv_tokens(T + 16, H, d, seed=4)).to(dev).to(torch.bfloat16)
    V = torch.from_numpy(hq_synth.kv_tokens(T + 16, H, d, seed=5)).to(dev).to(torch.bfloat16)
    q = torch.from_numpy(hq_synth.activations(QH, d, seed=6)).to(dev).to(torch.bfloat16)
    kv = ctx.kv_create(H, d, T + 64, hq.Lattice.E8, snr_kv, (0, 0), 4, rotation=1, dither=1, window=32)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    kv.append(K[:T], V[:T])
    torch.cuda.synchronize()
    bulk_s = time.perf_counter() - t0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(16):
        kv.append(K[T + i:T + i + 1], V[T + i:T + i + 1])
    e1.record()
    torch.cuda.synchronize()
    app_us = 1e3 * e0.elapsed_time(e1) / 16
    o = torch.empty_like(q)
    att_ms = _time_cuda(lambda: kv.attend(q, out=o), reps=10, warm=2)
    ex = kv.export()
    Tn = int(ex["n_tokens"])
    payload_bits = float(ex["upos"].astype(np.int64).sum()) + 2.0 * H * Tn * float(ex["rbits"])
    scal = 2.0 * H * Tn * d
    alg_bytes = (payload_bits + 32.0 * 2 * H * Tn) / 8.0
    gbs = alg_bytes / (att_ms * 1e-3) / 1e9
    res = {"bound": "hbm", "unit": "GB/s", "achieved": gbs, "peak": peak_gbs, "frac": gbs / peak_gbs,
           "attend_us": 1e3 * att_ms, "alg_bytes": alg_bytes, "append_us_per_token": app_us,
           "bulk_append_Mscalars_per_s": 2.0 * H * T * d / bulk_s / 1e6,
           "bits_per_scalar_payload": payload_bits / scal, "bits_per_scalar_total": 8.0 * alg_bytes / scal,
           "kv_compression_vs_bf16": 16.0 / (8.0 * alg_bytes / scal),
           "workload": "BASELINE configs[3]: 8 KV heads x 128, 32768 tokens, E8 2 bps, signs rotation, dither, window 32; 32 query heads"}
    kv.free(); del K, V
    return res


def measure_layer_step(ctx, hq, dev, layers, peak_gbs, context=32768, steps=12, short=True):
    """SURVEY §8(f)3 / PAPER.md Table 10's decode shape (L496-511): one token through whole decoder layers
    (hq_layer_decode: RMSNorm and SiLU.mul folded into the linears' prologues, residuals into their epilogues, KV append,
    attend) on the bench's compressed Llama-3.1-8B-shaped layers, each with its own 2-bps KV cache at `context` tokens.
    Launched eagerly (the cache position is host state), 7 launches per layer; the layers are cycled so weights and
    caches come from HBM."""
    import torch
    H, d, QH, hidden = 8, 128, 32, 4096
    snr_kv = float(np.float32(9.68))
    K = torch.from_numpy(hq_synth.kv_tokens(context, H, d, seed=4)).to(dev).to(torch.bfloat16)
    V = torch.from_numpy(hq_synth.kv_tokens(context, H, d, seed=5)).to(dev).to(torch.bfloat16)
    g = torch.ones((hidden,), dtype=torch.bfloat16, device=dev)
    objs, kv_bytes = [], 0.0
    for l, ws in enumerate(layers):
        kv = ctx.kv_create(H, d, context + 256, hq.Lattice.E8, snr_kv, (0, 0), 4 + l, rotation=1, dither=1, window=32,
                           device_position=True)
        kv.append(K, V)
        ex = kv.export()
        Tn = int(ex["n_tokens"])
        kv_bytes += (float(ex["upos"].astype(np.int64).sum()) + 2.0 * H * Tn * float(ex["rbits"]) + 32.0 * 2 * H * Tn) / 8.0
        objs.append((ctx.layer(ws["q"], ws["k"], ws["v"], ws["o"], ws["gate"], ws["up"], ws["down"], g, g, 1e-5, kv, QH), kv))
    del K, V
    kv_bytes /= len(layers)
    w_bytes = float(np.mean([sum((w.info.payload_bits + w.info.norm_bits + w.info.length_bits) / 8.0 for w in ws.values())
                             for ws in layers]))
    h = torch.from_numpy(hq_synth.activations(1, hidden, seed=99)[0]).to(dev).to(torch.bfloat16)
    h_out = torch.empty_like(h)

    def token():   # one token through all layers (fresh h per layer keeps the magnitudes of the synthetic weights bounded)
        for layer, _ in objs:
            layer.decode(h, h_out)
    for _ in range(3):
        token()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        token()
    e1.record()
    torch.cuda.synchronize()
    us = 1e3 * e0.elapsed_time(e1) / (steps * len(objs))
    ok = bool(torch.isfinite(h_out.float()).all())
    # the same token step as ONE CUDA graph per layer: the caches keep their position on the device, every replay is the
    # next token (tests/test_gpu_graph.py: bit-identical to the eager calls)
    st = torch.cuda.Stream()
    graphs = []
    with torch.cuda.stream(st):
        for layer, _ in objs:
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st):
                layer.decode(h, h_out)
            graphs.append(g)
        for _ in range(2):
            for g in graphs:
                g.replay()
        st.synchronize()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(st)
        for _ in range(steps):
            for g in graphs:
                g.replay()
        g1.record(st)
        st.synchronize()
    us_graph = 1e3 * g0.elapsed_time(g1) / (steps * len(objs))
    ok = ok and bool(torch.isfinite(h_out.float()).all()) and objs[0][1].sync_position() == context + 3 + steps + 2 + steps
    alg = w_bytes + kv_bytes
    gbs = alg / (us * 1e-6) / 1e9
    for layer, kv in objs:
        kv.free()
    short_ctx = None
    if short:   # the launch-bound end of the same call: 1024 tokens of context
        r = measure_layer_step(ctx, hq, dev, layers, peak_gbs, context=1024, steps=steps, short=False)
        short_ctx = {"context_tokens": 1024, "us_per_layer_step": r["us_per_layer_step"],
                     "us_per_layer_step_graph": r["us_per_layer_step_graph"], "finite": r["finite"]}
    return {"bound": "hbm", "unit": "GB/s", "achieved": gbs, "peak": peak_gbs, "frac": gbs / peak_gbs,
            "us_per_layer_step": us, "us_per_layer_step_graph": us_graph, "tokens_per_s_at_32_layers": 1e6 / (32.0 * min(us, us_graph)),
            "context_tokens": context,
            "launches_per_layer": 7, "alg_bytes_per_layer_step": alg, "weight_bytes": w_bytes, "kv_bytes": kv_bytes,
            "finite": ok, "short_context": short_ctx, "bf16_bytes_per_layer_step": 2.0 * 218103808 + 2.0 * 2 * H * d * context,
            "call": "hq_layer_decode (eager, and as one CUDA graph per layer on device_position caches): q+k+v [RMSNorm fold] -> hq_kv_append -> hq_attend (split + combine) -> o [+ residual] -> gate+up [RMSNorm fold] -> down [SiLU.mul fold, + residual]",
            "workload": "Llama-3.1-8B-shaped decoder layer, E8 4 bps weights, E8 2 bps KV cache (signs rotation, dither, window 32), batch 1"}


def measure_config3(ctx, hq, dev, copies=5):
    """BASELINE config 3 (reduced): a 14336 x 4096 Gaussian weight; lattice x rate at tile 128, E8 4 bps at tiles 64 / 256.
    `copies` distinct weights per point (5 x ~31 MB > the 126 MB L2) are cycled so the GEMV reads HBM, not L2."""
    import torch
    Ws = [torch.from_numpy(hq_synth.gaussian_weight(14336, 4096, seed=30 + c)).to(dev).to(torch.bfloat16) for c in range(copies)]
    x = torch.from_numpy(hq_synth.activations(1, 4096, seed=9)).to(dev).to(torch.bfloat16)
    combos = [(lat, bps, 128) for lat in ("E8", "D4", "A2", "Z") for bps in (3.0, 4.0, 5.0)] + [("E8", 4.0, 64), ("E8", 4.0, 256)]
    rows = []
    for lat, bps, n_tile in combos:
        s32, _ = hq.snr_for_bps(hq.Lattice.BY_NAME[lat], bps)       # the library's calibration table (§5.4)
        ws = [ctx.encode_weights(W, hq.Lattice.BY_NAME[lat], n_tile, s32, seed=3) for W in Ws]
        info, st = ws[0].info, ws[0].stats()
        sc = float(info.m_out * info.n_in)
        yv = torch.empty((1, 14336), dtype=torch.bfloat16, device=dev)
        state = {"i": 0}

        def one():
            ws[state["i"] % copies].linear(x, y=yv)
            state["i"] += 1
        ms = _time_cuda(one, reps=2 * copies, warm=copies)
        nbytes = (info.payload_bits + info.norm_bits + info.length_bits) / 8.0
        # MSE of the reconstruction, measured in the rotated domain (the RHT is orthonormal) on the first 512 rows
        R = 512
        _, _, u = ws[0].act_quant(Ws[0][:R], want_u=True)
        codes, norms = ws[0].decode_int8()
        c = codes[:R].float().view(R, -1, n_tile)
        if lat == "A2":
            c[..., 0::2] *= 3.0 ** 0.5
        rho = norms[:R].view(torch.float16).float()
        scale = rho / (info.alpha * n_tile ** 0.5)
        mse = float(((u.view(R, -1, n_tile) - scale[..., None] * c) ** 2).mean())
        pred = float((rho ** 2).mean() / n_tile / 10 ** (s32 / 10))
        rows.append({"lattice": lat, "target_bps": bps, "snr_db": s32, "n_tile": n_tile, "k": [info.rice_k[0], info.rice_k[1]],
                     "bits_payload": info.payload_bits / sc, "bits_total": 8.0 * nbytes / sc,
                     "tile_bits_min_max": [st.tile_bits_min, st.tile_bits_max],
                     "mse": mse, "mse_predicted": pred, "gemv_us": 1e3 * ms, "GBps_compressed": nbytes / (ms * 1e-3) / 1e9})
        for w in ws:
            w.free()
    return {"copies_cycled": copies, "rows": rows}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=4)
    ap.add_argument("--layers", type=int, default=4)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--skip-extras", action="store_true")
    ap.add_argument("--only", choices=("decode_ceiling", "large_m", "attend", "config3", "layer_step"), default=None,
                    help="run one secondary measurement alone and print its JSON (the command the ncu captures under profiles/ name)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_2606_23406_b200 as hq

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    ctx = hq.Context(local)

    if args.only:
        if args.only == "decode_ceiling":
            W = torch.from_numpy(hq_synth.llama_weight(0, "q")).to(dev).to(torch.bfloat16)
            w = ctx.encode_weights(W, hq.Lattice.E8, 128, SNR_E8_4BPS, seed=0)
            out = {"scalars_per_s": [w.decode_ceiling(200) for _ in range(3)]}
        elif args.only == "large_m":
            out = measure_large_m(ctx, hq, dev, reps=3)
        elif args.only == "attend":
            out = measure_attend(ctx, hq, dev, peaks()[0])
        elif args.only == "layer_step":
            lw = []
            for l in range(args.layers):
                lw.append({name: ctx.encode_weights(torch.from_numpy(hq_synth.llama_weight(l, name)).to(dev).to(torch.bfloat16),
                                                    hq.Lattice.E8, 128, SNR_E8_4BPS, seed=l) for name in NAMES})
            out = measure_layer_step(ctx, hq, dev, lw, peaks()[0])
        else:
            out = measure_config3(ctx, hq, dev)
        print(json.dumps({"only": args.only, "result": out}))
        return

    # ---- build the workload (untimed): L layers x 7 compressed matrices, replicas on every rank
    layers, alg_bytes = [], []
    for l in range(args.layers):
        ws, nb = {}, 0.0
        for name in NAMES:
            W = torch.from_numpy(hq_synth.llama_weight(l, name)).to(dev).to(torch.bfloat16)
            w = ctx.encode_weights(W, hq.Lattice.E8, 128, SNR_E8_4BPS, seed=l)
            del W
            ws[name] = w
            nb += (w.info.payload_bits + w.info.norm_bits + w.info.length_bits) / 8.0 + 2 * (w.n_in + w.m)
        layers.append(ws)
        alg_bytes.append(nb)
    bytes_per_step = float(np.mean(alg_bytes))
    scalars_per_step = sum(m * n for m, n in hq_synth.LLAMA_SHAPES.values())
    bps_total = 8.0 * np.mean([sum((w.info.payload_bits + w.info.norm_bits + w.info.length_bits) / 8.0
                                   for w in ws.values()) for ws in layers]) / scalars_per_step
    bps_payload = np.mean([sum(w.info.payload_bits for w in ws.values()) for ws in layers]) / scalars_per_step

    def make_io(B):
        xs = {n_in: torch.from_numpy(hq_synth.activations(B, n_in, seed=77 + n_in)).to(dev).to(torch.bfloat16)
              for n_in in (4096, 14336)}
        ys = {name: torch.empty((B, hq_synth.LLAMA_SHAPES[name][0]), dtype=torch.bfloat16, device=dev) for name in NAMES}
        return xs, ys

    GROUPS = [["q", "k", "v"], ["o"], ["gate", "up"], ["down"]]   # matrices that share an input share a launch

    def step(i, xs, ys):
        ws = layers[i % args.layers]
        for g in GROUPS:
            ctx.linear_group([ws[n] for n in g], xs[ws[g[0]].n_in], ys=[ys[n] for n in g])

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    def timed(B, steps, warmup, profile=False, graph=True):
        """K steps between two CUDA events on the launching stream.  graph=True replays one captured CUDA graph per
        layer (the seven hq_linear calls of a step, exactly the kernels the eager path launches); the per-kernel
        profile pass runs eagerly with the library's own event brackets."""
        xs, ys = make_io(B)
        st = torch.cuda.Stream(device=dev)
        with torch.cuda.stream(st):
            for i in range(max(warmup, args.layers)):
                step(i, xs, ys)
            st.synchronize()
            graphs = None
            if graph and not profile:
                graphs = []
                for l in range(args.layers):
                    g = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(g, stream=st):
                        step(l, xs, ys)
                    graphs.append(g)
                for l in range(args.layers):
                    graphs[l].replay()
            barrier()
            ctx.profile(profile)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            for i in range(steps):
                if graphs is not None:
                    graphs[(warmup + i) % args.layers].replay()
                else:
                    step(warmup + i, xs, ys)
            e1.record(st)
            barrier()
        ms = e0.elapsed_time(e1)
        kern = ctx.profile_read() if profile else (0.0, 0)
        ctx.profile(False)
        ms = max_over_ranks(ms, dev)
        return ms, kern

    # ---- headline: batch 1, device-resident inputs
    sampler = ClockSampler(local)
    sampler.start()
    ms, _ = timed(1, args.steps, args.warmup)
    ms_per_step = ms / args.steps
    value = aggregate_value(bytes_per_step, ms_per_step, world)

    # ---- roofline of the dominant kernel.  At batch 1 a step IS four launches of k_gemv_e8 and nothing else (the
    # activation cast, the decode, the MMA and the split-K reduction are one kernel), so the kernel's average launch
    # duration in the schedule the step runs in (graph replay, PDL between the launches) is ms_per_step / 4: kernel
    # time == step time by construction.  The eager per-launch bracket (library events around every launch, no overlap)
    # is reported beside it.
    ms_p, (kern_ms, kern_n) = timed(1, args.steps, 2, profile=True)
    peak, peak_src = peaks()
    n_launch = len(GROUPS)
    achieved = bytes_per_step / (ms_per_step * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": None, "alg_bytes_per_launch": bytes_per_step / n_launch,
                "kernel": "k_gemv_e8<K=2,NWG=5> (one launch per hq_linear_group; 4 per step)", "peak_source": peak_src,
                "avg_launch_us": 1e3 * ms_per_step / n_launch, "launches_per_step": n_launch,
                "timing": "CUDA events around K graph replays on the launching stream; the step holds only this kernel",
                "eager_avg_launch_us": 1e3 * kern_ms / max(kern_n, 1), "eager_launches_timed": kern_n,
                "alg_bytes_per_scalar": bytes_per_step / scalars_per_step,
                "frac_of_nominal_8TBs": achieved / 8000.0}
    clocks_now = sampler.summary()
    sm_clock_hz = 1e6 * float(clocks_now["sm_mhz"] or 1965)
    n_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    budget = n_sms * 128 * sm_clock_hz / (0.70 * peak * 1e9 / (bytes_per_step / scalars_per_step))
    roofline["co_bound"] = {"bound": "alu", "unit": "warp-instr/clk/SM", "peak": 4.0,
                            "budget_for_70pct_hbm_lane_instr_per_scalar": budget,
                            "peak_source": "profiles/r01_issue_rates.md (4 warp-instructions per clock per SM)"}
    if os.path.exists(NCU_STEP_JSON):   # written by the ncu pass of a named commit: profiles/r02_ncu_step.md
        nc = json.load(open(NCU_STEP_JSON))
        roofline["traffic"] = nc["dram_bytes_per_step"] / n_launch
        roofline["traffic_source"] = f"ncu --set full at commit {nc['commit']} ({os.path.relpath(NCU_STEP_JSON, ROOT)})"
        ipc = nc["warp_instr_per_step"] / (ms_per_step * 1e-3 * n_sms * sm_clock_hz)
        roofline["co_bound"].update({"achieved": ipc, "frac": ipc / 4.0,
                                     "lane_instr_per_scalar": nc["warp_instr_per_step"] * 32 / scalars_per_step,
                                     "source": roofline["traffic_source"]})
    # the decode-only ceiling, measured live: the fused kernel's decode phases on register-resident data
    try:
        ceil = layers[0]["q"].decode_ceiling(200)
        roofline["decode_ceiling"] = {"scalars_per_s": ceil, "equivalent_GBps": ceil * bytes_per_step / scalars_per_step / 1e9,
                                      "frac_of_hbm_peak": ceil * bytes_per_step / scalars_per_step / 1e9 / peak,
                                      "what": "hq_measure_decode_ceiling: phase 1 + phase 2 only, no loads, no MMA (profiles/r02_decode_ceiling.md)"}
    except Exception as ex:  # noqa: BLE001
        roofline["decode_ceiling"] = f"failed: {ex}"

    # ---- end to end: host (pinned) x -> device, linears, y -> host, every step.  The step's two activation vectors
    # live in one pinned buffer and its seven outputs in one device / one pinned buffer, so a step is ONE H2D copy,
    # four grouped launches and ONE D2H copy.
    offs, tot_m = {}, 0
    for name in NAMES:
        offs[name] = tot_m
        tot_m += hq_synth.LLAMA_SHAPES[name][0]
    xbuf = torch.empty((1, 4096 + 14336), dtype=torch.bfloat16, device=dev)
    ybuf = torch.empty((1, tot_m), dtype=torch.bfloat16, device=dev)
    hxbuf = torch.cat([torch.from_numpy(hq_synth.activations(1, n, seed=77 + n)) for n in (4096, 14336)], dim=1) \
        .to(torch.bfloat16).pin_memory()
    hybuf = torch.empty((1, tot_m), dtype=torch.bfloat16).pin_memory()
    xs = {4096: xbuf[:, :4096], 14336: xbuf[:, 4096:]}
    ys = {name: ybuf[:, offs[name]:offs[name] + hq_synth.LLAMA_SHAPES[name][0]] for name in NAMES}
    h2d = hxbuf.numel() * 2
    d2h = hybuf.numel() * 2

    def e2e_step(i):
        ws = layers[i % args.layers]
        xbuf.copy_(hxbuf, non_blocking=True)
        for g in GROUPS:
            ctx.linear_group([ws[n] for n in g], xs[ws[g[0]].n_in], ys=[ys[n] for n in g])
        hybuf.copy_(ybuf, non_blocking=True)
    # one CUDA graph per layer, like the device-resident arm: H2D copy nodes from pinned host memory, the four grouped
    # launches, D2H copy nodes to pinned host memory; wall clock around K replays + the final synchronize
    st2 = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(st2):
        for i in range(max(3, args.layers)):
            e2e_step(i)
        st2.synchronize()
        e2e_graphs = []
        for l in range(args.layers):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st2):
                e2e_step(l)
            e2e_graphs.append(g)
        for l in range(args.layers):
            e2e_graphs[l].replay()
        barrier()
        t0 = time.perf_counter()
        for i in range(args.steps):
            e2e_graphs[i % args.layers].replay()
        st2.synchronize()
        e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, dev)
    sampler.stop_flag = True   # clocks were sampled over the three timed passes (headline, per-kernel, end to end)
    sampler.join()
    e2e = {"value": world * bytes_per_step * args.steps / e2e_s / 1e9, "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h}

    extras = {}
    if not args.skip_extras and rank == 0:
        # batch 16 on the same weights (also part of BASELINE configs[1])
        n16 = max(4, args.steps // 2)
        ms16, _ = timed(16, n16, 2)
        g16 = bytes_per_step / (ms16 / n16 * 1e-3) / 1e9
        roofline["batch16"] = {"bound": "hbm", "unit": "GB/s", "achieved": g16, "peak": peak, "frac": g16 / peak,
                               "ms_per_step": ms16 / n16, "kernel": "k_act_blob + k_linear_e8<NB=16> per group"}
        # practical baseline on the same box: bf16 GEMV by cuBLAS on uncompressed weights (one layer, cycled 4x)
        try:
            dense = [{n: torch.randn(hq_synth.LLAMA_SHAPES[n], device=dev, dtype=torch.bfloat16) * 0.02 for n in NAMES}
                     for _ in range(2)]
            xs1, _ = make_io(1)
            for i in range(3):
                for n in NAMES:
                    torch.matmul(xs1[dense[0][n].shape[1]], dense[i % 2][n].t())
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for i in range(10):
                for n in NAMES:
                    torch.matmul(xs1[dense[0][n].shape[1]], dense[i % 2][n].t())
            e1.record()
            torch.cuda.synchronize()
            extras["cublas_bf16_gemv_ms_per_layer"] = e0.elapsed_time(e1) / 10
            del dense
        except Exception as ex:  # noqa: BLE001
            extras["cublas_bf16_gemv_ms_per_layer"] = f"failed: {ex}"
        if world == 1:
            for key, fn in (("large_m", lambda: measure_large_m(ctx, hq, dev)),
                            ("attend", lambda: measure_attend(ctx, hq, dev, peak)),
                            ("layer_step", lambda: measure_layer_step(ctx, hq, dev, layers, peak))):
                try:
                    roofline[key] = fn()
                except Exception as ex:  # noqa: BLE001
                    roofline[key] = f"failed: {ex}"
            try:
                extras["config3_sweep"] = measure_config3(ctx, hq, dev)
            except Exception as ex:  # noqa: BLE001
                extras["config3_sweep"] = f"failed: {ex}"

    # ---- CPU baseline: the oracle on a bounded sample, rank 0, N=1 only
    cpu = None
    if rank == 0 and world == 1:
        one_pass, nbytes, sample = oracle_sample()
        one_pass()
        reps, t0 = 0, time.perf_counter()
        while time.perf_counter() - t0 < 12.0 and reps < 100000:   # about 12 s of CPU work on the bounded sample
            one_pass()
            reps += 1
        dt = time.perf_counter() - t0
        cpu = {"value": nbytes * reps / dt / 1e9, "unit": UNIT, "cores": len(os.sched_getaffinity(0)), "kind": "oracle",
               "sample": f"{sample}; {reps} passes in {dt:.1f} s"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "int8", "data": "synthetic",
                "config": base_config(args.layers),
                "rate": {"bits_per_scalar_payload": bps_payload, "bits_per_scalar_total": bps_total},
                "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": args.steps * len(GROUPS),
                "roofline": roofline, "cpu_baseline": cpu, "extras": extras}
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
