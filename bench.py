#!/usr/bin/env python
"""bench.py — HyperQuant hot path on B200: fused Rice-decode + tcgen05 INT8 GEMV over one Llama-3.1-8B-shaped
decoder layer's linears (BASELINE.json configs[1]: E8, 4 bps, RHT tile 128, batch 1), seeded synthetic weights.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--layers L] [--impl reference]

A step = the seven linears (q,k,v,o,gate,up,down) of one layer at batch 1 through hq_linear_group (matrices that
share an input share a launch: activation RHT + INT8 cast, fused decode+MMA, split-K finalize).  L distinct layers (L x ~116 MB compressed > the 126 MB L2) are
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
# dram__bytes_read.sum + dram__bytes_write.sum of the four k_linear_e8 launches of one step, from the ncu --set full
# capture summarised in profiles/r01c_e8_grouped_kernel.md §3 (14.01 + 9.40 + 64.73+0.57 + 32.62 MB)
NCU_DRAM_BYTES_PER_STEP = 121.34e6
# smsp__inst_executed.sum of the same four launches (10.24 + 7.17 + 43.85 + 22.43 M warp-instructions)
NCU_WARP_INSTR_PER_STEP = 83.69e6
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
            "config": {"workload": WORKLOAD, "lattice": "E8", "bps": 4.0, "n_tile": 128, "batch": 1},
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


def run_extras(ctx, hq, dev, peak_gbs):
    """The other BASELINE configs, each a bounded, seeded, synthetic run through the public API (parity for the
    same code paths is in tests/): config 5 (large-M INT8 TOPS), config 4 (KV append / attend), config 3 (reduced
    lattice / rate / tile sweep at batch 1)."""
    import torch
    out = {}
    # ---- config 5: 8192 tokens x (4096 -> 16384), E8 4 bps, tile 128, INT8 MMA
    try:
        W = torch.from_numpy(hq_synth.gaussian_weight(16384, 4096, seed=5)).to(dev).to(torch.bfloat16)
        w = ctx.encode_weights(W, hq.Lattice.E8, 128, SNR_E8_4BPS, seed=5)
        del W
        X = torch.from_numpy(hq_synth.activations(8192, 4096, seed=6)).to(dev).to(torch.bfloat16)
        y = torch.empty((8192, 16384), dtype=torch.bfloat16, device=dev)
        ms = _time_cuda(lambda: w.linear(X, y=y), reps=3)
        ops = 2.0 * 8192 * 16384 * 4096
        c5 = {"workload": "8192 tokens x 4096->16384, E8 4 bps, tile 128", "ms": ms, "int8_TOPS": ops / (ms * 1e-3) / 1e12,
              "nominal_dense_int8_TOPS": 4500.0}
        try:
            a = torch.randint(-127, 127, (8192, 8192), dtype=torch.int8, device=dev)
            b = torch.randint(-127, 127, (8192, 8192), dtype=torch.int8, device=dev)
            ms_mm = _time_cuda(lambda: torch._int_mm(a, b), reps=5, warm=2)
            c5["measured_int8_peak_TOPS_torch_int_mm_8192"] = 2.0 * 8192 ** 3 / (ms_mm * 1e-3) / 1e12
            c5["frac_of_measured_int8_peak"] = c5["int8_TOPS"] / c5["measured_int8_peak_TOPS_torch_int_mm_8192"]
            del a, b
        except Exception as ex:  # noqa: BLE001
            c5["measured_int8_peak_TOPS_torch_int_mm_8192"] = f"unavailable: {ex}"
        c5["frac_of_nominal_int8_peak"] = c5["int8_TOPS"] / 4500.0
        # Roofline of the large-M path: the INT8 tensor pipe.  peak = torch._int_mm measured beside it (a plain library
        # GEMM with one drain per output tile); this path must drain and rescale the INT32 accumulator once per K-tile of
        # 128 (both scales are per tile, PAPER §4.8), which costs >= 2 issue slots per accumulator (I2F + half of a packed
        # multiply and a packed FMA): DESIGN.md §6.3 derives that co-bound and profiles/r01d_large_m_path.md shows it.
        meas = c5.get("measured_int8_peak_TOPS_torch_int_mm_8192")
        peak = meas if isinstance(meas, float) else 4500.0
        c5["roofline"] = {"bound": "tensor", "achieved": c5["int8_TOPS"], "peak": peak, "unit": "TOPS",
                          "frac": c5["int8_TOPS"] / peak,
                          "peak_source": "torch._int_mm 8192^3 measured in this run" if isinstance(meas, float) else "nominal dense INT8",
                          "note": "whole call: activation blob + weight decode into the operand-layout scratch copy + GEMM"}
        c5["path"] = "k_act_blob + k_e8_decode_ablob + k_e8_gemm_large (hq_linear_large.cuh)"
        out["config5_large_m"] = c5
        w.free(); del X, y
    except Exception as ex:  # noqa: BLE001
        out["config5_large_m"] = f"failed: {ex}"
    # ---- config 4: KV cache, 8 heads x 128, 32768 tokens, E8 2 bps, signs rotation, dither, window 32
    try:
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
        att_ms = _time_cuda(lambda: kv.attend(q, out=o), reps=5)
        ex = kv.export()
        Tn = int(ex["n_tokens"])
        payload_bits = float(ex["upos"].astype(np.int64).sum()) + 2.0 * H * Tn * float(ex["rbits"])
        scal = 2.0 * H * Tn * d
        alg_bytes = (payload_bits + 32.0 * 2 * H * Tn) / 8.0
        out["config4_kv"] = {"workload": "8 KV heads x 128, 32768 tokens, E8 2 bps, signs rotation, dither, window 32; 32 query heads",
                             "bulk_append_Mscalars_per_s": 2.0 * H * T * d / bulk_s / 1e6, "append_us_per_token": app_us,
                             "attend_ms": att_ms, "attend_GBps_compressed": alg_bytes / (att_ms * 1e-3) / 1e9,
                             "attend_frac_of_hbm_roofline": alg_bytes / (att_ms * 1e-3) / 1e9 / peak_gbs,
                             "bits_per_scalar_payload": payload_bits / scal, "bits_per_scalar_total": 8.0 * alg_bytes / scal,
                             "kv_compression_vs_bf16": 16.0 / (8.0 * alg_bytes / scal)}
        kv.free(); del K, V
    except Exception as ex:  # noqa: BLE001
        out["config4_kv"] = f"failed: {ex}"
    # ---- config 3 (reduced): one 14336 x 4096 Gaussian weight; lattice x rate at tile 128, E8 4 bps at tiles 64 / 256
    try:
        Wn = hq_synth.gaussian_weight(14336, 4096, seed=3)
        W = torch.from_numpy(Wn).to(dev).to(torch.bfloat16)
        x = torch.from_numpy(hq_synth.activations(1, 4096, seed=9)).to(dev).to(torch.bfloat16)
        snr = {"E8": (16.50, 22.68, 28.73), "D4": (16.4, 22.5, 28.6), "A2": (16.02, 22.21, 28.26), "Z": (15.8, 21.9, 27.9)}
        combos = [(lat, s, 128) for lat in ("E8", "D4", "A2", "Z") for s in snr[lat]] + [("E8", 22.68, 64), ("E8", 22.68, 256)]
        rows = []
        for lat, s, n_tile in combos:
            s32 = float(np.float32(s))
            w = ctx.encode_weights(W, hq.Lattice.BY_NAME[lat], n_tile, s32, seed=3)
            info = w.info
            sc = float(info.m_out * info.n_in)
            yv = torch.empty((1, 14336), dtype=torch.bfloat16, device=dev)
            ms = _time_cuda(lambda: w.linear(x, y=yv), reps=5, warm=2)
            nbytes = (info.payload_bits + info.norm_bits + info.length_bits) / 8.0
            # MSE of the reconstruction, measured in the rotated domain (the RHT is orthonormal) on the first 512 rows
            R = 512
            _, _, u = w.act_quant(W[:R], want_u=True)
            codes, norms = w.decode_int8()
            c = codes[:R].float().view(R, -1, n_tile)
            if lat == "A2":
                c[..., 0::2] *= 3.0 ** 0.5
            rho = norms[:R].view(torch.float16).float()
            scale = rho / (info.alpha * n_tile ** 0.5)
            mse = float(((u.view(R, -1, n_tile) - scale[..., None] * c) ** 2).mean())
            pred = float((rho ** 2).mean() / n_tile / 10 ** (s32 / 10))
            rows.append({"lattice": lat, "snr_db": s, "n_tile": n_tile, "k": [info.rice_k[0], info.rice_k[1]],
                         "bits_payload": info.payload_bits / sc, "bits_total": 8.0 * nbytes / sc,
                         "mse": mse, "mse_predicted": pred, "gemv_us": 1e3 * ms, "GBps_compressed": nbytes / (ms * 1e-3) / 1e9})
            w.free()
        out["config3_sweep"] = rows
    except Exception as ex:  # noqa: BLE001
        out["config3_sweep"] = f"failed: {ex}"
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=4)
    ap.add_argument("--layers", type=int, default=4)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--skip-extras", action="store_true")
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

    # ---- roofline of the dominant kernel (fused decode+MMA), CUDA events around each launch
    ms_p, (kern_ms, kern_n) = timed(1, args.steps, 2, profile=True)
    weight_bytes_per_step = bytes_per_step
    achieved = weight_bytes_per_step * args.steps / (kern_ms * 1e-3) / 1e9 if kern_ms > 0 else 0.0
    peak, peak_src = peaks()
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": NCU_DRAM_BYTES_PER_STEP / len(GROUPS), "alg_bytes_per_launch": bytes_per_step / len(GROUPS),
                "traffic_source": "ncu --set full, profiles/r01c_e8_grouped_kernel.md", "kernel": "k_linear_e8<K=2,NB=16,BC=1,NWG=6,CPS=1> (one launch per hq_linear_group)", "peak_source": peak_src,
                "kernel_share_of_step": kern_ms / ms_p if ms_p > 0 else None,
                "launches_timed": kern_n, "avg_launch_us": 1e3 * kern_ms / max(kern_n, 1),
                "alg_bytes_per_scalar": bytes_per_step / scalars_per_step,
                "frac_of_nominal_8TBs": achieved / 8000.0}
    # co-bound: the kernel is limited by the ALU work of the Rice decode.  Issue rate achieved =
    # warp-instructions of the four launches (ncu) / (their summed duration x SMs x SM clock); peak = 4 warp-instr/clk/SM
    sm_clock_hz, n_sms = 1.965e9, 148
    kern_s_per_step = kern_ms * 1e-3 / args.steps if kern_ms > 0 else float("nan")
    ipc = NCU_WARP_INSTR_PER_STEP / (kern_s_per_step * n_sms * sm_clock_hz)
    roofline["co_bound"] = {"bound": "alu", "achieved": ipc, "peak": 4.0, "unit": "warp-instr/clk/SM", "frac": ipc / 4.0,
                            "lane_instr_per_scalar": NCU_WARP_INSTR_PER_STEP * 32 / scalars_per_step,
                            "budget_for_70pct_hbm_lane_instr_per_scalar": n_sms * 128 * sm_clock_hz /
                            (0.70 * peak * 1e9 / (bytes_per_step / scalars_per_step)),
                            "source": "instruction count: ncu, profiles/r01c_e8_grouped_kernel.md; peak: profiles/r01_issue_rates.md"}

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
        # batch 16 on the same weights
        ms16, _ = timed(16, max(4, args.steps // 2), 2)
        extras["batch16"] = {"ms_per_step": ms16 / max(4, args.steps // 2),
                             "GBps_compressed": bytes_per_step / (ms16 / max(4, args.steps // 2) * 1e-3) / 1e9}
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
            extras.update(run_extras(ctx, hq, dev, peaks()[0]))

    # ---- CPU baseline: the oracle on a bounded sample, rank 0, N=1 only
    cpu = None
    if rank == 0 and world == 1:
        one_pass, nbytes, sample = oracle_sample()
        one_pass()
        reps, t0 = 0, time.perf_counter()
        while time.perf_counter() - t0 < 10.0 and reps < 50:
            one_pass()
            reps += 1
        dt = time.perf_counter() - t0
        cpu = {"value": nbytes * reps / dt / 1e9, "unit": UNIT, "cores": len(os.sched_getaffinity(0)), "kind": "oracle",
               "sample": f"{sample}; {reps} passes in {dt:.1f} s"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "int8", "data": "synthetic",
                "config": {"workload": WORKLOAD, "lattice": "E8", "snr_db": SNR_E8_4BPS, "n_tile": 128, "batch": 1,
                           "layers_cycled": args.layers, "l2_policy": "inputs larger than L2 (layers cycled)", "launch": "one CUDA graph per layer: hq_linear_group x 4 (q+k+v, o, gate+up, down)",
                           "scalars_per_step": scalars_per_step, "bits_per_scalar_payload": bps_payload,
                           "bits_per_scalar_total": bps_total, "parallelism": "replicas only"},
                "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": args.steps * (len(GROUPS) * 2 + len(NAMES)),
                "roofline": roofline, "cpu_baseline": cpu, "extras": extras}
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
