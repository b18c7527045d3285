"""ctypes binding of libhq.so (include/hq.h).  Argument marshalling only."""
import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
HQ_F32, HQ_BF16 = 0, 1


class Lattice:
    Z, A2, D4, E8 = 1, 2, 4, 8
    BY_NAME = {"Z": 1, "A2": 2, "D4": 4, "E8": 8}


class HQError(RuntimeError):
    pass


_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_void_p, C.c_size_t)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class _Allocator(C.Structure):
    _fields_ = [("alloc", _ALLOC_FN), ("free", _FREE_FN), ("user", C.c_void_p)]


class _CodecConfig(C.Structure):
    _fields_ = [("lattice", C.c_int32), ("n_tile", C.c_int32), ("snr_db", C.c_float), ("rice_k", C.c_int32 * 2),
                ("seed", C.c_uint64)]


class _KVConfig(C.Structure):
    _fields_ = [("kv_heads", C.c_int32), ("head_dim", C.c_int32), ("max_tokens", C.c_int64), ("codec", _CodecConfig),
                ("rotation", C.c_int32), ("dither", C.c_int32), ("window", C.c_int32), ("una_capacity_bits", C.c_int64),
                ("qjl_dev", C.c_void_p), ("device_position", C.c_int32)]


class _WeightInfo(C.Structure):
    _fields_ = [("m_out", C.c_int64), ("n_in", C.c_int64), ("lattice", C.c_int32), ("n_tile", C.c_int32),
                ("rice_k", C.c_int32 * 2), ("snr_db", C.c_float), ("alpha", C.c_double), ("seed", C.c_uint64),
                ("payload_bits", C.c_int64), ("norm_bits", C.c_int64), ("length_bits", C.c_int64),
                ("blob_bytes", C.c_int64), ("n_groups", C.c_int64), ("clamp_count", C.c_int64)]


class _Stats(C.Structure):
    _fields_ = [("payload_bits", C.c_int64), ("norm_bits", C.c_int64), ("length_bits", C.c_int64),
                ("offset_bits", C.c_int64), ("padding_bits", C.c_int64), ("clamp_count", C.c_int64),
                ("n_tiles", C.c_int64), ("tile_bits_min", C.c_int32), ("tile_bits_max", C.c_int32),
                ("bits_per_scalar_payload", C.c_double), ("bits_per_scalar_total", C.c_double)]


class WeightHeader(C.Structure):
    _fields_ = [("magic", C.c_uint32), ("version", C.c_uint32), ("m_out", C.c_int64), ("n_in", C.c_int64),
                ("lattice", C.c_int32), ("n_tile", C.c_int32), ("rice_k", C.c_int32 * 2), ("snr_db", C.c_float),
                ("seed", C.c_uint64), ("blob_bytes", C.c_int64), ("n_groups", C.c_int64),
                ("payload_bits", C.c_int64), ("clamp_count", C.c_int64), ("ulen_min", C.c_int32),
                ("ulen_max", C.c_int32)]


class _Fold(C.Structure):
    _fields_ = [("mode", C.c_int32), ("eps", C.c_float), ("aux_dev", C.c_void_p), ("residuals_dev", C.POINTER(C.c_void_p))]


class _Layer(C.Structure):
    _fields_ = [("wq", C.c_void_p), ("wk", C.c_void_p), ("wv", C.c_void_p), ("wo", C.c_void_p), ("wgate", C.c_void_p),
                ("wup", C.c_void_p), ("wdown", C.c_void_p), ("g_attn_dev", C.c_void_p), ("g_mlp_dev", C.c_void_p),
                ("eps", C.c_float), ("kv", C.c_void_p), ("q_heads", C.c_int32)]


class _LayerScratch(C.Structure):
    _fields_ = [(n, C.c_size_t) for n in ("q", "k", "v", "a", "h2", "gate", "up", "total")]


FOLD_NONE, FOLD_RMSNORM, FOLD_SILU_MUL = 0, 1, 2
CAST_INT8, CAST_FP8_E4M3 = 0, 1


class _KVView(C.Structure):
    _fields_ = [("n_tokens", C.c_int64), ("rbits", C.c_int64), ("rem_dev", C.c_void_p), ("una_dev", C.c_void_p),
                ("ulen_dev", C.c_void_p), ("norm_dev", C.c_void_p), ("blk_off_dev", C.c_void_p),
                ("upos_dev", C.c_void_p), ("rem_words", C.c_int64), ("una_words", C.c_int64),
                ("clamp_count", C.c_int64)]


def lib_path() -> str:
    return os.path.join(HERE, "libhq.so")


_lib = None

EXPORTS = ["hq_create", "hq_destroy", "hq_last_error", "hq_measure_decode_ceiling", "hq_alpha", "hq_snr_for_bps", "hq_profile_enable", "hq_profile_read",
           "hq_encode_weights", "hq_weight_free", "hq_weight_get_info", "hq_weight_stats", "hq_weight_export",
           "hq_weight_export_host", "hq_weight_import", "hq_decode_int8", "hq_act_quant", "hq_linear",
           "hq_linear_cast", "hq_linear_group", "hq_linear_group_fold", "hq_layer_scratch_view", "hq_layer_decode", "hq_linear_static", "hq_linear_workspace_bytes", "hq_kv_create", "hq_kv_free", "hq_kv_append", "hq_kv_sync_position", "hq_attend", "hq_kv_export",
           "hq_kv_decode_int8"]


def load_library():
    """dlopen libhq.so; fails loudly if it has not been built (python -m paper_2606_23406_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise HQError(f"{path} is missing: build it with `python -m paper_2606_23406_b200.build` (no CPU fallback)")
    lib = C.CDLL(path)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    lib.hq_create.argtypes = [C.POINTER(vp), C.POINTER(_Allocator), C.c_int]
    lib.hq_destroy.argtypes = [vp]; lib.hq_destroy.restype = None
    lib.hq_last_error.argtypes = [vp]; lib.hq_last_error.restype = C.c_char_p
    lib.hq_alpha.argtypes = [i32, C.c_double]; lib.hq_alpha.restype = C.c_double
    lib.hq_snr_for_bps.argtypes = [vp, i32, C.c_double, C.POINTER(C.c_float), C.POINTER(i32)]
    lib.hq_weight_stats.argtypes = [vp, C.POINTER(_Stats)]
    lib.hq_weight_export_host.argtypes = [vp, vp, C.POINTER(WeightHeader), vp, vp, vp]
    lib.hq_weight_import.argtypes = [vp, C.POINTER(WeightHeader), vp, vp, vp, C.POINTER(vp)]
    lib.hq_measure_decode_ceiling.argtypes = [vp, vp, i32, vp, C.POINTER(C.c_double)]
    lib.hq_profile_enable.argtypes = [vp, i32]
    lib.hq_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(i64)]
    lib.hq_encode_weights.argtypes = [vp, vp, i32, i64, i64, i64, C.POINTER(_CodecConfig), vp, C.POINTER(vp)]
    lib.hq_weight_free.argtypes = [vp, vp]; lib.hq_weight_free.restype = None
    lib.hq_weight_get_info.argtypes = [vp, C.POINTER(_WeightInfo)]
    lib.hq_weight_export.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
    lib.hq_decode_int8.argtypes = [vp, vp, vp, vp, vp]
    lib.hq_act_quant.argtypes = [vp, vp, vp, i32, i64, i64, vp, vp, vp, vp]
    lib.hq_linear.argtypes = [vp, vp, vp, i32, i64, i64, vp, i64, vp, vp, vp]
    lib.hq_linear_cast.argtypes = [vp, vp, vp, i32, i64, i64, vp, i64, vp, vp, i32, vp]
    lib.hq_linear_static.argtypes = [vp, vp, vp, i32, vp, vp, vp]
    lib.hq_linear_group.argtypes = [vp, C.POINTER(vp), i32, vp, i32, i64, i64, C.POINTER(vp), C.POINTER(i64), C.POINTER(vp), vp]
    lib.hq_linear_group_fold.argtypes = [vp, C.POINTER(vp), i32, vp, C.POINTER(_Fold), C.POINTER(vp), C.POINTER(vp), vp]
    lib.hq_layer_scratch_view.argtypes = [C.POINTER(_Layer), C.POINTER(_LayerScratch)]
    lib.hq_layer_decode.argtypes = [vp, C.POINTER(_Layer), vp, vp, vp, C.c_size_t, vp]
    lib.hq_linear_workspace_bytes.argtypes = [vp, i64, C.POINTER(C.c_size_t)]
    lib.hq_kv_create.argtypes = [vp, C.POINTER(_KVConfig), C.POINTER(vp)]
    lib.hq_kv_free.argtypes = [vp, vp]; lib.hq_kv_free.restype = None
    lib.hq_kv_append.argtypes = [vp, vp, vp, vp, i64, vp]
    lib.hq_kv_sync_position.argtypes = [vp, vp, C.POINTER(i64)]
    lib.hq_attend.argtypes = [vp, vp, vp, i32, vp, vp, vp]
    lib.hq_kv_export.argtypes = [vp, vp, C.POINTER(_KVView)]
    lib.hq_kv_decode_int8.argtypes = [vp, vp, i32, i64, i64, vp, vp]
    _lib = lib
    return lib


def alpha(lattice: int, snr_db: float) -> float:
    return load_library().hq_alpha(lattice, float(snr_db))


def snr_for_bps(lattice: int, target_bps: float):
    """(snr_db as the float32 the codec config carries, (k0, k1)) from the library's calibration table (host only)."""
    snr, k = C.c_float(), (C.c_int32 * 2)()
    st = load_library().hq_snr_for_bps(None, lattice, float(target_bps), C.byref(snr), k)
    if st != 0:
        raise HQError(f"hq_snr_for_bps: status {st} (target outside the table's range?)")
    return float(snr.value), (int(k[0]), int(k[1]))


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.float32:
        return HQ_F32
    if t.dtype == torch.bfloat16:
        return HQ_BF16
    raise HQError(f"unsupported dtype {t.dtype}")


def _stream_ptr(device) -> int:
    return torch.cuda.current_stream(device).cuda_stream


class Context:
    """hq_ctx with device memory lent by torch's caching allocator."""

    def __init__(self, device: int = 0):
        if not torch.cuda.is_available():
            raise HQError("no CUDA device: libhq has no CPU fallback")
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        self._live = {}

        def _alloc(user, nbytes):
            try:
                t = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
            except Exception:
                return None
            self._live[t.data_ptr()] = t
            return t.data_ptr()

        def _free(user, ptr):
            self._live.pop(ptr, None)

        self._alloc_cb, self._free_cb = _ALLOC_FN(_alloc), _FREE_FN(_free)
        self._allocator = _Allocator(self._alloc_cb, self._free_cb, None)
        h = C.c_void_p()
        st = self.lib.hq_create(C.byref(h), C.byref(self._allocator), device)
        if st != 0:
            raise HQError(f"hq_create failed with status {st} (needs an sm_100 device)")
        self.h = h

    def check(self, st: int):
        if st != 0:
            raise HQError(f"libhq status {st}: {self.lib.hq_last_error(self.h).decode()}")

    def profile(self, on: bool):
        self.check(self.lib.hq_profile_enable(self.h, 1 if on else 0))

    def profile_read(self):
        """(summed ms of the bracketed dominant kernels, their count) since the last read."""
        ms, n = C.c_double(), C.c_int64()
        self.check(self.lib.hq_profile_read(self.h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def close(self):
        if getattr(self, "h", None):
            self.lib.hq_destroy(self.h)
            self.h = None

    # ---- weights ----
    def encode_weights(self, W: torch.Tensor, lattice: int, n_tile: int, snr_db: float, seed: int, rice_k=(-1, -1)):
        assert W.is_cuda and W.dim() == 2 and W.stride(1) == 1
        cfg = _CodecConfig(lattice, n_tile, float(snr_db), (C.c_int32 * 2)(int(rice_k[0]), int(rice_k[1])), seed)
        h = C.c_void_p()
        self.check(self.lib.hq_encode_weights(self.h, W.data_ptr(), _dtype_code(W), W.shape[0], W.shape[1],
                                              W.stride(0), C.byref(cfg), _stream_ptr(self.device), C.byref(h)))
        return Weight(self, h)

    def linear_group(self, weights, x: torch.Tensor, ys=None, want_f32=False):
        """[w_i x for w_i in weights] in one fused launch (weights that share x: q/k/v, gate/up)."""
        n = len(weights)
        assert 1 <= n <= 4 and x.is_cuda and x.dim() == 2 and x.stride(1) == 1
        B = x.shape[0]
        if ys is None:
            ys = [torch.empty((B, w.m), dtype=torch.bfloat16, device=self.device) for w in weights]
        y32 = [torch.empty((B, w.m), dtype=torch.float32, device=self.device) for w in weights] if want_f32 else None
        wa = (C.c_void_p * n)(*[w.h for w in weights])
        ya = (C.c_void_p * n)(*[y.data_ptr() for y in ys])
        la = (C.c_int64 * n)(*[y.stride(0) for y in ys])
        fa = (C.c_void_p * n)(*[t.data_ptr() for t in y32]) if want_f32 else None
        self.check(self.lib.hq_linear_group(self.h, wa, n, x.data_ptr(), _dtype_code(x), B, x.stride(0), ya, la, fa,
                                            _stream_ptr(self.device)))
        return (ys, y32) if want_f32 else ys

    def linear_group_fold(self, weights, x: torch.Tensor, mode=FOLD_NONE, aux: torch.Tensor = None, eps=0.0,
                          residuals=None, ys=None, want_f32=False):
        """hq_linear_group_fold: batch-1 linears with RMSNorm / SiLU.mul folded into the prologue and an optional
        residual add in the epilogue (x, aux, residuals: bf16 vectors)."""
        n = len(weights)
        assert 1 <= n <= 4 and x.is_cuda and x.dtype == torch.bfloat16 and x.dim() == 1 and x.is_contiguous()
        if ys is None:
            ys = [torch.empty((w.m,), dtype=torch.bfloat16, device=self.device) for w in weights]
        y32 = [torch.empty((w.m,), dtype=torch.float32, device=self.device) for w in weights] if want_f32 else None
        wa = (C.c_void_p * n)(*[w.h for w in weights])
        ya = (C.c_void_p * n)(*[y.data_ptr() for y in ys])
        fa = (C.c_void_p * n)(*[t.data_ptr() for t in y32]) if want_f32 else None
        ra = (C.c_void_p * n)(*[(r.data_ptr() if r is not None else None) for r in residuals]) if residuals else None
        fold = _Fold(int(mode), float(eps), aux.data_ptr() if aux is not None else None, ra)
        self.check(self.lib.hq_linear_group_fold(self.h, wa, n, x.data_ptr(), C.byref(fold), ya, fa, _stream_ptr(self.device)))
        return (ys, y32) if want_f32 else ys

    def layer(self, wq, wk, wv, wo, wgate, wup, wdown, g_attn: torch.Tensor, g_mlp: torch.Tensor, eps, kv, q_heads):
        return Layer(self, (wq, wk, wv, wo, wgate, wup, wdown), g_attn, g_mlp, eps, kv, q_heads)

    def import_weight(self, header: "WeightHeader", blob, sub_off):
        """hq_weight_import from host numpy arrays (the pair Weight.export_host returns)."""
        import numpy as np
        blob = np.ascontiguousarray(blob, dtype=np.uint8); sub_off = np.ascontiguousarray(sub_off, dtype=np.uint32)
        h = C.c_void_p()
        self.check(self.lib.hq_weight_import(self.h, C.byref(header), blob.ctypes.data, sub_off.ctypes.data,
                                             _stream_ptr(self.device), C.byref(h)))
        return Weight(self, h)

    # ---- KV ----
    def kv_create(self, kv_heads, head_dim, max_tokens, lattice, snr_db, rice_k, seed, rotation=1, dither=1,
                  window=32, una_capacity_bits=0, qjl: torch.Tensor = None, device_position=False):
        """rotation 2 (qjl): `qjl` = the Haar matrix S [head_dim, head_dim] fp32 on the device (copied by the library)."""
        codec = _CodecConfig(lattice, head_dim, float(snr_db), (C.c_int32 * 2)(int(rice_k[0]), int(rice_k[1])), seed)
        if qjl is not None:
            assert qjl.is_cuda and qjl.dtype == torch.float32 and qjl.is_contiguous() and tuple(qjl.shape) == (head_dim, head_dim)
        cfg = _KVConfig(kv_heads, head_dim, max_tokens, codec, rotation, dither, window, int(una_capacity_bits),
                        qjl.data_ptr() if qjl is not None else None, 1 if device_position else 0)
        h = C.c_void_p()
        self.check(self.lib.hq_kv_create(self.h, C.byref(cfg), C.byref(h)))
        return KVCache(self, h, kv_heads, head_dim, max_tokens)


class Weight:
    def __init__(self, ctx: Context, h):
        self.ctx, self.h = ctx, h
        info = _WeightInfo()
        ctx.check(ctx.lib.hq_weight_get_info(h, C.byref(info)))
        self.info = info
        self.m, self.n_in, self.n_tile = info.m_out, info.n_in, info.n_tile
        self.k = (info.rice_k[0], info.rice_k[1])

    def free(self):
        if self.h:
            self.ctx.lib.hq_weight_free(self.ctx.h, self.h)
            self.h = None

    def export(self):
        """(blob uint8 [blob_bytes], sub_off uint32 [n_groups+1]) as host numpy arrays (FORMAT §5)."""
        blob_p, goff_p = C.c_void_p(), C.c_void_p()
        self.ctx.check(self.ctx.lib.hq_weight_export(self.h, C.byref(blob_p), C.byref(goff_p)))
        torch.cuda.synchronize(self.ctx.device)
        blob = _wrap(blob_p.value, self.info.blob_bytes, self.ctx.device).cpu().numpy()
        goff = _wrap(goff_p.value, (self.info.n_groups + 1) * 4, self.ctx.device).cpu().numpy().view("uint32")
        return blob, goff

    def decode_ceiling(self, reps=200):
        """Decode-only issue ceiling of the E8 decoder on this weight's data (scalars per second)."""
        v = C.c_double()
        self.ctx.check(self.ctx.lib.hq_measure_decode_ceiling(self.ctx.h, self.h, reps, _stream_ptr(self.ctx.device),
                                                              C.byref(v)))
        return v.value

    def stats(self):
        st = _Stats()
        self.ctx.check(self.ctx.lib.hq_weight_stats(self.h, C.byref(st)))
        return st

    def export_host(self):
        """(header, blob uint8, sub_off uint32): the encoded weight as host data (hq_weight_export_host)."""
        import numpy as np
        hd = WeightHeader()
        self.ctx.check(self.ctx.lib.hq_weight_export_host(self.ctx.h, self.h, C.byref(hd), None, None, None))
        blob = np.empty(hd.blob_bytes, np.uint8); goff = np.empty(hd.n_groups + 1, np.uint32)
        self.ctx.check(self.ctx.lib.hq_weight_export_host(self.ctx.h, self.h, C.byref(hd), blob.ctypes.data,
                                                          goff.ctypes.data, _stream_ptr(self.ctx.device)))
        return hd, blob, goff

    def decode_int8(self):
        dev = self.ctx.device
        codes = torch.empty((self.m, self.n_in), dtype=torch.int8, device=dev)
        norms = torch.empty((self.m, self.n_in // self.n_tile), dtype=torch.int16, device=dev)
        self.ctx.check(self.ctx.lib.hq_decode_int8(self.ctx.h, self.h, codes.data_ptr(), norms.data_ptr(),
                                                   _stream_ptr(dev)))
        return codes, norms

    def act_quant(self, x: torch.Tensor, want_u=False):
        dev = self.ctx.device
        assert x.is_cuda and x.dim() == 2 and x.shape[1] == self.n_in and x.stride(1) == 1
        B = x.shape[0]
        q = torch.empty((B, self.n_in), dtype=torch.int8, device=dev)
        s_x = torch.empty((B, self.n_in // self.n_tile), dtype=torch.float32, device=dev)
        u = torch.empty((B, self.n_in), dtype=torch.float32, device=dev) if want_u else None
        self.ctx.check(self.ctx.lib.hq_act_quant(self.ctx.h, self.h, x.data_ptr(), _dtype_code(x), B, x.stride(0),
                                                 q.data_ptr(), s_x.data_ptr(), u.data_ptr() if want_u else None,
                                                 _stream_ptr(dev)))
        return (q, s_x, u) if want_u else (q, s_x)

    def linear(self, x: torch.Tensor, y: torch.Tensor = None, want_f32=False, want_acc=False):
        """y = Ŵ x through the fused decode + INT8 MMA kernel. x [B, n_in] (bf16 or f32) -> y [B, m] bf16."""
        dev = self.ctx.device
        assert x.is_cuda and x.dim() == 2 and x.shape[1] == self.n_in and x.stride(1) == 1
        B = x.shape[0]
        if y is None:
            y = torch.empty((B, self.m), dtype=torch.bfloat16, device=dev)
        y32 = torch.empty((B, self.m), dtype=torch.float32, device=dev) if want_f32 else None
        acc = torch.empty((self.n_in // self.n_tile, B, self.m), dtype=torch.int32, device=dev) if want_acc else None
        self.ctx.check(self.ctx.lib.hq_linear(self.ctx.h, self.h, x.data_ptr(), _dtype_code(x), B, x.stride(0),
                                              y.data_ptr(), y.stride(0), y32.data_ptr() if want_f32 else None,
                                              acc.data_ptr() if want_acc else None, _stream_ptr(dev)))
        if want_f32 or want_acc:
            return y, y32, acc
        return y


    def linear_cast(self, x: torch.Tensor, cast: int, y: torch.Tensor = None, want_f32=False, want_acc=False):
        """hq_linear_cast: cast 0 = INT8 (hq_linear), 1 = FP8-E4M3 operands with an fp32 tensor-core accumulator."""
        dev = self.ctx.device
        assert x.is_cuda and x.dim() == 2 and x.stride(1) == 1
        B = x.shape[0]
        if y is None:
            y = torch.empty((B, self.m), dtype=torch.bfloat16, device=dev)
        y32 = torch.empty((B, self.m), dtype=torch.float32, device=dev) if want_f32 else None
        acc = None
        if want_acc:   # [n_kt, B, m]: int32 (INT8 cast) or the fp32 tensor-core accumulator (FP8 cast)
            acc = torch.empty((self.n_in // self.n_tile, B, self.m), dtype=torch.float32 if cast == CAST_FP8_E4M3 else torch.int32,
                              device=dev)
        self.ctx.check(self.ctx.lib.hq_linear_cast(self.ctx.h, self.h, x.data_ptr(), _dtype_code(x), B, x.stride(0),
                                                   y.data_ptr(), y.stride(0), y32.data_ptr() if want_f32 else None,
                                                   acc.data_ptr() if want_acc else None, int(cast), _stream_ptr(dev)))
        if want_acc:
            return (y, y32, acc) if want_f32 else (y, acc)
        return (y, y32) if want_f32 else y

    def linear_static(self, x: torch.Tensor, y: torch.Tensor, y32: torch.Tensor = None):
        """hq_linear_static: one activation row, outputs given by the caller, no allocation anywhere in the call."""
        assert x.is_cuda and x.numel() == self.n_in and x.is_contiguous()
        assert y is None or (y.is_cuda and y.dtype == torch.bfloat16 and y.numel() == self.m and y.is_contiguous())
        assert y32 is None or (y32.is_cuda and y32.dtype == torch.float32 and y32.numel() == self.m and y32.is_contiguous())
        self.ctx.check(self.ctx.lib.hq_linear_static(self.ctx.h, self.h, x.data_ptr(), _dtype_code(x),
                                                     y.data_ptr() if y is not None else None,
                                                     y32.data_ptr() if y32 is not None else None, _stream_ptr(self.ctx.device)))
        return y


class Layer:
    """hq_layer / hq_layer_decode: one decode step of a decoder layer (seven launches, glue folded into the linears)."""

    def __init__(self, ctx: Context, weights, g_attn, g_mlp, eps, kv, q_heads):
        self.ctx, self.weights, self.g_attn, self.g_mlp, self.kv = ctx, weights, g_attn, g_mlp, kv
        self.c = _Layer(*[w.h for w in weights], g_attn.data_ptr(), g_mlp.data_ptr(), float(eps), kv.h, int(q_heads))
        self.view = _LayerScratch()
        ctx.check(ctx.lib.hq_layer_scratch_view(C.byref(self.c), C.byref(self.view)))
        self.scratch = torch.empty((self.view.total,), dtype=torch.uint8, device=ctx.device)

    def decode(self, h_in: torch.Tensor, h_out: torch.Tensor = None):
        assert h_in.is_cuda and h_in.dtype == torch.bfloat16 and h_in.is_contiguous()
        if h_out is None:
            h_out = torch.empty_like(h_in)
        self.ctx.check(self.ctx.lib.hq_layer_decode(self.ctx.h, C.byref(self.c), h_in.data_ptr(), h_out.data_ptr(),
                                                    self.scratch.data_ptr(), self.view.total, _stream_ptr(self.ctx.device)))
        return h_out

    def scratch_tensor(self, name):
        """bf16 view of one intermediate (q, k, v, a, h2, gate, up) of the last decode() - for parity tests."""
        w = self.weights
        n = {"q": w[0].m, "k": w[1].m, "v": w[2].m, "a": w[0].m, "h2": w[3].m, "gate": w[4].m, "up": w[5].m}[name]
        off = getattr(self.view, name)
        return self.scratch[off:off + 2 * n].view(torch.bfloat16)


class KVCache:
    def __init__(self, ctx: Context, h, kv_heads, head_dim, max_tokens):
        self.ctx, self.h = ctx, h
        self.kv_heads, self.head_dim, self.max_tokens = kv_heads, head_dim, max_tokens

    def free(self):
        if self.h:
            self.ctx.lib.hq_kv_free(self.ctx.h, self.h)
            self.h = None

    def append(self, k: torch.Tensor, v: torch.Tensor):
        assert k.is_cuda and k.dtype == torch.bfloat16 and k.is_contiguous() and v.is_contiguous() and k.shape == v.shape
        assert tuple(k.shape[1:]) == (self.kv_heads, self.head_dim)
        self.ctx.check(self.ctx.lib.hq_kv_append(self.ctx.h, self.h, k.data_ptr(), v.data_ptr(), k.shape[0],
                                                 _stream_ptr(self.ctx.device)))

    def sync_position(self) -> int:
        """hq_kv_sync_position: the held-token count (read back from the device for device_position caches)."""
        n = C.c_int64(0)
        self.ctx.check(self.ctx.lib.hq_kv_sync_position(self.ctx.h, self.h, C.byref(n)))
        return int(n.value)

    def attend(self, q: torch.Tensor, out: torch.Tensor = None, want_f32=False):
        dev = self.ctx.device
        assert q.is_cuda and q.dtype == torch.bfloat16 and q.is_contiguous() and q.shape[1] == self.head_dim
        if out is None:
            out = torch.empty_like(q)
        o32 = torch.empty(q.shape, dtype=torch.float32, device=dev) if want_f32 else None
        self.ctx.check(self.ctx.lib.hq_attend(self.ctx.h, self.h, q.data_ptr(), q.shape[0], out.data_ptr(),
                                              o32.data_ptr() if want_f32 else None, _stream_ptr(dev)))
        return (out, o32) if want_f32 else out

    def export(self):
        """Host copies of the FORMAT §6 container: dict of numpy arrays."""
        v = _KVView()
        self.ctx.check(self.ctx.lib.hq_kv_export(self.ctx.h, self.h, C.byref(v)))
        dev, H, mt = self.ctx.device, self.kv_heads, self.max_tokens
        n_blk = (mt + 127) // 128

        def arr(ptr, count, np_dtype, itemsize):
            return _wrap(ptr, count * itemsize, dev).cpu().numpy().view(np_dtype)

        return dict(
            n_tokens=v.n_tokens, rbits=v.rbits, clamp_count=v.clamp_count,
            rem=arr(v.rem_dev, 2 * H * v.rem_words, "uint32", 4).reshape(2, H, v.rem_words),
            una=arr(v.una_dev, 2 * H * v.una_words, "uint32", 4).reshape(2, H, v.una_words),
            ulen=arr(v.ulen_dev, 2 * H * mt, "uint16", 2).reshape(2, H, mt),
            norm=arr(v.norm_dev, 2 * H * mt, "uint16", 2).reshape(2, H, mt),
            blk_off=arr(v.blk_off_dev, 2 * H * (n_blk + 1), "uint32", 4).reshape(2, H, n_blk + 1),
            upos=arr(v.upos_dev, 2 * H, "uint32", 4).reshape(2, H))

    def decode_int8(self, role, t0, n):
        codes = torch.empty((n, self.kv_heads, self.head_dim), dtype=torch.int8, device=self.ctx.device)
        self.ctx.check(self.ctx.lib.hq_kv_decode_int8(self.ctx.h, self.h, role, t0, n, codes.data_ptr(),
                                                      _stream_ptr(self.ctx.device)))
        return codes


class _DevMem:
    """__cuda_array_interface__ view of raw device memory (no ownership)."""

    def __init__(self, ptr, nbytes):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def _wrap(ptr, nbytes, device):
    return torch.as_tensor(_DevMem(ptr, int(nbytes)), device=device)
