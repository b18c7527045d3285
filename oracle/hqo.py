"""ctypes front end of the oracle (oracle/hq_oracle.c).  TEST INFRASTRUCTURE ONLY — see the C header.

Argument marshalling only; every step of the method is in the C file.  Never imported by the
product package.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

Z, A2, D4, E8 = 1, 2, 4, 8
LATTICES = {"Z": Z, "A2": A2, "D4": D4, "E8": E8}

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.hqo_alpha.restype = C.c_double
        _lib.hqo_alpha.argtypes = [C.c_int, C.c_double]
        _lib.hqo_second_moment.restype = C.c_double
        _lib.hqo_second_moment.argtypes = [C.c_int]
        _lib.hqo_f16_bits_to_f32.restype = C.c_float
        _lib.hqo_f16_bits_to_f32.argtypes = [C.c_uint16]
        _lib.hqo_f32_to_f16_bits.restype = C.c_uint16
        _lib.hqo_f32_to_f16_bits.argtypes = [C.c_float]
        for name in ("hqo_tile_bits", "hqo_write_tile", "hqo_read_tile", "hqo_rice_reference_bits",
                     "hqo_quantize_weights", "hqo_total_bits", "hqo_pack_weights",
                     "hqo_kv_quantize", "hqo_kv_pack_head", "hqo_kv_unpack_token"):
            getattr(_lib, name).restype = C.c_int64
    return _lib


def _p(a, t=None):
    return a.ctypes.data_as(C.c_void_p)


def _c(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _karr(k):
    k = list(k) if np.ndim(k) else [int(k), int(k)]
    return np.array([k[0], k[1] if len(k) > 1 else k[0]], dtype=np.int32)


# ---------------------------------------------------------------- RNG / signs
def philox(ctr, key):
    ctr = _c(ctr, np.uint32); key = _c(key, np.uint32); out = np.zeros(4, np.uint32)
    lib().hqo_philox4x32_10(_p(ctr), _p(key), _p(out))
    return out


def signs(seed, stream, n):
    out = np.zeros(n, np.int8)
    lib().hqo_signs(C.c_uint64(seed), C.c_uint32(stream), C.c_int64(n), _p(out))
    return out


# ---------------------------------------------------------------- RHT
def fwht(v):
    v = _c(v, np.float32).copy()
    lib().hqo_fwht_f32(_p(v), C.c_int(v.size))
    return v


def rht_f32(x, d):
    x = _c(x, np.float32); d = _c(d, np.int8); u = np.zeros_like(x)
    lib().hqo_rht_f32(_p(x), _p(d), C.c_int(x.size), _p(u))
    return u


def rht_dense_f64(x, d):
    x = _c(x, np.float64); d = _c(d, np.int8); u = np.zeros_like(x)
    lib().hqo_rht_dense_f64(_p(x), _p(d), C.c_int(x.size), _p(u))
    return u


def alpha(lattice, snr_db):
    return lib().hqo_alpha(lattice, float(snr_db))


def second_moment(lattice):
    return lib().hqo_second_moment(lattice)


def f16_bits_to_f32(h):
    return np.array([lib().hqo_f16_bits_to_f32(int(v)) for v in np.ravel(h)], np.float32).reshape(np.shape(h))


def f32_to_f16_bits(f):
    return np.array([lib().hqo_f32_to_f16_bits(float(v)) for v in np.ravel(f)], np.uint16).reshape(np.shape(f))


# ---------------------------------------------------------------- quantizer pieces
def nearest(lattice, y, clamp=True):
    y = _c(y, np.float32); c = np.zeros(lattice, np.int32)
    if clamp:
        lib().hqo_nearest(lattice, _p(y), _p(c))
    else:
        lib().hqo_nearest_noclamp(lattice, _p(y), _p(c))
    return c


def dither_block(lattice, seed, blk, token, head, role):
    U = np.zeros(lattice, np.float32)
    lib().hqo_dither_block(lattice, C.c_uint64(seed), C.c_uint32(blk), C.c_uint32(token),
                           C.c_uint32(head), C.c_uint32(role), _p(U))
    return U


def strip(lattice, c):
    c = _c(c, np.int32); z = np.zeros(lattice, np.int32)
    lib().hqo_strip(lattice, _p(c), _p(z))
    return z


def unstrip(lattice, z):
    z = _c(z, np.int32); c = np.zeros(lattice, np.int32)
    lib().hqo_unstrip(lattice, _p(z), _p(c))
    return c


# ---------------------------------------------------------------- tile streams
def tile_bits(lattice, codes, k):
    codes = _c(codes, np.int8); k = _karr(k)
    return lib().hqo_tile_bits(lattice, _p(codes), C.c_int(codes.size), _p(k))


def write_tile(lattice, codes, k, words, pos):
    codes = _c(codes, np.int8); k = _karr(k)
    return lib().hqo_write_tile(lattice, _p(codes), C.c_int(codes.size), _p(k), _p(words), C.c_uint64(pos))


def read_tile(lattice, n, k, words, pos):
    k = _karr(k); codes = np.zeros(n, np.int8)
    L = lib().hqo_read_tile(lattice, C.c_int(n), _p(k), _p(words), C.c_uint64(pos), _p(codes))
    return codes, L


def rice_reference_bits(lattice, codes, k):
    codes = _c(codes, np.int8); k = _karr(k)
    words = np.zeros(codes.size * 9 + 8, np.uint32)
    L = lib().hqo_rice_reference_bits(lattice, _p(codes), C.c_int(codes.size), _p(k), _p(words))
    return L, words


def symbol_histogram(lattice, codes, n):
    codes = _c(codes, np.int8)
    hist = np.zeros((lattice, 512), np.int64)
    lib().hqo_symbol_histogram(lattice, _p(codes), C.c_int64(codes.size // n), C.c_int(n), _p(hist))
    return hist


# ---------------------------------------------------------------- weights (O1, O2)
def quantize_weights(W, lattice, n_tile, snr_db, seed):
    W = _c(W, np.float32); m, n_in = W.shape
    codes = np.zeros((m, n_in), np.int8); norms = np.zeros((m, n_in // n_tile), np.uint16)
    clamps = lib().hqo_quantize_weights(_p(W), C.c_int64(m), C.c_int64(n_in), C.c_int64(n_in), lattice,
                                        C.c_int(n_tile), C.c_double(snr_db), C.c_uint64(seed),
                                        _p(codes), _p(norms))
    return codes, norms, clamps


def total_bits(codes, lattice, n_tile, k):
    codes = _c(codes, np.int8); k = _karr(k)
    return lib().hqo_total_bits(_p(codes), C.c_int64(codes.size // n_tile), lattice, C.c_int(n_tile), _p(k))


def choose_k(codes, lattice, n_tile):
    codes = _c(codes, np.int8); k = np.zeros(2, np.int32)
    lib().hqo_choose_k(_p(codes), C.c_int64(codes.size // n_tile), lattice, C.c_int(n_tile), _p(k))
    return k


def pack_weights(codes, norms, lattice, n_tile, k):
    codes = _c(codes, np.int8); norms = _c(norms, np.uint16); k = _karr(k)
    m, n_in = codes.shape
    G4 = 4 * ((m + 127) // 128) * (n_in // n_tile)          # sub-groups of 32 rows x one K-tile (FORMAT §5)
    goff = np.zeros(G4 + 1, np.uint32)
    args = (_p(codes), _p(norms), C.c_int64(m), C.c_int64(n_in), lattice, C.c_int(n_tile), _p(k))
    size = lib().hqo_pack_weights(*args, None, _p(goff))
    if size < 0:
        raise ValueError("a tile's U-section exceeds 8160 bits (FORMAT §5)")
    blob = np.zeros(size, np.uint8)
    lib().hqo_pack_weights(*args, _p(blob), _p(goff))
    return blob, goff


def unpack_weights(blob, goff, m, n_in, lattice, n_tile, k):
    blob = _c(blob, np.uint8); goff = _c(goff, np.uint32); k = _karr(k)
    codes = np.zeros((m, n_in), np.int8); norms = np.zeros((m, n_in // n_tile), np.uint16)
    lib().hqo_unpack_weights(_p(blob), _p(goff), C.c_int64(m), C.c_int64(n_in), lattice, C.c_int(n_tile),
                             _p(k), _p(codes), _p(norms))
    return codes, norms


def encode_weights(W, lattice, n_tile, snr_db, seed, k=(-1, -1)):
    """O1 end to end. Returns dict(codes, norms, k, blob, group_off, clamps, payload_bits)."""
    codes, norms, clamps = quantize_weights(W, lattice, n_tile, snr_db, seed)
    k = _karr(k)
    if k[0] < 0:
        k = choose_k(codes, lattice, n_tile)
    blob, goff = pack_weights(codes, norms, lattice, n_tile, k)
    return dict(codes=codes, norms=norms, k=k, blob=blob, group_off=goff, clamps=clamps,
                payload_bits=total_bits(codes, lattice, n_tile, k))


# ---------------------------------------------------------------- linear (O3)
def act_quant(x, lattice, n_tile, seed, want_u=False):
    x = _c(x, np.float32); B, n_in = x.shape
    q = np.zeros((B, n_in), np.int8); s_x = np.zeros((B, n_in // n_tile), np.float32)
    u = np.zeros((B, n_in), np.float32) if want_u else None
    lib().hqo_act_quant(_p(x), C.c_int64(B), C.c_int64(n_in), C.c_int64(n_in), lattice, C.c_int(n_tile),
                        C.c_uint64(seed), _p(q), _p(s_x), _p(u) if want_u else None)
    return (q, s_x, u) if want_u else (q, s_x)


def linear(codes, norms, lattice, n_tile, snr_db, q, s_x, want_acc=True):
    codes = _c(codes, np.int8); norms = _c(norms, np.uint16); q = _c(q, np.int8); s_x = _c(s_x, np.float32)
    m, n_in = codes.shape; B = q.shape[0]
    acc = np.zeros((n_in // n_tile, B, m), np.int32) if want_acc else None
    y = np.zeros((B, m), np.float64)
    lib().hqo_linear(_p(codes), _p(norms), C.c_int64(m), C.c_int64(n_in), lattice, C.c_int(n_tile),
                     C.c_double(snr_db), _p(q), _p(s_x), C.c_int64(B), _p(acc) if want_acc else None, _p(y))
    return acc, y


def linear_sampled(codes, norms, lattice, n_tile, snr_db, q, s_x, bs, rs):
    codes = _c(codes, np.int8); norms = _c(norms, np.uint16); q = _c(q, np.int8); s_x = _c(s_x, np.float32)
    bs = _c(bs, np.int64); rs = _c(rs, np.int64)
    m, n_in = codes.shape; B = q.shape[0]; ns = bs.size
    acc = np.zeros((ns, n_in // n_tile), np.int32); y = np.zeros(ns, np.float64)
    lib().hqo_linear_sampled(_p(codes), _p(norms), C.c_int64(m), C.c_int64(n_in), lattice, C.c_int(n_tile),
                             C.c_double(snr_db), _p(q), _p(s_x), C.c_int64(B), C.c_int64(ns), _p(bs), _p(rs),
                             _p(acc), _p(y))
    return acc, y


def dequant_weights(codes, norms, lattice, n_tile, snr_db, seed):
    codes = _c(codes, np.int8); norms = _c(norms, np.uint16); m, n_in = codes.shape
    What = np.zeros((m, n_in), np.float64)
    lib().hqo_dequant_weights(_p(codes), _p(norms), C.c_int64(m), C.c_int64(n_in), lattice, C.c_int(n_tile),
                              C.c_double(snr_db), C.c_uint64(seed), _p(What))
    return What


# ---------------------------------------------------------------- KV (O1 with rotate + dither, O4)
def kv_quantize(kv, token0, role, lattice, snr_db, rotation, dither, seed, qjl=None):
    """rotation 2 (qjl): `qjl` is the dense orthogonal matrix S [d, d] (row-major fp32), an input (§3.4)."""
    kv = _c(kv, np.float32); n_tok, heads, d = kv.shape
    codes = np.zeros((n_tok, heads, d), np.int8); norms = np.zeros((n_tok, heads), np.uint16)
    Q = _c(qjl, np.float32) if qjl is not None else None
    assert (rotation == 2) == (Q is not None) and (Q is None or Q.shape == (d, d))
    clamps = lib().hqo_kv_quantize_q(_p(kv), C.c_int64(n_tok), C.c_int(heads), C.c_int(d), C.c_int64(token0),
                                     C.c_int(role), lattice, C.c_double(snr_db), C.c_int(rotation),
                                     C.c_int(dither), C.c_uint64(seed), _p(Q) if Q is not None else None,
                                     _p(codes), _p(norms))
    return codes, norms, clamps


def rbits(lattice, n, k):
    k = _karr(k)
    return lib().hqo_rbits(lattice, C.c_int(n), _p(k))


def kv_pack_head(codes, head, lattice, k, rem, una, upos0, t0=0):
    """FORMAT §6: R-sections to rem at (t0+t)*Rbits, U-sections appended to una from bit upos0."""
    codes = _c(codes, np.int8); n_tok, heads, d = codes.shape; k = _karr(k)
    ulen = np.zeros(n_tok, np.uint16)
    pos = lib().hqo_kv_pack_head(_p(codes), C.c_int64(n_tok), C.c_int(heads), C.c_int(d), C.c_int(head),
                                 lattice, _p(k), C.c_int64(t0), _p(rem), _p(una), C.c_int64(upos0), _p(ulen))
    return pos, ulen


def kv_unpack_token(lattice, d, k, rem, t, una, upos):
    k = _karr(k); codes = np.zeros(d, np.int8)
    used = lib().hqo_kv_unpack_token(lattice, C.c_int(d), _p(k), _p(rem), C.c_int64(t), _p(una),
                                     C.c_int64(upos), _p(codes))
    return codes, used


def kv_reconstruct(codes, norms, token0, role, lattice, snr_db, rotation, dither, seed, qjl=None):
    codes = _c(codes, np.int8); norms = _c(norms, np.uint16); n_tok, heads, d = codes.shape
    out = np.zeros((n_tok, heads, d), np.float64)
    Q = _c(qjl, np.float32) if qjl is not None else None
    assert (rotation == 2) == (Q is not None)
    lib().hqo_kv_reconstruct_q(_p(codes), _p(norms), C.c_int64(n_tok), C.c_int(heads), C.c_int(d),
                               C.c_int64(token0), C.c_int(role), lattice, C.c_double(snr_db), C.c_int(rotation),
                               C.c_int(dither), C.c_uint64(seed), _p(Q) if Q is not None else None, _p(out))
    return out


def attend(Khat, Vhat, Kexact, Vexact, window, q):
    Khat = _c(Khat, np.float64); Vhat = _c(Vhat, np.float64)
    Kexact = _c(Kexact, np.float32); Vexact = _c(Vexact, np.float32); q = _c(q, np.float32)
    T, heads, d = Khat.shape; q_heads = q.shape[0]
    out = np.zeros((q_heads, d), np.float64)
    lib().hqo_attend(_p(Khat), _p(Vhat), _p(Kexact), _p(Vexact), C.c_int64(T), C.c_int(heads), C.c_int(d),
                     C.c_int(window), _p(q), C.c_int(q_heads), _p(out))
    return out


# ---------------------------------------------------------------- calibration (B.1 L857, §5.4)
def calib_point(tiles, lattice, snr_db):
    """Quantize iid-Gaussian tiles at one SNR: returns (bps at auto k, k, realized snr_db, codes)."""
    tiles = _c(tiles, np.float32); nt, n = tiles.shape
    codes = np.zeros((nt, n), np.int8); sp = C.c_double(0); ep = C.c_double(0)
    lib().hqo_calib_quantize(_p(tiles), C.c_int64(nt), C.c_int(n), lattice, C.c_double(snr_db), _p(codes),
                             C.byref(sp), C.byref(ep))
    k = choose_k(codes, lattice, n)
    bps = total_bits(codes, lattice, n, k) / codes.size
    return bps, k, 10.0 * np.log10(sp.value / ep.value), codes


def snr_for_bps(tiles, lattice, target_bps, lo=0.0, hi=45.0, iters=18):
    """Invert the monotone empirical rate curve b(SNR) by bisection on the same tiles (L863)."""
    for _ in range(iters):
        mid = 0.5 * (lo + hi)
        if calib_point(tiles, lattice, mid)[0] < target_bps:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


# ---- layer glue that folds into the activation cast (FORMAT R8-R10)
def bf16_round(x):
    x = _c(x, np.float32); out = np.empty_like(x)
    lib().hqo_bf16_round_array(_p(x), C.c_int64(x.size), _p(out))
    return out


def rmsnorm_bf16(h, g, eps):
    h = _c(h, np.float32); g = _c(g, np.float32); x = np.empty_like(h)
    lib().hqo_rmsnorm_bf16(_p(h), _p(g), C.c_int64(h.size), C.c_float(eps), _p(x))
    return x


def exp_c(t):
    f = lib().hqo_exp_c; f.restype = C.c_float; f.argtypes = [C.c_float]
    return np.array([f(float(v)) for v in np.asarray(t, np.float32).reshape(-1)], np.float32)


def silu_mul_bf16(a, b):
    a = _c(a, np.float32); b = _c(b, np.float32); x = np.empty_like(a)
    lib().hqo_silu_mul_bf16(_p(a), _p(b), C.c_int64(a.size), _p(x))
    return x


# ---- FP8-E4M3 MMA cast (§4.8, §6.3; FORMAT R12)
def e4m3_round(x):
    x = _c(x, np.float32); out = np.empty_like(x)
    lib().hqo_e4m3_round_array(_p(x), C.c_int64(x.size), _p(out))
    return out


def act_quant_fp8(x, n_tile, seed):
    x = _c(x, np.float32); B, n_in = x.shape
    q8 = np.zeros((B, n_in), np.float32); s_x = np.zeros((B, n_in // n_tile), np.float32)
    lib().hqo_act_quant_fp8(_p(x), C.c_int64(B), C.c_int64(n_in), C.c_int64(n_in), C.c_int(n_tile), C.c_uint64(seed),
                            _p(q8), _p(s_x))
    return q8, s_x


def linear_fp8(codes, norms, lattice, n_tile, snr_db, q8, s_x, want_acc=False):
    codes = _c(codes, np.int8); norms = _c(norms, np.uint16); q8 = _c(q8, np.float32); s_x = _c(s_x, np.float32)
    m, n_in = codes.shape; B = q8.shape[0]
    y = np.zeros((B, m), np.float64)
    acc = np.zeros((n_in // n_tile, B, m), np.float64) if want_acc else None
    acc_abs = np.zeros((n_in // n_tile, B, m), np.float64) if want_acc else None
    lib().hqo_linear_fp8(_p(codes), _p(norms), C.c_int64(m), C.c_int64(n_in), lattice, C.c_int(n_tile),
                         C.c_double(snr_db), _p(q8), _p(s_x), C.c_int64(B), _p(y),
                         _p(acc) if want_acc else None, _p(acc_abs) if want_acc else None)
    return (y, acc, acc_abs) if want_acc else y
