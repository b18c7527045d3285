"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

Holds none of the method's arithmetic: only random draws, dtype rounding and shapes (DESIGN.md §4
states the recipe and what each input stands in for).  numpy only.
"""
import numpy as np


def to_bf16_f32(a: np.ndarray) -> np.ndarray:
    """Round fp32 values to the nearest bf16 (RNE) and return them widened back to fp32."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    u = a.view(np.uint32).astype(np.uint64)
    r = ((u + 0x7FFF + ((u >> 16) & 1)) >> 16) << 16
    return r.astype(np.uint32).view(np.float32).reshape(a.shape)


def bf16_bits(a: np.ndarray) -> np.ndarray:
    """uint16 bit patterns of bf16-representable fp32 values."""
    return (np.ascontiguousarray(a, dtype=np.float32).view(np.uint32) >> 16).astype(np.uint16)


def c1_weight():
    """Config 1: W 256x256 fp32 ~ N(0, 0.02^2), seed 0; x fp32 ~ N(0,1), length 256, seed 1."""
    W = (np.random.default_rng(0).standard_normal((256, 256)) * 0.02).astype(np.float32)
    x = np.random.default_rng(1).standard_normal((1, 256)).astype(np.float32)
    return W, x


LLAMA_SHAPES = {  # name -> (m_out, n_in); Llama-3.1-8B decoder-layer linears (config 2)
    "q": (4096, 4096), "k": (1024, 4096), "v": (1024, 4096), "o": (4096, 4096),
    "gate": (14336, 4096), "up": (14336, 4096), "down": (4096, 14336),
}


def gaussian_weight(m, n_in, seed, outliers=False, std=0.02):
    """bf16-valued N(0, std^2) weight; optionally round(0.001*n_in) seeded input columns x20."""
    rng = np.random.default_rng(seed)
    W = rng.standard_normal((m, n_in), dtype=np.float32) * np.float32(std)
    if outliers:
        cols = rng.choice(n_in, size=max(1, round(0.001 * n_in)), replace=False)
        W[:, cols] *= np.float32(20.0)
    return to_bf16_f32(W)


def llama_weight(layer, name, scale_rows=1.0):
    idx = list(LLAMA_SHAPES).index(name)
    m, n_in = LLAMA_SHAPES[name]
    m = int(m * scale_rows)
    return gaussian_weight(m, n_in, seed=layer * 16 + idx, outliers=True)


def activations(batch, n_in, seed, bf16=True):
    x = np.random.default_rng(seed).standard_normal((batch, n_in), dtype=np.float32)
    return to_bf16_f32(x) if bf16 else x


def kv_tokens(n_tok, heads, d, seed, token0=0):
    """K or V rows [n_tok, heads, d]: N(0,1) x per-channel LogNormal(0,1) scale (fixed per seed), bf16."""
    scale = np.exp(np.random.default_rng(seed).standard_normal((heads, d))).astype(np.float32)
    rng = np.random.default_rng([seed, 1, token0])
    x = rng.standard_normal((n_tok, heads, d), dtype=np.float32) * scale[None]
    return to_bf16_f32(x)


def haar_matrix(d, seed):
    """A Haar-uniform orthogonal matrix S [d, d] (the qjl rotation, §3.4: drawn once per layer): QR of a
    Gaussian matrix with the sign convention that makes the distribution uniform; fp32."""
    g = np.random.default_rng([seed, 7]).standard_normal((d, d))
    q, r = np.linalg.qr(g)
    return np.ascontiguousarray((q * np.sign(np.diag(r))[None, :]).astype(np.float32))


def calib_tiles(nt, n, seed=42):
    """iid N(0,1) calibration tiles (B.1: ~1e5 tiles, seed 42)."""
    return np.random.default_rng(seed).standard_normal((nt, n), dtype=np.float32)
