"""Pins of the oracle's qjl rotation (FORMAT R11; §3.4 eq.(2) x_rot = S^T Q_Lambda(S x), Table 4).

The rotation is a dense matrix product, so the plausible mistakes are a transposed operand, a wrong place in the
pipeline and a missing inverse: each pin below fails for one of them."""
import numpy as np

import hq_synth
from oracle import hqo

SNR = float(np.float32(22.68))
SEED = 5


def _snr_db(x, xh):
    return 10 * np.log10(np.sum(x.astype(np.float64) ** 2) / np.sum((xh - x) ** 2))


def test_haar_matrix_is_orthogonal_and_not_symmetric():
    Q = hq_synth.haar_matrix(128, 3).astype(np.float64)
    assert np.abs(Q @ Q.T - np.eye(128)).max() < 1e-5
    assert np.abs(Q - Q.T).max() > 0.1


def test_identity_and_sign_matrices_reduce_to_the_other_rotations_bit_for_bit():
    X = hq_synth.kv_tokens(40, 2, 128, seed=4)
    c0, n0, _ = hqo.kv_quantize(X, 0, 0, hqo.E8, SNR, 0, 1, SEED)
    cI, nI, _ = hqo.kv_quantize(X, 0, 0, hqo.E8, SNR, 2, 1, SEED, qjl=np.eye(128, dtype=np.float32))
    assert (c0 == cI).all() and (n0 == nI).all()                       # fma(1, u, 0) = u and fma(0, u, acc) = acc: exact
    s = np.zeros(128, np.int8)
    hqo.lib().hqo_signs(hqo.C.c_uint64(SEED), hqo.C.c_uint32(2), hqo.C.c_int64(128), s.ctypes.data_as(hqo.C.c_void_p))
    c1, n1, _ = hqo.kv_quantize(X, 0, 0, hqo.E8, SNR, 1, 1, SEED)
    cS, nS, _ = hqo.kv_quantize(X, 0, 0, hqo.E8, SNR, 2, 1, SEED, qjl=np.diag(s.astype(np.float32)))
    assert (c1 == cS).all() and (n1 == nS).all()


def test_index_convention_u_prime_i_equals_sum_j_Q_ij_u_j():
    """A cyclic-shift permutation matrix (not symmetric) on a vector whose RHT is exactly c * e_j0: the single non-zero
    code must land at i = j0 + 1 (where Q[i, j0] = 1), not at j0 - 1 (what Q^T would give)."""
    d, j0, c = 64, 10, 4.0
    D = np.zeros(d, np.int8)
    hqo.lib().hqo_signs(hqo.C.c_uint64(SEED), hqo.C.c_uint32(1), hqo.C.c_int64(d), D.ctypes.data_as(hqo.C.c_void_p))
    H = np.array([[(-1) ** bin(i & j).count("1") for j in range(d)] for i in range(d)], np.float64)
    x = (c * D * H[:, j0] / 8.0).astype(np.float32)                    # RHT(x) = H D x / 8 = c e_j0, every step exact
    _, _, u = hqo.act_quant(x[None], hqo.Z, d, SEED, want_u=True)
    assert u[0, j0] == c and np.count_nonzero(u) == 1
    P = np.zeros((d, d), np.float32)
    for j in range(d):
        P[(j + 1) % d, j] = 1.0
    codes, norms, _ = hqo.kv_quantize(x.reshape(1, 1, d), 0, 0, hqo.Z, SNR, 2, 0, SEED, qjl=P)
    nz = np.flatnonzero(codes[0, 0])
    assert list(nz) == [j0 + 1] and codes[0, 0, j0 + 1] > 0


def test_reconstruction_inverts_the_rotation():
    """S^T after the quantizer (eq.(2)): with a Haar (non-symmetric) S the long-way reconstruction reaches the target
    SNR; a missing or transposed inverse would sit near 0 dB."""
    Q = hq_synth.haar_matrix(128, 9)
    X = hq_synth.kv_tokens(64, 2, 128, seed=6)
    for dither in (0, 1):
        c, n, _ = hqo.kv_quantize(X, 0, 1, hqo.E8, SNR, 2, dither, SEED, qjl=Q)
        Xh = hqo.kv_reconstruct(c, n, 0, 1, hqo.E8, SNR, 2, dither, SEED, qjl=Q)
        assert abs(_snr_db(X, Xh) - SNR) < 0.5
        bad = hqo.kv_reconstruct(c, n, 0, 1, hqo.E8, SNR, 2, dither, SEED, qjl=np.ascontiguousarray(Q.T))
        assert _snr_db(X, bad) < 3.0                                   # negative control


def test_rotation_spreads_channel_anisotropy():
    """What the rotation is for (§6.2): after S the per-coordinate energy of anisotropic K rows is flat, so fewer inputs hit
    the INT8 pre-clamp than without rotation at a high rate."""
    X = hq_synth.kv_tokens(256, 2, 128, seed=8)
    Q = hq_synth.haar_matrix(128, 10)
    snr_hi = float(np.float32(34.0))
    _, _, cl_none = hqo.kv_quantize(X, 0, 0, hqo.E8, snr_hi, 0, 0, SEED)
    _, _, cl_qjl = hqo.kv_quantize(X, 0, 0, hqo.E8, snr_hi, 2, 0, SEED, qjl=Q)
    assert cl_qjl <= cl_none
