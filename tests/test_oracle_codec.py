"""Pins for the oracle's strip, Rice tile stream, container, calibration and linear/attend (no GPU)."""
import itertools
import json
import os

import numpy as np
import pytest

import hq_synth
from oracle import hqo

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))
NAME = {1: "Z", 2: "A2", 4: "D4", 8: "E8"}
S3 = np.sqrt(3.0)


def _members(lattice, cand):
    if lattice == hqo.Z:
        return np.ones(len(cand), bool)
    if lattice in (hqo.D4, hqo.A2):
        return cand.sum(1) % 2 == 0
    c0 = cand[:, :1] & 1
    return ((cand & 1) == c0).all(1) & (((cand - c0) // 2).sum(1) % 2 == 0)


# ------------------------------------------------------------------ strip (§4.6, Table 3)
@pytest.mark.parametrize("lattice,R", [(hqo.Z, 20), (hqo.A2, 12), (hqo.D4, 4), (hqo.E8, 2)])
def test_strip_is_a_bijection_lattice_to_Zn(lattice, R):
    dim = lattice
    box = np.array(list(itertools.product(range(-R, R + 1), repeat=dim)), np.int64)
    pts = box[_members(lattice, box)]
    syms = np.stack([hqo.strip(lattice, p) for p in pts])
    assert (syms >= 0).all()                                             # zig-zagged
    assert len(np.unique(syms, axis=0)) == len(pts)                      # injective
    back = np.stack([hqo.unstrip(lattice, z) for z in syms])
    assert (back == pts).all()                                           # lossless
    # surjective: every small non-negative symbol tuple un-strips to a lattice member and strips back
    tup = np.array(list(itertools.product(range(0, 3 if dim == 8 else 6), repeat=dim)), np.int32)
    pts2 = np.stack([hqo.unstrip(lattice, z) for z in tup]).astype(np.int64)
    assert _members(lattice, pts2).all()
    assert (np.stack([hqo.strip(lattice, p) for p in pts2]) == tup).all()


@pytest.mark.parametrize("lattice", [hqo.Z, hqo.A2, hqo.D4, hqo.E8])
def test_bits_stripped_per_scalar_table3(lattice):
    # raw code vector needs log2(box) bits/coordinate; lattice ∩ box has box/covolume-index points, so a
    # bijection onto Z^n saves log2(index)/n bits per scalar: 1.00 / 0.25 / 0.50 / 0  (Table 3)
    dim, R = lattice, {1: 64, 2: 32, 4: 8, 8: 2}[lattice]
    box = np.array(list(itertools.product(range(-R, R), repeat=dim)), np.int64)
    frac = _members(lattice, box).mean()
    assert abs(-np.log2(frac) / dim - GOLD["bits_stripped_per_scalar"][NAME[lattice]]) < 1e-9


def test_zigzag_values():
    # zigzag(n) = 2n (n>=0), -2n-1 (n<0)  (L270), via the Z lattice whose strip is the identity
    for v, z in [(0, 0), (1, 2), (-1, 1), (2, 4), (-2, 3), (127, 254), (-127, 253)]:
        assert hqo.strip(hqo.Z, [v])[0] == z and hqo.unstrip(hqo.Z, [z])[0] == v
    # E8 comb = 2*zigzag(t) + c (L274): the point (1,1,1,1,1,1,1,1+2*2) has c=1, s=(0,..,0,2), p=0, t=1
    assert list(hqo.strip(hqo.E8, [1, 1, 1, 1, 1, 1, 1, 5])) == [0] * 7 + [2 * 2 + 1]
    # D4: (1,0,0,3): p=1, t=1 ; A2: (n_y,n_x)=(3,1): p=1,t_y=1
    assert list(hqo.strip(hqo.D4, [1, 0, 0, 3])) == [2, 0, 0, 2]
    assert list(hqo.strip(hqo.A2, [3, 1])) == [2, 2]


# ------------------------------------------------------------------ Rice tile stream (§3.3, §4.7, FORMAT §4)
def _random_codes(lattice, n, rng, sigma):
    y = rng.standard_normal((n // lattice, lattice)) * sigma
    if lattice == hqo.A2:
        y[:, 0] *= S3
    return np.concatenate([hqo.nearest(lattice, b.astype(np.float32)) for b in y]).astype(np.int8)


@pytest.mark.parametrize("lattice", [hqo.Z, hqo.A2, hqo.D4, hqo.E8])
@pytest.mark.parametrize("n", [64, 128, 256])
def test_tile_stream_roundtrip_and_rice_length(lattice, n):
    rng = np.random.default_rng(100 * lattice + n)
    for sigma, k in [(1.6, (0, 0)), (3.5, (1, 0)), (7.3, (2, 1)), (7.3, (2, 3)), (14.6, (3, 2)), (30.0, (1, 5))]:
        codes = _random_codes(lattice, n, rng, sigma)
        L = hqo.tile_bits(lattice, codes, k)
        # textbook interleaved Rice code of the same symbols has the same length, and its first
        # codeword is literally q zeros, a one, then r in k bits
        Lref, wref = hqo.rice_reference_bits(lattice, codes, k)
        assert L == Lref
        z0 = hqo.strip(lattice, codes[:lattice].astype(np.int32))[0]
        q0, bits = z0 >> k[0], [(int(wref[p >> 5]) >> (31 - (p & 31))) & 1 for p in range((z0 >> k[0]) + 1 + k[0])]
        assert bits[:q0] == [0] * q0 and bits[q0] == 1
        assert sum(b << (k[0] - 1 - i) for i, b in enumerate(bits[q0 + 1:])) == z0 & ((1 << k[0]) - 1)
        for pos in (0, 5, 31, 37):                                      # bit-granular placement
            words = np.zeros((pos + L) // 32 + 2, np.uint32)
            assert hqo.write_tile(lattice, codes, k, words, pos) == L
            if pos:
                assert words[0] >> (32 - min(pos, 32)) == 0             # nothing written before pos
            back, used = hqo.read_tile(lattice, n, k, words, pos)
            assert used == L and (back == codes).all()
            total_ones = sum(bin(int(w)).count("1") for w in words)
            assert total_ones >= n                                      # n unary terminators at least


def test_adversarial_tiles_roundtrip():
    # G8: all energy in one coordinate, maximal codes, all-zero tile
    for lattice in (hqo.Z, hqo.A2, hqo.D4, hqo.E8):
        n = 128
        y = np.zeros(n, np.float32); y[5] = 166.0
        c1 = np.concatenate([hqo.nearest(lattice, y[i:i + lattice]) for i in range(0, n, lattice)]).astype(np.int8)
        c2 = np.concatenate([hqo.nearest(lattice, np.full(lattice, 500.0, np.float32) * (-1) ** i)
                             for i in range(n // lattice)]).astype(np.int8)
        for codes in (c1, c2, np.zeros(n, np.int8)):
            for k in ((0, 0), (2, 2)):
                L = hqo.tile_bits(lattice, codes, k)
                words = np.zeros(L // 32 + 2, np.uint32)
                hqo.write_tile(lattice, codes, k, words, 0)
                assert (hqo.read_tile(lattice, n, k, words, 0)[0] == codes).all()


@pytest.mark.parametrize("lattice,n_tile,m", [(hqo.E8, 64, 256), (hqo.D4, 128, 130), (hqo.A2, 64, 200), (hqo.Z, 256, 128)])
def test_weight_container_roundtrip(lattice, n_tile, m):
    W = hq_synth.gaussian_weight(m, 512, seed=lattice + m)
    enc = hqo.encode_weights(W, lattice, n_tile, 22.0, seed=9)
    codes, norms = hqo.unpack_weights(enc["blob"], enc["group_off"], m, 512, lattice, n_tile, enc["k"])
    assert (codes == enc["codes"]).all() and (norms == enc["norms"]).all()
    # layout facts of FORMAT §5, re-derived here from the codes alone: sub-groups of 32 rows x one K-tile,
    # header = ulen[32] | norm[32], R words interleaved over rows, U word-rows compacted in row order
    n_kt, n_rb = 512 // n_tile, (m + 127) // 128
    Rbits = hqo.rbits(lattice, n_tile, enc["k"])
    RW = (Rbits + 31) // 32
    goff = enc["group_off"].astype(np.int64)
    assert len(goff) == 4 * n_rb * n_kt + 1 and goff[-1] * 16 == enc["blob"].size
    lens_total = 0
    for sg in range(4 * n_rb * n_kt):
        g, w = sg // 4, sg % 4
        rb, kt = g // n_kt, g % n_kt
        base = 16 * goff[sg]
        hdr = enc["blob"][base: base + 128].view(np.uint16)
        rows = int(np.clip(m - (128 * rb + 32 * w), 0, 32))
        assert (hdr[rows:32] == 0).all() and (hdr[32 + rows:] == 0).all()
        nw = (hdr[:32].astype(np.int64) + 31) // 32
        size = 128 + 4 * (RW * 32 + int(nw.sum()))
        assert goff[sg + 1] - goff[sg] == (size + 15) // 16
        area = enc["blob"][base + 128: base + size].view(np.uint32)
        uarea = area[RW * 32:]
        for i in range(rows):
            r = 128 * rb + 32 * w + i
            tile = enc["codes"][r, kt * n_tile:(kt + 1) * n_tile]
            assert hdr[i] + Rbits == hqo.tile_bits(lattice, tile, enc["k"])
            # the row's logical stream, written on its own, is what the container interleaves
            words = np.zeros(RW + int(nw[i]) + 2, np.uint32)
            hqo.write_tile(lattice, tile, enc["k"], words, 0)
            if Rbits % 32 == 0:
                assert (area[np.arange(RW) * 32 + i] == words[:RW]).all()
                for t in range(int(nw[i])):
                    at = int(np.minimum(nw, t).sum()) + int((nw[:i] > t).sum())   # earlier word-rows + earlier rows
                    assert uarea[at] == words[RW + t]
        lens_total += int(hdr[:32].sum()) + rows * Rbits
    assert lens_total == enc["payload_bits"]


def test_e8_stream_order_groups_coordinates_of_four_blocks():
    # FORMAT §3: stream position p = 32c + 8w + 2b + e holds coordinate 2w+e of block 4c+b.  A tile whose only
    # non-zero code sits in (block, coordinate) must put its only non-zero symbol at that stream position:
    # with k = 0 the U-section is "1" per zero symbol and q zeros + "1" for the non-zero one.
    n = 64
    for blk in range(8):
        for coord in range(7):                       # coordinates 0..6 carry zigzag(s_i) themselves (L261-270)
            codes = np.zeros(n, np.int8)
            codes[8 * blk + coord] = 2                # even coset, s = 1 -> zigzag 2; parity of the block flips s_7:
            codes[8 * blk + 7] = 2                    # keep the point in 2E8: s_7 = 1 = 2*0 + parity(1)
            words = np.zeros(8, np.uint32)
            hqo.write_tile(hqo.E8, codes, (0, 0), words, 0)
            bits = "".join(format(int(x), "032b") for x in words)
            c, b = blk // 4, blk % 4
            p = 32 * c + 8 * (coord // 2) + 2 * b + (coord % 2)
            assert bits[:p] == "1" * p and bits[p:p + 3] == "001"
            assert (hqo.read_tile(hqo.E8, n, (0, 0), words, 0)[0] == codes).all()


def test_field_plane_layout_is_swar_extractable():
    # FORMAT §4: in a full chunk of 32 symbols (four blocks of 8), group g = 2*block + parity holds the
    # w-bit fields of the block's even (parity 0) or odd (parity 1) symbols, one symbol per byte:
    # (V[g // (8/w)] >> (w * (g % (8/w)))) & (mask_w * 0x01010101).
    rng = np.random.default_rng(5)
    for k in range(1, 8):
        zz = rng.integers(0, 1 << k, size=64)          # Z lattice: symbol = zigzag(code), q = 0
        codes = np.where(zz & 1, -((zz + 1) >> 1), zz >> 1).astype(np.int8)
        words = np.zeros(64, np.uint32)
        L = hqo.write_tile(hqo.Z, codes, (k, k), words, 0)
        assert L == 64 * (k + 1) and hqo.rbits(hqo.Z, 64, (k, k)) == 64 * k
        wi = 0
        for ch in range(2):
            lo = 0
            for wd in (1, 2, 4):
                if not k & wd:
                    continue
                per = 8 // wd
                for g in range(8):
                    V = int(words[wi + g // per])
                    f4 = (V >> (wd * (g % per))) & (((1 << wd) - 1) * 0x01010101)
                    for u in range(4):
                        sym = 32 * ch + 8 * (g // 2) + 2 * u + (g % 2)
                        assert (f4 >> (8 * u)) & 0xFF == (int(zz[sym]) >> lo) & ((1 << wd) - 1)
                wi += wd
                lo += wd
        # U-section: q = 0 everywhere -> 64 one bits right after the R-section
        assert words[wi] == 0xFFFFFFFF and words[wi + 1] == 0xFFFFFFFF and words[wi + 2] == 0


def test_auto_k_is_argmin():
    codes = hqo.quantize_weights(hq_synth.gaussian_weight(64, 512, 3), hqo.E8, 128, 22.7, 1)[0]
    k = hqo.choose_k(codes, hqo.E8, 128)
    tots = [hqo.total_bits(codes, hqo.E8, 128, (kk, kk)) for kk in range(8)]
    assert k[0] == int(np.argmin(tots)) == 2
    codes = hqo.quantize_weights(hq_synth.gaussian_weight(64, 512, 3), hqo.D4, 128, 22.7, 1)[0]
    k = hqo.choose_k(codes, hqo.D4, 128)
    tots = [hqo.total_bits(codes, hqo.D4, 128, (kk, max(kk - 1, 0))) for kk in range(8)]
    assert k[0] == int(np.argmin(tots)) and k[1] == max(k[0] - 1, 0)   # the halving identity (L272, L865)


# ------------------------------------------------------------------ calibration pins (B.1, B.2, Tables 11, 14)
@pytest.fixture(scope="module")
def tiles():
    return hq_synth.calib_tiles(20000, 128, seed=42)


@pytest.mark.parametrize("lattice", [hqo.E8, hqo.D4, hqo.A2, hqo.Z])
def test_rice_rate_at_21dB(tiles, lattice):
    bps, k, snr, codes = hqo.calib_point(tiles, lattice, 21.0)
    assert abs(bps - GOLD["rice_rate_at_21dB"][NAME[lattice]]) < 0.025      # L289
    assert abs(snr - 21.0) < 0.1                                            # realized SNR (L874)
    R_ideal = 0.5 * np.log2(10 ** 2.1) + 0.5 * np.log2(2 * np.pi * np.e * GOLD["table2_G"][NAME[lattice]])
    assert 0.03 < bps - R_ideal < 0.15                                      # "~0.1 bps above the ideal" (L861)
    # B.4: marginal entropy of the stripped symbols = lattice ideal within ~0.02 bps (L908, L927)
    hist = hqo.symbol_histogram(lattice, codes, 128).astype(np.float64)
    p = hist / hist.sum(1, keepdims=True)
    H = -(np.where(p > 0, p * np.log2(np.where(p > 0, p, 1)), 0)).sum(1).mean()
    assert abs(H - R_ideal) < 0.03


def test_alpha_at_5bps_table14(tiles):
    for lattice in (hqo.E8, hqo.A2, hqo.Z):
        snr = hqo.snr_for_bps(tiles, lattice, 5.0, lo=20, hi=40, iters=12)
        assert abs(hqo.alpha(lattice, snr) - GOLD["alpha_at_5bps"][NAME[lattice]]) < 0.15
    snr = hqo.snr_for_bps(tiles, hqo.D4, 5.0, lo=20, hi=40, iters=12)
    assert abs(hqo.alpha(hqo.D4, snr) - 8.6) < 0.15       # G7: eq.(9) with D4 ⊂ Z^4; the printed 17.3 is 2·D4


def test_a2_snr_table11_and_e8_z_gap(tiles):
    for bps, snr_paper in GOLD["a2_snr_db"].items():
        if bps == "cite":
            continue
        snr = hqo.snr_for_bps(tiles, hqo.A2, float(bps), lo=5, hi=40, iters=12)
        assert abs(snr - snr_paper) < 0.12
        b, k, real, _ = hqo.calib_point(tiles, hqo.A2, snr)
        assert abs(b - float(bps)) < 0.01 and abs(real - snr) < 0.1        # rate within ~0.01 bps (L295)
    for bps, gap in [(3.0, 0.81), (5.0, 0.65)]:
        g = hqo.snr_for_bps(tiles, hqo.E8, bps, 5, 40, 12) - hqo.snr_for_bps(tiles, hqo.Z, bps, 5, 40, 12)
        assert abs(g - gap) < 0.06                                          # L383


def test_e8_operating_points_and_code_range(tiles):
    # E8: k = 0,1,2,3 at 2,3,4,5 bps; largest coordinate ≈ 3.4σ, |Y| ≈ 50 over 20-30 dB (L894)
    for bps, k_expect in [(2.0, 0), (3.0, 1), (4.0, 2), (5.0, 3)]:
        snr = hqo.snr_for_bps(tiles, hqo.E8, bps, 0, 40, 12)
        b, k, real, codes = hqo.calib_point(tiles, hqo.E8, snr)
        assert k[0] == k_expect
    b, k, real, codes = hqo.calib_point(tiles, hqo.E8, 30.0)
    amax = np.abs(codes.astype(np.int32)).max()
    assert 45 <= amax <= 90 and amax / hqo.alpha(hqo.E8, 30.0) < 5.5


# ------------------------------------------------------------------ linear (O3)
def test_linear_matches_numpy_and_dequantized_weights():
    W, x = hq_synth.c1_weight()
    snr = 22.68
    enc = hqo.encode_weights(W, hqo.E8, 64, snr, seed=5)
    q, s_x, u = hqo.act_quant(x, hqo.E8, 64, seed=5, want_u=True)
    acc, y = hqo.linear(enc["codes"], enc["norms"], hqo.E8, 64, snr, q, s_x)
    # the INT8 contraction, re-done with a library matmul per tile
    c = enc["codes"].astype(np.int64).reshape(256, 4, 64); qq = q.astype(np.int64).reshape(1, 4, 64)
    assert (acc == np.einsum("rki,bki->kbr", c, qq)).all()
    # activations: u is the RHT of x (1e-5), q = rint(u*127/amax)
    d = hqo.signs(5, 1, 256)
    for kt in range(4):
        ref = hqo.rht_dense_f64(x[0, kt * 64:(kt + 1) * 64].astype(np.float64), d[kt * 64:(kt + 1) * 64])
        assert np.max(np.abs(u[0, kt * 64:(kt + 1) * 64] - ref)) < 1e-5 * np.abs(ref).max()
        amax = np.abs(ref).max()
        assert abs(s_x[0, kt] - amax / 127) < 1e-6 * amax
        assert np.abs(q[0, kt * 64:(kt + 1) * 64] - ref * 127 / amax).max() <= 0.5 + 1e-3
    # y ≈ Ŵ x with Ŵ reconstructed the long way (inverse RHT of the scaled codes): only the
    # activation cast separates them (G5: ~0.4 % of |y|)
    What = hqo.dequant_weights(enc["codes"], enc["norms"], hqo.E8, 64, snr, seed=5)
    y_exact = x.astype(np.float64) @ What.T
    assert np.linalg.norm(y - y_exact) / np.linalg.norm(y_exact) < 0.01
    # and Ŵ ≈ W at the calibrated SNR (L874: within ≈0.1 dB; small matrix -> 0.3)
    snr_real = 10 * np.log10((W.astype(np.float64) ** 2).sum() / ((What - W) ** 2).sum())
    assert abs(snr_real - snr) < 0.3
    # sampled variant agrees with the full one
    bs, rs = np.zeros(5, np.int64), np.array([0, 17, 100, 200, 255])
    acc_s, y_s = hqo.linear_sampled(enc["codes"], enc["norms"], hqo.E8, 64, snr, q, s_x, bs, rs)
    assert (acc_s == acc[:, 0, rs].T).all() and np.allclose(y_s, y[0, rs], rtol=1e-12)


def test_a2_linear_uses_sqrt3_on_even_coordinates():
    W = hq_synth.gaussian_weight(128, 128, 4); x = hq_synth.activations(2, 128, 5)
    enc = hqo.encode_weights(W, hqo.A2, 128, 25.0, seed=2)
    q, s_x = hqo.act_quant(x, hqo.A2, 128, seed=2)
    _, y = hqo.linear(enc["codes"], enc["norms"], hqo.A2, 128, 25.0, q, s_x)
    What = hqo.dequant_weights(enc["codes"], enc["norms"], hqo.A2, 128, 25.0, seed=2)
    y_exact = x.astype(np.float64) @ What.T
    assert np.linalg.norm(y - y_exact) / np.linalg.norm(y_exact) < 0.01
    assert abs(10 * np.log10((W.astype(np.float64) ** 2).sum() / ((What - W) ** 2).sum()) - 25.0) < 0.4


# ------------------------------------------------------------------ KV: unbiasedness (Cor. 2-3, Prop. 1-2) and attend
def test_subtractive_dither_is_unbiased_per_vector():
    heads, d, snr = 1, 128, 9.68                       # E8 at ~2 bps
    x = hq_synth.kv_tokens(1, heads, d, seed=4)
    qv = np.random.default_rng(3).standard_normal(d)
    N = 100000                                         # north_star: 1e5 dithers per rotation
    for rotation in (0, 1):
        # the same vector presented as tokens 0..N-1: a fresh dither per token (L190)
        X = np.repeat(x, N, axis=0)
        codes, norms, _ = hqo.kv_quantize(X, 0, 0, hqo.E8, snr, rotation, 1, seed=77)
        xh = hqo.kv_reconstruct(codes, norms, 0, 0, hqo.E8, snr, rotation, 1, seed=77)[:, 0]
        err = xh @ qv - x[0, 0].astype(np.float64) @ qv
        rho = float(hqo.f16_bits_to_f32(norms[0, 0]))
        sigma = np.sqrt(hqo.second_moment(hqo.E8) * (qv @ qv)) * rho / (hqo.alpha(hqo.E8, snr) * np.sqrt(d))
        assert abs(err.mean()) < 3 * sigma / np.sqrt(N) + 1e-3 * sigma      # mean within 3σ (eq.(4), Cor.2)
        assert abs(err.std() / sigma - 1) < 0.05                            # Var = σ²_V ||q||² (Cor.3 L806)
        # negative control (Prop. 2): without dither the error is one fixed non-zero vector
        c0, n0, _ = hqo.kv_quantize(X[:4], 0, 0, hqo.E8, snr, rotation, 0, seed=77)
        x0 = hqo.kv_reconstruct(c0, n0, 0, 0, hqo.E8, snr, rotation, 0, seed=77)[:, 0]
        assert (x0 == x0[0]).all() and np.abs(x0[0] - x[0, 0]).max() > 1e-3


def test_attend_window_covers_everything_equals_exact_attention():
    T, heads, d, qh = 40, 2, 128, 8
    K = hq_synth.kv_tokens(T, heads, d, seed=4); V = hq_synth.kv_tokens(T, heads, d, seed=5)
    q = hq_synth.activations(qh, d, seed=6)
    junk = np.full((T, heads, d), 1e9)
    out = hqo.attend(junk, junk, K, V, window=T, q=q)                      # G15
    for i in range(qh):
        h = i // (qh // heads)
        s = (K[:, h].astype(np.float64) @ q[i].astype(np.float64)) / np.sqrt(d)
        p = np.exp(s - s.max()); p /= p.sum()
        assert np.allclose(out[i], p @ V[:, h].astype(np.float64), rtol=1e-12, atol=1e-12)
    # with quantized history: high SNR reconstruction converges to the exact answer
    ck, nk, _ = hqo.kv_quantize(K, 0, 0, hqo.E8, 34.0, 1, 1, seed=1)
    cv, nv, _ = hqo.kv_quantize(V, 0, 1, hqo.E8, 34.0, 1, 1, seed=1)
    Kh = hqo.kv_reconstruct(ck, nk, 0, 0, hqo.E8, 34.0, 1, 1, seed=1)
    Vh = hqo.kv_reconstruct(cv, nv, 0, 1, hqo.E8, 34.0, 1, 1, seed=1)
    assert abs(10 * np.log10((K.astype(np.float64) ** 2).sum() / ((Kh - K) ** 2).sum()) - 34.0) < 0.5
    out8 = hqo.attend(Kh, Vh, K, V, window=8, q=q)
    assert np.abs(out8 - out).max() < 0.05 * np.abs(out).max()


def test_kv_stream_pack_and_lengths():
    T, heads, d = 20, 2, 128
    K = hq_synth.kv_tokens(T, heads, d, seed=4)
    for snr, k in ((9.68, (0, 0)), (22.68, (2, 2))):
        codes, norms, _ = hqo.kv_quantize(K, 0, 0, hqo.E8, snr, 1, 1, seed=1)
        Rbits = hqo.rbits(hqo.E8, d, k)
        rem = np.zeros(T * Rbits // 32 + 4, np.uint32); una = np.zeros(4096, np.uint32)
        # appended in two calls: the second continues where the first stopped (FORMAT §6)
        pos1, l1 = hqo.kv_pack_head(codes[:7], 1, hqo.E8, k, rem, una, 0, t0=0)
        pos, l2 = hqo.kv_pack_head(codes[7:], 1, hqo.E8, k, rem, una, pos1, t0=7)
        ulen = np.concatenate([l1, l2])
        assert pos == ulen.astype(np.int64).sum()
        p = 0
        for t in range(T):
            back, used = hqo.kv_unpack_token(hqo.E8, d, k, rem, t, una, p)
            assert used == ulen[t] and (back == codes[t, 1]).all()
            assert used + Rbits == hqo.tile_bits(hqo.E8, codes[t, 1], k)
            p += used
        if k[0] == 0:
            # ~2 bps + fp16 norm: effective 2.25-2.4 bits/scalar incl. u16 length -> KV× ≈ 6.4-6.6 (L587-590)
            eff = (ulen.mean() + Rbits + 32) / d
            assert 2.0 < eff < 2.6
