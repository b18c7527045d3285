"""Pins for the oracle's RNG, RHT, fp16, nearest-point decoders and dither (no GPU).

Each check ties oracle/hq_oracle.c to something other than itself: published known-answer vectors,
the dense definition, brute force over the lattice's membership definition, and the closed-form
constants the paper prints (tests/golden/paper_values.json).
"""
import itertools
import json
import os

import numpy as np
import pytest

from oracle import hqo

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))
S3 = np.sqrt(3.0)


def test_philox_known_answers():
    for v in GOLD["philox4x32_10_kat"]["vectors"]:
        out = hqo.philox([int(x, 16) for x in v["ctr"]], [int(x, 16) for x in v["key"]])
        assert [f"{int(x):08x}" for x in out] == v["out"]


def test_signs_balanced_and_seeded():
    a = hqo.signs(7, 1, 4096)
    assert set(np.unique(a)) == {-1, 1}
    assert abs(int(a.sum())) < 4 * 64          # 4 sigma
    assert (hqo.signs(7, 1, 4096) == a).all()
    assert (hqo.signs(8, 1, 4096) != a).any() and (hqo.signs(7, 2, 4096) != a).any()
    # prefix property: a layer's sign vector does not depend on its length
    assert (hqo.signs(7, 1, 300) == a[:300]).all()


@pytest.mark.parametrize("n", [64, 128, 256])
def test_hadamard_is_sylvester_and_HHt_is_nI(n):
    # G1: the butterfly applied to unit vectors gives the integer ±1 Sylvester matrix, H Hᵀ = n I exactly
    H = np.stack([hqo.fwht(np.eye(n, dtype=np.float32)[i]) for i in range(n)]).astype(np.int64)
    assert set(np.unique(H)) == {-1, 1}
    i, j = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    par = np.array([[bin(a & b).count("1") & 1 for b in range(n)] for a in range(n)])
    assert (H == 1 - 2 * par).all()
    assert (H @ H.T == n * np.eye(n, dtype=np.int64)).all()


@pytest.mark.parametrize("n", [64, 128, 256])
def test_rht_matches_dense_definition_and_is_orthonormal(n):
    rng = np.random.default_rng(n)
    d = hqo.signs(3, 1, n)
    x = rng.standard_normal(n).astype(np.float32) * 3
    w = rng.standard_normal(n).astype(np.float32)
    u32 = hqo.rht_f32(x, d)
    u64 = hqo.rht_dense_f64(x.astype(np.float64), d)
    # the fp32 butterfly vs the dense double definition: the 1e-5 criterion of north_star
    assert np.max(np.abs(u32 - u64)) <= 1e-5 * np.max(np.abs(u64))
    # independent numpy restatement of eq.(1): H D x / sqrt n
    H = np.array([[1 - 2 * (bin(a & b).count("1") & 1) for b in range(n)] for a in range(n)], np.float64)
    assert np.allclose(u64, H @ (d * x.astype(np.float64)) / np.sqrt(n), rtol=0, atol=1e-12)
    # orthonormal: norms and inner products preserved (W = (W Hᵀ) H, L212)
    w64 = hqo.rht_dense_f64(w.astype(np.float64), d)
    assert abs(u64 @ w64 - x.astype(np.float64) @ w.astype(np.float64)) < 1e-10
    # inverse = D H / sqrt n  (round trip)
    back = d * (H @ u64) / np.sqrt(n)
    assert np.max(np.abs(back - x)) < 1e-12 * 10


def test_fp16_rounding_matches_ieee():
    rng = np.random.default_rng(0)
    vals = np.concatenate([rng.standard_normal(2000) * 10 ** rng.uniform(-9, 5, 2000),
                           [0.0, 65504.0, 65519.0, 65520.0, 1e9, 2.0 ** -24, 2.0 ** -25, 3 * 2.0 ** -25,
                            6.1e-5, 6.103515625e-05, 1.0, 1.00048828125, 1.000732421875]]).astype(np.float32)
    vals = np.abs(vals)
    got = hqo.f32_to_f16_bits(vals)
    ref = vals.astype(np.float16)
    ref_bits = ref.view(np.uint16).copy()
    ref_bits[np.isinf(ref)] = 0x7BFF                      # FORMAT R3: saturating
    assert (got == ref_bits).all()
    assert (hqo.f16_bits_to_f32(got) == np.where(np.isinf(ref), 65504.0, ref.astype(np.float32))).all()


# ------------------------------------------------------------------ nearest point: brute force
def _members(lattice, cand):
    """Membership by the DEFINITIONS of §4.5-4.6 (L241, L253-255), not by the decoder."""
    if lattice == hqo.Z:
        return np.ones(len(cand), bool)
    if lattice == hqo.D4 or lattice == hqo.A2:
        return cand.sum(1) % 2 == 0
    c0 = cand[:, :1] & 1
    same = ((cand & 1) == c0).all(1)
    half = (cand - c0) // 2
    return same & (half.sum(1) % 2 == 0)


def _brute(lattice, y):
    dim = lattice
    scale = np.array([S3, 1.0]) if lattice == hqo.A2 else np.ones(dim)
    base = np.rint(np.asarray(y, np.float64) / scale).astype(np.int64)
    offs = np.array(list(itertools.product(range(-3, 4), repeat=dim)) if dim <= 4
                    else list(itertools.product(range(-2, 3), repeat=dim)), np.int64)
    cand = base + offs
    cand = cand[_members(lattice, cand)]
    d2 = ((np.asarray(y, np.float64) - cand * scale) ** 2).sum(1)
    return cand, d2


@pytest.mark.parametrize("lattice,count", [(hqo.Z, 300), (hqo.A2, 300), (hqo.D4, 300), (hqo.E8, 60)])
def test_nearest_point_vs_brute_force(lattice, count):
    rng = np.random.default_rng(lattice)
    dim = lattice
    ys = [rng.standard_normal(dim) * s for s in (0.3, 2.0, 9.0) for _ in range(count // 3)]
    # adversarial: zeros, half-integers, exact ties between cosets, deep holes
    ys += [np.zeros(dim), np.full(dim, 0.5), np.full(dim, 1.0), np.full(dim, -0.5), np.full(dim, 1.5),
           np.r_[1.0, np.zeros(dim - 1)], np.r_[0.5, np.zeros(dim - 1)], np.r_[-2.5, np.full(dim - 1, 0.5)]]
    for y in ys:
        y = np.asarray(y, np.float32)
        c = hqo.nearest(lattice, y, clamp=False).astype(np.int64)
        assert _members(lattice, c[None])[0], (y, c)
        cand, d2 = _brute(lattice, y)
        scale = np.array([S3, 1.0]) if lattice == hqo.A2 else np.ones(dim)
        mine = ((y.astype(np.float64) - c * scale) ** 2).sum()
        assert mine <= d2.min() * (1 + 1e-6) + 1e-9, (y, c, cand[d2.argmin()])
        if np.sort(d2)[1] - d2.min() > 1e-4:          # away from ties the answer is unique
            assert (c == cand[d2.argmin()]).all()


@pytest.mark.parametrize("lattice", [hqo.Z, hqo.A2, hqo.D4, hqo.E8])
def test_voronoi_second_moment_matches_table2(lattice):
    # (1/n) E||y - Q(y)||^2 for y uniform over many cells = G(Λ)·V^{2/N} (eq.(9): within 5 %)
    rng = np.random.default_rng(11)
    dim = lattice
    N = 40000
    ys = (rng.uniform(-8, 8, (N, dim)) * (np.array([S3, 1.0]) if lattice == hqo.A2 else 1.0)).astype(np.float32)
    scale = np.array([S3, 1.0]) if lattice == hqo.A2 else np.ones(dim)
    e2 = 0.0
    for y in ys:
        c = hqo.nearest(lattice, y, clamp=False)
        e2 += ((y.astype(np.float64) - c * scale) ** 2).sum()
    m = e2 / (N * dim)
    G = GOLD["table2_G"][{1: "Z", 2: "A2", 4: "D4", 8: "E8"}[lattice]]
    V2N = {1: 1.0, 2: 2 * S3, 4: np.sqrt(2.0), 8: 4.0}[lattice]
    assert abs(m / (G * V2N) - 1) < 0.02
    assert abs(hqo.second_moment(lattice) / (G * V2N) - 1) < 1e-5
    if lattice == hqo.E8:
        assert abs(m - GOLD["sigma2_V"]["E8"]) < 0.006          # "≈0.287 in our scaling", L808


def test_clamp_keeps_codes_in_int8_and_in_lattice():
    # G8: adversarial tiles (all energy in one coordinate: α√n ≈ 166 at 5 bps / 128) stay valid
    for lattice in (hqo.Z, hqo.A2, hqo.D4, hqo.E8):
        dim = lattice
        for v in (126.4, 126.5, 127.49, 127.5, 166.0, 400.0, -126.5, -127.5, -166.0, 1e6):
            for pos in range(dim):
                y = np.full(dim, 0.49, np.float32); y[pos] = v
                c = hqo.nearest(lattice, y).astype(np.int64)
                assert np.abs(c).max() <= 127 and _members(lattice, c[None])[0], (lattice, y, c)


# ------------------------------------------------------------------ dither (A.6, Thm 1)
@pytest.mark.parametrize("lattice", [hqo.Z, hqo.A2, hqo.D4, hqo.E8])
def test_dither_uniform_on_voronoi_cell(lattice):
    dim = lattice
    N = 20000
    U = np.stack([hqo.dither_block(lattice, 5, blk % 16, blk // 16, 1, 0) for blk in range(N)]).astype(np.float64)
    # U lies in V(Λ): its nearest lattice point is the origin
    inside = sum((hqo.nearest(lattice, u.astype(np.float32), clamp=False) == 0).all() for u in U[:500])
    assert inside >= 495                                   # boundary ties only
    m2 = (U ** 2).sum() / (N * dim)
    assert abs(m2 / hqo.second_moment(lattice) - 1) < 0.03        # paper asks 5 % (L847)
    assert np.abs(U.mean(0)).max() < 5 * np.sqrt(hqo.second_moment(lattice) / N)   # mean 0 (eq.(7))
    cov = U.T @ U / N
    assert np.abs(cov - np.eye(dim) * hqo.second_moment(lattice)).max() < 0.03 * dim ** 0.5   # isotropic (L808)
    if lattice == hqo.Z:
        assert abs(m2 - GOLD["sigma2_V"]["Z"]) < 0.002


def test_dither_is_a_function_of_its_counter_only():
    a = hqo.dither_block(hqo.E8, 9, 3, 77, 2, 1)
    assert (a == hqo.dither_block(hqo.E8, 9, 3, 77, 2, 1)).all()
    for other in [(10, 3, 77, 2, 1), (9, 4, 77, 2, 1), (9, 3, 78, 2, 1), (9, 3, 77, 3, 1), (9, 3, 77, 2, 0)]:
        assert (a != hqo.dither_block(hqo.E8, *other)).any()
