"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol include/hq.h declares."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "hq.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hq_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_header_symbols():
    from paper_2606_23406_b200 import build, EXPORTS
    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert len(names) >= 15 and {"hq_encode_weights", "hq_linear", "hq_kv_append", "hq_attend"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in hq.h but not exported"
    assert sorted(EXPORTS) == names                 # the binding covers the whole header


def test_no_gpu_means_loud_failure_not_fallback():
    import pytest
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2606_23406_b200 as hq
    with pytest.raises(hq.HQError):
        hq.Context(0)
    lib = hq.load_library()
    assert abs(lib.hq_alpha(8, 20.0) - (10 ** 2.0 * 0.0717 * 4) ** 0.5) < 1e-12   # eq.(9), host-only call


def test_snr_for_bps_table_reproduces_the_papers_anchors():
    """hq_snr_for_bps (host-only lookup in the committed calibration table, G17) against what the paper prints:
    Rice rates at 21 dB on iid Gaussian tiles 3.74 / 3.77 / 3.81 / 3.84 bps for E8 / D4 / A2 / Z;
    A2 + Rice SNR 16.02 / 22.21 / 28.26 dB at 3 / 4 / 5 bps (Table 11); alpha(5 bps) = 14.7 / 13.6 / 7.4 for
    E8 / A2 / Z (Table 14); E8 - Z gap 0.81 dB at 3 bps -> 0.65 dB at 5 bps (L383)."""
    import pytest
    import paper_2606_23406_b200 as hq
    E8, D4, A2, Z = 8, 4, 2, 1
    for lat, bps in ((E8, 3.74), (D4, 3.77), (A2, 3.81), (Z, 3.84)):
        assert abs(hq.snr_for_bps(lat, bps)[0] - 21.0) < 0.15                       # 0.02 bps ~ 0.12 dB
    for bps, snr in ((3.0, 16.02), (4.0, 22.21), (5.0, 28.26)):
        assert abs(hq.snr_for_bps(A2, bps)[0] - snr) < 0.1
    for lat, a in ((E8, 14.7), (A2, 13.6), (Z, 7.4)):
        assert abs(hq.alpha(lat, hq.snr_for_bps(lat, 5.0)[0]) - a) < 0.15
    gap3 = hq.snr_for_bps(E8, 3.0)[0] - hq.snr_for_bps(Z, 3.0)[0]
    gap5 = hq.snr_for_bps(E8, 5.0)[0] - hq.snr_for_bps(Z, 5.0)[0]
    assert abs(gap3 - 0.81) < 0.06 and abs(gap5 - 0.65) < 0.06
    assert hq.snr_for_bps(E8, 4.0)[1] == (2, 2) and hq.snr_for_bps(E8, 2.0)[1] == (0, 0)   # k = 0,1,2,3 at 2,3,4,5 bps (G10)
    with pytest.raises(hq.HQError):
        hq.snr_for_bps(E8, 50.0)                                                    # outside the table


def test_calibration_table_matches_the_oracle_at_sampled_grid_points():
    """The committed table is what oracle/make_calib_table.py writes: re-run the oracle on three grid points."""
    import numpy as np
    import hq_synth
    import paper_2606_23406_b200 as hq
    from oracle import hqo
    tiles = hq_synth.calib_tiles(100000, 128, 42)
    for lat, snr in ((hqo.E8, 22.75), (hqo.D4, 12.0), (hqo.Z, 30.5)):
        bps, k, _, _ = hqo.calib_point(tiles, lat, snr)
        got, kk = hq.snr_for_bps(lat, float(np.float32(round(bps, 5))))
        assert abs(got - snr) < 2e-3 and tuple(int(v) for v in k) == kk


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2606_23406_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("oracle/", "").lower() or f in ("hq_common.cuh", "hq_calib_table.inc"), f
