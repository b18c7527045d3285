"""hq_linear_static: the batch-1 fused kernel with its scratch in a file-scope device array (include/hq.h).

Collected last on purpose (the suite runs with pytest -x).  The new entry point must give what hq_linear gives at batch 1
- same kernel, same flat tile partition, scratch elsewhere - on two calls in a row (the array keeps the first call's
contents), must allocate nothing, and must reject weights whose scratch does not fit.  Passes alone in a fresh process
and after the other GPU tests (it builds its own context and weights).
"""
import numpy as np
import pytest

import hq_synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

SNR_E8_4BPS = float(np.float32(22.68))


def _rel_err(y, ref, floor=1e-3):
    """max |y - ref| / max(|ref|, floor * rms(ref)): the linear-output measure of tests/test_gpu_parity.py (G16)."""
    ref = np.asarray(ref, np.float64)
    rms = np.sqrt((ref ** 2).mean())
    return np.max(np.abs(np.asarray(y, np.float64) - ref) / np.maximum(np.abs(ref), floor * rms + 1e-30))


@pytest.fixture(scope="module")
def ctx():
    import paper_2606_23406_b200 as hq
    c = hq.Context(0)
    yield c
    c.close()


# (m_out, n_in): a Llama-shaped square, a wide-K matrix whose row blocks are cut into many split-K segments, a ragged
# row count below one row block per warp group
@pytest.mark.parametrize("m,n_in", [(4096, 4096), (1024, 14336), (300, 1024)])
def test_linear_static_matches_hq_linear_on_two_calls_in_a_row(ctx, m, n_in):
    import paper_2606_23406_b200 as hq
    dev = torch.device("cuda", 0)
    W = torch.from_numpy(hq_synth.gaussian_weight(m, n_in, seed=11)).to(dev).to(torch.bfloat16)
    w = ctx.encode_weights(W, hq.Lattice.E8, 128, SNR_E8_4BPS, seed=3)
    xs = [torch.from_numpy(hq_synth.activations(1, n_in, seed=s)).to(dev).to(torch.bfloat16) for s in (21, 22)]
    # the existing path first (it may grow the context's workspace: that is its business)
    refs = []
    for x in xs:
        y, y32, _ = w.linear(x, want_f32=True)
        refs.append((y.clone(), y32.clone()))
    torch.cuda.synchronize()
    y = torch.empty(m, dtype=torch.bfloat16, device=dev)
    y32 = torch.empty(m, dtype=torch.float32, device=dev)
    for call, x in enumerate(xs):          # two calls in a row on the shared array, different inputs
        y.fill_(float("nan")); y32.fill_(float("nan"))
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated(dev)
        w.linear_static(x.view(-1), y, y32)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated(dev) == before       # nothing came from the allocator the context was given
        ref_bf16, ref_f32 = refs[call]
        assert torch.isfinite(y32).all()
        # tolerance of test_linear_group_is_bit_identical_to_separate_calls at batch 1 (fp32 re-association, G14)
        assert _rel_err(y32.cpu().numpy(), ref_f32.view(-1).cpu().numpy()) < 1e-5, (m, n_in, call)
        d = (y.float() - ref_bf16.view(-1).float()).abs()
        assert (d <= ref_bf16.view(-1).float().abs() * 2.0 ** -7 + 1e-6).all()      # within one bf16 ulp
    w.free()


def test_linear_static_bf16_only_and_f32_input(ctx):
    import paper_2606_23406_b200 as hq
    dev = torch.device("cuda", 0)
    m, n_in = 512, 2048
    W = torch.from_numpy(hq_synth.gaussian_weight(m, n_in, seed=12)).to(dev)
    w = ctx.encode_weights(W, hq.Lattice.E8, 128, SNR_E8_4BPS, seed=4)
    x = torch.from_numpy(hq_synth.activations(1, n_in, seed=23)).to(dev)            # fp32 activations
    ref = w.linear(x)
    y = torch.empty(m, dtype=torch.bfloat16, device=dev)
    for _ in range(2):
        y.zero_()
        w.linear_static(x.view(-1), y)
        torch.cuda.synchronize()
        d = (y.float() - ref.view(-1).float()).abs()
        assert (d <= ref.view(-1).float().abs() * 2.0 ** -7 + 1e-6).all()
    w.free()


def test_linear_static_rejects_what_does_not_fit_or_is_not_its_path(ctx):
    import paper_2606_23406_b200 as hq
    from paper_2606_23406_b200.binding import HQError
    dev = torch.device("cuda", 0)
    # another lattice: not the kernel this entry point wraps
    W = torch.from_numpy(hq_synth.gaussian_weight(256, 512, seed=13)).to(dev)
    wd4 = ctx.encode_weights(W, hq.Lattice.D4, 128, float(np.float32(22.5)), seed=5)
    x = torch.from_numpy(hq_synth.activations(1, 512, seed=24)).to(dev)
    y = torch.empty(256, dtype=torch.bfloat16, device=dev)
    with pytest.raises(HQError, match="E8"):
        wd4.linear_static(x.view(-1), y)
    wd4.free()
    # beyond the stated maximum: m_out = 262144 + 128 rows need 2049 x 16 counter bytes > 32 KiB
    m = 262144 + 128
    Wb = torch.from_numpy(hq_synth.gaussian_weight(m, 128, seed=14)).to(dev).to(torch.bfloat16)
    wb = ctx.encode_weights(Wb, hq.Lattice.E8, 128, SNR_E8_4BPS, seed=6)
    del Wb
    xb = torch.from_numpy(hq_synth.activations(1, 128, seed=25)).to(dev).to(torch.bfloat16)
    yb = torch.empty(m, dtype=torch.bfloat16, device=dev)
    with pytest.raises(HQError, match="static scratch holds"):
        wb.linear_static(xb.view(-1), yb)
    ref = wb.linear(xb)                     # the allocating path still takes it
    assert torch.isfinite(ref.float()).all()
    wb.free()
    # a large weight inside the limit (m_out <= 160 000 always fits) runs and agrees
    m2 = 159872
    W2 = torch.from_numpy(hq_synth.gaussian_weight(m2, 256, seed=15)).to(dev).to(torch.bfloat16)
    w2 = ctx.encode_weights(W2, hq.Lattice.E8, 128, SNR_E8_4BPS, seed=7)
    del W2
    x2 = torch.from_numpy(hq_synth.activations(1, 256, seed=26)).to(dev).to(torch.bfloat16)
    y2 = torch.empty(m2, dtype=torch.bfloat16, device=dev)
    w2.linear_static(x2.view(-1), y2)
    ref2 = w2.linear(x2)
    torch.cuda.synchronize()
    d = (y2.float() - ref2.view(-1).float()).abs()
    assert (d <= ref2.view(-1).float().abs() * 2.0 ** -7 + 1e-6).all()
    w2.free()
