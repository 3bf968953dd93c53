"""mc_edep_total_static (include/mc.h): the energy-ledger total for callers that may not allocate GPU memory.

Some users of this library cannot call cudaMalloc: the process around them has given nearly all device memory to a
framework's caching allocator (a raw allocation fails), or another thread is recording a CUDA graph in the global capture
mode (an allocation anywhere in the process is illegal then), or they sit in a loop that cannot take the device-wide stall
an allocation causes.  For them the library has one call that creates no device state: the caller passes the per-batch
energy grids and a place for the result, and the partial sums live in a fixed array inside the library's device image.

The tests check that call against the path that existed before it — sum_kernel, whose result mc_get_stats returns as
e_deposited_MeV — on two calls in a row with different inputs and sizes, so a ticket or a partial left over from the first
call would show in the second.  The bar is the one tests/test_gpu_coupled.py uses for fp64 statistics of the fp32 grids
(rtol 1e-6); both sides add the same floats in fp64 and differ only in rounding order, so a plain fp64 sum on the host is
checked far more tightly as well.

The file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide another test), and it
must pass both alone in a fresh process and after the rest of the suite — it assumes nothing about what ran before."""
import numpy as np
import pytest

import paper_1503_01722_b200 as mc
from paper_1503_01722_b200 import workloads as W


def test_sizes_beyond_the_fixed_scratch_are_refused_with_a_message():
    # argument checks come before any CUDA call, so this part runs without a GPU; the pointer is never dereferenced
    lim = mc.mc_edep_total_static_max()
    assert lim == 2 ** 28
    dummy = np.zeros(4, np.float32)
    with pytest.raises(mc.McError) as e:
        mc.mc_edep_total_static(dummy, lim + 1)
    assert e.value.status == mc.MC_ERR_INVALID_ARG and "larger than the fixed scratch" in str(e.value) and str(lim) in str(e.value)
    with pytest.raises(mc.McError) as e:
        mc.mc_edep_total_static(dummy, 0)
    assert e.value.status == mc.MC_ERR_INVALID_ARG
    with pytest.raises(mc.McError) as e:
        mc.mc_edep_total_static(None, 16)
    assert e.value.status == mc.MC_ERR_INVALID_ARG and "null" in str(e.value)


@pytest.mark.gpu
def test_static_scratch_total_matches_the_ledger_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available()
    cfg = W.config(1)
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    # call 1: a large input (many chunks, ragged tail); call 2: a smaller one with other contents — stale partials beyond
    # its last chunk and the previous ticket must not leak into it; call 3: the first input again
    cases = [(40000, 7, 11), (20000, 3, 12), (40000, 7, 11)]
    seen = {}
    for n, B, seed in cases:
        p = mc.mc_edep_buffer(eng.ctx, B)
        mc.mc_run_range(eng.ctx, cfg["beam"], n, 0, n, seed, B, p)
        ledger = mc.mc_get_stats(eng.ctx)["e_deposited_MeV"]  # the existing path: sum_kernel + fp64 atomics
        assert ledger > 0
        count = B * eng.nvox
        assert count % 4096 != 0  # ragged last chunk
        got = mc.mc_edep_total_static(p, count)
        assert abs(got - ledger) <= 1e-6 * ledger, (got, ledger)
        # the same histories into a caller-owned buffer, whose plain fp64 sum on the host side is the tight reference
        dev = torch.zeros(count, dtype=torch.float32, device="cuda")
        mc.mc_run_range(eng.ctx, cfg["beam"], n, 0, n, seed, B, dev)
        ref = float(dev.double().sum().item())
        got_dev = mc.mc_edep_total_static(dev, count, torch.cuda.current_stream().cuda_stream)
        assert abs(got_dev - ref) <= 1e-12 * ref, (got_dev, ref)
        # fixed summation order: the same data gives the same bits, call after call
        assert mc.mc_edep_total_static(dev, count) == got_dev
        # the first input again after a different one: the same total up to the fp32 order of the scoring atomics (two runs
        # of the same histories give grids that differ in the last bits; include/mc.h, mc_run)
        seen.setdefault((n, B, seed), got_dev)
        assert abs(seen[(n, B, seed)] - got_dev) <= 1e-6 * got_dev
    eng.close()


@pytest.mark.gpu
def test_static_scratch_total_on_known_arrays_and_device_output():
    import torch
    assert torch.cuda.is_available()
    g = torch.Generator(device="cpu").manual_seed(5)
    for count in (1, 255, 4096, 4097, 3 * 4096 * 1184 + 17, 2 ** 22 + 3):  # one element .. more chunks than CTAs
        a = torch.rand(count, generator=g, dtype=torch.float32)
        ref = float(a.double().sum().item())
        d = a.cuda()
        assert abs(mc.mc_edep_total_static(d, count) - ref) <= 1e-12 * ref + 1e-300
        out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")  # the result may also stay on the device
        mc.mc_edep_total_static(d, count, 0, out)
        assert abs(float(out.item()) - ref) <= 1e-12 * ref
        # a view that starts in the middle of the buffer (not 16-byte aligned) sums just as well
        if count > 8:
            ref1 = float(a[1:].double().sum().item())
            assert abs(mc.mc_edep_total_static(d.data_ptr() + 4, count - 1) - ref1) <= 1e-12 * ref1
    # host memory is refused, not read
    with pytest.raises(mc.McError) as e:
        mc.mc_edep_total_static(np.ones(8, np.float32), 8)
    assert e.value.status == mc.MC_ERR_INVALID_ARG and "not device memory" in str(e.value)
