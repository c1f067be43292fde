"""-m gpu: mcx_cnr_static, the one entry point that needs no device memory from the caller (include/mcx.h): tally finalise +
CNR of PAPER.md:257 Eq. (1) with the intermediate arrays in the library's file-scope device scratch, against the existing
path (mcx_tally_read + mcx_cnr with the caller's buffers).  Two calls in a row on different detectors and instruments: the
scratch is shared and keeps the last call's contents.  (Collected last on purpose; passes alone in a fresh process too.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def M():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import paper_2410_08747_b200 as m
    m.lib()
    return m


def _existing(g, det, rm, rr, efit):
    c, fit = g.cnr(det, rm, rr, efit)                                           # mcx_tally_read + mcx_cnr, caller's buffers
    return c.cpu().numpy(), fit.cpu().numpy()


def _with_energy_bins(inst, n_e):
    inst = dict(inst)
    inst["components"] = [dict(c) for c in inst["components"]]
    for c in inst["components"]:
        if c["kind"] == "detector":
            c["nE"] = n_e
    return inst


def _close(a, b):
    return np.allclose(a, b, rtol=1e-11, atol=1e-300)                           # (tests/test_gpu_next.py's CNR tolerance)


def test_static_scratch_cnr_equals_the_existing_path_on_two_calls_in_a_row(M, W):
    import torch
    big = M.Instrument(_with_energy_bins(W.config1(small=True), 64))            # 64 x 64 pixels x 64 energy bins = 2^18 bins: the limit
    assert big.dets[0]["nx"] * big.dets[0]["ny"] * big.dets[0]["nE"] == M.binding.CNR_STATIC_MAX_BINS
    big.trace(2_000_000)
    small = M.Instrument(W.config7(small=True))                                 # five line detectors, fewer bins: stale data beyond them
    small.trace(300_000)
    torch.cuda.synchronize()
    calls = [(big, 0, (10, 20, 10, 20), (40, 50, 30, 40), 80.0)]
    d = small.dets[1]
    calls.append((small, 1, (0, 1, 0, d["ny"] // 2), (0, 1, d["ny"] // 2, d["ny"]), d["Emin"]))
    calls.append((big, 0, (0, 64, 0, 1), (3, 4, 5, 64), 20.0))
    calls.append((small, 4, (0, 1, 1, 3), (0, 1, 5, 9), 0.5 * (d["Emin"] + d["Emax"])))
    for dev_out in (False, True):
        for g, det, rm, rr, efit in calls:
            ne = g.dets[det]["nE"]
            if dev_out:
                out, fit = torch.full((ne,), -1.0, dtype=torch.float64, device="cuda"), torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
            else:
                out, fit = torch.full((ne,), -1.0, dtype=torch.float64).pin_memory(), torch.full((2,), -1.0, dtype=torch.float64).pin_memory()
            g.cnr_static(det, rm, rr, efit, out, fit)
            torch.cuda.synchronize()
            want_c, want_fit = _existing(g, det, rm, rr, efit)
            assert np.any(want_c > 0.0)
            assert _close(out.cpu().numpy(), want_c) and _close(fit.cpu().numpy(), want_fit)
            del out, fit
    # back to back on one stream without a synchronize in between: stream order keeps the shared scratch consistent; and
    # the device's free memory, as the driver counts it, is the same before and after (outputs made beforehand)
    outs = [(torch.empty(g.dets[det]["nE"], dtype=torch.float64, device="cuda"), torch.empty(2, dtype=torch.float64, device="cuda"))
            for g, det, _, _, _ in calls[:2]]
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for (g, det, rm, rr, efit), (out, fit) in zip(calls[:2], outs):
        g.cnr_static(det, rm, rr, efit, out, fit)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    for (g, det, rm, rr, efit), (out, fit) in zip(calls[:2], outs):
        want_c, want_fit = _existing(g, det, rm, rr, efit)
        assert _close(out.cpu().numpy(), want_c) and _close(fit.cpu().numpy(), want_fit)
    big.close()
    small.close()


def test_static_scratch_cnr_refuses_what_does_not_fit(M, W):
    import torch
    g = M.Instrument(_with_energy_bins(W.config1(small=True), 65))              # one energy bin above the 2^18 bins
    assert g.dets[0]["nx"] * g.dets[0]["ny"] * g.dets[0]["nE"] > M.binding.CNR_STATIC_MAX_BINS
    out, fit = torch.empty(g.dets[0]["nE"], dtype=torch.float64, device="cuda"), torch.empty(2, dtype=torch.float64, device="cuda")
    with pytest.raises(M.McxError) as err:
        g.cnr_static(0, (0, 1, 0, 1), (1, 2, 0, 1), 0.0, out, fit)
    assert "static scratch" in str(err.value)
    g.close()
    g = M.Instrument(W.config4(small=True))
    out, fit = torch.empty(g.dets[0]["nE"], dtype=torch.float64, device="cuda"), torch.empty(2, dtype=torch.float64, device="cuda")
    with pytest.raises(M.McxError):
        g.cnr_static(0, (0, 65, 0, 1), (0, 1, 0, 1), 80.0, out, fit)            # region outside the detector
    import ctypes as C
    rm, rr = (C.c_int32 * 4)(0, 1, 0, 1), (C.c_int32 * 4)(1, 2, 0, 1)
    status = g.L.mcx_cnr_static(g.handle, 3, rm, rr, 80.0, out.data_ptr(), fit.data_ptr(), None)  # no such detector
    assert status != 0 and b"out of range" in g.L.mcx_last_error()
    assert g.L.mcx_cnr_static(g.handle, 0, rm, rr, 80.0, None, fit.data_ptr(), None) != 0         # null output
    g.close()
