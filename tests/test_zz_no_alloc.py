"""taiga_detector_histogram_static against taiga_detector_histogram (run on the B200 box: -m gpu).

Who needs the static entry point: a caller that may not allocate once its loop is running -- an evaluation between
plasma shots that shares the GPU with other streams (cudaMalloc / cudaFree make every stream of the device wait), or
a process whose memory pool already owns the GPU, where a late cudaMalloc fails.  taiga_detector_histogram allocates
its edge buffer (device) and its staging buffer (pinned) on first use; the static variant keeps the edges in a fixed
32 KB array of the library, so it is limited to nu + nw <= 2048 segments and its calls must not overlap on the GPU.

The binning is integer work, so the bar is the one the other histogram tests use: counters, summary, ions.cell and
ions.flags bit for bit.  Two calls in a row, the second with a smaller, gapped detector: the shared array still holds
the first call's edges beyond the second call's, and none of them may show.  The file sorts last on purpose (pytest -x
would otherwise hide every later test behind a failure here) and depends on no state other tests leave behind: it makes
its own contexts, and the array's contents before the first call are irrelevant by construction."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2506_15812_b200 import workloads as wl  # noqa: E402


def _np(t):
    return t.detach().cpu().numpy()


def _binned(tg, call, ions, traced, det, n_hist):
    """Restore the traced per-ion results (the histogram rewrites cell and flags), bin, return everything it wrote."""
    ions.a["cell"].copy_(traced["cell"])
    ions.a["flags"].copy_(traced["flags"])
    counts = torch.zeros((n_hist, det.nw, det.nu), dtype=torch.int64, device="cuda")
    summary = torch.zeros((n_hist, 6), dtype=torch.int64, device="cuda")
    call(ions, det, n_hist, counts, summary)
    torch.cuda.synchronize()
    return _np(counts).copy(), _np(summary).copy(), _np(ions.cell).copy(), _np(ions.flags).copy()


def test_static_histogram_matches_the_allocating_one_on_two_calls_in_a_row():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2506_15812_b200 import taiga
    tg = taiga.Taiga(0)
    try:
        cfg = wl.config(1, n_override=20000 + 13)             # several 256-thread blocks and a ragged tail
        ions, _, _ = taiga.run_config(tg, cfg)                # a1-a4 (+ one ordinary a5) on the product path
        torch.cuda.synchronize()
        # what a3/a4 left: crossers carry CELL_MISS again, flags without the edge bit
        cell = ions.cell.clone()
        cell[cell >= 0] = taiga.CELL_MISS
        traced = dict(cell=cell, flags=(ions.flags & ~torch.tensor(taiga.FLAG_EDGE, dtype=torch.uint8, device="cuda")).clone())
        big = wl.uniform_detector(*wl.DETECTOR_CENTRES["cfg1"], 96, 2.5e-4)          # 9216 counters: the global-atomic path
        small = wl.gapped_detector(cfg.detector)                                     # 8 x 8 with gaps: binary search, smem path
        for det in (big, small):                              # two calls in a row on the shared array
            ref = _binned(tg, tg.detector_histogram, ions, traced, det, cfg.n_hist)
            got = _binned(tg, tg.detector_histogram_static, ions, traced, det, cfg.n_hist)
            assert ref[1][0, 0] > 1000, "the case must put ions on the detector"
            for r, g, what in zip(ref, got, ("counts", "summary", "cell", "flags")):
                assert np.array_equal(r, g), what
        # accumulation into existing counters, as the allocating call does
        counts = torch.ones((1, small.nw, small.nu), dtype=torch.int64, device="cuda")
        summary = torch.zeros((1, 6), dtype=torch.int64, device="cuda")
        ions.a["cell"].copy_(traced["cell"])
        tg.detector_histogram_static(ions, small, 1, counts, summary)
        torch.cuda.synchronize()
        assert np.array_equal(_np(counts), got[0] + 1)
    finally:
        tg.close()


def test_static_histogram_refuses_detectors_beyond_its_fixed_table():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2506_15812_b200 import taiga
    tg = taiga.Taiga(0)
    try:
        ions = taiga.Ions(64)
        ions.a["cell"].fill_(taiga.CELL_MISS)
        nu = taiga.STATIC_MAX_SEGMENTS - 3                    # nu + nw = limit + 1
        det = wl.uniform_detector(0.0, 0.0, nu, 1e-5)
        det.w_lo, det.w_hi = det.w_lo[:4].copy(), det.w_hi[:4].copy()
        counts = torch.zeros((1, 4, nu), dtype=torch.int64, device="cuda")
        summary = torch.zeros((1, 6), dtype=torch.int64, device="cuda")
        with pytest.raises(taiga.TaigaError) as e:
            tg.detector_histogram_static(ions, det, 1, counts, summary)
        assert e.value.code == taiga.E_ARG and "TAIGA_STATIC_MAX_SEGMENTS" in str(e.value)
        torch.cuda.synchronize()
        assert int(counts.sum()) == 0 and int(summary.sum()) == 0          # nothing was enqueued
        det.w_lo, det.w_hi = det.w_lo[:3].copy(), det.w_hi[:3].copy()      # exactly at the limit: accepted
        counts = torch.zeros((1, 3, nu), dtype=torch.int64, device="cuda")
        tg.detector_histogram_static(ions, det, 1, counts, summary)
        ref_c, ref_s = torch.zeros_like(counts), torch.zeros_like(summary)
        ions.a["cell"].fill_(taiga.CELL_MISS)
        ions.a["flags"].zero_()
        tg.detector_histogram(ions, det, 1, ref_c, ref_s)
        torch.cuda.synchronize()
        assert torch.equal(counts, ref_c) and torch.equal(summary, ref_s) and int(summary[0, :2].sum()) == 64
    finally:
        tg.close()
