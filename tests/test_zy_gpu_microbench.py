"""GPU micro-benchmark (-m gpu) of the two SM units the hot kernels are bound by, re-measured from the tree
(imager_debug_probe, csrc/probe.cu).  DESIGN.md 6.1 and bench.py's `roofline.lsu_floor_ms` rest on: a warp-wide LDS.64 costs
about 2.1 clocks per SM whatever its lane mask (so 16 idle lanes buy nothing), and a warp-wide FFMA2 about 0.565 clocks per
SM (113 of the nominal 128 FMA lanes per clock).  The windows below are those claims with room for clock and scheduling
noise; the measured values are printed (run with -s).  Collected near the end so that a shifted number on another box
cannot hide the parity tests under `pytest -x`."""
import pytest

pytestmark = pytest.mark.gpu


def test_lds64_and_ffma2_issue_rates():
    import torch
    assert torch.cuda.is_available()
    from paper_2206_15117_b200.binding import debug_probe
    r = debug_probe()
    print(f"LDS.64: {r['lds64_clk']:.3f} clk per warp instruction per SM (32 lanes), {r['lds64_half_mask_clk']:.3f} (16 lanes); "
          f"FFMA2: {r['ffma2_clk']:.3f}; {r['n_sm']} SMs")
    assert 1.9 <= r["lds64_clk"] <= 2.4                                   # 256 B per instruction through 128 B/clk
    assert abs(r["lds64_half_mask_clk"] - r["lds64_clk"]) <= 0.15 * r["lds64_clk"]      # the mask does not make it cheaper
    assert 0.49 <= r["ffma2_clk"] <= 0.65                                 # 4 schedulers x at most one instruction per 2 clk
