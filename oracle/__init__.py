"""CPU ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, obviously-correct restatement of what the gridding / degridding hot path of
arxiv/paper_2206_15117 computes, written from the paper and, where the paper is
silent, from the readings listed in DESIGN.md ("Readings") which restate SURVEY.md section 8(c)
steps O0-O7.  Arithmetic is fp64 / complex128 throughout (visibilities, weights and kernel
tables are complex64/float32 inputs, as the paper's GPU path would hold them).

Rules (task statement, item 3):
  * only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
    leg may import or execute anything in here;
  * nothing in here imports `paper_2206_15117_b200` or reads any file the CUDA path produced;
  * no blocking, fusion or re-ordering beyond what each cited definition states.

Modules
  index.py    O1 visibility -> (cell, sub-cell, signed w-plane, kernel set, drop), O2 bucket key + stable sort
  kernels.py  O6 kernel tables (DELTA, PSWF, WPROJ, AWPROJ_ADJOINT, AWPROJ_PAPER, MOSAIC_PB), Eq. 2-6 helpers
  gridder.c   O4 gridding, O5 degridding (plain C loops, double accumulation, OpenMP over rows / visibilities)
  gridder.py  ctypes wrapper of gridder.c
  imaging.py  O0/O7 grid<->image DFT with taper correction, direct DFT, Eq. 1 mosaic weighting

Pins (tests/test_oracle_*.py, `-m "not gpu"`): P1-P14 of DESIGN.md.  Parity unpinned: see DESIGN.md
"Parity unpinned" (config-level choices only: support schedule, PA binning, channel width, latitude).
"""
