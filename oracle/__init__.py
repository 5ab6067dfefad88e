"""Oracle: plain, slow, fp64 CPU implementation of the w-projection gridding path.

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import, call, link or execute anything in this
directory.  The product path (``paper_1905_03213_b200`` + ``libwpgrid.so``)
shares no code with it and never routes through it.

What it computes (the readings listed in DESIGN.md):

=========  ==================================================================
module     definition followed
=========  ==================================================================
taper      O2  prolate-spheroidal taper psi(nu), c = 3*pi (north_star:
               "prolate-spheroidal taper"; paper silent)
wkernel    O3  K1-K6 oversampled W-kernel stack, direct-DFT form
               ("new convolution kernel function"; PAPER.md:108
               "number of w-projection planes is 23, full support size 9")
gridder    O4  G1-G7 convolutional gridding (data model
               row x channel PAPER.md:56), plain C loops in grid_oracle.c;
               degrid(): its adjoint with unit weights;
               flux(): P11's right-hand side and the grid's first moments in
               O(nvis) without a grid (checks full-size GPU runs);
               cells(): single grid cells one by one, G5 read as a gather
               (full-size GPU runs on sampled outputs)
image      O5  dirty image = centred inverse FFT / taper
           O6  brute-force direct 3-D DFT image (pin for the whole chain)
baseline_  Eqs. (1)-(2): baseline index from antenna IDs, count array C, exclusive
order      prefix sum, stable baseline-then-time re-order
=========  ==================================================================

Parity pins (tests/ -m "not gpu"): P1 taper vs independent Legendre recipe and
printed values, P2 direct double sum vs zero-padded FFT route, P3 symmetries,
P4 w=0 separability, P5 slice sums ~ 1, P6/P7 worked index/plane examples
(tests/golden/), P8 stored kernel values (tests/golden/), P9 gridded dirty
image vs direct 3-D DFT, P10 single-visibility footprint, P11 flux
conservation (and oracle_flux against the Python P11 sum, hand-written moment
sums and the gridded result; oracle_cells against the gather written out in
Python and against the scatter-form grid, every cell), P12 linearity/chunking; Eqs. (1)-(2): worked example, bijection onto the antenna
triangle, closed-form row starts, numpy cumsum / stable argsort
(tests/test_oracle_baseline_order.py); degridder: adjoint identity, single-cell
grids, prediction of the measurement model (tests/test_oracle_degrid.py).  No function here is "parity unpinned".
"""
