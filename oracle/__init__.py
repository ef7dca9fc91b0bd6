"""CPU oracle for the AMPLFI data-generation hot path (arXiv 2407.19048, section 3).

THIS PACKAGE IS TEST INFRASTRUCTURE, NOT PRODUCT.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import it.  The product (``paper_2407_19048_b200``) never imports it and has no
CPU fallback.  It shares no code, header, table or constant generator with the CUDA path.

Everything is plain numpy in fp64 (complex128), written in the order of the paper's own
statement of the steps (section 3.2):

    waveform  -> oracle.waveform
    detector projection -> oracle.project
    power-spectrum estimate -> oracle.welch
    injection + whitening -> oracle.whiten
    two data views d, d' -> oracle.views
    Fourier transforms -> oracle.fft  (naive O(N^2) DFT for N <= 64,
                                          plain recursive radix-2 FFT above that)

The paper prints none of the formulas; each function states the passage it follows and the
DESIGN.md reading it takes.  Pins live in tests/test_oracle_*.py (``-m "not gpu"``).

Parity status of the oracle itself:
  * oracle.fft, oracle.welch, oracle.whiten, oracle.project, TaylorF2 in oracle.waveform:
    pinned (numpy.fft / scipy.signal.welch / numpy.interp agreement, closed forms,
    brute force, worked-example values under tests/golden/).
  * oracle.waveform.imrphenomd: every closed-form ingredient is pinned (aligned-spin PN phase and
    amplitude coefficients against the (chi_s, chi_a, delta) form of [32] App. B, test-mass limits of
    the remnant fits, exchange symmetry, C1 junctions, the time-domain peak at t_c:
    tests/test_oracle_phenomd_pins.py; the Kerr (2,2,0) mode against published values and the
    defining continued fractions: tests/test_oracle_qnm.py).  What stays **parity unpinned** is
    oracle.phenomd_coeffs.TABLE, the 19 x 11 fitted numbers of [32] Table V, typed as recalled:
    lalsimulation is not available and PAPER.md prints none of them (DESIGN.md R-W1).
"""
