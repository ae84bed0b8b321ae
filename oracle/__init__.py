"""CPU oracle for the LSE+OBC hot path of arxiv/paper_2602_03438 (Eqs. 1-2).

TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct NumPy (complex128; the dense
tier optionally in 80-bit extended precision).  Only `tests/`, `__graft_entry__.smoke()`
and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import this package.
It shares no code with `paper_2602_03438_b200/` (the CUDA path) and imports nothing from it.

Tiers:
  dense.py        tier 0 - the DEFINITION: G^R = (zS - H - Sigma^R)^-1, G^<> = G^R Sigma^<> G^A,
                  full dense inversion (fp64 LAPACK, or hand-written extended-precision Gauss-Jordan).
  rgf.py          tier 1 - the recursive Green's function sweeps S3-S6, block by block,
                  in the order and notation of SURVEY.md 8(a)/(c-1).
  obc.py          Sancho-Rubio decimation of the lead blocks.
  observables.py  density, LDOS, transmission, bond and contact currents (readings R11-R13).
  pipeline.py     the whole path for one workload, chaining the above (what bench.py times).
  convolution.py  Eq. 3 for M1 = M2 = I: the discrete energy convolution / correlation
                  of selected blocks as the written-out double sum.

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): tier 1 vs tier 0 on random tiny and
config-shaped inputs; tier 0 fp64 vs extended precision; 1D-chain closed form for the
decimation; integer transmission of a translation-invariant device; current conservation
(PAPER.md:86); selected-block residuals of Eqs. 1-2; anti-Hermiticity; the corrected spectral
identity; hand-solved 1x1/2x2 cases; for the convolution a shifted delta, a polynomial product
with binomial coefficients, np.convolve per element and an np.fft route.  No function here is "parity unpinned".
"""
