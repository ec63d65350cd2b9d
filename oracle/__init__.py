"""CPU oracle for the TDVP hot path of arXiv:1907.12044 -- TEST INFRASTRUCTURE ONLY.

A plain, slow, obviously-correct numpy implementation (complex128 / float64) of what the CUDA
path in ``paper_1907_12044_b200/`` computes, written from the paper (``PAPER.md``) step by step
in the paper's order and notation.  It shares no code with the CUDA path; neither imports the
other.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import it.

Modules (SURVEY.md section 8(c) numbering):
  model.py         O1  Frenkel-Holstein Hamiltonian (Eq. 45) -> MPO (Eq. 11), Kronecker-sum H
  contractions.py  O2  H_eff apply (Eq. 29/43), environment updates (Eq. 30-32), bond apply (Eq. 44)
  lanczos.py       O3  Lanczos/Krylov exponential
  tdvp_ps.py       O4  TDVP-PS symmetric sweep (Eq. 42-44)
  tdvp_mu.py       O5  TDVP-MU derivative (Eq. 27, 33, 36-38) + one Dormand-Prince 5(4) step
  tdvp_cmf.py      O5b TDVP-MU with constant-mean-field integration, second-order midpoint scheme
  observables.py   O6  populations, norm, energy
  exact.py         O7  full-Hilbert-space propagation (tiny chains only)

Pins (tests/test_oracle_pins.py, run with -m "not gpu"): p1-p9 of SURVEY.md 8(c); p12, p13 for the CMF
scheme (its local right-hand side is the pinned MU derivative; second order in the step, the paper's
Fig. 7 slope, and agreement with TDVP-PS).  The paper states neither the predictor of the midpoint
mean field nor the local Runge-Kutta method of CMF: those two choices are readings (DESIGN.md c19),
parity unpinned against the paper's own (unstated) ones.
Parity unpinned: the adaptive Krylov stopping rule and the adaptive RK45 step controller (the
paper gives no formula for either) -- the contract mode is fixed k / fixed h;
and the paper's own Tables II/III and Figs. 4-7, which need FMO parameters that are not available.
"""
