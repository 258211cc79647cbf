"""CPU oracle for the ILE hot path of arxiv/paper_2505_11655 ("Narrowing RIFT").

TEST INFRASTRUCTURE ONLY.  Plain, slow, double-precision numpy written from the paper
 and the readings listed in DESIGN.md section 3.  Only ``tests/``,
``__graft_entry__.smoke()``, ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` leg and
``oracle/make_injections.py`` may import it.  It shares no code with
``paper_2505_11655_b200`` (the CUDA path) and never imports it; the product path never
imports this package.

Pin status (tests/test_oracle_*.py, ``-m "not gpu"``):
  likelihood.antenna, .ylm, .lnL ............ pinned (P1-P6, P8: closed forms, sum rules,
                                              zero-noise injection rho^2/2, quadrature)
  reduce.reduce_lnw ......................... pinned (P7: constant / Gaussian closed forms)
  philox.philox4x32_10 ...................... pinned against cuRAND's host generator
                                              (library routine), plus uniformity tests
  integrators.AC / AV / GMM / Portfolio ..... algorithm constants (eps, beta, P_thr, N_min*,
                                              EM schedule) are this build's readings of a
                                              paper that defers them to refs [23],[64]:
                                              **parity unpinned** w.r.t. RIFT's own code;
                                              pinned only through closed-form integrals and
                                              invariants (P9-P11)
  distance-table lookup ..................... pinned (P12: quadrature, Laplace limit)
"""
