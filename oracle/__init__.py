"""CPU oracle for the chi0*dV hot path of arXiv 2203.05623 (Eq. 10-11).

THIS PACKAGE IS TEST INFRASTRUCTURE.  It is a plain, slow, fp64 NumPy statement of what
the path computes, written from the paper.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import it.  It shares no code with
``paper_2203_05623_b200/`` (the CUDA path) and never imports it; the only module both sides use
is ``synth/`` (seeded inputs, none of the method's arithmetic).

Parity pins (tests/test_oracle_*.py, all ``-m "not gpu"``):
  gsphere      brute-force count identities, involution of -G, paper Table 5 (tests/golden/table5_npw.txt)
  fft          numpy.fft is the library routine; delta -> plane wave closed form, Parseval, round trip
  hamiltonian  dense (index arithmetic) vs matrix-free (FFT) are two independent codes; Hermiticity;
               V=0,D=0 -> |G|^2 c; V=const -> shift; time reversal
  chi0         sum-over-states vs dense Sternheimer solve vs finite-field derivative of the density;
               free-electron Lindhard sum; symmetry/negativity of <dV_j, dn_i>; charge conservation
  pcg/cocg     (full-size sampled columns) true residual < 1e-10 and agreement with sum-over-states
No function in this package is "parity unpinned".
"""
