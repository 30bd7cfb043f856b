"""CPU oracle for H|psi> -- TEST INFRASTRUCTURE, not the product.

Plain, slow, obviously-correct implementation of what the hot path computes,
written from /root/reference/PAPER.md (cited per function as PAPER.md:<line>).
Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` /
``--impl reference`` legs of ``bench.py`` may import this package.  It shares
no code with ``paper_2308_07277_b200`` and neither imports the other.

Parts:
  O1  gsphere.py      G-sphere enumeration, sphere->box index map, |k+G|^2
  O2  hpsi.py         H apply by direct O(N_G^2) G-space summation
                      (dense-matrix numpy form for small N_G; the same triple
                      sum as explicit C loops in hpsi_direct.c for large N_G)
  O3  dft.py          naive DFT straight from the definition (8^3-size checks)
  O5  subspace.py     subspace products <psi_i|phi_j>
  O7  propagate.py    Taylor-series exp(-i dt H) psi, eq. 52, and the split-operator form, eq. 53 (8(f) rank 3;
                      PAPER.md:1131-1139)
  O8  mtxel.py        GW plane-wave matrix elements M_nn'(k,q,G), eq. 56 (8(f) rank 4)
  O6  density.py      n(r) = sum_i f_i |psi_i(r)|^2 by direct synthesis (8(f) rank 2)

Pins (tests/test_oracle_*.py, ``-m "not gpu"``): the paper's printed bcc
example, closed-form plane-wave
eigenvalues, single-Fourier-component shift, rank-1 projector, Hermiticity,
naive-DFT brute force on 8^3, numpy fftn identity; for O5 unit
vectors, a geometric-sequence closed form, the inner-product axioms, np.vdot.
Parity unpinned: none of the functions here; absolute physical energies of
real Si are out of scope (no pseudopotential data).
"""
