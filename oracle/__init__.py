"""CPU oracle for the U(1)xSU(2)-symmetric two-site TDVP hot path (arxiv/paper_2606_04771).

TEST INFRASTRUCTURE ONLY.  Plain, slow numpy code written from the paper
 and from the readings listed in DESIGN.md.  Nothing
under ``paper_2606_04771_b200/`` may import this package; only ``tests/``,
``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs
of ``bench.py`` do.  It shares no code with the CUDA path.

Modules
-------
su2        Clebsch-Gordan coefficients (Racah formula) and the recoupling
           coefficients coefL / coefR as explicit sums over six CGs.
fermi      Jordan-Wigner site operators, dense Hamiltonian Eq. (1), exact
           diagonalisation (O-ED), pseudospin generators Eqs. (4)-(6).
u0         U=0 closed form by single-particle propagation (O-U0).
dense_tdvp dense, non-symmetric two-site TDVP (O-D).
symm       symmetric block-sparse reference (O-S): sector tables, reduced
           MPO, dense embedding, environments, H_eff, SVD split, task lists.
symm_tdvp  two-site TDVP driver on top of ``symm`` (O-S driver).

Parity status: every function is pinned by tests/test_oracle_*.py (-m "not gpu");
see DESIGN.md section "Oracle pins".
"""
