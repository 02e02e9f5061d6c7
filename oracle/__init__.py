"""CPU FP64 oracle for the DMRG hot path.  TEST INFRASTRUCTURE ONLY.

Plain, slow, obviously-correct numpy implementations of what the CUDA library
computes.  Only `tests/`,
`__graft_entry__.smoke()` and the `cpu_baseline` / `--impl reference` legs of
`bench.py` may import this package.  It shares no code with
`paper_2603_28648_b200/`; both read the seeded inputs of `fixtures/`.

Pins (tests/test_oracle_*.py, `-m "not gpu"`):
  fock.py     FCI: V=0 closed form, Hubbard dimer closed form, Lanczos = dense
              eigh = Jacobi, [H,N]=[H,Sz]=[H,S^2]=0, hermiticity.
  abelian.py  cut identity and blocking identities as operator identities vs
              Jordan-Wigner matrices (L=4); H_eff.psi and renormalization vs the
              brute-force projected Hamiltonian P^T H P (L=4,6,8).
  su2.py      Wigner 6j/9j vs orthogonality sums and exact values; reduced
              operators vs Wigner-Eckart projections of Jordan-Wigner matrices;
              H_eff.psi vs Clebsch-Gordan expansion into Fock space.
  davidson.py monotone Ritz values bounded by the dense lowest eigenvalue;
              cfg0 sweep energy = FCI within 1e-8 Eh.
Large configs (cfg2..cfg4 full size): parity unpinned beyond the sampled
blocks and invariants.
"""
