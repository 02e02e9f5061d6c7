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
              brute-force projected Hamiltonian P^T H P (six cases with L=4,5).
  su2.py      the SU(2) result DEFINED by Clebsch-Gordan expansion into abelian.py;
              Clebsch-Gordan exact values, closed forms, orthogonality.
  wigner.py   6j/9j vs exact rationals, closed forms, orthogonality sums, the
              Clebsch-Gordan definition of the 9j, sympy for j <= 3.
  su2_loopnest.py  loop-nest H_eff.psi / renormalization on reduced elements with
              6j/9j recoupling (part c4): = su2.py on eight systems to 1e-12.
  abelian_terms.py, falg.py  un-enlarged term list (= abelian.py) and the
              algorithmic flop count F_alg (brute-force enumeration).
  davidson.py monotone Ritz values bounded by the dense lowest eigenvalue;
              cfg0 sweep energy = FCI within 1e-8 Eh.
Large configs (cfg2..cfg4 full size): checked on seeded samples of output blocks
with su2_loopnest.py (tests/test_gpu_fullsize.py).
"""
