"""CPU oracle for the sparse-SYK hot path of arxiv 2311.00639 -- TEST INFRASTRUCTURE ONLY.

This package is the slow, plain, fp64 definition of what the CUDA library must compute.
It is written from /root/reference/PAPER.md (cited as "PAPER.md:<line>") and DESIGN.md's
readings, builds matrices (Kronecker products, monomial rows) rather than bit-mask tables,
and shares no code, header, table or constant generator with `paper_2311_00639_b200/`.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import it.  The product path never does.

Modules
  rng          counter-based generator, Bernoulli/Gaussian sampling of Eq. (1)   (O1)
  majorana     dense Majorana matrices: Jordan-Wigner and the paper's Eq. (S1)   (O2)
  hamiltonian  dense H, monomial-row evaluation, derived integer tables, H.v     (O3-O5)
  evolve       exact exp(-i tau H) by full diagonalisation; Chebyshev series     (O6, O8)
  otoc         same-psi and exact-trace regularised OTOC                        (O7)
  green        same-psi and exact-trace retarded Green function
  pauli        generic sums of Pauli strings / spin chains by Kronecker products
  parity       parity blocks H_UU / H_DD, gamma blocks, block OTOC / Green function
  nonhermitian complex-coupling SYK Hamiltonian; exp(-i tau H) v by the dense matrix exponential
  alg1         literal transcription of the paper's Algorithm 1 (Python + C)    (P6)

Pins (tests/test_oracle_*.py, `-m "not gpu"`): Clifford algebra, Hermiticity/trace/parity,
Tr H^2 closed form, hand-worked Pauli products (tests/golden/), two representations with one
spectrum, literal Algorithm 1 vs dense, exactly solvable exponentials, group properties,
OTOC and Green-function closed forms, nilpotent / diagonal / anti-Hermitian exponentials.  Parity unpinned: none of the functions here; what stays unpinned is
agreement with the paper's Fig. 1 curves and its iteration counts (no data in PAPER.md).
"""
