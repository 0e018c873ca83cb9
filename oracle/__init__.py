"""ORACLE — test infrastructure, NOT part of the product.

A plain, slow, obviously-correct CPU implementation (numpy, fp64) of what the hot path of
arxiv 2208.05637 computes: the local energy E_loc(x) = sum_p alpha_p <x|P_p|x^p> f(x^p)/f(x)
(Eq. 15) of a MADE + phase-MLP wavefunction (Eq. 8-10).

Rules:
  * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
    import this package; the product (paper_2208_05637_b200/) never does, and this package never
    imports the product (not even its input generators: every function takes plain arrays);
  * every function cites the passage it follows; nothing is blocked, fused or reordered beyond
    what the paper's definition states (chunking over terms only bounds memory);
  * every function is pinned in tests/test_oracle_*.py to something other than itself (dense
    Kronecker matrices, Slater-Condon, normalisation over 2^n, closed forms).
    Every function has such a pin: the phase net, "parity unpinned" in round 1, is pinned through an independent
    torch fp64 evaluation and a position-order test (tests/test_oracle_made.py); oracle.grad (Eq. 7) by
    finite differences, torch autograd and exact enumeration against the dense Hamiltonian (tests/test_oracle_grad.py).
"""
