"""oracle/ -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

A plain, slow, float64 CPU restatement of what the NUFFT hot path of arxiv 1710.03197 (PyNUFFT)
computes: A = V F S (eq. 1), A^H = S^H F^H V^H (eq. 2), A^H A (PAPER.md:96,
eq. 5), the multi-coil operator (eqs. 34-35) and the solvers built on them
(PAPER.md:124-198).

Rules this package lives under:
  * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import it;
  * it imports nothing from paper_1710_03197_b200/ (the CUDA path) and the CUDA path imports nothing from
    here; the two share no kernels, tables, constants or helpers;
  * numpy only, float64/complex128 throughout, no blocking / fusion / reordering beyond what the paper's
    statement of each step says.

Modules:
  nufft_oracle.py    kernel, scaling factors, stencil, V, V^H, forward, adjoint, selfadjoint, direct NDFT,
                     multi-coil
  solvers_oracle.py  gradient, shrink, CG, L1TV-OLS
  next_oracle.py     density compensation (eqs. 6-7), Toeplitz A^H A

Parity status of every function is listed in each module's header.
"""
