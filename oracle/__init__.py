"""CPU oracle for the PSWF-LR reciprocal-space path (arxiv/paper_2606_06617).

TEST INFRASTRUCTURE ONLY.  Plain, slow, float64.  Shares no code with the CUDA
path in ``paper_2606_06617_b200/`` and is never imported by it.  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import, call, link or execute anything in here.

Modules (each function cites the PAPER.md passage it follows):

  pswf.py      psi_0^c, lambda_0, C_0              Eq. (7)-(9), (S37)-(S41)
  kernels.py   S^_p(k), Phi^_p(k), k=0 constants,  Theorem 1 (S47)-(S52), (S60),
               S_p(r), S_p(0)                      (S17)-(S33), (S67), (S73)-(S79)
  direct.py    oracle A: direct non-uniform        Eq. (5)-(6)
               Fourier sums for E, phi, F;
               virial_direct (strain derivative)
  direct_sum.c same sums in plain C/OpenMP for the
               large configurations
  gridded.py   oracle B: spread/FFT/scale/iFFT/    Eq. (20)-(26)
               gather in float64 numpy
  scaffold.py  real-space complement, self term,   (S64)-(S68), Eq. (12)
               classical erfc Ewald; real_space_parts is
               the parity target of pswf_lr_execute_real

Pins (tests/test_oracle_*.py) and their status are listed in DESIGN.md §3.
Parity unpinned: none of the functions used for GPU parity; the paper's own
fp32 error tables S1-S3 are context only (cells and P not given).
"""
