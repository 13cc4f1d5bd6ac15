"""CPU oracle for the DMRG hot path of arXiv:1309.5571 -- TEST INFRASTRUCTURE ONLY.

Plain, slow, obviously-correct numpy FP64 code written from /root/reference/PAPER.md.
It shares no code with the CUDA library in ``paper_1309_5571_b200/`` and neither
imports the other.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import it; the
product path never does and fails loudly when the CUDA library is missing.

Modules:
  ed        O-ED   site-level Hamiltonians on the full 2^N / 4^N space  (Eq. 1-8)
  blocks    O-BLK  exact left/right blocks cut into sector blocks        (L165)
  kron      O-KRON the definition: H = sum_a c_a kron(A_a, B_a) restricted to Q (Eq. 9)
  rec       O-REC  block-wise records  X'_jl += A_{i->j} X_ik B_{k->l}^T  (Eq. 11)
  davidson  O-DAV  textbook Davidson following Alg. 3 line by line

Parity status: every function on the path is pinned by tests/test_oracle_*.py
(closed forms, brute-force ED, invariants); nothing is "parity unpinned".
"""
