"""B200-native hot path of the block-time-step Hermite direct N-body method of arXiv:1312.1789
(PAPER.md:15, :43): j-predictor, O(N_act N) force with derivatives, corrector + block time step.

`paper_1312_1789_b200.nbody`     -- thin ctypes binding of the C-ABI library (include/nbody.h); importing it
                                     fails loudly if csrc/libnbody.so is missing (no CPU fallback exists).
`paper_1312_1789_b200.workloads` -- seeded synthetic inputs (no method arithmetic).
`paper_1312_1789_b200.build`     -- nvcc build of csrc/ for sm_100a.
"""
