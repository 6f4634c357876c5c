"""darts-b200: B200-native group-rollout decoding for DARTS (arxiv/paper_2605_30859).

`paper_2605_30859_b200.api`       thin ctypes binding over the C-ABI library (include/darts.h);
                                  importing it loads csrc/libdarts.so and fails loudly if absent.
`paper_2605_30859_b200.workloads` seeded synthetic inputs (no method arithmetic; shared with tests).
`paper_2605_30859_b200.build`     nvcc build of csrc/ into libdarts.so (sm_100a).
"""
