"""B200-native non-symmetric Laplace-transform J/K build (arxiv/paper_2607_05622 hot path).

`ltjk`   -- ctypes binding of the C ABI (include/ltjk.h) around libltjk.so (CUDA, sm_100a)
`inputs` -- seeded synthetic workloads (no method arithmetic)
`build`  -- in-tree build of libltjk.so
"""
