"""B200-native GRPIC hot path (arxiv 2503.04558): GR particle push fused with
charge-conserving current deposition, GR Maxwell field update, cell sort and compaction,
as hand-written sm_100a CUDA kernels behind the C-ABI library `libgrpic.so`
(include/grpic.h).  `grpic` is the thin ctypes binding; `inputs` the seeded synthetic
input generators.  There is no CPU fallback: using `grpic` without the built library or
without a GPU raises."""
