"""B200-native batched ADMM-QP hot path of TurboMPC (arxiv/paper_2606_24039).

`binding` mirrors the C ABI of include/tmpc.h (libtmpc.so, hand-written sm_100a CUDA kernels); `solver.Solver`
bundles a handle with device tensors; `workloads` holds the seeded synthetic input generators (no method arithmetic).
Nothing here imports the CPU oracle (oracle/ is test infrastructure)."""
