"""B200-native hot path of the He-4 variational Monte Carlo of arXiv:1312.1282.

`binding` is the ctypes layer over the C ABI of include/qmc.h (libqmc_b200.so, built in-tree by `build`);
`workloads` holds the seeded inputs of BASELINE.json's five configs; `parallel` shards walkers over ranks;
`observables` normalises g(r) and reblocks energy series on the host.  Nothing here computes a step of the
method: every step of the path runs in the CUDA kernels under csrc/.
"""
