"""B200-native hot path of the submatrix method (arXiv:2004.10811): C-ABI library + thin binding.

`binding` marshals arguments to libsubmatrix_b200.so (include/submatrix.h); every step of the
path runs in the library's CUDA kernels.  `workloads` fabricates seeded synthetic inputs."""
