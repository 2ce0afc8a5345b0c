"""B200-native Landau Jacobian hot path (arxiv 2104.10000): CUDA kernels behind a C ABI."""
