"""B200-native pressure projection (forward + adjoint), MGPCG and advection for NeuralFluid
(arXiv 2405.14903).  The product is the C-ABI library built from csrc/ (include/nf.h); `api` is the thin
ctypes binding; `workloads` are the seeded synthetic inputs.  There is no CPU fallback: using `api`
without the built CUDA library raises."""
__all__ = ["api", "workloads"]
