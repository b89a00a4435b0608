// ca_fused.cuh -- temporally fused reaction-diffusion kernel (all n_sub sub-steps of S1 in one pass).
// Placeholder interface for the first bring-up: reports "unsupported", so the per-sub-step kernel runs.
#pragma once
#include "ca_device.cuh"

namespace ca {
inline void fused_configure(const KParams &) {}
inline bool fused_supported(const KParams &) { return false; }
inline void launch_fused(const KParams &, const Lattice &, int, const long long *, int, cudaStream_t) {}
}  // namespace ca
