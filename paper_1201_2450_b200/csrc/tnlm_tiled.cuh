// Tiled sm_100a TNLM sweep kernel (placeholder until the first measured design lands).
#pragma once
#include "tnlm_common.cuh"

namespace tnlm {

inline bool tiled_supported(const tnlm_params &) { return false; }
inline size_t tiled_scratch_bytes(const tnlm_params &) { return 0; }
inline const char *tiled_name(const tnlm_params &) { return "none"; }
inline int tiled_launches_per_sweep(const tnlm_params &) { return 1; }
inline cudaError_t launch_tiled(const tnlm_params &, const Dims &, const float *, const float *, const float *,
                                float *, void *, size_t, cudaStream_t)
{
    return cudaErrorNotSupported;
}

}  // namespace tnlm
