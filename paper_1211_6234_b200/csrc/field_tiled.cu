// field_tiled.cu -- placeholder until the register-tiled kernel lands.
#include "dsmc_internal.cuh"
size_t dsmc_wk_floats(int) { return 64; }
bool dsmc_tiled_supported(int, int) { return false; }
cudaError_t launch_make_wk(const float *, float *, int, cudaStream_t, uint64_t *) { return cudaSuccess; }
cudaError_t launch_field_tiled(const float *, const float *, float *, float *, int, int, int, int, cudaStream_t,
                               uint64_t *) { return cudaErrorNotSupported; }
