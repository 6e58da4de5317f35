// temporary: variant 1 not built yet
#include "v1_kernels.cuh"
cudaError_t v1_prepare_weights(const DevModel &, const double *, const double *, V1Weights &) { return cudaSuccess; }
void v1_release_weights(V1Weights &) {}
size_t v1_workspace_bytes(const DevModel &, int64_t) { return 256; }
cudaError_t v1_pass1(const DevModel &, const ChunkView &, const V1Weights &, cudaStream_t) { return cudaErrorNotSupported; }
cudaError_t v1_fit(const DevModel &, const ChunkView &, const V1Weights &, const double *, void *, double *, cudaStream_t) { return cudaErrorNotSupported; }
cudaError_t v1_pass2(const DevModel &, const ChunkView &, const V1Weights &, double *, double *, cudaStream_t) { return cudaErrorNotSupported; }
