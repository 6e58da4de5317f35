// tc_kernels.cuh — interface of the mixed-precision (tcgen05 / TMEM) kernels.  Internal.
#pragma once
#include "common.cuh"

// Embedding nets as shared-memory images: TF32 hi / lo operand panels (K-major, 128-byte swizzle) + fp32 vectors.
struct TCWeights {
  float *emb = nullptr;       // ntypes^2 images
  size_t net_stride = 0;      // floats per image
  bool ready = false;
};

cudaError_t tc_prepare_weights(const DevModel &P, const double *emb_h, TCWeights &W);
void tc_release_weights(TCWeights &W);

// flattened list of the real (non-padded) slots per neighbour-type section of one chunk
size_t tc_pair_workspace_bytes(const DevModel &P, int64_t chunk);
cudaError_t tc_build_pairs(const DevModel &P, const ChunkView &C, void *pair_ws, cudaStream_t st);

cudaError_t tc_pass1(const DevModel &P, const ChunkView &C, const TCWeights &W, const void *pair_ws, cudaStream_t st);
size_t tc_pass2_workspace_bytes(const DevModel &P, int64_t chunk);      // fp32 copy of dT
cudaError_t tc_pass2(const DevModel &P, const ChunkView &C, const TCWeights &W, const void *pair_ws, void *ws2,
                     double *force, double *virial, cudaStream_t st);
