// v1_kernels.cuh — interface of the fused DMMA kernels (variant 1).  Internal.
#pragma once
#include "common.cuh"

// Embedding weights re-laid-out for the m8n8k4 fp64 tensor-core tiles (see embed_dmma.cu for the layout).
struct V1Weights {
  double *emb = nullptr;      // ntypes^2 padded nets
  long long net_stride = 0;   // doubles per padded net
  int SP = 0;                 // feature slots per lane quarter and copy: ceil(s1 / 4)
  bool ready = false;
  void *fit = nullptr;        // padded fitting weights (fit_dmma.cu)
};

cudaError_t v1_prepare_fit(const DevModel &P, const double *fit_h, V1Weights &W);
void v1_release_fit(V1Weights &W);

cudaError_t v1_prepare_weights(const DevModel &P, const double *emb_h, const double *fit_h, V1Weights &W);
void v1_release_weights(V1Weights &W);
size_t v1_workspace_bytes(const DevModel &P, int64_t chunk);
cudaError_t v1_pass1(const DevModel &P, const ChunkView &C, const V1Weights &W, cudaStream_t st);
cudaError_t v1_fit(const DevModel &P, const ChunkView &C, const V1Weights &W, const double *fit, void *ws,
                   double *atom_energy, cudaStream_t st);
cudaError_t v1_pass2(const DevModel &P, const ChunkView &C, const V1Weights &W, double *force, double *virial,
                     cudaStream_t st);
