// tc_kernels.cuh — interface of the mixed-precision (tcgen05 / TMEM) kernels.  Internal.
#pragma once
#include "common.cuh"

// Embedding nets as shared-memory images: TF32 hi / lo operand panels (K-major, 128-byte swizzle) + fp32 vectors.
struct TCWeights {
  float *emb = nullptr;       // ntypes^2 images
  size_t net_stride = 0;      // floats per image
  bool ready = false;
  void *fit = nullptr;        // fitting weights as B operand images (fit_tc.cu)
};

cudaError_t tc_prepare_weights(const DevModel &P, const double *emb_h, TCWeights &W);
void tc_release_weights(TCWeights &W);

// flattened list of the real (non-padded) slots per neighbour-type section of one chunk
size_t tc_pair_workspace_bytes(const DevModel &P, int64_t chunk);
cudaError_t tc_build_pairs(const DevModel &P, const ChunkView &C, void *pair_ws, cudaStream_t st);

cudaError_t tc_pass1(const DevModel &P, const ChunkView &C, const TCWeights &W, const void *pair_ws, cudaStream_t st);
size_t tc_pass2_workspace_bytes(const DevModel &P, int64_t chunk);      // fp32 copy of dT
cudaError_t tc_pass2(const DevModel &P, const ChunkView &C, const TCWeights &W, const void *pair_ws, const float *dT32,
                     double *force, double *virial, cudaStream_t st);

// fitting stage (fit_tc.cu): E_i and dT (fp64 in C.dT and the fp32 copy dT32) from C.T
// opf: operand format of the fitting GEMMs: 0 = 3xTF32, 1 = BF16 x 6 products, 2 = plain BF16 (fit_tc.cu)
cudaError_t tc_prepare_fit(const DevModel &P, const double *fit_h, TCWeights &W, int opf);
void tc_release_fit(TCWeights &W);
size_t tc_fit_workspace_bytes(const DevModel &P, int64_t chunk, int opf);
cudaError_t tc_fit(const DevModel &P, const ChunkView &C, const TCWeights &W, void *ws, float *dT32, double *atom_energy,
                   cudaStream_t st, bool want_dT64);   // want_dT64: also write C.dT (fp64 view of dT for the debug hook)
