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
double *v1_fit_preact(const V1Weights &W, void *ws, int64_t n, int *row_len);
cudaError_t v1_pass1(const DevModel &P, const ChunkView &C, const V1Weights &W, cudaStream_t st);
cudaError_t v1_fit(const DevModel &P, const ChunkView &C, const V1Weights &W, const double *fit, void *ws,
                   double *atom_energy, cudaStream_t st);
cudaError_t v1_pass2(const DevModel &P, const ChunkView &C, const V1Weights &W, double *force, double *virial,
                     cudaStream_t st);

cudaError_t v1_plain_gemm(int64_t rows, const double *A, int lda, const double *B, int ldb, int K, int N,
                          const double *Cin, double *Cout, int ldc, const int *range, cudaStream_t st);

// Variant 2 ("paper pipeline", strawman.cu): padded-dense, unfused embedding stage of PAPER.md
// section 3.2.3 — GEMMs over all padded slots with the bias folded in, concat as a GEMM with (I, I), separate tanh /
// tanh-grad kernels, G and every activation materialised.
struct V2Weights {
  double *buf = nullptr;      // per net: B0 B1 II1 B2 II2 B2T II2T B1T II1T B0T (padded, see strawman.cu)
  int *range = nullptr;       // device {0, INT_MAX}
  int LD0 = 0, LD1 = 0, LD2 = 0;
  long long net_stride = 0;
  bool ready = false;
};
cudaError_t v2_prepare_weights(const DevModel &P, const double *emb_h, V2Weights &W);
void v2_release_weights(V2Weights &W);
size_t v2_slot_bytes(const V2Weights &W);                         // workspace per padded slot of a net batch
cudaError_t v2_pass1(const DevModel &P, const ChunkView &C, const V2Weights &W, const int *type_start_h, void *ws,
                     cudaStream_t st);
cudaError_t v2_pass2(const DevModel &P, const ChunkView &C, const V2Weights &W, const int *type_start_h, void *ws,
                     double *force, double *virial, cudaStream_t st);

#ifdef __CUDACC__
// tanh(x) = 1 - 2 / (exp(2x) + 1) with exp(2x) = 2^n 2^f: n = rint(2x log2 e) by the 1.5 * 2^52 trick, 2^f by a
// degree-10 polynomial on [-0.5, 0.5] (relative error 2.9e-16), the reciprocal from MUFU.RCP64H refined by one cubic
// step.  18 fp64-pipe instructions; absolute error <= 4.5e-16 against libdevice on [-25, 25], [-1, 1], [-0.01, 0.01]
// and [-1e-6, 1e-6] (4e7 points each, profiles/r1_fp64_peaks.md); libdevice's tanh costs 2.2x the pipe slots.
__device__ __forceinline__ double dp_tanh(double x) {
  const int hi = __double2hiint(x);
  const bool big = (hi & 0x7fffffff) >= 0x40340000;                 // |x| >= 20: tanh = +-1 in fp64
  const double xc = big ? __hiloint2double((hi & 0x80000000) | 0x40340000, 0) : x;
  const double tm = fma(xc, 2.8853900817779268, 6755399441055744.0); // 2 log2(e) x + 1.5 * 2^52
  const int ni = __double2loint(tm);
  const double f = fma(xc, 2.8853900817779268, 6755399441055744.0 - tm);   // t - rint(t), one rounding
  double p = 7.0725859492692236999e-9;
  p = fma(p, f, 1.0208690299958305835e-7);
  p = fma(p, f, 1.3215442587921689653e-6);
  p = fma(p, f, 0.000015252657260200837064);
  p = fma(p, f, 0.00015403530441736050155);
  p = fma(p, f, 0.0013333558230164973899);
  p = fma(p, f, 0.0096181291076068885273);
  p = fma(p, f, 0.055504108664447719166);
  p = fma(p, f, 0.2402265069591009822);
  p = fma(p, f, 0.69314718055994998286);
  p = fma(p, f, 1.0);
  const double d = __hiloint2double(__double2hiint(p) + ni * 1048576, __double2loint(p)) + 1.0;
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
  const double err = fma(-d, r, 1.0);
  const double tq = fma(err, err, err);
  r = fma(r, tq, r);
  return fma(-2.0, r, 1.0);
}
#endif
