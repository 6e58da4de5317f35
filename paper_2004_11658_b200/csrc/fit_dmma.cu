// fit_dmma.cu — variant 1 of S5 (D = T T^<T), S6 (fitting net forward), S7 (fitting backward + dT).
// TEMPORARY: routes to the variant-0 GEMM kernels until the DMMA fitting kernels land.
#include "v1_kernels.cuh"

size_t v1_workspace_bytes(const DevModel &P, int64_t chunk) {
  return sizeof(double) * (size_t)chunk * (2 * (size_t)P.dim + 7 * (size_t)P.fw) + 256;
}

cudaError_t v1_fit(const DevModel &P, const ChunkView &C, const V1Weights &W, const double *fit, void *ws,
                   double *atom_energy, cudaStream_t st) {
  (void)W;
  double *p = reinterpret_cast<double *>(ws);
  const size_t n = (size_t)C.n;
  V0Scratch S;
  S.D = p; p += n * P.dim;
  S.dD = p; p += n * P.dim;
  S.Z0 = p; p += n * P.fw;
  S.U1 = p; p += n * P.fw;
  S.Z1 = p; p += n * P.fw;
  S.U2 = p; p += n * P.fw;
  S.Z2 = p; p += n * P.fw;
  S.G = p; p += n * P.fw;
  S.dZ = p;
  return launch_fit_v0(P, C, fit, S, atom_energy, nullptr, st);
}
