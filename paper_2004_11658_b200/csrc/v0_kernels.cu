// v0_kernels.cu — variant 0: plain, unfused CUDA kernels for S3..S9 (thread-per-output FMA loops, libdevice tanh).
// They are the correctness-first strawman the fused DMMA kernels (variant 1) are measured against; both are
// checked against the CPU oracle by tests/.  Equation references: see include/dpb.h.
#include "common.cuh"

#define RG 8   // neighbour rows processed together by the embedding kernels

// Env-matrix row of a real slot (Eq. 5; Alg. 2 :212-238): s = w(r)/r, R~ = (s, s d/r).
__device__ __forceinline__ void env_row(const DevModel &P, const double4 v, double e[4]) {
  double w, dw;
  dp_switch(v.w, P.rcs, P.rc, w, dw);
  const double ir = 1.0 / v.w;
  const double s = w * ir;
  e[0] = s; e[1] = s * v.x * ir; e[2] = s * v.y * ir; e[3] = s * v.z * ir;
}

// ---------------------------------------------------------------------------------------------------------
// S3 + S4 + S5 (forward): T_i = sum_k g_k (x) R~_k (Eq. 4 left factor).  Block per atom, thread o owns T[o][0..3].
__global__ void k_pass1_v0(DevModel P, ChunkView C, const double *__restrict__ emb) {
  extern __shared__ double sm[];
  const int s1 = P.s1, s2 = 2 * P.s1, M = P.M;
  double *env = sm;                 // [RG][4]
  double *h0 = env + RG * 4;        // [RG][s1]
  double *h1 = h0 + RG * s1;        // [RG][2 s1]
  const int tid = threadIdx.x, q = blockIdx.x;
  const int i = C.s_idx[C.p0 + q];
  (void)i;
  // centre type from the sorted position
  int a = 0;
  while (C.p0 + q >= C.type_start[a + 1]) ++a;
  double Tacc[4] = {0.0, 0.0, 0.0, 0.0};
  for (int t = 0; t < P.ntypes; ++t) {
    const double *W0 = emb + (size_t)(a * P.ntypes + t) * P.emb_net_size;
    const double *b0 = W0 + s1, *W1 = b0 + s1, *b1 = W1 + (size_t)s1 * s2, *W2 = b1 + s2, *b2 = W2 + (size_t)s2 * M;
    const int n = C.nreal[(size_t)q * P.ntypes + t];
    const double4 *dr = C.dr + (size_t)q * P.nm + P.sec_start[t];
    for (int r0 = 0; r0 < n; r0 += RG) {
      const int nr = min(RG, n - r0);
      if (tid < RG) {
        double e[4] = {0.0, 0.0, 0.0, 0.0};
        if (tid < nr) env_row(P, dr[r0 + tid], e);
        env[tid * 4 + 0] = e[0]; env[tid * 4 + 1] = e[1]; env[tid * 4 + 2] = e[2]; env[tid * 4 + 3] = e[3];
      }
      __syncthreads();
      // layer 0 (Eq. 8): h0 = tanh(x W0 + b0)
      for (int idx = tid; idx < RG * s1; idx += blockDim.x) {
        const int r = idx / s1, k = idx - r * s1;
        h0[idx] = tanh(env[r * 4] * W0[k] + b0[k]);
      }
      __syncthreads();
      // layer 1 (Eq. 9): h1 = (h0, h0) + tanh(h0 W1 + b1)
      for (int idx = tid; idx < RG * s2; idx += blockDim.x) {
        const int r = idx / s2, o = idx - r * s2;
        double acc = b1[o];
        for (int k = 0; k < s1; ++k) acc += h0[r * s1 + k] * W1[(size_t)k * s2 + o];
        h1[idx] = h0[r * s1 + (o % s1)] + tanh(acc);
      }
      __syncthreads();
      // layer 2 (Eq. 9): g = (h1, h1) + tanh(h1 W2 + b2);  T[o][c] += g[o] R~[c]
      if (tid < M) {
        const int o = tid;
        double acc[RG];
#pragma unroll
        for (int r = 0; r < RG; ++r) acc[r] = b2[o];
        for (int k = 0; k < s2; ++k) {
          const double w = W2[(size_t)k * M + o];
#pragma unroll
          for (int r = 0; r < RG; ++r) acc[r] += h1[r * s2 + k] * w;
        }
#pragma unroll
        for (int r = 0; r < RG; ++r) {
          if (r < nr) {
            const double g = h1[r * s2 + (o % s2)] + tanh(acc[r]);
#pragma unroll
            for (int c = 0; c < 4; ++c) Tacc[c] += g * env[r * 4 + c];
          }
        }
      }
      __syncthreads();
    }
  }
  if (tid < M) {
    double *T = C.T + ((size_t)q * M + tid) * 4;
    T[0] = Tacc[0]; T[1] = Tacc[1]; T[2] = Tacc[2]; T[3] = Tacc[3];
  }
}

cudaError_t launch_pass1_v0(const DevModel &P, const ChunkView &C, const double *emb, cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  const int threads = ((P.M + 31) / 32) * 32;
  const size_t smem = sizeof(double) * (RG * 4 + RG * P.s1 + RG * 2 * P.s1);
  k_pass1_v0<<<C.n, threads, smem, st>>>(P, C, emb);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// S8 + S9: per real slot, dE_i/dR~_k and dE_i/dx through the embedding net (forward-mode tangent g' = dg/dx, so
// that dx = <dT R~_k, g'>), chained to the displacement (O10) and scattered: F_i += f_ik, F_j -= f_ik,
// Xi -= d_ik (x) f_ik (ProdForce / ProdVirial).
__global__ void k_pass2_v0(DevModel P, ChunkView C, const double *__restrict__ emb, double *__restrict__ force,
                           double *__restrict__ virial) {
  extern __shared__ double sm[];
  const int s1 = P.s1, s2 = 2 * P.s1, M = P.M;
  double *env = sm;                   // [RG][4]
  double *h0 = env + RG * 4;          // [RG][s1]
  double *h0p = h0 + RG * s1;         // [RG][s1]   d h0 / dx
  double *h1 = h0p + RG * s1;         // [RG][2 s1]
  double *h1p = h1 + RG * s2;         // [RG][2 s1]
  double *red = h1p + RG * s2;        // [nwarps][RG][5]
  double *out = red + (blockDim.x / 32) * RG * 5;   // [RG][5] dR~[0..3], dx
  __shared__ double facc[RG][3], vacc[RG][9];
  const int tid = threadIdx.x, q = blockIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
  const int i = C.s_idx[C.p0 + q];
  int a = 0;
  while (C.p0 + q >= C.type_start[a + 1]) ++a;
  double dTo[4] = {0.0, 0.0, 0.0, 0.0};
  if (tid < M) {
    const double *d = C.dT + ((size_t)q * M + tid) * 4;
    dTo[0] = d[0]; dTo[1] = d[1]; dTo[2] = d[2]; dTo[3] = d[3];
  }
  if (tid < RG) {
    for (int c = 0; c < 3; ++c) facc[tid][c] = 0.0;
    for (int c = 0; c < 9; ++c) vacc[tid][c] = 0.0;
  }
  __syncthreads();
  for (int t = 0; t < P.ntypes; ++t) {
    const double *W0 = emb + (size_t)(a * P.ntypes + t) * P.emb_net_size;
    const double *b0 = W0 + s1, *W1 = b0 + s1, *b1 = W1 + (size_t)s1 * s2, *W2 = b1 + s2, *b2 = W2 + (size_t)s2 * M;
    const int n = C.nreal[(size_t)q * P.ntypes + t];
    const double4 *dr = C.dr + (size_t)q * P.nm + P.sec_start[t];
    const int *nl = C.nl + (size_t)q * P.nm + P.sec_start[t];
    for (int r0 = 0; r0 < n; r0 += RG) {
      const int nr = min(RG, n - r0);
      if (tid < RG) {
        double e[4] = {0.0, 0.0, 0.0, 0.0};
        if (tid < nr) env_row(P, dr[r0 + tid], e);
        env[tid * 4 + 0] = e[0]; env[tid * 4 + 1] = e[1]; env[tid * 4 + 2] = e[2]; env[tid * 4 + 3] = e[3];
      }
      __syncthreads();
      for (int idx = tid; idx < RG * s1; idx += blockDim.x) {
        const int r = idx / s1, k = idx - r * s1;
        const double t0 = tanh(env[r * 4] * W0[k] + b0[k]);
        h0[idx] = t0;
        h0p[idx] = (1.0 - t0 * t0) * W0[k];                      // d tanh = 1 - tanh^2
      }
      __syncthreads();
      for (int idx = tid; idx < RG * s2; idx += blockDim.x) {
        const int r = idx / s2, o = idx - r * s2;
        double acc = b1[o], accp = 0.0;
        for (int k = 0; k < s1; ++k) {
          const double w = W1[(size_t)k * s2 + o];
          acc += h0[r * s1 + k] * w;
          accp += h0p[r * s1 + k] * w;
        }
        const double t1 = tanh(acc);
        h1[idx] = h0[r * s1 + (o % s1)] + t1;
        h1p[idx] = h0p[r * s1 + (o % s1)] + (1.0 - t1 * t1) * accp;
      }
      __syncthreads();
      double part[RG][5];
#pragma unroll
      for (int r = 0; r < RG; ++r)
#pragma unroll
        for (int c = 0; c < 5; ++c) part[r][c] = 0.0;
      if (tid < M) {
        const int o = tid;
        double acc[RG], accp[RG];
#pragma unroll
        for (int r = 0; r < RG; ++r) { acc[r] = b2[o]; accp[r] = 0.0; }
        for (int k = 0; k < s2; ++k) {
          const double w = W2[(size_t)k * M + o];
#pragma unroll
          for (int r = 0; r < RG; ++r) {
            acc[r] += h1[r * s2 + k] * w;
            accp[r] += h1p[r * s2 + k] * w;
          }
        }
#pragma unroll
        for (int r = 0; r < RG; ++r) {
          const double t2 = tanh(acc[r]);
          const double g = h1[r * s2 + (o % s2)] + t2;
          const double gp = h1p[r * s2 + (o % s2)] + (1.0 - t2 * t2) * accp[r];
          double dg = 0.0;                                         // dg[o] = sum_c dT[o][c] R~[c]
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            part[r][c] = dTo[c] * g;                               // dR~[c] = sum_o dT[o][c] g[o]
            dg += dTo[c] * env[r * 4 + c];
          }
          part[r][4] = dg * gp;                                    // dx = sum_o dg[o] g'[o]
        }
      }
      // block reduction over o of the RG x 5 partials
#pragma unroll
      for (int r = 0; r < RG; ++r)
#pragma unroll
        for (int c = 0; c < 5; ++c) {
          double v = part[r][c];
#pragma unroll
          for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
          if (lane == 0) red[(wid * RG + r) * 5 + c] = v;
        }
      __syncthreads();
      if (tid < RG * 5) {
        double v = 0.0;
        for (int w = 0; w < nw; ++w) v += red[w * RG * 5 + tid];
        out[tid] = v;
      }
      __syncthreads();
      if (tid < nr) {
        // O10: derivative of R~ with respect to the displacement; f_ik[c] = sum_m dR~[m] dR~_m/dd_c
        const double4 v = dr[r0 + tid];
        const double d[3] = {v.x, v.y, v.z};
        const double r = v.w;
        double w, dw;
        dp_switch(r, P.rcs, P.rc, w, dw);
        const double ir = 1.0 / r;
        const double s = w * ir, qq = s * ir;
        const double sp = dw * ir - w * ir * ir;
        const double qp = sp * ir - s * ir * ir;
        const double dR0 = out[tid * 5 + 0] + out[tid * 5 + 4];
        const double dRv[3] = {out[tid * 5 + 1], out[tid * 5 + 2], out[tid * 5 + 3]};
        const double dot = dRv[0] * d[0] + dRv[1] * d[1] + dRv[2] * d[2];
        double f[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) f[c] = (dR0 * sp + qp * dot) * d[c] * ir + qq * dRv[c];
        const int j = nl[r0 + tid];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          facc[tid][c] += f[c];
          if (force) atomicAdd(&force[3 * (size_t)j + c], -f[c]);
        }
#pragma unroll
        for (int x = 0; x < 3; ++x)
#pragma unroll
          for (int y = 0; y < 3; ++y) vacc[tid][3 * x + y] -= d[x] * f[y];
      }
      __syncthreads();
    }
  }
  if (tid < 3 && force) {
    double s = 0.0;
    for (int r = 0; r < RG; ++r) s += facc[r][tid];
    atomicAdd(&force[3 * (size_t)i + tid], s);
  }
  if (tid >= 32 && tid < 41 && virial) {
    double s = 0.0;
    for (int r = 0; r < RG; ++r) s += vacc[r][tid - 32];
    atomicAdd(&virial[tid - 32], s);
  }
}

cudaError_t launch_pass2_v0(const DevModel &P, const ChunkView &C, const double *emb, double *force, double *virial,
                            cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  int threads = ((P.M + 31) / 32) * 32;
  if (threads < 64) threads = 64;
  const size_t smem = sizeof(double) * (RG * 4 + 2 * RG * P.s1 + 2 * RG * 2 * P.s1 + (threads / 32) * RG * 5 + RG * 5);
  k_pass2_v0<<<C.n, threads, smem, st>>>(P, C, emb, force, virial);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// S5 (second factor): D[b][a] = sum_c T[b][c] T[a][c], a < M^< (Eq. 4; flatten b*M^< + a, R7).
__global__ void k_descr_v0(DevModel P, ChunkView C, double *__restrict__ D, double *dbgD) {
  const int q = blockIdx.x;
  const double *T = C.T + (size_t)q * P.M * 4;
  const int i = C.s_idx[C.p0 + q];
  for (int e = threadIdx.x; e < P.dim; e += blockDim.x) {
    const int b = e / P.Ma, a = e - b * P.Ma;
    double acc = 0.0;
#pragma unroll
    for (int c = 0; c < 4; ++c) acc += T[b * 4 + c] * T[a * 4 + c];
    D[(size_t)q * P.dim + e] = acc;
    if (dbgD) dbgD[(size_t)i * P.dim + e] = acc;
  }
}

// S7 (contraction backward): dT[b][c] = sum_a dD[b][a] T[a][c] + [b < M^<] sum_b' dD[b'][b] T[b'][c].
__global__ void k_dT_v0(DevModel P, ChunkView C, const double *__restrict__ dD) {
  const int q = blockIdx.x;
  const double *T = C.T + (size_t)q * P.M * 4;
  const double *dd = dD + (size_t)q * P.dim;
  for (int e = threadIdx.x; e < P.M * 4; e += blockDim.x) {
    const int b = e >> 2, c = e & 3;
    double acc = 0.0;
    for (int a = 0; a < P.Ma; ++a) acc += dd[b * P.Ma + a] * T[a * 4 + c];
    if (b < P.Ma)
      for (int bp = 0; bp < P.M; ++bp) acc += dd[bp * P.Ma + b] * T[bp * 4 + c];
    C.dT[(size_t)q * P.M * 4 + e] = acc;
  }
}

// Tiled fp64 GEMM for the fitting net of one species: rows = the chunk's atoms of type `ty` (a contiguous range
// of sorted positions read from the device), C = epi(A op(B)).  64x64 tile, BK = 16, 4x4 per thread.
//   EPI 0: out1 = tanh(acc + bias)                                   first fitting layer (reading R4)
//   EPI 1: out1 = u = tanh(acc + bias); out2 = zin + u               Eq. 3
//   EPI 2: out1 = zin + acc                                          backward through a skip layer
//   EPI 3: out1 = acc                                                dD = G0 W0^T
template <int EPI, bool TRANSB>
__global__ void __launch_bounds__(256)
k_gemm_v0(ChunkView C, int ty, int Ncols, int K, const double *__restrict__ A, int lda, const double *__restrict__ B,
          int ldb, const double *__restrict__ bias, const double *__restrict__ zin, double *__restrict__ out1,
          double *__restrict__ out2, int ldo) {
  __shared__ double As[16][64 + 1], Bs[16][64 + 1];
  const int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  const int m0 = row_lo + blockIdx.x * 64, n0 = blockIdx.y * 64;
  if (m0 >= row_hi) return;
  const int tid = threadIdx.x, tx = tid & 15, tyy = tid >> 4;
  double acc[4][4] = {};
  for (int k0 = 0; k0 < K; k0 += 16) {
    for (int e = tid; e < 64 * 16; e += 256) {
      const int m = e >> 4, k = e & 15;
      As[k][m] = (m0 + m < row_hi && k0 + k < K) ? A[(size_t)(m0 + m) * lda + k0 + k] : 0.0;
    }
    if (TRANSB) {
      for (int e = tid; e < 64 * 16; e += 256) {
        const int n = e >> 4, k = e & 15;
        Bs[k][n] = (n0 + n < Ncols && k0 + k < K) ? B[(size_t)(n0 + n) * ldb + k0 + k] : 0.0;
      }
    } else {
      for (int e = tid; e < 64 * 16; e += 256) {
        const int k = e >> 6, n = e & 63;
        Bs[k][n] = (n0 + n < Ncols && k0 + k < K) ? B[(size_t)(k0 + k) * ldb + n0 + n] : 0.0;
      }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      double av[4], bv[4];
#pragma unroll
      for (int x = 0; x < 4; ++x) { av[x] = As[k][tyy * 4 + x]; bv[x] = Bs[k][tx * 4 + x]; }
#pragma unroll
      for (int x = 0; x < 4; ++x)
#pragma unroll
        for (int y = 0; y < 4; ++y) acc[x][y] += av[x] * bv[y];
    }
    __syncthreads();
  }
#pragma unroll
  for (int x = 0; x < 4; ++x) {
    const int m = m0 + tyy * 4 + x;
    if (m >= row_hi) continue;
#pragma unroll
    for (int y = 0; y < 4; ++y) {
      const int n = n0 + tx * 4 + y;
      if (n >= Ncols) continue;
      const size_t o = (size_t)m * ldo + n;
      if (EPI == 0) {
        out1[o] = tanh(acc[x][y] + bias[n]);
      } else if (EPI == 1) {
        const double u = tanh(acc[x][y] + bias[n]);
        out1[o] = u;
        out2[o] = zin[o] + u;
      } else if (EPI == 2) {
        out1[o] = zin[o] + acc[x][y];
      } else {
        out1[o] = acc[x][y];
      }
    }
  }
}

// E_i = z2 . w3 + b3 (output layer, reading R4); also G2 = w3 (1 - u2^2) and dZ2 = w3 broadcast for the backward.
__global__ void k_fit_out_v0(DevModel P, ChunkView C, int ty, const double *__restrict__ w3, const double *__restrict__ Z2,
                             const double *__restrict__ U2, double *__restrict__ G, double *__restrict__ dZ,
                             double *__restrict__ atom_energy) {
  const int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  const int q = row_lo + blockIdx.x;
  if (q >= row_hi) return;
  __shared__ double part[8];
  double s = 0.0;
  for (int o = threadIdx.x; o < P.fw; o += blockDim.x) {
    const size_t e = (size_t)q * P.fw + o;
    s += Z2[e] * w3[o];
    const double u = U2[e];
    G[e] = w3[o] * (1.0 - u * u);
    dZ[e] = w3[o];
  }
  for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double e = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) e += part[w];
    if (atom_energy) atom_energy[C.s_idx[C.p0 + q]] = e + w3[P.fw];     // b3 follows w3
  }
}

// G = dZ (1 - U^2)
__global__ void k_mul_dtanh_v0(long long n, const double *__restrict__ dZ, const double *__restrict__ U,
                               double *__restrict__ G) {
  long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e < n) {
    const double u = U[e];
    G[e] = dZ[e] * (1.0 - u * u);
  }
}

cudaError_t launch_fit_v0(const DevModel &P, const ChunkView &C, const double *fit, const V0Scratch &S,
                          double *atom_energy, double *dbgD, cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  const int fw = P.fw, dim = P.dim;
  k_descr_v0<<<C.n, 256, 0, st>>>(P, C, S.D, dbgD);
  const int mt = (C.n + 63) / 64;
  const dim3 g_fw(mt, (fw + 63) / 64), g_dim(mt, (dim + 63) / 64);
  const long long nel = (long long)C.n * fw;
  const int eb = (int)((nel + 255) / 256);
  for (int ty = 0; ty < P.ntypes; ++ty) {
    const double *W0 = fit + (size_t)ty * P.fit_net_size;
    const double *b0 = W0 + (size_t)dim * fw, *W1 = b0 + fw, *b1 = W1 + (size_t)fw * fw, *W2 = b1 + fw,
                 *b2 = W2 + (size_t)fw * fw, *w3 = b2 + fw;
    // forward (Eq. 2-3)
    k_gemm_v0<0, false><<<g_fw, 256, 0, st>>>(C, ty, fw, dim, S.D, dim, W0, fw, b0, nullptr, S.Z0, nullptr, fw);
    k_gemm_v0<1, false><<<g_fw, 256, 0, st>>>(C, ty, fw, fw, S.Z0, fw, W1, fw, b1, S.Z0, S.U1, S.Z1, fw);
    k_gemm_v0<1, false><<<g_fw, 256, 0, st>>>(C, ty, fw, fw, S.Z1, fw, W2, fw, b2, S.Z1, S.U2, S.Z2, fw);
    k_fit_out_v0<<<C.n, 64, 0, st>>>(P, C, ty, w3, S.Z2, S.U2, S.G, S.dZ, atom_energy);
    // backward (O9): dZ1 = dZ2 + G2 W2^T; dZ0 = dZ1 + G1 W1^T; dD = G0 W0^T
    k_gemm_v0<2, true><<<g_fw, 256, 0, st>>>(C, ty, fw, fw, S.G, fw, W2, fw, nullptr, S.dZ, S.Z2, nullptr, fw);   // Z2 := dZ1
    k_mul_dtanh_v0<<<eb, 256, 0, st>>>(nel, S.Z2, S.U1, S.G);
    k_gemm_v0<2, true><<<g_fw, 256, 0, st>>>(C, ty, fw, fw, S.G, fw, W1, fw, nullptr, S.Z2, S.dZ, nullptr, fw);   // dZ := dZ0
    k_mul_dtanh_v0<<<eb, 256, 0, st>>>(nel, S.dZ, S.Z0, S.G);
    k_gemm_v0<3, true><<<g_dim, 256, 0, st>>>(C, ty, dim, fw, S.G, fw, W0, fw, nullptr, nullptr, S.dD, nullptr, dim);
  }
  k_dT_v0<<<C.n, 256, 0, st>>>(P, C, S.dD);
  DPB_LAUNCHED(2 + 9 * P.ntypes);
  return cudaGetLastError();
}
