// fit_dmma.cu — variant 1 of S5 (D = T T^<T), S6 (fitting net forward, Eq. 2-3) and S7 (fitting
// backward + dT): six GEMMs per species on fp64 tensor-core tiles (DMMA m8n8k4) with the activation,
// skip and d tanh = 1 - tanh^2 work fused into the epilogues:
//   G1  Z0 = tanh(D W0 + b0)                                   [rows x dim] [dim x w]
//   G2  U1 = tanh(Z0 W1 + b1),  Z1 = Z0 + U1
//   G3  U2 = tanh(Z1 W2 + b2),  Z2 = Z1 + U2,  Q2 = w3 (1 - U2^2)          E_i = Z2 . w3 + b3 (row dot)
//   G4  dZ1 = w3 + Q2 W2^T,     Q1 = dZ1 (1 - U1^2)
//   G5  dZ0 = dZ1 + Q1 W1^T,    Q0 = dZ0 (1 - Z0^2)
//   G6  dD = Q0 W0^T                                           [rows x w] [w x dim]
// Weights are re-laid-out once at model creation: zero-padded to multiples of 16, 16-byte aligned, and the
// transposes are stored explicitly so that every GEMM reads a row-major B.  Rows = the chunk's atoms of one species
// (a contiguous range of sorted positions, read from the device: no host synchronisation).
//
// Kernel: CTA tile 64 rows x (16 NBW) columns, 8 warps as 4 (rows) x 2 (columns), warp tile 16 x (8 NBW): two
// m-blocks share every B fragment, one A fragment feeds NBW n-blocks.  K tiles of 16 through a 3-stage cp.async
// pipeline; shared-memory leading dimensions are 4 (mod 16) doubles, which makes the fragment loads conflict-free.
#include "v1_kernels.cuh"

#include <cooperative_groups.h>
#include <vector>

#define FIT_STAGES 3

struct FitNet {            // device pointers into the padded fitting weights of one species
  const double *W0, *b0, *W1, *b1, *W2, *b2, *w3, *W0T, *W1T, *W2T;
  double b3;
};

struct FitWeights {
  double *buf = nullptr;
  int fwp = 0, dimp = 0;
  std::vector<FitNet> nets;
};

__device__ __forceinline__ void dmma884f(double &c0, double &c1, const double a, const double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc, bool valid) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  const int sz = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gsrc), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

enum { EPI_TANH = 0, EPI_TANH_SKIP = 1, EPI_L3 = 2, EPI_BWD = 3, EPI_STORE = 4, EPI_ATOMIC = 5, EPI_ADD = 6 };

struct GemmArgs {
  const double *A; int lda;          // [rows][lda], K columns used
  const double *B; int ldb;          // [K][ldb] row-major, N columns used
  int K, N;                          // multiples of 16 / 8
  const double *bias;                // [N] or null
  const double *in0; const double *in1; int ldi;
  double *out0; double *out1; int ldo;
};

// WM = warp rows per CTA: CTA tile = 16 WM rows x 16 NBW columns, 64 WM threads.  (2, 15 / 8): the throughput shape;
// (1, 3): 16 x 48 tiles for small systems, where the number of CTAs, not the tile efficiency, bounds the stage.
// FIT_BK = K tile: 16 for the throughput shape; 80 for small systems, where a K = 240 GEMM is then three tiles that are
// all in flight at once (one memory latency instead of fifteen; a ragged last tile is zero-filled).
template <int WM, int NBW, int EPI, int FIT_BK>
__global__ void __launch_bounds__(64 * WM, FIT_BK == 16 ? 2 : 1)
k_fit_gemm(ChunkView C, int ty, GemmArgs g) {
  if (FIT_BK != 16) { pdl_wait(); pdl_trigger(); }          // the small-system instantiations are launched with dpb_launch_pdl
  constexpr int FIT_BM = 16 * WM, FIT_THREADS = 64 * WM, FIT_LDA = FIT_BK + 4;
  constexpr int BN = 16 * NBW, LDB = BN + 4;
  extern __shared__ __align__(16) double smem[];
  double *As = smem;                                        // [STAGES][BM][LDA]
  double *Bs = smem + FIT_STAGES * FIT_BM * FIT_LDA;        // [STAGES][BK][LDB]
  int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  dpb_sub_range(C, row_lo, row_hi);
  const int m0 = row_lo + blockIdx.x * FIT_BM;
  if (m0 >= row_hi) return;
  const int n0 = blockIdx.y * BN;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, gq = lane >> 2, q = lane & 3;
  const int wm = warp >> 1, wn = warp & 1;                  // warp tile: rows 16 wm .., cols 8 NBW wn ..
  // split-K (EPI_ATOMIC, small systems): blockIdx.z takes the K tiles [kt0, kt1) and adds its partial sums to out0
  const int nkt_all = (g.K + FIT_BK - 1) / FIT_BK;
  const int kt0 = (int)(((long long)nkt_all * blockIdx.z) / gridDim.z);
  const int nkt = (int)(((long long)nkt_all * (blockIdx.z + 1)) / gridDim.z) - kt0;

  auto load_tile = [&](int kt, int stage) {
    double *as = As + stage * FIT_BM * FIT_LDA;
    double *bs = Bs + stage * FIT_BK * LDB;
    const int k0 = (kt0 + kt) * FIT_BK;
    for (int c = tid; c < FIT_BM * (FIT_BK / 2); c += FIT_THREADS) {
      const int m = c / (FIT_BK / 2), kk = (c - m * (FIT_BK / 2)) * 2;
      const bool ok = m0 + m < row_hi && k0 + kk < g.K;
      cp_async16(as + m * FIT_LDA + kk, g.A + (size_t)(m0 + m < row_hi ? m0 + m : m0) * g.lda + (ok ? k0 + kk : 0), ok);
    }
    for (int c = tid; c < FIT_BK * (BN / 2); c += FIT_THREADS) {
      const int k = c / (BN / 2), nn = (c - k * (BN / 2)) * 2;
      const bool ok = n0 + nn < g.N && k0 + k < g.K;
      cp_async16(bs + k * LDB + nn, g.B + (size_t)(ok ? k0 + k : 0) * g.ldb + (ok ? n0 + nn : 0), ok);
    }
  };

  double acc[2][NBW][2];
#pragma unroll
  for (int mb = 0; mb < 2; ++mb)
#pragma unroll
    for (int nb = 0; nb < NBW; ++nb) { acc[mb][nb][0] = 0.0; acc[mb][nb][1] = 0.0; }

#pragma unroll
  for (int s = 0; s < FIT_STAGES - 1; ++s) {
    if (s < nkt) load_tile(s, s);
    cp_async_commit();
  }
  for (int kt = 0; kt < nkt; ++kt) {
    cp_async_wait<FIT_STAGES - 2>();
    __syncthreads();
    {
      const int nk = kt + FIT_STAGES - 1;
      if (nk < nkt) load_tile(nk, nk % FIT_STAGES);
      cp_async_commit();
    }
    const double *as = As + (kt % FIT_STAGES) * FIT_BM * FIT_LDA + (16 * wm + gq) * FIT_LDA + q;
    const double *bs = Bs + (kt % FIT_STAGES) * FIT_BK * LDB + q * LDB + 8 * NBW * wn + gq;
#pragma unroll
    for (int ks = 0; ks < FIT_BK / 4; ++ks) {
      const double a0 = as[4 * ks], a1 = as[8 * FIT_LDA + 4 * ks];
#pragma unroll
      for (int nb = 0; nb < NBW; ++nb) {
        const double b = bs[4 * ks * LDB + 8 * nb];
        dmma884f(acc[0][nb][0], acc[0][nb][1], a0, b);
        dmma884f(acc[1][nb][0], acc[1][nb][1], a1, b);
      }
    }
  }
  cp_async_wait<0>();

  // epilogue: thread (gq, q) holds rows 16 wm + gq (+8), columns n0 + 8 NBW wn + 8 nb + 2 q (+1).
  // The element-wise inputs of one m-block are loaded first, all at once (the stores below may alias them as far as
  // the compiler knows, so loads interleaved with stores would serialise NBW global round trips per row).
  const double2 zero2 = make_double2(0.0, 0.0);
#pragma unroll
  for (int mb = 0; mb < 2; ++mb) {
    const int m = m0 + 16 * wm + gq + 8 * mb;
    if (m >= row_hi) continue;
    const int nbase = n0 + 8 * NBW * wn + 2 * q;
    double2 x0[NBW], x1[NBW];
#pragma unroll
    for (int nb = 0; nb < NBW; ++nb) {
      const int n = nbase + 8 * nb;
      const size_t oi = (size_t)m * g.ldi + n;
      x0[nb] = zero2; x1[nb] = zero2;
      if (n < g.N) {
        if (EPI == EPI_TANH_SKIP || EPI == EPI_L3 || EPI == EPI_ADD) x0[nb] = *reinterpret_cast<const double2 *>(g.in0 + oi);
        if (EPI == EPI_BWD) {
          if (g.in0) x0[nb] = *reinterpret_cast<const double2 *>(g.in0 + oi);
          x1[nb] = *reinterpret_cast<const double2 *>(g.in1 + oi);
        }
      }
    }
#pragma unroll
    for (int nb = 0; nb < NBW; ++nb) {
      const int n = nbase + 8 * nb;
      if (n >= g.N) continue;
      double v0 = acc[mb][nb][0], v1 = acc[mb][nb][1];
      const size_t oo = (size_t)m * g.ldo + n;
      if (EPI == EPI_TANH) {
        const double2 b = *reinterpret_cast<const double2 *>(g.bias + n);
        *reinterpret_cast<double2 *>(g.out0 + oo) = make_double2(dp_tanh(v0 + b.x), dp_tanh(v1 + b.y));
      } else if (EPI == EPI_TANH_SKIP) {
        const double2 b = *reinterpret_cast<const double2 *>(g.bias + n);
        const double u0 = dp_tanh(v0 + b.x), u1 = dp_tanh(v1 + b.y);
        *reinterpret_cast<double2 *>(g.out0 + oo) = make_double2(u0, u1);
        *reinterpret_cast<double2 *>(g.out1 + oo) = make_double2(x0[nb].x + u0, x0[nb].y + u1);
      } else if (EPI == EPI_L3) {
        // bias = b2, in1 = w3 (as a [N] vector), in0 = Z1: out1 = Z2 = Z1 + U2, out0 = Q2 = w3 (1 - U2^2)
        const double2 b = *reinterpret_cast<const double2 *>(g.bias + n);
        const double2 w = *reinterpret_cast<const double2 *>(g.in1 + n);
        const double u0 = dp_tanh(v0 + b.x), u1 = dp_tanh(v1 + b.y);
        *reinterpret_cast<double2 *>(g.out1 + oo) = make_double2(x0[nb].x + u0, x0[nb].y + u1);
        *reinterpret_cast<double2 *>(g.out0 + oo) = make_double2(w.x * (1.0 - u0 * u0), w.y * (1.0 - u1 * u1));
      } else if (EPI == EPI_BWD) {
        // dz = acc + bias[n] (w3, first backward step) + in0 (dZ of the next layer); out0 = dz; out1 = dz (1 - in1^2)
        if (g.bias) { const double2 b = *reinterpret_cast<const double2 *>(g.bias + n); v0 += b.x; v1 += b.y; }
        v0 += x0[nb].x; v1 += x0[nb].y;
        const double2 u = x1[nb];
        if (g.out0) *reinterpret_cast<double2 *>(g.out0 + oo) = make_double2(v0, v1);
        *reinterpret_cast<double2 *>(g.out1 + oo) = make_double2(v0 * (1.0 - u.x * u.x), v1 * (1.0 - u.y * u.y));
      } else if (EPI == EPI_ADD) {
        *reinterpret_cast<double2 *>(g.out0 + oo) = make_double2(v0 + x0[nb].x, v1 + x0[nb].y);
      } else if (EPI == EPI_ATOMIC) {
        atomicAdd(g.out0 + oo, v0);
        atomicAdd(g.out0 + oo + 1, v1);
      } else {
        *reinterpret_cast<double2 *>(g.out0 + oo) = make_double2(v0, v1);
      }
    }
  }
}

// S5: D[b][a] = sum_c T[b][c] T[a][c] (Eq. 4; flatten b M^< + a, reading R7), zero-padded to dimp.
__global__ void k_descr_v1(DevModel P, ChunkView C, int ty, int dimp, double *__restrict__ D) {
  pdl_trigger();                                           // (small systems: G1 behind it is launched with dpb_launch_pdl)
  const int q = blockIdx.x;
  {                                                         // one launch per species, on that species' stream
    int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  dpb_sub_range(C, row_lo, row_hi);
    if (q < row_lo || q >= row_hi) return;
  }
  __shared__ double Ts[256 * 5 + 16];            // row stride 5 doubles: the 16 rows a = 0..15 hit 16 distinct bank pairs
  const double *T = C.T + (size_t)q * P.M * 4;
  for (int k = threadIdx.x; k < P.M * 4; k += blockDim.x) Ts[(k >> 2) * 5 + (k & 3)] = T[k];
  __syncthreads();
  for (int e = threadIdx.x; e < dimp; e += blockDim.x) {
    double acc = 0.0;
    if (e < P.dim) {
      const int b = e / P.Ma, a = e - b * P.Ma;
#pragma unroll
      for (int c = 0; c < 4; ++c) acc += Ts[b * 5 + c] * Ts[a * 5 + c];
    }
    D[(size_t)q * dimp + e] = acc;
  }
}

// S7: dT[b][c] = sum_a dD[b][a] T[a][c] + [b < M^<] sum_b' dD[b'][b] T[b'][c].  The second term (M^< x 4 outputs, M terms
// each) is split over all threads in partial sums so that it does not serialise behind M^< x 4 threads.
__global__ void k_dT_v1(DevModel P, ChunkView C, int ty, int dimp, const double *__restrict__ dD) {
  const int q = blockIdx.x;
  {
    int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  dpb_sub_range(C, row_lo, row_hi);
    if (q < row_lo || q >= row_hi) return;                  // (block-uniform: before any barrier)
  }
  extern __shared__ double sm2[];
  double *Ts = sm2;                      // [M][4]
  const int ldr = P.Ma + 1;              // padded row stride: rows b, b + 1, ... fall into different banks
  double *dd = sm2 + P.M * 4;            // [M][Ma + 1]
  double *part = dd + P.M * ldr;         // [nparts][Ma * 4]
  const double *T = C.T + (size_t)q * P.M * 4;
  for (int k = threadIdx.x; k < P.M * 4; k += blockDim.x) Ts[k] = T[k];
  for (int k = threadIdx.x; k < P.dim; k += blockDim.x) dd[(k / P.Ma) * ldr + (k % P.Ma)] = dD[(size_t)q * dimp + k];
  __syncthreads();
  const int nout2 = P.Ma * 4;
  const int nparts = max(1, (int)blockDim.x / nout2);
  for (int idx = threadIdx.x; idx < nparts * nout2; idx += blockDim.x) {
    const int pt = idx / nout2, o = idx - pt * nout2, bcol = o >> 2, c = o & 3;
    const int per = (P.M + nparts - 1) / nparts, lo = pt * per, hi = min(P.M, lo + per);
    double acc = 0.0;
    for (int bp = lo; bp < hi; ++bp) acc += dd[bp * ldr + bcol] * Ts[bp * 4 + c];
    part[idx] = acc;
  }
  __syncthreads();
  for (int e = threadIdx.x; e < P.M * 4; e += blockDim.x) {
    const int b = e >> 2, c = e & 3;
    double acc = 0.0;
    for (int a = 0; a < P.Ma; ++a) acc += dd[b * ldr + a] * Ts[a * 4 + c];
    if (b < P.Ma)
      for (int pt = 0; pt < nparts; ++pt) acc += part[pt * nout2 + e];
    C.dT[dt_offset(P, C, q, b) + c] = acc;
  }
}

// S7 again, the kernel the launcher prefers (M^< in {4, 8, 16}): one WARP per atom, no block barrier, ONE coalesced pass
// over the atom's dD row.  A warp instruction loads 512 contiguous bytes; lane l holds dD[b][a0], dD[b][a0 + 1] with
// b = 32 / LPR * i + l / LPR, a0 = 2 (l mod LPR), LPR = M^< / 2 lanes per row.  First term: partial sum over the lane's
// two a (T[a0], T[a0 + 1] in registers), completed across the row's lanes by shuffles.  Second term: 2 x 4 accumulators
// (a, c) summed over the lane's rows, at the end across the lanes that share a0.  Only T is staged in shared memory.
#define DTV_WARPS 8
template <int LPR>
__global__ void __launch_bounds__(32 * DTV_WARPS) k_dT_v1s(DevModel P, ChunkView C, int ty, int dimp, const double *__restrict__ dD) {
  extern __shared__ double sm2[];
  constexpr int Ma = 2 * LPR, RPI = 32 / LPR;
  pdl_wait();                                               // (small systems launch it with dpb_launch_pdl behind G6)
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q = blockIdx.x * DTV_WARPS + warp;
  if (q >= C.n) return;
  {                                                         // one launch per species, at the tail of that species' chain
    int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  dpb_sub_range(C, row_lo, row_hi);
    if (q < row_lo || q >= row_hi) return;
  }
  const int M = P.M;
  double *Ts = sm2 + (size_t)warp * (M + 2 * Ma) * 4;      // [M][4]
  double *f1 = Ts + 4 * M, *t2 = f1 + 4 * Ma;              // [Ma][4] first term of rows b < M^<; [Ma][4] second term
  const double2 *T = reinterpret_cast<const double2 *>(C.T + (size_t)q * M * 4);
  for (int k = lane; k < 2 * M; k += 32) reinterpret_cast<double2 *>(Ts)[k] = T[k];
  __syncwarp();
  const int a0 = 2 * (lane % LPR), rl = lane / LPR;
  double ta[2][4], c2[2][4];
#pragma unroll
  for (int k = 0; k < 2; ++k)
#pragma unroll
    for (int c = 0; c < 4; ++c) { ta[k][c] = Ts[4 * (a0 + k) + c]; c2[k][c] = 0.0; }
  const double2 *row2 = reinterpret_cast<const double2 *>(dD + (size_t)q * dimp) + lane;
  auto one = [&](int b, const double2 d) {
    double s[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) s[c] = fma(d.x, ta[0][c], d.y * ta[1][c]);
#pragma unroll
    for (int off = 1; off < LPR; off <<= 1)
#pragma unroll
      for (int c = 0; c < 4; ++c) s[c] += __shfl_xor_sync(0xffffffffu, s[c], off);
    if (b < M) {
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const double tb = Ts[4 * b + c];
        c2[0][c] = fma(d.x, tb, c2[0][c]);
        c2[1][c] = fma(d.y, tb, c2[1][c]);
      }
      if (lane % LPR == 0) {
        double2 *o = reinterpret_cast<double2 *>(b < Ma ? f1 + 4 * b : C.dT + dt_offset(P, C, q, b));
        o[0] = make_double2(s[0], s[1]);
        o[1] = make_double2(s[2], s[3]);
      }
    }
  };
  const double2 z2 = make_double2(0.0, 0.0);
  const int NI = (M + RPI - 1) / RPI;                      // the same trip count for every lane: the shuffles are warp-wide
  int i = 0;
  for (; i + 2 <= NI; i += 2) {                            // two loads in flight
    const int b0 = i * RPI + rl, b1 = b0 + RPI;
    const double2 d0 = b0 < M ? row2[(size_t)i * 32] : z2;
    const double2 d1 = b1 < M ? row2[(size_t)(i + 1) * 32] : z2;
    one(b0, d0);
    one(b1, d1);
  }
  if (i < NI) {
    const int b0 = i * RPI + rl;
    one(b0, b0 < M ? row2[(size_t)i * 32] : z2);
  }
#pragma unroll
  for (int off = LPR; off < 32; off <<= 1)
#pragma unroll
    for (int k = 0; k < 2; ++k)
#pragma unroll
      for (int c = 0; c < 4; ++c) c2[k][c] += __shfl_xor_sync(0xffffffffu, c2[k][c], off);
  if (lane < LPR) {
#pragma unroll
    for (int k = 0; k < 2; ++k)
#pragma unroll
      for (int c = 0; c < 4; ++c) t2[4 * (a0 + k) + c] = c2[k][c];
  }
  __syncwarp();
  if (lane < Ma && lane < M) {
    double2 *o = reinterpret_cast<double2 *>(C.dT + dt_offset(P, C, q, lane));
    o[0] = make_double2(f1[4 * lane] + t2[4 * lane], f1[4 * lane + 1] + t2[4 * lane + 1]);
    o[1] = make_double2(f1[4 * lane + 2] + t2[4 * lane + 2], f1[4 * lane + 3] + t2[4 * lane + 3]);
  }
}

// Z0 = tanh(X + b0) in place, after a split-K G1 (small systems): rows of species ty.
__global__ void k_bias_tanh_v1(ChunkView C, int ty, int fwp, const double *__restrict__ bias, double *__restrict__ Z) {
  int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  dpb_sub_range(C, row_lo, row_hi);
  const int q = row_lo + blockIdx.x;
  if (q >= row_hi) return;
  for (int o = threadIdx.x; o < fwp; o += blockDim.x) Z[(size_t)q * fwp + o] = dp_tanh(Z[(size_t)q * fwp + o] + bias[o]);
}

// E_i = Z2 . w3 + b3 (output layer, reading R4): one warp per atom.
__global__ void k_rowdot_v1(ChunkView C, int ty, int fwp, const double *__restrict__ Z2, const double *__restrict__ w3,
                            double b3, double *__restrict__ atom_energy) {
  int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  dpb_sub_range(C, row_lo, row_hi);
  const int q = row_lo + blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (q >= row_hi) return;
  const int lane = threadIdx.x & 31;
  double s = 0.0;
  for (int o = lane; o < fwp; o += 32) s += Z2[(size_t)q * fwp + o] * w3[o];
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  if (lane == 0) atom_energy[C.s_idx[C.p0 + q]] = s + b3;
}

// ---------------------------------------------------------------------------------------------------------
// Small systems (BASELINE.json configs[0]): the middle of the fitting chain — bias + tanh of G1, G2, G3, the E_i row dot,
// G4 and G5 — as ONE kernel on thread-block clusters.  A cluster of fwp / 48 CTAs owns a tile of 16 atoms; CTA r owns the
// columns [48 r, 48 r + 48) of every layer (12 warps = 6 n-blocks x 2 m-blocks: three warps per scheduler) and streams
// only those columns of the four w x w matrices (halves of K through a 3-buffer cp.async pipeline that runs ahead across
// the layers).  A layer's full-width output, the next layer's A operand, is assembled in every CTA's shared memory by
// distributed-shared-memory stores, one cluster barrier per layer; U1, Z1 / dZ1, U2 and Z0 of the own columns stay in
// registers.  Replaces six dependent launches (10-14 us each at 192 atoms, bound by their latency) by one.  E_i is summed
// in a fixed order (lanes, warps, then the cluster's CTAs at rank 0): no reductions.
#define MID_NB 6                                              // n-blocks (8 columns) per CTA
#define MID_WARPS (2 * MID_NB)
#define MID_COLS (8 * MID_NB)
#define MID_LDB (MID_COLS + 4)
#define MID_ZI 5                                              // loads of the Z0 tile per thread (16 x 240 / 2 / 384)

__global__ void __launch_bounds__(32 * MID_WARPS, 1)
k_fit_mid_cluster(ChunkView C, int ty, int fwp, FitNet N, const double *__restrict__ Z0pre, double *__restrict__ Q,
                  double *__restrict__ atom_energy) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  dpb_sub_range(C, row_lo, row_hi);
  pdl_wait();                                                // launched behind the split-K G1 with the programmatic attribute
  pdl_trigger();
  const int m0 = row_lo + blockIdx.y * 16;
  if (m0 >= row_hi) return;                                  // the whole cluster (same blockIdx.y) leaves together
  const int ncl = (int)cluster.num_blocks(), r = (int)cluster.block_rank();
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, g = lane >> 2, q = lane & 3;
  const int nbk = w % MID_NB, row = g + 8 * (w / MID_NB);    // this warp's n-block and m-block: the thread's tile row
  const int lda = fwp + 4, kh = fwp / 2;
  extern __shared__ __align__(16) double smem[];
  double *bufA = smem, *bufB = bufA + 16 * lda;              // full-width activations [16][lda]
  double *Bs = bufB + 16 * lda;                              // 3 x [kh][MID_LDB]: one half (in K) of a matrix' own columns
  double *red = Bs + 3 * kh * MID_LDB;                       // [MID_NB][16] row sums of the warps
  double *clred = red + MID_NB * 16;                         // [8][16] row sums of the cluster's CTAs (used at rank 0)
  const int c0 = MID_COLS * r;                               // first own column

  auto load_half = [&](int h) {                              // h = 2 layer + half; matrices W1, W2, W2^T, W1^T
    if (h < 8) {
      const double *Wm = (h >> 1) == 0 ? N.W1 : (h >> 1) == 1 ? N.W2 : (h >> 1) == 2 ? N.W2T : N.W1T;
      const double *src = Wm + (size_t)(h & 1) * kh * fwp + c0;
      double *dst = Bs + (h % 3) * kh * MID_LDB;
      for (int c = tid; c < kh * (MID_COLS / 2); c += 32 * MID_WARPS) {
        const int k = c / (MID_COLS / 2), nn = (c - k * (MID_COLS / 2)) * 2;
        cp_async16(dst + k * MID_LDB + nn, src + (size_t)k * fwp + nn, true);
      }
    }
    cp_async_commit();
  };
  load_half(0);
  load_half(1);
  // Z0 = tanh(pre-activation + b0), the whole tile in every CTA of the cluster (16 x fwp tanh: cheaper than an exchange);
  // all loads of a thread first, then the arithmetic: one memory latency, not one per element
  {
    const int total = 16 * (fwp / 2);
    double2 v[MID_ZI], b[MID_ZI];
#pragma unroll
    for (int u = 0; u < MID_ZI; ++u) {
      const int c = tid + u * 32 * MID_WARPS;
      const int m = c / (fwp / 2), n = (c - m * (fwp / 2)) * 2;
      v[u] = make_double2(0.0, 0.0); b[u] = v[u];
      if (c < total) {
        b[u] = *reinterpret_cast<const double2 *>(N.b0 + n);
        if (m0 + m < row_hi) v[u] = *reinterpret_cast<const double2 *>(Z0pre + (size_t)(m0 + m) * fwp + n);
      }
    }
#pragma unroll
    for (int u = 0; u < MID_ZI; ++u) {
      const int c = tid + u * 32 * MID_WARPS;
      const int m = c / (fwp / 2), n = (c - m * (fwp / 2)) * 2;
      if (c < total)
        *reinterpret_cast<double2 *>(bufA + m * lda + n) = make_double2(dp_tanh(v[u].x + b[u].x), dp_tanh(v[u].y + b[u].y));
    }
    for (int c = tid + MID_ZI * 32 * MID_WARPS; c < total; c += 32 * MID_WARPS) {      // (wider than 240: not launched)
      const int m = c / (fwp / 2), n = (c - m * (fwp / 2)) * 2;
      double2 x = make_double2(0.0, 0.0);
      if (m0 + m < row_hi) x = *reinterpret_cast<const double2 *>(Z0pre + (size_t)(m0 + m) * fwp + n);
      const double2 bb = *reinterpret_cast<const double2 *>(N.b0 + n);
      *reinterpret_cast<double2 *>(bufA + m * lda + n) = make_double2(dp_tanh(x.x + bb.x), dp_tanh(x.y + bb.y));
    }
  }
  const int col = c0 + 8 * nbk + 2 * q;                      // this thread's columns col, col + 1 of row `row`
  double z0[2], u1[2], z1[2], acc[2][2];                     // [column]; acc: [k parity][column]

  auto gemm_half = [&](const double *A, int h) {             // acc += A[:, half of K] . B half (own columns)
    cp_async_wait<1>();
    __syncthreads();                                         // half h has landed; everyone is done with buffer (h + 2) % 3
    load_half(h + 2);
    const double *as = A + row * lda + (h & 1) * kh + q;
    const double *bs = Bs + (h % 3) * kh * MID_LDB + q * MID_LDB + 8 * nbk + g;
#pragma unroll 5
    for (int ks = 0; ks < kh / 4; ks += 2) {                 // kh / 4 is even: two independent accumulator sets
      dmma884f(acc[0][0], acc[0][1], as[4 * ks], bs[4 * ks * MID_LDB]);
      dmma884f(acc[1][0], acc[1][1], as[4 * ks + 4], bs[4 * (ks + 1) * MID_LDB]);
    }
  };
  auto clear_acc = [&]() { acc[0][0] = 0.0; acc[0][1] = 0.0; acc[1][0] = 0.0; acc[1][1] = 0.0; };
  auto broadcast = [&](double *buf, const double (&v)[2]) {  // own columns of a full-width tile, into every CTA
    for (int rr = 0; rr < ncl; ++rr)
      *reinterpret_cast<double2 *>(cluster.map_shared_rank(buf, rr) + row * lda + col) = make_double2(v[0], v[1]);
  };

  // G2: U1 = tanh(Z0 W1 + b1), Z1 = Z0 + U1
  clear_acc();
  gemm_half(bufA, 0);                                        // (its barrier also publishes the Z0 tile)
  z0[0] = bufA[row * lda + col]; z0[1] = bufA[row * lda + col + 1];
  gemm_half(bufA, 1);
  {
    const double2 b = *reinterpret_cast<const double2 *>(N.b1 + col);
    u1[0] = dp_tanh(acc[0][0] + acc[1][0] + b.x);
    u1[1] = dp_tanh(acc[0][1] + acc[1][1] + b.y);
    z1[0] = z0[0] + u1[0];
    z1[1] = z0[1] + u1[1];
    broadcast(bufB, z1);
  }
  cluster.sync();
  // G3: U2 = tanh(Z1 W2 + b2), Z2 = Z1 + U2, E_i = Z2 . w3 + b3, Q2 = w3 (1 - U2^2)
  const double2 w3 = *reinterpret_cast<const double2 *>(N.w3 + col);
  clear_acc();
  gemm_half(bufB, 2);
  gemm_half(bufB, 3);
  {
    const double2 b = *reinterpret_cast<const double2 *>(N.b2 + col);
    const double ua = dp_tanh(acc[0][0] + acc[1][0] + b.x), ub = dp_tanh(acc[0][1] + acc[1][1] + b.y);
    double es = fma(z1[0] + ua, w3.x, (z1[1] + ub) * w3.y);
    const double q2[2] = {w3.x * (1.0 - ua * ua), w3.y * (1.0 - ub * ub)};
    es += __shfl_xor_sync(0xffffffffu, es, 1);
    es += __shfl_xor_sync(0xffffffffu, es, 2);
    if (q == 0) red[nbk * 16 + row] = es;
    broadcast(bufA, q2);
    __syncthreads();
    if (tid < 16) {
      double s = 0.0;
#pragma unroll
      for (int nb = 0; nb < MID_NB; ++nb) s += red[nb * 16 + tid];
      cluster.map_shared_rank(clred, 0)[r * 16 + tid] = s;
    }
  }
  cluster.sync();
  if (r == 0 && tid < 16 && m0 + tid < row_hi) {
    double s = N.b3;
    for (int rr = 0; rr < ncl; ++rr) s += clred[rr * 16 + tid];
    atom_energy[C.s_idx[C.p0 + m0 + tid]] = s;
  }
  // G4: dZ1 = w3 + Q2 W2^T, Q1 = dZ1 (1 - U1^2)
  clear_acc();
  gemm_half(bufA, 4);
  gemm_half(bufA, 5);
  {
    z1[0] = w3.x + acc[0][0] + acc[1][0];                    // dZ1
    z1[1] = w3.y + acc[0][1] + acc[1][1];
    const double q1[2] = {z1[0] * (1.0 - u1[0] * u1[0]), z1[1] * (1.0 - u1[1] * u1[1])};
    broadcast(bufB, q1);
  }
  cluster.sync();
  // G5: dZ0 = dZ1 + Q1 W1^T, Q0 = dZ0 (1 - Z0^2): the A operand of G6
  clear_acc();
  gemm_half(bufB, 6);
  gemm_half(bufB, 7);
  if (m0 + row < row_hi) {
    const double da = z1[0] + acc[0][0] + acc[1][0], db = z1[1] + acc[0][1] + acc[1][1];
    *reinterpret_cast<double2 *>(Q + (size_t)(m0 + row) * fwp + col) =
        make_double2(da * (1.0 - z0[0] * z0[0]), db * (1.0 - z0[1] * z0[1]));
  }
  cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------------------
static int round_up(int x, int m) { return (x + m - 1) / m * m; }

// The padded fitting weights hang off V1Weights::fit (opaque pointer declared in v1_kernels.cuh).
cudaError_t v1_prepare_fit(const DevModel &P, const double *fit_h, V1Weights &W) {
  FitWeights *F = new FitWeights();
  const int fw = P.fw, dim = P.dim, fwp = round_up(fw, 16), dimp = round_up(dim, 16);
  F->fwp = fwp; F->dimp = dimp;
  const size_t per = (size_t)dimp * fwp * 2 + (size_t)fwp * fwp * 4 + 4 * (size_t)fwp;
  std::vector<double> h(per * P.ntypes, 0.0);
  std::vector<size_t> off;
  for (int ty = 0; ty < P.ntypes; ++ty) {
    const double *W0 = fit_h + (size_t)ty * P.fit_net_size;
    const double *b0 = W0 + (size_t)dim * fw, *W1 = b0 + fw, *b1 = W1 + (size_t)fw * fw, *W2 = b1 + fw,
                 *b2 = W2 + (size_t)fw * fw, *w3 = b2 + fw;
    double *base = h.data() + per * ty;
    double *pW0 = base, *pW0T = pW0 + (size_t)dimp * fwp, *pW1 = pW0T + (size_t)dimp * fwp,
           *pW1T = pW1 + (size_t)fwp * fwp, *pW2 = pW1T + (size_t)fwp * fwp, *pW2T = pW2 + (size_t)fwp * fwp,
           *pb0 = pW2T + (size_t)fwp * fwp, *pb1 = pb0 + fwp, *pb2 = pb1 + fwp, *pw3 = pb2 + fwp;
    for (int d = 0; d < dim; ++d)
      for (int o = 0; o < fw; ++o) {
        pW0[(size_t)d * fwp + o] = W0[(size_t)d * fw + o];
        pW0T[(size_t)o * dimp + d] = W0[(size_t)d * fw + o];
      }
    for (int a = 0; a < fw; ++a)
      for (int o = 0; o < fw; ++o) {
        pW1[(size_t)a * fwp + o] = W1[(size_t)a * fw + o];
        pW1T[(size_t)o * fwp + a] = W1[(size_t)a * fw + o];
        pW2[(size_t)a * fwp + o] = W2[(size_t)a * fw + o];
        pW2T[(size_t)o * fwp + a] = W2[(size_t)a * fw + o];
      }
    for (int o = 0; o < fw; ++o) { pb0[o] = b0[o]; pb1[o] = b1[o]; pb2[o] = b2[o]; pw3[o] = w3[o]; }
  }
  cudaError_t e = cudaMalloc(&F->buf, sizeof(double) * h.size());
  if (e != cudaSuccess) { delete F; return e; }
  e = cudaMemcpy(F->buf, h.data(), sizeof(double) * h.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { cudaFree(F->buf); delete F; return e; }
  for (int ty = 0; ty < P.ntypes; ++ty) {
    const double *base = F->buf + per * ty;
    FitNet n;
    n.W0 = base; n.W0T = n.W0 + (size_t)dimp * fwp; n.W1 = n.W0T + (size_t)dimp * fwp;
    n.W1T = n.W1 + (size_t)fwp * fwp; n.W2 = n.W1T + (size_t)fwp * fwp; n.W2T = n.W2 + (size_t)fwp * fwp;
    n.b0 = n.W2T + (size_t)fwp * fwp; n.b1 = n.b0 + fwp; n.b2 = n.b1 + fwp; n.w3 = n.b2 + fwp;
    n.b3 = fit_h[(size_t)ty * P.fit_net_size + P.fit_net_size - 1];
    F->nets.push_back(n);
  }
  W.fit = F;
  return cudaSuccess;
}

void v1_release_fit(V1Weights &W) {
  FitWeights *F = reinterpret_cast<FitWeights *>(W.fit);
  if (F) {
    if (F->buf) cudaFree(F->buf);
    delete F;
  }
  W.fit = nullptr;
}

size_t v1_workspace_bytes(const DevModel &P, int64_t chunk) {
  const size_t fwp = round_up(P.fw, 16), dimp = round_up(P.dim, 16);
  return sizeof(double) * (size_t)chunk * (2 * dimp + 6 * fwp) + 256;
}

template <int WM, int NBW, int EPI, int FIT_BK = 16>
static cudaError_t gemm_t(const ChunkView &C, int ty, const GemmArgs &g, cudaStream_t st, int splitk = 1) {
  constexpr int BN = 16 * NBW, FIT_BM = 16 * WM;
  const size_t smem = sizeof(double) * FIT_STAGES * (FIT_BM * (FIT_BK + 4) + FIT_BK * (BN + 4));
  static bool configured_d[DPB_MAX_DEVICES] = {};
  bool &configured = configured_d[dpb_device()];
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_fit_gemm<WM, NBW, EPI, FIT_BK>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid((C.n + FIT_BM - 1) / FIT_BM, (g.N + BN - 1) / BN, splitk);
  if (FIT_BK != 16) {
    cudaError_t el = dpb_launch_pdl(k_fit_gemm<WM, NBW, EPI, FIT_BK>, grid, dim3(64 * WM), smem, st, true, C, ty, g);
    if (el != cudaSuccess) return el;
  } else
  k_fit_gemm<WM, NBW, EPI, FIT_BK><<<grid, 64 * WM, smem, st>>>(C, ty, g);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

// Small systems (a chunk of at most FIT_SMALL_N atoms: BASELINE.json configs[0], 192 atoms) are bound by how many CTAs a
// GEMM offers, not by tile efficiency: 16 x 48 tiles give 5 (240 columns) or 34 (1600) CTAs per 16 rows.
#define FIT_SMALL_N 2048
template <int NBW, int EPI>
static cudaError_t gemm(const ChunkView &C, int ty, const GemmArgs &g, cudaStream_t st) {
  if (C.n <= FIT_SMALL_N) return gemm_t<1, 3, EPI, 80>(C, ty, g, st);
  return gemm_t<2, NBW, EPI>(C, ty, g, st);
}

// Plain GEMM on the same tiles for the strawman pipeline (strawman.cu): C[rows x N] = A[rows x K] B[K x N] (+ Cin).
// K and N even, lda / ldb / ldc even (16-byte rows); `range` = device int[2] {0, INT_MAX} (the kernel's row-range hook).
cudaError_t v1_plain_gemm(int64_t rows, const double *A, int lda, const double *B, int ldb, int K, int N,
                          const double *Cin, double *Cout, int ldc, const int *range, cudaStream_t st) {
  if (rows <= 0) return cudaSuccess;
  ChunkView C{};
  C.p0 = 0; C.n = (int)rows; C.type_start = range; C.sub_part = 0; C.sub_nparts = 1;
  GemmArgs g{A, lda, B, ldb, K, N, nullptr, Cin, nullptr, ldc, Cout, nullptr, ldc};
  if (N <= 32) return Cin ? gemm_t<2, 2, EPI_ADD>(C, 0, g, st) : gemm_t<2, 2, EPI_STORE>(C, 0, g, st);
  if (N <= 64) return Cin ? gemm_t<2, 4, EPI_ADD>(C, 0, g, st) : gemm_t<2, 4, EPI_STORE>(C, 0, g, st);
  if (N <= 112) return Cin ? gemm_t<2, 7, EPI_ADD>(C, 0, g, st) : gemm_t<2, 7, EPI_STORE>(C, 0, g, st);
  return Cin ? gemm_t<2, 8, EPI_ADD>(C, 0, g, st) : gemm_t<2, 8, EPI_STORE>(C, 0, g, st);
}

// The buffer of the first layer's pre-activations (split-K sums) inside the workspace of a chunk of n atoms, and its
// row length: what a caller clears on the side instead of the memset below (ChunkView::prezero).
double *v1_fit_preact(const V1Weights &W, void *ws, int64_t n, int *row_len) {
  const FitWeights *F = reinterpret_cast<const FitWeights *>(W.fit);
  if (!F || !ws) return nullptr;
  *row_len = F->fwp;
  return reinterpret_cast<double *>(ws) + 2 * (size_t)n * F->dimp;
}

cudaError_t v1_fit(const DevModel &P, const ChunkView &Cin, const V1Weights &W, const double *fit, void *ws,
                   double *atom_energy, cudaStream_t st) {
  (void)fit;
  const ChunkView &C = Cin;
  if (C.n <= 0) return cudaSuccess;
  const FitWeights *F = reinterpret_cast<const FitWeights *>(W.fit);
  if (!F) return cudaErrorNotSupported;
  const int fwp = F->fwp, dimp = F->dimp;
  const size_t n = (size_t)C.n;
  double *p = reinterpret_cast<double *>(ws);
  double *D = p; p += n * dimp;          // later reused as dD's input? no: dD has its own buffer
  double *dD = p; p += n * dimp;
  double *Z0 = p; p += n * fwp;
  double *U1 = p; p += n * fwp;
  double *Z1 = p; p += n * fwp;          // later dZ1
  double *Z2 = p; p += n * fwp;
  double *Q = p; p += n * fwp;           // Q2, then Q1 (ping-pong with Q')
  double *Q2 = p;                        // second Q buffer
  cudaError_t e;

  const bool splitk = C.n <= FIT_SMALL_N && !C.fslot;    // (not in deterministic mode: the partial sums are reductions)
  // small systems: the middle of the chain as one cluster kernel when the width is a multiple of 48 (clusters of <= 8 CTAs)
  const size_t smem_mid = sizeof(double) * (2 * 16 * (size_t)(fwp + 4) + 3 * (size_t)(fwp / 2) * MID_LDB + 16 * (MID_NB + 8));
  bool mid = splitk && fwp % MID_COLS == 0 && fwp / MID_COLS <= 8 && smem_mid <= 227 * 1024;
  if (mid) {
    // once per device and width: the shared-memory limit, and whether a cluster of this size can be resident at all (a
    // device or partition where it cannot falls back to the separate launches)
    static int mid_state_d[DPB_MAX_DEVICES] = {}, mid_fwp_d[DPB_MAX_DEVICES] = {};
    int &mid_state = mid_state_d[dpb_device()], &mid_fwp = mid_fwp_d[dpb_device()];
    if (mid_state == 0 || mid_fwp != fwp) {
      mid_fwp = fwp;
      mid_state = -1;
      if (cudaFuncSetAttribute(k_fit_mid_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(227 * 1024)) ==
          cudaSuccess) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(fwp / MID_COLS), 1, 1);
        cfg.blockDim = dim3(32 * MID_WARPS, 1, 1);
        cfg.dynamicSmemBytes = smem_mid;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)(fwp / MID_COLS); at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int nclusters = 0;
        if (cudaOccupancyMaxActiveClusters(&nclusters, k_fit_mid_cluster, &cfg) == cudaSuccess && nclusters > 0) mid_state = 1;
      }
      if (mid_state < 0) cudaGetLastError();
    }
    mid = mid_state > 0;
  }
  if (splitk && !C.prezero && (e = cudaMemsetAsync(Z0, 0, sizeof(double) * n * fwp, st)) != cudaSuccess) return e;
  // per-type chains on forked streams (common.cuh); their rows, hence every buffer row they touch, are disjoint.  The
  // descriptor and dT kernels (memory-bound) belong to the chains: one species' run beside the other's GEMMs
  const size_t sm = sizeof(double) * ((size_t)P.M * 4 + (size_t)P.M * (P.Ma + 1) + 256 + 4 * P.Ma);
  static size_t configured_d[DPB_MAX_DEVICES] = {};
  size_t &configured = configured_d[dpb_device()];
  if (sm > 48 * 1024 && sm > configured) {
    e = cudaFuncSetAttribute(k_dT_v1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    configured = sm;
  }
  const size_t sms = sizeof(double) * DTV_WARPS * 4 * ((size_t)P.M + 2 * P.Ma);
  const unsigned nbs = (unsigned)((C.n + DTV_WARPS - 1) / DTV_WARPS);
  // A single-species system has no second chain to overlap with: its rows are split into two parts that run as two chains
  // on forked streams (the memory-bound descriptor / dT kernels and the GEMM tails of one beside the GEMMs of the other:
  // Cu32k fitting 3.52 -> 3.30 ms).  With two species the chains already overlap; splitting them further was measured
  // and is slower (W24k 2.12 -> 2.17 ms in 2 parts, 2.28 in 4).
  const int split = P.ntypes == 1 && C.n >= 4096 ? 2 : 1;
  const int nbatch = P.ntypes * split;
  cudaStream_t ts[DPB_MAX_TYPES];
  const bool typed = C.typed_pipe && split == 1 && !splitk;   // species pipeline: pass 1 left the streams forked
  if ((e = typed ? dpb_forked_streams(nbatch, st, ts) : dpb_fork_streams(nbatch, st, ts)) != cudaSuccess) return e;
  for (int k = 0; k < nbatch; ++k) {
    const int ty = P.ntypes - 1 - k / split, part = k % split;
    cudaStream_t s = ts[k];
    const FitNet &N = F->nets[ty];
    GemmArgs g;
    ChunkView C = Cin;
    C.sub_part = part; C.sub_nparts = split;
    k_descr_v1<<<C.n, 256, 0, s>>>(P, C, ty, dimp, D);
    DPB_LAUNCHED(1);
    // G1: Z0 = tanh(D W0 + b0).  Small systems: split-K over 8 CTAs (K = dim is a serial loop of dim / 16 tiles for
    // the few CTAs a 192-atom box offers), partial sums added into the cleared Z0, bias and tanh in a second kernel.
    g = GemmArgs{D, dimp, N.W0, fwp, dimp, fwp, N.b0, nullptr, nullptr, fwp, Z0, nullptr, fwp};
    if (splitk && mid) {
      // bias + tanh of G1, G2, G3, E_i, G4, G5 in one cluster kernel (k_fit_mid_cluster): Z0 holds the pre-activation sums
      if ((e = gemm_t<1, 3, EPI_ATOMIC, 80>(C, ty, g, s, 8)) != cudaSuccess) return e;
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)(fwp / MID_COLS), (unsigned)((C.n + 15) / 16), 1);
      cfg.blockDim = dim3(32 * MID_WARPS, 1, 1);
      cfg.dynamicSmemBytes = smem_mid;
      cfg.stream = s;
      cudaLaunchAttribute at[2];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = (unsigned)(fwp / MID_COLS); at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
      at[1].val.programmaticStreamSerializationAllowed = 1;
      cfg.attrs = at; cfg.numAttrs = 2;
      if ((e = cudaLaunchKernelEx(&cfg, k_fit_mid_cluster, C, ty, fwp, N, (const double *)Z0, Q, atom_energy)) != cudaSuccess)
        return e;
      DPB_LAUNCHED(1);
    } else {
    if (splitk) {
      if ((e = gemm_t<1, 3, EPI_ATOMIC, 80>(C, ty, g, s, 8)) != cudaSuccess) return e;
      k_bias_tanh_v1<<<C.n, 64, 0, s>>>(C, ty, fwp, N.b0, Z0);
      DPB_LAUNCHED(1);
    } else if ((e = gemm<15, EPI_TANH>(C, ty, g, s)) != cudaSuccess) return e;
    // G2: U1 = tanh(Z0 W1 + b1); Z1 = Z0 + U1
    g = GemmArgs{Z0, fwp, N.W1, fwp, fwp, fwp, N.b1, Z0, nullptr, fwp, U1, Z1, fwp};
    if ((e = gemm<15, EPI_TANH_SKIP>(C, ty, g, s)) != cudaSuccess) return e;
    // G3: U2 = tanh(Z1 W2 + b2); Z2 = Z1 + U2; Q = w3 (1 - U2^2)
    g = GemmArgs{Z1, fwp, N.W2, fwp, fwp, fwp, N.b2, Z1, N.w3, fwp, Q, Z2, fwp};
    if ((e = gemm<15, EPI_L3>(C, ty, g, s)) != cudaSuccess) return e;
    k_rowdot_v1<<<(C.n + 7) / 8, 256, 0, s>>>(C, ty, fwp, Z2, N.w3, N.b3, atom_energy);
    DPB_LAUNCHED(1);
    // G4: dZ1 = w3 + Q W2^T (-> Z1 buffer); Q' = dZ1 (1 - U1^2)
    g = GemmArgs{Q, fwp, N.W2T, fwp, fwp, fwp, N.w3, nullptr, U1, fwp, Z1, Q2, fwp};
    if ((e = gemm<15, EPI_BWD>(C, ty, g, s)) != cudaSuccess) return e;
    // G5: dZ0 = dZ1 + Q' W1^T; Q = dZ0 (1 - Z0^2)
    g = GemmArgs{Q2, fwp, N.W1T, fwp, fwp, fwp, nullptr, Z1, Z0, fwp, nullptr, Q, fwp};
    if ((e = gemm<15, EPI_BWD>(C, ty, g, s)) != cudaSuccess) return e;
    }
    // G6: dD = Q W0^T
    g = GemmArgs{Q, fwp, N.W0T, dimp, fwp, dimp, nullptr, nullptr, nullptr, dimp, dD, nullptr, dimp};
    if ((e = gemm<8, EPI_STORE>(C, ty, g, s)) != cudaSuccess) return e;
    if (P.Ma == 16 && sms <= 48 * 1024 && C.n <= FIT_SMALL_N) {
      if ((e = dpb_launch_pdl(k_dT_v1s<8>, dim3(nbs), dim3(32 * DTV_WARPS), sms, s, true, P, C, ty, dimp, (const double *)dD)) !=
          cudaSuccess)
        return e;
    } else if (P.Ma == 16 && sms <= 48 * 1024) k_dT_v1s<8><<<nbs, 32 * DTV_WARPS, sms, s>>>(P, C, ty, dimp, dD);
    else if (P.Ma == 8 && sms <= 48 * 1024) k_dT_v1s<4><<<nbs, 32 * DTV_WARPS, sms, s>>>(P, C, ty, dimp, dD);
    else if (P.Ma == 4 && sms <= 48 * 1024) k_dT_v1s<2><<<nbs, 32 * DTV_WARPS, sms, s>>>(P, C, ty, dimp, dD);
    else k_dT_v1<<<C.n, 256, sm, s>>>(P, C, ty, dimp, dD);
    DPB_LAUNCHED(1);
  }
  if (!typed && (e = dpb_join_streams(nbatch, st, ts)) != cudaSuccess) return e;
  return cudaGetLastError();
}
