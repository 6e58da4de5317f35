// fit_tc.cu — mixed-precision (DPB_TF32) S5 (D = T T^<T), S6 (fitting net forward, Eq. 2-3) and S7
// (fitting backward + dT) on the 5th-generation tensor cores.  Same six GEMMs as fit_dmma.cu:
//   G1  Z0 = tanh(D W0 + b0)                    G4  dZ1 = w3 + Q2 W2^T,  Q1 = dZ1 S1,  S1 = 1 - U1^2
//   G2  U1 = tanh(Z0 W1 + b1), Z1 = Z0 + U1     G5  dZ0 = dZ1 + Q1 W1^T, Q0 = dZ0 S0,  S0 = 1 - Z0^2
//   G3  U2 = tanh(Z1 W2 + b2), E_i = (Z1 + U2) . w3 + b3,  Q2 = w3 (1 - U2^2)
//   G6  dD = Q0 W0^T
// each as tcgen05.mma kind::tf32 with the 3xTF32 operand split (tc_common.cuh) and fp32 accumulators in TMEM.
//
// Operand format ("images"): every GEMM operand lives in HBM as the exact shared-memory image the MMA reads:
// K-major, 128-byte swizzle, panels of 32 K-columns; hi and lo parts in separate arrays.  An A image is
// [row tile of 128][K panel][128 rows x 128 B]; a B image is [N tile][K panel][NT rows x 128 B].  A stage of the
// pipeline is therefore four contiguous bulk copies (cp.async.bulk, the TMA engine without a tensor map).  The
// epilogue of one GEMM writes the A image of the next (thread r of the epilogue warpgroup owns tile row r = TMEM lane
// r), plus the plain fp32 rows the later element-wise steps need.
//
// Kernel: one CTA per (row tile, N tile); warp 0 = bulk-copy producer, warp 1 = MMA issuer, warps 2-9 = two epilogue
// warpgroups (half of the N tile each).
#include <vector>

#include "tc_common.cuh"
#include "tc_kernels.cuh"

#define FT_APANEL (128 * 128)          // bytes of one A panel: 128 rows x 128 B (32 TF32 or 64 BF16 K-columns per row)

// Operand format of the GEMMs (tc_fit's `opf`).  An operand x is stored as NP pieces whose sum is x to fp32 accuracy; the
// product a b is the sum of the listed piece products (error-compensated split; the dropped products are below fp32's
// rounding):
//   0  3xTF32 (DPB_TF32):       x = hi + lo in TF32;       lo hi + hi lo + hi hi                  kind::tf32, K = 8 per MMA
//   1  BF16 x 6 (DPB_BF16):     x = p0 + p1 + p2 in BF16;  p2 p0 + p0 p2 + p1 p1 + p1 p0 + p0 p1 + p0 p0   kind::f16, K = 16
//   2  plain BF16 (DPB_BF16_PLAIN): x ~ p0;                p0 p0      (measured, not meant to meet the tolerance)
// KP = K columns per 128-byte panel row; CP = panels per accumulation chunk (K = 64, see FT_CP below).
template <int OPF> struct OpFmt;
template <> struct OpFmt<0> { static constexpr int NP = 2, KP = 32, CP = 2; };
template <> struct OpFmt<1> { static constexpr int NP = 3, KP = 64, CP = 1; };
template <> struct OpFmt<2> { static constexpr int NP = 1, KP = 64, CP = 1; };
static int opf_np(int opf) { return opf == 0 ? 2 : (opf == 1 ? 3 : 1); }
static int opf_kp(int opf) { return opf == 0 ? 32 : 64; }

enum { FE_TANH = 0, FE_TANH_SKIP = 1, FE_L3 = 2, FE_BWD1 = 3, FE_BWD0 = 4, FE_STORE = 5 };

struct FitTCNet {                      // device pointers of one species: B images per piece, fp32 vectors
  const uint8_t *W0[3], *W1[3], *W2[3], *W2T[3], *W1T[3], *W0T[3];
  const float *b0, *b1, *b2, *w3;
  float b3;
};

struct FitTC {
  uint8_t *buf = nullptr;
  int opf = 0;
  int fw = 0, fwp = 0, NT = 0;         // width, width padded to the K panel, N tile of the fw-wide GEMMs
  int dim = 0, dimp = 0, NT6 = 0;      // descriptor size, padded to the N tile of G6 (240: fewer re-reads of A than 128)
  std::vector<FitTCNet> nets;
};

struct FitTCArgs {
  const uint8_t *A[3];                 // A images per piece: [tile][KPAN][FT_APANEL bytes]
  const uint8_t *B[3];                 // B images per piece: [ntile][KPAN][NT * 128 bytes]
  int KPAN;                            // K panels
  int N;                               // real output columns (<= gridDim.y * NT)
  int KPAN_out;                        // K panels of the output image (its K = this GEMM's N)
  const float *bias, *w3;              // [N]
  const float *in0, *in1;              // plain fp32 [rows][ldp]
  float *out_plain0, *out_plain1;      // plain fp32 [rows][ldp]
  uint8_t *out[3];                     // output A image per piece, or out[0] == null
  int ldp;
  float b3;
  double *atom_energy;                 // FE_L3
  const int *s_idx;
};

// store 4 consecutive columns n0 .. n0 + 3 of row r into an A image in global memory (all pieces)
template <int OPF>
__device__ __forceinline__ void img_store4(uint8_t *const img[3], size_t tile, int kpan, int n0, int r, float v0,
                                           float v1, float v2, float v3) {
  constexpr int KP = OpFmt<OPF>::KP;
  const size_t pan = (tile * kpan + (size_t)(n0 / KP)) * FT_APANEL;
  if (OPF == 0) {
    float4 h, l;
    tc::split_tf32(v0, h.x, l.x);
    tc::split_tf32(v1, h.y, l.y);
    tc::split_tf32(v2, h.z, l.z);
    tc::split_tf32(v3, h.w, l.w);
    const size_t o = pan + tc::sw128_offset(r, n0 & 31);
    *reinterpret_cast<float4 *>(img[0] + o) = h;
    *reinterpret_cast<float4 *>(img[1] + o) = l;
  } else {
    uint32_t p[4][3];
    const float v[4] = {v0, v1, v2, v3};
#pragma unroll
    for (int i = 0; i < 4; ++i) tc::split_bf16x3(v[i], p[i][0], p[i][1], p[i][2]);
    const size_t o = pan + tc::sw128_offset_b16(r, n0 & 63);
#pragma unroll
    for (int q = 0; q < OpFmt<OPF>::NP; ++q)
      *reinterpret_cast<uint2 *>(img[q] + o) = make_uint2(p[0][q] | (p[1][q] << 16), p[2][q] | (p[3][q] << 16));
  }
}

// One group of 8 output columns of row m (tile row r): apply the GEMM's epilogue to the accumulators a[8].
// The plain fp32 activation arrays (Z0, S0, S1, Z1, dZ1) are private to these epilogues, which all map thread r to tile
// row r; they are stored tile-wise transposed, [tile][column / 4][row][4], so that the 32 lanes of a warp (32 rows) touch
// 512 contiguous bytes per access instead of 32 separate lines.  dD (FE_STORE) stays row-major for k_dT_tc.
template <int EPI, int OPF>
__device__ __forceinline__ void ft_epi8(const float a[8], int nn0, const FitTCArgs &g, size_t tile, int r, int m,
                                        double &edot) {
  float o0[8], o1[8];
#pragma unroll
  for (int q4 = 0; q4 < 2; ++q4) {
    const int nn = nn0 + 4 * q4;
    const bool live = nn < g.N;
    float4 bias = make_float4(0.f, 0.f, 0.f, 0.f), w3 = bias, i0 = bias, i1 = bias;
    const size_t pt = ((tile * (size_t)(g.ldp >> 2) + (size_t)(nn >> 2)) * 128 + (size_t)r) * 4;   // tiled offset
    if (live) {
      if (EPI == FE_TANH || EPI == FE_TANH_SKIP || EPI == FE_L3) bias = *reinterpret_cast<const float4 *>(g.bias + nn);
      if (EPI == FE_L3 || EPI == FE_BWD1) w3 = *reinterpret_cast<const float4 *>(g.w3 + nn);
      if (EPI == FE_TANH_SKIP || EPI == FE_L3 || EPI == FE_BWD0)
        i0 = *reinterpret_cast<const float4 *>(g.in0 + pt);
      if (EPI == FE_BWD1 || EPI == FE_BWD0) i1 = *reinterpret_cast<const float4 *>(g.in1 + pt);
    }
    const float bb[4] = {bias.x, bias.y, bias.z, bias.w}, ww[4] = {w3.x, w3.y, w3.z, w3.w};
    const float x0[4] = {i0.x, i0.y, i0.z, i0.w}, x1[4] = {i1.x, i1.y, i1.z, i1.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float av = a[4 * q4 + i];
      float p = 0.f, q = 0.f;                              // p -> image / plain0, q -> plain1
      if (live) {
        if (EPI == FE_TANH) {
          tc::tanh_d_f32(av + bb[i], p, q);                                // Z0 and S0 = 1 - Z0^2
        } else if (EPI == FE_TANH_SKIP) {
          float u;
          tc::tanh_d_f32(av + bb[i], u, q);                                // U1 and S1 = 1 - U1^2
          p = x0[i] + u;                                                   // Z1 = Z0 + U1
        } else if (EPI == FE_L3) {
          float u, s2;
          tc::tanh_d_f32(av + bb[i], u, s2);                               // U2 and 1 - U2^2
          edot = fma((double)(x0[i] + u), (double)ww[i], edot);            // E_i += Z2 w3
          p = ww[i] * s2;                                                  // Q2 = w3 (1 - U2^2)
        } else if (EPI == FE_BWD1) {
          q = ww[i] + av;                                                  // dZ1 = w3 + Q2 W2^T
          p = q * x1[i];                                                   // Q1 = dZ1 S1
        } else if (EPI == FE_BWD0) {
          const float dz = x0[i] + av;                                     // dZ0 = dZ1 + Q1 W1^T
          p = dz * x1[i];                                                  // Q0 = dZ0 S0
        } else {
          p = av;                                                          // dD
        }
      }
      o0[4 * q4 + i] = p;
      o1[4 * q4 + i] = q;
    }
  }
#pragma unroll
  for (int q4 = 0; q4 < 2; ++q4) {
    const int nn = nn0 + 4 * q4;
    if (g.out[0] && nn < g.KPAN_out * OpFmt<OPF>::KP)
      img_store4<OPF>(g.out, tile, g.KPAN_out, nn, r, o0[4 * q4], o0[4 * q4 + 1], o0[4 * q4 + 2], o0[4 * q4 + 3]);
    if (nn < g.ldp) {
      const size_t po = EPI == FE_STORE ? (size_t)m * g.ldp + nn
                                        : ((tile * (size_t)(g.ldp >> 2) + (size_t)(nn >> 2)) * 128 + (size_t)r) * 4;
      if (g.out_plain0)
        *reinterpret_cast<float4 *>(g.out_plain0 + po) = make_float4(o0[4 * q4], o0[4 * q4 + 1], o0[4 * q4 + 2], o0[4 * q4 + 3]);
      if (g.out_plain1)
        *reinterpret_cast<float4 *>(g.out_plain1 + po) = make_float4(o1[4 * q4], o1[4 * q4 + 1], o1[4 * q4 + 2], o1[4 * q4 + 3]);
    }
  }
}

__device__ __forceinline__ void mbar_arrive(uint64_t *mbar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(tc::smem_u32(mbar)) : "memory");
}

// The tensor core accumulates in fp32 with truncation; over a long K (1600 for G1) that bias reaches 1e-4 of the
// pre-activations and breaks the force tolerance (measured).  The accumulation is therefore
// chunked: the MMAs of CP K panels (K = 64) go to one of two TMEM accumulators starting from zero, and the epilogue
// warps add the finished chunk to fp32 registers (round-to-nearest) while the next chunk runs in the other buffer.

template <int NT, int EPI, int OPF>
__global__ void __launch_bounds__(320, 1)
k_fit_tc(ChunkView C, int ty, FitTCArgs g) {
  using F = OpFmt<OPF>;
  constexpr int NP = F::NP, FT_CP = F::CP;
  constexpr int BPANEL = NT * 128;                               // bytes of one B panel (one piece)
  constexpr int STAGE = NP * (FT_APANEL + BPANEL);               // pieces of A, then pieces of B
  constexpr int STAGES = (STAGE * 3 <= 200 * 1024) ? 3 : ((STAGE * 2 <= 200 * 1024) ? 2 : 1);
  constexpr int NH = NT / 2;                                     // columns per epilogue warpgroup
  static_assert(NH % 8 == 0 && NH <= 128, "");
  extern __shared__ __align__(1024) uint8_t smem[];
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + STAGES * STAGE);
  uint64_t *empty = full + STAGES;
  uint64_t *accfull = empty + STAGES, *accempty = accfull + 2;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(accempty + 2);
  double *edot_sh = reinterpret_cast<double *>(smem);            // reused after the main loop (FE_L3)

  const int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  const int tile = blockIdx.x, m0 = tile * 128;
  if (m0 >= row_hi || m0 + 128 <= row_lo) return;               // tile holds no atom of this species
  const int nt = blockIdx.y, n0 = nt * NT;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nchunks = (g.KPAN + FT_CP - 1) / FT_CP;

  if (warp == 0) tc::tmem_alloc<512>(tmem_slot);
  if (tid == 32) {
    for (int s = 0; s < STAGES; ++s) { tc::mbar_init(full + s, 1); tc::mbar_init(empty + s, 1); }
    for (int b = 0; b < 2; ++b) { tc::mbar_init(accfull + b, 1); tc::mbar_init(accempty + b, 8); }
    tc::fence_mbar_init();
  }
  tc::fence_before_sync();
  __syncthreads();
  tc::fence_after_sync();
  const uint32_t tmem = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {
      const size_t aoff = (size_t)tile * g.KPAN * FT_APANEL, boff = (size_t)nt * g.KPAN * BPANEL;
      for (int kp = 0; kp < g.KPAN; ++kp) {
        const int s = kp % STAGES;
        if (kp >= STAGES) tc::mbar_wait(empty + s, ((kp / STAGES) - 1) & 1);
        uint8_t *st = smem + s * STAGE;
        tc::mbar_arrive_expect_tx(full + s, STAGE);
#pragma unroll
        for (int q = 0; q < NP; ++q) {
          tc::bulk_g2s(st + q * FT_APANEL, g.A[q] + aoff + (size_t)kp * FT_APANEL, FT_APANEL, full + s);
          tc::bulk_g2s(st + NP * FT_APANEL + q * BPANEL, g.B[q] + boff + (size_t)kp * BPANEL, BPANEL, full + s);
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      constexpr uint32_t idesc = OPF == 0 ? tc::make_idesc_tf32(128, NT) : tc::make_idesc_bf16(128, NT);
      for (int c = 0; c < nchunks; ++c) {
        const int buf = c & 1;
        if (c >= 2) tc::mbar_wait(accempty + buf, ((c >> 1) - 1) & 1);
        tc::fence_after_sync();
        const uint32_t td = tmem + buf * 256;
        const int kp_hi = min(g.KPAN, (c + 1) * FT_CP);
        for (int kp = c * FT_CP; kp < kp_hi; ++kp) {
          const int s = kp % STAGES;
          tc::mbar_wait(full + s, (kp / STAGES) & 1);
          tc::fence_after_sync();
          const uint32_t sa = tc::smem_u32(smem + s * STAGE), sb = sa + NP * FT_APANEL;
#pragma unroll
          for (int ks = 0; ks < 4; ++ks) {                         // 32 bytes of K per MMA: 8 TF32 or 16 BF16 columns
            const uint32_t first = (kp > c * FT_CP || ks > 0) ? 1u : 0u;
            uint64_t da[NP], db[NP];
#pragma unroll
            for (int q = 0; q < NP; ++q) {
              da[q] = tc::make_desc_sw128(sa + q * FT_APANEL + ks * 32);
              db[q] = tc::make_desc_sw128(sb + q * BPANEL + ks * 32);
            }
            if constexpr (OPF == 0) {                              // pieces (hi, lo): lo hi + hi lo + hi hi
              tc::mma_tf32_ss(td, da[1], db[0], idesc, first);
              tc::mma_tf32_ss(td, da[0], db[1], idesc, 1u);
              tc::mma_tf32_ss(td, da[0], db[0], idesc, 1u);
            } else if constexpr (OPF == 1) {                       // pieces (p0, p1, p2), smallest products first
              tc::mma_f16_ss(td, da[2], db[0], idesc, first);
              tc::mma_f16_ss(td, da[0], db[2], idesc, 1u);
              tc::mma_f16_ss(td, da[1], db[1], idesc, 1u);
              tc::mma_f16_ss(td, da[1], db[0], idesc, 1u);
              tc::mma_f16_ss(td, da[0], db[1], idesc, 1u);
              tc::mma_f16_ss(td, da[0], db[0], idesc, 1u);
            } else {
              tc::mma_f16_ss(td, da[0], db[0], idesc, first);
            }
          }
          tc::mma_commit(empty + s);
        }
        tc::mma_commit(accfull + buf);
      }
    }
  } else {
    // two epilogue warpgroups (columns [e NH, e NH + NH)); thread r = TMEM lane r = tile row r
    const int e = (warp - 2) >> 2;
    const int r = 32 * (warp & 3) + lane, m = m0 + r;
    const bool ok = m >= row_lo && m < row_hi;
    const uint32_t lane_sel = (uint32_t)(32 * (warp & 3)) << 16;
    float acc[NH];
#pragma unroll
    for (int i = 0; i < NH; ++i) acc[i] = 0.0f;
    for (int c = 0; c < nchunks; ++c) {
      const int buf = c & 1;
      tc::mbar_wait(accfull + buf, (c >> 1) & 1);
      tc::fence_after_sync();
      const uint32_t ta = tmem + lane_sel + buf * 256 + e * NH;
      constexpr int P0 = NH < 64 ? NH : 64, P1 = NH - P0;
      {
        uint32_t v[P0];
        tc::tmem_ld_cols_nowait<P0>(ta, v);
        tc::tmem_wait_ld();
#pragma unroll
        for (int i = 0; i < P0; ++i) acc[i] += __uint_as_float(v[i]);
      }
      if (P1 > 0) {
        uint32_t v[P1 > 0 ? P1 : 8];
        tc::tmem_ld_cols_nowait<(P1 > 0 ? P1 : 8)>(ta + P0, v);
        tc::tmem_wait_ld();
#pragma unroll
        for (int i = 0; i < P1; ++i) acc[P0 + i] += __uint_as_float(v[i]);
      }
      tc::fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive(accempty + buf);
    }
    double edot = 0.0;
    if (ok) {
#pragma unroll
      for (int j = 0; j < NH; j += 8) ft_epi8<EPI, OPF>(acc + j, n0 + e * NH + j, g, (size_t)tile, r, m, edot);
      if (EPI != FE_STORE && g.out[0] && e == 1)              // image columns between NT and the padded K must be zero
        for (int nn = n0 + NT; nn < g.KPAN_out * F::KP; nn += 4)
          img_store4<OPF>(g.out, (size_t)tile, g.KPAN_out, nn, r, 0.f, 0.f, 0.f, 0.f);
    }
    if (EPI == FE_L3) {
      // all stages have been consumed (the last accfull implies every MMA read its operands): smem is free
      if (e == 1) edot_sh[r] = edot;
      tc::bar_sync(1, 256);
      if (e == 0 && ok) g.atom_energy[g.s_idx[C.p0 + m]] = edot + edot_sh[r] + (double)g.b3;
    }
  }
  tc::fence_before_sync();
  __syncthreads();
  if (warp == 0) tc::tmem_dealloc<512>(tmem);
}

// ---- S5: descriptor as the A image of G1 ---------------------------------------------------------------------------
// D[b M^< + a] = sum_c T[b][c] T[a][c] (Eq. 4; reading R7), from the fp64 T rounded to fp32, written
// straight into the hi / lo operand images (the descriptor never exists in another form).  Thread = atom (tile row).
#define DESCR_R 16                     // atoms per block
// D = T (T^<)^T (Eq. 4) written directly as the A operand of G1 (hi / lo images).  A block stages the fp32 copy of its
// atoms' T rows in shared memory (coalesced 16-byte loads of the contiguous fp64 rows), then walks (K panel, row, 16-byte
// chunk) tasks with the chunk index fastest: eight lanes write one full 128-byte image row, a warp four adjacent rows =
// 512 contiguous bytes per store (thread-per-row stores touched 32 separate lines, half a sector each).
template <int MA, int OPF>
__global__ void __launch_bounds__(256) k_descr_tc(DevModel P, ChunkView C, int ty, int kpan, FitTCArgs img) {
  constexpr int KP = OpFmt<OPF>::KP, CH = KP / 4;                  // 4-column chunks per panel row
  extern __shared__ float4 Ts[];                                   // [DESCR_R][M + 1]
  // one launch per species, on that species' stream: blocks outside its row range leave at once
  const int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  const int row0 = blockIdx.x * DESCR_R, nrow = min(DESCR_R, C.n - row0), M = P.M, ld = M + 1;
  if (row0 >= row_hi || row0 + DESCR_R <= row_lo) return;
  {
    const double2 *src = reinterpret_cast<const double2 *>(C.T + (size_t)row0 * M * 4);
    float2 *dst = reinterpret_cast<float2 *>(Ts);
    for (int k = threadIdx.x; k < nrow * M * 2; k += 256) {
      const double2 v = src[k];
      const int rl = k / (2 * M), w = k - rl * 2 * M;
      dst[rl * 2 * ld + w] = make_float2((float)v.x, (float)v.y);
    }
  }
  __syncthreads();
  const int ntask = DESCR_R * kpan * CH, kreal = M * MA;
  for (int q = threadIdx.x; q < ntask; q += 256) {
    const int j = q % CH, rl = (q / CH) & (DESCR_R - 1), pan = q / (CH * DESCR_R);
    const int m = row0 + rl, k0 = pan * KP + 4 * j;
    if (rl >= nrow || m < row_lo || m >= row_hi) continue;
    float d[4] = {0.f, 0.f, 0.f, 0.f};                             // image columns between dim and the padded K are zero
    if (k0 < kreal) {
      const int b = k0 / MA, a0 = k0 - b * MA;
      const float4 tb = Ts[rl * ld + b];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float4 ta = Ts[rl * ld + a0 + k];
        d[k] = fmaf(tb.x, ta.x, fmaf(tb.y, ta.y, fmaf(tb.z, ta.z, tb.w * ta.w)));
      }
    }
    img_store4<OPF>(img.out, (size_t)(m >> 7), kpan, k0, m & 127, d[0], d[1], d[2], d[3]);
  }
}

// ---- S7: dT[b][c] = sum_a dD[b][a] T[a][c] + [b < M^<] sum_b' dD[b'][b] T[b'][c] (one of the S7 contractions: fp32
// products and sums like the GEMMs), written as the fp32 copy pass 2 reads and, for the debug hook only, as fp64.
// One WARP per atom, no block barrier, ONE coalesced pass over the atom's dD row (M M^< floats): a warp instruction loads
// 512 contiguous bytes, lane l holds dD[b][a0 .. a0 + 3] with b = 32 / LPR * i + l / LPR, a0 = 4 (l mod LPR), LPR = M^< / 4
// lanes per row.  From that one load: the first term's partial sum over the lane's four a (T[a0 ..] kept in registers),
// completed across the LPR lanes of the row by shuffles; and the second term's 4 x 4 accumulators (a = a0 + k, c), summed
// over the lane's rows and at the end across the lanes that share a0.  Only the fp32 copy of T is in shared memory.
#define DT_WARPS 8
template <int LPR>
__global__ void __launch_bounds__(32 * DT_WARPS) k_dT_tc(DevModel P, ChunkView C, int ldd, const float *__restrict__ dD,
                                                         float *__restrict__ dT32, double *__restrict__ dT64, int ty) {
  extern __shared__ float4 sm4[];
  constexpr int Ma = 4 * LPR, RPI = 32 / LPR;                   // rows per warp instruction
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q = blockIdx.x * DT_WARPS + warp;
  // one launch per species, at the tail of that species' chain
  const int row_lo = max(C.p0, C.type_start[ty]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[ty + 1]) - C.p0;
  if (q >= C.n || q < row_lo || q >= row_hi) return;
  const int M = P.M;
  float4 *Ts = sm4 + warp * (M + 2 * Ma);                       // [M]   T[b][0..3] in fp32
  float4 *f1 = Ts + M, *t2 = f1 + Ma;                           // [Ma] first term of rows b < M^<; [Ma] second term
  const double2 *T = reinterpret_cast<const double2 *>(C.T + (size_t)q * M * 4);
  for (int k = lane; k < M; k += 32) {
    const double2 u = T[2 * k], v = T[2 * k + 1];
    Ts[k] = make_float4((float)u.x, (float)u.y, (float)v.x, (float)v.y);
  }
  __syncwarp();
  const int a0 = 4 * (lane % LPR), rl = lane / LPR;
  const float4 ta0 = Ts[a0], ta1 = Ts[a0 + 1], ta2 = Ts[a0 + 2], ta3 = Ts[a0 + 3];
  const float4 *row4 = reinterpret_cast<const float4 *>(dD + (size_t)q * ldd) + lane;
  float4 c0 = make_float4(0.f, 0.f, 0.f, 0.f), c1 = c0, c2 = c0, c3 = c0;      // second term, a = a0 + k
  auto one = [&](int b, const float4 d) {
    // first term, partial over a0 .. a0 + 3
    float s0 = fmaf(d.x, ta0.x, fmaf(d.y, ta1.x, fmaf(d.z, ta2.x, d.w * ta3.x)));
    float s1 = fmaf(d.x, ta0.y, fmaf(d.y, ta1.y, fmaf(d.z, ta2.y, d.w * ta3.y)));
    float s2 = fmaf(d.x, ta0.z, fmaf(d.y, ta1.z, fmaf(d.z, ta2.z, d.w * ta3.z)));
    float s3 = fmaf(d.x, ta0.w, fmaf(d.y, ta1.w, fmaf(d.z, ta2.w, d.w * ta3.w)));
#pragma unroll
    for (int off = 1; off < LPR; off <<= 1) {
      s0 += __shfl_xor_sync(0xffffffffu, s0, off); s1 += __shfl_xor_sync(0xffffffffu, s1, off);
      s2 += __shfl_xor_sync(0xffffffffu, s2, off); s3 += __shfl_xor_sync(0xffffffffu, s3, off);
    }
    if (b < M) {
      const float4 tb = Ts[b];
      c0.x = fmaf(d.x, tb.x, c0.x); c0.y = fmaf(d.x, tb.y, c0.y); c0.z = fmaf(d.x, tb.z, c0.z); c0.w = fmaf(d.x, tb.w, c0.w);
      c1.x = fmaf(d.y, tb.x, c1.x); c1.y = fmaf(d.y, tb.y, c1.y); c1.z = fmaf(d.y, tb.z, c1.z); c1.w = fmaf(d.y, tb.w, c1.w);
      c2.x = fmaf(d.z, tb.x, c2.x); c2.y = fmaf(d.z, tb.y, c2.y); c2.z = fmaf(d.z, tb.z, c2.z); c2.w = fmaf(d.z, tb.w, c2.w);
      c3.x = fmaf(d.w, tb.x, c3.x); c3.y = fmaf(d.w, tb.y, c3.y); c3.z = fmaf(d.w, tb.z, c3.z); c3.w = fmaf(d.w, tb.w, c3.w);
      if (lane % LPR == 0) {
        const float4 o4 = make_float4(s0, s1, s2, s3);
        if (b < Ma) f1[b] = o4;                                  // completed below with the second term
        else {
          reinterpret_cast<float4 *>(dT32)[(size_t)q * M + b] = o4;
          if (dT64) {
            double2 *o = reinterpret_cast<double2 *>(dT64 + ((size_t)q * M + b) * 4);
            o[0] = make_double2((double)s0, (double)s1);
            o[1] = make_double2((double)s2, (double)s3);
          }
        }
      }
    }
  };
  const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
  const int NI = (M + RPI - 1) / RPI;                           // the same trip count for every lane: the shuffles are warp-wide
  int i = 0;
  for (; i + 2 <= NI; i += 2) {                                 // two loads in flight
    const int b0 = i * RPI + rl, b1 = b0 + RPI;
    const float4 d0 = b0 < M ? row4[(size_t)i * 32] : z4;
    const float4 d1 = b1 < M ? row4[(size_t)(i + 1) * 32] : z4;
    one(b0, d0);
    one(b1, d1);
  }
  if (i < NI) {
    const int b0 = i * RPI + rl;
    one(b0, b0 < M ? row4[(size_t)i * 32] : z4);
  }
  // second term: sum over the lanes that share a0
#pragma unroll
  for (int off = LPR; off < 32; off <<= 1) {
    c0.x += __shfl_xor_sync(0xffffffffu, c0.x, off); c0.y += __shfl_xor_sync(0xffffffffu, c0.y, off);
    c0.z += __shfl_xor_sync(0xffffffffu, c0.z, off); c0.w += __shfl_xor_sync(0xffffffffu, c0.w, off);
    c1.x += __shfl_xor_sync(0xffffffffu, c1.x, off); c1.y += __shfl_xor_sync(0xffffffffu, c1.y, off);
    c1.z += __shfl_xor_sync(0xffffffffu, c1.z, off); c1.w += __shfl_xor_sync(0xffffffffu, c1.w, off);
    c2.x += __shfl_xor_sync(0xffffffffu, c2.x, off); c2.y += __shfl_xor_sync(0xffffffffu, c2.y, off);
    c2.z += __shfl_xor_sync(0xffffffffu, c2.z, off); c2.w += __shfl_xor_sync(0xffffffffu, c2.w, off);
    c3.x += __shfl_xor_sync(0xffffffffu, c3.x, off); c3.y += __shfl_xor_sync(0xffffffffu, c3.y, off);
    c3.z += __shfl_xor_sync(0xffffffffu, c3.z, off); c3.w += __shfl_xor_sync(0xffffffffu, c3.w, off);
  }
  if (lane < LPR) { t2[a0] = c0; t2[a0 + 1] = c1; t2[a0 + 2] = c2; t2[a0 + 3] = c3; }
  __syncwarp();
  if (lane < Ma && lane < M) {
    const float4 u = f1[lane], v = t2[lane];
    const float s0 = u.x + v.x, s1 = u.y + v.y, s2 = u.z + v.z, s3 = u.w + v.w;
    reinterpret_cast<float4 *>(dT32)[(size_t)q * M + lane] = make_float4(s0, s1, s2, s3);
    if (dT64) {
      double2 *o = reinterpret_cast<double2 *>(dT64 + ((size_t)q * M + lane) * 4);
      o[0] = make_double2((double)s0, (double)s1);
      o[1] = make_double2((double)s2, (double)s3);
    }
  }
}

// ---- host: weights as B images -------------------------------------------------------------------------------------
static int ft_round_up(int x, int m) { return (x + m - 1) / m * m; }

// B[n][k] for n < N, k < K (zero outside), as [ntiles][kpan][NT rows x 128 B] swizzled panels, one array per piece;
// appends the pieces to `out` (bytes) and returns their offsets
template <class F>
static void pack_B(int opf, F get, int N, int K, int NT, int ntiles, int kpan, std::vector<uint8_t> &out, size_t off[3]) {
  const int np = opf_np(opf), kp_cols = opf_kp(opf);
  const size_t sz = (size_t)ntiles * kpan * NT * 128;
  const size_t at = (out.size() + 1023) / 1024 * 1024;
  out.resize(at + np * sz, 0);
  for (int q = 0; q < 3; ++q) off[q] = at + (size_t)(q < np ? q : 0) * sz;
  for (int nt = 0; nt < ntiles; ++nt)
    for (int kp = 0; kp < kpan; ++kp) {
      const size_t base = ((size_t)nt * kpan + kp) * NT * 128;
      for (int rn = 0; rn < NT; ++rn) {
        const int n = nt * NT + rn;
        if (n >= N) continue;
        for (int kk = 0; kk < kp_cols; ++kk) {
          const int k = kp * kp_cols + kk;
          if (k >= K) continue;
          const double w = get(n, k);
          if (opf == 0) {
            const float hi = tc_host_tf32((float)w), lo = tc_host_tf32((float)(w - (double)hi));
            const size_t o = base + tc::sw128_offset(rn, kk);
            memcpy(&out[off[0] + o], &hi, 4);
            memcpy(&out[off[1] + o], &lo, 4);
          } else {
            float rem = (float)w;
            const size_t o = base + tc::sw128_offset_b16(rn, kk);
            for (int q = 0; q < np; ++q) {
              const uint16_t b = tc_host_bf16_bits(rem);
              memcpy(&out[off[q] + o], &b, 2);
              rem -= tc_host_bf16_value(b);
            }
          }
        }
      }
    }
}

static int ft_pick_nt(int fw) {
  if (fw <= 32) return 32;
  if (fw <= 64) return 64;
  if (fw <= 128) return 128;
  if (fw <= 240) return 240;
  if (fw <= 256) return 256;
  return 0;
}

cudaError_t tc_prepare_fit(const DevModel &P, const double *fit_h, TCWeights &W, int opf) {
  if (P.fw % 4 != 0 || ft_pick_nt(P.fw) == 0 || (P.Ma != 4 && P.Ma != 8 && P.Ma != 16)) return cudaErrorNotSupported;
  FitTC *F = new FitTC();
  const int KP = opf_kp(opf);
  F->opf = opf;
  F->fw = P.fw; F->fwp = ft_round_up(P.fw, KP); F->NT = ft_pick_nt(P.fw);
  F->NT6 = P.dim >= 960 ? 240 : 128;
  F->dim = P.dim; F->dimp = ft_round_up(P.dim, F->NT6);
  const int fw = P.fw, dim = P.dim, kpw = F->fwp / KP, kpd = ft_round_up(dim, KP) / KP, nt6 = F->dimp / F->NT6;
  std::vector<uint8_t> h;
  struct Off { size_t W0[3], W1[3], W2[3], W2T[3], W1T[3], W0T[3], b0, b1, b2, w3; };
  std::vector<Off> offs(P.ntypes);
  for (int ty = 0; ty < P.ntypes; ++ty) {
    const double *W0 = fit_h + (size_t)ty * P.fit_net_size;
    const double *b0 = W0 + (size_t)dim * fw, *W1 = b0 + fw, *b1 = W1 + (size_t)fw * fw, *W2 = b1 + fw,
                 *b2 = W2 + (size_t)fw * fw, *w3 = b2 + fw;
    Off &o = offs[ty];
    // forward GEMMs: C[r][n] = sum_k A[r][k] W[k][n]  ->  B[n][k] = W[k][n]
    pack_B(opf, [&](int n, int k) { return W0[(size_t)k * fw + n]; }, fw, dim, F->NT, 1, kpd, h, o.W0);
    pack_B(opf, [&](int n, int k) { return W1[(size_t)k * fw + n]; }, fw, fw, F->NT, 1, kpw, h, o.W1);
    pack_B(opf, [&](int n, int k) { return W2[(size_t)k * fw + n]; }, fw, fw, F->NT, 1, kpw, h, o.W2);
    // backward GEMMs: C[r][n] = sum_k Q[r][k] W[n][k]  ->  B[n][k] = W[n][k]
    pack_B(opf, [&](int n, int k) { return W2[(size_t)n * fw + k]; }, fw, fw, F->NT, 1, kpw, h, o.W2T);
    pack_B(opf, [&](int n, int k) { return W1[(size_t)n * fw + k]; }, fw, fw, F->NT, 1, kpw, h, o.W1T);
    pack_B(opf, [&](int n, int k) { return W0[(size_t)n * fw + k]; }, dim, fw, F->NT6, nt6, kpw, h, o.W0T);
    auto vecpad = [&](const double *src) {
      const size_t at = (h.size() + 15) / 16 * 16;
      h.resize(at + 256 * sizeof(float), 0);
      for (int i = 0; i < fw; ++i) { const float v = (float)src[i]; memcpy(&h[at + 4 * (size_t)i], &v, 4); }
      return at;
    };
    o.b0 = vecpad(b0); o.b1 = vecpad(b1); o.b2 = vecpad(b2); o.w3 = vecpad(w3);
  }
  cudaError_t e = cudaMalloc(&F->buf, h.size());
  if (e != cudaSuccess) { delete F; return e; }
  e = cudaMemcpy(F->buf, h.data(), h.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { cudaFree(F->buf); delete F; return e; }
  for (int ty = 0; ty < P.ntypes; ++ty) {
    const Off &o = offs[ty];
    const uint8_t *b = F->buf;
    FitTCNet n{};
    for (int q = 0; q < 3; ++q) {
      n.W0[q] = b + o.W0[q]; n.W1[q] = b + o.W1[q]; n.W2[q] = b + o.W2[q];
      n.W2T[q] = b + o.W2T[q]; n.W1T[q] = b + o.W1T[q]; n.W0T[q] = b + o.W0T[q];
    }
    n.b0 = reinterpret_cast<const float *>(b + o.b0); n.b1 = reinterpret_cast<const float *>(b + o.b1);
    n.b2 = reinterpret_cast<const float *>(b + o.b2); n.w3 = reinterpret_cast<const float *>(b + o.w3);
    n.b3 = (float)fit_h[(size_t)ty * P.fit_net_size + P.fit_net_size - 1];
    F->nets.push_back(n);
  }
  W.fit = F;
  return cudaSuccess;
}

void tc_release_fit(TCWeights &W) {
  FitTC *F = reinterpret_cast<FitTC *>(W.fit);
  if (F) {
    if (F->buf) cudaFree(F->buf);
    delete F;
  }
  W.fit = nullptr;
}

// images: D (NP pieces x tiles x kpd panels), X0 and X1 (NP x tiles x kpw each); plain fp32: Z0 S0 S1 Z1 dZ1 [rows][fwp], dD
size_t tc_fit_workspace_bytes(const DevModel &P, int64_t chunk, int opf) {
  const int KP = opf_kp(opf), np = opf_np(opf);
  const size_t tiles = (size_t)(chunk + 127) / 128, rows = tiles * 128;
  const size_t kpd = (size_t)ft_round_up(P.dim, KP) / KP, fwp = ft_round_up(P.fw, KP), kpw = fwp / KP,
               dimp = ft_round_up(P.dim, P.dim >= 960 ? 240 : 128);
  return (size_t)np * tiles * (kpd + 2 * kpw) * FT_APANEL + sizeof(float) * (5 * rows * fwp + rows * dimp) + 4096;
}

template <int NT, int EPI, int OPF>
static cudaError_t ft_launch(const ChunkView &C, int ty, const FitTCArgs &g, int ntiles_n, cudaStream_t st) {
  constexpr int STAGE = OpFmt<OPF>::NP * (FT_APANEL + NT * 128);
  constexpr int STAGES = (STAGE * 3 <= 200 * 1024) ? 3 : ((STAGE * 2 <= 200 * 1024) ? 2 : 1);
  constexpr int smem = STAGES * STAGE + 128;
  static_assert(smem <= 227 * 1024, "stage does not fit");
  static bool configured_d[DPB_MAX_DEVICES] = {};
  bool &configured = configured_d[dpb_device()];
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_fit_tc<NT, EPI, OPF>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid((C.n + 127) / 128, ntiles_n);
  k_fit_tc<NT, EPI, OPF><<<grid, 320, smem, st>>>(C, ty, g);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

struct FitTCBufs { uint8_t *D[3], *X0[3], *X1[3]; float *Z0, *S0, *S1, *Z1, *dZ1, *dD; };

template <int NT, int OPF>
static cudaError_t ft_run_type(const DevModel &P, const ChunkView &C, const FitTC &F, int ty, const FitTCBufs &B,
                               double *atom_energy, cudaStream_t st) {
  constexpr int KP = OpFmt<OPF>::KP;
  const FitTCNet &N = F.nets[ty];
  const int kpw = F.fwp / KP, kpd = ft_round_up(F.dim, KP) / KP, fw = F.fw, ldp = F.fwp;
  cudaError_t e;
  FitTCArgs g{};
  auto setA = [&](uint8_t *const a[3]) { for (int q = 0; q < 3; ++q) g.A[q] = a[q]; };
  auto setB = [&](const uint8_t *const b[3]) { for (int q = 0; q < 3; ++q) g.B[q] = b[q]; };
  auto setO = [&](uint8_t *const o[3]) { for (int q = 0; q < 3; ++q) g.out[q] = o ? o[q] : nullptr; };
  g.s_idx = C.s_idx; g.ldp = ldp; g.N = fw; g.KPAN_out = kpw;
  // G1: Z0 = tanh(D W0 + b0), S0 = 1 - Z0^2 (stored: recomputing it from the rounded Z0 loses the saturated units)
  setA(B.D); setB(N.W0); g.KPAN = kpd; g.bias = N.b0;
  g.out_plain0 = B.Z0; g.out_plain1 = B.S0; setO(B.X0);
  if ((e = ft_launch<NT, FE_TANH, OPF>(C, ty, g, 1, st)) != cudaSuccess) return e;
  // G2: U1 = tanh(Z0 W1 + b1), Z1 = Z0 + U1, S1 = 1 - U1^2
  setA(B.X0); setB(N.W1); g.KPAN = kpw; g.bias = N.b1; g.in0 = B.Z0;
  g.out_plain0 = B.Z1; g.out_plain1 = B.S1; setO(B.X1);
  if ((e = ft_launch<NT, FE_TANH_SKIP, OPF>(C, ty, g, 1, st)) != cudaSuccess) return e;
  // G3: U2 = tanh(Z1 W2 + b2), E_i = (Z1 + U2) . w3 + b3, Q2 = w3 (1 - U2^2)
  setA(B.X1); setB(N.W2); g.bias = N.b2; g.w3 = N.w3; g.in0 = B.Z1; g.b3 = N.b3;
  g.atom_energy = atom_energy; g.out_plain0 = nullptr; g.out_plain1 = nullptr; setO(B.X0);
  if ((e = ft_launch<NT, FE_L3, OPF>(C, ty, g, 1, st)) != cudaSuccess) return e;
  // G4: dZ1 = w3 + Q2 W2^T, Q1 = dZ1 S1
  setA(B.X0); setB(N.W2T); g.in0 = nullptr; g.in1 = B.S1;
  g.out_plain0 = nullptr; g.out_plain1 = B.dZ1; setO(B.X1);
  if ((e = ft_launch<NT, FE_BWD1, OPF>(C, ty, g, 1, st)) != cudaSuccess) return e;
  // G5: dZ0 = dZ1 + Q1 W1^T, Q0 = dZ0 S0
  setA(B.X1); setB(N.W1T); g.in0 = B.dZ1; g.in1 = B.S0;
  g.out_plain0 = nullptr; g.out_plain1 = nullptr; setO(B.X0);
  if ((e = ft_launch<NT, FE_BWD0, OPF>(C, ty, g, 1, st)) != cudaSuccess) return e;
  // G6: dD = Q0 W0^T
  setA(B.X0); setB(N.W0T); g.N = F.dim; g.ldp = F.dimp; g.KPAN_out = 0;
  g.out_plain0 = B.dD; setO(nullptr); g.in0 = nullptr; g.in1 = nullptr;
  if (F.NT6 == 240) return ft_launch<240, FE_STORE, OPF>(C, ty, g, F.dimp / 240, st);
  return ft_launch<128, FE_STORE, OPF>(C, ty, g, F.dimp / 128, st);
}

template <int OPF>
static cudaError_t tc_fit_fmt(const DevModel &P, const ChunkView &C, const FitTC *F, void *ws, float *dT32,
                              double *atom_energy, cudaStream_t st, bool want_dT64) {
  constexpr int KP = OpFmt<OPF>::KP, NP = OpFmt<OPF>::NP;
  const size_t tiles = (size_t)(C.n + 127) / 128, rows = tiles * 128;
  const size_t kpd = (size_t)ft_round_up(F->dim, KP) / KP, kpw = F->fwp / KP;
  uint8_t *pb = reinterpret_cast<uint8_t *>(ws);
  FitTCBufs B{};
  for (int q = 0; q < 3; ++q) { B.D[q] = pb + (size_t)(q < NP ? q : 0) * tiles * kpd * FT_APANEL; }
  pb += (size_t)NP * tiles * kpd * FT_APANEL;
  for (int q = 0; q < 3; ++q) { B.X0[q] = pb + (size_t)(q < NP ? q : 0) * tiles * kpw * FT_APANEL; }
  pb += (size_t)NP * tiles * kpw * FT_APANEL;
  for (int q = 0; q < 3; ++q) { B.X1[q] = pb + (size_t)(q < NP ? q : 0) * tiles * kpw * FT_APANEL; }
  pb += (size_t)NP * tiles * kpw * FT_APANEL;
  float *p = reinterpret_cast<float *>(pb);
  B.Z0 = p; p += rows * F->fwp;
  B.S0 = p; p += rows * F->fwp;
  B.S1 = p; p += rows * F->fwp;
  B.Z1 = p; p += rows * F->fwp;
  B.dZ1 = p; p += rows * F->fwp;
  B.dD = p;
  // The per-type chains (descriptor rows, six GEMMs, dT contraction) are independent: disjoint rows; a tile on the type
  // boundary is read by both and written row-wise by each.  G1-G5 of one type fill only as many SMs as that type has row
  // tiles (W24k: 64 and 128 of 148), and the descriptor / dT kernels are memory-bound while the GEMMs are not: forked
  // streams let one type's work take what the other leaves idle.  Largest type (last) on the caller's stream.
  const unsigned nbd = (unsigned)((C.n + DESCR_R - 1) / DESCR_R), nbt = (unsigned)((C.n + DT_WARPS - 1) / DT_WARPS);
  const size_t smd = (size_t)DESCR_R * (P.M + 1) * sizeof(float4);
  const size_t smt = sizeof(float4) * DT_WARPS * ((size_t)P.M + 2 * P.Ma);
  if (smt > 48 * 1024 || smd > 48 * 1024) return cudaErrorInvalidValue;   // M <= 256 is checked at model creation
  double *dT64 = want_dT64 ? C.dT : nullptr;
  cudaStream_t ts[DPB_MAX_TYPES];
  {
    cudaError_t e = dpb_fork_streams(P.ntypes, st, ts);
    if (e != cudaSuccess) return e;
  }
  FitTCArgs dimg{};
  for (int q = 0; q < 3; ++q) dimg.out[q] = B.D[q];
  for (int k = 0; k < P.ntypes; ++k) {
    const int ty = P.ntypes - 1 - k;
    cudaStream_t s = ts[k];
    switch (P.Ma) {
      case 4: k_descr_tc<4, OPF><<<nbd, 256, smd, s>>>(P, C, ty, (int)kpd, dimg); break;
      case 8: k_descr_tc<8, OPF><<<nbd, 256, smd, s>>>(P, C, ty, (int)kpd, dimg); break;
      default: k_descr_tc<16, OPF><<<nbd, 256, smd, s>>>(P, C, ty, (int)kpd, dimg); break;
    }
    DPB_LAUNCHED(1);
    cudaError_t e;
    switch (F->NT) {
      case 32: e = ft_run_type<32, OPF>(P, C, *F, ty, B, atom_energy, s); break;
      case 64: e = ft_run_type<64, OPF>(P, C, *F, ty, B, atom_energy, s); break;
      case 128: e = ft_run_type<128, OPF>(P, C, *F, ty, B, atom_energy, s); break;
      case 240: e = ft_run_type<240, OPF>(P, C, *F, ty, B, atom_energy, s); break;
      default: e = ft_run_type<256, OPF>(P, C, *F, ty, B, atom_energy, s); break;
    }
    if (e != cudaSuccess) return e;
    switch (P.Ma) {
      case 4: k_dT_tc<1><<<nbt, 32 * DT_WARPS, smt, s>>>(P, C, F->dimp, B.dD, dT32, dT64, ty); break;
      case 8: k_dT_tc<2><<<nbt, 32 * DT_WARPS, smt, s>>>(P, C, F->dimp, B.dD, dT32, dT64, ty); break;
      default: k_dT_tc<4><<<nbt, 32 * DT_WARPS, smt, s>>>(P, C, F->dimp, B.dD, dT32, dT64, ty); break;
    }
    DPB_LAUNCHED(1);
  }
  {
    cudaError_t e = dpb_join_streams(P.ntypes, st, ts);
    if (e != cudaSuccess) return e;
  }
  return cudaGetLastError();
}

cudaError_t tc_fit(const DevModel &P, const ChunkView &C, const TCWeights &W, void *ws, float *dT32, double *atom_energy,
                   cudaStream_t st, bool want_dT64) {
  if (C.n <= 0) return cudaSuccess;
  const FitTC *F = reinterpret_cast<const FitTC *>(W.fit);
  if (!F) return cudaErrorNotSupported;
  switch (F->opf) {
    case 0: return tc_fit_fmt<0>(P, C, F, ws, dT32, atom_energy, st, want_dT64);
    case 1: return tc_fit_fmt<1>(P, C, F, ws, dT32, atom_energy, st, want_dT64);
    default: return tc_fit_fmt<2>(P, C, F, ws, dT32, atom_energy, st, want_dT64);
  }
}
