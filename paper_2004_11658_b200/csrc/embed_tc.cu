// embed_tc.cu — mixed-precision (DPB_TF32) embedding passes on the 5th-generation tensor cores (BASELINE.json
// configs[3]).  S3-S5 (pass 1) and S8-S9 (pass 2) of the hot path:
//   * env matrix R~ (Eq. 5), the chain to the displacement (O10), and every accumulation of T, F, Xi stay in fp64;
//   * the embedding GEMMs (Eq. 8-9) run as tcgen05.mma kind::tf32 with fp32 accumulators in TMEM,
//     operands split x = hi + lo (3xTF32, tc_common.cuh) so that the contraction is accurate to fp32 rounding;
//   * tanh in fp32 (ex2.approx / rcp.approx).
// Work decomposition: the real (non-padded) slots of section t of all centre atoms of type a are flattened into one
// pair list (k_pair_scan / k_pair_expand); a tile is 128 consecutive pairs = the 128 TMEM lanes; thread r of a
// warpgroup owns row r through the whole net (layer outputs come back with tcgen05.ld 32x32b, one row per thread,
// so the concat skip [x || x] of Eq. 9 is a register add).  Two warpgroups per CTA work on independent tiles (own
// 64 KB operand slot, own TMEM columns, own mbarrier): while one waits for its MMAs the other runs its tanh epilogue.
#include <cstring>
#include <vector>

#include "tc_common.cuh"
#include "tc_kernels.cuh"

template <int S1>
struct TL {
  static constexpr int N1 = (2 * S1 + 7) / 8 * 8, N2 = (4 * S1 + 7) / 8 * 8;
  static constexpr int KS1 = (S1 + 7) / 8, KS2 = (2 * S1 + 7) / 8, PAN2 = (KS2 + 3) / 4;
  static constexpr int W1B = N1 * 128, W2P = N2 * 128, W2B = PAN2 * W2P;       // bytes of one hi (or lo) image
  static constexpr int oW1h = 0, oW1l = W1B, oW2h = 2 * W1B, oW2l = 2 * W1B + W2B, oVec = 2 * W1B + 2 * W2B;
  static constexpr int vW0 = 0, vb0 = 32, vb1 = 64, vb2 = 64 + N1, nv1 = 64 + N1 + N2;           // floats
  // the same vectors scaled by 2 log2(e) (pass 1 feeds them straight into ex2)
  static constexpr int sW0 = nv1, sb0 = nv1 + 32, sb1 = nv1 + 64, sb2 = nv1 + 64 + N1, nvec = 2 * nv1;
  static constexpr int img_bytes = (oVec + 4 * nvec + 1023) / 1024 * 1024;
  static constexpr int SLOT = 65536;                       // per-warpgroup operand slot
  static constexpr int oSlot = img_bytes, oEnv = oSlot + 2 * SLOT, oIds = oEnv + 2 * 128 * 32,
                       oBar = oIds + 2 * 256 * 4, oTmem = oBar + 16, smem_bytes = oTmem + 16;
  static_assert(S1 <= 32, "layer-1 operand is one 32-wide panel");
  static_assert(N2 <= 128 && PAN2 <= 2, "layer-2 operand: two 32-wide panels, 128 output columns");
};

// ---- host: pack one net into its shared-memory image ---------------------------------------------------------
template <int S1>
static void pack_net_tc(const double *net, std::vector<float> &out) {
  using L = TL<S1>;
  out.assign(L::img_bytes / 4, 0.0f);
  const double *W0 = net, *b0 = W0 + S1, *W1 = b0 + S1, *b1 = W1 + (size_t)S1 * 2 * S1, *W2 = b1 + 2 * S1,
               *b2 = W2 + (size_t)2 * S1 * 4 * S1;
  auto put = [&](int byte_base, int n, int k, double w) {
    const float hi = tc_host_tf32((float)w);
    const float lo = tc_host_tf32((float)(w - (double)hi));
    (void)lo;
    out[(byte_base + tc::sw128_offset(n, k)) / 4] = hi;
  };
  auto put_lo = [&](int byte_base, int n, int k, double w) {
    const float hi = tc_host_tf32((float)w);
    out[(byte_base + tc::sw128_offset(n, k)) / 4] = tc_host_tf32((float)(w - (double)hi));
  };
  for (int k = 0; k < S1; ++k)
    for (int n = 0; n < 2 * S1; ++n) {
      put(L::oW1h, n, k, W1[(size_t)k * 2 * S1 + n]);
      put_lo(L::oW1l, n, k, W1[(size_t)k * 2 * S1 + n]);
    }
  for (int k = 0; k < 2 * S1; ++k)
    for (int n = 0; n < 4 * S1; ++n) {
      const int pan = k / 32, kk = k % 32;
      put(L::oW2h + pan * L::W2P, n, kk, W2[(size_t)k * 4 * S1 + n]);
      put_lo(L::oW2l + pan * L::W2P, n, kk, W2[(size_t)k * 4 * S1 + n]);
    }
  float *vec = out.data() + L::oVec / 4;
  for (int s = 0; s < S1; ++s) { vec[L::vW0 + s] = (float)W0[s]; vec[L::vb0 + s] = (float)b0[s]; }
  for (int o = 0; o < 2 * S1; ++o) vec[L::vb1 + o] = (float)b1[o];
  for (int o = 0; o < 4 * S1; ++o) vec[L::vb2 + o] = (float)b2[o];
  const double c2 = 2.8853900817779268;
  for (int s = 0; s < S1; ++s) { vec[L::sW0 + s] = (float)(c2 * W0[s]); vec[L::sb0 + s] = (float)(c2 * b0[s]); }
  for (int o = 0; o < 2 * S1; ++o) vec[L::sb1 + o] = (float)(c2 * b1[o]);
  for (int o = 0; o < 4 * S1; ++o) vec[L::sb2 + o] = (float)(c2 * b2[o]);
}

static bool tc_supported_s1(int s1) { return s1 == 8 || s1 == 16 || s1 == 25 || s1 == 32; }

cudaError_t tc_prepare_weights(const DevModel &P, const double *emb_h, TCWeights &W) {
  W.ready = false;
  if (!tc_supported_s1(P.s1)) return cudaErrorNotSupported;
  std::vector<float> one, all;
  const int nets = P.ntypes * P.ntypes;
  for (int k = 0; k < nets; ++k) {
    const double *net = emb_h + (size_t)k * P.emb_net_size;
    switch (P.s1) {
      case 8: pack_net_tc<8>(net, one); break;
      case 16: pack_net_tc<16>(net, one); break;
      case 25: pack_net_tc<25>(net, one); break;
      default: pack_net_tc<32>(net, one); break;
    }
    W.net_stride = one.size();
    all.insert(all.end(), one.begin(), one.end());
  }
  cudaError_t e = cudaMalloc(&W.emb, sizeof(float) * all.size());
  if (e != cudaSuccess) return e;
  e = cudaMemcpy(W.emb, all.data(), sizeof(float) * all.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return e;
  W.ready = true;
  return cudaSuccess;
}

void tc_release_weights(TCWeights &W) {
  tc_release_fit(W);
  if (W.emb) cudaFree(W.emb);
  W.emb = nullptr;
  W.ready = false;
}

// ---- pair list -----------------------------------------------------------------------------------------------
// off[t][q] = number of real slots of section t over the chunk's atoms before sorted position q (q in [0, n]).
__global__ void __launch_bounds__(1024) k_pair_scan(int n, int ntypes, const int *__restrict__ nreal, int *__restrict__ off) {
  const int t = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  __shared__ int wsum[32];
  __shared__ int carry_s;
  int *o = off + (size_t)t * (n + 1);
  int carry = 0;
  // 1024 consecutive atoms per round (coalesced): warp scan, scan of the 32 warp totals, running carry
  for (int sb = 0; sb < n; sb += 32 * 1024) {
  int vals[32];                                              // 32 rounds' loads in flight before the first barrier
#pragma unroll
  for (int r = 0; r < 32; ++r) {
    const int q = sb + r * 1024 + tid;
    vals[r] = q < n ? nreal[(size_t)q * ntypes + t] : 0;
  }
#pragma unroll
  for (int r = 0; r < 32; ++r) {
    const int base = sb + r * 1024;
    if (base >= n) break;
    const int q = base + tid;
    const int v = vals[r];
    int incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += u;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      const int w = wsum[lane];
      int wi = w;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, wi, d);
        if (lane >= d) wi += u;
      }
      wsum[lane] = wi - w;                                   // exclusive prefix of the warp totals
      if (lane == 31) carry_s = wi;                          // total of this round
    }
    __syncthreads();
    if (q < n) o[q] = carry + wsum[warp] + incl - v;
    carry += carry_s;
    __syncthreads();                                         // wsum / carry_s are rewritten in the next round
  }
  }
  if (tid == 0) o[n] = carry;
}

// pidx[n sec_start[t] + off[t][q] + k] = q Nm + sec_start[t] + k  for every real slot k of section t of atom q.
// One warp per atom: only the real slots are visited (copper at sel = 512 is 65 % padding), stores are contiguous.
__global__ void __launch_bounds__(256) k_pair_expand(DevModel P, int n, const int *__restrict__ nreal,
                                                     const int *__restrict__ off, int *__restrict__ pidx) {
  const int q = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (q >= n) return;
  for (int t = 0; t < P.ntypes; ++t) {
    const int nr = nreal[(size_t)q * P.ntypes + t];
    int *dst = pidx + (size_t)n * P.sec_start[t] + off[(size_t)t * (n + 1) + q];
    const int base = q * P.nm + P.sec_start[t];
    for (int k = lane; k < nr; k += 32) dst[k] = base + k;
  }
}

size_t tc_pair_workspace_bytes(const DevModel &P, int64_t chunk) {
  return sizeof(int) * ((size_t)P.ntypes * (chunk + 1) + (size_t)chunk * P.nm) + 256;
}

cudaError_t tc_build_pairs(const DevModel &P, const ChunkView &C, void *ws, cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  int *off = reinterpret_cast<int *>(ws);
  int *pidx = off + (size_t)P.ntypes * (C.n + 1);
  k_pair_scan<<<P.ntypes, 1024, 0, st>>>(C.n, P.ntypes, C.nreal, off);
  k_pair_expand<<<(unsigned)((C.n + 7) / 8), 256, 0, st>>>(P, C.n, C.nreal, off, pidx);
  DPB_LAUNCHED(2);
  return cudaGetLastError();
}

// ---- device helpers ------------------------------------------------------------------------------------------
__device__ __forceinline__ void env_row4_tc(const DevModel &P, const double4 v, double e[4]) {
  double w, dw;
  dp_switch(v.w, P.rcs, P.rc, w, dw);
  const double ir = 1.0 / v.w;
  const double s = w * ir;
  const double sr = s * ir;
  e[0] = s; e[1] = sr * v.x; e[2] = sr * v.y; e[3] = sr * v.z;
}

// write 4 consecutive K entries (one 16-byte chunk j of the 128-byte row) of a SW128 K-major panel, hi and lo
__device__ __forceinline__ void store_split4(uint8_t *pan_hi, uint8_t *pan_lo, uint32_t rowbase, uint32_t r7, int j,
                                             float v0, float v1, float v2, float v3) {
  float4 h, l;
  tc::split_tf32(v0, h.x, l.x);
  tc::split_tf32(v1, h.y, l.y);
  tc::split_tf32(v2, h.z, l.z);
  tc::split_tf32(v3, h.w, l.w);
  const uint32_t off = rowbase + ((((uint32_t)j ^ r7) & 7u) << 4);
  *reinterpret_cast<float4 *>(pan_hi + off) = h;
  *reinterpret_cast<float4 *>(pan_lo + off) = l;
}

// D (+)= A B with the 3xTF32 split: hi hi + lo hi + hi lo.  One thread issues.
__device__ __forceinline__ void mma3(uint32_t tmem_d, uint32_t a_hi, uint32_t a_lo, uint32_t b_hi, uint32_t b_lo,
                                     uint32_t idesc, bool first) {
  const uint64_t dah = tc::make_desc_sw128(a_hi), dal = tc::make_desc_sw128(a_lo);
  const uint64_t dbh = tc::make_desc_sw128(b_hi), dbl = tc::make_desc_sw128(b_lo);
  tc::mma_tf32_ss(tmem_d, dal, dbh, idesc, first ? 0u : 1u);
  tc::mma_tf32_ss(tmem_d, dah, dbl, idesc, 1u);
  tc::mma_tf32_ss(tmem_d, dah, dbh, idesc, 1u);
}

#ifdef TC_PROF
#include <cstdio>
#define TCP(i) tp[i] = clock64()
#else
#define TCP(i)
#endif
// ---- pass 1 ----------------------------------------------------------------------------------------------------
template <int S1>
__global__ void __launch_bounds__(256, 1)
k_pass1_tc(DevModel P, ChunkView C, const float *__restrict__ all_img, size_t net_stride,
           const int *__restrict__ off_all, const int *__restrict__ pidx_all) {
  using L = TL<S1>;
  extern __shared__ __align__(1024) uint8_t smem[];
  const int tid = threadIdx.x, wg = tid >> 7, wt = tid & 127, warp = tid >> 5;
  const float *vec = reinterpret_cast<const float *>(smem + L::oVec);
  uint8_t *slot = smem + L::oSlot + wg * L::SLOT;
  float4 *envt = reinterpret_cast<float4 *>(smem + L::oEnv) + wg * 128;   // fp32 copy of the tile's R~ rows
  int *ids = reinterpret_cast<int *>(smem + L::oIds) + wg * 256, *segs = ids + 128;
  uint64_t *mbar = reinterpret_cast<uint64_t *>(smem + L::oBar) + wg;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + L::oTmem);

  if (warp == 0) tc::tmem_alloc<512>(tmem_slot);
  if (tid == 0) {
    tc::mbar_init(reinterpret_cast<uint64_t *>(smem + L::oBar), 1);
    tc::mbar_init(reinterpret_cast<uint64_t *>(smem + L::oBar) + 1, 1);
    tc::fence_mbar_init();
  }
  tc::fence_proxy_async();
  tc::fence_before_sync();
  __syncthreads();
  tc::fence_after_sync();
  const uint32_t tmem = *tmem_slot;
  // TMEM columns of this warpgroup: A1 hi [0,32) lo [32,64), D1 [64,128); then A2 hi [0,64) lo [64,128) over them (the
  // layer-1 operands and accumulator are dead by then), D2 [128,256).  The A operands are written with tcgen05.st, one
  // row per thread, and the MMA reads them from tensor memory: no swizzled stores, no proxy fence, and half of the
  // shared-memory operand traffic of an SS-mode MMA.
  const uint32_t tA = tmem + wg * 256, tD1 = tA + 64, tD2 = tA + 128;
  const uint32_t lane_sel = (uint32_t)(32 * (warp & 3)) << 16;
  const uint32_t slot_a = tc::smem_u32(slot), img_a = tc::smem_u32(smem);
  const uint32_t rowbase = (uint32_t)(wt >> 3) * 1024u + (uint32_t)(wt & 7) * 128u, r7 = wt & 7;

  // one launch walks all ntypes^2 nets (a = centre type, t = neighbour type): the CTA reloads the weight image at a net
  // switch, so only the last net has a tail in which SMs idle (four launches per pass had four)
  uint32_t phase = 0;
  for (int net = 0; net < P.ntypes * P.ntypes; ++net) {
  const int a = net / P.ntypes, t = net - a * P.ntypes;
  const int *off_t = off_all + (size_t)t * (C.n + 1), *pidx_t = pidx_all + (size_t)C.n * P.sec_start[t];
  __syncthreads();                                          // every MMA that read the previous image has completed
  {
    const float *net_img = all_img + (size_t)net * net_stride;
    for (int k = tid; k < L::img_bytes / 16; k += 256)
      reinterpret_cast<int4 *>(smem)[k] = reinterpret_cast<const int4 *>(net_img)[k];
  }
  tc::fence_proxy_async();
  __syncthreads();
  const int row_lo = max(C.p0, C.type_start[a]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[a + 1]) - C.p0;
  int flat0 = 0, flat1 = 0;
  if (row_hi > row_lo) { flat0 = off_t[row_lo]; flat1 = off_t[row_hi]; }
  const int ntiles = (flat1 - flat0 + 127) >> 7;
#ifdef TC_PROF
  long long tp[11];
#endif

  // the pair of the next tile, its centre atom and that atom's section bounds are fetched one tile ahead (a chain of
  // three dependent global loads that would otherwise sit at the head of the tile)
  int nx_qa = 0, nx_o0 = 0, nx_o1 = 0;
  double4 nx_dv = make_double4(0.0, 0.0, 0.0, 1.0);
  bool nx_valid = false;
  {
    const int t0 = blockIdx.x * 2 + wg, p0 = flat0 + t0 * 128 + wt;
    nx_valid = t0 < ntiles && p0 < flat1;
    if (nx_valid) {
      const int idx = pidx_t[p0];
      nx_dv = C.dr[idx];
      nx_qa = idx / P.nm;
      nx_o0 = off_t[nx_qa]; nx_o1 = off_t[nx_qa + 1];
    }
  }
  for (int tile = blockIdx.x * 2 + wg; tile < ntiles; tile += gridDim.x * 2) {
    const bool valid = nx_valid;
    const int nrows = min(128, flat1 - (flat0 + tile * 128));
    double e[4] = {0.0, 0.0, 0.0, 0.0};
    int qa = -1;
    TCP(0);
    if (valid) {
      qa = nx_qa;
      env_row4_tc(P, nx_dv, e);
    }
    ids[wt] = qa;
    if (valid) {
      const int tile0 = flat0 + tile * 128, seg_lo = nx_o0 - tile0, seg_hi = nx_o1 - tile0;
      segs[wt] = min(nrows, seg_hi) | ((seg_lo >= 0 && seg_hi <= 128) ? 256 : 0);
    }
    {
      // [row][component]: one broadcast 16-byte load gives the accumulation (e0, e1) and (e2, e3) as register pairs
      envt[wt] = make_float4((float)e[0], (float)e[1], (float)e[2], (float)e[3]);
    }
    const float x = (float)e[0];
    // layer 0 (Eq. 8): h0 = tanh(x W0 + b0)
    float h0[32];
#pragma unroll
    for (int s = 0; s < 32; ++s) h0[s] = s < S1 ? tc::tanh_prescaled_f32(fmaf(x, vec[L::sW0 + s], vec[L::sb0 + s])) : 0.0f;
    {
      uint32_t w[32];
#pragma unroll
      for (int s = 0; s < 32; ++s) { float fh, fl; tc::split_tf32(h0[s], fh, fl); w[s] = __float_as_uint(fh); }
      tc::tmem_st32_nowait(tA + lane_sel, w);
#pragma unroll
      for (int s = 0; s < 32; ++s) { float fh, fl; tc::split_tf32(h0[s], fh, fl); w[s] = __float_as_uint(fl); }
      tc::tmem_st32_nowait(tA + lane_sel + 32, w);
      tc::tmem_wait_st();
    }
    TCP(1);
    tc::fence_before_sync();
    tc::bar_sync(1 + wg, 128);
    TCP(2);
    if (wt == 0) {
      tc::fence_after_sync();
      constexpr uint32_t idesc = tc::make_idesc_tf32(128, L::N1);
#pragma unroll
      for (int ks = 0; ks < L::KS1; ++ks) {
        const uint64_t dbh = tc::make_desc_sw128(img_a + L::oW1h + ks * 32), dbl = tc::make_desc_sw128(img_a + L::oW1l + ks * 32);
        tc::mma_tf32_ts(tD1, tA + 32 + 8 * ks, dbh, idesc, ks == 0 ? 0u : 1u);
        tc::mma_tf32_ts(tD1, tA + 8 * ks, dbl, idesc, 1u);
        tc::mma_tf32_ts(tD1, tA + 8 * ks, dbh, idesc, 1u);
      }
      tc::mma_commit(mbar);
    }
    tc::mbar_wait(mbar, phase);
    phase ^= 1;
    tc::fence_after_sync();
    TCP(3);
    // layer 1 (Eq. 9): h1 = (h0, h0) + tanh(h0 W1 + b1)
    float h1[2 * S1];
    {
      uint32_t v[L::N1];
      tc::tmem_ld_cols_nowait<L::N1>(tD1 + lane_sel, v);
      tc::tmem_wait_ld();
#pragma unroll
      for (int o = 0; o < 2 * S1; ++o) h1[o] = h0[o % S1] + tc::tanh_prescaled_f32(fmaf(__uint_as_float(v[o]), TC_2LOG2E, vec[L::sb1 + o]));
    }
    TCP(4);
    {
      uint32_t w[32];
#pragma unroll
      for (int half = 0; half < (8 * L::KS2 > 32 ? 2 : 1); ++half) {
#pragma unroll
        for (int lo = 0; lo < 2; ++lo) {
#pragma unroll
          for (int s = 0; s < 32; ++s) {
            const int o = 32 * half + s;
            float fh, fl;
            tc::split_tf32(o < 2 * S1 ? h1[o] : 0.0f, fh, fl);
            w[s] = __float_as_uint(lo ? fl : fh);
          }
          tc::tmem_st32_nowait(tA + lane_sel + 64 * lo + 32 * half, w);
        }
      }
      tc::tmem_wait_st();
    }
    TCP(5);
    tc::fence_before_sync();
    tc::bar_sync(1 + wg, 128);
    if (wt == 0) {
      tc::fence_after_sync();
      constexpr uint32_t idesc = tc::make_idesc_tf32(128, L::N2);
#pragma unroll
      for (int ks = 0; ks < L::KS2; ++ks) {
        const uint32_t bo = (ks >> 2) * L::W2P + (ks & 3) * 32;
        const uint64_t dbh = tc::make_desc_sw128(img_a + L::oW2h + bo), dbl = tc::make_desc_sw128(img_a + L::oW2l + bo);
        tc::mma_tf32_ts(tD2, tA + 64 + 8 * ks, dbh, idesc, ks == 0 ? 0u : 1u);
        tc::mma_tf32_ts(tD2, tA + 8 * ks, dbl, idesc, 1u);
        tc::mma_tf32_ts(tD2, tA + 8 * ks, dbh, idesc, 1u);
      }
      tc::mma_commit(mbar);
    }
    tc::mbar_wait(mbar, phase);
    phase ^= 1;
    tc::fence_after_sync();
    TCP(6);
    // layer 2 (Eq. 9): g = (h1, h1) + tanh(h1 W2 + b2), written to the slot TRANSPOSED: gT[feature][row], 128 floats per
    // feature, the 16-byte chunk (4 rows) XOR-swizzled with the feature (conflict-free 4-byte stores by row threads and
    // 16-byte loads by feature threads)
    float *gt = reinterpret_cast<float *>(slot);
    {
      constexpr int CH = 32, NCH = (L::N2 + CH - 1) / CH;
      uint32_t va[CH], vb[CH];
      tc::tmem_ld_cols_nowait<(L::N2 < CH ? L::N2 : CH)>(tD2 + lane_sel, va);
      tc::tmem_wait_ld();
      float *gdst = gt + (wt & 3);
      const int rch = wt >> 2;
#pragma unroll
      for (int c = 0; c < NCH; ++c) {
        uint32_t *cur = (c & 1) ? vb : va, *nxt = (c & 1) ? va : vb;
        if (c + 1 < NCH) {
          if (L::N2 - (c + 1) * CH >= CH) tc::tmem_ld_cols_nowait<CH>(tD2 + lane_sel + (c + 1) * CH, nxt);
          else tc::tmem_ld_cols_nowait<(L::N2 % CH == 0 ? CH : L::N2 % CH)>(tD2 + lane_sel + (c + 1) * CH, nxt);
        }
#pragma unroll
        for (int j = 0; j < CH; ++j) {
          const int o = c * CH + j;
          if (o < 4 * S1)
            gdst[o * 128 + ((rch ^ (o & 7)) << 2)] =
                h1[o % (2 * S1)] + tc::tanh_prescaled_f32(fmaf(__uint_as_float(cur[j]), TC_2LOG2E, vec[L::sb2 + o]));
        }
        if (c + 1 < NCH) tc::tmem_wait_ld();
      }
    }
    TCP(7);
    tc::fence_before_sync();
    tc::bar_sync(1 + wg, 128);
    TCP(8);
    // prefetch the next tile's pair (two dependent global loads) behind the accumulation below
    {
      const int tn = tile + gridDim.x * 2, pn = flat0 + tn * 128 + wt;
      nx_valid = tn < ntiles && pn < flat1;
      if (nx_valid) {
        const int idx = pidx_t[pn];
        nx_dv = C.dr[idx];
        nx_qa = idx / P.nm;
        nx_o0 = off_t[nx_qa]; nx_o1 = off_t[nx_qa + 1];
      }
    }
    // S5: T_i += sum_rows g (x) R~.  Thread b owns feature b; rows are grouped by centre atom (segments, from the pair
    // offsets).  Four rows per step: one 16-byte load of gT, four broadcast loads of R~ rows (e0..e3 adjacent), eight
    // packed FMAs (FFMA2); products and partial sums of up to 8 rows in fp32, accumulation across them in fp64
    // (DESIGN.md "Mixed precision"); steps cut by a segment boundary take the masked path.
    if (wt < 4 * S1) {
      const int b = wt;
      const float4 *grow = reinterpret_cast<const float4 *>(gt + b * 128);
      const float4 *et = reinterpret_cast<const float4 *>(envt);       // [128]: R~ row of tile row r
      const int sw = b & 7;
      int row = 0;
      float2 s01 = make_float2(0.f, 0.f), s23 = s01;
      double a0, a1, a2, a3;
      auto step = [&](int k, const float4 g4) {
        const float4 r0 = et[4 * k], r1 = et[4 * k + 1], r2 = et[4 * k + 2], r3 = et[4 * k + 3];
        s01 = tc::ffma2(make_float2(g4.x, g4.x), make_float2(r0.x, r0.y), s01);
        s23 = tc::ffma2(make_float2(g4.x, g4.x), make_float2(r0.z, r0.w), s23);
        s01 = tc::ffma2(make_float2(g4.y, g4.y), make_float2(r1.x, r1.y), s01);
        s23 = tc::ffma2(make_float2(g4.y, g4.y), make_float2(r1.z, r1.w), s23);
        s01 = tc::ffma2(make_float2(g4.z, g4.z), make_float2(r2.x, r2.y), s01);
        s23 = tc::ffma2(make_float2(g4.z, g4.z), make_float2(r2.z, r2.w), s23);
        s01 = tc::ffma2(make_float2(g4.w, g4.w), make_float2(r3.x, r3.y), s01);
        s23 = tc::ffma2(make_float2(g4.w, g4.w), make_float2(r3.z, r3.w), s23);
      };
      auto flush = [&]() {
        a0 += (double)s01.x; a1 += (double)s01.y; a2 += (double)s23.x; a3 += (double)s23.y;
        s01 = make_float2(0.f, 0.f); s23 = s01;
      };
      auto masked_step = [&](int k, int lo_row, int hi_row) {   // a step cut by a segment boundary
        float4 g4 = grow[k ^ sw];
        const int r0 = 4 * k;
        if (r0 < lo_row || r0 >= hi_row) g4.x = 0.f;
        if (r0 + 1 < lo_row || r0 + 1 >= hi_row) g4.y = 0.f;
        if (r0 + 2 < lo_row || r0 + 2 >= hi_row) g4.z = 0.f;
        if (r0 + 3 < lo_row || r0 + 3 >= hi_row) g4.w = 0.f;
        step(k, g4);
        flush();
      };
      while (row < nrows) {
        const int cur = ids[row];
        const int se = segs[row];                           // end row of this atom's segment; bit 8: whole section in the tile
        const int hi = se & 255;
        a0 = 0.0; a1 = 0.0; a2 = 0.0; a3 = 0.0;
        // whole steps [kb, ke) in a branch-free loop (two steps = 8 rows per fp64 flush); the at most two steps that a
        // segment boundary cuts go through the masked path (uniform over the warp)
        int kb = row >> 2;
        const int ke = hi >> 2;
        if (row & 3) { masked_step(kb, row, hi); ++kb; }
        if ((hi & 3) && ke >= kb) masked_step(ke, row, hi);
        int k = kb;
        for (; k + 2 <= ke; k += 2) {
          const float4 ga = grow[k ^ sw], gb = grow[(k + 1) ^ sw];
          step(k, ga);
          step(k + 1, gb);
          flush();
        }
        if (k < ke) { step(k, grow[k ^ sw]); flush(); }
        double *dst = C.T + ((size_t)cur * P.M + b) * 4;
        if (P.ntypes == 1 && (se & 256)) {
          // one net only and the whole section of this atom lies inside the tile: nobody else writes T[cur][b][:]
          double2 *d2 = reinterpret_cast<double2 *>(dst);
          d2[0] = make_double2(a0, a1);
          d2[1] = make_double2(a2, a3);
        } else {
          atomicAdd(dst + 0, a0); atomicAdd(dst + 1, a1); atomicAdd(dst + 2, a2); atomicAdd(dst + 3, a3);
        }
        row = hi;
      }
    }
    TCP(9);
    tc::bar_sync(1 + wg, 128);                              // slot, env tile and ids are rewritten by the next tile
    TCP(10);
#ifdef TC_PROF
    if (blockIdx.x == 3 && wt == 0 && tile == blockIdx.x * 2 + wg + 4 * gridDim.x * 2)
      printf("wg %d a %d t %d: env+l0 %lld bar %lld mma1 %lld ld1+tanh %lld st2 %lld mma2 %lld ld2+tanh+g %lld bar %lld Tacc %lld bar %lld\n", wg, a, t,
             tp[1]-tp[0], tp[2]-tp[1], tp[3]-tp[2], tp[4]-tp[3], tp[5]-tp[4], tp[6]-tp[5], tp[7]-tp[6], tp[8]-tp[7], tp[9]-tp[8], tp[10]-tp[9]);
#endif
  }
  }                                                         // nets
  tc::fence_before_sync();
  __syncthreads();
  if (warp == 0) tc::tmem_dealloc<512>(tmem);
}

static int g_tc_sms_d[DPB_MAX_DEVICES] = {};        // per device
#define g_tc_sms (g_tc_sms_d[dpb_device()])

template <int S1>
static cudaError_t run_pass1_tc(const DevModel &P, const ChunkView &C, const TCWeights &W, const int *off,
                                const int *pidx, cudaStream_t st) {
  using L = TL<S1>;
  static bool configured_d[DPB_MAX_DEVICES] = {};
  bool &configured = configured_d[dpb_device()];
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_pass1_tc<S1>, cudaFuncAttributeMaxDynamicSharedMemorySize, L::smem_bytes);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  k_pass1_tc<S1><<<g_tc_sms, 256, L::smem_bytes, st>>>(P, C, W.emb, W.net_stride, off, pidx);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

cudaError_t tc_pass1(const DevModel &P, const ChunkView &C, const TCWeights &W, const void *pair_ws, cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  if (!W.ready) return cudaErrorNotSupported;
  if (g_tc_sms == 0) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&g_tc_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
  }
  cudaError_t e = cudaMemsetAsync(C.T, 0, sizeof(double) * (size_t)C.n * P.M * 4, st);
  if (e != cudaSuccess) return e;
  const int *off = reinterpret_cast<const int *>(pair_ws);
  const int *pidx = off + (size_t)P.ntypes * (C.n + 1);
  switch (P.s1) {
    case 8: return run_pass1_tc<8>(P, C, W, off, pidx, st);
    case 16: return run_pass1_tc<16>(P, C, W, off, pidx, st);
    case 25: return run_pass1_tc<25>(P, C, W, off, pidx, st);
    default: return run_pass1_tc<32>(P, C, W, off, pidx, st);
  }
}

// ---- pass 2 ----------------------------------------------------------------------------------------------------
// S8 + S9 in mixed precision.  Forward-mode derivative of the embedding net (its input is the scalar s(r)): the value
// row h and the tangent row h' = dh/dx go through the same tensor-core GEMMs (separate accumulators in TMEM), then
//   dE/dR~[c] = sum_o dT[o][c] g[o],   dE/dx = sum_o (dT R~)[o] g'[o]                     (O9, fp32 dots per row)
// and the chain to the displacement (O10), the force scatter and the virial (O11, ProdForce / ProdVirial,
// PAPER.md:240) in fp64.  dT32 is the fp32 copy of dE/dT written by the fitting stage.

template <int S1>
__global__ void __launch_bounds__(256, 1)
k_pass2_tc(DevModel P, ChunkView C, const float *__restrict__ all_img, size_t net_stride,
           const int *__restrict__ off_all, const int *__restrict__ pidx_all, const float *__restrict__ dT32,
           double *__restrict__ force, double *__restrict__ virial) {
  using L = TL<S1>;
  extern __shared__ __align__(1024) uint8_t smem[];
  const int tid = threadIdx.x, wg = tid >> 7, wt = tid & 127, warp = tid >> 5, lane = tid & 31;
  const float *vec = reinterpret_cast<const float *>(smem + L::oVec);
  uint8_t *slot = smem + L::oSlot + wg * L::SLOT;
  uint64_t *mbar = reinterpret_cast<uint64_t *>(smem + L::oBar) + wg;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + L::oTmem);
  double *vred = reinterpret_cast<double *>(smem + L::oEnv);           // [8 warps][9], used after the tile loop
  int *ids = reinterpret_cast<int *>(smem + L::oIds) + wg * 256;       // centre atom of every tile row

  if (warp == 0) tc::tmem_alloc<512>(tmem_slot);
  if (tid == 0) {
    tc::mbar_init(reinterpret_cast<uint64_t *>(smem + L::oBar), 1);
    tc::mbar_init(reinterpret_cast<uint64_t *>(smem + L::oBar) + 1, 1);
    tc::fence_mbar_init();
  }
  tc::fence_proxy_async();
  tc::fence_before_sync();
  __syncthreads();
  tc::fence_after_sync();
  const uint32_t tmem = *tmem_slot;
  const uint32_t tD1v = tmem + wg * 256, tD1t = tD1v + 64, tD2v = tD1v, tD2t = tD1v + 128;
  const uint32_t tA1 = tD1v + 128;                           // layer-1 A operands: v hi, v lo, t hi, t lo, 32 columns each
  const uint32_t lane_sel = (uint32_t)(32 * (warp & 3)) << 16;
  const uint32_t slot_a = tc::smem_u32(slot), img_a = tc::smem_u32(smem);
  const uint32_t rowbase = (uint32_t)(wt >> 3) * 1024u + (uint32_t)(wt & 7) * 128u, r7 = wt & 7;

  double vir[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) vir[k] = 0.0;
  // one launch walks all ntypes^2 nets (a = centre type, t = neighbour type): the CTA reloads the weight image at a net
  // switch, so only the last net has a tail in which SMs idle (four launches per pass had four)
  uint32_t phase = 0;
  for (int net = 0; net < P.ntypes * P.ntypes; ++net) {
  const int a = net / P.ntypes, t = net - a * P.ntypes;
  const int *off_t = off_all + (size_t)t * (C.n + 1), *pidx_t = pidx_all + (size_t)C.n * P.sec_start[t];
  __syncthreads();                                          // every MMA that read the previous image has completed
  {
    const float *net_img = all_img + (size_t)net * net_stride;
    for (int k = tid; k < L::img_bytes / 16; k += 256)
      reinterpret_cast<int4 *>(smem)[k] = reinterpret_cast<const int4 *>(net_img)[k];
  }
  tc::fence_proxy_async();
  __syncthreads();
  const int row_lo = max(C.p0, C.type_start[a]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[a + 1]) - C.p0;
  int flat0 = 0, flat1 = 0;
  if (row_hi > row_lo) { flat0 = off_t[row_lo]; flat1 = off_t[row_hi]; }
  const int ntiles = (flat1 - flat0 + 127) >> 7;

  int nx_idx = 0;
  double4 nx_dv = make_double4(0.0, 0.0, 0.0, 1.0);
  bool nx_valid = false;
  {
    const int t0 = blockIdx.x * 2 + wg, p0 = flat0 + t0 * 128 + wt;
    nx_valid = t0 < ntiles && p0 < flat1;
    if (nx_valid) { nx_idx = pidx_t[p0]; nx_dv = C.dr[nx_idx]; }
  }
  for (int tile = blockIdx.x * 2 + wg; tile < ntiles; tile += gridDim.x * 2) {
    const bool valid = nx_valid;
    const int idx = nx_idx;
    const double4 dv = nx_dv;
    const int qa = valid ? idx / P.nm : -1;
    ids[wt] = qa;
    double ed[4] = {0.0, 0.0, 0.0, 0.0};
    if (valid) env_row4_tc(P, dv, ed);
    const float e0 = (float)ed[0], e1 = (float)ed[1], e2 = (float)ed[2], e3 = (float)ed[3];
    // layer 0 and its tangent: h0' = (1 - t0^2) W0   (d tanh = 1 - tanh^2)
    float h0v[32], h0t[32];
#pragma unroll
    for (int s = 0; s < 32; ++s) {
      if (s < S1) {
        const float w0 = vec[L::vW0 + s];
        float t0, d0;
        tc::tanh_d_f32(fmaf(e0, w0, vec[L::vb0 + s]), t0, d0);
        h0v[s] = t0;
        h0t[s] = d0 * w0;
      } else {
        h0v[s] = 0.0f; h0t[s] = 0.0f;
      }
    }
    // layer-1 A operands (value and tangent, hi and lo) go to tensor memory, columns [128, 256) of the warpgroup — the
    // tangent accumulator of layer 2 lives there later — and the MMAs read them from there (TS form, as in pass 1)
    {
      uint32_t w[32];
#pragma unroll
      for (int part = 0; part < 4; ++part) {
#pragma unroll
        for (int s = 0; s < 32; ++s) {
          float fh, fl;
          tc::split_tf32(part < 2 ? h0v[s] : h0t[s], fh, fl);
          w[s] = __float_as_uint((part & 1) ? fl : fh);
        }
        tc::tmem_st32_nowait(tA1 + 32 * part + lane_sel, w);
      }
      tc::tmem_wait_st();
    }
    tc::fence_before_sync();
    tc::bar_sync(1 + wg, 128);
    if (wt == 0) {
      tc::fence_after_sync();
      constexpr uint32_t idesc = tc::make_idesc_tf32(128, L::N1);
#pragma unroll
      for (int ks = 0; ks < L::KS1; ++ks) {
        const uint64_t dbh = tc::make_desc_sw128(img_a + L::oW1h + ks * 32), dbl = tc::make_desc_sw128(img_a + L::oW1l + ks * 32);
        tc::mma_tf32_ts(tD1v, tA1 + 32 + 8 * ks, dbh, idesc, ks == 0 ? 0u : 1u);      // lo hi + hi lo + hi hi
        tc::mma_tf32_ts(tD1v, tA1 + 8 * ks, dbl, idesc, 1u);
        tc::mma_tf32_ts(tD1v, tA1 + 8 * ks, dbh, idesc, 1u);
        tc::mma_tf32_ts(tD1t, tA1 + 96 + 8 * ks, dbh, idesc, ks == 0 ? 0u : 1u);
        tc::mma_tf32_ts(tD1t, tA1 + 64 + 8 * ks, dbl, idesc, 1u);
        tc::mma_tf32_ts(tD1t, tA1 + 64 + 8 * ks, dbh, idesc, 1u);
      }
      tc::mma_commit(mbar);
    }
    tc::mbar_wait(mbar, phase);
    phase ^= 1;
    tc::fence_after_sync();
    // layer 1: h1 = (h0, h0) + t1, h1' = (h0', h0') + (1 - t1^2) (h0' W1)
    float h1v[2 * S1], h1t[2 * S1];
    {
      uint32_t v[L::N1], w[L::N1];
      tc::tmem_ld_cols_nowait<L::N1>(tD1v + lane_sel, v);
      tc::tmem_ld_cols_nowait<L::N1>(tD1t + lane_sel, w);
      tc::tmem_wait_ld();
#pragma unroll
      for (int o = 0; o < 2 * S1; ++o) {
        float t1, d1;
        tc::tanh_d_f32(__uint_as_float(v[o]) + vec[L::vb1 + o], t1, d1);
        h1v[o] = h0v[o % S1] + t1;
        h1t[o] = fmaf(d1, __uint_as_float(w[o]), h0t[o % S1]);
      }
    }
    // layer 2, value rows
#pragma unroll
    for (int j = 0; j < 2 * L::KS2; ++j) {
      const int pan = j >> 3;
      auto H = [&](int o) { return o < 2 * S1 ? h1v[o] : 0.0f; };
      store_split4(slot + pan * 16384, slot + 32768 + pan * 16384, rowbase, r7, j & 7, H(4 * j), H(4 * j + 1), H(4 * j + 2),
                   H(4 * j + 3));
    }
    tc::fence_proxy_async();
    tc::fence_before_sync();
    tc::bar_sync(1 + wg, 128);
    if (wt == 0) {
      tc::fence_after_sync();
      constexpr uint32_t idesc = tc::make_idesc_tf32(128, L::N2);
#pragma unroll
      for (int ks = 0; ks < L::KS2; ++ks) {
        const uint32_t ao = (ks >> 2) * 16384 + (ks & 3) * 32, bo = (ks >> 2) * L::W2P + (ks & 3) * 32;
        mma3(tD2v, slot_a + ao, slot_a + 32768 + ao, img_a + L::oW2h + bo, img_a + L::oW2l + bo, idesc, ks == 0);
      }
      tc::mma_commit(mbar);
    }
    tc::mbar_wait(mbar, phase);
    phase ^= 1;
    tc::fence_after_sync();
    // layer 2, tangent rows (the operand slot is free again: the value MMAs have completed)
#pragma unroll
    for (int j = 0; j < 2 * L::KS2; ++j) {
      const int pan = j >> 3;
      auto H = [&](int o) { return o < 2 * S1 ? h1t[o] : 0.0f; };
      store_split4(slot + pan * 16384, slot + 32768 + pan * 16384, rowbase, r7, j & 7, H(4 * j), H(4 * j + 1), H(4 * j + 2),
                   H(4 * j + 3));
    }
    tc::fence_proxy_async();
    tc::fence_before_sync();
    tc::bar_sync(1 + wg, 128);
    if (wt == 0) {
      tc::fence_after_sync();
      constexpr uint32_t idesc = tc::make_idesc_tf32(128, L::N2);
#pragma unroll
      for (int ks = 0; ks < L::KS2; ++ks) {
        const uint32_t ao = (ks >> 2) * 16384 + (ks & 3) * 32, bo = (ks >> 2) * L::W2P + (ks & 3) * 32;
        mma3(tD2t, slot_a + ao, slot_a + 32768 + ao, img_a + L::oW2h + bo, img_a + L::oW2l + bo, idesc, ks == 0);
      }
      tc::mma_commit(mbar);
    }
    // prefetch the next tile's pair behind the MMA wait
    {
      const int tn = tile + gridDim.x * 2, pn = flat0 + tn * 128 + wt;
      nx_valid = tn < ntiles && pn < flat1;
      if (nx_valid) { nx_idx = pidx_t[pn]; nx_dv = C.dr[nx_idx]; }
    }
    // ... and the first dT rows of this tile's centre atoms (staged in the operand slot once the MMAs are done)
    const float4 *dT4 = reinterpret_cast<const float4 *>(dT32);
    constexpr int CAP_AT = L::SLOT / (4 * S1 * 16);            // atoms whose rows fit the slot
    constexpr int DT_PF = 3;                                   // float4 per thread in flight over the MMA wait
    const int nrows_t = min(128, flat1 - (flat0 + tile * 128));
    const int qa0 = ids[0];
    const int nat = min(ids[nrows_t - 1] - qa0 + 1, CAP_AT);
    const float4 *dsrc = dT4 + (size_t)qa0 * P.M;
    float4 pf[DT_PF];
#pragma unroll
    for (int u = 0; u < DT_PF; ++u) {
      const int k = wt + 128 * u;
      pf[u] = k < nat * 4 * S1 ? dsrc[k] : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    tc::mbar_wait(mbar, phase);
    phase ^= 1;
    tc::fence_after_sync();
    // The operand slot is free again (the tangent MMAs have completed): stage the dT rows of the tile's centre atoms in
    // it (coalesced), so that the epilogue reads them from shared memory — with 221 KB of shared memory in use the L1
    // holds almost nothing and the per-feature global loads were the largest phase of the tile.
    const int jn = (valid && force) ? C.nl[idx] : 0;        // neighbour index for the force scatter: loaded ahead of its use
    const int in_ = (valid && force) ? C.s_idx[C.p0 + qa] : 0;   // ... and the centre atom's own index
    float4 *stage = reinterpret_cast<float4 *>(slot);
    {
#pragma unroll
      for (int u = 0; u < DT_PF; ++u) {
        const int k = wt + 128 * u;
        if (k < nat * 4 * S1) stage[k] = pf[u];
      }
      for (int k = wt + 128 * DT_PF; k < nat * 4 * S1; k += 128) stage[k] = dsrc[k];
    }
    tc::bar_sync(1 + wg, 128);
    // epilogue: g = (h1, h1) + t2, g' = (h1', h1') + (1 - t2^2) (h1' W2); dots with the atom's dT rows
    // packed FMAs: (pr0, pr1), (pr2, pr3) += g dT[o][:]; (q0, q1), (q2, q3) += g' dT[o][:], dotted with R~ at the end
    float2 pr01 = make_float2(0.f, 0.f), pr23 = pr01, q01 = pr01, q23 = pr01;
    const bool staged = valid && qa - qa0 < nat;
    const float4 *dTrow = staged ? stage + (qa - qa0) * (4 * S1) : dT4 + (size_t)(valid ? qa : 0) * P.M;
    {
      constexpr int CH = 16, NCH = (4 * S1 + CH - 1) / CH;
#pragma unroll
      for (int c = 0; c < NCH; ++c) {
        uint32_t v[CH], w[CH];
        constexpr int dummy = 0;
        (void)dummy;
        if (L::N2 - c * CH >= CH) {
          tc::tmem_ld_cols_nowait<CH>(tD2v + lane_sel + c * CH, v);
          tc::tmem_ld_cols_nowait<CH>(tD2t + lane_sel + c * CH, w);
        } else {
          tc::tmem_ld_cols_nowait<8>(tD2v + lane_sel + c * CH, v);
          tc::tmem_ld_cols_nowait<8>(tD2t + lane_sel + c * CH, w);
        }
        tc::tmem_wait_ld();
#pragma unroll
        for (int i = 0; i < CH; ++i) {
          const int o = c * CH + i;
          if (o < 4 * S1) {
            float t2, d2;
            tc::tanh_d_f32(__uint_as_float(v[i]) + vec[L::vb2 + o], t2, d2);
            const float gv = h1v[o % (2 * S1)] + t2;
            const float gp = fmaf(d2, __uint_as_float(w[i]), h1t[o % (2 * S1)]);
            const float4 d4 = dTrow[o];
            pr01 = tc::ffma2(make_float2(gv, gv), make_float2(d4.x, d4.y), pr01);
            pr23 = tc::ffma2(make_float2(gv, gv), make_float2(d4.z, d4.w), pr23);
            q01 = tc::ffma2(make_float2(gp, gp), make_float2(d4.x, d4.y), q01);
            q23 = tc::ffma2(make_float2(gp, gp), make_float2(d4.z, d4.w), q23);
          }
        }
      }
    }
    tc::fence_before_sync();                                // TMEM reads done before the next tile's MMAs overwrite
    tc::bar_sync(1 + wg, 128);                              // ... and the staged dT rows before the next tile's operands
    // O10 / O11 in fp64: f_ik = sum_m dR~[m] dR~_m/dd; F_j -= f, F_i += f, Xi -= d (x) f
    double f0 = 0.0, f1 = 0.0, f2 = 0.0;
    if (valid) {
      const double r = dv.w, ir = 1.0 / r;
      double w, dw;
      dp_switch(r, P.rcs, P.rc, w, dw);
      const double s = w * ir, qq = s * ir;
      const double sp = dw * ir - w * ir * ir;
      const double qp = sp * ir - s * ir * ir;
      const float dx = fmaf(q01.x, e0, fmaf(q01.y, e1, fmaf(q23.x, e2, q23.y * e3)));
      const double dR0 = (double)pr01.x + (double)dx, dR1 = (double)pr01.y, dR2 = (double)pr23.x, dR3 = (double)pr23.y;
      const double dot = dR1 * dv.x + dR2 * dv.y + dR3 * dv.z;
      const double cm = (dR0 * sp + qp * dot) * ir;
      f0 = fma(cm, dv.x, qq * dR1); f1 = fma(cm, dv.y, qq * dR2); f2 = fma(cm, dv.z, qq * dR3);
      if (force) {
        const int j = jn;
        atomicAdd(&force[3 * (size_t)j + 0], -f0);
        atomicAdd(&force[3 * (size_t)j + 1], -f1);
        atomicAdd(&force[3 * (size_t)j + 2], -f2);
      }
      vir[0] -= dv.x * f0; vir[1] -= dv.x * f1; vir[2] -= dv.x * f2;
      vir[3] -= dv.y * f0; vir[4] -= dv.y * f1; vir[5] -= dv.y * f2;
      vir[6] -= dv.z * f0; vir[7] -= dv.z * f1; vir[8] -= dv.z * f2;
    }
    // F_i += sum_k f_ik: rows of one atom are contiguous lanes -> segmented warp reduction, one RED per run head
    if (force) {
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const int qo = __shfl_down_sync(0xffffffffu, qa, off);
        const double g0 = __shfl_down_sync(0xffffffffu, f0, off), g1 = __shfl_down_sync(0xffffffffu, f1, off),
                     g2 = __shfl_down_sync(0xffffffffu, f2, off);
        if (lane + off < 32 && qo == qa) { f0 += g0; f1 += g1; f2 += g2; }
      }
      const int qprev = __shfl_up_sync(0xffffffffu, qa, 1);
      if (valid && (lane == 0 || qprev != qa)) {
        const size_t i = (size_t)in_;
        atomicAdd(&force[3 * i + 0], f0); atomicAdd(&force[3 * i + 1], f1); atomicAdd(&force[3 * i + 2], f2);
      }
    }
  }
  }                                                         // nets
  // virial: warp -> block -> one atomic per component and CTA
#pragma unroll
  for (int k = 0; k < 9; ++k) {
    double v = vir[k];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if (lane == 0) vred[warp * 9 + k] = v;
  }
  tc::fence_before_sync();
  __syncthreads();
  if (tid < 9 && virial) {
    double v = 0.0;
    for (int w = 0; w < 8; ++w) v += vred[w * 9 + tid];
    atomicAdd(&virial[tid], v);
  }
  if (warp == 0) tc::tmem_dealloc<512>(tmem);
}

size_t tc_pass2_workspace_bytes(const DevModel &P, int64_t chunk) { return sizeof(float) * (size_t)chunk * P.M * 4 + 256; }

template <int S1>
static cudaError_t run_pass2_tc(const DevModel &P, const ChunkView &C, const TCWeights &W, const int *off,
                                const int *pidx, const float *dT32, double *force, double *virial, cudaStream_t st) {
  using L = TL<S1>;
  static bool configured_d[DPB_MAX_DEVICES] = {};
  bool &configured = configured_d[dpb_device()];
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_pass2_tc<S1>, cudaFuncAttributeMaxDynamicSharedMemorySize, L::smem_bytes);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  k_pass2_tc<S1><<<g_tc_sms, 256, L::smem_bytes, st>>>(P, C, W.emb, W.net_stride, off, pidx, dT32, force, virial);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

cudaError_t tc_pass2(const DevModel &P, const ChunkView &C, const TCWeights &W, const void *pair_ws, const float *dT32,
                     double *force, double *virial, cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  if (!W.ready) return cudaErrorNotSupported;
  const int *off = reinterpret_cast<const int *>(pair_ws);
  const int *pidx = off + (size_t)P.ntypes * (C.n + 1);
  switch (P.s1) {
    case 8: return run_pass2_tc<8>(P, C, W, off, pidx, dT32, force, virial, st);
    case 16: return run_pass2_tc<16>(P, C, W, off, pidx, dT32, force, virial, st);
    case 25: return run_pass2_tc<25>(P, C, W, off, pidx, dT32, force, virial, st);
    default: return run_pass2_tc<32>(P, C, W, off, pidx, dT32, force, virial, st);
  }
}
