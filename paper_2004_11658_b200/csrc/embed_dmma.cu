// embed_dmma.cu — variant 1 of S3+S4+S5 (pass 1) and S8+S9 (pass 2): the embedding net on fp64 tensor-core tiles
// (mma.sync m8n8k4 = SASS DMMA.8x8x4, the only fp64 MMA primitive of sm_100a; tcgen05 has no f64 kind), fused with
// the env matrix, the G^T R~ reduction and the force / virial chain so that G never leaves the SM.
//
// Fragment layout of m8n8k4 (g = lane / 4, q = lane % 4):  A[row g][k q]   B[k q][col g]   C[row g][cols 2q, 2q+1].
// Rows are neighbours.  The output of one layer (C layout: thread (g, q) holds, for n-block nb, the columns 2q and
// 2q+1, called "slots" 2nb and 2nb+1 of lane quarter q) feeds the next layer as A operand WITHOUT any shuffle: the
// k-step `ks` of the next GEMM takes, from lane quarter q, its slot ks — a permutation of the contraction index that
// the weight rows follow.  Features are placed so that the concat skip [x || x] of Eq. 9 stays inside the thread:
//   feature o of a layer of width 2^l s1:  copy c = o / s1, r = o % s1  ->  quarter q = r % 4, slot = c * SP + r / 4,
// with SP = ceil(s1 / 4) slots per copy (pads are zero weights, zero bias: their activations are exactly 0).
// The padded weight matrices in shared memory are  W_l[4 * ks + q][8 * nb + 2 q' + e]  (input slot ks of quarter q,
// output slot 2 nb + e of quarter q'), leading dimension = 4 (mod 16) doubles so that B-fragment loads are
// conflict-free.
//
// Pass 2 differentiates the embedding net in forward mode: its input is the scalar s(r), so the tangent row
// h' = dh/dx runs through the same GEMM chain as the value row (second m-block, same B fragments), and
//   dE/dx = sum_o (dT R~)[o] g'[o],   dE/dR~[c] = sum_o dT[o][c] g[o]          (O9 of DESIGN.md / SURVEY.md §8(c)).
//
// Kernels: k_pass1_dmma<SP, RB, RU> (RU: same-species pair reuse, T_j += g (x) R~_ji by fp64 reductions),
// k_pass2_dmma<SP> and k_pass2_dmma_ru<SP> (pair reuse: the second direction reads dT_j slices staged by the TMA
// engine), k_pass2_dmma_st<SP, SA> (row stream over the atoms a warp takes; SA: the tanh outputs of the value chain are
// read from the records pass 1 stored, ChunkView::act, and only the tangent chain runs).  One launch per net; a warp takes work items (atom, or a segment of an atom's rows for small chunks) from a
// counter in global memory; the net's weights are staged by one TMA bulk copy per CTA.  DESIGN.md sections 6 and 12.
#include "v1_kernels.cuh"
#include "tc_common.cuh"

#include <vector>

#ifndef P1_WARPS
#define P1_WARPS 12           // warps per CTA, pass 1 (168 registers; 8 warps at 204-218: 3-4 % slower, 16: no better)
#endif
#ifndef P2_WARPS
#define P2_WARPS 8            // warps per CTA, pass 2
#endif

__device__ __forceinline__ void dmma884(double &c0, double &c1, const double a, const double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int SP>
struct EL {
  static constexpr int S0 = SP, S1 = 2 * SP, S2 = 4 * SP;
  static constexpr int NB1 = SP, NB2 = 2 * SP;
  static constexpr int LD1 = 8 * NB1 + 4, LD2 = 8 * NB2 + 4;
  static constexpr int oW0 = 0;                          // [4 SP]  position 4 s + q
  static constexpr int ob0 = 4 * SP;                     // [4 SP]
  static constexpr int oW1 = 8 * SP;                     // [4 SP][LD1]
  static constexpr int ob1 = oW1 + 4 * SP * LD1;         // [8 NB1]
  static constexpr int oW2 = ob1 + 8 * NB1;              // [8 SP][LD2]
  static constexpr int ob2 = oW2 + 8 * SP * LD2;         // [8 NB2]
  static constexpr int total = ob2 + 8 * NB2;
  static constexpr int LDG = 8 * SP + 4;                 // leading dimension of the per-warp g tile (one N chunk)
  static constexpr int tile1 = 16 * LDG + 16 * 4;        // pass 1, per warp: g tile [16][LDG] + env tile [16][4] (RB = 2)
  static constexpr int tile1s = 8 * LDG + 8 * 4;         // same for RB = 1
  static constexpr int tile2 = 16 * SP * 4;              // pass 2, per warp: dT tile [16 SP][4]
  // Stored activations (ChunkView::act): per row and lane quarter q the tanh outputs t0 [SP] (padded to an even count),
  // t1 [2 SP], t2 [4 SP] in slot order; element e of quarter q at (e / 2) * 8 + 2 q + e % 2, so that one 16-byte access
  // per lane covers 64 contiguous bytes per row (8 rows: 512 bytes per warp instruction).
  static constexpr int A0 = (SP + 1) & ~1;               // elements of t0 per lane
  static constexpr int AE = A0 + 6 * SP;                 // elements per lane
  static constexpr int REC = 4 * AE;                     // doubles per record
};

// streaming (evict-first) 16-byte accesses to the activation records: written once, read once, never reused — they must
// not push the dT tiles and the lists out of L2
__device__ __forceinline__ void act_store(double *p, const double a, const double b) {
  __stcs(reinterpret_cast<double2 *>(p), make_double2(a, b));
}
__device__ __forceinline__ double2 act_load(const double *p) { return __ldcs(reinterpret_cast<const double2 *>(p)); }
// one instruction of the TMA engine brings a whole record (bytes: multiple of 16) from DRAM into L2
__device__ __forceinline__ void act_prefetch(const double *p, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(p), "r"(bytes) : "memory");
}

// Row staging of the embedding passes: the (d, r) rows and neighbour indices of the next 32 slots are copied global ->
// shared with cp.async (no registers in flight) while the current 32 are processed, so that no 8-row block starts with
// a global-load round trip.  Per warp: 2 buffers x 32 rows x (32 B + 4 B).
#define EMB_STG 288                                        // doubles per warp: 2 x 32 double4 + 2 x 32 int
__device__ __forceinline__ void emb_cp16(void *smem_dst, const void *gsrc) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc));
}
__device__ __forceinline__ void emb_cp4(void *smem_dst, const void *gsrc) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc));
}
__device__ __forceinline__ void emb_cp_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void emb_cp_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }


// The net's padded weights (EL<SP>::total doubles: 67 KB for 25-50-100, 87 KB for 32-64-128) go global -> shared as ONE
// bulk copy of the TMA engine (cp.async.bulk, completion on an mbarrier): one memory round trip per CTA instead of a
// loop of dependent loads — what a 192-atom evaluation with a cold L2 waits for.
__device__ __forceinline__ void stage_net(double *W, const double *__restrict__ netp, int total, uint64_t *mbar) {
  if (threadIdx.x == 0) {
    tc::mbar_init(mbar, 1);
    tc::fence_mbar_init();
    tc::mbar_arrive_expect_tx(mbar, (unsigned)total * 8u);
    tc::bulk_g2s(W, netp, (unsigned)total * 8u, mbar);
  }
  __syncthreads();                                       // the initialised barrier is visible to every waiter
  tc::mbar_wait(mbar, 0);
}

// Work items are handed out dynamically: a warp takes the next (atom, segment) from a counter in global memory.  A static
// round-robin leaves a tail of 1 / (items per warp) — 15-20 % for the 8,192 oxygen atoms of the water box on 148 x 12 warps
// — and the pair reuse makes the items unequal (an atom evaluates between none and all of its same-species pairs).
__device__ __forceinline__ int next_item(int *counter, int lane) {
  int v = 0;
  if (lane == 0) v = atomicAdd(counter, 1);
  return __shfl_sync(0xffffffffu, v, 0);
}

static int sp_for(int s1) {
  if (s1 <= 8) return 2;
  if (s1 <= 16) return 4;
  if (s1 <= 28) return 7;
  if (s1 <= 32) return 8;
  return 0;                                              // wider nets: variant 0 kernels
}

// feature index held by (quarter q, slot s) of a layer with `copies` copies of s1, or -1 for a pad
static inline int feat_of(int q, int s, int SP, int s1, int copies) {
  const int c = s / SP, r = (s % SP) * 4 + q;
  if (c >= copies || r >= s1) return -1;
  return c * s1 + r;
}

template <int SP>
static void pack_net(const double *net, int s1, std::vector<double> &out) {
  using L = EL<SP>;
  out.assign(L::total, 0.0);
  const double *W0 = net, *b0 = W0 + s1, *W1 = b0 + s1, *b1 = W1 + (size_t)s1 * 2 * s1, *W2 = b1 + 2 * s1,
               *b2 = W2 + (size_t)2 * s1 * 4 * s1;
  for (int s = 0; s < SP; ++s)
    for (int q = 0; q < 4; ++q) {
      const int f = feat_of(q, s, SP, s1, 1);
      if (f >= 0) { out[L::oW0 + 4 * s + q] = W0[f]; out[L::ob0 + 4 * s + q] = b0[f]; }
    }
  for (int nb = 0; nb < L::NB1; ++nb)
    for (int qo = 0; qo < 4; ++qo)
      for (int e = 0; e < 2; ++e) {
        const int fo = feat_of(qo, 2 * nb + e, SP, s1, 2), col = 8 * nb + 2 * qo + e;
        if (fo < 0) continue;
        out[L::ob1 + col] = b1[fo];
        for (int ks = 0; ks < SP; ++ks)
          for (int q = 0; q < 4; ++q) {
            const int fi = feat_of(q, ks, SP, s1, 1);
            if (fi >= 0) out[L::oW1 + (4 * ks + q) * L::LD1 + col] = W1[(size_t)fi * 2 * s1 + fo];
          }
      }
  for (int nb = 0; nb < L::NB2; ++nb)
    for (int qo = 0; qo < 4; ++qo)
      for (int e = 0; e < 2; ++e) {
        const int fo = feat_of(qo, 2 * nb + e, SP, s1, 4), col = 8 * nb + 2 * qo + e;
        if (fo < 0) continue;
        out[L::ob2 + col] = b2[fo];
        for (int ks = 0; ks < 2 * SP; ++ks)
          for (int q = 0; q < 4; ++q) {
            const int fi = feat_of(q, ks, SP, s1, 2);
            if (fi >= 0) out[L::oW2 + (4 * ks + q) * L::LD2 + col] = W2[(size_t)fi * 4 * s1 + fo];
          }
      }
}

cudaError_t v1_prepare_weights(const DevModel &P, const double *emb_h, const double *fit_h, V1Weights &W) {
  W.SP = sp_for(P.s1);
  W.ready = false;
  if (W.SP == 0) return cudaSuccess;
  {
    cudaError_t ef = v1_prepare_fit(P, fit_h, W);
    if (ef != cudaSuccess) return ef;
  }
  std::vector<double> one, all;
  const int nets = P.ntypes * P.ntypes;
  for (int k = 0; k < nets; ++k) {
    const double *net = emb_h + (size_t)k * P.emb_net_size;
    switch (W.SP) {
      case 2: pack_net<2>(net, P.s1, one); break;
      case 4: pack_net<4>(net, P.s1, one); break;
      case 7: pack_net<7>(net, P.s1, one); break;
      default: pack_net<8>(net, P.s1, one); break;
    }
    W.net_stride = (long long)one.size();
    all.insert(all.end(), one.begin(), one.end());
  }
  cudaError_t e = cudaMalloc(&W.emb, sizeof(double) * all.size());
  if (e != cudaSuccess) return e;
  e = cudaMemcpy(W.emb, all.data(), sizeof(double) * all.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return e;
  W.ready = true;
  return cudaSuccess;
}

void v1_release_weights(V1Weights &W) {
  v1_release_fit(W);
  if (W.emb) cudaFree(W.emb);
  W.emb = nullptr;
  W.ready = false;
}

// Env-matrix row (Eq. 5) from the stored (d, r) of a real slot.
__device__ __forceinline__ void env_row4(const DevModel &P, const double4 v, double e[4]) {
  double w, dw;
  dp_switch(v.w, P.rcs, P.rc, w, dw);
  const double ir = 1.0 / v.w;
  const double s = w * ir;
  const double sr = s * ir;
  e[0] = s; e[1] = sr * v.x; e[2] = sr * v.y; e[3] = sr * v.z;
}

// ---------------------------------------------------------------------------------------------------------
// Pass 1.  One launch per (centre type a, neighbour type t): the CTA keeps net (a, t) in shared memory, each warp
// takes atoms of type a round-robin and walks the real slots of section t in blocks of 8 * RB rows (RB m-blocks that
// share every B fragment).  T_i is accumulated in registers (lane-owned features) through a per-warp g tile.
// RB = 1 keeps the fully unrolled loop body inside the instruction cache (RB = 2 measured 49 % stall_no_inst).
// RU (launched for the nets (a, a) when C.reuse): same-species pair reuse.  g depends on s(r_ij) = s(r_ji) only, so of
// the two directions of a pair whose atoms are both centres of this chunk only the atom with the lower row evaluates
// the embedding net; it adds g (x) R~_ik to its own T_i and g (x) R~_ki = g (x) (s, -s d/r) to T_k with warp-coalesced
// red.global.add.f64 (580 G/s measured, profiles/r1_fp64_peaks.md).  T rows are zeroed by the launcher and every
// accumulation of this launch into T is a reduction.  Taken only while no neighbour was dropped (n_overflow == 0).
template <int SP, int RB, bool RU>
__global__ void __launch_bounds__((32 * P1_WARPS), 1)
k_pass1_dmma(DevModel P, ChunkView C, const double *__restrict__ netp, int a, int t, int accumulate, int nseg,
             int *counter) {
  using L = EL<SP>;
  extern __shared__ __align__(16) double smem[];
  double *W = smem;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, q = lane & 3;
  double *gt = smem + ((L::total + 1) & ~1) + warp * (RB == 1 ? L::tile1s : L::tile1);     // [8 RB][LDG]
  double *envt = gt + 8 * RB * L::LDG;                             // [8 RB][4]
  // RU: per warp, the kept slots of the atom (slot index, row of the neighbour inside the chunk or -1)
  int *ksl = reinterpret_cast<int *>(smem + ((L::total + 1) & ~1) + P1_WARPS * (RB == 1 ? L::tile1s : L::tile1)) +
             warp * 2 * P.nm;
  int *krow = ksl + P.nm;
  const bool ru = RU && C.stats->n_overflow == 0ull;
  const bool store_act = C.act != nullptr && nseg == 1;     // pass 2 reads the records only when items are whole atoms
  // RU: offset inside a T tile of the element this lane adds in step k of N chunk ch (position p = lane / 4 + 8 k of
  // the g tile, component lane % 4), or -1 for a pad
  int toff[RU ? 2 : 1][RU ? SP : 1];
  if (RU) {
#pragma unroll
    for (int ch = 0; ch < 2; ++ch)
#pragma unroll
      for (int k = 0; k < SP; ++k) {
        const int p = (lane >> 2) + 8 * k, sg = ch * 2 * SP + (p >> 2), c = sg / SP, r = (sg % SP) * 4 + (p & 3);
        toff[ch][k] = r < P.s1 ? (c * P.s1 + r) * 4 + (lane & 3) : -1;
      }
  }
  __shared__ uint64_t wbar;
  stage_net(W, netp, L::total, &wbar);
  const double *W0p = W + L::oW0, *b0p = W + L::ob0, *W1p = W + L::oW1, *b1p = W + L::ob1, *W2p = W + L::oW2,
               *b2p = W + L::ob2;
  const int row_lo = max(C.p0, C.type_start[a]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[a + 1]) - C.p0;
  const int s1 = P.s1, M = P.M;

  // work item = (atom, segment of its section): nseg > 1 splits the rows of an atom over several warps when the chunk has
  // too few atoms to fill the GPU (configs[0]: 192 atoms); T is then accumulated with reductions (accumulate == 2)
  for (int item = next_item(counter, lane); item < (row_hi - row_lo) * nseg; item = next_item(counter, lane)) {
    const int qa = row_lo + item / nseg;
    int n = C.nreal[(size_t)qa * P.ntypes + t];
    int s_lo = 0;
    if (nseg > 1) {
      const int rs = (((n + nseg - 1) / nseg) + 7) & ~7;
      s_lo = min(n, (item % nseg) * rs);
      n = min(n, s_lo + rs);
    }
    if (s_lo >= n && accumulate) continue;               // (store mode still has to write the zero tile)
    const double4 *dr = C.dr + (size_t)qa * P.nm + P.sec_start[t];
    if (RU && ru) {                                      // keep the slots whose pair this atom evaluates
      // the sorted positions of the neighbours (written by k_nlist next to their input indices): the loads of up to
      // eight 32-slot batches are issued together — one memory latency per atom instead of two dependent ones per batch
      const int *nlpr = C.nlp + (size_t)qa * P.nm + P.sec_start[t];
      int nk = 0;
      __syncwarp();
      for (int base0 = s_lo; base0 < n; base0 += 256) {
        int pj[8];
#pragma unroll
        for (int b = 0; b < 8; ++b) {
          const int slot = base0 + 32 * b + lane;
          pj[b] = slot < n ? nlpr[slot] - C.p0 : -1;
        }
#pragma unroll
        for (int b = 0; b < 8; ++b) {
          const int slot = base0 + 32 * b + lane;
          if (base0 + 32 * b >= n) break;
          int qj = pj[b];
          if (qj < 0 || qj >= C.n) qj = -1;              // not a centre of this chunk (other chunk, ghost): one direction
          const bool keep = slot < n && (qj < 0 || qj > qa);
          const unsigned mk = __ballot_sync(0xffffffffu, keep);
          if (keep) {
            const int pos = nk + __popc(mk & ((1u << lane) - 1u));
            ksl[pos] = slot; krow[pos] = qj;
          }
          nk += __popc(mk);
        }
      }
      n = nk;
      __syncwarp();
    } else {
      dr += s_lo;
      n -= s_lo;
    }
    double Tacc[2][2][4];
#pragma unroll
    for (int ch = 0; ch < 2; ++ch)
#pragma unroll
      for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int c = 0; c < 4; ++c) Tacc[ch][u][c] = 0.0;

    // the (d, r) row of the NEXT block is fetched while this one is computed: no block starts with a global round trip
    double4 dvn[RB];
#pragma unroll
    for (int rb = 0; rb < RB; ++rb) {
      const int row = g + 8 * rb;
      dvn[rb] = make_double4(0.0, 0.0, 0.0, 1.0);
      if (row < n) dvn[rb] = dr[(RU && ru) ? ksl[row] : row];
    }
    for (int r0 = 0; r0 < n; r0 += 8 * RB) {
      double x[RB];
      double *recp[RB];                                  // this lane's piece of the row's activation record, or nullptr
#pragma unroll
      for (int rb = 0; rb < RB; ++rb) {
        const int row = r0 + g + 8 * rb;
        double e[4] = {0.0, 0.0, 0.0, 0.0};
        const double4 dvc = dvn[rb];
        {
          const int rown = row + 8 * RB;
          if (rown < n) dvn[rb] = dr[(RU && ru) ? ksl[rown] : rown];
        }
        recp[rb] = nullptr;
        if (store_act && row < n)
          recp[rb] = C.act + ((size_t)qa * P.nm + P.sec_start[t] + ((RU && ru) ? ksl[row] : s_lo + row)) * L::REC + 2 * q;
        if (row < n) env_row4(P, dvc, e);
        x[rb] = e[0];
        if (q == 0) {
          double *dst = envt + (g + 8 * rb) * 4;
          dst[0] = e[0]; dst[1] = e[1]; dst[2] = e[2]; dst[3] = e[3];
        }
      }
      // layer 0 (Eq. 8): h0 = tanh(x W0 + b0)
      double h0[RB][SP];
#pragma unroll
      for (int s = 0; s < SP; ++s) {
        const double w0 = W0p[4 * s + q], bb = b0p[4 * s + q];
#pragma unroll
        for (int rb = 0; rb < RB; ++rb) h0[rb][s] = dp_tanh(fma(x[rb], w0, bb));
      }
#pragma unroll
      for (int rb = 0; rb < RB; ++rb)
        if (recp[rb]) {
#pragma unroll
          for (int s = 0; s < SP; s += 2) act_store(recp[rb] + 4 * s, h0[rb][s], s + 1 < SP ? h0[rb][s + 1] : 0.0);
        }
      // layer 1 (Eq. 9): h1 = (h0, h0) + tanh(h0 W1 + b1)
      double h1[RB][2 * SP];
#pragma unroll
      for (int nb = 0; nb < L::NB1; ++nb) {
        const double2 bb = *reinterpret_cast<const double2 *>(b1p + 8 * nb + 2 * q);
#pragma unroll
        for (int rb = 0; rb < RB; ++rb) { h1[rb][2 * nb] = bb.x; h1[rb][2 * nb + 1] = bb.y; }
      }
#pragma unroll
      for (int ks = 0; ks < SP; ++ks) {
#pragma unroll
        for (int nb = 0; nb < L::NB1; ++nb) {
          const double b = W1p[(4 * ks + q) * L::LD1 + 8 * nb + g];
#pragma unroll
          for (int rb = 0; rb < RB; ++rb) dmma884(h1[rb][2 * nb], h1[rb][2 * nb + 1], h0[rb][ks], b);
        }
      }
#pragma unroll
      for (int s = 0; s < 2 * SP; s += 2)
#pragma unroll
        for (int rb = 0; rb < RB; ++rb) {
          const double ta = dp_tanh(h1[rb][s]), tb = dp_tanh(h1[rb][s + 1]);
          if (recp[rb]) act_store(recp[rb] + 4 * (L::A0 + s), ta, tb);
          h1[rb][s] = h0[rb][s % SP] + ta;
          h1[rb][s + 1] = h0[rb][(s + 1) % SP] + tb;
        }
      // layer 2 (Eq. 9) in two N chunks of SP n-blocks: g = (h1, h1) + tanh(h1 W2 + b2); T += g (x) R~
#pragma unroll
      for (int ch = 0; ch < 2; ++ch) {
        double acc[RB][2 * SP];
#pragma unroll
        for (int nb = 0; nb < SP; ++nb) {
          const double2 bb = *reinterpret_cast<const double2 *>(b2p + 8 * (ch * SP + nb) + 2 * q);
#pragma unroll
          for (int rb = 0; rb < RB; ++rb) { acc[rb][2 * nb] = bb.x; acc[rb][2 * nb + 1] = bb.y; }
        }
#pragma unroll
        for (int ks = 0; ks < 2 * SP; ++ks) {
#pragma unroll
          for (int nb = 0; nb < SP; ++nb) {
            const double b = W2p[(4 * ks + q) * L::LD2 + 8 * (ch * SP + nb) + g];
#pragma unroll
            for (int rb = 0; rb < RB; ++rb) dmma884(acc[rb][2 * nb], acc[rb][2 * nb + 1], h1[rb][ks], b);
          }
        }
        __syncwarp();                                    // previous chunk's T update has finished reading gt
        // slot ch*2SP + s of layer 2 takes its skip from slot s of layer 1 (same copy structure)
#pragma unroll
        for (int s = 0; s < 2 * SP; s += 2)
#pragma unroll
          for (int rb = 0; rb < RB; ++rb) {
            const double ta = dp_tanh(acc[rb][s]), tb = dp_tanh(acc[rb][s + 1]);
            if (recp[rb]) act_store(recp[rb] + 4 * (L::A0 + 2 * SP + ch * 2 * SP + s), ta, tb);
            gt[(g + 8 * rb) * L::LDG + 4 * s + q] = h1[rb][s] + ta;
            gt[(g + 8 * rb) * L::LDG + 4 * (s + 1) + q] = h1[rb][s + 1] + tb;
          }
        __syncwarp();
#pragma unroll
        for (int row = 0; row < 8 * RB; ++row) {
          const double4 e4a = *reinterpret_cast<const double4 *>(envt + row * 4);
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            const int p = lane + 32 * u;
            if (p < 8 * SP) {
              const double gv = gt[row * L::LDG + p];
              Tacc[ch][u][0] = fma(gv, e4a.x, Tacc[ch][u][0]);
              Tacc[ch][u][1] = fma(gv, e4a.y, Tacc[ch][u][1]);
              Tacc[ch][u][2] = fma(gv, e4a.z, Tacc[ch][u][2]);
              Tacc[ch][u][3] = fma(gv, e4a.w, Tacc[ch][u][3]);
            }
          }
        }
        if (RU && ru) {                                  // T_k += g (x) R~_ki, 8 positions x 4 components per instruction
          // The phase must be SHORT: while a warp is in it, it feeds the fp64 pipe nothing.  Row targets come from one
          // load per lane + shuffles, and all shared-memory loads of a row (its R~ component, SP values of g) are issued
          // before the first reduction (the compiler keeps loads behind atomics in program order).
          const int comp = lane & 3;
          const int myq = (lane < 8 * RB && r0 + lane < n) ? krow[r0 + lane] : -1;
#pragma unroll 2
          for (int row = 0; row < 8 * RB; ++row) {
            const int qj = __shfl_sync(0xffffffffu, myq, row);
            if (qj < 0) continue;
            const double e0 = envt[row * 4 + comp];
            const double *gr = gt + row * L::LDG + (lane >> 2);
            double gv[SP];
#pragma unroll
            for (int k = 0; k < SP; ++k) gv[k] = gr[8 * k];
            const double ev = comp == 0 ? e0 : -e0;
            double *Tj = C.T + (size_t)qj * M * 4;
#pragma unroll
            for (int k = 0; k < SP; ++k) {
              const int o = toff[ch][k];
              if (o >= 0) atomicAdd(Tj + o, gv[k] * ev);
            }
          }
        }
      }
      __syncwarp();                                      // envt / gt are rewritten by the next row block
    }
    // T_i rows of the lane-owned features (position p = 4 s + q inside chunk ch)
#pragma unroll
    for (int ch = 0; ch < 2; ++ch)
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int p = lane + 32 * u;
        if (p < 8 * SP) {
          const int s = ch * 2 * SP + (p >> 2), qq = p & 3;
          const int c = s / SP, r = (s % SP) * 4 + qq;
          if (r < s1) {
            double *dst = C.T + ((size_t)qa * M + c * s1 + r) * 4;
            if ((RU && ru) || accumulate == 2) {
              atomicAdd(dst + 0, Tacc[ch][u][0]); atomicAdd(dst + 1, Tacc[ch][u][1]);
              atomicAdd(dst + 2, Tacc[ch][u][2]); atomicAdd(dst + 3, Tacc[ch][u][3]);
            } else if (accumulate) {
              dst[0] += Tacc[ch][u][0]; dst[1] += Tacc[ch][u][1]; dst[2] += Tacc[ch][u][2]; dst[3] += Tacc[ch][u][3];
            } else {
              dst[0] = Tacc[ch][u][0]; dst[1] = Tacc[ch][u][1]; dst[2] = Tacc[ch][u][2]; dst[3] = Tacc[ch][u][3];
            }
          }
        }
      }
  }
}

// ---------------------------------------------------------------------------------------------------------
// Pass 2.  Same launch structure; per warp 8 neighbours at a time: m-block 0 carries the values, m-block 1 the
// tangents d/dx.  Epilogue per N chunk: partial dots with the atom's dT tile (shared memory), quad reduction, then
// one lane per neighbour chains to the displacement (O10) and scatters force / virial (O11).
template <int SP>
__global__ void __launch_bounds__((32 * P2_WARPS), 1)
k_pass2_dmma(DevModel P, ChunkView C, const double *__restrict__ netp, int a, int t, double *__restrict__ force,
             double *__restrict__ virial, int nseg, int *counter) {
  using L = EL<SP>;
  extern __shared__ __align__(16) double smem[];
  double *W = smem;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, q = lane & 3;
  double *dTt = smem + ((L::total + 1) & ~1) + warp * L::tile2;    // [16 SP][4], position 4 s + q
  double4 *drs = reinterpret_cast<double4 *>(smem + ((L::total + 1) & ~1) + P2_WARPS * L::tile2 + warp * EMB_STG);
  int *nls = reinterpret_cast<int *>(drs + 64);
  __shared__ double vred[P2_WARPS][9];
  __shared__ uint64_t wbar;
  stage_net(W, netp, L::total, &wbar);
  const double *W0p = W + L::oW0, *b0p = W + L::ob0, *W1p = W + L::oW1, *b1p = W + L::ob1, *W2p = W + L::oW2,
               *b2p = W + L::ob2;
  const int row_lo = max(C.p0, C.type_start[a]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[a + 1]) - C.p0;
  double vir[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) vir[k] = 0.0;

  for (int item = next_item(counter, lane); item < (row_hi - row_lo) * nseg; item = next_item(counter, lane)) {
    const int qa = row_lo + item / nseg;                 // work item = (atom, segment of its section), as in pass 1
    int n = C.nreal[(size_t)qa * P.ntypes + t];
    int s_lo = 0;
    if (nseg > 1) {
      const int rs = (((n + nseg - 1) / nseg) + 7) & ~7;
      s_lo = min(n, (item % nseg) * rs);
      n = min(n, s_lo + rs) - s_lo;
    }
    if (n <= 0) continue;
    const double4 *dr = C.dr + (size_t)qa * P.nm + P.sec_start[t] + s_lo;
    const int *nl = C.nl + (size_t)qa * P.nm + P.sec_start[t] + s_lo;
    __syncwarp();
    {                                                    // dT is stored in lane order (ChunkView::dt_pad): a plain copy
      const double4 *src = reinterpret_cast<const double4 *>(C.dT + (size_t)qa * C.dt_rows * 4);
      for (int p = lane; p < 16 * SP; p += 32) *reinterpret_cast<double4 *>(dTt + 4 * p) = src[p];
    }
    __syncwarp();
    double fi[3] = {0.0, 0.0, 0.0};
    auto stage_rows = [&](int base, int buf) {
      const int r = base + lane;
      if (r < n) {
        emb_cp16(drs + buf * 32 + lane, dr + r);
        emb_cp16(reinterpret_cast<double *>(drs + buf * 32 + lane) + 2, reinterpret_cast<const double *>(dr + r) + 2);
        emb_cp4(nls + buf * 32 + lane, nl + r);
      }
      emb_cp_commit();
    };
    stage_rows(0, 0);

    for (int r0 = 0; r0 < n; r0 += 8) {
      if ((r0 & 31) == 0) {
        stage_rows(r0 + 32, ((r0 >> 5) + 1) & 1);        // next 32 rows in flight (possibly an empty group)
        emb_cp_wait<1>();
        __syncwarp();
      }
      const int row = r0 + g;
      const bool valid = row < n;
      const int sl = ((r0 >> 5) & 1) * 32 + (row & 31);
      double e[4] = {0.0, 0.0, 0.0, 0.0};
      double4 dv = make_double4(0.0, 0.0, 0.0, 1.0);
      int jn = 0;                                       // neighbour index for the scatter
      if (valid) { dv = drs[sl]; jn = nls[sl]; env_row4(P, dv, e); }
      // layer 0 and its tangent: h0' = (1 - t0^2) W0   (d tanh = 1 - tanh^2)
      double h0v[SP], h0t[SP];
#pragma unroll
      for (int s = 0; s < SP; ++s) {
        const double w0 = W0p[4 * s + q], bb = b0p[4 * s + q];
        const double t0 = dp_tanh(fma(e[0], w0, bb));
        h0v[s] = t0;
        h0t[s] = fma(-t0, t0, 1.0) * w0;
      }
      double h1v[2 * SP], h1t[2 * SP];
#pragma unroll
      for (int nb = 0; nb < L::NB1; ++nb) {
        const double2 bb = *reinterpret_cast<const double2 *>(b1p + 8 * nb + 2 * q);
        h1v[2 * nb] = bb.x; h1v[2 * nb + 1] = bb.y;
        h1t[2 * nb] = 0.0; h1t[2 * nb + 1] = 0.0;
      }
#pragma unroll
      for (int ks = 0; ks < SP; ++ks) {
#pragma unroll
        for (int nb = 0; nb < L::NB1; ++nb) {
          const double b = W1p[(4 * ks + q) * L::LD1 + 8 * nb + g];
          dmma884(h1v[2 * nb], h1v[2 * nb + 1], h0v[ks], b);
          dmma884(h1t[2 * nb], h1t[2 * nb + 1], h0t[ks], b);
        }
      }
#pragma unroll
      for (int s = 0; s < 2 * SP; ++s) {
        const double t1 = dp_tanh(h1v[s]);
        h1v[s] = h0v[s % SP] + t1;
        h1t[s] = fma(fma(-t1, t1, 1.0), h1t[s], h0t[s % SP]);
      }
      double pr[5] = {0.0, 0.0, 0.0, 0.0, 0.0};         // partial dR~[0..3], dx over this thread's features
#pragma unroll
      for (int ch = 0; ch < 2; ++ch) {
        double av[2 * SP], at[2 * SP];
#pragma unroll
        for (int nb = 0; nb < SP; ++nb) {
          const double2 bb = *reinterpret_cast<const double2 *>(b2p + 8 * (ch * SP + nb) + 2 * q);
          av[2 * nb] = bb.x; av[2 * nb + 1] = bb.y;
          at[2 * nb] = 0.0; at[2 * nb + 1] = 0.0;
        }
#pragma unroll
        for (int ks = 0; ks < 2 * SP; ++ks) {
#pragma unroll
          for (int nb = 0; nb < SP; ++nb) {
            const double b = W2p[(4 * ks + q) * L::LD2 + 8 * (ch * SP + nb) + g];
            dmma884(av[2 * nb], av[2 * nb + 1], h1v[ks], b);
            dmma884(at[2 * nb], at[2 * nb + 1], h1t[ks], b);
          }
        }
#pragma unroll
        for (int s = 0; s < 2 * SP; ++s) {
          const double t2 = dp_tanh(av[s]);
          const double gv = h1v[s] + t2;
          const double gp = fma(fma(-t2, t2, 1.0), at[s], h1t[s]);
          const double4 d4 = *reinterpret_cast<const double4 *>(dTt + 4 * (4 * (ch * 2 * SP + s) + q));
          pr[0] = fma(d4.x, gv, pr[0]);
          pr[1] = fma(d4.y, gv, pr[1]);
          pr[2] = fma(d4.z, gv, pr[2]);
          pr[3] = fma(d4.w, gv, pr[3]);
          const double dg = fma(d4.x, e[0], fma(d4.y, e[1], fma(d4.z, e[2], d4.w * e[3])));
          pr[4] = fma(dg, gp, pr[4]);
        }
      }
#pragma unroll
      for (int k = 0; k < 5; ++k) {
        pr[k] += __shfl_xor_sync(0xffffffffu, pr[k], 1);
        pr[k] += __shfl_xor_sync(0xffffffffu, pr[k], 2);
      }
      if (valid && q == 0) {
        // O10: derivative of R~ with respect to the displacement; f_ik[c] = sum_m dR~[m] dR~_m / dd_c
        const double r = dv.w, ir = 1.0 / r;
        double w, dw;
        dp_switch(r, P.rcs, P.rc, w, dw);
        const double s = w * ir, qq = s * ir;
        const double sp = dw * ir - w * ir * ir;
        const double qp = sp * ir - s * ir * ir;
        const double dR0 = pr[0] + pr[4];
        const double dot = pr[1] * dv.x + pr[2] * dv.y + pr[3] * dv.z;
        const double cm = (dR0 * sp + qp * dot) * ir;
        const double f0 = fma(cm, dv.x, qq * pr[1]), f1 = fma(cm, dv.y, qq * pr[2]), f2 = fma(cm, dv.z, qq * pr[3]);
        if (C.fslot) {
          // deterministic mode: keep dE_i/dd_ik per slot; forces and virial are gathered in a fixed order afterwards
          double *fs = C.fslot + ((size_t)qa * P.nm + P.sec_start[t] + s_lo + row) * 3;
          fs[0] = f0; fs[1] = f1; fs[2] = f2;
        } else {
        const int j = jn;
        if (force) {
          atomicAdd(&force[3 * (size_t)j + 0], -f0);
          atomicAdd(&force[3 * (size_t)j + 1], -f1);
          atomicAdd(&force[3 * (size_t)j + 2], -f2);
        }
        fi[0] += f0; fi[1] += f1; fi[2] += f2;
        vir[0] -= dv.x * f0; vir[1] -= dv.x * f1; vir[2] -= dv.x * f2;
        vir[3] -= dv.y * f0; vir[4] -= dv.y * f1; vir[5] -= dv.y * f2;
        vir[6] -= dv.z * f0; vir[7] -= dv.z * f1; vir[8] -= dv.z * f2;
        }
      }
    }
    // F_i += sum_k f_ik (ProdForce)
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      double v = fi[k];                                 // only the q == 0 lanes hold contributions
      v += __shfl_xor_sync(0xffffffffu, v, 1);
      v += __shfl_xor_sync(0xffffffffu, v, 2);
      v += __shfl_xor_sync(0xffffffffu, v, 4);
      v += __shfl_xor_sync(0xffffffffu, v, 8);
      v += __shfl_xor_sync(0xffffffffu, v, 16);
      fi[k] = v;
    }
    if (lane < 3 && force && !C.fslot) atomicAdd(&force[3 * (size_t)C.s_idx[C.p0 + qa] + lane], lane == 0 ? fi[0] : (lane == 1 ? fi[1] : fi[2]));
  }
  // virial (ProdVirial): warp -> block -> one atomic per component and CTA
#pragma unroll
  for (int k = 0; k < 9; ++k) {
    double v = vir[k];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if (lane == 0) vred[warp][k] = v;
  }
  __syncthreads();
  if (tid < 9 && virial && !C.fslot) {
    double v = 0.0;
    for (int w = 0; w < P2_WARPS; ++w) v += vred[w][tid];
    atomicAdd(&virial[tid], v);
  }
}


// ---------------------------------------------------------------------------------------------------------
// Pass 2 with same-species pair reuse (nets (a, a); dpb_model_set_pair_reuse).  The embedding net
// depends on s(r_ij) = s(r_ji) only (Eq. 5, 8-9): of the two directions of a pair whose atoms are both
// centres of this chunk, ONE atom (the lower row when the row sum is even, the higher one otherwise: every atom keeps
// about half of its pairs) runs the value and tangent chains and applies the epilogue twice — with its own dT tile and
// R~_ij, and with dT_j and R~_ji = (s, -s d/r).  The dT_j slices of the 8 rows of a block are fetched from L2 by the
// TMA engine (cp.async.bulk, one 1 KB piece per row and N chunk, completion on a per-warp mbarrier) while the DMMAs of
// that chunk run; the force on the pair is f_ij - f_ji (F_i += f, F_j -= f, Xi -= d_ij (x) f).  Pairs whose neighbour
// is not a centre of this chunk (another chunk, a ghost) are evaluated in one direction as before.  Layer 2 runs as a
// two-trip loop over halves of N (two N chunks each), which also keeps the unrolled body inside the instruction cache.
template <int SP>
struct P2R {
  static constexpr int NBA = (SP + 1) / 2, NBB = SP - NBA;   // n-blocks of the two N chunks of a half (SP n-blocks)
  static constexpr int SLICE = 32 * NBA + 16;                // doubles per staged row slice (+128 B: rows on distinct banks)
  static constexpr int RING = 64;                            // kept rows in flight per warp
  // per warp: own dT tile [16 SP][4] | dT_j slices [8][SLICE] | ring (d, r) [RING] | ring j [RING] | ring row of j | mbarrier
  //           | staging of 32 raw slots: (d, r) [32], j [32], sorted position of j [32]
  static constexpr int per_warp = 64 * SP + 8 * SLICE + 4 * RING + RING / 2 + RING / 2 + 2 + 4 * 32 + 16 + 16;
};

// value and tangent MMAs of NB n-blocks (starting at n-block NB0 of the half), then the epilogue over their 2 NB slots
template <int SP, int NB, int NB0>
__device__ __forceinline__ void p2r_chunk(const double *__restrict__ W2h, const double *__restrict__ b2h,
                                          const double *__restrict__ dTh, const double *__restrict__ jrow,
                                          const bool anyboth, uint64_t *mbar, unsigned &parity,
                                          const double (&h1v)[2 * SP], const double (&h1t)[2 * SP],
                                          const double (&e)[4], const int g, const int q, double (&pr)[5],
                                          double (&pj)[5]) {
  using L = EL<SP>;
  double av[2 * NB], at[2 * NB];
#pragma unroll
  for (int nb = 0; nb < NB; ++nb) {
    const double2 bb = *reinterpret_cast<const double2 *>(b2h + 8 * (NB0 + nb) + 2 * q);
    av[2 * nb] = bb.x; av[2 * nb + 1] = bb.y;
    at[2 * nb] = 0.0; at[2 * nb + 1] = 0.0;
  }
#pragma unroll
  for (int ks = 0; ks < 2 * SP; ++ks) {
#pragma unroll
    for (int nb = 0; nb < NB; ++nb) {
      const double b = W2h[(4 * ks + q) * L::LD2 + 8 * (NB0 + nb) + g];
      dmma884(av[2 * nb], av[2 * nb + 1], h1v[ks], b);
      dmma884(at[2 * nb], at[2 * nb + 1], h1t[ks], b);
    }
  }
  // g and g' of the chunk's slots (left in av / at), and the direction i -> j against the atom's own dT tile
#pragma unroll
  for (int s = 0; s < 2 * NB; ++s) {
    const int sl = 2 * NB0 + s;                             // slot inside the half: the skip comes from slot sl of layer 1
    const double t2 = dp_tanh(av[s]);
    const double gv = h1v[sl] + t2;
    const double gp = fma(fma(-t2, t2, 1.0), at[s], h1t[sl]);
    av[s] = gv; at[s] = gp;
    const double4 d4 = *reinterpret_cast<const double4 *>(dTh + 4 * (4 * sl + q));
    pr[0] = fma(d4.x, gv, pr[0]);
    pr[1] = fma(d4.y, gv, pr[1]);
    pr[2] = fma(d4.z, gv, pr[2]);
    pr[3] = fma(d4.w, gv, pr[3]);
    const double dg = fma(d4.x, e[0], fma(d4.y, e[1], fma(d4.z, e[2], d4.w * e[3])));
    pr[4] = fma(dg, gp, pr[4]);
  }
  if (anyboth) {                                            // direction j -> i: dT_j (staged slice), R~_ji = (s, -s d/r)
    tc::mbar_wait(mbar, parity);
    parity ^= 1u;
#pragma unroll
    for (int s = 0; s < 2 * NB; ++s) {
      const double4 d4 = *reinterpret_cast<const double4 *>(jrow + 4 * (4 * s + q));
      pj[0] = fma(d4.x, av[s], pj[0]);
      pj[1] = fma(d4.y, av[s], pj[1]);
      pj[2] = fma(d4.z, av[s], pj[2]);
      pj[3] = fma(d4.w, av[s], pj[3]);
      const double dg = fma(d4.x, e[0], -fma(d4.y, e[1], fma(d4.z, e[2], d4.w * e[3])));
      pj[4] = fma(dg, at[s], pj[4]);
    }
  }
}

template <int SP>
__global__ void __launch_bounds__((32 * P2_WARPS), 1)
k_pass2_dmma_ru(DevModel P, ChunkView C, const double *__restrict__ netp, int a, int t, double *__restrict__ force,
                double *__restrict__ virial, int nseg, int *counter) {
  using L = EL<SP>;
  using R = P2R<SP>;
  extern __shared__ __align__(16) double smem[];
  double *W = smem;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, q = lane & 3;
  double *dTt = smem + ((L::total + 1) & ~1) + warp * R::per_warp;      // [16 SP][4], position 4 s + q
  double *jbuf = dTt + 64 * SP;                                         // [8][SLICE]
  double4 *rdv = reinterpret_cast<double4 *>(jbuf + 8 * R::SLICE);      // ring of kept rows: (d, r)
  int *rjn = reinterpret_cast<int *>(rdv + R::RING);                    //   input index of the neighbour (force scatter)
  int *rqj = rjn + R::RING;                                             //   its row in this chunk when both directions run, else -1
  uint64_t *mbar = reinterpret_cast<uint64_t *>(rqj + R::RING);
  double4 *sdr = reinterpret_cast<double4 *>(mbar + 2);                 // staged raw slots (cp.async, one batch ahead)
  int *snl = reinterpret_cast<int *>(sdr + 32);
  int *snlp = snl + 32;
  __shared__ double vred[P2_WARPS][9];
  __shared__ uint64_t wbar;
  if (lane == 0) tc::mbar_init(mbar, 1);
  tc::fence_mbar_init();
  stage_net(W, netp, L::total, &wbar);
  const double *W0p = W + L::oW0, *b0p = W + L::ob0, *W1p = W + L::oW1, *b1p = W + L::ob1, *W2p = W + L::oW2,
               *b2p = W + L::ob2;
  const int row_lo = max(C.p0, C.type_start[a]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[a + 1]) - C.p0;
  // pairs are shared for the nets (a, a) only, and only while no neighbour was dropped (that breaks the list symmetry)
  const bool ru = a == t && C.stats->n_overflow == 0ull;
  const size_t dt_tile = (size_t)C.dt_rows * 4;          // doubles per dT tile (= 64 SP)
  unsigned parity = 0;
  double vir[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) vir[k] = 0.0;

  for (int item = next_item(counter, lane); item < (row_hi - row_lo) * nseg; item = next_item(counter, lane)) {
    const int qa = row_lo + item / nseg;                 // work item = (atom, segment of its section), as in pass 1
    int n = C.nreal[(size_t)qa * P.ntypes + t];
    int s_lo = 0;
    if (nseg > 1) {
      const int rs = (((n + nseg - 1) / nseg) + 7) & ~7;
      s_lo = min(n, (item % nseg) * rs);
      n = min(n, s_lo + rs);
    }
    if (s_lo >= n) continue;                             // the raw slots [s_lo, n) of the section
    const double4 *dr = C.dr + (size_t)qa * P.nm + P.sec_start[t];
    const int *nl = C.nl + (size_t)qa * P.nm + P.sec_start[t];
    const int *nlp = C.nlp + (size_t)qa * P.nm + P.sec_start[t];
    __syncwarp();
    {
      const double4 *src = reinterpret_cast<const double4 *>(C.dT + (size_t)qa * dt_tile);
      for (int p = lane; p < 16 * SP; p += 32) *reinterpret_cast<double4 *>(dTt + 4 * p) = src[p];
    }
    // kept rows: sweep 0 keeps the pairs this atom evaluates in both directions, sweep 1 the one-direction pairs.  The raw
    // slots travel global -> shared one batch of 32 AHEAD of their use (cp.async issued before a row block is computed,
    // consumed after it), so that the compaction into the ring never waits for a memory round trip.
    int head = 0, cnt = 0, rawpos = s_lo, sweep = ru ? 0 : 1, st_base = 0, st_sweep = 0;
    bool done = false, staged = false;
    auto stage = [&]() {
      if (done || staged) return;
      const int slot = rawpos + lane;
      if (slot < n) {
        emb_cp16(sdr + lane, dr + slot);
        emb_cp16(reinterpret_cast<double *>(sdr + lane) + 2, reinterpret_cast<const double *>(dr + slot) + 2);
        emb_cp4(snl + lane, nl + slot);
        emb_cp4(snlp + lane, nlp + slot);
      }
      emb_cp_commit();
      st_base = rawpos; st_sweep = sweep; staged = true;
      rawpos += 32;
      if (rawpos >= n) {
        if (ru && sweep == 0) { sweep = 1; rawpos = s_lo; } else done = true;
      }
    };
    auto consume = [&]() {
      if (!staged) return;
      emb_cp_wait<0>();
      __syncwarp();
      const int slot = st_base + lane;
      bool keep = false;
      int qj = -1;
      if (slot < n) {
        if (ru) {
          const int pj = snlp[lane] - C.p0;
          const bool inchunk = pj >= 0 && pj < C.n;
          if (st_sweep == 0) { keep = inchunk && ((((qa + pj) & 1) == 0) == (qa < pj)); qj = pj; }
          else keep = !inchunk;
        } else {
          keep = true;
        }
      }
      const unsigned mk = __ballot_sync(0xffffffffu, keep);
      if (keep) {
        const int pos = (head + cnt + __popc(mk & ((1u << lane) - 1u))) & (R::RING - 1);
        rdv[pos] = sdr[lane]; rjn[pos] = snl[lane]; rqj[pos] = qj;
      }
      cnt += __popc(mk);
      staged = false;
      __syncwarp();                                      // ring rows visible; the staging area may be refilled
    };
    auto fill = [&]() {
      while (cnt < 16 && (staged || !done)) { stage(); consume(); }
    };
    // both-direction rows of the block at the ring head, and (lanes 0..7) the row of neighbour j of ring row `lane`
    int myqj = -1;
    auto block_mask = [&]() -> unsigned {
      myqj = (lane < 8 && lane < cnt) ? rqj[(head + lane) & (R::RING - 1)] : -1;
      return __ballot_sync(0xffffffffu, myqj >= 0);
    };
    // TMA: the dT_j slices of N chunk k (0..3) of the block at the ring head -> jbuf rows
    auto issue = [&](const unsigned bm, const int k) {
      if (bm == 0u) return;
      const int slot0 = (k >> 1) * 2 * SP + ((k & 1) ? 2 * R::NBA : 0);
      const unsigned bytes = ((k & 1) ? R::NBB : R::NBA) * 256u;
      if (lane == 0) tc::mbar_arrive_expect_tx(mbar, (unsigned)__popc(bm) * bytes);
      __syncwarp();
      if (myqj >= 0) tc::bulk_g2s(jbuf + lane * R::SLICE, C.dT + (size_t)myqj * dt_tile + 16 * slot0, bytes, mbar);
    };
    fill();
    if (cnt <= 32) stage();
    unsigned bmask = block_mask();
    issue(bmask, 0);
    double fi[3] = {0.0, 0.0, 0.0};

    while (cnt > 0) {
      const int nrows = min(cnt, 8);
      const bool valid = g < nrows;
      const bool both = (bmask >> g) & 1u;
      const bool anyboth = bmask != 0u;
      double e[4] = {0.0, 0.0, 0.0, 0.0};
      double4 dv = make_double4(0.0, 0.0, 0.0, 1.0);
      int jn = 0;
      if (valid) {
        const int ri = (head + g) & (R::RING - 1);
        dv = rdv[ri]; jn = rjn[ri];
        env_row4(P, dv, e);
      }
      // layer 0 and its tangent: h0' = (1 - t0^2) W0   (d tanh = 1 - tanh^2)
      double h0v[SP], h0t[SP];
#pragma unroll
      for (int s = 0; s < SP; ++s) {
        const double w0 = W0p[4 * s + q], bb = b0p[4 * s + q];
        const double t0 = dp_tanh(fma(e[0], w0, bb));
        h0v[s] = t0;
        h0t[s] = fma(-t0, t0, 1.0) * w0;
      }
      double h1v[2 * SP], h1t[2 * SP];
#pragma unroll
      for (int nb = 0; nb < L::NB1; ++nb) {
        const double2 bb = *reinterpret_cast<const double2 *>(b1p + 8 * nb + 2 * q);
        h1v[2 * nb] = bb.x; h1v[2 * nb + 1] = bb.y;
        h1t[2 * nb] = 0.0; h1t[2 * nb + 1] = 0.0;
      }
#pragma unroll
      for (int ks = 0; ks < SP; ++ks) {
#pragma unroll
        for (int nb = 0; nb < L::NB1; ++nb) {
          const double b = W1p[(4 * ks + q) * L::LD1 + 8 * nb + g];
          dmma884(h1v[2 * nb], h1v[2 * nb + 1], h0v[ks], b);
          dmma884(h1t[2 * nb], h1t[2 * nb + 1], h0t[ks], b);
        }
      }
#pragma unroll
      for (int s = 0; s < 2 * SP; ++s) {
        const double t1 = dp_tanh(h1v[s]);
        h1v[s] = h0v[s % SP] + t1;
        h1t[s] = fma(fma(-t1, t1, 1.0), h1t[s], h0t[s % SP]);
      }
      double pr[5] = {0.0, 0.0, 0.0, 0.0, 0.0};         // partial dR~_ij[0..3], dx over this thread's features
      double pj[5] = {0.0, 0.0, 0.0, 0.0, 0.0};         // the same for the direction j -> i
      const double *jrow = jbuf + g * R::SLICE;
#pragma unroll 1
      for (int half = 0; half < 2; ++half) {
        const double *W2h = W2p + 8 * half * SP, *b2h = b2p + 8 * half * SP, *dTh = dTt + 32 * half * SP;
        p2r_chunk<SP, R::NBA, 0>(W2h, b2h, dTh, jrow, anyboth, mbar, parity, h1v, h1t, e, g, q, pr, pj);
        __syncwarp();                                    // every lane has read its slice: the next one may land
        issue(bmask, 2 * half + 1);
        if (R::NBB > 0) p2r_chunk<SP, R::NBB, R::NBA>(W2h, b2h, dTh, jrow, anyboth, mbar, parity, h1v, h1t, e, g, q, pr, pj);
        __syncwarp();
        if (half == 0) issue(bmask, 2);
      }
#pragma unroll
      for (int k = 0; k < 5; ++k) {
        pr[k] += __shfl_xor_sync(0xffffffffu, pr[k], 1);
        pr[k] += __shfl_xor_sync(0xffffffffu, pr[k], 2);
      }
      if (anyboth) {
#pragma unroll
        for (int k = 0; k < 5; ++k) {
          pj[k] += __shfl_xor_sync(0xffffffffu, pj[k], 1);
          pj[k] += __shfl_xor_sync(0xffffffffu, pj[k], 2);
        }
      }
      // advance the ring and start the next block's first slices before the scalar tail of this one
      head = (head + nrows) & (R::RING - 1);
      cnt -= nrows;
      consume();
      fill();
      if (cnt <= 32) stage();
      bmask = block_mask();
      issue(bmask, 0);
      if (valid && q == 0) {
        // O10: derivative of R~ with respect to the displacement; f_ik[c] = sum_m dR~[m] dR~_m / dd_c
        const double r = dv.w, ir = 1.0 / r;
        double w, dw;
        dp_switch(r, P.rcs, P.rc, w, dw);
        const double s = w * ir, qq = s * ir;
        const double sp = dw * ir - w * ir * ir;
        const double qp = sp * ir - s * ir * ir;
        const double dot = pr[1] * dv.x + pr[2] * dv.y + pr[3] * dv.z;
        const double cm = ((pr[0] + pr[4]) * sp + qp * dot) * ir;
        double f0 = fma(cm, dv.x, qq * pr[1]), f1 = fma(cm, dv.y, qq * pr[2]), f2 = fma(cm, dv.z, qq * pr[3]);
        if (both) {                                      // f_ji = dE_j/dd_ji with d_ji = -d_ij; the pair force is f_ij - f_ji
          const double dotj = -(pj[1] * dv.x + pj[2] * dv.y + pj[3] * dv.z);
          const double cmj = ((pj[0] + pj[4]) * sp + qp * dotj) * ir;
          f0 -= fma(-cmj, dv.x, qq * pj[1]);
          f1 -= fma(-cmj, dv.y, qq * pj[2]);
          f2 -= fma(-cmj, dv.z, qq * pj[3]);
        }
        if (force) {
          atomicAdd(&force[3 * (size_t)jn + 0], -f0);
          atomicAdd(&force[3 * (size_t)jn + 1], -f1);
          atomicAdd(&force[3 * (size_t)jn + 2], -f2);
        }
        fi[0] += f0; fi[1] += f1; fi[2] += f2;
        vir[0] -= dv.x * f0; vir[1] -= dv.x * f1; vir[2] -= dv.x * f2;
        vir[3] -= dv.y * f0; vir[4] -= dv.y * f1; vir[5] -= dv.y * f2;
        vir[6] -= dv.z * f0; vir[7] -= dv.z * f1; vir[8] -= dv.z * f2;
      }
    }
    // F_i += sum_k f_ik (ProdForce)
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      double v = fi[k];                                 // only the q == 0 lanes hold contributions; every lane gets the sum
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
      fi[k] = v;
    }
    if (lane < 3 && force) atomicAdd(&force[3 * (size_t)C.s_idx[C.p0 + qa] + lane], lane == 0 ? fi[0] : (lane == 1 ? fi[1] : fi[2]));
  }
#pragma unroll
  for (int k = 0; k < 9; ++k) {
    double v = vir[k];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if (lane == 0) vred[warp][k] = v;
  }
  __syncthreads();
  if (tid < 9 && virial) {
    double v = 0.0;
    for (int w = 0; w < P2_WARPS; ++w) v += vred[w][tid];
    atomicAdd(&virial[tid], v);
  }
}


// ---------------------------------------------------------------------------------------------------------
// Pass 2, row-stream kernel (every net; chunks large enough that a work item is a whole atom).  The kept rows of the atoms a
// warp takes (pair reuse as in k_pass2_dmma_ru for a == t) form ONE stream of 8-row blocks: only the last block of a
// WARP is ragged, not the last block of every atom and net (W24k: 8.6 % of the pass-2 rows were padding, Cu32k 4 %).
// A block may therefore hold rows of two atoms (never more: it is cut short otherwise): the dE/dT slices of the (at
// most two) centre atoms of a block come from L2 by the same TMA copies as the neighbours' slices, per N chunk, instead
// of a per-atom tile in shared memory; F_i is added per row.
template <int SP, bool BOTH = true>
struct P2S {
  static constexpr int JR = BOTH ? 8 : 0;                    // staged dT_j rows (none for a net without shared pairs)
  static constexpr int NBA = (SP + 1) / 2, NBB = SP - NBA;   // n-blocks of the two N chunks of a half (SP n-blocks)
  static constexpr int SLICE = 32 * NBA + 16;                // doubles per staged row slice (+128 B: rows on distinct banks)
  static constexpr int RING = 64;
  // per warp: dT_i slices [2][SLICE] | dT_j slices [8][SLICE] | ring (d, r) [RING] | ring ints j, row of j, centre row, i,
  //           record index [RING] | mbarrier | staging of 32 raw slots: (d, r) [32], j [32], sorted position of j [32]
  static constexpr int per_warp = (2 + JR) * SLICE + 4 * RING + 2 * RING + RING / 2 + 2 + 4 * 32 + 16 + 16;
};

// SA: the value chain is not run; t2v holds the stored tanh outputs of this chunk's slots (ChunkView::act).
template <int SP, int NB, int NB0, bool SA>
__device__ __forceinline__ void p2s_chunk(const double *__restrict__ W2h, const double *__restrict__ b2h,
                                          const double *__restrict__ irow, const double *__restrict__ jrow,
                                          const bool anyboth, uint64_t *mbar, unsigned &parity,
                                          const double (&h1v)[2 * SP], const double (&h1t)[2 * SP],
                                          const double (&t2v)[2 * NB],
                                          const double (&e)[4], const int g, const int q, double (&pr)[5],
                                          double (&pj)[5]) {
  using L = EL<SP>;
  double av[2 * NB], at[2 * NB];
#pragma unroll
  for (int nb = 0; nb < NB; ++nb) {
    if (!SA) {
      const double2 bb = *reinterpret_cast<const double2 *>(b2h + 8 * (NB0 + nb) + 2 * q);
      av[2 * nb] = bb.x; av[2 * nb + 1] = bb.y;
    }
    at[2 * nb] = 0.0; at[2 * nb + 1] = 0.0;
  }
#pragma unroll
  for (int ks = 0; ks < 2 * SP; ++ks) {
#pragma unroll
    for (int nb = 0; nb < NB; ++nb) {
      const double b = W2h[(4 * ks + q) * L::LD2 + 8 * (NB0 + nb) + g];
      if (!SA) dmma884(av[2 * nb], av[2 * nb + 1], h1v[ks], b);
      dmma884(at[2 * nb], at[2 * nb + 1], h1t[ks], b);
    }
  }
  tc::mbar_wait(mbar, parity);                              // the slices of this chunk (dT_i always, dT_j if any) have landed
  parity ^= 1u;
#pragma unroll
  for (int s = 0; s < 2 * NB; ++s) {
    const int sl = 2 * NB0 + s;                             // slot inside the half: the skip comes from slot sl of layer 1
    const double t2 = SA ? t2v[s] : dp_tanh(av[s]);
    const double gv = h1v[sl] + t2;
    const double gp = fma(fma(-t2, t2, 1.0), at[s], h1t[sl]);
    av[s] = gv; at[s] = gp;
    const double4 d4 = *reinterpret_cast<const double4 *>(irow + 4 * (4 * s + q));
    pr[0] = fma(d4.x, gv, pr[0]);
    pr[1] = fma(d4.y, gv, pr[1]);
    pr[2] = fma(d4.z, gv, pr[2]);
    pr[3] = fma(d4.w, gv, pr[3]);
    const double dg = fma(d4.x, e[0], fma(d4.y, e[1], fma(d4.z, e[2], d4.w * e[3])));
    pr[4] = fma(dg, gp, pr[4]);
  }
  if (anyboth) {                                            // direction j -> i: dT_j, R~_ji = (s, -s d/r)
#pragma unroll
    for (int s = 0; s < 2 * NB; ++s) {
      const double4 d4 = *reinterpret_cast<const double4 *>(jrow + 4 * (4 * s + q));
      pj[0] = fma(d4.x, av[s], pj[0]);
      pj[1] = fma(d4.y, av[s], pj[1]);
      pj[2] = fma(d4.z, av[s], pj[2]);
      pj[3] = fma(d4.w, av[s], pj[3]);
      const double dg = fma(d4.x, e[0], -fma(d4.y, e[1], fma(d4.z, e[2], d4.w * e[3])));
      pj[4] = fma(dg, at[s], pj[4]);
    }
  }
}

// NW warps per CTA; BOTH = false: a net without shared pairs (a != t) — no dT_j slices, no second direction, and with SA
// few enough registers and little enough shared memory for 12 warps
template <int SP, bool SA, int NW, bool BOTH>
__global__ void __launch_bounds__((32 * NW), 1)
k_pass2_dmma_st(DevModel P, ChunkView C, const double *__restrict__ netp, int a, int t, double *__restrict__ force,
                double *__restrict__ virial, int *counter) {
  using L = EL<SP>;
  using R = P2S<SP, BOTH>;
  extern __shared__ __align__(16) double smem[];
  double *W = smem;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, q = lane & 3;
  double *ibuf = smem + ((L::total + 1) & ~1) + warp * R::per_warp;     // [2][SLICE] dT slices of the block's centre atoms
  double *jbuf = ibuf + 2 * R::SLICE;                                   // [8][SLICE] dT slices of the rows' neighbours
  double4 *rdv = reinterpret_cast<double4 *>(jbuf + R::JR * R::SLICE);      // ring of kept rows: (d, r)
  int *rjn = reinterpret_cast<int *>(rdv + R::RING);                    //   input index of the neighbour
  int *rqj = rjn + R::RING;                                             //   its row in this chunk when both directions run, else -1
  int *rqa = rqj + R::RING;                                             //   row of the centre atom in this chunk
  int *rio = rqa + R::RING;                                             //   input index of the centre atom
  int *rrec = rio + R::RING;                                            //   index of the row's activation record (SA)
  uint64_t *mbar = reinterpret_cast<uint64_t *>(rrec + R::RING);
  double4 *sdr = reinterpret_cast<double4 *>(mbar + 2);                 // staged raw slots (cp.async, one batch ahead)
  int *snl = reinterpret_cast<int *>(sdr + 32);
  int *snlp = snl + 32;
  __shared__ double vred[NW][9];
  __shared__ uint64_t wbar;
  if (lane == 0) tc::mbar_init(mbar, 1);
  tc::fence_mbar_init();
  stage_net(W, netp, L::total, &wbar);
  const double *W0p = W + L::oW0, *b0p = W + L::ob0, *W1p = W + L::oW1, *b1p = W + L::ob1, *W2p = W + L::oW2,
               *b2p = W + L::ob2;
  const int row_lo = max(C.p0, C.type_start[a]) - C.p0, row_hi = min(C.p0 + C.n, C.type_start[a + 1]) - C.p0;
  const bool ru = BOTH && a == t && C.stats->n_overflow == 0ull;
  const size_t dt_tile = (size_t)C.dt_rows * 4;
  unsigned parity = 0;
  double vir[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) vir[k] = 0.0;

  // The ring of kept rows lives across work items: a warp takes one atom at a time from the counter (fine-grained, for the
  // tail of the launch), and the rows an atom leaves over (< 8) are computed together with the first rows of the warp's
  // next atom, whichever that is — rows carry their centre atom.  Only the last block of a WARP is ragged.
  const int natom = max(row_hi - row_lo, 0);
  int head = 0, cnt = 0;
  int qa = 0, n = 0, io = 0, rawpos = 0, sweep = 1;      // the atom being swept: chunk row, real slots, input index
  bool have = false, nomore = false;
  {
    // next atom with rows, or nomore
    auto next_atom = [&]() {
      have = false;
      while (!nomore && !have) {
        const int item = next_item(counter, lane);
        if (item >= natom) { nomore = true; break; }
        qa = row_lo + item;
        n = C.nreal[(size_t)qa * P.ntypes + t];
        if (n > 0) { io = C.s_idx[C.p0 + qa]; rawpos = 0; sweep = ru ? 0 : 1; have = true; }
      }
    };
    // one batch of 32 raw slots of the current atom: global -> shared (cp.async), kept rows -> ring
    auto batch = [&]() {
      const int slot = rawpos + lane;
      if (slot < n) {
        const size_t o = (size_t)qa * P.nm + P.sec_start[t] + slot;
        emb_cp16(sdr + lane, C.dr + o);
        emb_cp16(reinterpret_cast<double *>(sdr + lane) + 2, reinterpret_cast<const double *>(C.dr + o) + 2);
        emb_cp4(snl + lane, C.nl + o);
        emb_cp4(snlp + lane, C.nlp + o);
      }
      emb_cp_commit();
      emb_cp_wait<0>();
      __syncwarp();
      bool keep = false;
      int qj = -1;
      if (slot < n) {
        if (ru) {
          const int pj = snlp[lane] - C.p0;
          const bool inchunk = pj >= 0 && pj < C.n;
          // sweep 0 keeps the pairs this atom evaluates in both directions, sweep 1 the one-direction pairs.
          // SA: the evaluating atom is the one whose row pass 1 stored — the lower row, as in k_pass1_dmma<.., RU>
          if (sweep == 0) { keep = inchunk && (SA ? qa < pj : ((((qa + pj) & 1) == 0) == (qa < pj))); qj = pj; }
          else keep = !inchunk;
        } else {
          keep = true;
        }
      }
      const unsigned mk = __ballot_sync(0xffffffffu, keep);
      if (keep) {
        const int pos = (head + cnt + __popc(mk & ((1u << lane) - 1u))) & (R::RING - 1);
        rdv[pos] = sdr[lane]; rjn[pos] = snl[lane]; rqj[pos] = qj; rqa[pos] = qa; rio[pos] = io;
        if (SA) rrec[pos] = qa * P.nm + P.sec_start[t] + slot;
      }
      cnt += __popc(mk);
      __syncwarp();
      rawpos += 32;
      if (rawpos >= n) {
        if (ru && sweep == 0) { sweep = 1; rawpos = 0; } else have = false;
      }
    };
    auto fill = [&]() {
      while (cnt < 16 && !nomore) {
        if (!have) { next_atom(); continue; }
        batch();
      }
    };
    // the block at the ring head: its rows (at most 8, of at most two atoms), which of them run both directions, and
    // (lanes 0..7) the neighbour row, (lanes 8, 9) the centre rows whose dT slices the TMA fetches
    int nrows = 0, myrow = -1, islot = 0;
    unsigned bmask = 0;
    auto block_setup = [&]() {
      const int avail = min(cnt, 8);
      const int rq = lane < avail ? rqa[(head + lane) & (R::RING - 1)] : -1;
      const int a0 = __shfl_sync(0xffffffffu, rq, 0);
      const unsigned m0 = __ballot_sync(0xffffffffu, lane < avail && rq == a0);
      const unsigned rest = ((1u << avail) - 1u) & ~m0;
      int a1 = -1;
      unsigned m1 = 0;
      if (rest) {
        a1 = __shfl_sync(0xffffffffu, rq, __ffs(rest) - 1);
        m1 = __ballot_sync(0xffffffffu, lane < avail && rq == a1);
      }
      nrows = __popc(m0 | m1);                              // rows are ordered by atom: a prefix of the ring
      const int qjl = lane < nrows ? rqj[(head + lane) & (R::RING - 1)] : -1;
      bmask = BOTH ? __ballot_sync(0xffffffffu, qjl >= 0) : 0u;
      myrow = BOTH ? qjl : -1;                              // lanes 0..7: row of the neighbour (or -1)
      if (lane == 8) myrow = nrows > 0 ? a0 : -1;
      if (lane == 9) myrow = a1;
      const int rqg = __shfl_sync(0xffffffffu, rq, g);      // centre row of this thread's tile row
      islot = (g < nrows && rqg == a1) ? 1 : 0;
    };
    auto issue = [&](const int k) {                         // N chunk k (0..3) of the block at the ring head
      if (nrows == 0) return;
      const int slot0 = (k >> 1) * 2 * SP + ((k & 1) ? 2 * R::NBA : 0);
      const unsigned bytes = ((k & 1) ? R::NBB : R::NBA) * 256u;
      const unsigned want = __ballot_sync(0xffffffffu, lane < 10 && myrow >= 0);
      if (lane == 0) tc::mbar_arrive_expect_tx(mbar, (unsigned)__popc(want) * bytes);
      __syncwarp();
      if (lane < 10 && myrow >= 0) {
        double *dst = lane < 8 ? jbuf + lane * R::SLICE : ibuf + (lane - 8) * R::SLICE;
        tc::bulk_g2s(dst, C.dT + (size_t)myrow * dt_tile + 16 * slot0, bytes, mbar);
      }
    };
    fill();
    block_setup();
    issue(0);

    while (cnt > 0) {
      const int nr = nrows;
      const bool valid = g < nr;
      const bool both = BOTH && ((bmask >> g) & 1u);
      const bool anyboth = BOTH && bmask != 0u;
      // SA: the records are streamed from DRAM (written once by pass 1, read once here): the 8 ring rows behind this block
      // are prefetched into L2 now, one block (about 2,500 cycles) before their loads
      if (SA && lane < 8 && 8 + lane < cnt)
        act_prefetch(C.act + (size_t)rrec[(head + 8 + lane) & (R::RING - 1)] * L::REC, (unsigned)(L::REC * 8));
      double e[4] = {0.0, 0.0, 0.0, 0.0};
      double4 dv = make_double4(0.0, 0.0, 0.0, 1.0);
      int jn = 0, ri_io = 0;
      if (valid) {
        const int ri = (head + g) & (R::RING - 1);
        dv = rdv[ri]; jn = rjn[ri]; ri_io = rio[ri];
        env_row4(P, dv, e);
      }
      // SA: this lane's piece of the row's activation record (written by pass 1)
      const double *recp = nullptr;
      if (SA && valid) recp = C.act + (size_t)rrec[(head + g) & (R::RING - 1)] * L::REC + 2 * q;
      double t01[SA ? L::A0 + 2 * SP : 2];                  // t0 [A0] | t1 [2 SP]
      double t2a[2 * R::NBA], t2b[2 * R::NBB];              // NBB >= 1 for every SP in use
      if (SA) {
#pragma unroll
        for (int s = 0; s < L::A0 + 2 * SP; s += 2) {
          double2 v = make_double2(0.0, 0.0);
          if (recp) v = act_load(recp + 4 * s);
          t01[s] = v.x; t01[s + 1] = v.y;
        }
#pragma unroll
        for (int s = 0; s < 2 * R::NBA; s += 2) {           // N chunk 0 of layer 2
          double2 v = make_double2(0.0, 0.0);
          if (recp) v = act_load(recp + 4 * (L::A0 + 2 * SP + s));
          t2a[s] = v.x; t2a[s + 1] = v.y;
        }
      }
      double h0v[SP], h0t[SP];
#pragma unroll
      for (int s = 0; s < SP; ++s) {
        const double w0 = W0p[4 * s + q], bb = b0p[4 * s + q];
        const double t0 = SA ? t01[s] : dp_tanh(fma(e[0], w0, bb));
        h0v[s] = t0;
        h0t[s] = fma(-t0, t0, 1.0) * w0;
      }
      double h1v[2 * SP], h1t[2 * SP];
#pragma unroll
      for (int nb = 0; nb < L::NB1; ++nb) {
        if (!SA) {
          const double2 bb = *reinterpret_cast<const double2 *>(b1p + 8 * nb + 2 * q);
          h1v[2 * nb] = bb.x; h1v[2 * nb + 1] = bb.y;
        }
        h1t[2 * nb] = 0.0; h1t[2 * nb + 1] = 0.0;
      }
#pragma unroll
      for (int ks = 0; ks < SP; ++ks) {
#pragma unroll
        for (int nb = 0; nb < L::NB1; ++nb) {
          const double b = W1p[(4 * ks + q) * L::LD1 + 8 * nb + g];
          if (!SA) dmma884(h1v[2 * nb], h1v[2 * nb + 1], h0v[ks], b);
          dmma884(h1t[2 * nb], h1t[2 * nb + 1], h0t[ks], b);
        }
      }
#pragma unroll
      for (int s = 0; s < 2 * SP; ++s) {
        const double t1 = SA ? t01[L::A0 + s] : dp_tanh(h1v[s]);
        h1v[s] = h0v[s % SP] + t1;
        h1t[s] = fma(fma(-t1, t1, 1.0), h1t[s], h0t[s % SP]);
      }
      double pr[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      double pj[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      const double *irow = ibuf + islot * R::SLICE, *jrow = jbuf + g * R::SLICE;
#pragma unroll 1
      for (int half = 0; half < 2; ++half) {
        const double *W2h = W2p + 8 * half * SP, *b2h = b2p + 8 * half * SP;
        // the stored t2 of a chunk are fetched one chunk ahead (BOTH: 2 warps per scheduler) or just before the chunk's
        // DMMAs, which then cover the load (!BOTH: 12 warps at 168 registers — the lookahead's registers would spill)
        auto load_t2a = [&](const int hf) {
#pragma unroll
          for (int s = 0; s < 2 * R::NBA; s += 2) {
            double2 v = make_double2(0.0, 0.0);
            if (recp) v = act_load(recp + 4 * (L::A0 + 2 * SP + hf * 2 * SP + s));
            t2a[s] = v.x; t2a[s + 1] = v.y;
          }
        };
        auto load_t2b = [&](const int hf) {
#pragma unroll
          for (int s = 0; s < 2 * R::NBB; s += 2) {
            double2 v = make_double2(0.0, 0.0);
            if (recp) v = act_load(recp + 4 * (L::A0 + 2 * SP + hf * 2 * SP + 2 * R::NBA + s));
            t2b[s] = v.x; t2b[s + 1] = v.y;
          }
        };
        if (SA && !BOTH && half == 1) load_t2a(1);
        if (SA && BOTH) load_t2b(half);
        p2s_chunk<SP, R::NBA, 0, SA>(W2h, b2h, irow, jrow, anyboth, mbar, parity, h1v, h1t, t2a, e, g, q, pr, pj);
        __syncwarp();
        issue(2 * half + 1);
        if (SA && BOTH && half == 0) load_t2a(1);
        if (SA && !BOTH) load_t2b(half);
        p2s_chunk<SP, R::NBB, R::NBA, SA>(W2h, b2h, irow, jrow, anyboth, mbar, parity, h1v, h1t, t2b, e, g, q, pr, pj);
        __syncwarp();
        if (half == 0) issue(2);
      }
#pragma unroll
      for (int k = 0; k < 5; ++k) {
        pr[k] += __shfl_xor_sync(0xffffffffu, pr[k], 1);
        pr[k] += __shfl_xor_sync(0xffffffffu, pr[k], 2);
      }
      if (anyboth) {
#pragma unroll
        for (int k = 0; k < 5; ++k) {
          pj[k] += __shfl_xor_sync(0xffffffffu, pj[k], 1);
          pj[k] += __shfl_xor_sync(0xffffffffu, pj[k], 2);
        }
      }
      head = (head + nr) & (R::RING - 1);
      cnt -= nr;
      fill();
      block_setup();
      issue(0);
      if (valid && q == 0) {
        const double r = dv.w, ir = 1.0 / r;
        double w, dw;
        dp_switch(r, P.rcs, P.rc, w, dw);
        const double s = w * ir, qq = s * ir;
        const double sp = dw * ir - w * ir * ir;
        const double qp = sp * ir - s * ir * ir;
        const double dot = pr[1] * dv.x + pr[2] * dv.y + pr[3] * dv.z;
        const double cm = ((pr[0] + pr[4]) * sp + qp * dot) * ir;
        double f0 = fma(cm, dv.x, qq * pr[1]), f1 = fma(cm, dv.y, qq * pr[2]), f2 = fma(cm, dv.z, qq * pr[3]);
        if (both) {
          const double dotj = -(pj[1] * dv.x + pj[2] * dv.y + pj[3] * dv.z);
          const double cmj = ((pj[0] + pj[4]) * sp + qp * dotj) * ir;
          f0 -= fma(-cmj, dv.x, qq * pj[1]);
          f1 -= fma(-cmj, dv.y, qq * pj[2]);
          f2 -= fma(-cmj, dv.z, qq * pj[3]);
        }
        if (force) {
          atomicAdd(&force[3 * (size_t)jn + 0], -f0);
          atomicAdd(&force[3 * (size_t)jn + 1], -f1);
          atomicAdd(&force[3 * (size_t)jn + 2], -f2);
          atomicAdd(&force[3 * (size_t)ri_io + 0], f0);
          atomicAdd(&force[3 * (size_t)ri_io + 1], f1);
          atomicAdd(&force[3 * (size_t)ri_io + 2], f2);
        }
        vir[0] -= dv.x * f0; vir[1] -= dv.x * f1; vir[2] -= dv.x * f2;
        vir[3] -= dv.y * f0; vir[4] -= dv.y * f1; vir[5] -= dv.y * f2;
        vir[6] -= dv.z * f0; vir[7] -= dv.z * f1; vir[8] -= dv.z * f2;
      }
    }
  }
#pragma unroll
  for (int k = 0; k < 9; ++k) {
    double v = vir[k];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if (lane == 0) vred[warp][k] = v;
  }
  __syncthreads();
  if (tid < 9 && virial) {
    double v = 0.0;
    for (int w = 0; w < NW; ++w) v += vred[w][tid];
    atomicAdd(&virial[tid], v);
  }
}

// ---------------------------------------------------------------------------------------------------------
static int g_sm_count_d[DPB_MAX_DEVICES] = {};      // per device
#define g_sm_count (g_sm_count_d[dpb_device()])

// Segments per atom (work items per atom and net): 1 when the chunk has enough atoms to give every warp of the GPU two
// of them (counting all nets); up to 8 for small chunks (configs[0]: 192 atoms on 148 SMs x 8 warps).
static int seg_count(int n_atoms, int warps, int nets) {
  const long long want = 2ll * g_sm_count * warps / (nets > 0 ? nets : 1);   // the nets' launches run side by side
  long long k = (want + n_atoms - 1) / (n_atoms > 0 ? n_atoms : 1);
  return (int)(k < 1 ? 1 : (k > 8 ? 8 : k));
}

template <int SP>
static cudaError_t run_pass1(const DevModel &P, const ChunkView &C, const V1Weights &W, cudaStream_t st) {
  using L = EL<SP>;
  const size_t smem = sizeof(double) * (((L::total + 1) & ~1) + P1_WARPS * L::tile1s);
  const size_t smem_ru = smem + sizeof(int) * 2 * (size_t)P.nm * P1_WARPS;
  const bool reuse = C.reuse && C.nlp && smem_ru <= 227 * 1024;
  static bool configured_d[DPB_MAX_DEVICES] = {};
  bool &configured = configured_d[dpb_device()];
  static size_t configured_ru_d[DPB_MAX_DEVICES] = {};
  size_t &configured_ru = configured_ru_d[dpb_device()];
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_pass1_dmma<SP, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  if (reuse && smem_ru > configured_ru) {
    cudaError_t e = cudaFuncSetAttribute(k_pass1_dmma<SP, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ru);
    if (e != cudaSuccess) return e;
    configured_ru = smem_ru;
  }
  const int nseg = C.fslot ? 1 : seg_count(C.n, P1_WARPS, P.ntypes * P.ntypes);   // deterministic mode: no reductions into T
  if ((reuse || nseg > 1) && !C.prezero) {               // every accumulation into T is then an addition
    cudaError_t e = cudaMemsetAsync(C.T, 0, sizeof(double) * (size_t)C.n * P.M * 4, st);
    if (e != cudaSuccess) return e;
  }
  const int grid = (int)min((long long)g_sm_count, ((long long)C.n * nseg + P1_WARPS - 1) / P1_WARPS);
  // nets of one centre type a accumulate into the same T rows (t = 0 stores, t > 0 adds): one stream per a, so that the
  // tail of one launch overlaps the start of another centre type's
  // (with row segments every accumulation is a reduction: then every net gets its own stream)
  cudaStream_t ts[DPB_MAX_TYPES];
  const int ns = nseg > 1 ? min(P.ntypes * P.ntypes, DPB_MAX_TYPES) : P.ntypes;
  cudaError_t e = dpb_fork_streams(ns, st, ts);
  if (e != cudaSuccess) return e;
  for (int a = 0; a < P.ntypes; ++a)
    for (int t = 0; t < P.ntypes; ++t) {
      const double *net = W.emb + (size_t)(a * P.ntypes + t) * W.net_stride;
      cudaStream_t s = nseg > 1 ? ts[(a * P.ntypes + t) % ns] : ts[P.ntypes - 1 - a];
      if (reuse && a == t)
        k_pass1_dmma<SP, 1, true><<<grid, (32 * P1_WARPS), smem_ru, s>>>(P, C, net, a, t, nseg > 1 ? 2 : 1, nseg,
                                                                        C.counters + a * P.ntypes + t);
      else
        k_pass1_dmma<SP, 1, false><<<grid, (32 * P1_WARPS), smem, s>>>(P, C, net, a, t,
                                                                      nseg > 1 ? 2 : (reuse ? 1 : t > 0), nseg,
                                                                      C.counters + a * P.ntypes + t);
      DPB_LAUNCHED(1);
    }
  if (!(C.typed_pipe && nseg == 1) && (e = dpb_join_streams(ns, st, ts)) != cudaSuccess) return e;
  return cudaGetLastError();
}

template <int SP>
static cudaError_t run_pass2(const DevModel &P, const ChunkView &C, const V1Weights &W, double *force, double *virial,
                             cudaStream_t st) {
  using L = EL<SP>;
  const size_t smem = sizeof(double) * (((L::total + 1) & ~1) + P2_WARPS * (L::tile2 + EMB_STG));
  static bool configured_d[DPB_MAX_DEVICES] = {};
  bool &configured = configured_d[dpb_device()];
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_pass2_dmma<SP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  using R = P2R<SP>;
  const size_t smem_ru = sizeof(double) * (((L::total + 1) & ~1) + P2_WARPS * R::per_warp);
  const bool reuse = C.reuse2 && !C.fslot && C.nlp && C.dt_pad == 4 * SP && smem_ru <= 227 * 1024;
  static bool configured_ru_d[DPB_MAX_DEVICES] = {};
  bool &configured_ru = configured_ru_d[dpb_device()];
  if (reuse && !configured_ru) {
    cudaError_t e = cudaFuncSetAttribute(k_pass2_dmma_ru<SP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ru);
    if (e != cudaSuccess) return e;
    configured_ru = true;
  }
  const int nseg = C.fslot ? 1 : seg_count(C.n, P2_WARPS, P.ntypes * P.ntypes);
  using S = P2S<SP>;
  const size_t smem_st = sizeof(double) * (((L::total + 1) & ~1) + P2_WARPS * S::per_warp);
  // the row-stream kernel serves every net when an item is a run of whole atoms (no row segments, no per-slot output)
  const bool stream = reuse && nseg == 1 && smem_st <= 227 * 1024;
  // stored activations: pass 1 wrote a record for every row it evaluated (same nseg == 1 condition there)
  const bool sa = stream && C.act != nullptr && C.act_stride == L::REC &&
                  seg_count(C.n, P1_WARPS, P.ntypes * P.ntypes) == 1;
  // nets a != t with stored activations: no staged neighbour slices and no second direction -> 12 warps per CTA
  constexpr int NW1 = 12;
  const size_t smem_one = sizeof(double) * (((L::total + 1) & ~1) + NW1 * P2S<SP, false>::per_warp);
  static bool configured_st_d[DPB_MAX_DEVICES] = {};
  bool &configured_st = configured_st_d[dpb_device()];
  if (stream && !configured_st) {
    cudaError_t e = cudaFuncSetAttribute(k_pass2_dmma_st<SP, false, P2_WARPS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem_st);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(k_pass2_dmma_st<SP, true, P2_WARPS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               (int)smem_st);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(k_pass2_dmma_st<SP, true, NW1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               (int)smem_one);
    if (e != cudaSuccess) return e;
    configured_st = true;
  }
  const int grid = (int)min((long long)g_sm_count, ((long long)C.n * nseg + P2_WARPS - 1) / P2_WARPS);
  // the nets are independent here (forces and virial are atomic sums, slot stores are disjoint): a stream per net, so
  // that the tail of every launch is filled by the others
  cudaStream_t ts[DPB_MAX_TYPES];
  const bool typed = C.typed_pipe && nseg == 1;            // species pipeline: the streams of pass 1 / fitting, not joined yet
  const int ns = typed ? P.ntypes : min(P.ntypes * P.ntypes, DPB_MAX_TYPES);
  cudaError_t e = typed ? dpb_forked_streams(ns, st, ts) : dpb_fork_streams(ns, st, ts);
  if (e != cudaSuccess) return e;
  for (int a = P.ntypes - 1; a >= 0; --a)
    for (int t = P.ntypes - 1; t >= 0; --t) {
      const int net = a * P.ntypes + t;
      cudaStream_t s = typed ? ts[P.ntypes - 1 - a] : ts[(P.ntypes * P.ntypes - 1 - net) % ns];
      if (sa && a != t)
        k_pass2_dmma_st<SP, true, NW1, false><<<grid, (32 * NW1), smem_one, s>>>(P, C, W.emb + (size_t)net * W.net_stride, a,
                                                                                   t, force, virial, C.counters + 64 + net);
      else if (sa)
        k_pass2_dmma_st<SP, true, P2_WARPS, true><<<grid, (32 * P2_WARPS), smem_st, s>>>(
            P, C, W.emb + (size_t)net * W.net_stride, a, t, force, virial, C.counters + 64 + net);
      else if (stream)
        k_pass2_dmma_st<SP, false, P2_WARPS, true><<<grid, (32 * P2_WARPS), smem_st, s>>>(
            P, C, W.emb + (size_t)net * W.net_stride, a, t, force, virial, C.counters + 64 + net);
      else if (reuse && a == t)
        k_pass2_dmma_ru<SP><<<grid, (32 * P2_WARPS), smem_ru, s>>>(P, C, W.emb + (size_t)net * W.net_stride, a, t, force,
                                                                     virial, nseg, C.counters + 64 + net);
      else
        k_pass2_dmma<SP><<<grid, (32 * P2_WARPS), smem, s>>>(P, C, W.emb + (size_t)net * W.net_stride, a, t, force,
                                                              virial, nseg, C.counters + 64 + net);
      DPB_LAUNCHED(1);
    }
  if ((e = dpb_join_streams(ns, st, ts)) != cudaSuccess) return e;
  return cudaGetLastError();
}

static cudaError_t ensure_sm_count() {
  if (g_sm_count > 0) return cudaSuccess;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  return cudaDeviceGetAttribute(&g_sm_count, cudaDevAttrMultiProcessorCount, dev);
}

cudaError_t v1_pass1(const DevModel &P, const ChunkView &C, const V1Weights &W, cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  if (!W.ready) return cudaErrorNotSupported;                  // api.cu routes nets wider than 32 to variant 0
  cudaError_t e = ensure_sm_count();
  if (e != cudaSuccess) return e;
  switch (W.SP) {
    case 2: return run_pass1<2>(P, C, W, st);
    case 4: return run_pass1<4>(P, C, W, st);
    case 7: return run_pass1<7>(P, C, W, st);
    default: return run_pass1<8>(P, C, W, st);
  }
}

cudaError_t v1_pass2(const DevModel &P, const ChunkView &C, const V1Weights &W, double *force, double *virial,
                     cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  cudaError_t e = ensure_sm_count();
  if (e != cudaSuccess) return e;
  switch (W.SP) {
    case 2: return run_pass2<2>(P, C, W, force, virial, st);
    case 4: return run_pass2<4>(P, C, W, force, virial, st);
    case 7: return run_pass2<7>(P, C, W, force, virial, st);
    default: return run_pass2<8>(P, C, W, force, virial, st);
  }
}
