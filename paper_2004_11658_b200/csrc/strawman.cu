// strawman.cu — variant 2: the embedding stage the way the paper's section 3.2.3 runs it, as a measured
// strawman on B200.  What it keeps from the paper and the fused kernels (variant 1) drop:
//   * every GEMM runs over ALL padded slots of a (centre type a, neighbour type t) batch: rows = N_a x sel[t]
//     (4,096 x 92 = 376,832 rows for the O-H batch of the 12,288-atom water box); padded slots carry
//     R~ = 0, their G is computed and then multiplied by zero (:105);
//   * the bias is folded into the GEMM: the activations carry a constant-1 column and the weight matrix a bias row (:264);
//   * the concat skip (x, x) of Eq. 9 is a GEMM with (I, I) (Eq. 12, :266-271), accumulated onto tanh(xW + b);
//   * tanh and its gradient 1 - tanh^2 are separate element-wise kernels (:273);
//   * G and every activation are materialised in HBM between the kernels (Eq. 13, :279-290) and read by the backward
//     pass, which is reverse mode (delta W^T GEMMs and the transposed (I, I) fold), as TensorFlow's autodiff does.
// The GEMMs are this library's own DMMA tiles (fit_dmma.cu, v1_plain_gemm), not cuBLAS.  The fitting stage is variant
// 1's.  Same results as the other variants (tests compare it with the oracle); only the time and the bytes differ.
#include "v1_kernels.cuh"

#include <climits>
#include <vector>

static int ru16(int x) { return (x + 15) / 16 * 16; }

// padded matrices of one net, in order; sizes in doubles
struct V2Off { size_t B0, B1, II1, B2, II2, B2T, II2T, B1T, II1T, B0T, total; };
static V2Off v2_offsets(int LD0, int LD1, int LD2) {
  V2Off o;
  size_t p = 0;
  o.B0 = p; p += 2 * (size_t)LD0;
  o.B1 = p; p += (size_t)LD0 * LD1;
  o.II1 = p; p += (size_t)LD0 * LD1;
  o.B2 = p; p += (size_t)LD1 * LD2;
  o.II2 = p; p += (size_t)LD1 * LD2;
  o.B2T = p; p += (size_t)LD2 * LD1;
  o.II2T = p; p += (size_t)LD2 * LD1;
  o.B1T = p; p += (size_t)LD1 * LD0;
  o.II1T = p; p += (size_t)LD1 * LD0;
  o.B0T = p; p += (size_t)LD0 * 2;
  o.total = p;
  return o;
}

cudaError_t v2_prepare_weights(const DevModel &P, const double *emb_h, V2Weights &W) {
  const int s1 = P.s1;
  W.LD0 = ru16(s1 + 1); W.LD1 = ru16(2 * s1 + 1); W.LD2 = ru16(4 * s1);
  const int LD0 = W.LD0, LD1 = W.LD1, LD2 = W.LD2;
  const V2Off o = v2_offsets(LD0, LD1, LD2);
  W.net_stride = (long long)o.total;
  const int nets = P.ntypes * P.ntypes;
  std::vector<double> h((size_t)nets * o.total, 0.0);
  for (int k = 0; k < nets; ++k) {
    const double *W0 = emb_h + (size_t)k * P.emb_net_size, *b0 = W0 + s1, *W1 = b0 + s1, *b1 = W1 + (size_t)s1 * 2 * s1,
                 *W2 = b1 + 2 * s1, *b2 = W2 + (size_t)2 * s1 * 4 * s1;
    double *q = h.data() + (size_t)k * o.total;
    for (int c = 0; c < s1; ++c) { q[o.B0 + c] = W0[c]; q[o.B0 + LD0 + c] = b0[c]; q[o.B0T + 2 * (size_t)c] = W0[c]; }
    for (int r = 0; r < s1; ++r)
      for (int c = 0; c < 2 * s1; ++c) {
        q[o.B1 + (size_t)r * LD1 + c] = W1[(size_t)r * 2 * s1 + c];
        q[o.B1T + (size_t)c * LD0 + r] = W1[(size_t)r * 2 * s1 + c];
      }
    for (int c = 0; c < 2 * s1; ++c) q[o.B1 + (size_t)s1 * LD1 + c] = b1[c];            // bias row (the constant-1 column)
    for (int r = 0; r < s1; ++r)
      for (int e = 0; e < 2; ++e) {
        q[o.II1 + (size_t)r * LD1 + e * s1 + r] = 1.0;                                     // (I, I), Eq. 12
        q[o.II1T + (size_t)(e * s1 + r) * LD0 + r] = 1.0;
      }
    q[o.II1 + (size_t)s1 * LD1 + 2 * s1] = 1.0;                                            // carries the constant 1 along
    for (int r = 0; r < 2 * s1; ++r)
      for (int c = 0; c < 4 * s1; ++c) {
        q[o.B2 + (size_t)r * LD2 + c] = W2[(size_t)r * 4 * s1 + c];
        q[o.B2T + (size_t)c * LD1 + r] = W2[(size_t)r * 4 * s1 + c];
      }
    for (int c = 0; c < 4 * s1; ++c) q[o.B2 + (size_t)(2 * s1) * LD2 + c] = b2[c];
    for (int r = 0; r < 2 * s1; ++r)
      for (int e = 0; e < 2; ++e) {
        q[o.II2 + (size_t)r * LD2 + e * 2 * s1 + r] = 1.0;
        q[o.II2T + (size_t)(e * 2 * s1 + r) * LD1 + r] = 1.0;
      }
  }
  cudaError_t e = cudaMalloc(&W.buf, sizeof(double) * h.size());
  if (e != cudaSuccess) return e;
  e = cudaMemcpy(W.buf, h.data(), sizeof(double) * h.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return e;
  const int rg[2] = {0, INT_MAX};
  e = cudaMalloc(&W.range, sizeof(rg));
  if (e != cudaSuccess) return e;
  e = cudaMemcpy(W.range, rg, sizeof(rg), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return e;
  W.ready = true;
  return cudaSuccess;
}

void v2_release_weights(V2Weights &W) {
  if (W.buf) cudaFree(W.buf);
  if (W.range) cudaFree(W.range);
  W.buf = nullptr; W.range = nullptr; W.ready = false;
}

// doubles per padded slot: kept from pass 1 to pass 2 (R~, H0, U1, U2, G) and per-batch scratch (A0, H1 / D1, dG, D0, DX, dR~)
static size_t v2_kept(const V2Weights &W) { return 4 + (size_t)W.LD0 + W.LD1 + 2 * (size_t)W.LD2; }
static size_t v2_scratch(const V2Weights &W) { return 2 + (size_t)W.LD1 + W.LD2 + W.LD0 + 2 + 4; }
size_t v2_slot_bytes(const V2Weights &W) { return sizeof(double) * (v2_kept(W) + v2_scratch(W)); }

// ---- kernels --------------------------------------------------------------------------------------------------------
// S3 for a batch: R~ of every padded slot (zero when padded) and the layer-0 input (s, 1).
__global__ void k_v2_env(DevModel P, ChunkView C, int t, int row_lo, long long nslot, double *__restrict__ Rt,
                         double *__restrict__ A0) {
  const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= nslot) return;
  const int sel = P.sel[t], qa = row_lo + (int)(w / sel), k = (int)(w % sel);
  double e[4] = {0.0, 0.0, 0.0, 0.0};
  if (k < C.nreal[(size_t)qa * P.ntypes + t]) {
    const double4 v = C.dr[(size_t)qa * P.nm + P.sec_start[t] + k];
    double sw, dw;
    dp_switch(v.w, P.rcs, P.rc, sw, dw);
    const double ir = 1.0 / v.w, s = sw * ir, sr = s * ir;
    e[0] = s; e[1] = sr * v.x; e[2] = sr * v.y; e[3] = sr * v.z;
  }
  reinterpret_cast<double4 *>(Rt)[w] = make_double4(e[0], e[1], e[2], e[3]);
  reinterpret_cast<double2 *>(A0)[w] = make_double2(e[0], 1.0);
}

// separate activation kernel: X <- tanh(X) on the first `width` columns; one_col (>= 0) is set to 1
__global__ void k_v2_tanh(long long nslot, double *__restrict__ X, int ld, int width, int one_col) {
  const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= nslot * ld) return;
  const int c = (int)(w % ld);
  double v = 0.0;
  if (c < width) v = dp_tanh(X[w]);
  else if (c == one_col) v = 1.0;
  X[w] = v;
}

// separate tanh-grad kernel: U <- D (1 - U^2)
__global__ void k_v2_tanh_grad(long long n, const double *__restrict__ D, double *__restrict__ U) {
  const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= n) return;
  const double u = U[w];
  U[w] = D[w] * (1.0 - u * u);
}

// S5 left factor: T_i (+)= G^T R~ over the sel[t] slots of atom qa (Eq. 4).  Block = atom, thread = feature.
__global__ void k_v2_GtR(DevModel P, ChunkView C, int t, int row_lo, const double *__restrict__ G, int ld,
                         const double *__restrict__ Rt, int accumulate) {
  const int qa = row_lo + blockIdx.x, sel = P.sel[t];
  const size_t s0 = (size_t)blockIdx.x * sel;
  extern __shared__ double4 rs[];
  for (int k = threadIdx.x; k < sel; k += blockDim.x) rs[k] = reinterpret_cast<const double4 *>(Rt)[s0 + k];
  __syncthreads();
  for (int b = threadIdx.x; b < P.M; b += blockDim.x) {
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    for (int k = 0; k < sel; ++k) {
      const double g = G[(s0 + k) * ld + b];
      const double4 e = rs[k];
      a0 = fma(g, e.x, a0); a1 = fma(g, e.y, a1); a2 = fma(g, e.z, a2); a3 = fma(g, e.w, a3);
    }
    double *dst = C.T + ((size_t)qa * P.M + b) * 4;
    if (accumulate) { dst[0] += a0; dst[1] += a1; dst[2] += a2; dst[3] += a3; }
    else { dst[0] = a0; dst[1] = a1; dst[2] = a2; dst[3] = a3; }
  }
}

// backward of the contraction: dG[k][b] = sum_c dT[b][c] R~[k][c] (all LD2 columns written, pads zero);
// dR~[k][c] = sum_b dT[b][c] G[k][b].  Block = atom.
__global__ void k_v2_dG(DevModel P, ChunkView C, int t, int row_lo, const double *__restrict__ G, int ld,
                        const double *__restrict__ Rt, double *__restrict__ dG, double *__restrict__ dRt) {
  const int qa = row_lo + blockIdx.x, sel = P.sel[t], M = P.M;
  const size_t s0 = (size_t)blockIdx.x * sel;
  extern __shared__ double4 dts[];                          // [M] dT rows of the atom
  for (int b = threadIdx.x; b < M; b += blockDim.x) {
    const double *src = C.dT + dt_offset(P, C, qa, b);
    dts[b] = make_double4(src[0], src[1], src[2], src[3]);
  }
  __syncthreads();
  for (long long w = threadIdx.x; w < (long long)sel * ld; w += blockDim.x) {
    const int k = (int)(w / ld), b = (int)(w % ld);
    double v = 0.0;
    if (b < M) {
      const double4 e = reinterpret_cast<const double4 *>(Rt)[s0 + k], d = dts[b];
      v = fma(d.x, e.x, fma(d.y, e.y, fma(d.z, e.z, d.w * e.w)));
    }
    dG[(s0 + k) * ld + b] = v;
  }
  for (int k = threadIdx.x; k < sel; k += blockDim.x) {
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    for (int b = 0; b < M; ++b) {
      const double g = G[(s0 + k) * ld + b];
      const double4 d = dts[b];
      a0 = fma(d.x, g, a0); a1 = fma(d.y, g, a1); a2 = fma(d.z, g, a2); a3 = fma(d.w, g, a3);
    }
    reinterpret_cast<double4 *>(dRt)[s0 + k] = make_double4(a0, a1, a2, a3);
  }
}

// ProdForce / ProdVirial for a batch: dR~[0] += dx, chain to the displacement (O10), scatter.
__global__ void k_v2_force(DevModel P, ChunkView C, int t, int row_lo, long long nslot, const double *__restrict__ dRt,
                           const double *__restrict__ DX, double *__restrict__ force, double *__restrict__ virial) {
  const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double vir[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
  if (w < nslot) {
    const int sel = P.sel[t], qa = row_lo + (int)(w / sel), k = (int)(w % sel);
    if (k < C.nreal[(size_t)qa * P.ntypes + t]) {
      const size_t slot = (size_t)qa * P.nm + P.sec_start[t] + k;
      const double4 dv = C.dr[slot];
      const double4 p = reinterpret_cast<const double4 *>(dRt)[w];
      const double dR0 = p.x + DX[2 * w];
      const double r = dv.w, ir = 1.0 / r;
      double sw, dw;
      dp_switch(r, P.rcs, P.rc, sw, dw);
      const double s = sw * ir, qq = s * ir, sp = dw * ir - sw * ir * ir, qp = sp * ir - s * ir * ir;
      const double dot = p.y * dv.x + p.z * dv.y + p.w * dv.z;
      const double cm = (dR0 * sp + qp * dot) * ir;
      const double f[3] = {fma(cm, dv.x, qq * p.y), fma(cm, dv.y, qq * p.z), fma(cm, dv.z, qq * p.w)};
      const int j = C.nl[slot], i = C.s_idx[C.p0 + qa];
      const double d[3] = {dv.x, dv.y, dv.z};
      if (force)
#pragma unroll
        for (int c = 0; c < 3; ++c) { atomicAdd(&force[3 * (size_t)j + c], -f[c]); atomicAdd(&force[3 * (size_t)i + c], f[c]); }
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) vir[3 * a + b] = -d[a] * f[b];
    }
  }
  if (virial) {
#pragma unroll
    for (int k = 0; k < 9; ++k) {
      double v = vir[k];
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
      if ((threadIdx.x & 31) == 0 && v != 0.0) atomicAdd(&virial[k], v);
    }
  }
}

// ---- host ------------------------------------------------------------------------------------------------------------
struct V2Batch { int a, t, row_lo, na; long long nslot, off; };

static std::vector<V2Batch> v2_batches(const DevModel &P, const ChunkView &C, const int *ts) {
  std::vector<V2Batch> out;
  long long off = 0;
  for (int a = 0; a < P.ntypes; ++a) {
    const int lo = (ts[a] > C.p0 ? ts[a] : C.p0) - C.p0, hi = (ts[a + 1] < C.p0 + C.n ? ts[a + 1] : C.p0 + C.n) - C.p0;
    for (int t = 0; t < P.ntypes; ++t) {
      V2Batch b{a, t, lo, hi > lo ? hi - lo : 0, 0, off};
      b.nslot = (long long)b.na * P.sel[t];
      off += b.nslot;
      out.push_back(b);
    }
  }
  return out;
}

struct V2Bufs { double *Rt, *H0, *U1, *U2, *G, *A0, *H1, *dG, *D0, *DX, *dRt; };

// kept arrays are laid out [all slots of the chunk]; scratch arrays are sized for the chunk as well (a batch uses a prefix)
static V2Bufs v2_bufs(const DevModel &P, const ChunkView &C, const V2Weights &W, void *ws) {
  const size_t ns = (size_t)C.n * P.nm;
  double *p = reinterpret_cast<double *>(ws);
  V2Bufs B;
  B.Rt = p; p += 4 * ns;
  B.H0 = p; p += (size_t)W.LD0 * ns;
  B.U1 = p; p += (size_t)W.LD1 * ns;
  B.U2 = p; p += (size_t)W.LD2 * ns;
  B.G = p; p += (size_t)W.LD2 * ns;
  B.A0 = p; p += 2 * ns;
  B.H1 = p; p += (size_t)W.LD1 * ns;
  B.dG = p; p += (size_t)W.LD2 * ns;
  B.D0 = p; p += (size_t)W.LD0 * ns;
  B.DX = p; p += 2 * ns;
  B.dRt = p;
  return B;
}

#define V2(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return e_; } while (0)
static unsigned nblk(long long n) { return (unsigned)((n + 255) / 256); }

cudaError_t v2_pass1(const DevModel &P, const ChunkView &C, const V2Weights &W, const int *ts, void *ws, cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  const V2Bufs B = v2_bufs(P, C, W, ws);
  const V2Off o = v2_offsets(W.LD0, W.LD1, W.LD2);
  const int s1 = P.s1, LD0 = W.LD0, LD1 = W.LD1, LD2 = W.LD2;
  int stored_a = -1;                                       // centre type whose T rows already hold a first contribution
  for (const V2Batch &b : v2_batches(P, C, ts)) {
    if (b.na > 0 && b.t == 0 && P.sel[0] == 0) {           // no slots of type 0: T starts from zero
      V2(cudaMemsetAsync(C.T + (size_t)b.row_lo * P.M * 4, 0, sizeof(double) * (size_t)b.na * P.M * 4, st));
      stored_a = b.a;
    }
    if (b.nslot == 0) continue;
    const double *net = W.buf + (size_t)(b.a * P.ntypes + b.t) * W.net_stride;
    double *Rt = B.Rt + 4 * b.off, *H0 = B.H0 + (size_t)LD0 * b.off, *U1 = B.U1 + (size_t)LD1 * b.off,
           *U2 = B.U2 + (size_t)LD2 * b.off, *G = B.G + (size_t)LD2 * b.off;
    k_v2_env<<<nblk(b.nslot), 256, 0, st>>>(P, C, b.t, b.row_lo, b.nslot, Rt, B.A0);
    DPB_LAUNCHED(1);
    // layer 0 (Eq. 8): X0 = (s, 1) (W0; b0), H0 = tanh(X0), constant-1 column behind it
    V2(v1_plain_gemm(b.nslot, B.A0, 2, net + o.B0, LD0, 2, LD0, nullptr, H0, LD0, W.range, st));
    k_v2_tanh<<<nblk(b.nslot * LD0), 256, 0, st>>>(b.nslot, H0, LD0, s1, s1);
    DPB_LAUNCHED(1);
    // layer 1 (Eq. 9, 12): U1 = tanh((H0, 1) (W1; b1)), H1 = H0 (I, I) + U1
    V2(v1_plain_gemm(b.nslot, H0, LD0, net + o.B1, LD1, LD0, LD1, nullptr, U1, LD1, W.range, st));
    k_v2_tanh<<<nblk(b.nslot * LD1), 256, 0, st>>>(b.nslot, U1, LD1, 2 * s1, -1);
    DPB_LAUNCHED(1);
    V2(v1_plain_gemm(b.nslot, H0, LD0, net + o.II1, LD1, LD0, LD1, U1, B.H1, LD1, W.range, st));
    // layer 2: U2 = tanh((H1, 1) (W2; b2)), G = H1 (I, I) + U2
    V2(v1_plain_gemm(b.nslot, B.H1, LD1, net + o.B2, LD2, LD1, LD2, nullptr, U2, LD2, W.range, st));
    k_v2_tanh<<<nblk(b.nslot * LD2), 256, 0, st>>>(b.nslot, U2, LD2, 4 * s1, -1);
    DPB_LAUNCHED(1);
    V2(v1_plain_gemm(b.nslot, B.H1, LD1, net + o.II2, LD2, LD1, LD2, U2, G, LD2, W.range, st));
    // T_i (+)= G^T R~
    k_v2_GtR<<<b.na, 128, sizeof(double4) * P.sel[b.t], st>>>(P, C, b.t, b.row_lo, G, LD2, Rt, stored_a == b.a);
    DPB_LAUNCHED(1);
    stored_a = b.a;
  }
  return cudaGetLastError();
}

cudaError_t v2_pass2(const DevModel &P, const ChunkView &C, const V2Weights &W, const int *ts, void *ws, double *force,
                     double *virial, cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  const V2Bufs B = v2_bufs(P, C, W, ws);
  const V2Off o = v2_offsets(W.LD0, W.LD1, W.LD2);
  const int LD0 = W.LD0, LD1 = W.LD1, LD2 = W.LD2;
  for (const V2Batch &b : v2_batches(P, C, ts)) {
    if (b.nslot == 0) continue;
    const double *net = W.buf + (size_t)(b.a * P.ntypes + b.t) * W.net_stride;
    double *Rt = B.Rt + 4 * b.off, *H0 = B.H0 + (size_t)LD0 * b.off, *U1 = B.U1 + (size_t)LD1 * b.off,
           *U2 = B.U2 + (size_t)LD2 * b.off, *G = B.G + (size_t)LD2 * b.off;
    double *D1 = B.H1;                                     // dE/dH1 (scratch shared with the forward H1)
    k_v2_dG<<<b.na, 256, sizeof(double4) * P.M, st>>>(P, C, b.t, b.row_lo, G, LD2, Rt, B.dG, B.dRt);
    DPB_LAUNCHED(1);
    // delta2 = dG (1 - U2^2); dH1 = delta2 W2^T + dG (I, I)^T
    k_v2_tanh_grad<<<nblk(b.nslot * LD2), 256, 0, st>>>(b.nslot * LD2, B.dG, U2);
    DPB_LAUNCHED(1);
    V2(v1_plain_gemm(b.nslot, U2, LD2, net + o.B2T, LD1, LD2, LD1, nullptr, D1, LD1, W.range, st));
    V2(v1_plain_gemm(b.nslot, B.dG, LD2, net + o.II2T, LD1, LD2, LD1, D1, D1, LD1, W.range, st));
    // delta1 = dH1 (1 - U1^2); dH0 = delta1 W1^T + dH1 (I, I)^T
    k_v2_tanh_grad<<<nblk(b.nslot * LD1), 256, 0, st>>>(b.nslot * LD1, D1, U1);
    DPB_LAUNCHED(1);
    V2(v1_plain_gemm(b.nslot, U1, LD1, net + o.B1T, LD0, LD1, LD0, nullptr, B.D0, LD0, W.range, st));
    V2(v1_plain_gemm(b.nslot, D1, LD1, net + o.II1T, LD0, LD1, LD0, B.D0, B.D0, LD0, W.range, st));
    // delta0 = dH0 (1 - H0^2); dx = delta0 W0^T
    k_v2_tanh_grad<<<nblk(b.nslot * LD0), 256, 0, st>>>(b.nslot * LD0, B.D0, H0);
    DPB_LAUNCHED(1);
    V2(v1_plain_gemm(b.nslot, H0, LD0, net + o.B0T, 2, LD0, 2, nullptr, B.DX, 2, W.range, st));
    k_v2_force<<<nblk(b.nslot), 256, 0, st>>>(P, C, b.t, b.row_lo, b.nslot, B.dRt, B.DX, force, virial);
    DPB_LAUNCHED(1);
  }
  return cudaGetLastError();
}
