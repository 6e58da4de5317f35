// nlist.cu — S1 cell binning and S2 neighbour search + format (Alg. 1; Fig. 2(a) :159).
//
// The paper formats a raw LAMMPS list with a CUB block sort on a packed 64-bit key (Eq. 11), which
// quantises r to 1e-8 A and needs j < 1e5.  Here (reading R10) the exact key of Alg. 1 line 4/7 — (alpha_j, |r_ij|
// as fp64, j) — is ranked by counting inside one thread block per atom, after a cell-list search on the GPU:
//   k_keys / k_scan / k_fill : counting sort of the atoms by (type, cell)            [S1]
//   k_nlist                  : stencil scan -> in-range hits in shared memory -> rank -> write slots / pad [S2]
// The displacement uses dp_displacement (reading R2) on a cell-sorted COPY of the raw coordinates (same bits).
#include "common.cuh"

// dp_displacement with the division and the square root skipped where their result is known in advance — the
// values produced are bit-identical to the pinned sequence (reading R2):
//   |d| < 0.4999 L          =>  |RN(d / L)| < 0.5            =>  k = rint(d / L) = 0
//   0.5001 L < |d| < 1.4999 L  =>  0.5 < |RN(d / L)| < 1.5   =>  k = +-1
//   r2 > rc^2 (1 + 1e-9)    =>  sqrt(r2) > rc                =>  not a neighbour, r is not needed (returns false)
__device__ __forceinline__ bool displacement_in_range(const double xi[3], const double xj[3], const double L[3],
                                                      double rc2_hi, double d[3], double &r) {
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const double dc = __dsub_rn(xj[c], xi[c]);
    const double a = fabs(dc);
    double k;
    if (a < 0.4999 * L[c]) k = 0.0;
    else if (a > 0.5001 * L[c] && a < 1.4999 * L[c]) k = copysign(1.0, dc);
    else k = rint(__ddiv_rn(dc, L[c]));
    d[c] = __fma_rn(-k, L[c], dc);
  }
  const double r2 = __fma_rn(d[2], d[2], __fma_rn(d[1], d[1], __dmul_rn(d[0], d[0])));
  if (r2 > rc2_hi) return false;
  r = __dsqrt_rn(r2);
  return true;
}

// ---------------------------------------------------------------------------------------------------------
__global__ void k_keys(DevModel P, DevGrid G, int n, const double *__restrict__ coord, const int *__restrict__ type,
                       int *__restrict__ key, int *__restrict__ count, DevStats *stats) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int ic[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double f = coord[3 * (size_t)i + c] / G.L[c];
    f -= floor(f);
    int v = (int)(f * G.nc[c]);
    v = v < 0 ? 0 : v;
    ic[c] = v >= G.nc[c] ? G.nc[c] - 1 : v;
  }
  int t = type[i];
  if (t < 0 || t >= P.ntypes) {
    atomicExch(&stats->err_type, 1);
    t = 0;
  }
  int k = t * G.ncell + (ic[0] * G.nc[1] + ic[1]) * G.nc[2] + ic[2];
  key[i] = k;
  atomicAdd(&count[k], 1);
}

// Exclusive scan of count[0..nkeys) by one block; also writes cursor = start and type_start[t] = start[t*ncell].
__global__ void k_scan(int nkeys, int ncell, int ntypes, const int *__restrict__ count, int *__restrict__ start,
                       int *__restrict__ cursor, int *__restrict__ type_start) {
  __shared__ int part[1024];
  const int tid = threadIdx.x;
  const int seg = (nkeys + 1023) / 1024;
  const int lo = tid * seg, hi = min(nkeys, lo + seg);
  int s = 0;
  for (int k = lo; k < hi; ++k) s += count[k];
  part[tid] = s;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {
    int v = tid >= off ? part[tid - off] : 0;
    __syncthreads();
    part[tid] += v;
    __syncthreads();
  }
  int run = tid ? part[tid - 1] : 0;
  for (int k = lo; k < hi; ++k) {
    start[k] = run;
    cursor[k] = run;
    if (k % ncell == 0) type_start[k / ncell] = run;
    run += count[k];
  }
  if (tid == 1023) {
    start[nkeys] = part[1023];
    type_start[ntypes] = part[1023];
  }
}

__global__ void k_fill(int n, const double *__restrict__ coord, const int *__restrict__ key, int *__restrict__ cursor,
                       int *__restrict__ s_idx, double *__restrict__ s_xyz) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int p = atomicAdd(&cursor[key[i]], 1);   // order inside a (type, cell) bucket is irrelevant: Alg. 1's key is total
  s_idx[p] = i;
  s_xyz[3 * (size_t)p + 0] = coord[3 * (size_t)i + 0];
  s_xyz[3 * (size_t)p + 1] = coord[3 * (size_t)i + 1];
  s_xyz[3 * (size_t)p + 2] = coord[3 * (size_t)i + 2];
}

cudaError_t launch_cell_sort(const DevModel &P, const DevGrid &G, int64_t natoms, const double *coord, const int *type,
                             int *key, int *count, int *start, int *cursor, int *s_idx, double *s_xyz,
                             DevStats *stats, cudaStream_t st) {
  const int nkeys = P.ntypes * G.ncell;
  cudaError_t e = cudaMemsetAsync(count, 0, sizeof(int) * (size_t)nkeys, st);
  if (e != cudaSuccess) return e;
  const int n = (int)natoms;
  if (n > 0) k_keys<<<(n + 255) / 256, 256, 0, st>>>(P, G, n, coord, type, key, count, stats);
  // type_start lives right behind start[nkeys + 1]
  k_scan<<<1, 1024, 0, st>>>(nkeys, G.ncell, P.ntypes, count, start, cursor, start + nkeys + 1);
  if (n > 0) k_fill<<<(n + 255) / 256, 256, 0, st>>>(n, coord, key, cursor, s_idx, s_xyz);
  DPB_LAUNCHED(n > 0 ? 3 : 1);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// S2.  One block per atom (sorted position p).  Shared memory: the stencil's (type, cell) ranges with a prefix sum,
// then the in-range hits S(i,k) = (alpha_j, |r_ij|, j) of Alg. 1 line 4.
#define NL_THREADS 128
#define NL_MAX_RANGES (27 * DPB_MAX_TYPES)

__global__ void __launch_bounds__(NL_THREADS)
k_nlist(DevModel P, DevGrid G, ChunkView C, const double *__restrict__ s_xyz, const int *__restrict__ start, int cap,
        int *__restrict__ nlist_out, DevStats *stats) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *hr = reinterpret_cast<double *>(smem_raw);            // [cap] distance
  int *hj = reinterpret_cast<int *>(hr + cap);                    // [cap] atom index j
  int *hp = hj + cap;                                             // [cap] sorted position of j
  int *ht = hp + cap;                                             // [cap] type of j
  __shared__ int r_start[NL_MAX_RANGES], r_pref[NL_MAX_RANGES + 1], r_type[NL_MAX_RANGES];
  __shared__ int n_ranges, n_hit, cnt[DPB_MAX_TYPES];

  const int tid = threadIdx.x;
  const int q = blockIdx.x;             // row inside the chunk
  const int p = C.p0 + q;               // sorted position
  const int i = C.s_idx[p];
  const double xi[3] = {s_xyz[3 * (size_t)p], s_xyz[3 * (size_t)p + 1], s_xyz[3 * (size_t)p + 2]};

  // stencil ranges: one thread per (type, stencil cell), then a serial compaction of the <= 27 ntypes entries
  __shared__ int c_start[NL_MAX_RANGES], c_cnt[NL_MAX_RANGES];
  for (int ent = tid; ent < 27 * P.ntypes; ent += NL_THREADS) {
    // cell of atom i, recomputed exactly as in k_keys
    int ic[3], lo[3], num[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double f = xi[c] / G.L[c];
      f -= floor(f);
      int v = (int)(f * G.nc[c]);
      v = v < 0 ? 0 : v;
      ic[c] = v >= G.nc[c] ? G.nc[c] - 1 : v;
      if (G.lo_mode[c]) { lo[c] = ic[c] - 1; num[c] = 3; } else { lo[c] = 0; num[c] = G.nc[c]; }
    }
    const int t = ent / 27, w = ent - 27 * t;
    const int a = w / 9, b = (w / 3) % 3, c = w % 3;
    int cntv = 0, s0 = 0;
    if (a < num[0] && b < num[1] && c < num[2]) {      // fewer than 3 cells in a dimension: each cell once
      const int ja = (lo[0] + a + G.nc[0]) % G.nc[0];
      const int jb = (lo[1] + b + G.nc[1]) % G.nc[1];
      const int jc = (lo[2] + c + G.nc[2]) % G.nc[2];
      const int k = t * G.ncell + (ja * G.nc[1] + jb) * G.nc[2] + jc;
      s0 = start[k];
      cntv = start[k + 1] - s0;
    }
    c_start[ent] = s0;
    c_cnt[ent] = cntv;
  }
  __syncthreads();
  if (tid == 0) {
    int nr = 0, run = 0;
    for (int e = 0; e < 27 * P.ntypes; ++e) {
      const int cv = c_cnt[e];
      if (cv > 0) {
        r_start[nr] = c_start[e]; r_pref[nr] = run; r_type[nr] = e / 27;
        run += cv; ++nr;
      }
    }
    r_pref[nr] = run;
    n_ranges = nr;
    n_hit = 0;
    for (int t = 0; t < DPB_MAX_TYPES; ++t) cnt[t] = 0;
  }
  __syncthreads();

  const double rc2_hi = P.rc * P.rc * (1.0 + 1e-9);
  const int ncand = r_pref[n_ranges];
  int rp = 0;
  for (int c = tid; c < ncand; c += NL_THREADS) {
    while (c >= r_pref[rp + 1]) ++rp;
    const int pj = r_start[rp] + (c - r_pref[rp]);
    if (pj == p) continue;                                         // j != i (reading R19)
    const double xj[3] = {s_xyz[3 * (size_t)pj], s_xyz[3 * (size_t)pj + 1], s_xyz[3 * (size_t)pj + 2]};
    double d[3], r;
    if (displacement_in_range(xi, xj, G.L, rc2_hi, d, r) && r <= P.rc) {   // "<=" as printed, PAPER.md:80 (R9)
      const int t = r_type[rp];
      atomicAdd(&cnt[t], 1);
      const int h = atomicAdd(&n_hit, 1);
      if (h < cap) { hr[h] = r; hj[h] = C.s_idx[pj]; hp[h] = pj; ht[h] = t; }
    }
  }
  __syncthreads();

  int nh = n_hit;
  if (nh > cap) {
    if (tid == 0) atomicExch(&stats->err_cap, 1);
    nh = cap;
  }
  int *nl_row = C.nl + (size_t)q * P.nm;
  double4 *dr_row = C.dr + (size_t)q * P.nm;
  int *out_row = nlist_out ? nlist_out + (size_t)i * P.nm : nullptr;

  // Alg. 1 line 7: order by (type, distance, index).  rank = number of hits of the same type that
  // precede this one; the first sel[t] go to section t (line 8-9, :186-193), the others are dropped (reading R8).
  for (int h = tid; h < nh; h += NL_THREADS) {
    const double r = hr[h];
    const int j = hj[h], t = ht[h];
    int rank = 0;
    for (int g = 0; g < nh; ++g) {
      const double rg = hr[g];
      rank += (ht[g] == t) && (rg < r || (rg == r && hj[g] < j));
    }
    if (rank < P.sel[t]) {
      const int slot = P.sec_start[t] + rank;
      nl_row[slot] = j;
      if (out_row) out_row[slot] = j;
      const int pj = hp[h];
      const double xj[3] = {s_xyz[3 * (size_t)pj], s_xyz[3 * (size_t)pj + 1], s_xyz[3 * (size_t)pj + 2]};
      double d[3], rr;
      dp_displacement(xi, xj, G.L, d, rr);
      dr_row[slot] = make_double4(d[0], d[1], d[2], rr);
    }
  }
  // padding: -1 at the tail of each section
  for (int slot = tid; slot < P.nm; slot += NL_THREADS) {
    int t = 0;
    while (slot >= P.sec_start[t + 1]) ++t;
    if (slot - P.sec_start[t] >= cnt[t]) {
      nl_row[slot] = -1;
      if (out_row) out_row[slot] = -1;
    }
  }
  if (tid < P.ntypes) {
    const int c = cnt[tid], kept = min(c, P.sel[tid]);
    C.nreal[(size_t)q * P.ntypes + tid] = kept;
    atomicMax(&stats->max_nei[tid], c);
    if (c > kept) atomicAdd(&stats->n_overflow, (unsigned long long)(c - kept));
    atomicAdd(&stats->n_real_pairs, (unsigned long long)kept);
  }
}

cudaError_t launch_nlist(const DevModel &P, const DevGrid &G, const ChunkView &C, const double *s_xyz,
                         const int *start, int cap, int *nlist_out, DevStats *stats, cudaStream_t st) {
  if (C.n <= 0) return cudaSuccess;
  const size_t smem = (size_t)cap * (sizeof(double) + 3 * sizeof(int));
  static size_t configured = 0;
  if (smem > 48 * 1024 && smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(k_nlist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  k_nlist<<<C.n, NL_THREADS, smem, st>>>(P, G, C, s_xyz, start, cap, nlist_out, stats);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// E = sum_i E_i (Eq. 1) in a fixed order: one block, strided partial sums then a tree.
__global__ void k_reduce_energy(long long n, const double *__restrict__ ei, double *__restrict__ e) {
  __shared__ double part[1024];
  double s = 0.0;
  for (long long k = threadIdx.x; k < n; k += 1024) s += ei[k];
  part[threadIdx.x] = s;
  __syncthreads();
  for (int off = 512; off > 0; off >>= 1) {
    if ((int)threadIdx.x < off) part[threadIdx.x] += part[threadIdx.x + off];
    __syncthreads();
  }
  if (threadIdx.x == 0) *e = part[0];
}

cudaError_t launch_reduce_energy(int64_t natoms, const double *atom_energy, double *energy, cudaStream_t st) {
  k_reduce_energy<<<1, 1024, 0, st>>>((long long)natoms, atom_energy, energy);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

// Test hook: copy the chunk's T / dT rows to buffers indexed by the original atom index.
__global__ void k_scatter_debug(DevModel P, ChunkView C, double *dbgT, double *dbgdT) {
  const int q = blockIdx.x;
  const int i = C.s_idx[C.p0 + q];
  const int n = P.M * 4;
  for (int k = threadIdx.x; k < n; k += blockDim.x) {
    if (dbgT) dbgT[(size_t)i * n + k] = C.T[(size_t)q * n + k];
    if (dbgdT) dbgdT[(size_t)i * n + k] = C.dT[(size_t)q * n + k];
  }
}

cudaError_t launch_scatter_debug(const DevModel &P, const ChunkView &C, double *dbgT, double *dbgdT, cudaStream_t st) {
  if (C.n <= 0 || (!dbgT && !dbgdT)) return cudaSuccess;
  k_scatter_debug<<<C.n, 128, 0, st>>>(P, C, dbgT, dbgdT);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}
