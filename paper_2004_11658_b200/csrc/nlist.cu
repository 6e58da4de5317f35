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
__device__ __forceinline__ int sort_key(const DevModel &P, const DevGrid &G, int i, const double *__restrict__ coord,
                                        const int *__restrict__ type, DevStats *stats) {
  int ic[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const double x = coord[3 * (size_t)i + c] - G.org[c];
    if (G.open && !(x >= 0.0 && x <= G.ext[c])) atomicExch(&stats->err_bounds, 1);
    double f = x / G.L[c];
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
  if (G.ngrp == 2 && i >= G.nloc) t += P.ntypes;                   // ghosts: behind every local atom
  return t * G.ncell + (ic[0] * G.nc[1] + ic[1]) * G.nc[2] + ic[2];
}

__global__ void k_keys(DevModel P, DevGrid G, int n, const double *__restrict__ coord, const int *__restrict__ type,
                       int *__restrict__ key, int *__restrict__ count, DevStats *stats) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int k = sort_key(P, G, i, coord, type, stats);
  key[i] = k;
  atomicAdd(&count[k], 1);
}

// Exclusive scan of count[0..nkeys) by one block; also writes cursor = start and type_start[t] = start[t*ncell].
__device__ __forceinline__ void scan_block(int nkeys, int ncell, int ntypes, const int *count, int *start, int *cursor,
                                           int *type_start, int *part) {
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

__global__ void k_scan(int nkeys, int ncell, int ntypes, const int *__restrict__ count, int *__restrict__ start,
                       int *__restrict__ cursor, int *__restrict__ type_start) {
  __shared__ int part[1024];
  scan_block(nkeys, ncell, ntypes, count, start, cursor, type_start, part);
}

__device__ __forceinline__ void fill_one(int i, const double *__restrict__ coord, const int *key, int *cursor,
                                         int *__restrict__ s_idx, double *__restrict__ s_xyz, int *__restrict__ pos_of) {
  int p = atomicAdd(&cursor[key[i]], 1);   // order inside a (type, cell) bucket is irrelevant: Alg. 1's key is total
  s_idx[p] = i;
  if (pos_of) pos_of[i] = p;
  s_xyz[3 * (size_t)p + 0] = coord[3 * (size_t)i + 0];
  s_xyz[3 * (size_t)p + 1] = coord[3 * (size_t)i + 1];
  s_xyz[3 * (size_t)p + 2] = coord[3 * (size_t)i + 2];
}

__global__ void k_fill(int n, const double *__restrict__ coord, const int *__restrict__ key, int *__restrict__ cursor,
                       int *__restrict__ s_idx, double *__restrict__ s_xyz, int *__restrict__ pos_of) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  fill_one(i, coord, key, cursor, s_idx, s_xyz, pos_of);
}

// Small systems: keys, scan and fill by ONE block (a 192-atom evaluation is bound by its chain of dependent launches:
// three launches and a memset become one; same arithmetic, same arrays).
#define SORT_SMALL_N 4096
__global__ void __launch_bounds__(1024)
k_sort_small(DevModel P, DevGrid G, int n, int nkeys, const double *__restrict__ coord, const int *__restrict__ type,
             int *key, int *count, int *start, int *cursor, int *__restrict__ s_idx, double *__restrict__ s_xyz,
             DevStats *stats, int *__restrict__ pos_of, ZeroJobs Z) {
  __shared__ int part[1024];
  pdl_trigger();                                           // the list kernel behind may be scheduled now (it waits in pdl_wait)
  for (int k = threadIdx.x; k < nkeys; k += 1024) count[k] = 0;
  if (Z.stats) for (int k = threadIdx.x; k < Z.stats_bytes / 4; k += 1024) reinterpret_cast<int *>(Z.stats)[k] = 0;
  if (Z.counters) for (int k = threadIdx.x; k < Z.ncounters; k += 1024) Z.counters[k] = 0;
  __syncthreads();
  for (int i = threadIdx.x; i < n; i += 1024) {
    const int k = sort_key(P, G, i, coord, type, stats);
    key[i] = k;
    atomicAdd(&count[k], 1);
  }
  __syncthreads();
  scan_block(nkeys, G.ncell, P.ntypes * G.ngrp, count, start, cursor, start + nkeys + 1, part);
  __syncthreads();
  for (int i = threadIdx.x; i < n; i += 1024) fill_one(i, coord, key, cursor, s_idx, s_xyz, pos_of);
}

cudaError_t launch_cell_sort(const DevModel &P, const DevGrid &G, int64_t natoms, const double *coord, const int *type,
                             int *key, int *count, int *start, int *cursor, int *s_idx, double *s_xyz,
                             DevStats *stats, cudaStream_t st, int *pos_of, const ZeroJobs *zero) {
  const int nkeys = P.ntypes * G.ngrp * G.ncell;
  const int n = (int)natoms;
  ZeroJobs Z{};
  if (zero) Z = *zero;
  if (n > 0 && n <= SORT_SMALL_N && nkeys <= 4 * SORT_SMALL_N) {
    k_sort_small<<<1, 1024, 0, st>>>(P, G, n, nkeys, coord, type, key, count, start, cursor, s_idx, s_xyz, stats, pos_of, Z);
    DPB_LAUNCHED(1);
    return cudaGetLastError();
  }
  cudaError_t e = cudaMemsetAsync(count, 0, sizeof(int) * (size_t)nkeys, st);
  if (e == cudaSuccess && Z.stats) e = cudaMemsetAsync(Z.stats, 0, (size_t)Z.stats_bytes, st);
  if (e == cudaSuccess && Z.counters) e = cudaMemsetAsync(Z.counters, 0, sizeof(int) * (size_t)Z.ncounters, st);
  if (e != cudaSuccess) return e;
  if (n > 0) k_keys<<<(n + 255) / 256, 256, 0, st>>>(P, G, n, coord, type, key, count, stats);
  // type_start lives right behind start[nkeys + 1]
  k_scan<<<1, 1024, 0, st>>>(nkeys, G.ncell, P.ntypes * G.ngrp, count, start, cursor, start + nkeys + 1);
  if (n > 0) k_fill<<<(n + 255) / 256, 256, 0, st>>>(n, coord, key, cursor, s_idx, s_xyz, pos_of);
  DPB_LAUNCHED(n > 0 ? 3 : 1);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// S2.  One block per atom (sorted position p).  Shared memory: the stencil's (type, cell-run) ranges with a prefix sum,
// then the in-range hits S(i,k) = (alpha_j, |r_ij|, j) of Alg. 1 line 4.
// Cells are numbered z-fastest, so the three z-neighbours of a stencil column are one contiguous run of sorted
// positions (two runs when the column wraps around the box): 9 x 2 entries per type instead of 27.
#define NL_THREADS 128
#define NL_BUCKETS 32           // distance buckets per type, uniform in r^3: the ranking only compares inside a bucket

struct __align__(16) NlHit { double r; int j; int t; };


// MODE 0: candidates from the cell stencil (cells >= r_c).  MODE 1 (MD, rebuild step): cells >= r_c + skin; every
// candidate within r_c + skin is also appended to the atom's raw list (the paper's LAMMPS skin list, PAPER.md:193,
// :298).  MODE 2 (MD, reuse step): candidates are the raw list — Alg. 1 proper: format a raw list.
// ZERO: the instantiation of small evaluations that also clears the later stages' buffers (ZeroJobs); the other one must
// not see that code at all (its 48 registers and 10 blocks per SM are tuned: +4-6 % with the test compiled in).
template <int MODE, bool ZERO = false>
__global__ void __launch_bounds__(NL_THREADS, MODE == 0 ? 10 : 1)   // 48 registers: 10 blocks per SM (64 gave 8: +11 %)
k_nlist(DevModel P, DevGrid G, ChunkView C, const double *__restrict__ s_xyz, const int *__restrict__ start, int cap,
        int *__restrict__ nlist_out, DevStats *stats, NlRaw R, ZeroJobs Z) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  if (ZERO) pdl_wait();                                             // launched behind k_sort_small with dpb_launch_pdl
  if (ZERO) {                                                       // small evaluations: the memsets of the later stages
    const int zb = blockIdx.x, zt = threadIdx.x, zn = blockDim.x;
    if (Z.T) for (int k = zt; k < Z.t_len; k += zn) Z.T[(size_t)zb * Z.t_len + k] = 0.0;
    if (Z.Z0) for (int k = zt; k < Z.z_len; k += zn) Z.Z0[(size_t)zb * Z.z_len + k] = 0.0;
    if (Z.force && zt < 3) Z.force[3 * (size_t)zb + zt] = 0.0;
    if (Z.virial && zb == 0 && zt < 9) Z.virial[zt] = 0.0;
  }
  NlHit *hit = reinterpret_cast<NlHit *>(smem_raw);               // [cap] (distance, atom index j, type of j)
  int *hp = reinterpret_cast<int *>(hit + cap);                   // [cap] sorted position of j
  int *order = hp + cap;                                          // [cap] hits grouped by (type, distance bucket)
  __shared__ int bcnt[DPB_MAX_TYPES * NL_BUCKETS], bstart[DPB_MAX_TYPES * NL_BUCKETS + 1];
  const int nent_all = 18 * P.ntypes * G.ngrp;                    // stencil ranges: sized by the launcher
  int *r_start = order + cap, *r_pref = r_start + nent_all, *r_type = r_pref + nent_all + 1;
  __shared__ int n_ranges, n_hit, n_raw, cnt[DPB_MAX_TYPES];

  const int tid = threadIdx.x, lane = tid & 31, nthr = blockDim.x;      // 64 or 128 threads (launch_nlist)
  const int q = blockIdx.x;             // row inside the chunk
  const int p = C.p0 + q;               // sorted position
  const int i = C.s_idx[p];
  const double xi[3] = {s_xyz[3 * (size_t)p], s_xyz[3 * (size_t)p + 1], s_xyz[3 * (size_t)p + 2]};

  if (tid < DPB_MAX_TYPES) cnt[tid] = 0;
  for (int k = tid; k < DPB_MAX_TYPES * NL_BUCKETS; k += nthr) bcnt[k] = 0;
  const double binv = (double)NL_BUCKETS / (P.rc * P.rc * P.rc);
  if (tid == 0) { n_hit = 0; n_raw = 0; }
  // stencil ranges, built and compacted by warp 0 (ballot + warp scan): entry = (type, x offset, y offset, part)
  if (MODE != 2 && tid < 32) {
    int ic[3], lo[3], num[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {                                  // cell of atom i, recomputed exactly as in k_keys
      double f = (xi[c] - G.org[c]) / G.L[c];
      f -= floor(f);
      int v = (int)(f * G.nc[c]);
      v = v < 0 ? 0 : v;
      ic[c] = v >= G.nc[c] ? G.nc[c] - 1 : v;
      if (G.lo_mode[c]) { lo[c] = ic[c] - 1; num[c] = 3; } else { lo[c] = 0; num[c] = G.nc[c]; }
    }
    // z runs: [z0, z0 + len0) and, if the stencil wraps, [z1, z1 + len1)
    int z0, len0, z1 = 0, len1 = 0;
    if (!G.lo_mode[2]) { z0 = 0; len0 = G.nc[2]; }
    else if (lo[2] < 0) { z0 = 0; len0 = 2; z1 = G.nc[2] - 1; len1 = 1; }
    else if (lo[2] + 2 >= G.nc[2]) { z0 = lo[2]; len0 = 2; z1 = 0; len1 = 1; }
    else { z0 = lo[2]; len0 = 3; }
    const int nent = nent_all;
    int nr = 0, run = 0;
    for (int base = 0; base < nent; base += 32) {
      const int ent = base + lane;
      int cntv = 0, s0 = 0, t = 0;
      if (ent < nent) {
        const int pt = ent / 18;                                     // pseudo-type: (group, type)
        t = pt >= P.ntypes ? pt - P.ntypes : pt;
        const int w = ent - 18 * pt, part = w & 1, ab = w >> 1, a = ab / 3, b = ab - 3 * a;
        const int zz = part ? z1 : z0, ln = part ? len1 : len0;
        if (a < num[0] && b < num[1] && ln > 0) {                  // fewer than 3 cells in a dimension: each cell once
          const int ja = (lo[0] + a + G.nc[0]) % G.nc[0];
          const int jb = (lo[1] + b + G.nc[1]) % G.nc[1];
          const int k = pt * G.ncell + (ja * G.nc[1] + jb) * G.nc[2] + zz;
          s0 = start[k];
          cntv = start[k + ln] - s0;
        }
      }
      const unsigned m = __ballot_sync(0xffffffffu, cntv > 0);
      int incl = cntv;                                             // inclusive warp scan of the counts
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += v;
      }
      if (cntv > 0) {
        const int pos = nr + __popc(m & ((1u << lane) - 1u));
        r_start[pos] = s0; r_pref[pos] = run + incl - cntv; r_type[pos] = t;
      }
      nr += __popc(m);
      run += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) { r_pref[nr] = run; n_ranges = nr; }
  }
  __syncthreads();

  const double rc2_hi = P.rc * P.rc * (1.0 + 1e-9);
  if (MODE != 2) {
    const int ncand = r_pref[n_ranges];
    const double lim = MODE == 1 ? R.rs2_hi : rc2_hi;
    int *raw_row = MODE == 1 ? R.raw + (size_t)p * R.cap : nullptr;
    int rp = 0;
    for (int c = tid; c < ncand; c += nthr) {
      while (c >= r_pref[rp + 1]) ++rp;
      const int pj = r_start[rp] + (c - r_pref[rp]);
      if (pj == p) continue;                                         // j != i (reading R19)
      const double xj[3] = {s_xyz[3 * (size_t)pj], s_xyz[3 * (size_t)pj + 1], s_xyz[3 * (size_t)pj + 2]};
      double d[3], r;
      if (displacement_in_range(xi, xj, G.L, lim, d, r)) {
        if (MODE == 1) {
          const int k = atomicAdd(&n_raw, 1);
          if (k < R.cap) raw_row[k] = pj;
        }
        if (r <= P.rc) {                                             // "<=" as printed, PAPER.md:80 (R9)
          const int t = r_type[rp];
          atomicAdd(&cnt[t], 1);
          const int h = atomicAdd(&n_hit, 1);
          if (h < cap) {
            const int b = min(NL_BUCKETS - 1, (int)(r * r * r * binv));     // monotone in r: consistent with the order
            hit[h].r = r; hit[h].j = C.s_idx[pj]; hit[h].t = t * NL_BUCKETS + b; hp[h] = pj;
            atomicAdd(&bcnt[t * NL_BUCKETS + b], 1);
          }
        }
      }
    }
  } else {
    const int ncand = min(R.nraw[p], R.cap);
    const int *raw_row = R.raw + (size_t)p * R.cap;
    for (int c = tid; c < ncand; c += nthr) {
      const int pj = raw_row[c];
      const double xj[3] = {s_xyz[3 * (size_t)pj], s_xyz[3 * (size_t)pj + 1], s_xyz[3 * (size_t)pj + 2]};
      double d[3], r;
      if (displacement_in_range(xi, xj, G.L, rc2_hi, d, r) && r <= P.rc) {
        int t = 0;
        while (t + 1 < P.ntypes && pj >= C.type_start[t + 1]) ++t;   // sorted positions are grouped by type
        atomicAdd(&cnt[t], 1);
        const int h = atomicAdd(&n_hit, 1);
        if (h < cap) {
          const int b = min(NL_BUCKETS - 1, (int)(r * r * r * binv));
          hit[h].r = r; hit[h].j = C.s_idx[pj]; hit[h].t = t * NL_BUCKETS + b; hp[h] = pj;
          atomicAdd(&bcnt[t * NL_BUCKETS + b], 1);
        }
      }
    }
  }
  __syncthreads();

  int nh = n_hit;
  if (nh > cap) {
    // More in-range candidates than staging slots (DPB_ECAP): cnt[] counted every hit but only `cap` were staged, so
    // the ranks below could not fill the slots that nreal would promise.  The row is written as EMPTY (all -1,
    // nreal = 0): the passes that are enqueued behind this kernel never touch an unwritten slot; the evaluation is
    // reported as failed through err_cap.
    if (tid == 0) atomicExch(&stats->err_cap, 1);
    if (tid < DPB_MAX_TYPES) cnt[tid] = 0;
    nh = 0;
  }
  if (MODE == 1 && tid == 0) {
    R.nraw[p] = n_raw;
    if (n_raw > R.cap) atomicExch(&stats->err_cap, 1);
  }
  int *nl_row = C.nl + (size_t)q * P.nm;
  int *nlp_row = C.nlp ? const_cast<int *>(C.nlp) + (size_t)q * P.nm : nullptr;
  double4 *dr_row = C.dr + (size_t)q * P.nm;
  int *out_row = nlist_out ? nlist_out + (size_t)i * P.nm : nullptr;

  // Alg. 1 line 7: order by (type, distance, index).  Hits are grouped by (type, bucket of r^3) with a
  // counting sort; the rank of a hit inside its type = hits in earlier buckets + hits of its own bucket that precede
  // it under the exact key (r as fp64, then j).  The first sel[t] go to section t (line 8-9, :186-193), the others are
  // dropped (reading R8).
  const int nb = P.ntypes * NL_BUCKETS;
  if (tid < 32) {                                             // exclusive scan of the bucket counts (<= 256 entries)
    const int per = (nb + 31) / 32, lo = tid * per;
    int sum = 0;
    for (int k = lo; k < min(nb, lo + per); ++k) sum += bcnt[k];
    int incl = sum;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const int v = __shfl_up_sync(0xffffffffu, incl, off);
      if (lane >= off) incl += v;
    }
    int run = incl - sum;
    for (int k = lo; k < min(nb, lo + per); ++k) { bstart[k] = run; run += bcnt[k]; bcnt[k] = 0; }
    if (tid == 31) bstart[nb] = incl;
  }
  __syncthreads();
  for (int h = tid; h < nh; h += nthr) {
    const int bk = hit[h].t;
    order[bstart[bk] + atomicAdd(&bcnt[bk], 1)] = h;
  }
  __syncthreads();
  for (int pos = tid; pos < nh; pos += nthr) {
    const int h = order[pos];
    const NlHit me = hit[h];
    const int t = me.t / NL_BUCKETS, lo = bstart[me.t], hi = bstart[me.t + 1];
    int less = 0;
    for (int g = lo; g < hi; ++g) {
      const NlHit u = hit[order[g]];
      less += (u.r < me.r) | ((u.r == me.r) & (u.j < me.j));
    }
    const int rank = lo - bstart[t * NL_BUCKETS] + less;
    if (rank < P.sel[t]) {
      const int slot = P.sec_start[t] + rank;
      nl_row[slot] = me.j;
      if (out_row) out_row[slot] = me.j;
      const int pj = hp[h];
      if (nlp_row) nlp_row[slot] = pj;
      const double xj[3] = {s_xyz[3 * (size_t)pj], s_xyz[3 * (size_t)pj + 1], s_xyz[3 * (size_t)pj + 2]};
      double d[3], rr;
      dp_displacement(xi, xj, G.L, d, rr);
      dr_row[slot] = make_double4(d[0], d[1], d[2], rr);
    }
  }
  // padding: -1 at the tail of each section
  for (int slot = tid; slot < P.nm; slot += nthr) {
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
                         const int *start, int cap, int *nlist_out, DevStats *stats, cudaStream_t st, int mode,
                         const NlRaw *raw, const ZeroJobs *zero) {
  if (C.n <= 0) return cudaSuccess;
  ZeroJobs Z{};
  if (zero && mode == 0) Z = *zero;
  const size_t smem = (size_t)cap * (sizeof(NlHit) + 2 * sizeof(int)) + sizeof(int) * (3 * 18 * (size_t)P.ntypes * G.ngrp + 1);
  static size_t configured_d[DPB_MAX_DEVICES] = {};
  size_t &configured = configured_d[dpb_device()];
  if (smem > 48 * 1024 && smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(k_nlist<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_nlist<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_nlist<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_nlist<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  NlRaw R{};
  if (raw) R = *raw;
  // one block per atom: 64 threads when the lists are short (water: ~660 candidates for ~90 hits; 192 -> 182 us on W24k),
  // 128 otherwise (copper, ~1,200 candidates: 64 threads take 586 instead of 416 us on Cu32k)
  const int nthr = P.nm <= 192 ? 64 : NL_THREADS;
  if (mode == 1) k_nlist<1><<<C.n, nthr, smem, st>>>(P, G, C, s_xyz, start, cap, nlist_out, stats, R, Z);
  else if (mode == 2) k_nlist<2><<<C.n, nthr, smem, st>>>(P, G, C, s_xyz, start, cap, nlist_out, stats, R, Z);
  else if (zero) {
    cudaError_t el = dpb_launch_pdl(k_nlist<0, true>, dim3(C.n), dim3(nthr), smem, st, true, P, G, C, s_xyz, start, cap,
                                    nlist_out, stats, R, Z);
    if (el != cudaSuccess) return el;
  }
  else k_nlist<0><<<C.n, nthr, smem, st>>>(P, G, C, s_xyz, start, cap, nlist_out, stats, R, Z);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

// MD reuse step: refresh the cell-sorted coordinate copy from the current coordinates (the sorted order of the last
// rebuild stays) and track the largest displacement since that rebuild (skin criterion: must stay below skin / 2).
__global__ void k_gather_sorted(int n, const double *__restrict__ coord, const int *__restrict__ s_idx,
                                double *__restrict__ s_xyz, const double *__restrict__ xyz0, DevStats *stats) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  double d2 = 0.0;
  if (p < n) {
    const int i = s_idx[p];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double x = coord[3 * (size_t)i + c];
      s_xyz[3 * (size_t)p + c] = x;
      const double d = x - xyz0[3 * (size_t)p + c];
      d2 += d * d;
    }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) d2 = fmax(d2, __shfl_xor_sync(0xffffffffu, d2, off));
  if ((threadIdx.x & 31) == 0 && d2 > 0.0)
    atomicMax(reinterpret_cast<unsigned long long *>(&stats->max_disp2), (unsigned long long)__double_as_longlong(d2));
}

cudaError_t launch_gather_sorted(int64_t natoms, const double *coord, const int *s_idx, double *s_xyz,
                                 const double *xyz0, DevStats *stats, cudaStream_t st) {
  const int n = (int)natoms;
  if (n <= 0) return cudaSuccess;
  k_gather_sorted<<<(n + 255) / 256, 256, 0, st>>>(n, coord, s_idx, s_xyz, xyz0, stats);
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
    if (dbgdT) dbgdT[(size_t)i * n + k] = C.dT[dt_offset(P, C, q, k >> 2) + (k & 3)];
  }
}

cudaError_t launch_scatter_debug(const DevModel &P, const ChunkView &C, double *dbgT, double *dbgdT, cudaStream_t st) {
  if (C.n <= 0 || (!dbgT && !dbgdT)) return cudaSuccess;
  k_scatter_debug<<<C.n, 128, 0, st>>>(P, C, dbgT, dbgdT);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}
