// det.cu — deterministic reduction of forces and virial (SURVEY.md §7 hard part 6).  In this mode pass 2 stores
// f_ik = dE_i/dd_ik per slot instead of scattering it with fp64 atomics; here every atom gathers
//   F_i = sum_k f_ik - sum_{j : i in L(j)} f_{j, slot of i in L(j)}          (O11: F_i += f_ik, F_j -= f_ik)
// using the symmetry j in L(i) <=> i in L(j) (valid when no neighbour was dropped by a full type section), and
// Xi = -sum_i sum_k d_ik (x) f_ik, both in a fixed summation order: lane k-stride, then a fixed shuffle tree, then a
// fixed-order sum over atoms.  The result is bitwise reproducible from run to run.
//
// Sub-region mode (dpb_eval_local): only the nloc local atoms are centres, so only they have f_ik
// rows.  api.cu also builds the formatted list of every GHOST (list only, no network): by the same symmetry it names the
// local atoms j whose lists contain the ghost, and F_ghost = - sum_{j local, ghost in L(j)} f_{j, slot of ghost}.  A local
// atom skips the reverse term of its ghost neighbours (a ghost is no centre).  The virial parts are the local atoms'.
#include "common.cuh"

#define DET_WARPS 8

__global__ void __launch_bounds__(32 * DET_WARPS)
k_force_gather(DevModel P, DevGrid G, int n, int nloc, const int *__restrict__ s_idx, const int *__restrict__ pos_of,
               const int *__restrict__ type_start, const double *__restrict__ s_xyz, const int *__restrict__ nl_all,
               const int *__restrict__ nreal_all, const double *__restrict__ fslot, double *__restrict__ force,
               double *__restrict__ vpart) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int p = blockIdx.x * DET_WARPS + warp;
  if (p >= n) return;
  const int i = s_idx[p];
  const bool centre = p < nloc;           // sorted positions [0, nloc) are the local atoms (all of them in a periodic box)
  int a = 0;                              // (group, type) section of p in the sorted order; the species is a mod ntypes
  while (a + 1 < P.ntypes * G.ngrp && p >= type_start[a + 1]) ++a;
  if (a >= P.ntypes) a -= P.ntypes;
  const double xi[3] = {s_xyz[3 * (size_t)p], s_xyz[3 * (size_t)p + 1], s_xyz[3 * (size_t)p + 2]};
  double acc[3] = {0.0, 0.0, 0.0}, vir[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) vir[k] = 0.0;
  for (int t = 0; t < P.ntypes; ++t) {
    const int nr = nreal_all[(size_t)p * P.ntypes + t];
    for (int k = lane; k < nr; k += 32) {
      const size_t slot = (size_t)p * P.nm + P.sec_start[t] + k;
      const int j = nl_all[slot];
      const int pj = pos_of[j];
      double f[3] = {0.0, 0.0, 0.0};     // a ghost (p >= nloc) is no centre: no rows of its own
      if (centre) { f[0] = fslot[3 * slot]; f[1] = fslot[3 * slot + 1]; f[2] = fslot[3 * slot + 2]; }
      // slot of i in j's list: section of type a
      const int nrj = pj < nloc ? nreal_all[(size_t)pj * P.ntypes + a] : 0;      // ... and neither is a ghost j
      const size_t basej = (size_t)pj * P.nm + P.sec_start[a];
      double g[3] = {0.0, 0.0, 0.0};
      for (int kk = 0; kk < nrj; ++kk)
        if (nl_all[basej + kk] == i) {
          g[0] = fslot[3 * (basej + kk)]; g[1] = fslot[3 * (basej + kk) + 1]; g[2] = fslot[3 * (basej + kk) + 2];
          break;
        }
      const double xj[3] = {s_xyz[3 * (size_t)pj], s_xyz[3 * (size_t)pj + 1], s_xyz[3 * (size_t)pj + 2]};
      double d[3], r;
      dp_displacement(xi, xj, G.L, d, r);
#pragma unroll
      for (int c = 0; c < 3; ++c) acc[c] += f[c] - g[c];
#pragma unroll
      for (int x = 0; x < 3; ++x)
#pragma unroll
        for (int y = 0; y < 3; ++y) vir[3 * x + y] -= d[x] * f[y];
    }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
    for (int c = 0; c < 3; ++c) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], off);
#pragma unroll
    for (int k = 0; k < 9; ++k) vir[k] += __shfl_xor_sync(0xffffffffu, vir[k], off);
  }
  if (lane == 0) {
    if (force) { force[3 * (size_t)i] = acc[0]; force[3 * (size_t)i + 1] = acc[1]; force[3 * (size_t)i + 2] = acc[2]; }
#pragma unroll
    if (centre)                                                       // local atoms are the first nloc ORIGINAL indices
      for (int k = 0; k < 9; ++k) vpart[9 * (size_t)i + k] = vir[k];  // by original index: the cell-sort order varies
  }
}

// Xi[k] = sum_p vpart[p][k] in a fixed order: one block, strided partial sums then a tree.
__global__ void k_reduce_virial(int n, const double *__restrict__ vpart, double *__restrict__ virial) {
  __shared__ double part[1024];
  for (int k = 0; k < 9; ++k) {
    double s = 0.0;
    for (int p = threadIdx.x; p < n; p += 1024) s += vpart[9 * (size_t)p + k];
    part[threadIdx.x] = s;
    __syncthreads();
    for (int off = 512; off > 0; off >>= 1) {
      if ((int)threadIdx.x < off) part[threadIdx.x] += part[threadIdx.x + off];
      __syncthreads();
    }
    if (threadIdx.x == 0) virial[k] = part[0];
    __syncthreads();
  }
}

// Overflow and staging-cap flags of the ghost rows (second DevStats) count like the local rows' in dpb_eval_info: a
// dropped neighbour anywhere breaks the symmetry the gather relies on.
__global__ void k_merge_ghost_stats(DevStats *stats) {
  if (stats[1].n_overflow) atomicAdd(&stats[0].n_overflow, stats[1].n_overflow);
  if (stats[1].err_cap) stats[0].err_cap = 1;
}

cudaError_t launch_merge_ghost_stats(DevStats *stats, cudaStream_t st) {
  k_merge_ghost_stats<<<1, 1, 0, st>>>(stats);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

cudaError_t launch_force_gather(const DevModel &P, const DevGrid &G, int64_t natoms, int64_t nloc, const int *s_idx, const int *pos_of,
                                const int *type_start, const double *s_xyz, const int *nl_all, const int *nreal_all,
                                const double *fslot, double *force, double *vpart, double *virial, cudaStream_t st) {
  const int n = (int)natoms;
  if (n <= 0) return cudaSuccess;
  k_force_gather<<<(n + DET_WARPS - 1) / DET_WARPS, 32 * DET_WARPS, 0, st>>>(P, G, n, (int)nloc, s_idx, pos_of, type_start,
                                                                           s_xyz, nl_all, nreal_all, fslot, force, vpart);
  DPB_LAUNCHED(1);
  if (virial) {
    k_reduce_virial<<<1, 1024, 0, st>>>((int)nloc, vpart, virial);
    DPB_LAUNCHED(1);
  }
  return cudaGetLastError();
}
