// cell.cu — general periodic cells through explicit images (the paper's own
// formulation of periodicity — the atoms of the cell are the local atoms, their lattice images within r_c of the cell are
// ghosts, the ghost force increments are added to the atoms they are images of).  dpb_eval_cell (api.cu) runs
//   k_cell_wrap    fractional coordinates s = x A^-1 wrapped into [0, 1), local atoms x' = s A
//   k_cell_images  every lattice image t = s + shift with -m_c <= t_c <= 1 + m_c (m_c = r_c / h_c, h_c the perpendicular
//                  height of the cell) is appended as a ghost (position, type, owner)
//   dpb_eval_local arithmetic on local + ghost atoms (unchanged kernels)
//   k_cell_fold    F_owner += F_ghost (fp64 reductions: an atom has several images)
#include "common.cuh"

__global__ void k_cell_wrap(int n, const double *__restrict__ coord, const int *__restrict__ type, CellGeom G,
                            double *__restrict__ frac, double *__restrict__ xall, int *__restrict__ tall,
                            int *__restrict__ owner) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double x[3] = {coord[3 * (size_t)i], coord[3 * (size_t)i + 1], coord[3 * (size_t)i + 2]};
  double s[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double v = x[0] * G.Ainv[c] + x[1] * G.Ainv[3 + c] + x[2] * G.Ainv[6 + c];
    v -= floor(v);
    if (v >= 1.0) v = 0.0;                                 // -tiny - floor(-tiny) rounds to 1
    s[c] = v;
    frac[3 * (size_t)i + c] = v;
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) xall[3 * (size_t)i + c] = s[0] * G.A[c] + s[1] * G.A[3 + c] + s[2] * G.A[6 + c];
  tall[i] = type[i];
  owner[i] = i;
}

// one thread per (atom, shift); warp-aggregated slot allocation behind the n local atoms; rows beyond cap are counted only
__global__ void k_cell_images(int n, long long nshift, const double *__restrict__ frac, const int *__restrict__ type,
                              CellGeom G, long long cap, double *__restrict__ xall, int *__restrict__ tall,
                              int *__restrict__ owner, unsigned long long *__restrict__ count) {
  const long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  bool keep = false;
  double t[3] = {0.0, 0.0, 0.0};
  int i = 0;
  if (w < (long long)n * nshift) {
    i = (int)(w / nshift);
    long long k = w - (long long)i * nshift;
    const int d2 = 2 * G.nshell[2] + 1, d1 = 2 * G.nshell[1] + 1;
    const int sh[3] = {(int)(k / ((long long)d1 * d2)) - G.nshell[0], (int)((k / d2) % d1) - G.nshell[1],
                       (int)(k % d2) - G.nshell[2]};
    if (sh[0] != 0 || sh[1] != 0 || sh[2] != 0) {
      keep = true;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        t[c] = frac[3 * (size_t)i + c] + (double)sh[c];
        keep = keep && t[c] >= -G.margin[c] && t[c] <= 1.0 + G.margin[c];
      }
    }
  }
  const unsigned m = __ballot_sync(0xffffffffu, keep);
  if (m == 0) return;
  unsigned long long base = 0;
  if (lane == __ffs(m) - 1) base = atomicAdd(count, (unsigned long long)__popc(m));
  base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
  if (keep) {
    const unsigned long long slot = base + __popc(m & ((1u << lane) - 1u));
    if ((long long)slot < cap) {
      const size_t o = (size_t)n + slot;
#pragma unroll
      for (int c = 0; c < 3; ++c) xall[3 * o + c] = t[0] * G.A[c] + t[1] * G.A[3 + c] + t[2] * G.A[6 + c];
      tall[o] = type[i];
      owner[o] = i;
    }
  }
}

__global__ void k_cell_fold(long long nall, int n, const int *__restrict__ owner, const double *__restrict__ fall,
                            double *__restrict__ force) {
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= 3 * nall) return;
  const long long a = e / 3;
  const int c = (int)(e - 3 * a);
  if (a < n) force[3 * a + c] = fall[e] + 0.0;            // local rows first: plain store (launch 1), images add (launch 2)
}

__global__ void k_cell_fold_images(long long nall, int n, const int *__restrict__ owner, const double *__restrict__ fall,
                                   double *__restrict__ force) {
  const long long e = 3 * (long long)n + (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= 3 * nall) return;
  const long long a = e / 3;
  const int c = (int)(e - 3 * a);
  atomicAdd(&force[3 * (size_t)owner[a] + c], fall[e]);
}

cudaError_t launch_cell_wrap(int64_t n, const double *coord, const int *type, const CellGeom &G, double *frac,
                             double *xall, int *tall, int *owner, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_cell_wrap<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((int)n, coord, type, G, frac, xall, tall, owner);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

cudaError_t launch_cell_images(int64_t n, const double *frac, const int *type, const CellGeom &G, int64_t cap,
                               double *xall, int *tall, int *owner, unsigned long long *count, cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(count, 0, sizeof(unsigned long long), st);
  if (e != cudaSuccess || n <= 0) return e;
  const long long nshift = (long long)(2 * G.nshell[0] + 1) * (2 * G.nshell[1] + 1) * (2 * G.nshell[2] + 1);
  const long long work = (long long)n * nshift;
  k_cell_images<<<(unsigned)((work + 255) / 256), 256, 0, st>>>((int)n, nshift, frac, type, G, (long long)cap, xall, tall,
                                                                owner, count);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

cudaError_t launch_cell_fold(int64_t nall, int64_t n, const int *owner, const double *fall, double *force,
                             cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_cell_fold<<<(unsigned)((3 * n + 255) / 256), 256, 0, st>>>((long long)nall, (int)n, owner, fall, force);
  DPB_LAUNCHED(1);
  if (nall > n) {
    k_cell_fold_images<<<(unsigned)((3 * (nall - n) + 255) / 256), 256, 0, st>>>((long long)nall, (int)n, owner, fall,
                                                                                force);
    DPB_LAUNCHED(1);
  }
  return cudaGetLastError();
}
