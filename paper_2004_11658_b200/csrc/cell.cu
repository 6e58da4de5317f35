// cell.cu — general periodic cells through explicit images (the paper's own
// formulation of periodicity — the atoms of the cell are the local atoms, their lattice images within r_c of the cell are
// ghosts, the ghost force increments are added to the atoms they are images of).  dpb_eval_cell (api.cu) runs
//   k_cell_wrap    fractional coordinates s = x A^-1 wrapped into [0, 1)
//   k_cell_count / k_cell_scan / k_cell_fill
//                  local atoms x' = s A; every lattice image t = s + shift with -m_c <= t_c <= 1 + m_c (m_c = r_c / h_c, h_c the perpendicular
//                  height of the cell) is appended as a ghost (position, type), an atom's images in consecutive rows
//   dpb_eval_local arithmetic on local + ghost atoms (unchanged kernels)
//   k_cell_fold    F_i = F of the local row + F of its image rows, in row order
#include "common.cuh"

__global__ void k_cell_wrap(int n, const double *__restrict__ coord, CellGeom G, double *__restrict__ frac) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double x[3] = {coord[3 * (size_t)i], coord[3 * (size_t)i + 1], coord[3 * (size_t)i + 2]};
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double v = x[0] * G.Ainv[c] + x[1] * G.Ainv[3 + c] + x[2] * G.Ainv[6 + c];
    v -= floor(v);
    if (v >= 1.0) v = 0.0;                                 // -tiny - floor(-tiny) rounds to 1
    frac[3 * (size_t)i + c] = v;
  }
}

// Image k of atom i (k indexes the shifts, slowest dimension first): fractional coordinate t = s_i + shift; kept when it
// lies within the margins of the cell and the shift is not zero.
__device__ __forceinline__ bool cell_image(const CellGeom &G, const double *__restrict__ frac_i, long long k, double t[3]) {
  const int d2 = 2 * G.nshell[2] + 1, d1 = 2 * G.nshell[1] + 1;
  const int sh[3] = {(int)(k / ((long long)d1 * d2)) - G.nshell[0], (int)((k / d2) % d1) - G.nshell[1],
                     (int)(k % d2) - G.nshell[2]};
  bool keep = sh[0] != 0 || sh[1] != 0 || sh[2] != 0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    t[c] = frac_i[c] + (double)sh[c];
    keep = keep && t[c] >= -G.margin[c] && t[c] <= 1.0 + G.margin[c];
  }
  return keep;
}

// The images of atom i take the rows [n + off[i], n + off[i + 1]) in shift order: the row of an image does not depend on
// the scheduling, so a list's order of equidistant images (an atom's own +a and -a images) and the fold below are the
// same in every run.  k_cell_count -> k_cell_scan (exclusive, one block) -> k_cell_fill.
__global__ void k_cell_count(int n, long long nshift, const double *__restrict__ frac, CellGeom G, int *__restrict__ off) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double s[3] = {frac[3 * (size_t)i], frac[3 * (size_t)i + 1], frac[3 * (size_t)i + 2]};
  double t[3];
  int c = 0;
  for (long long k = 0; k < nshift; ++k) c += cell_image(G, s, k, t) ? 1 : 0;
  off[i] = c;
}

__global__ void __launch_bounds__(1024) k_cell_scan(int n, int *__restrict__ off) {      // off[n] = number of images
  __shared__ long long part[1024];
  const int per = (n + 1023) / 1024, lo = min(n, (int)threadIdx.x * per), hi = min(n, lo + per);
  long long s = 0;
  for (int i = lo; i < hi; ++i) s += off[i];
  part[threadIdx.x] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    long long run = 0;
    for (int k = 0; k < 1024; ++k) { const long long v = part[k]; part[k] = run; run += v; }
    off[n] = (int)(run > 2000000000ll ? 2000000000ll : run);
  }
  __syncthreads();
  long long run = part[threadIdx.x];
  for (int i = lo; i < hi; ++i) { const int v = off[i]; off[i] = (int)run; run += v; }
}

__global__ void k_cell_fill(int n, long long nshift, const double *__restrict__ frac, const int *__restrict__ type,
                            CellGeom G, const int *__restrict__ off, double *__restrict__ xall, int *__restrict__ tall) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double s[3] = {frac[3 * (size_t)i], frac[3 * (size_t)i + 1], frac[3 * (size_t)i + 2]};
  const int ty = type[i];
#pragma unroll
  for (int c = 0; c < 3; ++c) xall[3 * (size_t)i + c] = s[0] * G.A[c] + s[1] * G.A[3 + c] + s[2] * G.A[6 + c];
  tall[i] = ty;                                            // row i: the atom itself, wrapped into the cell
  size_t o = (size_t)n + off[i];
  double t[3];
  for (long long k = 0; k < nshift; ++k)
    if (cell_image(G, s, k, t)) {
#pragma unroll
      for (int c = 0; c < 3; ++c) xall[3 * o + c] = t[0] * G.A[c] + t[1] * G.A[3 + c] + t[2] * G.A[6 + c];
      tall[o] = ty;
      ++o;
    }
}

// F_i = F of the local row + the image rows of i, added in row order (no reductions: bitwise reproducible)
__global__ void k_cell_fold(int n, const int *__restrict__ off, const double *__restrict__ fall, double *__restrict__ force) {
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= 3 * (long long)n) return;
  const int i = (int)(e / 3), c = (int)(e - 3 * (long long)i);
  double f = fall[e];
  for (int k = off[i]; k < off[i + 1]; ++k) f += fall[3 * ((size_t)n + k) + c];
  force[e] = f;
}

cudaError_t launch_cell_wrap(int64_t n, const double *coord, const CellGeom &G, double *frac, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_cell_wrap<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((int)n, coord, G, frac);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

cudaError_t launch_cell_images(int64_t n, const double *frac, const int *type, const CellGeom &G, int *off, double *xall,
                               int *tall, int fill, cudaStream_t st) {
  if (n <= 0) return fill ? cudaSuccess : cudaMemsetAsync(off, 0, sizeof(int), st);
  const long long nshift = (long long)(2 * G.nshell[0] + 1) * (2 * G.nshell[1] + 1) * (2 * G.nshell[2] + 1);
  const unsigned grid = (unsigned)((n + 127) / 128);
  if (!fill) {                                   // the caller reads off[n] before the rows are written
    k_cell_count<<<grid, 128, 0, st>>>((int)n, nshift, frac, G, off);
    k_cell_scan<<<1, 1024, 0, st>>>((int)n, off);
    DPB_LAUNCHED(2);
  } else {
    k_cell_fill<<<grid, 128, 0, st>>>((int)n, nshift, frac, type, G, off, xall, tall);
    DPB_LAUNCHED(1);
  }
  return cudaGetLastError();
}

cudaError_t launch_cell_fold(int64_t n, const int *off, const double *fall, double *force, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  k_cell_fold<<<(unsigned)((3 * n + 255) / 256), 256, 0, st>>>((int)n, off, fall, force);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}
