// dd.cu — pack / unpack kernels of the domain decomposition's ghost exchange (
// PAPER.md:145-149).  A stage of the forward exchange sends, along one dimension, the atoms within r_c of the brick's
// upper face to the + neighbour and those within r_c of the lower face to the - neighbour; at the box boundary the
// sender applies the periodic shift.  The reverse exchange adds the returned ghost force increments at the sender's
// indices.  Messages are rows of four doubles (x, y, z, type) so that one transfer carries an atom.
#include "common.cuh"

// One pass over the atoms: warp-aggregated slot allocation per direction (order inside a message is arbitrary; the
// index list written next to it is what the reverse exchange uses).  Rows beyond `cap` are counted but not written.
__global__ void k_dd_pack(int n, const double *__restrict__ coord, const int *__restrict__ type, int dim,
                          double cut_minus, double cut_plus, double shift_minus, double shift_plus, int cap,
                          double *__restrict__ pack_minus, int *__restrict__ idx_minus,
                          double *__restrict__ pack_plus, int *__restrict__ idx_plus, int *__restrict__ counts) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  double x[3] = {0.0, 0.0, 0.0};
  int t = 0;
  bool to_minus = false, to_plus = false;
  if (i < n) {
    x[0] = coord[3 * (size_t)i]; x[1] = coord[3 * (size_t)i + 1]; x[2] = coord[3 * (size_t)i + 2];
    t = type[i];
    to_minus = x[dim] < cut_minus;
    to_plus = x[dim] >= cut_plus;
  }
#pragma unroll
  for (int dir = 0; dir < 2; ++dir) {
    const bool mine = dir ? to_plus : to_minus;
    const unsigned m = __ballot_sync(0xffffffffu, mine);
    if (m == 0) continue;
    int base = 0;
    if (lane == __ffs(m) - 1) base = atomicAdd(&counts[dir], __popc(m));
    base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
    if (mine) {
      const int slot = base + __popc(m & ((1u << lane) - 1u));
      if (slot < cap) {
        double *row = (dir ? pack_plus : pack_minus) + 4 * (size_t)slot;
        double y[3] = {x[0], x[1], x[2]};
        y[dim] += dir ? shift_plus : shift_minus;
        reinterpret_cast<double2 *>(row)[0] = make_double2(y[0], y[1]);
        reinterpret_cast<double2 *>(row)[1] = make_double2(y[2], (double)t);
        (dir ? idx_plus : idx_minus)[slot] = i;
      }
    }
  }
}

// Received rows -> the tail of the atom arrays.
__global__ void k_dd_unpack(int k, const double *__restrict__ pack, double *__restrict__ coord_out,
                            int *__restrict__ type_out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= k) return;
  const double2 a = reinterpret_cast<const double2 *>(pack)[2 * (size_t)i];
  const double2 b = reinterpret_cast<const double2 *>(pack)[2 * (size_t)i + 1];
  coord_out[3 * (size_t)i] = a.x; coord_out[3 * (size_t)i + 1] = a.y; coord_out[3 * (size_t)i + 2] = b.x;
  type_out[i] = (int)b.y;
}

// Reverse exchange: force[idx[i]] += fin[i].  An index occurs at most once per message, and the two messages of a
// stage are applied by two launches on one stream, so plain read-modify-write is enough.
__global__ void k_dd_add_forces(int k, const int *__restrict__ idx, const double *__restrict__ fin,
                                double *__restrict__ force) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= 3 * k) return;
  const int i = e / 3, c = e - 3 * i;
  force[3 * (size_t)idx[i] + c] += fin[e];
}

cudaError_t launch_dd_pack(int64_t n, const double *coord, const int *type, int dim, double cut_minus, double cut_plus,
                           double shift_minus, double shift_plus, int64_t cap, double *pack_minus, int *idx_minus,
                           double *pack_plus, int *idx_plus, int *counts, cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(counts, 0, 2 * sizeof(int), st);
  if (e != cudaSuccess || n <= 0) return e;
  k_dd_pack<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((int)n, coord, type, dim, cut_minus, cut_plus, shift_minus,
                                                          shift_plus, (int)cap, pack_minus, idx_minus, pack_plus, idx_plus,
                                                          counts);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

cudaError_t launch_dd_unpack(int64_t k, const double *pack, double *coord_out, int *type_out, cudaStream_t st) {
  if (k <= 0) return cudaSuccess;
  k_dd_unpack<<<(unsigned)((k + 255) / 256), 256, 0, st>>>((int)k, pack, coord_out, type_out);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}

cudaError_t launch_dd_add_forces(int64_t k, const int *idx, const double *fin, double *force, cudaStream_t st) {
  if (k <= 0) return cudaSuccess;
  k_dd_add_forces<<<(unsigned)((3 * k + 255) / 256), 256, 0, st>>>((int)k, idx, fin, force);
  DPB_LAUNCHED(1);
  return cudaGetLastError();
}
