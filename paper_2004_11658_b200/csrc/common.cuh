// common.cuh — internal declarations shared by the translation units of libdpb.so (CUDA, sm_100a).
// Not installed; the public interface is include/dpb.h.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/dpb.h"

#define DPB_MAX_TYPES 8

// Model parameters passed to kernels by value.
struct DevModel {
  int ntypes, nm, s1, M, Ma, dim, fw;
  double rc, rcs;
  int sel[DPB_MAX_TYPES];
  int sec_start[DPB_MAX_TYPES + 1];   // slot offset of neighbour-type section t; sec_start[ntypes] = nm
  long long emb_net_size, fit_net_size;
};

// Cell grid of one evaluation (orthorhombic box).
struct DevGrid {
  double L[3];
  int nc[3];
  int ncell;
  int lo_mode[3];   // 1: nc >= 3, use the +-1 stencil; 0: fewer than 3 cells, visit every cell of that dimension once
  // Sub-region mode (dpb_eval_local): no periodic box.  The atoms live in [org, org + ext]; L is that
  // extent padded by more than r_c, so that the minimum image of any pair within r_c is the pair itself and the
  // periodic kernels serve unchanged.  Atoms [0, nloc) are local, the rest ghosts: the sort key puts the ghosts behind
  // all local atoms (ngrp = 2 groups of ntypes pseudo-types), so the sorted positions [0, nloc) are the centres.
  double org[3], ext[3];
  int open;         // 1: sub-region mode
  int ngrp;         // 1 (periodic) or 2 (local, ghost)
  int nloc;
};

// Stats accumulated on the device by the neighbour kernel.
struct DevStats {
  unsigned long long n_real_pairs;
  unsigned long long n_overflow;
  int max_nei[DPB_MAX_TYPES];
  int err_type;      // an atom had a type index outside [0, ntypes)
  int err_cap;       // an atom had more in-range candidates than the staging capacity
  int err_bounds;    // sub-region mode: an atom lies outside the bounds the caller gave
  double max_disp2;  // MD: largest squared displacement of an atom since the last neighbour rebuild (bits ordered as u64)
};

// Raw (skin) neighbour list of the MD driver: sorted positions of the atoms within r_c + skin at the last rebuild.
struct NlRaw {
  int *raw;          // [N][cap]
  int *nraw;         // [N]
  int cap;
  double rs2_hi;     // (r_c + skin)^2 (1 + 1e-9)
};

// Per-chunk views (chunk = sorted positions [p0, p0 + n)).
struct ChunkView {
  int p0, n;
  const int *s_idx;        // [N] original atom index of sorted position p
  const int *type_start;   // [ntypes + 1] first sorted position of each type (device)
  int *nl;                 // [n][nm] neighbour index per slot (chunk-local copy of the nlist rows)
  double4 *dr;             // [n][nm] (dx, dy, dz, r) of real slots
  int *nreal;              // [n][ntypes] real (non-padded) slots per section
  double *T;               // [n][M][4]
  double *dT;              // [n][dt_rows][4]: dE_i/dT_i, row of feature b given by dt_offset() below
  // Layout of dT.  dt_pad == 0: plain, row = b, dt_rows = M.  dt_pad = 4 SP > 0 (fp64 variant 1): every copy of s1
  // features is padded to 4 SP rows, row = (b / s1) * dt_pad + b % s1, dt_rows = 4 dt_pad — the order in which the lanes
  // of the DMMA embedding kernels hold the features (embed_dmma.cu), so that any run of feature slots is one contiguous
  // piece of the tile (bulk-copied as such by pass 2).  Pad rows are zero (the buffer is cleared when it is allocated
  // and no kernel writes them).
  int dt_pad, dt_rows;
  const int *nlp;          // [n][nm] sorted position of the neighbour in each real slot (nl holds its input index)
  double *fslot;           // deterministic mode: [n][nm][3] dE_i/dd_ik per slot (pass 2 stores instead of scattering)  // same-species pair reuse in pass 1 (fp64 variant 1): g(s(r_ij)) = g(s(r_ji)) for a net (a, a), so
  // the atom with the lower sorted position evaluates the pair once and adds g (x) R~_ji to T_j with red.global.add.f64
  const int *pos_of;       // [N] sorted position of original atom index (nullptr: no reuse)
  const DevStats *stats;   // reuse is taken only while stats->n_overflow == 0 (a dropped neighbour breaks the symmetry)
  int sub_part, sub_nparts; // the fitting kernels of one launch cover part sub_part of sub_nparts of a species' rows (default 0 of 1)
  int *counters;           // [128] work-item counters of the embedding launches (pass 1: net, pass 2: 64 + net), zeroed per chunk
  int reuse;               // pass 1
  int reuse2;              // pass 2 (k_pass2_dmma_ru): both directions of a same-species pair from one evaluation
  // Stored activations (fp64 variant 1, embed_dmma.cu): pass 1 writes the tanh outputs of the three
  // embedding layers of every row it evaluates, pass 2 reads them instead of recomputing the value chain.  Record of
  // slot (row, section slot) at act + ((size_t)row * nm + slot) * act_stride; nullptr: pass 2 recomputes.
  double *act;
  int act_stride;          // doubles per record: 4 * (even(SP) + 6 SP)
  int prezero;             // T and the split-K pre-activations were cleared by the list kernel (ZeroJobs): no memsets
  // Species pipeline (ntypes > 1, large chunks): pass 1, the fitting chain and pass 2 of centre type a touch only rows of
  // type a (T_a, the fitting buffers of a, dT_a — with the pair reuse T_j and dT_j are of type a too), so they run back to
  // back on the stream of type a without the barriers between the stages; the streams join after pass 2.
  int typed_pipe;
};

// Small single-chunk evaluations are a chain of dependent graph nodes, and every memset is one of them (stats, counters,
// force, virial, T, the split-K pre-activations: 15 us of a 230 us evaluation of 192 atoms).  The cell-sort and list kernels
// clear these on the side instead.  Null pointers: nothing to do.
struct ZeroJobs {
  void *stats; int stats_bytes;        // k_sort_small, before the keys (multiple of 4 bytes)
  int *counters; int ncounters;        // k_sort_small
  double *T; int t_len;                // k_nlist<0>: block q clears T[q][0 .. t_len)
  double *Z0; int z_len;               // k_nlist<0>: block q clears Z0[q][0 .. z_len)
  double *force;                       // k_nlist<0>: block q clears force[q][0..3) (one block per atom of the evaluation)
  double *virial;                      // k_nlist<0>: block 0 clears virial[0..9)
};

// The per-type fitting chains are independent (disjoint rows) and one type's GEMM launch fills only as many SMs as that
// type has row tiles; they run on forked streams so that the types share the GPU.  fork: s[0] = st, s[ty > 0] = auxiliary
// streams that wait for everything enqueued on st so far; join: st waits for everything enqueued on them.
cudaError_t dpb_fork_streams(int ntypes, cudaStream_t st, cudaStream_t s[DPB_MAX_TYPES]);
cudaError_t dpb_join_streams(int ntypes, cudaStream_t st, cudaStream_t s[DPB_MAX_TYPES]);
// the streams of an earlier fork that has not been joined yet (no event is recorded, nothing waits)
cudaError_t dpb_forked_streams(int ntypes, cudaStream_t st, cudaStream_t s[DPB_MAX_TYPES]);

// dd.cu: pack / unpack kernels of the domain decomposition's ghost exchange
cudaError_t launch_dd_pack(int64_t n, const double *coord, const int *type, int dim, double cut_minus, double cut_plus,
                           double shift_minus, double shift_plus, int64_t cap, double *pack_minus, int *idx_minus,
                           double *pack_plus, int *idx_plus, int *counts, cudaStream_t st);
cudaError_t launch_dd_unpack(int64_t k, const double *pack, double *coord_out, int *type_out, cudaStream_t st);
cudaError_t launch_dd_add_forces(int64_t k, const int *idx, const double *fin, double *force, cudaStream_t st);

// cell.cu: explicit lattice images of a general periodic cell (dpb_eval_cell)
struct CellGeom {
  double A[9], Ainv[9];      // rows of A = lattice vectors; x = s A, s = x Ainv
  double margin[3];          // r_c / h_c, h_c = perpendicular height of the cell along lattice direction c
  int nshell[3];             // ceil(r_c / h_c) image shells
};
cudaError_t launch_cell_wrap(int64_t n, const double *coord, const CellGeom &G, double *frac, cudaStream_t st);
// fill = 0: off[i] = first image row of atom i (relative to row n), off[n] = number of images; fill = 1: write the rows
// (the wrapped atoms in rows [0, n), their images behind them)
cudaError_t launch_cell_images(int64_t n, const double *frac, const int *type, const CellGeom &G, int *off, double *xall,
                               int *tall, int fill, cudaStream_t st);
cudaError_t launch_cell_fold(int64_t n, const int *off, const double *fall, double *force, cudaStream_t st);

// Per-device launch configuration: cudaFuncSetAttribute and the SM count belong to a device, so the "already done" flags
// of the launchers are kept per device (a process that drives several GPUs creates models on each of them).
#define DPB_MAX_DEVICES 32
static inline int dpb_device() {
  int d = 0;
  if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= DPB_MAX_DEVICES) d = 0;
  return d;
}

// Programmatic dependent launch (small evaluations: a chain of dependent launches on one stream).  A kernel launched
// with dpb_launch_pdl may be scheduled while its predecessor on the stream still runs; it must call pdl_wait() before it
// touches anything the predecessor writes (or writes anything the predecessor reads).  pdl_wait() is a no-op in a kernel
// launched the ordinary way.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// ... and the predecessor says when its successor may be scheduled (it still waits in pdl_wait for the whole grid to end)
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <class... KArgs, class... Args>
static inline cudaError_t dpb_launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                         bool pdl, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// Process-wide count of kernels launched by this library (reported by dpb_kernel_launches()).
extern unsigned long long g_dpb_launches;
#define DPB_LAUNCHED(n) (g_dpb_launches += (unsigned long long)(n))

// ---- launchers implemented in the .cu files (all asynchronous on `st`; return cudaGetLastError()) ----------
cudaError_t launch_cell_sort(const DevModel &P, const DevGrid &G, int64_t natoms, const double *coord, const int *type,
                             int *key, int *count, int *start, int *cursor, int *s_idx, double *s_xyz,
                             DevStats *stats, cudaStream_t st, int *pos_of = nullptr, const ZeroJobs *zero = nullptr);
// deterministic force / virial reduction (det.cu)
cudaError_t launch_merge_ghost_stats(DevStats *stats, cudaStream_t st);
cudaError_t launch_force_gather(const DevModel &P, const DevGrid &G, int64_t natoms, int64_t nloc, const int *s_idx, const int *pos_of,
                                const int *type_start, const double *s_xyz, const int *nl_all, const int *nreal_all,
                                const double *fslot, double *force, double *vpart, double *virial, cudaStream_t st);
cudaError_t launch_nlist(const DevModel &P, const DevGrid &G, const ChunkView &C, const double *s_xyz,
                         const int *start, int cap, int *nlist_out, DevStats *stats, cudaStream_t st, int mode = 0,
                         const NlRaw *raw = nullptr, const ZeroJobs *zero = nullptr);
cudaError_t launch_gather_sorted(int64_t natoms, const double *coord, const int *s_idx, double *s_xyz,
                                 const double *xyz0, DevStats *stats, cudaStream_t st);

// variant 0 ("v0"): plain unfused kernels
struct V0Scratch {
  double *D, *dD;                       // [n][dim]
  double *Z0, *U1, *Z1, *U2, *Z2;       // [n][fw]
  double *G, *dZ;                       // [n][fw]
};
cudaError_t launch_pass1_v0(const DevModel &P, const ChunkView &C, const double *emb, cudaStream_t st);
cudaError_t launch_fit_v0(const DevModel &P, const ChunkView &C, const double *fit, const V0Scratch &S,
                          double *atom_energy, double *dbgD, cudaStream_t st);
cudaError_t launch_pass2_v0(const DevModel &P, const ChunkView &C, const double *emb, double *force, double *virial,
                            cudaStream_t st);

cudaError_t launch_scatter_debug(const DevModel &P, const ChunkView &C, double *dbgT, double *dbgdT, cudaStream_t st);
cudaError_t launch_reduce_energy(int64_t natoms, const double *atom_energy, double *energy, cudaStream_t st);

// molecular-dynamics driver (md.cu)
cudaError_t launch_md_kick_drift(int64_t n, double *coord, double *vel, const double *force, const int *type,
                                 const double *hm, double dt, cudaStream_t st);
cudaError_t launch_md_kick(int64_t n, double *vel, const double *force, const int *type, const double *hm,
                           cudaStream_t st);
cudaError_t launch_md_ekin(int64_t n, const double *vel, const int *type, const double *mass_ev, double *ekin,
                           cudaStream_t st);
cudaError_t launch_md_thermo(int64_t n, const double *vel, const int *type, const double *mass_ev, const double *epot,
                             const double *virial, double volume, double *thermo, int slot, cudaStream_t st);

// ---- device helpers ---------------------------------------------------------------------------------------
#ifdef __CUDACC__
// Minimum-image displacement d = r_j - r_i and |d| (Alg. 1 line 3-4), one pinned sequence of
// IEEE-754 operations on the raw coordinates (reading R2) so that the neighbour list is reproducible bit for bit:
//   d = x_j - x_i;  k = rint(d / L);  d = fma(-k, L, d);  r2 = fma(dz,dz, fma(dy,dy, dx*dx));  r = sqrt(r2).
__device__ __forceinline__ void dp_displacement(const double xi[3], const double xj[3], const double L[3], double d[3],
                                                double &r) {
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double dc = __dsub_rn(xj[c], xi[c]);
    double k = rint(__ddiv_rn(dc, L[c]));
    d[c] = __fma_rn(-k, L[c], dc);
  }
  double r2 = __fma_rn(d[2], d[2], __fma_rn(d[1], d[1], __dmul_rn(d[0], d[0])));
  r = __dsqrt_rn(r2);
}

// Part `sub_part` of `sub_nparts` of the row range [lo, hi) of a species (cut at multiples of 32 rows from lo).
__device__ __forceinline__ void dpb_sub_range(const ChunkView &C, int &lo, int &hi) {
  if (C.sub_nparts <= 1) return;
  const int n = hi > lo ? hi - lo : 0;
  const int per = ((n + C.sub_nparts - 1) / C.sub_nparts + 31) / 32 * 32;
  const int a = lo + C.sub_part * per, b = a + per;
  lo = a < hi ? a : hi;
  hi = (C.sub_part == C.sub_nparts - 1 || b > hi) ? hi : b;
}

// Offset (in doubles) of dT[q][b][0] in the chunk's dT buffer (layouts: ChunkView::dt_pad).
__device__ __forceinline__ size_t dt_offset(const DevModel &P, const ChunkView &C, int q, int b) {
  const int row = C.dt_pad ? (b / P.s1) * C.dt_pad + (b % P.s1) : b;
  return ((size_t)q * C.dt_rows + row) * 4;
}

// Gate w(r) of Eq. 5, reading R1: quintic between r_cs and r_c.
__device__ __forceinline__ void dp_switch(double r, double rcs, double rc, double &w, double &dw) {
  if (r < rcs) {
    w = 1.0; dw = 0.0;
  } else if (r < rc) {
    double inv = 1.0 / (rc - rcs);
    double u = (r - rcs) * inv;
    w = u * u * u * (-6.0 * u * u + 15.0 * u - 10.0) + 1.0;
    dw = -30.0 * u * u * (u - 1.0) * (u - 1.0) * inv;
  } else {
    w = 0.0; dw = 0.0;
  }
}
#endif
