// api.cu — the C ABI of libdpb.so (include/dpb.h): model object, grow-only device workspace, host dispatcher.
// One dpb_eval = S1 (cell sort) once, then for each chunk of atoms (sorted by type, then cell):
//   S2 nlist -> S3-S5 pass 1 (T) -> S5-S7 fitting fwd/bwd (E_i, dT) -> S8-S9 pass 2 (F, virial); finally E = sum E_i.
// Everything is enqueued on the caller's stream; no host synchronisation unless the caller asks for `info`.
// The chunk size is automatic (effective_chunk); small evaluations are replayed from a CUDA graph (eval_graphed);
// dpb_eval_cell builds lattice images and dispatches to the sub-region mode of run_eval; variant 2 (strawman.cu) is the
// paper's padded-dense pipeline.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "common.cuh"
#include "v1_kernels.cuh"
#include "tc_kernels.cuh"

static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

unsigned long long g_dpb_launches = 0;

// Auxiliary streams and events are per device (one process per GPU is the design, but a process that drives several
// devices must not wait on another device's stream).
struct ForkState {
  cudaStream_t aux[DPB_MAX_TYPES];
  cudaEvent_t ev_fork, ev_join[DPB_MAX_TYPES];
};
static ForkState g_fork[DPB_MAX_DEVICES] = {};

static cudaError_t fork_state(ForkState **out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= DPB_MAX_DEVICES) return cudaErrorInvalidDevice;
  *out = &g_fork[dev];
  return cudaSuccess;
}

cudaError_t dpb_fork_streams(int ntypes, cudaStream_t st, cudaStream_t s[DPB_MAX_TYPES]) {
  cudaError_t e;
  s[0] = st;
  if (ntypes <= 1) return cudaSuccess;
  ForkState *F;
  if ((e = fork_state(&F)) != cudaSuccess) return e;
  if (!F->ev_fork && (e = cudaEventCreateWithFlags(&F->ev_fork, cudaEventDisableTiming)) != cudaSuccess) return e;
  if ((e = cudaEventRecord(F->ev_fork, st)) != cudaSuccess) return e;
  for (int ty = 1; ty < ntypes; ++ty) {
    if (!F->aux[ty] && (e = cudaStreamCreateWithFlags(&F->aux[ty], cudaStreamNonBlocking)) != cudaSuccess) return e;
    if ((e = cudaStreamWaitEvent(F->aux[ty], F->ev_fork, 0)) != cudaSuccess) return e;
    s[ty] = F->aux[ty];
  }
  return cudaSuccess;
}

cudaError_t dpb_join_streams(int ntypes, cudaStream_t st, cudaStream_t s[DPB_MAX_TYPES]) {
  cudaError_t e;
  if (ntypes <= 1) return cudaSuccess;
  ForkState *F;
  if ((e = fork_state(&F)) != cudaSuccess) return e;
  for (int ty = 1; ty < ntypes; ++ty) {
    if (!F->ev_join[ty] && (e = cudaEventCreateWithFlags(&F->ev_join[ty], cudaEventDisableTiming)) != cudaSuccess) return e;
    if ((e = cudaEventRecord(F->ev_join[ty], s[ty])) != cudaSuccess) return e;
    if ((e = cudaStreamWaitEvent(st, F->ev_join[ty], 0)) != cudaSuccess) return e;
  }
  return cudaSuccess;
}
cudaError_t dpb_forked_streams(int ntypes, cudaStream_t st, cudaStream_t s[DPB_MAX_TYPES]) {
  s[0] = st;
  if (ntypes <= 1) return cudaSuccess;
  ForkState *F;
  cudaError_t e = fork_state(&F);
  if (e != cudaSuccess) return e;
  for (int ty = 1; ty < ntypes; ++ty) {
    if (!F->aux[ty]) return cudaErrorInvalidResourceHandle;
    s[ty] = F->aux[ty];
  }
  return cudaSuccess;
}
extern "C" int64_t dpb_kernel_launches(void) { return (int64_t)g_dpb_launches; }

extern "C" const char *dpb_last_error(void) { return g_err; }
extern "C" const char *dpb_version(void) { return "dpb 1 sm_100a"; }

// Bumped whenever a workspace buffer is (re)allocated or released: captured CUDA graphs hold the old pointers.
static unsigned long long g_ws_epoch = 1;

struct Buf {
  void *p = nullptr;
  size_t cap = 0;
  cudaError_t reserve(size_t bytes, bool zero = false, bool exact = false) {
    if (bytes <= cap) return cudaSuccess;
    ++g_ws_epoch;
    if (p) cudaFree(p);
    p = nullptr; cap = 0;
    size_t want = exact ? bytes : bytes + bytes / 8 + 256;      // exact: the activation records (tens of GB)
    cudaError_t e = cudaMalloc(&p, want);
    if (e == cudaSuccess) cap = want;
    if (e == cudaSuccess && zero) e = cudaMemset(p, 0, want);      // (re)allocation only: synchronous, rare
    return e;
  }
  void release() { if (p) { cudaFree(p); ++g_ws_epoch; } p = nullptr; cap = 0; }
  template <class T> T *as() const { return reinterpret_cast<T *>(p); }
};

// One captured evaluation (dpb_model_set_graph): every argument that is baked into the kernel parameters is part of the key.
struct GraphKey {
  int64_t natoms;
  const void *ptr[7];       // coord, type, energy, atom_energy, force, virial, nlist
  double box[9];
  bool operator==(const GraphKey &o) const { return memcmp(this, &o, sizeof(GraphKey)) == 0; }
};
struct GraphEntry {
  GraphKey key;
  cudaGraphExec_t exec = nullptr;
  unsigned long long epoch = 0, stamp = 0;   // workspace / configuration state the entry belongs to; last use
  long long kernels = 0;                     // kernel launches inside the graph
  bool failed = false;                       // capture did not work for this call: run it eagerly from now on
};
#define DPB_GRAPH_SLOTS 32
#define DPB_GRAPH_AUTO_ATOMS 4096

struct dpb_model {
  DevModel P;
  int graph_mode = 1;                        // 0 off, 1 evaluations of at most DPB_GRAPH_AUTO_ATOMS atoms, 2 always
  unsigned long long cfg_epoch = 1, graph_clock = 0;
  std::vector<GraphEntry> graphs;
  int precision = 0, variant = 1, timing = 0, deterministic = 0, pair_reuse = 1, stored_act = 1;
  int species_pipe = 1;         // dpb_model_set_species_pipeline
  double *atom_virial = nullptr;        // caller's [N][9] buffer (dpb_model_set_atom_virial)
  int64_t chunk = 0;            // atoms per pass; 0 = automatic (effective_chunk)
  size_t ws_budget = 0;         // bytes the per-chunk workspace may take in automatic mode (half of the memory free at creation)
  int device = 0;
  Buf emb, fit;                 // raw weights (layout of dpb_model_desc)
  V1Weights v1;                 // re-laid-out weights of the fused kernels
  TCWeights tcw;                // mixed precision: TF32 hi / lo operand images (embed_tc.cu)
  V2Weights v2;                 // variant 2 (strawman.cu): padded matrices of the paper's pipeline, built on first use
  Buf v2ws;
  // workspace
  Buf key, count, start, cursor, s_idx, s_xyz, stats, ei;
  Buf nl, nlp, dr, nreal, T, dT, counters;
  Buf act;                      // activation records of the chunk (ChunkView::act)
  int dt_pad_alloc = -1;          // layout the dT buffer was last used with (pad rows must be zero: cleared on a change)
  Buf v0[9];
  Buf v1ws;
  Buf tcfit;                    // mixed precision: operand images and activations of the fitting stage
  Buf dT32;                     // mixed precision: fp32 copy of dE/dT of the chunk
  Buf pairs;                    // mixed precision: flattened real-slot lists of the chunk
  Buf h_coord, h_type, h_out;   // device staging of dpb_eval_host
  // molecular dynamics driver (dpb_md_run): skin list of the last rebuild, forces, thermo output
  // deterministic mode: inverse of s_idx, full-size lists, per-slot dE_i/dd_ik, per-atom virial parts
  Buf pos_of, nl_all, nreal_all, fslot, vpart;
  Buf md_raw, md_nraw, md_xyz0, md_force, md_scal, md_mass;
  Buf cell_frac, cell_x, cell_t, cell_off, cell_f;   // dpb_eval_cell: local + image atoms
  int md_cap_raw = 0;
  double md_skin = 0.0;
  DevGrid md_grid;
  double *dbgT = nullptr, *dbgD = nullptr, *dbgdT = nullptr;
  std::vector<cudaEvent_t> evs;   // stage timers: [0] start, [1] after S1, then 4 per chunk, then the end
  int ev_chunks = 0;              // chunks of the last timed evaluation
  int64_t last_natoms = -1;       // atoms of the last evaluation (dpb_debug_sorted_order)
};

static int nm_of(const DevModel &P) { return P.nm; }

// doubles per activation record (ChunkView::act_stride), or 0 when the stored activations cannot apply to this model
static int act_record_doubles(const dpb_model *m) {
  if (!m->stored_act || m->precision != DPB_FP64 || m->variant != 1 || !m->v1.ready || m->deterministic ||
      m->pair_reuse < 1)
    return 0;
  const int sp = m->v1.SP;
  return 4 * (((sp + 1) & ~1) + 6 * sp);
}

// Atoms per chunk.  An explicit dpb_model_set_chunk wins; otherwise the largest chunk whose workspace (lists, (d, r)
// rows, T, dT and the fitting activations: 73 KB per atom for the copper model in fp64) stays inside the budget fixed
// at model creation, at least 32768 atoms.  Larger chunks are faster, not only smaller in launch count: the
// same-species pair reuse only shares pairs whose two atoms are centres of the same chunk.
// ncentre > 0: the number of centres of the evaluation.  When the activation records (stored activations, DESIGN.md
// section 12) of ONE chunk over all centres do not fit the budget but those of a chunk of at least 32768 centres do, the
// evaluation is cut into equal chunks of that size: on the 864,000-atom copper box 10 chunks of 87,040 with the records
// (326 ms) beat one chunk without them (365 ms) although the pairs across a chunk boundary are evaluated twice.
static int64_t effective_chunk(const dpb_model *m, int64_t ncentre = -1) {
  if (m->chunk > 0) return m->chunk;
  if (m->precision != DPB_FP64) return 32768;            // mixed precision: the tile / pair-list kernels are sized for this
  const DevModel &P = m->P;
  size_t per = (size_t)P.nm * (4 + 4 + 32) + (size_t)P.ntypes * 4 + (size_t)P.M * 32 + (size_t)(16 * 8 + P.M) * 32;
  if (m->precision == DPB_FP64) {
    if (m->variant == 0 || !m->v1.ready) per += sizeof(double) * (2 * (size_t)P.dim + 7 * (size_t)P.fw);
    else per += v1_workspace_bytes(P, 1024) / 1024;
    if (m->variant == 2) per += (size_t)P.nm * v2_slot_bytes(m->v2);       // Eq. 13's tensors: every padded slot
  } else {
    per += (tc_pair_workspace_bytes(P, 1024) + tc_pass2_workspace_bytes(P, 1024) + tc_fit_workspace_bytes(P, 1024, m->precision - DPB_TF32)) / 1024;
  }
  int64_t c = (int64_t)(m->ws_budget / (per + 1));
  c -= c % 1024;
  c = c < 32768 ? 32768 : c;
  const int rec = act_record_doubles(m);
  if (rec > 0 && ncentre > 0) {
    int64_t c_sa = (int64_t)(m->ws_budget / (per + (size_t)P.nm * rec * sizeof(double) + 1));
    c_sa -= c_sa % 1024;
    if (ncentre > c_sa && c_sa >= 32768) {
      const int64_t nch = (ncentre + c_sa - 1) / c_sa;
      int64_t bal = (ncentre + nch - 1) / nch;               // equal chunks
      bal = (bal + 1023) / 1024 * 1024;
      c = bal <= c_sa ? bal : c_sa;
    }
  }
  return c;
}

extern "C" int dpb_model_nm(const dpb_model *m) { return m ? nm_of(m->P) : DPB_EINVAL; }

extern "C" int dpb_model_create(const dpb_model_desc *d, int precision, dpb_model **out) {
  if (!d || !out) return fail(DPB_EINVAL, "dpb_model_create: null argument");
  *out = nullptr;
  if (precision < DPB_FP64 || precision > DPB_BF16_PLAIN)
    return fail(DPB_EINVAL, "dpb_model_create: precision must be DPB_FP64, DPB_TF32, DPB_BF16 or DPB_BF16_PLAIN");
  if (d->ntypes < 1 || d->ntypes > DPB_MAX_TYPES) return fail(DPB_EINVAL, "ntypes must be in [1, %d]", DPB_MAX_TYPES);
  if (!d->sel || !d->emb_weights || !d->fit_weights) return fail(DPB_EINVAL, "null sel / weights");
  if (d->emb_s1 < 1 || d->emb_s1 > 64) return fail(DPB_EINVAL, "emb_s1 must be in [1, 64]");
  if (d->m_axis < 1 || d->m_axis > 4 * d->emb_s1) return fail(DPB_EINVAL, "m_axis must be in [1, 4 s1]");
  if (d->fit_width < 1 || d->fit_width > 1024) return fail(DPB_EINVAL, "fit_width must be in [1, 1024]");
  if (!(d->rcut > 0.0) || !(d->rcut_smth >= 0.0) || !(d->rcut_smth < d->rcut))
    return fail(DPB_EINVAL, "need 0 <= rcut_smth < rcut");
  dpb_model *m = new (std::nothrow) dpb_model();
  if (!m) return fail(DPB_ENOMEM, "host allocation failed");
  DevModel &P = m->P;
  memset(&P, 0, sizeof(P));
  P.ntypes = d->ntypes; P.s1 = d->emb_s1; P.M = 4 * d->emb_s1; P.Ma = d->m_axis; P.dim = P.M * P.Ma;
  P.fw = d->fit_width; P.rc = d->rcut; P.rcs = d->rcut_smth;
  int nm = 0;
  for (int t = 0; t < P.ntypes; ++t) {
    if (d->sel[t] < 0) { delete m; return fail(DPB_EINVAL, "sel[%d] < 0", t); }
    P.sel[t] = d->sel[t]; P.sec_start[t] = nm; nm += d->sel[t];
  }
  P.sec_start[P.ntypes] = nm;
  for (int t = P.ntypes + 1; t <= DPB_MAX_TYPES; ++t) P.sec_start[t] = nm;
  P.nm = nm;
  const long long s1 = P.s1;
  P.emb_net_size = s1 + s1 + s1 * 2 * s1 + 2 * s1 + 2 * s1 * 4 * s1 + 4 * s1;
  P.fit_net_size = (long long)P.dim * P.fw + P.fw + 2 * ((long long)P.fw * P.fw + P.fw) + P.fw + 1;
  cudaGetDevice(&m->device);
  {
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) m->ws_budget = free_b / 2;
  }
  const size_t eb = sizeof(double) * (size_t)P.emb_net_size * P.ntypes * P.ntypes;
  const size_t fb = sizeof(double) * (size_t)P.fit_net_size * P.ntypes;
  cudaError_t e = m->emb.reserve(eb);
  if (e == cudaSuccess) e = m->fit.reserve(fb);
  if (e == cudaSuccess) e = m->stats.reserve(2 * sizeof(DevStats));      // [1]: ghost rows of the deterministic local mode
  if (e == cudaSuccess) e = cudaMemcpy(m->emb.p, d->emb_weights, eb, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(m->fit.p, d->fit_weights, fb, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = v1_prepare_weights(P, d->emb_weights, d->fit_weights, m->v1);
  m->precision = precision;
  if (e == cudaSuccess && precision != DPB_FP64) {
    e = tc_prepare_weights(P, d->emb_weights, m->tcw);
    if (e == cudaSuccess) e = tc_prepare_fit(P, d->fit_weights, m->tcw, precision - DPB_TF32);
    if (e == cudaErrorNotSupported) {
      dpb_model_destroy(m);
      return fail(DPB_ENOTIMPL, "mixed precision is built for emb_s1 in {8, 16, 25, 32}, m_axis in {4, 8, 16} and "
                                "fit_width %% 4 == 0, <= 256 (got %d, %d, %d)", d->emb_s1, d->m_axis, d->fit_width);
    }
  }
  if (e != cudaSuccess) {
    int code = (e == cudaErrorMemoryAllocation) ? DPB_ENOMEM : DPB_ECUDA;
    dpb_model_destroy(m);
    return fail(code, "dpb_model_create: %s", cudaGetErrorString(e));
  }
  *out = m;
  return DPB_OK;
}

extern "C" int dpb_model_destroy(dpb_model *m) {
  if (!m) return DPB_OK;
  Buf *all[] = {&m->emb, &m->fit, &m->key, &m->count, &m->start, &m->cursor, &m->s_idx, &m->s_xyz, &m->stats, &m->ei,
                &m->nl, &m->nlp, &m->dr, &m->v2ws, &m->counters, &m->nreal, &m->T, &m->dT, &m->v1ws, &m->pairs, &m->dT32, &m->tcfit, &m->h_coord, &m->h_type, &m->h_out,
                &m->pos_of, &m->nl_all, &m->nreal_all, &m->fslot, &m->vpart,
                &m->md_raw, &m->md_nraw, &m->md_xyz0, &m->md_force, &m->md_scal, &m->md_mass,
                &m->cell_frac, &m->cell_x, &m->cell_t, &m->cell_off, &m->cell_f, &m->act};
  for (Buf *b : all) b->release();
  for (Buf &b : m->v0) b.release();
  v1_release_weights(m->v1);
  v2_release_weights(m->v2);
  tc_release_weights(m->tcw);
  for (cudaEvent_t &e : m->evs) cudaEventDestroy(e);
  for (GraphEntry &g : m->graphs) if (g.exec) cudaGraphExecDestroy(g.exec);
  delete m;
  return DPB_OK;
}

extern "C" int dpb_model_set_chunk(dpb_model *m, int64_t chunk) {
  if (!m || chunk < 0) return fail(DPB_EINVAL, "dpb_model_set_chunk: chunk must be >= 1, or 0 for the automatic size");
  m->chunk = chunk;
  ++m->cfg_epoch;
  return DPB_OK;
}

extern "C" int dpb_model_set_variant(dpb_model *m, int variant) {
  if (!m || variant < 0 || variant > 2) return fail(DPB_EINVAL, "dpb_model_set_variant: variant must be 0, 1 or 2");
  if (variant == 2) {
    if (m->precision != DPB_FP64 || !m->v1.ready)
      return fail(DPB_ENOTIMPL, "variant 2 (the paper's padded-dense pipeline) is built for DPB_FP64 and emb_s1 <= 32");
    if (!m->v2.ready) {                                    // the raw weights live on the device: fetch them once
      const DevModel &P = m->P;
      std::vector<double> h((size_t)P.emb_net_size * P.ntypes * P.ntypes);
      cudaError_t e = cudaMemcpy(h.data(), m->emb.p, sizeof(double) * h.size(), cudaMemcpyDeviceToHost);
      if (e == cudaSuccess) e = v2_prepare_weights(P, h.data(), m->v2);
      if (e != cudaSuccess) return fail(DPB_ECUDA, "variant 2 weights: %s", cudaGetErrorString(e));
    }
  }
  m->variant = variant;
  ++m->cfg_epoch;
  return DPB_OK;
}

extern "C" int dpb_model_set_atom_virial(dpb_model *m, double *atom_virial) {
  if (!m) return fail(DPB_EINVAL, "null model");
  m->atom_virial = atom_virial;
  ++m->cfg_epoch;
  return DPB_OK;
}

extern "C" int dpb_model_set_deterministic(dpb_model *m, int on) {
  if (!m) return fail(DPB_EINVAL, "null model");
  m->deterministic = on ? 1 : 0;
  ++m->cfg_epoch;
  return DPB_OK;
}

extern "C" int dpb_model_set_pair_reuse(dpb_model *m, int on) {
  if (!m) return fail(DPB_EINVAL, "null model");
  if (on < 0 || on > 2) return fail(DPB_EINVAL, "pair reuse: 0 (off), 1 (single-chunk evaluations) or 2 (always)");
  m->pair_reuse = on;
  ++m->cfg_epoch;
  return DPB_OK;
}

extern "C" int dpb_model_set_species_pipeline(dpb_model *m, int on) {
  if (!m) return fail(DPB_EINVAL, "null model");
  if (on < 0 || on > 1) return fail(DPB_EINVAL, "species pipeline: 0 (off) or 1 (on)");
  m->species_pipe = on;
  ++m->cfg_epoch;
  return DPB_OK;
}

extern "C" int dpb_model_set_stored_activations(dpb_model *m, int on) {
  if (!m) return fail(DPB_EINVAL, "null model");
  if (on < 0 || on > 1) return fail(DPB_EINVAL, "stored activations: 0 (off) or 1 (when the records fit)");
  m->stored_act = on;
  if (!on) m->act.release();
  ++m->cfg_epoch;
  return DPB_OK;
}

extern "C" int dpb_set_debug_buffers(dpb_model *m, double *T, double *D, double *dT) {
  if (!m) return fail(DPB_EINVAL, "null model");
  m->dbgT = T; m->dbgD = D; m->dbgdT = dT;
  ++m->cfg_epoch;
  return DPB_OK;
}

extern "C" int dpb_debug_sorted_order(dpb_model *m, void *stream, int64_t natoms, int32_t *order) {
  if (!m || !order) return fail(DPB_EINVAL, "dpb_debug_sorted_order: null argument");
  if (m->last_natoms < 0 || natoms != m->last_natoms)
    return fail(DPB_EINVAL, "dpb_debug_sorted_order: natoms differs from the last evaluation (%lld)", (long long)m->last_natoms);
  if (natoms == 0) return DPB_OK;
  cudaError_t e = cudaMemcpyAsync(order, m->s_idx.p, sizeof(int) * (size_t)natoms, cudaMemcpyDeviceToDevice,
                                  reinterpret_cast<cudaStream_t>(stream));
  if (e != cudaSuccess) return fail(DPB_ECUDA, "dpb_debug_sorted_order: %s", cudaGetErrorString(e));
  return DPB_OK;
}

extern "C" int dpb_model_set_timing(dpb_model *m, int on) {
  if (!m) return fail(DPB_EINVAL, "null model");
  m->timing = on ? 1 : 0;
  ++m->cfg_epoch;
  return DPB_OK;
}

extern "C" int dpb_model_stage_us(const dpb_model *m, float us[8]) {
  if (!m || !us) return fail(DPB_EINVAL, "null argument");
  memset(us, 0, sizeof(float) * 8);
  if (m->ev_chunks <= 0 || m->evs.size() < 3 + 4 * (size_t)m->ev_chunks)
    return fail(DPB_EINVAL, "no timed evaluation yet (dpb_model_set_timing)");
  float ms = 0.f;
  cudaError_t e = cudaEventElapsedTime(&ms, m->evs[0], m->evs[1]);
  if (e != cudaSuccess) return fail(DPB_ECUDA, "stage events not complete: %s", cudaGetErrorString(e));
  us[0] = ms * 1e3f;
  for (int c = 0; c < m->ev_chunks; ++c) {
    const int b = 2 + 4 * c;
    if (cudaEventElapsedTime(&ms, m->evs[b - 1], m->evs[b]) == cudaSuccess) us[1] += ms * 1e3f;
    for (int k = 0; k < 3; ++k)
      if (cudaEventElapsedTime(&ms, m->evs[b + k], m->evs[b + k + 1]) == cudaSuccess) us[2 + k] += ms * 1e3f;
  }
  const int last = 2 + 4 * m->ev_chunks;
  if (cudaEventElapsedTime(&ms, m->evs[last - 1], m->evs[last]) == cudaSuccess) us[5] = ms * 1e3f;
  return DPB_OK;
}

// ---------------------------------------------------------------------------------------------------------
static int make_grid(const DevModel &P, const double box[9], DevGrid &G, double rsearch) {
  if (box[1] != 0.0 || box[2] != 0.0 || box[3] != 0.0 || box[5] != 0.0 || box[6] != 0.0 || box[7] != 0.0)
    return fail(DPB_EBOX, "box must be orthorhombic (off-diagonal entries are not zero)");
  G.L[0] = box[0]; G.L[1] = box[4]; G.L[2] = box[8];
  long long ncell = 1;
  for (int c = 0; c < 3; ++c) {
    if (!(G.L[c] > 0.0) || !(rsearch < 0.5 * G.L[c]))
      return fail(DPB_EBOX, "need rcut (+ skin) < L/2 in every dimension (L[%d] = %g, search radius = %g)", c, G.L[c],
                  rsearch);
    // cell edge >= rc (1 + 1e-6): the +-1 stencil then covers every r <= rc even when rounding moves an atom that
    // sits on a cell face into the neighbouring cell
    double f = floor(G.L[c] / (rsearch * (1.0 + 1e-6)));
    int n = f < 1.0 ? 1 : (f > 512.0 ? 512 : (int)f);
    G.nc[c] = n;
    ncell *= n;
  }
  while (ncell * P.ntypes > (1ll << 22)) {           // bound the histogram: coarser cells are still correct
    int big = 0;
    for (int c = 1; c < 3; ++c) if (G.nc[c] > G.nc[big]) big = c;
    ncell = ncell / G.nc[big];
    G.nc[big] = (G.nc[big] + 1) / 2;
    ncell *= G.nc[big];
  }
  for (int c = 0; c < 3; ++c) G.lo_mode[c] = G.nc[c] >= 3 ? 1 : 0;
  G.ncell = (int)ncell;
  for (int c = 0; c < 3; ++c) { G.org[c] = 0.0; G.ext[c] = G.L[c]; }
  G.open = 0; G.ngrp = 1; G.nloc = 0;
  return DPB_OK;
}

// Sub-region mode: the atoms lie in [lo, hi]; the grid is that of a periodic box of edge max(hi - lo + 1.001 rc,
// 2.002 rc) at origin lo.  Two atoms inside the bounds are less than L - 1.001 rc apart in every coordinate, so every
// periodic image other than the pair itself is farther than r_c: the minimum image is the plain difference wherever
// it matters, and rc < L / 2 holds.
static int make_grid_open(const DevModel &P, const double bounds[6], int64_t nloc, DevGrid &G) {
  double box[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
  for (int c = 0; c < 3; ++c) {
    const double ext = bounds[3 + c] - bounds[c];
    if (!(ext >= 0.0) || !(ext < 1e15)) return fail(DPB_EBOX, "bounds: need lo <= hi, finite (dimension %d)", c);
    const double a = ext + 1.001 * P.rc, b = 2.002 * P.rc;
    box[4 * c] = a > b ? a : b;
  }
  int rc = make_grid(P, box, G, P.rc);
  if (rc != DPB_OK) return rc;
  for (int c = 0; c < 3; ++c) { G.org[c] = bounds[c]; G.ext[c] = bounds[3 + c] - bounds[c]; }
  G.open = 1; G.ngrp = 2; G.nloc = (int)nloc;
  return DPB_OK;
}

static int cuda_fail(cudaError_t e, const char *what) {
  return fail(e == cudaErrorMemoryAllocation ? DPB_ENOMEM : DPB_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

#define CU(call, what) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, what); } while (0)

static int neighbour_cap(const DevModel &P) {
  int cap = 2 * P.nm;
  if (cap < 256) cap = 256;
  if (cap > 9000) cap = 9000;         // 24 B per hit: 211 KB of shared memory at most
  return cap;
}

// nl_mode 0: neighbour search from the cell list (every dpb_eval); 1 / 2: MD rebuild / reuse step (md.cu).
static int run_eval(dpb_model *m, cudaStream_t st, int64_t natoms, const double *coord, const int32_t *type,
                    const double box[9], double *energy, double *atom_energy, double *force, double *virial,
                    int32_t *nlist, bool nlist_only, int nl_mode = 0, int64_t nloc = -1) {
  // nloc >= 0: sub-region mode (dpb_eval_local): `box` holds the bounds (lo[3], hi[3]); atoms [0, nloc) are the centres
  const DevModel &P = m->P;
  if (natoms < 0 || natoms > 2000000000ll) return fail(DPB_EINVAL, "natoms out of range");
  if (natoms > 0 && (!coord || !type)) return fail(DPB_EINVAL, "null coord / type");
  if (nloc > natoms) return fail(DPB_EINVAL, "nloc > nall");
  DevGrid G;
  int rc = DPB_OK;
  if (nloc >= 0) rc = make_grid_open(P, box, nloc, G);
  else if (nl_mode == 2) G = m->md_grid;
  else rc = make_grid(P, box, G, nl_mode == 1 ? P.rc + m->md_skin : P.rc);
  if (rc != DPB_OK) return rc;
  if (nl_mode == 1) m->md_grid = G;
  const int N = (int)natoms;
  const int nkeys = P.ntypes * G.ngrp * G.ncell;
  const int64_t ncentre = nloc >= 0 ? nloc : natoms;
  const int64_t chunk_cap = effective_chunk(m, nlist_only ? -1 : ncentre);
  const int64_t chunk = chunk_cap < ncentre ? chunk_cap : (ncentre > 0 ? ncentre : 1);

  CU(m->key.reserve(sizeof(int) * (size_t)(N + 1)), "workspace");
  CU(m->count.reserve(sizeof(int) * (size_t)(nkeys + 1)), "workspace");
  CU(m->start.reserve(sizeof(int) * (size_t)(nkeys + 1 + P.ntypes * G.ngrp + 1)), "workspace");
  CU(m->cursor.reserve(sizeof(int) * (size_t)(nkeys + 1)), "workspace");
  CU(m->s_idx.reserve(sizeof(int) * (size_t)(N + 1)), "workspace");
  CU(m->s_xyz.reserve(sizeof(double) * 3 * (size_t)(N + 1)), "workspace");
  CU(m->ei.reserve(sizeof(double) * (size_t)(N + 1)), "workspace");
  const bool det = m->deterministic && !nlist_only;
  if (det && (m->precision != DPB_FP64 || m->variant != 1 || !m->v1.ready))
    return fail(DPB_ENOTIMPL, "the deterministic reduction is built for DPB_FP64, variant 1");
  if (m->atom_virial && !nlist_only && !det)
    return fail(DPB_ENOTIMPL, "the per-atom virial comes from the deterministic reduction: switch it on "
                              "(dpb_model_set_deterministic) or clear the buffer");
  CU(m->pos_of.reserve(sizeof(int) * (size_t)(N + 1)), "workspace");
  if (det) {
    CU(m->nl_all.reserve(sizeof(int) * (size_t)(N + 1) * P.nm), "workspace");
    CU(m->nreal_all.reserve(sizeof(int) * (size_t)(N + 1) * P.ntypes), "workspace");
    CU(m->fslot.reserve(sizeof(double) * 3 * (size_t)(N + 1) * P.nm), "workspace");
    CU(m->vpart.reserve(sizeof(double) * 9 * (size_t)(N + 1)), "workspace");
  }
  int dt_pad = 0;
  // deterministic sub-region mode: the ghosts' lists are built too (list only), in chunks of their own
  const int64_t nghost = (det && nloc > 0) ? natoms - nloc : 0;
  const int64_t gchunk = chunk_cap < nghost ? chunk_cap : nghost;
  const int64_t lrows = chunk > gchunk ? chunk : gchunk;
  CU(m->nl.reserve(sizeof(int) * (size_t)chunk * P.nm), "workspace");
  CU(m->nlp.reserve(sizeof(int) * (size_t)lrows * P.nm), "workspace");
  CU(m->counters.reserve(sizeof(int) * 128), "workspace");
  CU(m->dr.reserve(sizeof(double4) * (size_t)lrows * P.nm), "workspace");
  CU(m->nreal.reserve(sizeof(int) * (size_t)chunk * P.ntypes), "workspace");
  // Stored activations (dpb_model_set_stored_activations): one record per (centre, slot) of the chunk, taken when the
  // records fit into the workspace budget and the chunk is large enough for whole-atom work items
  int act_stride = 0;
  if (!nlist_only && act_record_doubles(m) > 0 && chunk >= 4096 && (size_t)chunk * P.nm < 2000000000ull) {
    const int stride = act_record_doubles(m);
    const size_t bytes = sizeof(double) * (size_t)chunk * P.nm * stride;
    if (bytes <= m->ws_budget) {
      const cudaError_t ea = m->act.reserve(bytes, false, true);
      if (ea == cudaSuccess) act_stride = stride;
      else if (ea == cudaErrorMemoryAllocation) cudaGetLastError();      // no room today: pass 2 recomputes
      else return cuda_fail(ea, "workspace of the stored activations");
    }
  }
  if (!nlist_only) {
    CU(m->T.reserve(sizeof(double) * (size_t)chunk * P.M * 4), "workspace");
    // fp64 variant 1 keeps dT in the padded lane order of the DMMA kernels (ChunkView::dt_pad); the pad rows are zero
    dt_pad = (m->precision == DPB_FP64 && m->variant == 1 && m->v1.ready) ? 4 * m->v1.SP : 0;
    const size_t dt_bytes = sizeof(double) * (size_t)chunk * (dt_pad ? 4 * dt_pad : P.M) * 4;
    if (dt_pad != m->dt_pad_alloc) { m->dT.release(); m->dt_pad_alloc = dt_pad; }
    CU(m->dT.reserve(dt_bytes, true), "workspace");
    if (m->precision == DPB_FP64 && (m->variant == 0 || !m->v1.ready)) {
      CU(m->v0[0].reserve(sizeof(double) * (size_t)chunk * P.dim), "workspace");
      CU(m->v0[1].reserve(sizeof(double) * (size_t)chunk * P.dim), "workspace");
      for (int k = 2; k < 9; ++k) CU(m->v0[k].reserve(sizeof(double) * (size_t)chunk * P.fw), "workspace");
    } else {
      CU(m->v1ws.reserve(v1_workspace_bytes(P, chunk)), "workspace");
    }
    if (m->precision == DPB_FP64 && m->variant == 2)
      CU(m->v2ws.reserve((size_t)chunk * P.nm * v2_slot_bytes(m->v2)), "workspace of the paper pipeline");
    if (m->precision != DPB_FP64) {
      CU(m->pairs.reserve(tc_pair_workspace_bytes(P, chunk)), "workspace");
      CU(m->dT32.reserve(tc_pass2_workspace_bytes(P, chunk)), "workspace");
      CU(m->tcfit.reserve(tc_fit_workspace_bytes(P, chunk, m->precision - DPB_TF32)), "workspace");
    }
  }
  DevStats *stats = m->stats.as<DevStats>();
  // Small single-chunk periodic evaluations: the memsets (each a node in the chain of dependent launches) are folded into
  // the cell-sort and list kernels (ZeroJobs, common.cuh)
  const bool fold = !nlist_only && nl_mode == 0 && nloc < 0 && natoms > 0 && natoms <= 4096 && chunk >= ncentre &&
                    m->precision == DPB_FP64 && m->variant == 1 && m->v1.ready && !det;
  ZeroJobs zj{};
  if (fold) {
    zj.stats = stats; zj.stats_bytes = (int)(2 * sizeof(DevStats));
    zj.counters = m->counters.as<int>(); zj.ncounters = 128;
    zj.T = m->T.as<double>(); zj.t_len = P.M * 4;
    zj.Z0 = v1_fit_preact(m->v1, m->v1ws.p, ncentre, &zj.z_len);
    zj.force = force; zj.virial = virial;
  }
  if (nl_mode == 0 && !fold) CU(cudaMemsetAsync(stats, 0, 2 * sizeof(DevStats), st), "memset stats");   // MD: kept over the run
  NlRaw raw{};
  if (nl_mode != 0) {
    raw.raw = m->md_raw.as<int>(); raw.nraw = m->md_nraw.as<int>(); raw.cap = m->md_cap_raw;
    const double rs = P.rc + m->md_skin;
    raw.rs2_hi = rs * rs * (1.0 + 1e-9);
  }
  const bool timing = m->timing && !nlist_only;
  const int nchunks = (int)((ncentre + chunk - 1) / chunk);
  if (timing) {
    const size_t need = 3 + 4 * (size_t)nchunks;
    while (m->evs.size() < need) {
      cudaEvent_t e;
      CU(cudaEventCreate(&e), "cudaEventCreate");
      m->evs.push_back(e);
    }
    m->ev_chunks = nchunks;
    cudaEventRecord(m->evs[0], st);
  }

  m->last_natoms = natoms;
  int *start = m->start.as<int>();
  if (nl_mode == 2) {
    CU(launch_gather_sorted(natoms, coord, m->s_idx.as<int>(), m->s_xyz.as<double>(), m->md_xyz0.as<double>(), stats,
                            st), "gather");
  } else {
    CU(launch_cell_sort(P, G, natoms, coord, type, m->key.as<int>(), m->count.as<int>(), start, m->cursor.as<int>(),
                        m->s_idx.as<int>(), m->s_xyz.as<double>(), stats, st, m->pos_of.as<int>(), fold ? &zj : nullptr),
       "cell sort");
    if (nl_mode == 1 && natoms > 0)
      CU(cudaMemcpyAsync(m->md_xyz0.p, m->s_xyz.p, sizeof(double) * 3 * (size_t)natoms, cudaMemcpyDeviceToDevice, st),
         "copy of the rebuild coordinates");
  }
  if (timing) cudaEventRecord(m->evs[1], st);
  int ts_h[DPB_MAX_TYPES + 1] = {0};
  if (m->precision == DPB_FP64 && m->variant == 2 && !nlist_only) {      // batch sizes of the padded GEMMs: one host sync
    CU(cudaMemcpyAsync(ts_h, start + nkeys + 1, sizeof(int) * (P.ntypes + 1), cudaMemcpyDeviceToHost, st), "type counts");
    CU(cudaStreamSynchronize(st), "stream synchronise");
  }

  double *ei = atom_energy ? atom_energy : m->ei.as<double>();
  if (!nlist_only && !fold) {
    if (force) CU(cudaMemsetAsync(force, 0, sizeof(double) * 3 * (size_t)natoms, st), "memset force");
    if (virial) CU(cudaMemsetAsync(virial, 0, sizeof(double) * 9, st), "memset virial");
  }
  const int cap = neighbour_cap(P);
  int ci = 0;
  bool energy_done = false;
  for (int64_t p0 = 0; p0 < ncentre; p0 += chunk, ++ci) {
    ChunkView C;
    C.p0 = (int)p0;
    C.n = (int)((ncentre - p0) < chunk ? (ncentre - p0) : chunk);
    C.s_idx = m->s_idx.as<int>();
    C.type_start = start + nkeys + 1;
    C.nl = m->nl.as<int>();
    C.dr = m->dr.as<double4>();
    C.nreal = m->nreal.as<int>();
    C.T = m->T.as<double>();
    C.dT = m->dT.as<double>();
    C.dt_pad = dt_pad;
    C.dt_rows = dt_pad ? 4 * dt_pad : P.M;
    C.nlp = m->nlp.as<int>();
    C.counters = m->counters.as<int>();
    C.sub_part = 0; C.sub_nparts = 1;
    if (!nlist_only && !fold) CU(cudaMemsetAsync(C.counters, 0, sizeof(int) * 128, st), "memset counters");
    C.fslot = nullptr;
    C.pos_of = m->pos_of.as<int>();
    C.stats = stats;
    C.reuse = (!det && (m->pair_reuse == 2 || (m->pair_reuse == 1 && (nchunks == 1 || chunk >= 32768)))) ? 1 : 0;
    C.reuse2 = (!det && m->pair_reuse >= 1) ? 1 : 0;     // pass 2 only reads dT_j: no bookkeeping, any chunking
    C.act = act_stride ? m->act.as<double>() : nullptr;
    C.act_stride = act_stride;
    C.prezero = fold ? 1 : 0;
    C.typed_pipe = (P.ntypes > 1 && C.n >= 4096 && !timing && !det && m->precision == DPB_FP64 && m->variant == 1 &&
                    m->v1.ready && !m->dbgT && !m->dbgD && !m->dbgdT && m->species_pipe) ? 1 : 0;
    if (det) {                                           // full-size lists: the gather needs every atom's row
      C.nl = m->nl_all.as<int>() + (size_t)p0 * P.nm;
      C.nreal = m->nreal_all.as<int>() + (size_t)p0 * P.ntypes;
      C.fslot = m->fslot.as<double>() + 3 * (size_t)p0 * P.nm;
    }
    CU(launch_nlist(P, G, C, m->s_xyz.as<double>(), start, cap, nlist, stats, st, nl_mode, nl_mode ? &raw : nullptr,
                    fold ? &zj : nullptr), "nlist");
    if (nlist_only) continue;
    if (timing) cudaEventRecord(m->evs[2 + 4 * ci], st);
    if (m->precision != DPB_FP64) {
      CU(tc_build_pairs(P, C, m->pairs.p, st), "pair list");
      CU(tc_pass1(P, C, m->tcw, m->pairs.p, st), "pass1 tf32");
      if (timing) cudaEventRecord(m->evs[3 + 4 * ci], st);
      CU(tc_fit(P, C, m->tcw, m->tcfit.p, m->dT32.as<float>(), ei, st, m->dbgdT != nullptr), "fit tf32");
      CU(launch_scatter_debug(P, C, m->dbgT, m->dbgdT, st), "debug scatter");
      if (timing) cudaEventRecord(m->evs[4 + 4 * ci], st);
      CU(tc_pass2(P, C, m->tcw, m->pairs.p, m->dT32.as<float>(), force, virial, st), "pass2 tf32");
      if (timing) cudaEventRecord(m->evs[5 + 4 * ci], st);
    } else if (m->variant == 2) {
      CU(v2_pass1(P, C, m->v2, ts_h, m->v2ws.p, st), "pass1 v2");
      if (timing) cudaEventRecord(m->evs[3 + 4 * ci], st);
      CU(v1_fit(P, C, m->v1, m->fit.as<double>(), m->v1ws.p, ei, st), "fit");
      CU(launch_scatter_debug(P, C, m->dbgT, m->dbgdT, st), "debug scatter");
      if (timing) cudaEventRecord(m->evs[4 + 4 * ci], st);
      CU(v2_pass2(P, C, m->v2, ts_h, m->v2ws.p, force, virial, st), "pass2 v2");
      if (timing) cudaEventRecord(m->evs[5 + 4 * ci], st);
    } else if (m->variant == 0 || !m->v1.ready) {
      V0Scratch S;
      S.D = m->v0[0].as<double>(); S.dD = m->v0[1].as<double>();
      S.Z0 = m->v0[2].as<double>(); S.U1 = m->v0[3].as<double>(); S.Z1 = m->v0[4].as<double>();
      S.U2 = m->v0[5].as<double>(); S.Z2 = m->v0[6].as<double>(); S.G = m->v0[7].as<double>();
      S.dZ = m->v0[8].as<double>();
      CU(launch_pass1_v0(P, C, m->emb.as<double>(), st), "pass1 v0");
      if (timing) cudaEventRecord(m->evs[3 + 4 * ci], st);
      CU(launch_fit_v0(P, C, m->fit.as<double>(), S, ei, m->dbgD, st), "fit v0");
      CU(launch_scatter_debug(P, C, m->dbgT, m->dbgdT, st), "debug scatter");
      if (timing) cudaEventRecord(m->evs[4 + 4 * ci], st);
      CU(launch_pass2_v0(P, C, m->emb.as<double>(), force, virial, st), "pass2 v0");
      if (timing) cudaEventRecord(m->evs[5 + 4 * ci], st);
    } else {
      CU(v1_pass1(P, C, m->v1, st), "pass1");
      if (timing) cudaEventRecord(m->evs[3 + 4 * ci], st);
      CU(v1_fit(P, C, m->v1, m->fit.as<double>(), m->v1ws.p, ei, st), "fit");
      CU(launch_scatter_debug(P, C, m->dbgT, m->dbgdT, st), "debug scatter");
      if (timing) cudaEventRecord(m->evs[4 + 4 * ci], st);
      // Small single-chunk evaluations: E = sum E_i (complete once the fitting stage has run) goes on a forked stream
      // beside pass 2 instead of behind it — one dependent launch less in a chain that is bound by its launches.
      cudaStream_t es[DPB_MAX_TYPES];
      const bool early_e = energy && !timing && nchunks == 1 && ncentre <= 4096;
      if (early_e) {
        CU(dpb_fork_streams(2, st, es), "fork");
        CU(launch_reduce_energy(ncentre, ei, energy, es[1]), "energy reduction");
        energy_done = true;
      }
      CU(v1_pass2(P, C, m->v1, force, virial, st), "pass2");
      if (early_e) CU(dpb_join_streams(2, st, es), "join");
      if (timing) cudaEventRecord(m->evs[5 + 4 * ci], st);
    }
  }
  for (int64_t p0 = nloc; nghost > 0 && p0 < natoms; p0 += gchunk) {      // ghost rows of the full-size list
    ChunkView C{};
    C.p0 = (int)p0;
    C.n = (int)((natoms - p0) < gchunk ? (natoms - p0) : gchunk);
    C.s_idx = m->s_idx.as<int>();
    C.type_start = start + nkeys + 1;
    C.nl = m->nl_all.as<int>() + (size_t)p0 * P.nm;
    C.nreal = m->nreal_all.as<int>() + (size_t)p0 * P.ntypes;
    C.dr = m->dr.as<double4>();
    C.nlp = m->nlp.as<int>();
    C.pos_of = m->pos_of.as<int>();
    C.sub_nparts = 1;
    C.stats = stats + 1;
    CU(launch_nlist(P, G, C, m->s_xyz.as<double>(), start, cap, nullptr, stats + 1, st, 0, nullptr), "nlist of the ghosts");
  }
  if (nghost > 0) CU(launch_merge_ghost_stats(stats, st), "ghost statistics");
  if (det && ncentre > 0)
    CU(launch_force_gather(P, G, natoms, ncentre, m->s_idx.as<int>(), m->pos_of.as<int>(), start + nkeys + 1,
                           m->s_xyz.as<double>(), m->nl_all.as<int>(), m->nreal_all.as<int>(), m->fslot.as<double>(),
                           force, m->atom_virial ? m->atom_virial : m->vpart.as<double>(), virial, st),
       "deterministic force gather");
  if (!nlist_only) {
    if (energy && !energy_done) CU(launch_reduce_energy(ncentre, ei, energy, st), "energy reduction");
    if (timing) cudaEventRecord(m->evs[2 + 4 * nchunks], st);
  }
  return DPB_OK;
}

static int finish_info(dpb_model *m, cudaStream_t st, int64_t natoms, dpb_eval_info *info) {
  DevStats hs;
  CU(cudaMemcpyAsync(&hs, m->stats.p, sizeof(DevStats), cudaMemcpyDeviceToHost, st), "stats copy");
  CU(cudaStreamSynchronize(st), "stream synchronise");
  if (hs.err_type) return fail(DPB_EINVAL, "an atom has a type index outside [0, ntypes)");
  if (hs.err_cap) return fail(DPB_ECAP, "an atom has more in-range candidates than the staging capacity (%d)",
                              neighbour_cap(m->P));
  if (hs.err_bounds) return fail(DPB_EBOX, "an atom lies outside the bounds given to dpb_eval_local");
  if (info) {
    memset(info, 0, sizeof(*info));
    info->n_real_pairs = (int64_t)hs.n_real_pairs;
    info->n_overflow = (int64_t)hs.n_overflow;
    for (int t = 0; t < 8 && t < DPB_MAX_TYPES; ++t) info->max_nei[t] = hs.max_nei[t];
    const int64_t chunk = effective_chunk(m, natoms);
    info->n_chunks = (int32_t)((natoms + chunk - 1) / chunk);
  }
  return DPB_OK;
}

extern "C" int dpb_model_status(dpb_model *m, void *stream) {
  if (!m) return fail(DPB_EINVAL, "dpb_model_status: null model");
  return finish_info(m, reinterpret_cast<cudaStream_t>(stream), 0, nullptr);
}

extern "C" int dpb_model_set_graph(dpb_model *m, int mode) {
  if (!m || mode < 0 || mode > 2) return fail(DPB_EINVAL, "dpb_model_set_graph: mode must be 0, 1 or 2");
  m->graph_mode = mode;
  return DPB_OK;
}

// dpb_eval through a CUDA graph.  The first call with a given argument set runs eagerly (it sizes the workspace and sets
// the kernel attributes), the second one is captured — run_eval only enqueues work, forks and joins included — and
// instantiated, later ones replay the graph: one launch instead of ~30, which is what a 192-atom evaluation is bound
// by.  Returns 1 if the call was served by a graph, 0 if the caller has to run it eagerly, < 0 on error.
static int eval_graphed(dpb_model *m, cudaStream_t st, int64_t natoms, const double *coord, const int32_t *type,
                        const double box[9], double *energy, double *atom_energy, double *force, double *virial,
                        int32_t *nlist) {
  if (m->graph_mode == 0 || m->timing || m->variant == 2 || (m->graph_mode == 1 && natoms > DPB_GRAPH_AUTO_ATOMS)) return 0;
  GraphKey key;
  memset(&key, 0, sizeof(key));
  key.natoms = natoms;
  const void *ptrs[7] = {coord, type, energy, atom_energy, force, virial, nlist};
  memcpy(key.ptr, ptrs, sizeof(ptrs));
  memcpy(key.box, box, sizeof(key.box));
  const unsigned long long epoch = g_ws_epoch * 1000003ull + m->cfg_epoch;
  GraphEntry *hit = nullptr;
  for (GraphEntry &g : m->graphs) if (g.key == key) { hit = &g; break; }
  if (hit && hit->epoch != epoch) {                       // workspace or configuration changed since: start over
    if (hit->exec) cudaGraphExecDestroy(hit->exec);
    hit->exec = nullptr; hit->failed = false; hit->epoch = 0;
  }
  if (!hit) {
    if (m->graphs.size() < DPB_GRAPH_SLOTS) { m->graphs.emplace_back(); hit = &m->graphs.back(); }
    else {
      hit = &m->graphs[0];
      for (GraphEntry &g : m->graphs) if (g.stamp < hit->stamp) hit = &g;
      if (hit->exec) cudaGraphExecDestroy(hit->exec);
      *hit = GraphEntry();
    }
    hit->key = key;
  }
  hit->stamp = ++m->graph_clock;
  if (hit->failed) return 0;
  if (hit->exec) {
    cudaError_t e = cudaGraphLaunch(hit->exec, st);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGraphLaunch");
    DPB_LAUNCHED(hit->kernels);
    return 1;
  }
  if (hit->epoch == 0) { hit->epoch = epoch; return 0; }  // first sighting: eager (may grow the workspace: new epoch)
  // second call in the same state: capture
  const unsigned long long l0 = g_dpb_launches;
  cudaError_t e = cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed);
  if (e != cudaSuccess) { cudaGetLastError(); hit->failed = true; return 0; }
  const int rc = run_eval(m, st, natoms, coord, type, box, energy, atom_energy, force, virial, nlist, false);
  cudaGraph_t graph = nullptr;
  e = cudaStreamEndCapture(st, &graph);
  const long long kernels = (long long)(g_dpb_launches - l0);
  g_dpb_launches = l0;                                    // nothing has run yet
  if (rc != DPB_OK || e != cudaSuccess || !graph || g_ws_epoch * 1000003ull + m->cfg_epoch != epoch) {
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    hit->failed = true;
    return rc != DPB_OK ? rc : 0;
  }
  e = cudaGraphInstantiate(&hit->exec, graph, 0);
  cudaGraphDestroy(graph);
  if (e != cudaSuccess) { cudaGetLastError(); hit->exec = nullptr; hit->failed = true; return 0; }
  hit->kernels = kernels;
  e = cudaGraphLaunch(hit->exec, st);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGraphLaunch");
  DPB_LAUNCHED(hit->kernels);
  return 1;
}

extern "C" int dpb_eval(dpb_model *m, void *stream, int64_t natoms, const double *coord, const int32_t *type,
                        const double box[9], double *energy, double *atom_energy, double *force, double *virial,
                        int32_t *nlist, dpb_eval_info *info) {
  if (!m || !box) return fail(DPB_EINVAL, "dpb_eval: null model / box");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (!info) {
    const int g = eval_graphed(m, st, natoms, coord, type, box, energy, atom_energy, force, virial, nlist);
    if (g != 0) return g < 0 ? g : DPB_OK;
  }
  int rc = run_eval(m, st, natoms, coord, type, box, energy, atom_energy, force, virial, nlist, false);
  if (rc != DPB_OK) return rc;
  if (info) return finish_info(m, st, natoms, info);
  return DPB_OK;
}

extern "C" int dpb_eval_local(dpb_model *m, void *stream, int64_t nloc, int64_t nall, const double *coord,
                              const int32_t *type, const double bounds[6], double *energy, double *atom_energy,
                              double *force, double *virial, int32_t *nlist, dpb_eval_info *info) {
  if (!m || !bounds) return fail(DPB_EINVAL, "dpb_eval_local: null model / bounds");
  if (nloc < 0) return fail(DPB_EINVAL, "dpb_eval_local: nloc < 0");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  int rc = run_eval(m, st, nall, coord, type, bounds, energy, atom_energy, force, virial, nlist, false, 0, nloc);
  if (rc != DPB_OK) return rc;
  if (info) return finish_info(m, st, nloc, info);
  return DPB_OK;
}

// ---- general periodic cell through explicit images ---------------------------
extern "C" int dpb_eval_cell(dpb_model *m, void *stream, int64_t natoms, const double *coord, const int32_t *type,
                             const double cell[9], double *energy, double *atom_energy, double *force, double *virial,
                             dpb_eval_info *info) {
  if (!m || !cell) return fail(DPB_EINVAL, "dpb_eval_cell: null model / cell");
  if (natoms < 0 || natoms > 2000000000ll) return fail(DPB_EINVAL, "natoms out of range");
  if (natoms > 0 && (!coord || !type)) return fail(DPB_EINVAL, "null coord / type");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const DevModel &P = m->P;
  CellGeom G;
  const double *a = cell;
  for (int k = 0; k < 9; ++k) G.A[k] = a[k];
  const double cr[3][3] = {{a[4] * a[8] - a[5] * a[7], a[5] * a[6] - a[3] * a[8], a[3] * a[7] - a[4] * a[6]},   // a1 x a2
                           {a[7] * a[2] - a[8] * a[1], a[8] * a[0] - a[6] * a[2], a[6] * a[1] - a[7] * a[0]},   // a2 x a0
                           {a[1] * a[5] - a[2] * a[4], a[2] * a[3] - a[0] * a[5], a[0] * a[4] - a[1] * a[3]}};  // a0 x a1
  const double det = a[0] * cr[0][0] + a[1] * cr[0][1] + a[2] * cr[0][2];
  if (!(fabs(det) > 0.0) || !std::isfinite(det)) return fail(DPB_EBOX, "dpb_eval_cell: the cell is singular");
  long long nshift = 1;
  for (int c = 0; c < 3; ++c) {
    const double nrm = sqrt(cr[c][0] * cr[c][0] + cr[c][1] * cr[c][1] + cr[c][2] * cr[c][2]);
    const double h = fabs(det) / nrm;                      // perpendicular height along lattice direction c
    G.margin[c] = P.rc / h;
    const double ns = ceil(G.margin[c]);
    if (!(ns <= 16.0)) return fail(DPB_EBOX, "dpb_eval_cell: the cell is thinner than r_c / 16 along lattice vector %d", c);
    G.nshell[c] = (int)ns;
    nshift *= 2 * G.nshell[c] + 1;
    for (int r = 0; r < 3; ++r) G.Ainv[3 * r + c] = cr[c][r] / det;      // column c of A^-1 = (a_j x a_k) / det
  }
  // bounds: the 8 corners of the parallelepiped widened by the margins
  double bounds[6] = {1e300, 1e300, 1e300, -1e300, -1e300, -1e300}, big = 0.0;
  for (int k = 0; k < 8; ++k) {
    double f[3], x[3] = {0.0, 0.0, 0.0};
    for (int c = 0; c < 3; ++c) f[c] = ((k >> c) & 1) ? 1.0 + G.margin[c] : -G.margin[c];
    for (int c = 0; c < 3; ++c) x[c] = f[0] * a[c] + f[1] * a[3 + c] + f[2] * a[6 + c];
    for (int c = 0; c < 3; ++c) {
      if (x[c] < bounds[c]) bounds[c] = x[c];
      if (x[c] > bounds[3 + c]) bounds[3 + c] = x[c];
      if (fabs(x[c]) > big) big = fabs(x[c]);
    }
  }
  for (int c = 0; c < 3; ++c) { bounds[c] -= 1e-9 * (1.0 + big); bounds[3 + c] += 1e-9 * (1.0 + big); }
  CU(m->cell_frac.reserve(sizeof(double) * 3 * ((size_t)natoms + 1)), "cell workspace");
  CU(m->cell_off.reserve(sizeof(int) * ((size_t)natoms + 1)), "cell workspace");
  int *off = m->cell_off.as<int>();
  CU(launch_cell_wrap(natoms, coord, G, m->cell_frac.as<double>(), st), "cell wrap");
  CU(launch_cell_images(natoms, m->cell_frac.as<double>(), type, G, off, nullptr, nullptr, 0, st), "cell image count");
  int nimg = 0;                                            // the number of images sizes the evaluation: one host sync
  CU(cudaMemcpyAsync(&nimg, off + natoms, sizeof(int), cudaMemcpyDeviceToHost, st), "image count");
  CU(cudaStreamSynchronize(st), "stream synchronise");
  const int64_t nall = natoms + (int64_t)nimg;
  if (nall > 2000000000ll - 1)                             // (k_cell_scan saturates the count at 2e9)
    return fail(DPB_EINVAL, "dpb_eval_cell: too many lattice images (at least %lld)", (long long)nimg);
  CU(m->cell_x.reserve(sizeof(double) * 3 * ((size_t)nall + 1)), "cell workspace");
  CU(m->cell_t.reserve(sizeof(int) * ((size_t)nall + 1)), "cell workspace");
  CU(m->cell_f.reserve(sizeof(double) * 3 * ((size_t)nall + 1)), "cell workspace");
  CU(launch_cell_images(natoms, m->cell_frac.as<double>(), type, G, off, m->cell_x.as<double>(), m->cell_t.as<int>(), 1,
                        st), "cell images");
  int rc = run_eval(m, st, nall, m->cell_x.as<double>(), m->cell_t.as<int>(), bounds, energy, atom_energy,
                    force ? m->cell_f.as<double>() : nullptr, virial, nullptr, false, 0, natoms);
  if (rc != DPB_OK) return rc;
  if (force) CU(launch_cell_fold(natoms, off, m->cell_f.as<double>(), force, st), "cell fold");
  if (info) return finish_info(m, st, natoms, info);
  return DPB_OK;
}

// ---- velocity-Verlet pieces for drivers that own the time loop (the decomposition's MD driver, dd.py) -----------------
extern "C" int dpb_md_coefficients(const double *mass_h, int32_t ntypes, double dt_fs, double *coeff_h) {
  if (!mass_h || !coeff_h || ntypes < 1 || ntypes > DPB_MAX_TYPES || !(dt_fs > 0.0))
    return fail(DPB_EINVAL, "dpb_md_coefficients: bad argument");
  const double AMU = 103.6426965268;                           // 1 amu A^2/fs^2 in eV (CODATA 2018)
  for (int t = 0; t < ntypes; ++t) {
    if (!(mass_h[t] > 0.0)) return fail(DPB_EINVAL, "dpb_md_coefficients: mass[%d] <= 0", t);
    coeff_h[t] = 0.5 * dt_fs / (mass_h[t] * AMU);
    coeff_h[ntypes + t] = mass_h[t] * AMU;
  }
  return DPB_OK;
}

extern "C" int dpb_md_kick_drift(void *stream, int64_t n, double *coord, double *vel, const double *force,
                                 const int32_t *type, const double *coeff, double dt_fs) {
  if (n < 0 || n > 2000000000ll) return fail(DPB_EINVAL, "dpb_md_kick_drift: n out of range");
  if (n > 0 && (!coord || !vel || !force || !type || !coeff)) return fail(DPB_EINVAL, "dpb_md_kick_drift: null argument");
  CU(launch_md_kick_drift(n, coord, vel, force, type, coeff, dt_fs, reinterpret_cast<cudaStream_t>(stream)), "kick + drift");
  return DPB_OK;
}

extern "C" int dpb_md_kick(void *stream, int64_t n, double *vel, const double *force, const int32_t *type,
                           const double *coeff) {
  if (n < 0 || n > 2000000000ll) return fail(DPB_EINVAL, "dpb_md_kick: n out of range");
  if (n > 0 && (!vel || !force || !type || !coeff)) return fail(DPB_EINVAL, "dpb_md_kick: null argument");
  CU(launch_md_kick(n, vel, force, type, coeff, reinterpret_cast<cudaStream_t>(stream)), "kick");
  return DPB_OK;
}

extern "C" int dpb_md_kinetic_energy(void *stream, int64_t n, const double *vel, const int32_t *type,
                                     const double *mass_ev, double *ekin) {
  if (n < 0 || n > 2000000000ll || !ekin) return fail(DPB_EINVAL, "dpb_md_kinetic_energy: bad argument");
  if (n > 0 && (!vel || !type || !mass_ev)) return fail(DPB_EINVAL, "dpb_md_kinetic_energy: null argument");
  CU(launch_md_ekin(n, vel, type, mass_ev, ekin, reinterpret_cast<cudaStream_t>(stream)), "kinetic energy");
  return DPB_OK;
}

extern "C" int dpb_dd_pack(void *stream, int64_t n, const double *coord, const int32_t *type, int32_t dim,
                           double cut_minus, double cut_plus, double shift_minus, double shift_plus, int64_t cap,
                           double *pack_minus, int32_t *idx_minus, double *pack_plus, int32_t *idx_plus,
                           int32_t *counts) {
  if (n < 0 || n > 2000000000ll || cap < 0 || cap > 2000000000ll || dim < 0 || dim > 2)
    return fail(DPB_EINVAL, "dpb_dd_pack: n / cap / dim out of range");
  if (!counts || (n > 0 && (!coord || !type)) || (cap > 0 && (!pack_minus || !idx_minus || !pack_plus || !idx_plus)))
    return fail(DPB_EINVAL, "dpb_dd_pack: null argument");
  CU(launch_dd_pack(n, coord, type, dim, cut_minus, cut_plus, shift_minus, shift_plus, cap, pack_minus, idx_minus,
                    pack_plus, idx_plus, counts, reinterpret_cast<cudaStream_t>(stream)), "dd pack");
  return DPB_OK;
}

extern "C" int dpb_dd_unpack(void *stream, int64_t k, const double *pack, double *coord_out, int32_t *type_out) {
  if (k < 0 || k > 2000000000ll) return fail(DPB_EINVAL, "dpb_dd_unpack: k out of range");
  if (k > 0 && (!pack || !coord_out || !type_out)) return fail(DPB_EINVAL, "dpb_dd_unpack: null argument");
  CU(launch_dd_unpack(k, pack, coord_out, type_out, reinterpret_cast<cudaStream_t>(stream)), "dd unpack");
  return DPB_OK;
}

extern "C" int dpb_dd_add_forces(void *stream, int64_t k, const int32_t *idx, const double *fin, double *force) {
  if (k < 0 || k > 2000000000ll) return fail(DPB_EINVAL, "dpb_dd_add_forces: k out of range");
  if (k > 0 && (!idx || !fin || !force)) return fail(DPB_EINVAL, "dpb_dd_add_forces: null argument");
  CU(launch_dd_add_forces(k, idx, fin, force, reinterpret_cast<cudaStream_t>(stream)), "dd add forces");
  return DPB_OK;
}

extern "C" int dpb_build_nlist(dpb_model *m, void *stream, int64_t natoms, const double *coord, const int32_t *type,
                               const double box[9], int32_t *nlist, int64_t *n_overflow) {
  if (!m || !box || !nlist) return fail(DPB_EINVAL, "dpb_build_nlist: null argument");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  int rc = run_eval(m, st, natoms, coord, type, box, nullptr, nullptr, nullptr, nullptr, nlist, true);
  if (rc != DPB_OK) return rc;
  if (n_overflow) {
    dpb_eval_info info;
    rc = finish_info(m, st, natoms, &info);
    if (rc != DPB_OK) return rc;
    *n_overflow = info.n_overflow;
  }
  return DPB_OK;
}

// ---- dpb_build_nlist_static: Alg. 1 without any allocation -------------------------------------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
// The kernels are those of dpb_build_nlist (k_keys / k_scan / k_fill / k_nlist); what differs is where their scratch
// lives: not in the model's workspace (Buf::reserve -> cudaMalloc) but in ONE file-scope device array of fixed size that
// every GPU which loads the library holds until the process exits.  Limits (checked, DPB_EINVAL beyond them):
#define DPB_STATIC_MAX_ATOMS 4096                     // natoms
#define DPB_STATIC_MAX_SLOTS (1 << 18)                // natoms * Nm       (W192: 26,496)
#define DPB_STATIC_MAX_KEYS 16384                     // ntypes * cells of the search grid
// Layout of the array (byte offsets, every piece 256-byte aligned):
#define SN_AL(x) (((size_t)(x) + 255) & ~(size_t)255)
#define SN_STATS 0
#define SN_KEY (SN_STATS + SN_AL(sizeof(DevStats)))
#define SN_SIDX (SN_KEY + SN_AL(4 * (DPB_STATIC_MAX_ATOMS + 1)))
#define SN_SXYZ (SN_SIDX + SN_AL(4 * (DPB_STATIC_MAX_ATOMS + 1)))
#define SN_COUNT (SN_SXYZ + SN_AL(24 * (DPB_STATIC_MAX_ATOMS + 1)))
#define SN_START (SN_COUNT + SN_AL(4 * (DPB_STATIC_MAX_KEYS + 1)))
#define SN_CURSOR (SN_START + SN_AL(4 * (DPB_STATIC_MAX_KEYS + 1 + DPB_MAX_TYPES + 1)))
#define SN_NREAL (SN_CURSOR + SN_AL(4 * (DPB_STATIC_MAX_KEYS + 1)))
#define SN_NL (SN_NREAL + SN_AL(4 * DPB_STATIC_MAX_ATOMS * DPB_MAX_TYPES))
#define SN_DR (SN_NL + SN_AL(4 * (size_t)DPB_STATIC_MAX_SLOTS))
#define SN_TOTAL (SN_DR + SN_AL(32 * (size_t)DPB_STATIC_MAX_SLOTS))            // 9.9 MB
static __device__ __align__(256) unsigned char g_static_scratch[SN_TOTAL];

// In host code `g_static_scratch` is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, once per device, with that device current.
static unsigned char *g_static_ptr[DPB_MAX_DEVICES] = {};

static int static_scratch(unsigned char **out) {
  int dev = 0;
  CU(cudaGetDevice(&dev), "cudaGetDevice");
  if (dev < 0 || dev >= DPB_MAX_DEVICES) return fail(DPB_EINVAL, "device index %d beyond DPB_MAX_DEVICES", dev);
  if (!g_static_ptr[dev]) {
    void *p = nullptr;
    CU(cudaGetSymbolAddress(&p, g_static_scratch), "cudaGetSymbolAddress of the static scratch");
    if (!p) return fail(DPB_ECUDA, "cudaGetSymbolAddress returned a null address");
    g_static_ptr[dev] = static_cast<unsigned char *>(p);
  }
  *out = g_static_ptr[dev];
  return DPB_OK;
}

// status[0..3] = real pairs, dropped neighbours (n_overflow), error bits (1: type out of range, 2: staging cap), largest
// candidate count of any (atom, type)
__global__ void k_static_status(const DevStats *__restrict__ s, int ntypes, long long *__restrict__ status) {
  int mx = 0;
  for (int t = 0; t < ntypes; ++t) mx = s->max_nei[t] > mx ? s->max_nei[t] : mx;
  status[0] = (long long)s->n_real_pairs;
  status[1] = (long long)s->n_overflow;
  status[2] = (s->err_type ? 1 : 0) | (s->err_cap ? 2 : 0);
  status[3] = mx;
}

extern "C" int dpb_build_nlist_static(const dpb_model *m, void *stream, int64_t natoms, const double *coord,
                                      const int32_t *type, const double box[9], int32_t *nlist, int64_t *status) {
  if (!m || !box) return fail(DPB_EINVAL, "dpb_build_nlist_static: null model / box");
  const DevModel &P = m->P;
  if (natoms < 0) return fail(DPB_EINVAL, "dpb_build_nlist_static: natoms < 0");
  if (natoms > DPB_STATIC_MAX_ATOMS)
    return fail(DPB_EINVAL, "dpb_build_nlist_static: %lld atoms exceed the static scratch (at most %d atoms); use "
                            "dpb_build_nlist", (long long)natoms, DPB_STATIC_MAX_ATOMS);
  if (natoms * (int64_t)P.nm > DPB_STATIC_MAX_SLOTS)
    return fail(DPB_EINVAL, "dpb_build_nlist_static: natoms * Nm = %lld exceeds the static scratch (at most %d slots); "
                            "use dpb_build_nlist", (long long)(natoms * P.nm), DPB_STATIC_MAX_SLOTS);
  if (natoms > 0 && (!coord || !type || !nlist)) return fail(DPB_EINVAL, "dpb_build_nlist_static: null coord / type / nlist");
  DevGrid G;
  int rc = make_grid(P, box, G, P.rc);
  if (rc != DPB_OK) return rc;
  const int nkeys = P.ntypes * G.ncell;
  if (nkeys > DPB_STATIC_MAX_KEYS)
    return fail(DPB_EINVAL, "dpb_build_nlist_static: ntypes * cells = %d exceeds the static scratch (at most %d); use "
                            "dpb_build_nlist", nkeys, DPB_STATIC_MAX_KEYS);
  unsigned char *base = nullptr;
  if ((rc = static_scratch(&base)) != DPB_OK) return rc;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  DevStats *stats = reinterpret_cast<DevStats *>(base + SN_STATS);
  int *start = reinterpret_cast<int *>(base + SN_START);
  // the array keeps the last call's contents: the statistics start at zero (the cell counts are cleared by the sort)
  CU(cudaMemsetAsync(stats, 0, sizeof(DevStats), st), "memset stats");
  CU(launch_cell_sort(P, G, natoms, coord, type, reinterpret_cast<int *>(base + SN_KEY),
                      reinterpret_cast<int *>(base + SN_COUNT), start, reinterpret_cast<int *>(base + SN_CURSOR),
                      reinterpret_cast<int *>(base + SN_SIDX), reinterpret_cast<double *>(base + SN_SXYZ), stats, st,
                      nullptr), "cell sort");
  ChunkView C{};
  C.p0 = 0;
  C.n = (int)natoms;
  C.s_idx = reinterpret_cast<int *>(base + SN_SIDX);
  C.type_start = start + nkeys + 1;
  C.nl = reinterpret_cast<int *>(base + SN_NL);
  C.dr = reinterpret_cast<double4 *>(base + SN_DR);
  C.nreal = reinterpret_cast<int *>(base + SN_NREAL);
  C.nlp = nullptr;
  C.stats = stats;
  C.sub_nparts = 1;
  CU(launch_nlist(P, G, C, reinterpret_cast<double *>(base + SN_SXYZ), start, neighbour_cap(P), nlist, stats, st, 0,
                  nullptr), "nlist");
  if (status) {
    k_static_status<<<1, 1, 0, st>>>(stats, P.ntypes, reinterpret_cast<long long *>(status));
    DPB_LAUNCHED(1);
    CU(cudaGetLastError(), "status");
  }
  return DPB_OK;
}

extern "C" int dpb_eval_host(dpb_model *m, void *stream, int64_t natoms, const double *coord_h, const int32_t *type_h,
                             const double box[9], double *energy_h, double *atom_energy_h, double *force_h,
                             double *virial_h, int32_t *nlist_h, dpb_eval_info *info) {
  if (!m || !box) return fail(DPB_EINVAL, "dpb_eval_host: null model / box");
  if (natoms < 0) return fail(DPB_EINVAL, "natoms < 0");
  if (natoms > 0 && (!coord_h || !type_h)) return fail(DPB_EINVAL, "null coord / type");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const size_t n = (size_t)natoms;
  CU(m->h_coord.reserve(sizeof(double) * 3 * (n + 1)), "staging");
  CU(m->h_type.reserve(sizeof(int) * (n + 1)), "staging");
  // outputs: E[1] (padded to 2), virial[9] (padded to 10), E_i[N], F[N][3], then nlist
  const size_t out_d = 2 + 10 + n + 3 * n;
  const size_t nl_bytes = nlist_h ? sizeof(int) * n * (size_t)m->P.nm : 0;
  CU(m->h_out.reserve(sizeof(double) * out_d + nl_bytes + 16), "staging");
  double *d_e = m->h_out.as<double>(), *d_v = d_e + 2, *d_ei = d_v + 10, *d_f = d_ei + n;
  int *d_nl = nlist_h ? reinterpret_cast<int *>(d_f + 3 * n) : nullptr;
  if (natoms > 0) {
    CU(cudaMemcpyAsync(m->h_coord.p, coord_h, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, st), "H2D coord");
    CU(cudaMemcpyAsync(m->h_type.p, type_h, sizeof(int) * n, cudaMemcpyHostToDevice, st), "H2D type");
  }
  int rc = run_eval(m, st, natoms, m->h_coord.as<double>(), m->h_type.as<int>(), box, energy_h ? d_e : nullptr,
                    atom_energy_h ? d_ei : nullptr, force_h ? d_f : nullptr, virial_h ? d_v : nullptr, d_nl, false);
  if (rc != DPB_OK) return rc;
  if (energy_h) CU(cudaMemcpyAsync(energy_h, d_e, sizeof(double), cudaMemcpyDeviceToHost, st), "D2H energy");
  if (virial_h) CU(cudaMemcpyAsync(virial_h, d_v, sizeof(double) * 9, cudaMemcpyDeviceToHost, st), "D2H virial");
  if (atom_energy_h && natoms > 0)
    CU(cudaMemcpyAsync(atom_energy_h, d_ei, sizeof(double) * n, cudaMemcpyDeviceToHost, st), "D2H atom energy");
  if (force_h && natoms > 0)
    CU(cudaMemcpyAsync(force_h, d_f, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost, st), "D2H force");
  if (nlist_h && natoms > 0)
    CU(cudaMemcpyAsync(nlist_h, d_nl, nl_bytes, cudaMemcpyDeviceToHost, st), "D2H nlist");
  if (info) return finish_info(m, st, natoms, info);
  CU(cudaStreamSynchronize(st), "stream synchronise");
  return DPB_OK;
}

// ---------------------------------------------------------------------------------------------------------
// molecular dynamics.  Velocity-Verlet NVE; one force evaluation per step
// through run_eval; with rebuild_every > 1 the neighbour search runs on a skin list (cells and raw list over
// r_c + skin, rebuilt every rebuild_every steps; in between, Alg. 1 formats the raw list).  Everything is enqueued on
// the stream without host synchronisation until the thermo output is copied back at the end.
extern "C" int dpb_md_run(dpb_model *m, void *stream, int64_t natoms, double *coord, double *vel, const int32_t *type,
                          const double *mass_h, const double box[9], const dpb_md_params *prm, double *thermo_h,
                          dpb_md_info *info) {
  if (!m || !box || !prm || !mass_h) return fail(DPB_EINVAL, "dpb_md_run: null argument");
  if (natoms < 0 || (natoms > 0 && (!coord || !vel || !type))) return fail(DPB_EINVAL, "dpb_md_run: null coord / vel / type");
  if (!(prm->dt_fs > 0.0) || prm->nsteps < 0 || prm->thermo_every < 1 || prm->rebuild_every < 1 || !(prm->skin >= 0.0))
    return fail(DPB_EINVAL, "dpb_md_run: need dt > 0, nsteps >= 0, thermo_every >= 1, rebuild_every >= 1, skin >= 0");
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const DevModel &P = m->P;
  const bool reuse = prm->rebuild_every > 1;
  const size_t n = (size_t)natoms;
  const int nth = prm->nsteps / prm->thermo_every + 1;
  const double AMU = 103.6426965268;
  std::vector<double> hm(2 * DPB_MAX_TYPES, 0.0);              // [0..8): (dt/2)/(m AMU); [8..16): m AMU
  for (int t = 0; t < P.ntypes; ++t) {
    if (!(mass_h[t] > 0.0)) return fail(DPB_EINVAL, "dpb_md_run: mass[%d] must be positive", t);
    hm[t] = 0.5 * prm->dt_fs / (mass_h[t] * AMU);
    hm[DPB_MAX_TYPES + t] = mass_h[t] * AMU;
  }
  CU(m->md_force.reserve(sizeof(double) * 3 * (n + 1)), "md workspace");
  CU(m->md_scal.reserve(sizeof(double) * (12 + 4 * (size_t)nth)), "md workspace");
  CU(m->md_mass.reserve(sizeof(double) * 2 * DPB_MAX_TYPES), "md workspace");
  CU(cudaMemcpyAsync(m->md_mass.p, hm.data(), sizeof(double) * 2 * DPB_MAX_TYPES, cudaMemcpyHostToDevice, st), "H2D masses");
  if (reuse) {
    const double f = (P.rc + prm->skin) / P.rc;
    long long cap = (long long)(1.3 * f * f * f * P.nm) + 32;
    if (cap > 8192) cap = 8192;
    m->md_cap_raw = (int)cap;
    m->md_skin = prm->skin;
    CU(m->md_raw.reserve(sizeof(int) * (n + 1) * (size_t)cap), "md skin list");
    CU(m->md_nraw.reserve(sizeof(int) * (n + 1)), "md skin list");
    CU(m->md_xyz0.reserve(sizeof(double) * 3 * (n + 1)), "md skin list");
  }
  double *force = m->md_force.as<double>(), *epot = m->md_scal.as<double>(), *vir = epot + 2, *thermo = epot + 12;
  const double volume = box[0] * box[4] * box[8];
  const double *d_hm = m->md_mass.as<double>(), *d_mev = d_hm + DPB_MAX_TYPES;
  CU(cudaMemsetAsync(m->stats.p, 0, sizeof(DevStats), st), "memset stats");
  int rebuilds = 0;
  auto eval = [&](int step) -> int {
    int mode = 0;
    if (reuse) { mode = (step % prm->rebuild_every == 0) ? 1 : 2; rebuilds += mode == 1; }
    else CU(cudaMemsetAsync(m->stats.p, 0, sizeof(DevStats), st), "memset stats");
    return run_eval(m, st, natoms, coord, type, box, epot, nullptr, force, vir, nullptr, false, mode);
  };
  int rc = eval(0);
  if (rc != DPB_OK) return rc;
  int slot = 0;
  for (int step = 0;; ++step) {
    if (step % prm->thermo_every == 0) CU(launch_md_thermo(natoms, vel, type, d_mev, epot, vir, volume, thermo, slot++, st), "thermo");
    if (step == prm->nsteps) break;
    CU(launch_md_kick_drift(natoms, coord, vel, force, type, d_hm, prm->dt_fs, st), "kick + drift");
    rc = eval(step + 1);
    if (rc != DPB_OK) return rc;
    CU(launch_md_kick(natoms, vel, force, type, d_hm, st), "kick");
  }
  if (thermo_h) CU(cudaMemcpyAsync(thermo_h, thermo, sizeof(double) * 4 * (size_t)nth, cudaMemcpyDeviceToHost, st), "D2H thermo");
  DevStats hs;
  CU(cudaMemcpyAsync(&hs, m->stats.p, sizeof(DevStats), cudaMemcpyDeviceToHost, st), "stats copy");
  CU(cudaStreamSynchronize(st), "stream synchronise");
  if (hs.err_type) return fail(DPB_EINVAL, "an atom has a type index outside [0, ntypes)");
  if (hs.err_cap) return fail(DPB_ECAP, "an atom has more candidates than the staging / skin-list capacity");
  if (info) {
    memset(info, 0, sizeof(*info));
    info->n_thermo = nth;
    info->n_rebuilds = reuse ? rebuilds : prm->nsteps + 1;
    info->max_displacement = sqrt(hs.max_disp2);
    info->skin_violated = reuse && info->max_displacement > 0.5 * prm->skin;
  }
  return DPB_OK;
}
