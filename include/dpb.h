/* include/dpb.h — C ABI of libdpb.so: one Deep Potential (smooth edition, se_a) energy / force / virial
 * evaluation over a periodic box on one NVIDIA B200 (sm_100a).
 *
 * What is computed (arXiv 2004.11658, cited as PAPER.md:<line>; readings R1..R26 are listed in DESIGN.md):
 *   E = sum_i E_i,  E_i = N_{alpha_i}( D( R~_i ) )                                  Eq. 1
 *   neighbour list L~(i,:): type-sorted, distance-sorted, index-tie-broken, padded     Alg. 1
 *   environment matrix R~_i (Nm x 4), rows s(r)(1, x/r, y/r, z/r), zero when padded    Eq. 5 / Alg. 2, :98-105, :212-238
 *   embedding net G (1 -> s1 -> 2 s1 -> 4 s1 = M, tanh, concat skip)                   Eq. 6-9, :105-121
 *   descriptor D_i = (G^T R~)(R~^T G^<)  (M x M^<, row-major flatten b*M^< + a)        Eq. 4, :94-96
 *   fitting net (D -> w -> w -> w -> 1, tanh, identity skip on the square layers)       Eq. 2-3, :84-92
 *   F_i = -dE/dr_i by back-propagation, virial Xi = -sum_{i,k} d_ik (x) dE_i/dd_ik      Eq. 10, :125-135; ProdForce/ProdVirial :240
 *
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback.  All calls return 0 on success or a
 * negative dpb_status; on error the outputs are undefined and dpb_last_error() describes the failure.
 * Nothing here throws or aborts.  Units: Angstrom, eV, eV/Angstrom.  All matrices row-major.
 *
 * Concurrency: one host thread per process and GPU drives the library (the design is one process per GPU); calls are not
 * thread-safe.  Work is enqueued on the caller's stream; internally independent launches (the nets of a pass, the
 * species' fitting chains) are forked onto library-owned streams and joined by events before the call's last kernel, so
 * for the caller everything is ordered as if it ran on `stream` alone.
 */
#ifndef DPB_H
#define DPB_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dpb_model dpb_model;   /* opaque; owns device copies of the weights and a grow-only workspace */

typedef enum {
  DPB_FP64 = 0,   /* everything in fp64 (the paper's precision)                              */
  DPB_TF32 = 1,   /* mixed precision (BASELINE.json configs[3]): embedding and fitting GEMM operands in TF32 with
                     the error-compensated 3xTF32 split, fp32 accumulate (tcgen05 / TMEM), tanh in fp32; neighbour
                     list, env matrix, chain to the displacement and the T, F, virial, E accumulations in fp64.
                     Built for emb_s1 in {8, 16, 25, 32}, m_axis in {4, 8, 16}, fit_width % 4 == 0 and <= 256.   */
  DPB_BF16 = 2,   /* BASELINE.json configs[3] "and a BF16 variant": the FITTING-net GEMMs (Eq. 2-3 and their backward: the
                     K = 1600 / 240 contractions) with BF16 operands on tcgen05 kind::f16 — every operand split into three
                     BF16 pieces (8 + 8 + 8 significant bits), six piece products per product, fp32 accumulate; the
                     embedding-net GEMMs run as in DPB_TF32 (their tcgen05 kernels are written for 32-bit operand cells).
                     Meets the same tolerance as DPB_TF32 at the same tensor-pipe cost (6 K=16 MMAs against 3 K=8 MMAs).  */
  DPB_BF16_PLAIN = 3 /* as DPB_BF16 with ONE BF16 piece per operand (plain BF16 GEMMs in the fitting net): kept to MEASURE
                     what plain BF16 costs in accuracy on this model; it misses the mixed-precision tolerance by orders of
                     magnitude (tests record the error) and is not meant for production use.        */
} dpb_precision;

typedef enum {
  DPB_OK = 0,
  DPB_EINVAL = -1,   /* bad argument, shape or type index                                                  */
  DPB_EBOX = -2,     /* box not orthorhombic, or r_c >= min(L)/2 (reading R18: minimum image must be unique) */
  DPB_ENOMEM = -3,   /* device or host allocation failed                                                   */
  DPB_ECUDA = -4,    /* a CUDA runtime call or kernel launch failed                                        */
  DPB_ECAP = -5,     /* an atom has more in-range candidates than the neighbour staging capacity           */
  DPB_ENOTIMPL = -6  /* precision / model shape not supported by this build                                */
} dpb_status;

/* Model description.  All pointers are HOST pointers, read during dpb_model_create only (not retained). */
typedef struct {
  int32_t ntypes;             /* number of species (Remark 1)                                 */
  double rcut;                /* r_c                                                          */
  double rcut_smth;           /* r_cs: the gate w(r) of Eq. 5 is 1 below it (reading R1)                    */
  const int32_t *sel;         /* sel[ntypes]: padded slot count per neighbour type; Nm = sum */
  int32_t emb_s1;             /* embedding widths s1 -> 2 s1 -> 4 s1 = M (Eq. 8-9)        */
  int32_t m_axis;             /* M^<, 1 <= M^< <= M                                          */
  int32_t fit_width;          /* fitting hidden width (240)                                   */
  const double *emb_weights;  /* ntypes^2 nets; net (a = centre type, t = neighbour type) at a*ntypes + t:
                                 W0[1][s1] b0[s1] W1[s1][2s1] b1[2s1] W2[2s1][4s1] b2[4s1], [in][out]       */
  const double *fit_weights;  /* ntypes nets: W0[M*M^<][w] b0[w] W1[w][w] b1[w] W2[w][w] b2[w] w3[w] b3[1]   */
} dpb_model_desc;

/* Filled by dpb_eval when info != NULL (this makes the call synchronise the stream). */
typedef struct {
  int64_t n_real_pairs;       /* number of non-padded neighbour slots over all atoms                        */
  int64_t n_overflow;         /* neighbours dropped because a type section was full (reading R8)            */
  int32_t max_nei[8];         /* max over atoms of in-range neighbours of type t (before truncation), t < 8 */
  int32_t n_chunks;           /* atom chunks the evaluation was split into                                  */
  int32_t reserved;
} dpb_eval_info;

/* Create / destroy.  dpb_model_create copies (and re-lays-out) the weights to the current CUDA device.
 * Errors: DPB_EINVAL (shape, precision), DPB_ENOTIMPL (mixed precision with an unsupported shape), DPB_ENOMEM, DPB_ECUDA. */
int dpb_model_create(const dpb_model_desc *desc, int precision, dpb_model **out);
int dpb_model_destroy(dpb_model *model);

/* Nm = sum_t sel[t]. */
int dpb_model_nm(const dpb_model *model);

/* Upper bound on the atoms processed per pass (bounds the workspace: about 73 KB per atom for the copper model, plus the
 * activation records where they are stored: Nm * 1.6-1.8 KB per atom).
 * chunk_atoms = 0 (the default) sizes it automatically inside a budget of half of the device memory that was free when
 * the model was created: one chunk if workspace and activation records of all centres fit (W24k, Cu32k); otherwise equal
 * chunks of the largest size whose workspace and records fit, if that is at least 32768 atoms (the 864,000-atom copper
 * box: 10 chunks of 87,040, 88 GB in use, 326 ms); otherwise the largest chunk whose workspace alone fits, at least
 * 32768 atoms, and pass 2 recomputes.  Larger chunks are faster: the same-species pair reuse shares only pairs whose two
 * atoms are centres of the same chunk.  Returns DPB_EINVAL if chunk < 0. */
int dpb_model_set_chunk(dpb_model *model, int64_t chunk_atoms);

/* Select the kernel generation: 0 = plain reference kernels ("v0": unfused, thread-per-output FMA loops),
 * 1 = fused DMMA kernels (default), 2 = the paper's own embedding pipeline as a measured strawman (
 * PAPER.md:250-290): GEMMs over ALL padded slots of every (centre type, neighbour type) batch with the bias folded in,
 * the concat skip as a GEMM with (I, I) (Eq. 12), separate tanh / tanh-grad kernels, G and every activation materialised
 * in HBM (Eq. 13: about 4.8 KB per padded slot for the water model) and a reverse-mode backward; DPB_FP64 only, one host
 * synchronisation per evaluation (the batch sizes).  All compute the same path; tests compare each with the oracle. */
int dpb_model_set_variant(dpb_model *model, int variant);

/* Reproducibility.  In the default mode two evaluations of the same input differ at the 1e-16 relative level, in F and the
 * virial (fp64 atomics in the force scatter) AND in E and E_i: with the same-species pair reuse (on by default) and, for
 * small systems, with the row segments and the split-K first fitting layer, T (Eq. 4's G^T R~) and the first-layer
 * pre-activations are accumulated with fp64 reductions whose order varies from run to run.  The deterministic mode below
 * switches all of these off (fixed summation order everywhere): bitwise identical E, E_i, F and virial.
 *
 * Deterministic reduction (DPB_FP64, variant 1): forces and virial are summed in a fixed order instead of with fp64
 * atomics, so two evaluations of the same input agree bit for bit (the paper reports E / F / virial reproducible to
 * 15 / 10 / 13 digits; the default atomics mode differs at the 1e-16 relative level from run to run).
 * Costs about N * Nm * 28 bytes of extra workspace and one gather kernel.  Exact only when no neighbour was dropped
 * by a full type section (info.n_overflow == 0).  Other precisions / variants: dpb_eval returns DPB_ENOTIMPL.
 * dpb_eval_local and dpb_eval_cell take part: the formatted lists of the ghost atoms are built as well (list only; by
 * the same symmetry a ghost's list names the local atoms whose lists contain it), N above is then nall, and n_overflow
 * also counts neighbours dropped from a ghost's list.  dpb_eval_cell lays out and folds its images in a fixed order. */
int dpb_model_set_deterministic(dpb_model *model, int on);

/* CUDA-graph replay of dpb_eval (calls with info == NULL and the stage timers off).  The first call with a given set of
 * arguments (natoms, every pointer, the box) runs eagerly, the second one is captured into a CUDA graph, later ones
 * replay it — one launch instead of about 30, which is what bounds a 192-atom evaluation (the paper's regime below
 * ~1000 atoms per GPU).  The library keeps the 32 most recent argument sets; a change of the
 * workspace or of any model setting drops them.  The buffers named by the arguments must stay valid while the model may
 * replay them (as for any asynchronous call).  mode: 0 off, 1 (default) evaluations of at most 4096 atoms, 2 always.
 * dpb_eval_local, dpb_eval_host and dpb_md_run always run eagerly. */
int dpb_model_set_graph(dpb_model *model, int mode);

/* Same-species pair reuse (DPB_FP64, variant 1; on by default, off while the deterministic reduction is on).
 * The embedding net of a pair depends on s(r_ij) = s(r_ji) only (Eq. 5 and 8-9), so for the nets
 * G^{a,a} one evaluation serves both directions.  Pass 1: the atom with the lower sorted position adds g (x) R~_ik to its
 * own T_i (Eq. 4's G^T R~) and g (x) R~_ki to T_k with fp64 reductions.  Pass 2: one atom of the pair runs the value and
 * tangent chains and applies the backward epilogue with its own dE/dT tile and with the neighbour's (read from memory);
 * the pair force is f_ik - f_ki.  Only pairs whose two atoms are centres of the same chunk are shared; it is switched
 * off on the device for an evaluation in which a neighbour was dropped by a full type section (n_overflow > 0), because
 * the two lists are then not symmetric.  T is summed in a different (and, with the reductions, run-to-run varying)
 * order: results move at the 1e-15 relative level.  Other precisions ignore it.
 *   on = 0  off (both passes)
 *   on = 1  (default) pass 2 always; pass 1 in evaluations that run as a single chunk or in chunks of at least 32768
 *           centres (dpb_model_set_chunk): only the pairs inside a chunk can be shared, and with thin chunks pass 1's
 *           bookkeeping (clearing T, every accumulation a reduction) costs more than the sharing saves
 *   on = 2  both passes always (pairs across a chunk boundary are evaluated in both directions)
 * Returns DPB_EINVAL for any other value. */
int dpb_model_set_pair_reuse(dpb_model *model, int on);

/* Stored activations (DPB_FP64, variant 1; on by default).  Pass 2 differentiates the embedding net (Eq. 8-9,
 * PAPER.md:113-123) along the value chain of pass 1.  on = 1: pass 1 writes the tanh outputs of the three layers of every
 * row it evaluates (7 s1 fp64 numbers per pair, streamed: written once, read once) and pass 2 reads them instead of
 * running the value chain and its tanh again; the arithmetic that remains is the same, so results do not change beyond
 * the summation order of the pair reuse.  Taken per evaluation when the records of a chunk (chunk * Nm * 7 * s1 * 8
 * bytes, padded: 1,600 B per slot for s1 = 25) fit into the workspace budget (half of the memory that was free when the
 * model was created; the automatic chunk size is chosen so that they do, see dpb_model_set_chunk), the chunk has at least
 * 4096 centres, the pair reuse is on and the deterministic reduction is off; otherwise, and with on = 0, pass 2
 * recomputes (the paper's Eq. 13 tensors are then never written).  Returns DPB_EINVAL for any other value. */
int dpb_model_set_stored_activations(dpb_model *model, int on);

/* Species pipeline (DPB_FP64, variant 1, more than one species, chunks of at least 4096 centres; on by default).  Pass 1,
 * the fitting chain and pass 2 of centre type a touch only rows of type a — T_a, the fitting buffers of a, dE/dT_a; with
 * the pair reuse the neighbour's rows are of type a as well — so with on = 1 they run back to back on the stream of type
 * a, without the barriers between the stages, and the streams join after pass 2 (Eq. 1 sums over atoms: the
 * species are independent until then).  Same arithmetic, same results up to the order of the force reductions.  Switched
 * off while the stage timers or the debug buffers are on.  on = 0: the three stages are separated by joins (what the
 * stage times of bench.py describe).  Returns DPB_EINVAL for any other value. */
int dpb_model_set_species_pipeline(dpb_model *model, int on);

/* Per-atom virial.  The paper gives no per-atom split (the virial is only named through the
 * ProdVirial operator); this library assigns every term to its centre atom:
 *     atom_virial[i][a][b] = -sum_k d_ik[a] (dE_i/dd_ik)[b],     sum_i atom_virial[i] = virial of dpb_eval.
 * atom_virial: DEVICE fp64 [N][9] that the following dpb_eval calls fill (indexed by the input atom order), or NULL to
 * switch the output off.  The caller owns the buffer and keeps it alive.  Produced by the gather of the deterministic
 * reduction: dpb_eval returns DPB_ENOTIMPL while a buffer is set and dpb_model_set_deterministic is off.
 * dpb_eval_local fills the rows of the nloc local atoms only ([nloc][9]; the terms of an atom's own neighbourhood, ghost
 * neighbours included), dpb_eval_cell the rows of the N atoms of the cell. */
int dpb_model_set_atom_virial(dpb_model *model, double *atom_virial);

/* One evaluation (the paper's problem statement: coordinates, types and box in; E, E_i, F_i and the virial out).
 *   stream       cudaStream_t (as void*) on which all work is enqueued; NULL = the legacy default stream
 *   natoms       N >= 0
 *   coord        DEVICE fp64 [N][3], raw (unwrapped is allowed) Cartesian positions
 *   type         DEVICE int32 [N], 0 <= type < ntypes, any order
 *   box          HOST fp64 [9], rows = cell vectors; must be orthorhombic with r_c < min(L)/2 (DPB_EBOX otherwise)
 *   energy       DEVICE fp64 [1]            E                      (may be NULL)
 *   atom_energy  DEVICE fp64 [N]            E_i                    (may be NULL)
 *   force        DEVICE fp64 [N][3]         F_i = -dE/dr_i         (may be NULL)
 *   virial       DEVICE fp64 [9]            Xi[a][b] = -sum_i sum_k d_ik[a] dE_i/dd_ik[b]  (may be NULL)
 *   nlist        DEVICE int32 [N][Nm]       formatted neighbour list, -1 padded  (may be NULL)
 *   info         HOST, may be NULL; non-NULL synchronises the stream before returning
 * The caller owns every buffer; the library neither frees nor retains them.  Work is asynchronous with
 * respect to the host unless info != NULL.  Neighbour overflow is not an error: the nearest sel[t] are kept. */
int dpb_eval(dpb_model *model, void *stream, int64_t natoms, const double *coord, const int32_t *type,
             const double box[9], double *energy, double *atom_energy, double *force, double *virial,
             int32_t *nlist, dpb_eval_info *info);

/* Deferred input errors.  Three conditions are detected on the device and therefore only reported by a call that
 * synchronises (dpb_eval / dpb_eval_local / dpb_eval_host with info != NULL, dpb_build_nlist with n_overflow != NULL,
 * dpb_md_run) — with info == NULL the call returns DPB_OK and its outputs are undefined:
 *   DPB_EINVAL  an atom's type index lies outside [0, ntypes) (it is evaluated as type 0)
 *   DPB_ECAP    an atom has more in-range candidates than the staging capacity max(256, 2 Nm) (its row is written empty)
 *   DPB_EBOX    dpb_eval_local: an atom lies outside `bounds`
 * dpb_model_status synchronises `stream` and returns the status of the LAST evaluation enqueued for this model
 * (DPB_OK, or one of the three above with dpb_last_error set), for callers that run with info == NULL. */
int dpb_model_status(dpb_model *model, void *stream);

/* Same call with HOST buffers for coord/type and for every output (end-to-end entry: host->device copies of the
 * inputs, the evaluation, and device->host copies of the requested outputs, all on `stream`, then a stream
 * synchronise).  Pinned host memory makes the copies asynchronous, pageable memory is accepted. */
int dpb_eval_host(dpb_model *model, void *stream, int64_t natoms, const double *coord_h, const int32_t *type_h,
                  const double box[9], double *energy_h, double *atom_energy_h, double *force_h, double *virial_h,
                  int32_t *nlist_h, dpb_eval_info *info);

/* One sub-region with explicit ghost atoms (a sub-region owns
 * its local atoms, the atoms of neighbouring sub-regions and the periodic images within r_c of it are present as
 * ghosts; the ghost forces go home in the reverse exchange).  There is no box and no minimum image: displacements are
 * plain differences, so r_c >= L/2 is handled by supplying the images as ghosts.
 *   nloc, nall   atoms [0, nloc) are local, [nloc, nall) ghosts (nall >= nloc >= 0)
 *   coord, type  DEVICE, [nall][3] / [nall]
 *   bounds       HOST fp64 [6]: lo[3], hi[3] of a region that contains every one of the nall atoms (e.g. the brick
 *                widened by r_c); an atom outside it is DPB_EBOX, reported when info != NULL
 *   energy       DEVICE fp64 [1]       sum of E_i over the LOCAL atoms
 *   atom_energy  DEVICE fp64 [nloc]
 *   force        DEVICE fp64 [nall][3] -dE/dr of that energy, on local and ghost atoms
 *   virial       DEVICE fp64 [9]       the local atoms' part, -sum_{i<nloc} sum_k d_ik (x) dE_i/dd_ik
 *   nlist        DEVICE int32 [nloc][Nm], indices into [0, nall)
 * Summed over the sub-regions of a periodic system (ghost forces added to their owners) the outputs equal dpb_eval's.
 * Ownership, asynchrony and info as for dpb_eval. */
int dpb_eval_local(dpb_model *model, void *stream, int64_t nloc, int64_t nall, const double *coord,
                   const int32_t *type, const double bounds[6], double *energy, double *atom_energy, double *force,
                   double *virial, int32_t *nlist, dpb_eval_info *info);

/* General periodic cell: triclinic cells and cells thinner than 2 r_c, which dpb_eval refuses.
 * Evaluated the way the paper formulates periodicity: the atoms, wrapped into the cell, are the local
 * atoms; every lattice image whose fractional coordinate lies within r_c / h_c of the cell (h_c = perpendicular height
 * along lattice vector c; ceil(r_c / h_c) image shells) is a ghost; dpb_eval_local's kernels do the arithmetic; the
 * ghost force increments are added to the atoms they are images of.  Image construction and fold-back are kernels of
 * this library (csrc/cell.cu).
 *   cell         HOST fp64 [9], rows = lattice vectors (any non-singular cell; DPB_EBOX if singular or thinner than r_c/16)
 *   coord, type  DEVICE, [N][3] / [N]; raw positions (wrapped internally)
 *   energy [1], atom_energy [N], force [N][3], virial [9]: DEVICE, as dpb_eval (any may be NULL)
 *   info         HOST or NULL; n_real_pairs etc. refer to the N atoms of the cell
 * One host synchronisation (the number of images sizes the evaluation), otherwise asynchronous on `stream`.  An atom's
 * images take consecutive rows in shift order and are folded back in that order, so the result does not depend on the
 * scheduling (bitwise reproducible together with dpb_model_set_deterministic). */
int dpb_eval_cell(dpb_model *model, void *stream, int64_t natoms, const double *coord, const int32_t *type,
                  const double cell[9], double *energy, double *atom_energy, double *force, double *virial,
                  dpb_eval_info *info);

/* Velocity-Verlet pieces for a driver that owns the time loop — the decomposition's MD driver in
 * paper_2004_11658_b200/dd.py, where an evaluation is ghost exchange + dpb_eval_local + reverse exchange.
 * dpb_md_coefficients (HOST -> HOST): coeff_h[t] = (dt/2) / (m_t u) and coeff_h[ntypes + t] = m_t u with
 *   u = 103.6426965268 eV fs^2 / (amu A^2); the caller copies the 2 ntypes doubles to the device.
 * dpb_md_kick_drift: v <- v + coeff[type] F;  x <- x + dt v     (n atoms; all pointers DEVICE, coeff = first half)
 * dpb_md_kick:       v <- v + coeff[type] F
 * dpb_md_kinetic_energy: ekin[0] = sum_i 1/2 mass_ev[type_i] v_i^2 in eV (mass_ev = second half of the coefficients),
 *   fixed summation order; the sum over sub-regions is the caller's all-reduce.
 * Asynchronous on `stream`; the caller owns every buffer. */
int dpb_md_coefficients(const double *mass_h, int32_t ntypes, double dt_fs, double *coeff_h);
int dpb_md_kick_drift(void *stream, int64_t n, double *coord, double *vel, const double *force, const int32_t *type,
                      const double *coeff, double dt_fs);
int dpb_md_kick(void *stream, int64_t n, double *vel, const double *force, const int32_t *type, const double *coeff);
int dpb_md_kinetic_energy(void *stream, int64_t n, const double *vel, const int32_t *type, const double *mass_ev,
                          double *ekin);

/* Ghost exchange of the domain decomposition (the driver is paper_2004_11658_b200/dd.py).  All
 * pointers DEVICE, all work asynchronous on `stream`; messages are rows of four fp64 (x, y, z, type).
 * dpb_dd_pack: one stage of the forward exchange along dimension dim (0, 1, 2).  Atoms with coord[dim] < cut_minus go to
 *   pack_minus (coord[dim] += shift_minus), atoms with coord[dim] >= cut_plus to pack_plus (+= shift_plus); an atom may
 *   go both ways.  idx_* [cap] receives the atom index of each row (for the reverse exchange), counts[2] = rows wanted
 *   for (minus, plus); rows beyond cap are counted but not written, so counts[d] > cap means: grow and call again.
 *   Row order inside a message is arbitrary.
 * dpb_dd_unpack: k received rows -> coord_out [k][3], type_out [k] (the tail of the atom arrays).
 * dpb_dd_add_forces: reverse exchange, force[idx[i]][:] += fin[i][:] for i < k; idx must not repeat within one call. */
int dpb_dd_pack(void *stream, int64_t n, const double *coord, const int32_t *type, int32_t dim, double cut_minus,
                double cut_plus, double shift_minus, double shift_plus, int64_t cap, double *pack_minus,
                int32_t *idx_minus, double *pack_plus, int32_t *idx_plus, int32_t *counts);
int dpb_dd_unpack(void *stream, int64_t k, const double *pack, double *coord_out, int32_t *type_out);
int dpb_dd_add_forces(void *stream, int64_t k, const int32_t *idx, const double *fin, double *force);

/* Alg. 1 only (cell binning + neighbour search + format): nlist DEVICE int32 [N][Nm].  n_overflow HOST, may be
 * NULL (non-NULL synchronises). */
int dpb_build_nlist(dpb_model *model, void *stream, int64_t natoms, const double *coord, const int32_t *type,
                    const double box[9], int32_t *nlist, int64_t *n_overflow);

/* dpb_build_nlist without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  Same kernels, same result (Alg. 1: cell binning,
 * neighbour search, sort by (type, distance, index), -1 padding); the scratch of the kernels lives in one file-scope
 * device array of 9.9 MB that every GPU which loads this library holds until the process exits, instead of in the
 * model's workspace.  The call performs no cudaMalloc / cudaFree and calls no allocating library routine; it does not
 * touch the model's workspace (the model only supplies r_c, sel and the number of types).
 *   Limits: natoms <= 4096, natoms * Nm <= 262144, ntypes * (cells of the search grid) <= 16384.  Beyond any of them:
 *           DPB_EINVAL with a message naming the limit; nothing is launched.  dpb_build_nlist has no such limits.
 *   coord, type  DEVICE fp64 [N][3] / int32 [N];  box HOST fp64 [9] as for dpb_eval (DPB_EBOX otherwise)
 *   nlist        DEVICE int32 [N][Nm], caller-owned output
 *   status       DEVICE int64 [4], caller-owned, may be NULL: real pairs, neighbours dropped by a full type section,
 *                error bits (1: a type index outside [0, ntypes), 2: an atom has more in-range candidates than the
 *                staging capacity — its row is then written empty), largest candidate count of any (atom, type).
 *                The call never synchronises: the deferred input errors are reported here, not by the return code.
 * Every call on a device shares the one array, which keeps the previous call's contents (what must start at zero is
 * cleared on `stream` first): calls that overlap on the GPU — different streams, different models, different host
 * threads — race.  Serialise them (one stream, or events).  The first call on a device looks up the array's device
 * address (cudaGetSymbolAddress) and sets the kernels' shared-memory limit: make that call outside graph capture. */
int dpb_build_nlist_static(const dpb_model *model, void *stream, int64_t natoms, const double *coord,
                           const int32_t *type, const double box[9], int32_t *nlist, int64_t *status);

/* Test / profiling hook, not part of the contract: DEVICE buffers (any may be NULL) that the following
 * dpb_eval calls also fill, indexed by the ORIGINAL atom index:
 *   T  [N][M][4]   = G^T R~                    (Eq. 4, left factor)
 *   D  [N][M*M^<]  = descriptor                (only written by variant 0)
 *   dT [N][M][4]   = dE_i/dT_i
 * Pass all NULL to switch it off. */
int dpb_set_debug_buffers(dpb_model *model, double *T, double *D, double *dT);

/* Test hook, not part of the contract: order DEVICE int32 [natoms] receives, for every sorted position p of the LAST
 * evaluation of this model (atoms are processed in the order (ghost?, type, cell); chunk c covers the positions
 * [c * chunk_atoms, (c + 1) * chunk_atoms)), the input index of the atom at p.  Lets a test pick atoms on both sides of
 * a chunk boundary.  Asynchronous on `stream`; DPB_EINVAL before the first evaluation or if natoms differs from it. */
int dpb_debug_sorted_order(dpb_model *model, void *stream, int64_t natoms, int32_t *order);

/* Per-stage device time of the last dpb_eval issued after dpb_model_set_timing(model, 1), in microseconds (CUDA
 * events recorded on the caller's stream between the stages; the caller must have synchronised that stream):
 * [0] cell binning, [1] neighbour search + format, [2] env + embedding + T, [3] descriptor + fitting fwd/bwd + dT,
 * [4] embedding backward + force/virial, [5] energy reduction; summed over chunks.  DPB_ECUDA if not complete. */
int dpb_model_set_timing(dpb_model *model, int on);
int dpb_model_stage_us(const dpb_model *model, float stage_us[8]);

/* ---- molecular dynamics with the DP forces ---------------------------------
 * Velocity-Verlet, NVE: v += (dt/2) F/m; x += dt v; F = F(x); v += (dt/2) F/m.  Units: Angstrom, fs, amu, eV
 * (1 amu A^2/fs^2 = 103.6426965268 eV; T = 2 E_kin / (3 N k_B), k_B = 8.617333262e-5 eV/K; pressure from the virial
 * theorem, P = (2 E_kin + tr Xi) / (3 V), 1 eV/A^3 = 1.602176634e6 bar — the thermo quantities of PAPER.md:298).
 * Neighbour reuse (2 A skin, rebuilt every 50 steps): with rebuild_every > 1 the cell search runs
 * over r_c + skin every rebuild_every steps and stores a raw list; the steps in between format that raw list (Alg. 1).
 * The formatted list equals a fresh search as long as no atom moves more than skin / 2 between rebuilds
 * (reported in dpb_md_info, not enforced).  rebuild_every == 1: fresh cell search every step, skin unused. */
typedef struct {
  double dt_fs;              /* time step                                                                  */
  int32_t nsteps;            /* number of steps (>= 0)                                                     */
  int32_t thermo_every;      /* thermo rows at steps 0, thermo_every, 2 thermo_every, ... (>= 1)           */
  int32_t rebuild_every;     /* >= 1                                                                       */
  int32_t reserved;
  double skin;               /* Angstrom; needs r_c + skin < min(L) / 2 when rebuild_every > 1             */
} dpb_md_params;

typedef struct {
  int32_t n_thermo;          /* rows written to thermo                                                     */
  int32_t n_rebuilds;        /* neighbour searches from the cell list                                      */
  int32_t skin_violated;     /* 1 if some atom moved more than skin / 2 between two rebuilds               */
  int32_t reserved;
  double max_displacement;   /* largest displacement of an atom since the rebuild before it (Angstrom)     */
} dpb_md_info;

/* coord DEVICE fp64 [N][3] and vel DEVICE fp64 [N][3] (A/fs) are updated in place; type DEVICE int32 [N]; mass HOST
 * [ntypes] (amu); box HOST [9]; thermo HOST [nsteps / thermo_every + 1][4] = (E_pot [eV], E_kin [eV], T [K], P [bar]) or NULL; info HOST or
 * NULL.  All work is enqueued on `stream`; the call returns after the stream has been synchronised.  The model must
 * not be used by another call while the run is in flight.  Errors as dpb_eval. */
int dpb_md_run(dpb_model *model, void *stream, int64_t natoms, double *coord, double *vel, const int32_t *type,
               const double *mass, const double box[9], const dpb_md_params *params, double *thermo,
               dpb_md_info *info);

/* Thread-local description of the last error returned on this thread; valid until the next call. */
const char *dpb_last_error(void);

/* Number of CUDA kernels this library has launched in this process so far (all models, all calls). */
int64_t dpb_kernel_launches(void);

/* Version string of the library ("dpb <n> sm_100a"). */
const char *dpb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DPB_H */
