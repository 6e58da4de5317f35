/* oracle/dpo.h — TEST INFRASTRUCTURE, NOT PART OF THE PRODUCT.
 *
 * Plain, slow, fp64 CPU implementation of one Deep Potential (smooth edition, se_a) energy / force / virial
 * evaluation, written from the equations of arXiv 2004.11658 (cited below as PAPER.md:<line>) and the readings
 * listed in DESIGN.md ("Readings of the paper").  It exists to check the CUDA library (libdpb.so) and to be
 * timed as the CPU baseline.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load it.  It shares no code with paper_2004_11658_b200/csrc (no headers, no helpers, no
 * tables); the CUDA path never calls it.
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py (brute force, closed forms,
 * finite differences, invariances, an independent PyTorch-autograd model).  What is NOT pinned, and cannot
 * be: the absolute energies / forces of the paper's trained water and copper models (weights and
 * configurations are not available) — "parity unpinned" for the paper's physical outputs only.
 *
 * All pointers are HOST pointers.  Matrices are row-major.  Units: Angstrom, eV.
 */
#ifndef DPO_H
#define DPO_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Model description: same field meaning as dpb_model_desc in include/dpb.h (declared independently). */
typedef struct {
  int32_t ntypes;            /* number of species                                                         */
  double rcut;               /* r_c                                                          */
  double rcut_smth;          /* r_cs: w(r) = 1 below it (reading R1)                            */
  const int32_t *sel;        /* sel[ntypes]: padded slot count per neighbour type           */
  int32_t emb_s1;            /* embedding widths s1 -> 2 s1 -> 4 s1 = M                 */
  int32_t m_axis;            /* M^<                                                         */
  int32_t fit_width;         /* fitting hidden width (240)                                  */
  const double *emb_weights; /* ntypes^2 nets, net (a,t) at a*ntypes+t: W0[1][s1] b0[s1] W1[s1][2s1]
                                b1[2s1] W2[2s1][4s1] b2[4s1], row-major [in][out]                         */
  const double *fit_weights; /* ntypes nets: W0[M*M^<][w] b0[w] W1[w][w] b1[w] W2[w][w] b2[w] w3[w] b3[1] */
} dpo_model_desc;

enum { DPO_OK = 0, DPO_EINVAL = -1, DPO_EBOX = -2, DPO_ENOMEM = -3 };

int dpo_nm(const dpo_model_desc *m);                       /* Nm = sum_t sel[t]                          */

/* w(r) and dw/dr — gating function of Eq. 5, reading R1. */
void dpo_switch(double r, double rcs, double rc, double *w, double *dw);

/* Minimum-image displacement d = r_j - r_i and |d| with the pinned IEEE operation sequence (reading R2). */
void dpo_displacement(const double ri[3], const double rj[3], const double L[3], double d[3], double *r);

/* Brute-force O(N) per row neighbour search + Alg. 1 formatting for the atoms listed in
 * rows[0..nrows) (rows == NULL: atoms 0..nrows-1).  nlist_out is [nrows][Nm] int32, padded with -1.
 * n_overflow (may be NULL) counts neighbours dropped because a type section was full (reading R8). */
int dpo_build_nlist_rows(const dpo_model_desc *m, int64_t natoms, const double *coord, const int32_t *type,
                         const double box[9], int64_t nrows, const int64_t *rows, int32_t *nlist_out,
                         int64_t *n_overflow);

/* Same result from the oracle's own cell list (all atoms); validated against the brute force in tests. */
int dpo_build_nlist_cells(const dpo_model_desc *m, int64_t natoms, const double *coord, const int32_t *type,
                          const double box[9], int32_t *nlist_out, int64_t *n_overflow);

/* Environment matrix (Alg. 2; Eq. 5) for one atom: env[Nm][4], and its derivative with
 * respect to the displacement d_ik: denv[Nm][4][3]; disp[Nm][3] (any output may be NULL). */
int dpo_env_row(const dpo_model_desc *m, int64_t natoms, const double *coord, const double box[9], int64_t i,
                const int32_t *nlist_row, double *env, double *denv, double *disp);

/* Embedding net forward (Eq. 7-9): g[4 s1] = G(x) for one net (pointer to its W0). */
void dpo_embed(const double *net, int32_t s1, double x, double *g);

/* Fitting net forward (Eq. 2-3, reading R4): returns E_i for descriptor D[dim]. */
double dpo_fit(const double *net, int32_t dim, int32_t width, const double *D);

/* Per-atom evaluation for the listed rows, given their formatted nlist rows [nrows][Nm]:
 *   atom_energy[nrows]; fslot[nrows][Nm][3] = dE_i/d d_ik (zero on padded slots);
 *   optional T_out[nrows][M][4], D_out[nrows][M*M^<], dT_out[nrows][M][4] (NULL to skip). */
int dpo_atom_rows(const dpo_model_desc *m, int64_t natoms, const double *coord, const int32_t *type,
                  const double box[9], int64_t nrows, const int64_t *rows, const int32_t *nlist_rows,
                  double *atom_energy, double *fslot, double *T_out, double *D_out, double *dT_out);

/* One full evaluation (PAPER.md:80 Eq. 1, :125 Eq. 10, :240 ProdForce/ProdVirial): energy[1], atom_energy[N],
 * force[N][3], virial[9]; nlist_out [N][Nm] or NULL.  use_cells != 0 selects the cell-list search. */
int dpo_eval(const dpo_model_desc *m, int64_t natoms, const double *coord, const int32_t *type,
             const double box[9], double *energy, double *atom_energy, double *force, double *virial,
             int32_t *nlist_out, int use_cells);

/* NEXT #3: per-atom virial, centre-atom split of reading R14: atom_virial[i][a][b] =
 * -sum_k d_ik[a] (dE_i/dd_ik)[b]; sums to the virial of dpo_eval.  atom_virial is [N][9]. */
int dpo_atom_virial(const dpo_model_desc *m, int64_t natoms, const double *coord, const int32_t *type,
                    const double box[9], double *atom_virial);

/* NEXT #2 / #3: one sub-region with explicit ghost atoms, no box.  Atoms
 * 0..nloc-1 are local, nloc..nall-1 ghosts; energy[1] and atom_energy[nloc] cover the local atoms, force[nall][3] is
 * -dE/dr of that energy on local and ghost atoms, virial[9] the local atoms' part; nlist_out [nloc][Nm] or NULL. */
int dpo_eval_local(const dpo_model_desc *m, int64_t nloc, int64_t nall, const double *coord, const int32_t *type,
                   double *energy, double *atom_energy, double *force, double *virial, int32_t *nlist_out);

/* NEXT #1: velocity-Verlet NVE molecular dynamics with the DP forces.
 * coord [N][3] (A) and vel [N][3] (A/fs) are updated in place; mass[ntypes] in amu; thermo [nsteps / thermo_every + 1][4]
 * = (E_pot [eV], E_kin [eV], T [K], P [bar]) at steps 0, thermo_every, ... (may be NULL).  Neighbours are searched from scratch every step. */
int dpo_md_run(const dpo_model_desc *m, int64_t natoms, double *coord, double *vel, const int32_t *type,
               const double *mass, const double box[9], double dt_fs, int64_t nsteps, int64_t thermo_every,
               double *thermo, int use_cells);

int dpo_num_threads(void);                                  /* OpenMP threads the loops over atoms use     */

#ifdef __cplusplus
}
#endif
#endif
