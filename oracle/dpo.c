/* oracle/dpo.c — TEST INFRASTRUCTURE, NOT PART OF THE PRODUCT (see oracle/dpo.h).
 *
 * Plain fp64 C restatement of the Deep Potential se_a definitions of arXiv 2004.11658.  Straightforward loops,
 * libm tanh/sqrt, no blocking, no fusion, no reordering beyond what the equations state.  Steps O1..O11 are
 * the ones listed in SURVEY.md §8(c) / DESIGN.md "Oracle"; each function cites the passage it follows.
 * Compile with -O2 -ffp-contract=off (so that only the explicit fma() calls of reading R2 are fused).
 * OpenMP is used only as "for each atom i" (Alg. 1 line 1 / Alg. 2 line 1); every reduction that
 * crosses atoms (E, F, virial) is done serially in atom / slot order, so results do not depend on threads.
 */
#include "dpo.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int dpo_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

int dpo_nm(const dpo_model_desc *m) {
  int nm = 0;
  for (int t = 0; t < m->ntypes; ++t) nm += m->sel[t];
  return nm;
}

static int64_t emb_net_size(int s1) {
  return (int64_t)s1 + s1 + (int64_t)s1 * 2 * s1 + 2 * s1 + (int64_t)2 * s1 * 4 * s1 + 4 * s1;
}
static int64_t fit_net_size(int dim, int w) {
  return (int64_t)dim * w + w + 2 * ((int64_t)w * w + w) + w + 1;
}

/* O1: argument checks.  Orthorhombic box (rows = cell vectors), r_c < min(L)/2 so that the minimum image is
 * unique and j identifies the pair (reading R18: one periodic box replaces the paper's ghost atoms,
 * PAPER.md:145-147). */
static int check_inputs(const dpo_model_desc *m, const double box[9], double L[3]) {
  if (!m || m->ntypes < 1 || !m->sel || m->emb_s1 < 1 || m->m_axis < 1 || m->m_axis > 4 * m->emb_s1 ||
      m->fit_width < 1)
    return DPO_EINVAL;
  if (!(m->rcut > 0.0) || !(m->rcut_smth >= 0.0) || !(m->rcut_smth < m->rcut)) return DPO_EINVAL;
  for (int t = 0; t < m->ntypes; ++t)
    if (m->sel[t] < 0) return DPO_EINVAL;
  if (box[1] != 0.0 || box[2] != 0.0 || box[3] != 0.0 || box[5] != 0.0 || box[6] != 0.0 || box[7] != 0.0)
    return DPO_EBOX;
  L[0] = box[0]; L[1] = box[4]; L[2] = box[8];
  for (int c = 0; c < 3; ++c)
    if (!(L[c] > 0.0) || !(m->rcut < 0.5 * L[c])) return DPO_EBOX;
  return DPO_OK;
}

/* O5 (reading R1): the gating function w of Eq. 5 ("decays smoothly from 1 to 0 at r_c").
 * u = (r - rcs)/(rc - rcs);  w = 1 (r < rcs);  u^3(-6u^2 + 15u - 10) + 1 (rcs <= r < rc);  0 (r >= rc).
 * dw/dr = -30 u^2 (u-1)^2 / (rc - rcs). */
void dpo_switch(double r, double rcs, double rc, double *w, double *dw) {
  if (r < rcs) {
    *w = 1.0; *dw = 0.0;
  } else if (r < rc) {
    double u = (r - rcs) / (rc - rcs);
    *w = u * u * u * (-6.0 * u * u + 15.0 * u - 10.0) + 1.0;
    *dw = -30.0 * u * u * (u - 1.0) * (u - 1.0) / (rc - rcs);
  } else {
    *w = 0.0; *dw = 0.0;
  }
}

/* O2 (reading R2): r_ij = r_j - r_i (PAPER.md:80; Alg. 1 line 3-4, :177) under the minimum-image convention,
 * with ONE pinned sequence of IEEE-754 operations on the raw input coordinates so that the neighbour list can
 * be compared bit for bit:  d = x_j - x_i;  k = rint(d / L);  d = fma(-k, L, d);
 * r2 = fma(dz,dz, fma(dy,dy, dx*dx));  r = sqrt(r2). */
void dpo_displacement(const double ri[3], const double rj[3], const double L[3], double d[3], double *r) {
  for (int c = 0; c < 3; ++c) {
    double dc = rj[c] - ri[c];
    double k = rint(dc / L[c]);
    d[c] = fma(-k, L[c], dc);
  }
  double r2 = fma(d[2], d[2], fma(d[1], d[1], d[0] * d[0]));
  *r = sqrt(r2);
}

/* S(i,k) = (alpha_j, |r_ij|, j) of Alg. 1 line 4. */
typedef struct { int32_t type; double r; int32_t j; } cand_t;

/* Alg. 1 line 7 (Fig. 2(a) :159; :165, :193): sort by type, then distance, then atom index. */
static int cand_cmp(const void *pa, const void *pb) {
  const cand_t *a = (const cand_t *)pa, *b = (const cand_t *)pb;
  if (a->type != b->type) return a->type < b->type ? -1 : 1;
  if (a->r != b->r) return a->r < b->r ? -1 : 1;
  if (a->j != b->j) return a->j < b->j ? -1 : 1;
  return 0;
}

/* O4: Alg. 1 lines 7-9 (sort, pad, keep j).  Section t occupies slots [sum_{t'<t} sel[t'], +sel[t]); the
 * first sel[t] neighbours of type t are written, the rest of the section is -1.  Neighbours
 * beyond sel[t] are dropped and counted (reading R8). */
static int64_t format_row(const dpo_model_desc *m, cand_t *cand, int64_t ncand, int32_t *row) {
  int nm = dpo_nm(m);
  int64_t dropped = 0;
  qsort(cand, (size_t)ncand, sizeof(cand_t), cand_cmp);
  for (int k = 0; k < nm; ++k) row[k] = -1;
  int64_t c = 0;
  int start = 0;
  for (int t = 0; t < m->ntypes; ++t) {
    int filled = 0;
    while (c < ncand && cand[c].type == t) {
      if (filled < m->sel[t]) row[start + filled++] = cand[c].j;
      else ++dropped;
      ++c;
    }
    start += m->sel[t];
  }
  return dropped;
}

/* O3 + O4: L(i) = { j != i : |r_ij| <= r_c } ("<=" as printed, reading R9/R19) by brute force
 * over all atoms, then Alg. 1. */
int dpo_build_nlist_rows(const dpo_model_desc *m, int64_t natoms, const double *coord, const int32_t *type,
                         const double box[9], int64_t nrows, const int64_t *rows, int32_t *nlist_out,
                         int64_t *n_overflow) {
  double L[3];
  int rc = check_inputs(m, box, L);
  if (rc != DPO_OK) return rc;
  for (int64_t i = 0; i < natoms; ++i)
    if (type[i] < 0 || type[i] >= m->ntypes) return DPO_EINVAL;
  int nm = dpo_nm(m);
  int64_t dropped_total = 0;
  int err = 0;
#pragma omp parallel
  {
    int64_t cap = 1024, dropped = 0;
    cand_t *cand = (cand_t *)malloc((size_t)cap * sizeof(cand_t));
    if (!cand) {
#pragma omp atomic write
      err = 1;
    }
#pragma omp for schedule(dynamic, 16)
    for (int64_t q = 0; q < nrows; ++q) {
      if (err) continue;
      int64_t i = rows ? rows[q] : q;
      int64_t nc = 0;
      for (int64_t j = 0; j < natoms; ++j) {
        if (j == i) continue;
        double d[3], r;
        dpo_displacement(coord + 3 * i, coord + 3 * j, L, d, &r);
        if (r <= m->rcut) {
          if (nc == cap) {
            cap *= 2;
            cand_t *nw = (cand_t *)realloc(cand, (size_t)cap * sizeof(cand_t));
            if (!nw) {
#pragma omp atomic write
              err = 1;
              break;
            }
            cand = nw;
          }
          cand[nc].type = type[j]; cand[nc].r = r; cand[nc].j = (int32_t)j;
          ++nc;
        }
      }
      if (!err) dropped += format_row(m, cand, nc, nlist_out + q * nm);
    }
#pragma omp atomic
    dropped_total += dropped;
    free(cand);
  }
  if (err) return DPO_ENOMEM;
  if (n_overflow) *n_overflow = dropped_total;
  return DPO_OK;
}

/* The same L(i) from a cell list (used only where the brute force is too slow, N >= 1e5).  Cells have an edge
 * >= r_c(1 + 1e-6); atoms are binned by their wrapped fractional coordinate; candidates come from the 27
 * surrounding cells (each distinct cell once when a dimension has fewer than 3 cells); distances use
 * dpo_displacement on the RAW coordinates, so the result is bit-identical to the brute force
 * (tests/test_oracle_nlist.py checks exactly that). */
int dpo_build_nlist_cells(const dpo_model_desc *m, int64_t natoms, const double *coord, const int32_t *type,
                          const double box[9], int32_t *nlist_out, int64_t *n_overflow) {
  double L[3];
  int rc = check_inputs(m, box, L);
  if (rc != DPO_OK) return rc;
  for (int64_t i = 0; i < natoms; ++i)
    if (type[i] < 0 || type[i] >= m->ntypes) return DPO_EINVAL;
  int nm = dpo_nm(m);
  int nc[3];
  for (int c = 0; c < 3; ++c) {
    nc[c] = (int)floor(L[c] / (m->rcut * (1.0 + 1e-6)));
    if (nc[c] < 1) nc[c] = 1;
  }
  int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
  int64_t *cell_of = (int64_t *)malloc((size_t)natoms * sizeof(int64_t));
  int64_t *start = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
  int64_t *members = (int64_t *)malloc((size_t)natoms * sizeof(int64_t));
  if (!cell_of || !start || !members) { free(cell_of); free(start); free(members); return DPO_ENOMEM; }
  for (int64_t i = 0; i < natoms; ++i) {
    int ic[3];
    for (int c = 0; c < 3; ++c) {
      double f = coord[3 * i + c] / L[c];
      f -= floor(f);
      ic[c] = (int)(f * nc[c]);
      if (ic[c] >= nc[c]) ic[c] = nc[c] - 1;
      if (ic[c] < 0) ic[c] = 0;
    }
    cell_of[i] = ((int64_t)ic[0] * nc[1] + ic[1]) * nc[2] + ic[2];
    start[cell_of[i] + 1]++;
  }
  for (int64_t c = 0; c < ncell; ++c) start[c + 1] += start[c];
  {
    int64_t *fill = (int64_t *)malloc((size_t)ncell * sizeof(int64_t));
    if (!fill) { free(cell_of); free(start); free(members); return DPO_ENOMEM; }
    memcpy(fill, start, (size_t)ncell * sizeof(int64_t));
    for (int64_t i = 0; i < natoms; ++i) members[fill[cell_of[i]]++] = i;   /* ascending atom index per cell */
    free(fill);
  }
  int64_t dropped_total = 0;
  int err = 0;
#pragma omp parallel
  {
    int64_t cap = 1024, dropped = 0;
    cand_t *cand = (cand_t *)malloc((size_t)cap * sizeof(cand_t));
    if (!cand) {
#pragma omp atomic write
      err = 1;
    }
#pragma omp for schedule(dynamic, 64)
    for (int64_t i = 0; i < natoms; ++i) {
      if (err) continue;
      int64_t ci = cell_of[i];
      int ic[3] = { (int)(ci / ((int64_t)nc[1] * nc[2])), (int)((ci / nc[2]) % nc[1]), (int)(ci % nc[2]) };
      int lo[3], cnt[3];
      for (int c = 0; c < 3; ++c) {
        if (nc[c] >= 3) { lo[c] = ic[c] - 1; cnt[c] = 3; }
        else { lo[c] = 0; cnt[c] = nc[c]; }           /* fewer than 3 cells: visit each cell once */
      }
      int64_t ncand = 0;
      for (int a = 0; a < cnt[0] && !err; ++a)
        for (int b = 0; b < cnt[1] && !err; ++b)
          for (int c = 0; c < cnt[2] && !err; ++c) {
            int ja = ((lo[0] + a) % nc[0] + nc[0]) % nc[0];
            int jb = ((lo[1] + b) % nc[1] + nc[1]) % nc[1];
            int jc = ((lo[2] + c) % nc[2] + nc[2]) % nc[2];
            int64_t cj = ((int64_t)ja * nc[1] + jb) * nc[2] + jc;
            for (int64_t p = start[cj]; p < start[cj + 1]; ++p) {
              int64_t j = members[p];
              if (j == i) continue;
              double d[3], r;
              dpo_displacement(coord + 3 * i, coord + 3 * j, L, d, &r);
              if (r <= m->rcut) {
                if (ncand == cap) {
                  cap *= 2;
                  cand_t *nw = (cand_t *)realloc(cand, (size_t)cap * sizeof(cand_t));
                  if (!nw) {
#pragma omp atomic write
                    err = 1;
                    break;
                  }
                  cand = nw;
                }
                cand[ncand].type = type[j]; cand[ncand].r = r; cand[ncand].j = (int32_t)j;
                ++ncand;
              }
            }
          }
      if (!err) dropped += format_row(m, cand, ncand, nlist_out + i * nm);
    }
#pragma omp atomic
    dropped_total += dropped;
    free(cand);
  }
  free(cell_of); free(start); free(members);
  if (err) return DPO_ENOMEM;
  if (n_overflow) *n_overflow = dropped_total;
  return DPO_OK;
}

/* O5 + O10: Alg. 2 and Eq. 5 (:100-103).  Real slot: s = w(r)/r,
 * R~ = (s, s dx/r, s dy/r, s dz/r); padded slot: zeros (:105, :238).
 * Derivative with respect to the displacement d (used by ProdForce / ProdVirial, :240), with q = s/r,
 * s' = w'/r - w/r^2, q' = s'/r - s/r^2:
 *   dR~_0/dd_c = s' d_c/r;   dR~_{1+b}/dd_c = q' d_b d_c / r + q delta_bc. */
int dpo_env_row(const dpo_model_desc *m, int64_t natoms, const double *coord, const double box[9], int64_t i,
                const int32_t *nlist_row, double *env, double *denv, double *disp) {
  double L[3];
  int rc = check_inputs(m, box, L);
  if (rc != DPO_OK) return rc;
  int nm = dpo_nm(m);
  for (int k = 0; k < nm; ++k) {
    int32_t j = nlist_row[k];
    double *e = env ? env + 4 * k : NULL;
    double *de = denv ? denv + 12 * k : NULL;
    double *dd = disp ? disp + 3 * k : NULL;
    if (j < 0) {
      if (e) memset(e, 0, 4 * sizeof(double));
      if (de) memset(de, 0, 12 * sizeof(double));
      if (dd) memset(dd, 0, 3 * sizeof(double));
      continue;
    }
    if (j >= natoms) return DPO_EINVAL;
    double d[3], r, w, dw;
    dpo_displacement(coord + 3 * i, coord + 3 * j, L, d, &r);
    dpo_switch(r, m->rcut_smth, m->rcut, &w, &dw);
    double s = w / r;
    double q = s / r;
    double sp = dw / r - w / (r * r);
    double qp = sp / r - s / (r * r);
    if (e) {
      e[0] = s;
      for (int b = 0; b < 3; ++b) e[1 + b] = s * d[b] / r;
    }
    if (de) {
      for (int c = 0; c < 3; ++c) de[0 * 3 + c] = sp * d[c] / r;
      for (int b = 0; b < 3; ++b)
        for (int c = 0; c < 3; ++c) de[(1 + b) * 3 + c] = qp * d[b] * d[c] / r + (b == c ? q : 0.0);
    }
    if (dd) { dd[0] = d[0]; dd[1] = d[1]; dd[2] = d[2]; }
  }
  return DPO_OK;
}

/* O6: embedding net, Eq. 7-9.  Layer 0 (Eq. 8, no skip): h0 = tanh(x W0 + b0), b0 in
 * R^{s1} (reading R2b: ":117 b0 in R" is a typo).  Layers k >= 1 (Eq. 9): h_k = (h_{k-1}, h_{k-1}) +
 * tanh(h_{k-1} W_k + b_k), where (x, x) is the concatenation [x || x] (Eq. 12 :268).
 * Keeps the tanh values t0, t1, t2 for the backward (d tanh = 1 - tanh^2, :273). */
static void embed_fwd(const double *net, int s1, double x, double *t0, double *t1, double *h1, double *t2,
                      double *g) {
  const double *W0 = net, *b0 = W0 + s1, *W1 = b0 + s1, *b1 = W1 + (int64_t)s1 * 2 * s1, *W2 = b1 + 2 * s1,
               *b2 = W2 + (int64_t)2 * s1 * 4 * s1;
  for (int a = 0; a < s1; ++a) t0[a] = tanh(x * W0[a] + b0[a]);
  for (int o = 0; o < 2 * s1; ++o) {
    double acc = 0.0;
    for (int a = 0; a < s1; ++a) acc += t0[a] * W1[a * 2 * s1 + o];
    t1[o] = tanh(acc + b1[o]);
    h1[o] = t0[o % s1] + t1[o];
  }
  for (int o = 0; o < 4 * s1; ++o) {
    double acc = 0.0;
    for (int a = 0; a < 2 * s1; ++a) acc += h1[a] * W2[a * 4 * s1 + o];
    t2[o] = tanh(acc + b2[o]);
    g[o] = h1[o % (2 * s1)] + t2[o];
  }
}

void dpo_embed(const double *net, int32_t s1, double x, double *g) {
  double *buf = (double *)malloc((size_t)(9 * s1) * sizeof(double));
  embed_fwd(net, s1, x, buf, buf + s1, buf + 3 * s1, buf + 5 * s1, g);
  free(buf);
}

/* O9 (embedding part): reverse mode through O6 ("back propagation").  Given dg = dE/dg returns
 * dE/dx.  delta2 = dg (1 - t2^2); dh1 = delta2 W2^T + dg[0:2s1] + dg[2s1:4s1]; delta1 = dh1 (1 - t1^2);
 * dh0 = delta1 W1^T + dh1[0:s1] + dh1[s1:2s1]; dx = sum (dh0 (1 - t0^2)) W0. */
static double embed_bwd(const double *net, int s1, const double *t0, const double *t1, const double *t2,
                        const double *dg, double *dh1, double *dh0) {
  const double *W0 = net, *b0 = W0 + s1, *W1 = b0 + s1, *b1 = W1 + (int64_t)s1 * 2 * s1, *W2 = b1 + 2 * s1;
  for (int a = 0; a < 2 * s1; ++a) {
    double acc = 0.0;
    for (int o = 0; o < 4 * s1; ++o) acc += dg[o] * (1.0 - t2[o] * t2[o]) * W2[a * 4 * s1 + o];
    dh1[a] = acc + dg[a] + dg[a + 2 * s1];
  }
  for (int a = 0; a < s1; ++a) {
    double acc = 0.0;
    for (int o = 0; o < 2 * s1; ++o) acc += dh1[o] * (1.0 - t1[o] * t1[o]) * W1[a * 2 * s1 + o];
    dh0[a] = acc + dh1[a] + dh1[a + s1];
  }
  double dx = 0.0;
  for (int a = 0; a < s1; ++a) dx += dh0[a] * (1.0 - t0[a] * t0[a]) * W0[a];
  return dx;
}

/* O8: fitting net, Eq. 2-3, one net per species (:123).  Reading R4: the first layer D -> w
 * has no skip (sizes differ), hidden layers w -> w are x + tanh(x W + b) (Eq. 3), the output layer is linear
 * w -> 1 with bias.  z0, u1, u2 (tanh values) and z1, z2 are kept for the backward. */
static double fit_fwd(const double *net, int dim, int w, const double *D, double *z0, double *u1, double *z1,
                      double *u2, double *z2) {
  const double *W0 = net, *b0 = W0 + (int64_t)dim * w, *W1 = b0 + w, *b1 = W1 + (int64_t)w * w, *W2 = b1 + w,
               *b2 = W2 + (int64_t)w * w, *w3 = b2 + w, *b3 = w3 + w;
  for (int o = 0; o < w; ++o) {
    double acc = 0.0;
    for (int d = 0; d < dim; ++d) acc += D[d] * W0[(int64_t)d * w + o];
    z0[o] = tanh(acc + b0[o]);
  }
  for (int o = 0; o < w; ++o) {
    double acc = 0.0;
    for (int a = 0; a < w; ++a) acc += z0[a] * W1[a * w + o];
    u1[o] = tanh(acc + b1[o]);
    z1[o] = z0[o] + u1[o];
  }
  for (int o = 0; o < w; ++o) {
    double acc = 0.0;
    for (int a = 0; a < w; ++a) acc += z1[a] * W2[a * w + o];
    u2[o] = tanh(acc + b2[o]);
    z2[o] = z1[o] + u2[o];
  }
  double e = 0.0;
  for (int o = 0; o < w; ++o) e += z2[o] * w3[o];
  return e + b3[0];
}

double dpo_fit(const double *net, int32_t dim, int32_t width, const double *D) {
  double *buf = (double *)malloc((size_t)(5 * width) * sizeof(double));
  double e = fit_fwd(net, dim, width, D, buf, buf + width, buf + 2 * width, buf + 3 * width, buf + 4 * width);
  free(buf);
  return e;
}

/* O9 (fitting part): dz2 = w3; dz1 = dz2 + (dz2 (1 - u2^2)) W2^T; dz0 = dz1 + (dz1 (1 - u1^2)) W1^T;
 * dD = (dz0 (1 - z0^2)) W0^T. */
static void fit_bwd(const double *net, int dim, int w, const double *z0, const double *u1, const double *u2,
                    double *dz1, double *dz0, double *dD) {
  const double *W0 = net, *b0 = W0 + (int64_t)dim * w, *W1 = b0 + w, *b1 = W1 + (int64_t)w * w, *W2 = b1 + w,
               *b2 = W2 + (int64_t)w * w, *w3 = b2 + w;
  for (int a = 0; a < w; ++a) {
    double acc = 0.0;
    for (int o = 0; o < w; ++o) acc += w3[o] * (1.0 - u2[o] * u2[o]) * W2[a * w + o];
    dz1[a] = w3[a] + acc;
  }
  for (int a = 0; a < w; ++a) {
    double acc = 0.0;
    for (int o = 0; o < w; ++o) acc += dz1[o] * (1.0 - u1[o] * u1[o]) * W1[a * w + o];
    dz0[a] = dz1[a] + acc;
  }
  for (int d = 0; d < dim; ++d) {
    double acc = 0.0;
    for (int o = 0; o < w; ++o) acc += dz0[o] * (1.0 - z0[o] * z0[o]) * W0[(int64_t)d * w + o];
    dD[d] = acc;
  }
}

/* O5..O10 for the listed atoms: E_i = N_{alpha_i}(D(R_i)) (Eq. 1) and dE_i/dd_ik. */
int dpo_atom_rows(const dpo_model_desc *m, int64_t natoms, const double *coord, const int32_t *type,
                  const double box[9], int64_t nrows, const int64_t *rows, const int32_t *nlist_rows,
                  double *atom_energy, double *fslot, double *T_out, double *D_out, double *dT_out) {
  double L[3];
  int rc = check_inputs(m, box, L);
  if (rc != DPO_OK) return rc;
  const int nm = dpo_nm(m), s1 = m->emb_s1, M = 4 * s1, Ma = m->m_axis, w = m->fit_width, dim = M * Ma;
  const int64_t esz = emb_net_size(s1), fsz = fit_net_size(dim, w);
  int err = 0;
#pragma omp parallel
  {
    /* per-thread workspace: env rows, per-slot activations (t0 s1, t1 2s1, h1 2s1, t2 4s1, g 4s1 = 13 s1) */
    size_t nd = (size_t)nm * 4 + (size_t)nm * 12 + (size_t)nm * 13 * s1 + (size_t)M * 4 * 2 + (size_t)dim * 2 +
                (size_t)w * 7 + (size_t)M + (size_t)3 * s1;
    double *ws = (double *)malloc(nd * sizeof(double));
    if (!ws) {
#pragma omp atomic write
      err = DPO_ENOMEM;
    }
    double *env = ws, *denv = env + (size_t)nm * 4, *act = denv + (size_t)nm * 12,
           *T = act + (size_t)nm * 13 * s1, *dT = T + M * 4, *D = dT + M * 4, *dD = D + dim, *z0 = dD + dim,
           *u1 = z0 + w, *z1 = u1 + w, *u2 = z1 + w, *z2 = u2 + w, *dz1 = z2 + w, *dz0 = dz1 + w,
           *dg = dz0 + w, *dh1 = dg + M, *dh0 = dh1 + 2 * s1;
#pragma omp for schedule(dynamic, 4)
    for (int64_t q = 0; q < nrows; ++q) {
      if (err) continue;
      const int64_t i = rows ? rows[q] : q;
      const int32_t *row = nlist_rows + q * nm;
      const int ti = type[i];
      int e2 = dpo_env_row(m, natoms, coord, box, i, row, env, denv, NULL);
      if (e2 != DPO_OK || ti < 0 || ti >= m->ntypes) {
#pragma omp atomic write
        err = DPO_EINVAL;
        continue;
      }
      /* O6 + O7: G_i rows for real slots; the slot's section gives the neighbour type t, net (alpha_i, t)
       * (Remark 1).  T = G^T R~ (M x 4), summed in slot order. */
      memset(T, 0, (size_t)M * 4 * sizeof(double));
      int k = 0;
      for (int t = 0; t < m->ntypes; ++t) {
        const double *net = m->emb_weights + (int64_t)(ti * m->ntypes + t) * esz;
        for (int kk = 0; kk < m->sel[t]; ++kk, ++k) {
          if (row[k] < 0) continue;                      /* padded: zero row of R~, contributes 0 (:105) */
          double *a = act + (size_t)k * 13 * s1;
          double *t0 = a, *t1 = a + s1, *h1 = a + 3 * s1, *t2 = a + 5 * s1, *g = a + 9 * s1;
          embed_fwd(net, s1, env[4 * k + 0], t0, t1, h1, t2, g);
          for (int b = 0; b < M; ++b)
            for (int c = 0; c < 4; ++c) T[b * 4 + c] += g[b] * env[4 * k + c];
        }
      }
      /* O7: D = (G^T R~)(R~^T G^<), Eq. 4, M x M^< row-major (reading R7):
       * D[b][a] = sum_c T[b][c] T[a][c], a < M^<. */
      for (int b = 0; b < M; ++b)
        for (int a = 0; a < Ma; ++a) {
          double acc = 0.0;
          for (int c = 0; c < 4; ++c) acc += T[b * 4 + c] * T[a * 4 + c];
          D[b * Ma + a] = acc;
        }
      /* O8, O9: fitting net of species alpha_i forward and backward. */
      const double *fnet = m->fit_weights + (int64_t)ti * fsz;
      atom_energy[q] = fit_fwd(fnet, dim, w, D, z0, u1, z1, u2, z2);
      fit_bwd(fnet, dim, w, z0, u1, u2, dz1, dz0, dD);
      /* O9: dT[b][c] = sum_a dD[b][a] T[a][c] + [b < M^<] sum_b' dD[b'][b] T[b'][c]. */
      for (int b = 0; b < M; ++b)
        for (int c = 0; c < 4; ++c) {
          double acc = 0.0;
          for (int a = 0; a < Ma; ++a) acc += dD[b * Ma + a] * T[a * 4 + c];
          if (b < Ma)
            for (int bp = 0; bp < M; ++bp) acc += dD[bp * Ma + b] * T[bp * 4 + c];
          dT[b * 4 + c] = acc;
        }
      if (T_out) memcpy(T_out + (size_t)q * M * 4, T, (size_t)M * 4 * sizeof(double));
      if (D_out) memcpy(D_out + (size_t)q * dim, D, (size_t)dim * sizeof(double));
      if (dT_out) memcpy(dT_out + (size_t)q * M * 4, dT, (size_t)M * 4 * sizeof(double));
      /* O9, O10 per real slot: dg = dT R~_k; dR~_k[c] = sum_b dT[b][c] g_k[b]; dR~_k[0] += dE/dx through the
       * embedding net; f_ik[c] = sum_m dR~_k[m] dR~_m/dd_c. */
      k = 0;
      for (int t = 0; t < m->ntypes; ++t) {
        const double *net = m->emb_weights + (int64_t)(ti * m->ntypes + t) * esz;
        for (int kk = 0; kk < m->sel[t]; ++kk, ++k) {
          double *f = fslot + ((size_t)q * nm + k) * 3;
          f[0] = f[1] = f[2] = 0.0;
          if (row[k] < 0) continue;
          double *a = act + (size_t)k * 13 * s1;
          double *t0 = a, *t1 = a + s1, *t2 = a + 5 * s1, *g = a + 9 * s1;
          double dR[4] = {0.0, 0.0, 0.0, 0.0};
          for (int b = 0; b < M; ++b) {
            double acc = 0.0;
            for (int c = 0; c < 4; ++c) acc += dT[b * 4 + c] * env[4 * k + c];
            dg[b] = acc;
          }
          for (int c = 0; c < 4; ++c)
            for (int b = 0; b < M; ++b) dR[c] += dT[b * 4 + c] * g[b];
          dR[0] += embed_bwd(net, s1, t0, t1, t2, dg, dh1, dh0);
          for (int c = 0; c < 3; ++c) {
            double acc = 0.0;
            for (int mm = 0; mm < 4; ++mm) acc += dR[mm] * denv[(size_t)k * 12 + mm * 3 + c];
            f[c] = acc;
          }
        }
      }
    }
    free(ws);
  }
  return err;
}

/* One full evaluation: E = sum_i E_i (Eq. 1), F_i = -dE/dr_i (Eq. 10, :125-127), virial
 * (ProdVirial, :240; reading R14).  O11: d_ik = r_j - r_i, so F_i += f_ik, F_j -= f_ik and
 * Xi[a][b] -= d_ik[a] f_ik[b], all accumulated serially in atom order, slot order. */
int dpo_eval(const dpo_model_desc *m, int64_t natoms, const double *coord, const int32_t *type,
             const double box[9], double *energy, double *atom_energy, double *force, double *virial,
             int32_t *nlist_out, int use_cells) {
  double L[3];
  int rc = check_inputs(m, box, L);
  if (rc != DPO_OK) return rc;
  const int nm = dpo_nm(m);
  int32_t *nlist = nlist_out ? nlist_out : (int32_t *)malloc((size_t)natoms * nm * sizeof(int32_t));
  double *fslot = (double *)malloc((size_t)natoms * nm * 3 * sizeof(double));
  double *ei = atom_energy ? atom_energy : (double *)malloc((size_t)natoms * sizeof(double));
  if (!nlist || !fslot || !ei) { rc = DPO_ENOMEM; goto done; }
  rc = use_cells ? dpo_build_nlist_cells(m, natoms, coord, type, box, nlist, NULL)
                 : dpo_build_nlist_rows(m, natoms, coord, type, box, natoms, NULL, nlist, NULL);
  if (rc != DPO_OK) goto done;
  rc = dpo_atom_rows(m, natoms, coord, type, box, natoms, NULL, nlist, ei, fslot, NULL, NULL, NULL);
  if (rc != DPO_OK) goto done;
  {
    double e = 0.0;
    for (int64_t i = 0; i < natoms; ++i) e += ei[i];
    if (energy) *energy = e;
  }
  if (force) memset(force, 0, (size_t)natoms * 3 * sizeof(double));
  if (virial) memset(virial, 0, 9 * sizeof(double));
  for (int64_t i = 0; i < natoms; ++i)
    for (int k = 0; k < nm; ++k) {
      int32_t j = nlist[i * nm + k];
      if (j < 0) continue;
      const double *f = fslot + ((size_t)i * nm + k) * 3;
      if (force)
        for (int c = 0; c < 3; ++c) { force[3 * i + c] += f[c]; force[3 * (int64_t)j + c] -= f[c]; }
      if (virial) {
        double d[3], r;
        dpo_displacement(coord + 3 * i, coord + 3 * (int64_t)j, L, d, &r);
        for (int a = 0; a < 3; ++a)
          for (int b = 0; b < 3; ++b) virial[3 * a + b] -= d[a] * f[b];
      }
    }
done:
  if (!nlist_out) free(nlist);
  if (!atom_energy) free(ei);
  free(fslot);
  return rc;
}

/* ---- NEXT #3: per-atom virial ------------------------------------------------------------
 * The paper names the virial only through the ProdVirial operator and gives no per-atom split.  Reading
 * R14 defines Xi = -sum_i sum_k d_ik (x) dE_i/dd_ik; the split used here assigns every term to its CENTRE atom:
 *     Xi_i[a][b] = -sum_k d_ik[a] (dE_i/dd_ik)[b],      sum_i Xi_i = Xi.
 * Xi_i is then minus the (transposed) derivative of E_i alone under a homogeneous strain of the configuration, which is
 * what tests/test_oracle_physics.py pins it to.  atom_virial is [N][9]. */
int dpo_atom_virial(const dpo_model_desc *m, int64_t natoms, const double *coord, const int32_t *type,
                    const double box[9], double *atom_virial) {
  double L[3];
  int rc = check_inputs(m, box, L);
  if (rc != DPO_OK) return rc;
  const int nm = dpo_nm(m);
  const size_t nrow = (size_t)(natoms > 0 ? natoms : 1);
  int32_t *nlist = (int32_t *)malloc(nrow * nm * sizeof(int32_t));
  double *fslot = (double *)malloc(nrow * nm * 3 * sizeof(double));
  double *ei = (double *)malloc(nrow * sizeof(double));
  if (!nlist || !fslot || !ei) { rc = DPO_ENOMEM; goto done; }
  rc = dpo_build_nlist_rows(m, natoms, coord, type, box, natoms, NULL, nlist, NULL);
  if (rc != DPO_OK) goto done;
  rc = dpo_atom_rows(m, natoms, coord, type, box, natoms, NULL, nlist, ei, fslot, NULL, NULL, NULL);
  if (rc != DPO_OK) goto done;
  memset(atom_virial, 0, (size_t)natoms * 9 * sizeof(double));
  for (int64_t i = 0; i < natoms; ++i)
    for (int k = 0; k < nm; ++k) {
      int32_t j = nlist[i * nm + k];
      if (j < 0) continue;
      const double *f = fslot + ((size_t)i * nm + k) * 3;
      double d[3], r;
      dpo_displacement(coord + 3 * i, coord + 3 * (int64_t)j, L, d, &r);
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) atom_virial[9 * i + 3 * a + b] -= d[a] * f[b];
    }
done:
  free(nlist); free(fslot); free(ei);
  return rc;
}

/* ---- NEXT #2 / #3: evaluation of one sub-region with explicit ghost atoms ------------
 * The paper's parallel formulation: a sub-region owns its "local" atoms; the atoms of the
 * neighbouring sub-regions (and the periodic images) that lie within r_c of it are present as explicit "ghost" atoms.
 * Atoms 0 .. nloc-1 are local, nloc .. nall-1 are ghosts.  There is no box: every displacement is the plain difference
 * r_j - r_i.  E = sum over LOCAL atoms of E_i; force[nall][3] = -dE/dr for local and ghost atoms alike (the ghost part
 * is what the reverse exchange sends home: grad_{r_i} E_j != -grad_{r_j} E_i, so it cannot be dropped);
 * virial = -sum over local i, slots k of d_ik (x) dE_i/dd_ik (reading R14).  Summed over the sub-regions of a periodic
 * system these give E, F and the virial of dpo_eval on the whole box: that identity is the pin (tests/test_oracle_local.py).
 * Implementation: dpo_displacement with box edges of 1e300 A, for which k = rint(dc / L) = 0 and fma(-0, L, dc) = dc. */
#define DPO_OPEN_EDGE 1e300

int dpo_eval_local(const dpo_model_desc *m, int64_t nloc, int64_t nall, const double *coord, const int32_t *type,
                   double *energy, double *atom_energy, double *force, double *virial, int32_t *nlist_out) {
  if (nloc < 0 || nall < nloc) return DPO_EINVAL;
  const double box[9] = {DPO_OPEN_EDGE, 0, 0, 0, DPO_OPEN_EDGE, 0, 0, 0, DPO_OPEN_EDGE};
  double L[3];
  int rc = check_inputs(m, box, L);
  if (rc != DPO_OK) return rc;
  const int nm = dpo_nm(m);
  const size_t nrow = (size_t)(nloc > 0 ? nloc : 1);
  int32_t *nlist = nlist_out ? nlist_out : (int32_t *)malloc(nrow * nm * sizeof(int32_t));
  double *fslot = (double *)malloc(nrow * nm * 3 * sizeof(double));
  double *ei = atom_energy ? atom_energy : (double *)malloc(nrow * sizeof(double));
  if (!nlist || !fslot || !ei) { rc = DPO_ENOMEM; goto done; }
  /* neighbours of the local atoms among ALL atoms; rows == NULL: atoms 0 .. nloc-1 */
  rc = dpo_build_nlist_rows(m, nall, coord, type, box, nloc, NULL, nlist, NULL);
  if (rc != DPO_OK) goto done;
  rc = dpo_atom_rows(m, nall, coord, type, box, nloc, NULL, nlist, ei, fslot, NULL, NULL, NULL);
  if (rc != DPO_OK) goto done;
  {
    double e = 0.0;
    for (int64_t i = 0; i < nloc; ++i) e += ei[i];
    if (energy) *energy = e;
  }
  if (force) memset(force, 0, (size_t)nall * 3 * sizeof(double));
  if (virial) memset(virial, 0, 9 * sizeof(double));
  for (int64_t i = 0; i < nloc; ++i)
    for (int k = 0; k < nm; ++k) {
      int32_t j = nlist[i * nm + k];
      if (j < 0) continue;
      const double *f = fslot + ((size_t)i * nm + k) * 3;
      if (force)
        for (int c = 0; c < 3; ++c) { force[3 * i + c] += f[c]; force[3 * (int64_t)j + c] -= f[c]; }
      if (virial)
        for (int a = 0; a < 3; ++a) {
          const double da = coord[3 * (int64_t)j + a] - coord[3 * i + a];
          for (int b = 0; b < 3; ++b) virial[3 * a + b] -= da * f[b];
        }
    }
done:
  if (!nlist_out) free(nlist);
  if (!atom_energy) free(ei);
  free(fslot);
  return rc;
}

/* ---- NEXT #1: molecular dynamics driver --------------------------------------------------
 * Velocity-Verlet integration of Newton's equations with the DP forces, NVE, as the paper runs it (PAPER.md:298:
 * velocity-Verlet, 0.5 fs for water, 1.0 fs for copper; thermo output every 20 steps).  One step:
 *     v <- v + (dt/2) F(x)/m;   x <- x + dt v;   F <- F(x);   v <- v + (dt/2) F/m.
 * The oracle searches neighbours from scratch at every step (the exact definition; a skin list that is rebuilt
 * every 50 steps, gives the same list as long as no atom moves more than half the skin).
 * Units: Angstrom, fs, amu, eV:  1 amu A^2/fs^2 = 103.6426965268 eV (CODATA 2018: 1.66053906660e-27 kg x 1e10 m^2/s^2 / 1.602176634e-19 C),
 * k_B = 8.617333262e-5 eV/K, T = 2 E_kin / (3 N k_B).  Coordinates are not wrapped (reading R2 takes raw values).
 * thermo[k][4] = (E_pot, E_kin, T, P) at steps 0, thermo_every, 2 thermo_every, ... <= nsteps ("kinetic
 * energy, potential energy, temperature, pressure ... every 20 time steps").  Pressure from the virial theorem,
 * P = (2 E_kin + tr Xi) / (3 V) with Xi = -sum d_ik (x) dE_i/dd_ik (reading R14), in bar: 1 eV/A^3 = 1.602176634e6 bar. */
#define DPO_AMU_A2_FS2_IN_EV 103.6426965268
#define DPO_KB_EV 8.617333262e-5
#define DPO_EV_A3_IN_BAR 1.602176634e6

int dpo_md_run(const dpo_model_desc *m, int64_t natoms, double *coord, double *vel, const int32_t *type,
               const double *mass, const double box[9], double dt_fs, int64_t nsteps, int64_t thermo_every,
               double *thermo, int use_cells) {
  if (natoms < 0 || nsteps < 0 || !(dt_fs > 0.0) || thermo_every < 1) return DPO_EINVAL;
  double *force = (double *)malloc((size_t)(natoms > 0 ? natoms : 1) * 3 * sizeof(double));
  if (!force) return DPO_ENOMEM;
  double epot = 0.0, vir[9];
  const double volume = box[0] * box[4] * box[8];
  int rc = dpo_eval(m, natoms, coord, type, box, &epot, NULL, force, vir, NULL, use_cells);
  int64_t nt = 0;
  for (int64_t step = 0; rc == DPO_OK; ++step) {
    if (step % thermo_every == 0 && thermo) {
      double ek = 0.0;
      for (int64_t i = 0; i < natoms; ++i) {
        const double *v = vel + 3 * i;
        ek += 0.5 * mass[type[i]] * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
      }
      ek *= DPO_AMU_A2_FS2_IN_EV;
      thermo[4 * nt + 0] = epot;
      thermo[4 * nt + 1] = ek;
      thermo[4 * nt + 2] = natoms > 0 ? 2.0 * ek / (3.0 * (double)natoms * DPO_KB_EV) : 0.0;
      thermo[4 * nt + 3] = (2.0 * ek + vir[0] + vir[4] + vir[8]) / (3.0 * volume) * DPO_EV_A3_IN_BAR;
      ++nt;
    }
    if (step == nsteps) break;
    for (int64_t i = 0; i < natoms; ++i) {
      const double h = 0.5 * dt_fs / (mass[type[i]] * DPO_AMU_A2_FS2_IN_EV);
      for (int c = 0; c < 3; ++c) {
        vel[3 * i + c] += h * force[3 * i + c];
        coord[3 * i + c] += dt_fs * vel[3 * i + c];
      }
    }
    rc = dpo_eval(m, natoms, coord, type, box, &epot, NULL, force, vir, NULL, use_cells);
    if (rc != DPO_OK) break;
    for (int64_t i = 0; i < natoms; ++i) {
      const double h = 0.5 * dt_fs / (mass[type[i]] * DPO_AMU_A2_FS2_IN_EV);
      for (int c = 0; c < 3; ++c) vel[3 * i + c] += h * force[3 * i + c];
    }
  }
  free(force);
  return rc;
}
