/*
 * tdpd_oracle.c — TEST INFRASTRUCTURE.  Plain, slow, fp64 CPU restatement of the tDPD + RBC
 * time step of arXiv:1611.06163, written from the paper's equations.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or constant generator with
 * the CUDA path under paper_1611_06163_b200/csrc/.
 *
 * Every function cites the passage it follows.  Readings of silent / garbled passages are the
 * ones listed in DESIGN.md §"Readings" (R1..), which follow SURVEY.md §8(c) A1..A26.
 *
 * Parity status: the cross-membrane coefficient reading (R15: kappa_ij by type pair), the form
 * of the source term Q^S (R-QS: zeroth-order source + first-order decay by species and type) and
 * the RBC parameter values are inputs / readings with no independent pin — "parity unpinned"
 * beyond conservation and the closed form of dC/dt = q - kC.  Everything else is
 * pinned by tests/test_oracle_*.py.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_T 4 /* max particle types   */
#define ORC_S 10 /* max chemical species (PAPER.md:218 benchmarks up to N_spec = 10) */

typedef struct {
  int32_t n_types, n_species;
  double box[3];
  double r_c, r_cc, dt, kBT, rho;
  double a[ORC_T][ORC_T], gamma[ORC_T][ORC_T], s_R[ORC_T][ORC_T];
  double kappa[ORC_S][ORC_T][ORC_T], s_c[ORC_S], m_s[ORC_S];
  double body_force[3];
  int32_t body_mode; /* 0 off, 1 uniform, 2 double Poiseuille in z */
  uint64_t seed;
  int32_t exclude_same_cell_membrane_pairs;
  /* Q^S of Eq 7 (reading R-QS): Q^S_i = source[s][type_i] - decay[s][type_i] C_i^s */
  double source[ORC_S][ORC_T], decay[ORC_S][ORC_T];
} orc_params;

typedef struct {
  double p, x0, m, gamma_T, gamma_C, k_g, k_l, k_v, k_b, theta0, VR_over_AR32;
} orc_rbc_params;

typedef struct {
  int64_t first_id;
  int32_t nv, ntri, nbond, ndih;
  int32_t *tri;  /* [ntri][3] local vertex indices, CCW from outside */
  int32_t *bond; /* [nbond][2] local, i<j */
  int32_t *dih;  /* [ndih][4] v1 v2 v3 v4: triangles (v1,v2,v3) and (v4,v3,v2) */
  double *h0, *kp; /* per bond */
  double *A0t;     /* per triangle */
  double A0, V0;
  double area, volume; /* totals of the last force evaluation (K-Gather) */
  double area_lag, volume_lag; /* totals of the force evaluation of the previous time step (PAPER.md:156 variant) */
  orc_rbc_params rp;
} orc_rbc;

typedef struct {
  orc_params P;
  int64_t n, cap;
  double *x, *v, *C;   /* [n][3], [n][3], [n][S] */
  int32_t *type, *rbc; /* rbc: 0 = solvent, k+1 = vertex of membrane k */
  double *F, *Fb, *Q, *g; /* pair force, bonded force, flux, body acceleration */
  int32_t n_rbc;
  orc_rbc *rbcs;
  int64_t step;        /* RNG step word of the last force evaluation */
  int have_forces;
  int use_brute;       /* 1: O(N^2) neighbour search */
  int lag_av;          /* 1: K-Apply uses the previous step's area / volume (Fig 2) */
  int lag_valid;       /* the lagged totals belong to step word lag_step */
  int64_t lag_step;
  /* pair census of the last force evaluation */
  int64_t n_cand, n_cc, n_c;
} orc_sim;

/* ------------------------------------------------------------------------------------------
 * Random numbers.  BASELINE north_star: "one specified counter-based hash of (min(i,j),
 * max(i,j), step, seed), for example Philox-4x32-10" (replaces the TEA scheme of PAPER.md:142).
 * Philox-4x32-10 as published by Salmon et al. (SC'11): 10 rounds; per round
 *   (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2, c' = (hi1^c1^k0, lo1, hi0^c3^k1, lo0),
 * key bumped by the Weyl constants between rounds.
 * ------------------------------------------------------------------------------------------ */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = M0 * (uint64_t)c0;
    uint64_t p1 = M1 * (uint64_t)c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* DESIGN.md R-RNG: 32-bit word -> uniform strictly inside (0,1), exactly representable in fp32
 * and fp64: u = ((x >> 9) + 1/2) 2^-23. */
static double orc_uniform(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

/* Box-Muller: R = sqrt(-2 ln ua), (g, g') = R (cos 2 pi ub, sin 2 pi ub). */
static void orc_box_muller(uint32_t xa, uint32_t xb, double *g_cos, double *g_sin) {
  double R = sqrt(-2.0 * log(orc_uniform(xa)));
  double t = 2.0 * M_PI * orc_uniform(xb);
  *g_cos = R * cos(t);
  *g_sin = R * sin(t);
}

/* Four Gaussians of the counter (min(id_i,id_j), max(id_i,id_j), step, tag), key = seed.
 * (x0,x1) -> g[0] (cos), g[1] (sin); (x2,x3) -> g[2] (cos), g[3] (sin). */
void orc_gauss4(int64_t id_i, int64_t id_j, int64_t step, uint32_t tag, uint64_t seed, double g[4]) {
  uint32_t lo = (uint32_t)(id_i < id_j ? id_i : id_j), hi = (uint32_t)(id_i < id_j ? id_j : id_i);
  uint32_t ctr[4] = {lo, hi, (uint32_t)step, tag};
  uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
  uint32_t x[4];
  orc_philox4x32_10(ctr, key, x);
  orc_box_muller(x[0], x[1], &g[0], &g[1]);
  orc_box_muller(x[2], x[3], &g[2], &g[3]);
}


/* Batch helpers for the statistical / bit-exact pins (tests only). */
void orc_philox_batch(int64_t n, const uint32_t *ctr /* [n][4] */, const uint32_t key[2], uint32_t *out /* [n][4] */) {
  for (int64_t i = 0; i < n; ++i) orc_philox4x32_10(&ctr[4 * i], key, &out[4 * i]);
}
void orc_gauss_batch(int64_t n, const int64_t *id_i, const int64_t *id_j, int64_t step, uint32_t tag, uint64_t seed,
                     double *g /* [n][4] */) {
  for (int64_t i = 0; i < n; ++i) orc_gauss4(id_i[i], id_j[i], step, tag, seed, &g[4 * i]);
}

/* ------------------------------------------------------------------------------------------ */
static double min_image(double d, double L) {
  /* nearest periodic image of a coordinate difference, box length L */
  return d - L * floor(d / L + 0.5);
}

static double wrap(double x, double L) {
  x -= L * floor(x / L);
  if (x >= L) x = 0.0; /* x was a tiny negative number */
  return x;
}

/* ------------------------------------------------------------------------------------------
 * One ordered pair (i <- j): non-bonded force on i (Eq 3-6) and flux into i
 * (Eq 8-10).  d = r_i - r_j (minimum image), dv = v_i - v_j.
 *   F_ij = [ a w_c - gamma w_R^2 (e.dv) + sigma w_R xi / sqrt(dt) ] e,  w_c = 1 - r/r_c  (R2),
 *          w_R = w_c^s (R3), sigma = sqrt(2 kBT gamma) (Eq 6), w_D = w_R^2 (Eq 6).
 *   Q_ij = -kappa w_cc^{s_c} (C_i - C_j)
 *          + sgn_ij m_s sqrt(kappa rho max(C_i+C_j,0)) w_cc^{s_c/2} zeta / sqrt(dt)     (R5)
 *          w_cc = 1 - r/r_cc, sgn_ij = +1 if id_i < id_j else -1 (zeta_ij = -zeta_ji).
 * Returns 0 (beyond r_cc or coincident, R22), 1 (flux only), 2 (force and flux).
 * ------------------------------------------------------------------------------------------ */
int orc_pair_terms(const orc_params *P, int64_t id_i, int64_t id_j, int ti, int tj, const double d[3],
                   const double dv[3], const double *Ci, const double *Cj, int64_t step,
                   double F[3], double *Qout) {
  double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
  F[0] = F[1] = F[2] = 0.0;
  for (int s = 0; s < P->n_species; ++s) Qout[s] = 0.0;
  if (r2 < 1e-12) return 0;
  if (!(r2 < P->r_cc * P->r_cc) && !(r2 < P->r_c * P->r_c)) return 0;
  double r = sqrt(r2);
  /* Gaussians (DESIGN.md R-RNG): tag 0 -> xi = g[0], zeta_0 = g[1], zeta_1 = g[2]; species 2 + 4q .. 5 + 4q take the
   * four Gaussians of tag 4 + q in order */
  double g[4], g2[(ORC_S + 1) / 4][4];
  orc_gauss4(id_i, id_j, step, 0u, P->seed, g);
  for (int q = 0; 2 + 4 * q < P->n_species; ++q) orc_gauss4(id_i, id_j, step, 4u + (uint32_t)q, P->seed, g2[q]);
  int kind = 0;
  double inv_sqrt_dt = 1.0 / sqrt(P->dt);
  if (r < P->r_cc) {
    kind = 1;
    double w = 1.0 - r / P->r_cc;
    double sgn = id_i < id_j ? 1.0 : -1.0;
    for (int s = 0; s < P->n_species; ++s) {
      double kap = P->kappa[s][ti][tj];
      double zeta = s == 0 ? g[1] : s == 1 ? g[2] : g2[(s - 2) / 4][(s - 2) % 4];
      double wdc = pow(w, P->s_c[s]);
      double wrc = pow(w, 0.5 * P->s_c[s]); /* Eq 10: w_DC = w_RC^2 */
      double csum = Ci[s] + Cj[s];
      if (csum < 0.0) csum = 0.0;
      double eps = P->m_s[s] * sqrt(kap * P->rho * csum); /* Eq 10 */
      Qout[s] = -kap * wdc * (Ci[s] - Cj[s]) + sgn * eps * wrc * zeta * inv_sqrt_dt;
    }
  }
  if (r < P->r_c) {
    kind = 2;
    double e[3] = {d[0] / r, d[1] / r, d[2] / r};
    double wc = 1.0 - r / P->r_c;
    double wR = pow(wc, P->s_R[ti][tj]);
    double wD = wR * wR;
    double gam = P->gamma[ti][tj];
    double sigma = sqrt(2.0 * P->kBT * gam);
    double edv = e[0] * dv[0] + e[1] * dv[1] + e[2] * dv[2];
    double f = P->a[ti][tj] * wc - gam * wD * edv + sigma * wR * g[0] * inv_sqrt_dt;
    F[0] = f * e[0]; F[1] = f * e[1]; F[2] = f * e[2];
  }
  return kind;
}

/* is the pair skipped because both are vertices of the same membrane (R16)? */
static int same_membrane(const orc_sim *S, int64_t i, int64_t j) {
  return S->P.exclude_same_cell_membrane_pairs && S->rbc[i] != 0 && S->rbc[i] == S->rbc[j];
}

static void accumulate_pair(orc_sim *S, int64_t i, int64_t j, int64_t *ncc, int64_t *nc) {
  const orc_params *P = &S->P;
  int ns = P->n_species;
  if (i == j || same_membrane(S, i, j)) return;
  double d[3], dv[3], F[3], Q[ORC_S];
  for (int a = 0; a < 3; ++a) {
    d[a] = min_image(S->x[3 * i + a] - S->x[3 * j + a], P->box[a]);
    dv[a] = S->v[3 * i + a] - S->v[3 * j + a];
  }
  int kind = orc_pair_terms(P, i, j, S->type[i], S->type[j], d, dv, &S->C[ns * i], &S->C[ns * j],
                            S->step, F, Q);
  if (kind >= 1) {
    ++*ncc;
    for (int s = 0; s < ns; ++s) S->Q[ns * i + s] += Q[s];
  }
  if (kind == 2) {
    ++*nc;
    for (int a = 0; a < 3; ++a) S->F[3 * i + a] += F[a];
  }
}

/* O(N^2) neighbour search: every j for every i (Eq 2 / Eq 7 sums over j != i within the cutoff). */
static void pair_forces_brute(orc_sim *S) {
  int64_t n = S->n, ncc = 0, nc = 0;
#pragma omp parallel for schedule(static) reduction(+ : ncc, nc)
  for (int64_t i = 0; i < n; ++i)
    for (int64_t j = 0; j < n; ++j) accumulate_pair(S, i, j, &ncc, &nc);
  S->n_cand = n * (n - 1);
  S->n_cc = ncc;
  S->n_c = nc;
}

/* The oracle's own fp64 cell list: cells of edge >= max(r_c, r_cc), 27-cell stencil.
 * Proven equal to the brute-force search on small boxes (tests/test_oracle_*.py). */
static int cell_dims(const orc_params *P, int nc[3]) {
  double rmax = P->r_cc > P->r_c ? P->r_cc : P->r_c;
  for (int a = 0; a < 3; ++a) {
    nc[a] = (int)floor(P->box[a] / rmax);
    if (nc[a] < 3) return 0;
  }
  return 1;
}

static void pair_forces_cells(orc_sim *S) {
  const orc_params *P = &S->P;
  int nc[3];
  if (!cell_dims(P, nc)) { pair_forces_brute(S); return; }
  int64_t n = S->n, ncell = (int64_t)nc[0] * nc[1] * nc[2];
  int64_t *head = malloc((ncell + 1) * sizeof *head), *cell = malloc(n * sizeof *cell),
          *order = malloc(n * sizeof *order);
  memset(head, 0, (ncell + 1) * sizeof *head);
  for (int64_t i = 0; i < n; ++i) {
    int c[3];
    for (int a = 0; a < 3; ++a) {
      c[a] = (int)floor(wrap(S->x[3 * i + a], P->box[a]) / P->box[a] * nc[a]);
      if (c[a] >= nc[a]) c[a] = nc[a] - 1;
    }
    cell[i] = ((int64_t)c[2] * nc[1] + c[1]) * nc[0] + c[0];
    ++head[cell[i] + 1];
  }
  for (int64_t c = 0; c < ncell; ++c) head[c + 1] += head[c];
  int64_t *fill = malloc(ncell * sizeof *fill);
  memcpy(fill, head, ncell * sizeof *fill);
  for (int64_t i = 0; i < n; ++i) order[fill[cell[i]]++] = i;
  int64_t ncand = 0, ncc = 0, ncs = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : ncand, ncc, ncs)
  for (int64_t i = 0; i < n; ++i) {
    int64_t ci = cell[i];
    int cx = (int)(ci % nc[0]), cy = (int)((ci / nc[0]) % nc[1]), cz = (int)(ci / ((int64_t)nc[0] * nc[1]));
    for (int dz = -1; dz <= 1; ++dz)
      for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
          int x = (cx + dx + nc[0]) % nc[0], y = (cy + dy + nc[1]) % nc[1], z = (cz + dz + nc[2]) % nc[2];
          int64_t c = ((int64_t)z * nc[1] + y) * nc[0] + x;
          for (int64_t k = head[c]; k < head[c + 1]; ++k) {
            int64_t j = order[k];
            if (j != i) ++ncand;
            accumulate_pair(S, i, j, &ncc, &ncs);
          }
        }
  }
  S->n_cand = ncand; S->n_cc = ncc; S->n_c = ncs;
  free(head); free(cell); free(order); free(fill);
}


/* Pair force and flux of the listed particles only (the same sums as orc_compute_forces, restricted to
 * i in ids[]), for sampled parity at sizes where a full evaluation takes minutes.  O(n_ids * N). */
void orc_pair_forces_subset(orc_sim *S, int64_t step, int64_t n_ids, const int64_t *ids, double *F_out, double *Q_out) {
  const orc_params *P = &S->P;
  int ns = P->n_species;
  double rmax = P->r_cc > P->r_c ? P->r_cc : P->r_c;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t q = 0; q < n_ids; ++q) {
    int64_t i = ids[q];
    double Fs[3] = {0, 0, 0}, Qs[ORC_S] = {0, 0, 0, 0};
    for (int64_t j = 0; j < S->n; ++j) {
      if (j == i || same_membrane(S, i, j)) continue;
      double d[3], dv[3], F[3], Q[ORC_S];
      d[0] = min_image(S->x[3 * i] - S->x[3 * j], P->box[0]);
      if (fabs(d[0]) > rmax) continue;
      d[1] = min_image(S->x[3 * i + 1] - S->x[3 * j + 1], P->box[1]);
      if (fabs(d[1]) > rmax) continue;
      d[2] = min_image(S->x[3 * i + 2] - S->x[3 * j + 2], P->box[2]);
      for (int a = 0; a < 3; ++a) dv[a] = S->v[3 * i + a] - S->v[3 * j + a];
      int kind = orc_pair_terms(P, i, j, S->type[i], S->type[j], d, dv, &S->C[ns * i], &S->C[ns * j], step, F, Q);
      if (kind >= 1) for (int s = 0; s < ns; ++s) Qs[s] += Q[s];
      if (kind == 2) for (int a = 0; a < 3; ++a) Fs[a] += F[a];
    }
    for (int a = 0; a < 3; ++a) F_out[3 * q + a] = Fs[a];
    for (int s = 0; s < ns; ++s) Q_out[ns * q + s] = Qs[s];
  }
}

/* ------------------------------------------------------------------------------------------
 * Membrane.  Vertices of one cell are unwrapped by minimum image relative to
 * the cell's vertex 0 (R: membranes across the periodic boundary).
 * ------------------------------------------------------------------------------------------ */
static void cross(const double a[3], const double b[3], double c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}
static double dot(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

static void unwrap_rbc(const orc_sim *S, const orc_rbc *R, double *r /* [nv][3] */) {
  const double *x0 = &S->x[3 * R->first_id];
  for (int v = 0; v < R->nv; ++v)
    for (int a = 0; a < 3; ++a)
      r[3 * v + a] = x0[a] + min_image(S->x[3 * (R->first_id + v) + a] - x0[a], S->P.box[a]);
}

/* WLC force magnitude dU_WLC/dh from Eq 13:
 * U = (kBT h_m / 4p) (3x^2 - 2x^3)/(1-x), x = h/h_m  =>  dU/dh = (kBT/p) (6x - 9x^2 + 4x^3) / (4 (1-x)^2). */
static double wlc_force(double kBT, double p, double x) {
  return kBT / p * (6.0 * x - 9.0 * x * x + 4.0 * x * x * x) / (4.0 * (1.0 - x) * (1.0 - x));
}

/* Bond terms on vertex i of bond (i,j), Eq 13-16; force on j is the negative.
 * d = r_i - r_j, dv = v_i - v_j, N = 3x3 iid N(0,1) (rows from Philox tags 1,2,3).
 *   conservative: (-dU_WLC/dh + k_p/h^m) e           (Eq 13, 14; -dU_POW/dh = k_p/h^m)
 *   dissipative : -gT dv - gC (dv.e) e                (Eq 15)
 *   random      : sqrt(2 kBT/dt) [ sqrt(2 gT) (N^S - tr(N) I/3) + (sqrt(3 gC - gT)/3) tr(N) I ] e
 *                 (Eq 16 with dW = sqrt(dt) N and the ".e" and "/dt" the text omits, R10). */
void orc_bond_terms(double kBT, double dt, const orc_rbc_params *rp, double h0, double kp,
                    const double d[3], const double dv[3], const double N[9],
                    double Fc[3], double Fd[3], double Fr[3]) {
  double h = sqrt(dot(d, d));
  double e[3] = {d[0] / h, d[1] / h, d[2] / h};
  double x = h / (rp->x0 * h0);
  double f = -wlc_force(kBT, rp->p, x) + kp / pow(h, rp->m);
  double edv = dot(e, dv);
  double tr = N[0] + N[4] + N[8];
  double cT = sqrt(2.0 * rp->gamma_T), cC = sqrt(3.0 * rp->gamma_C - rp->gamma_T) / 3.0;
  double pre = sqrt(2.0 * kBT / dt);
  for (int a = 0; a < 3; ++a) {
    Fc[a] = f * e[a];
    Fd[a] = -rp->gamma_T * dv[a] - rp->gamma_C * edv * e[a];
    double acc = 0.0;
    for (int b = 0; b < 3; ++b) {
      double NS = 0.5 * (N[3 * a + b] + N[3 * b + a]);
      double M = cT * (NS - (a == b ? tr / 3.0 : 0.0)) + (a == b ? cC * tr : 0.0);
      acc += M * e[b];
    }
    Fr[a] = pre * acc;
  }
}

/* Triangle (1,2,3) CCW from outside: xi = (r2-r1)x(r3-r1), A_t = |xi|/2, V_t = r1.(r2 x r3)/6
 * ("area and quasi-volume"). */
static void tri_area_volume(const double *r1, const double *r2, const double *r3, double *A, double *V,
                            double nhat[3]) {
  double a[3] = {r2[0] - r1[0], r2[1] - r1[1], r2[2] - r1[2]};
  double b[3] = {r3[0] - r1[0], r3[1] - r1[1], r3[2] - r1[2]};
  double xi[3], c[3];
  cross(a, b, xi);
  double len = sqrt(dot(xi, xi));
  *A = 0.5 * len;
  cross(r2, r3, c);
  *V = dot(r1, c) / 6.0;
  if (nhat) { nhat[0] = xi[0] / len; nhat[1] = xi[1] / len; nhat[2] = xi[2] / len; }
}

void orc_rbc_area_volume(const orc_rbc *R, const double *r, double *area, double *volume) {
  double A = 0.0, V = 0.0;
  for (int t = 0; t < R->ntri; ++t) {
    double At, Vt;
    tri_area_volume(&r[3 * R->tri[3 * t]], &r[3 * R->tri[3 * t + 1]], &r[3 * R->tri[3 * t + 2]], &At, &Vt, NULL);
    A += At; V += Vt;
  }
  *area = A; *volume = V;
}

/* K-Apply: -grad of Eq 17 + Eq 18 given the totals A, V.
 *   beta_t = -k_g (A-A0)/A0 - k_l (A_t-A0t)/A0t ; dA_t/dr1 = (1/2) nhat x (r3-r2) (cyclic)
 *   beta_v = -k_v (V-V0)/V0               ; dV/dr1  = (1/6) r2 x r3       (cyclic) */
static void area_volume_forces(const orc_rbc *R, const double *r, double A, double V, double *f) {
  const orc_rbc_params *rp = &R->rp;
  double beta_v = -rp->k_v * (V - R->V0) / R->V0;
  for (int t = 0; t < R->ntri; ++t) {
    const int32_t *T = &R->tri[3 * t];
    const double *p[3] = {&r[3 * T[0]], &r[3 * T[1]], &r[3 * T[2]]};
    double At, Vt, nh[3];
    tri_area_volume(p[0], p[1], p[2], &At, &Vt, nh);
    double beta_t = -rp->k_g * (A - R->A0) / R->A0 - rp->k_l * (At - R->A0t[t]) / R->A0t[t];
    for (int k = 0; k < 3; ++k) {
      const double *pa = p[(k + 1) % 3], *pb = p[(k + 2) % 3]; /* the other two, cyclic */
      double edge[3] = {pb[0] - pa[0], pb[1] - pa[1], pb[2] - pa[2]};
      double ga[3], gv[3];
      cross(nh, edge, ga);
      cross(pa, pb, gv);
      for (int a = 0; a < 3; ++a) f[3 * T[k] + a] += 0.5 * beta_t * ga[a] + beta_v / 6.0 * gv[a];
    }
  }
}

/* Bending, Eq 19: U = k_b (1 - cos(theta - theta0)) per shared edge.
 * Triangles (v1,v2,v3), (v4,v3,v2), both CCW from outside; xi = (r2-r1)x(r3-r1),
 * zeta = (r3-r4)x(r2-r4), e = r3-r2; cos th = xihat.zetahat, sin th = (xihat x zetahat).ehat.
 * F_v = -k_b sin(th - th0) dth/dr_v with
 *   dth/dr1 = -|e| xi/|xi|^2, dth/dr4 = -|e| zeta/|zeta|^2,
 *   s1 = (r1-r2).e/|e|^2, s4 = (r4-r2).e/|e|^2,
 *   dth/dr2 = -(1-s1) dth/dr1 - (1-s4) dth/dr4,  dth/dr3 = -s1 dth/dr1 - s4 dth/dr4. */
double orc_dihedral_terms(double k_b, double theta0, const double *r1, const double *r2, const double *r3,
                          const double *r4, double F[12]) {
  double a[3], b[3], c[3], dd[3], e[3], xi[3], ze[3], cr[3];
  for (int k = 0; k < 3; ++k) {
    a[k] = r2[k] - r1[k]; b[k] = r3[k] - r1[k];
    c[k] = r3[k] - r4[k]; dd[k] = r2[k] - r4[k];
    e[k] = r3[k] - r2[k];
  }
  cross(a, b, xi);
  cross(c, dd, ze);
  double xi2 = dot(xi, xi), ze2 = dot(ze, ze), e2 = dot(e, e);
  double lxi = sqrt(xi2), lze = sqrt(ze2), le = sqrt(e2);
  double cth = dot(xi, ze) / (lxi * lze);
  cross(xi, ze, cr);
  double sth = dot(cr, e) / (lxi * lze * le);
  double theta = atan2(sth, cth);
  double coef = -k_b * sin(theta - theta0);
  double g1[3], g4[3], d12[3], d42[3];
  for (int k = 0; k < 3; ++k) {
    g1[k] = -le * xi[k] / xi2;
    g4[k] = -le * ze[k] / ze2;
    d12[k] = r1[k] - r2[k];
    d42[k] = r4[k] - r2[k];
  }
  double s1 = dot(d12, e) / e2, s4 = dot(d42, e) / e2;
  for (int k = 0; k < 3; ++k) {
    F[k] = coef * g1[k];
    F[3 + k] = coef * (-(1.0 - s1) * g1[k] - (1.0 - s4) * g4[k]);
    F[6 + k] = coef * (-s1 * g1[k] - s4 * g4[k]);
    F[9 + k] = coef * g4[k];
  }
  return theta;
}

static void bonded_forces(orc_sim *S) {
  const orc_params *P = &S->P;
#pragma omp parallel for schedule(dynamic, 1)
  for (int m = 0; m < S->n_rbc; ++m) {
    orc_rbc *R = &S->rbcs[m];
    double *r = malloc(3 * R->nv * sizeof *r), *f = calloc(3 * R->nv, sizeof *f);
    unwrap_rbc(S, R, r);
    /* bonds */
    for (int b = 0; b < R->nbond; ++b) {
      int i = R->bond[2 * b], j = R->bond[2 * b + 1];
      int64_t gi = R->first_id + i, gj = R->first_id + j;
      double d[3], dv[3], N[9], Fc[3], Fd[3], Fr[3];
      for (int a = 0; a < 3; ++a) {
        d[a] = r[3 * i + a] - r[3 * j + a];
        dv[a] = S->v[3 * gi + a] - S->v[3 * gj + a];
      }
      for (uint32_t row = 0; row < 3; ++row) {
        double g[4];
        orc_gauss4(gi, gj, S->step, 1u + row, P->seed, g);
        N[3 * row] = g[0]; N[3 * row + 1] = g[1]; N[3 * row + 2] = g[2];
      }
      orc_bond_terms(P->kBT, P->dt, &R->rp, R->h0[b], R->kp[b], d, dv, N, Fc, Fd, Fr);
      for (int a = 0; a < 3; ++a) {
        double t = Fc[a] + Fd[a] + Fr[a];
        f[3 * i + a] += t;
        f[3 * j + a] -= t;
      }
    }
    /* K-Gather then K-Apply.  Sequential variant (R20, the definition): this step's totals.  Variant of PAPER.md:156
     * ("use the area/volume of previous time step in K-Apply"): the totals of the force evaluation of step k - 1
     * when there was one (the very first evaluation, and one after the state was replaced, use their own). */
    orc_rbc_area_volume(R, r, &R->area, &R->volume);
    if (S->lag_av && S->lag_valid && S->lag_step == S->step - 1) area_volume_forces(R, r, R->area_lag, R->volume_lag, f);
    else area_volume_forces(R, r, R->area, R->volume, f);
    /* bending */
    for (int q = 0; q < R->ndih; ++q) {
      const int32_t *D = &R->dih[4 * q];
      double F[12];
      orc_dihedral_terms(R->rp.k_b, R->rp.theta0, &r[3 * D[0]], &r[3 * D[1]], &r[3 * D[2]], &r[3 * D[3]], F);
      for (int k = 0; k < 4; ++k)
        for (int a = 0; a < 3; ++a) f[3 * D[k] + a] += F[3 * k + a];
    }
    for (int v = 0; v < R->nv; ++v)
      for (int a = 0; a < 3; ++a) S->Fb[3 * (R->first_id + v) + a] = f[3 * v + a];
    free(r); free(f);
  }
}

/* Body acceleration g_i, evaluated at the positions of the force evaluation (R-body; PAPER.md:178-184:
 * "+f from 0 to d, -f from d to 2d"). */
static void body_forces(orc_sim *S) {
  const orc_params *P = &S->P;
  for (int64_t i = 0; i < S->n; ++i) {
    double sgn = 0.0;
    if (P->body_mode == 1) sgn = 1.0;
    else if (P->body_mode == 2) sgn = wrap(S->x[3 * i + 2], P->box[2]) < 0.5 * P->box[2] ? 1.0 : -1.0;
    for (int a = 0; a < 3; ++a) S->g[3 * i + a] = sgn * P->body_force[a];
  }
}

void orc_compute_forces(orc_sim *S, int64_t step) {
  S->step = step;
  memset(S->F, 0, 3 * S->n * sizeof(double));
  memset(S->Fb, 0, 3 * S->n * sizeof(double));
  memset(S->Q, 0, (size_t)S->P.n_species * S->n * sizeof(double));
  if (S->use_brute) pair_forces_brute(S); else pair_forces_cells(S);
  /* source term Q^S_i of Eq 7: external source and first-order reaction, by species and particle type */
  for (int64_t i = 0; i < S->n; ++i)
    for (int s = 0; s < S->P.n_species; ++s)
      S->Q[(size_t)S->P.n_species * i + s] += S->P.source[s][S->type[i]] - S->P.decay[s][S->type[i]] * S->C[(size_t)S->P.n_species * i + s];
  bonded_forces(S);
  body_forces(S);
  S->have_forces = 1;
}

/* Velocity-Verlet (BASELINE north_star (4); the paper does not describe its integrator; R21):
 *  (1) v += dt/2 (F + g); C += dt/2 Q; x = wrap(x + dt v)
 *  (2) k += 1; (F, Q) = forces(x, v, C; step k)      [half-step v and C enter F^D and Q]
 *  (3) v += dt/2 (F + g); C += dt/2 Q.        Mass m = 1.  F^0 uses step word 0. */
static void half_kick(orc_sim *S) {
  double h = 0.5 * S->P.dt;
  int ns = S->P.n_species;
  for (int64_t i = 0; i < S->n; ++i) {
    for (int a = 0; a < 3; ++a) S->v[3 * i + a] += h * (S->F[3 * i + a] + S->Fb[3 * i + a] + S->g[3 * i + a]);
    for (int s = 0; s < ns; ++s) S->C[ns * i + s] += h * S->Q[ns * i + s];
  }
}

void orc_step(orc_sim *S, int32_t nsteps) {
  if (!S->have_forces) orc_compute_forces(S, 0);
  for (int32_t it = 0; it < nsteps; ++it) {
    half_kick(S);
    for (int64_t i = 0; i < S->n; ++i)
      for (int a = 0; a < 3; ++a) S->x[3 * i + a] = wrap(S->x[3 * i + a] + S->P.dt * S->v[3 * i + a], S->P.box[a]);
    for (int m = 0; m < S->n_rbc; ++m) { S->rbcs[m].area_lag = S->rbcs[m].area; S->rbcs[m].volume_lag = S->rbcs[m].volume; }
    S->lag_step = S->step; S->lag_valid = 1;
    orc_compute_forces(S, S->step + 1);
    half_kick(S);
  }
}

/* ------------------------------------------------------------------------------------------
 * Construction / access
 * ------------------------------------------------------------------------------------------ */
orc_sim *orc_create(const orc_params *P) {
  orc_sim *S = calloc(1, sizeof *S);
  S->P = *P;
  return S;
}

static void grow(orc_sim *S, int64_t extra) {
  int64_t need = S->n + extra;
  if (need <= S->cap) return;
  int64_t cap = need;
  int ns = S->P.n_species;
  S->x = realloc(S->x, 3 * cap * sizeof(double));
  S->v = realloc(S->v, 3 * cap * sizeof(double));
  S->C = realloc(S->C, (size_t)ns * cap * sizeof(double));
  S->F = realloc(S->F, 3 * cap * sizeof(double));
  S->Fb = realloc(S->Fb, 3 * cap * sizeof(double));
  S->g = realloc(S->g, 3 * cap * sizeof(double));
  S->Q = realloc(S->Q, (size_t)ns * cap * sizeof(double));
  S->type = realloc(S->type, cap * sizeof(int32_t));
  S->rbc = realloc(S->rbc, cap * sizeof(int32_t));
  S->cap = cap;
}

static void append(orc_sim *S, int64_t n, const float *pos, const float *vel, const int32_t *type,
                   int32_t fixed_type, const float *conc, int32_t rbc) {
  int ns = S->P.n_species;
  grow(S, n);
  for (int64_t i = 0; i < n; ++i) {
    int64_t k = S->n + i;
    for (int a = 0; a < 3; ++a) {
      S->x[3 * k + a] = pos[3 * i + a];
      S->v[3 * k + a] = vel ? vel[3 * i + a] : 0.0;
    }
    for (int s = 0; s < ns; ++s) S->C[ns * k + s] = conc ? conc[ns * i + s] : 0.0;
    S->type[k] = type ? type[i] : fixed_type;
    S->rbc[k] = rbc;
  }
  S->n += n;
  S->have_forces = 0;
}

void orc_load_particles(orc_sim *S, int64_t n, const float *pos, const float *vel, const int32_t *type,
                        const float *conc) {
  append(S, n, pos, vel, type, 0, conc, 0);
}

/* Adds one membrane; derives bonds (unique edges), dihedrals (one per shared edge), per-bond rest
 * length h0 = initial length (R11), k_p from force balance at h0, per-triangle A0t, A0 = sum A0t and
 * V0 = A0^{3/2} V^R/(A^R)^{3/2}.  Membrane vertices get particle type `mtype`.
 * Returns the membrane index, or -1 if the mesh is not a closed, consistently oriented manifold. */
int32_t orc_add_rbc_mesh(orc_sim *S, int32_t nv, const float *verts, const float *vel, const float *conc,
                         int32_t ntri, const int32_t *tri, const orc_rbc_params *rp, int32_t mtype) {
  /* directed-edge table: opp[a*nv+b] = third vertex of the triangle containing a->b, or -1 */
  int32_t *opp = malloc((size_t)nv * nv * sizeof *opp);
  for (int64_t k = 0; k < (int64_t)nv * nv; ++k) opp[k] = -1;
  for (int t = 0; t < ntri; ++t)
    for (int k = 0; k < 3; ++k) {
      int a = tri[3 * t + k], b = tri[3 * t + (k + 1) % 3], c = tri[3 * t + (k + 2) % 3];
      if (a < 0 || a >= nv || b < 0 || b >= nv || a == b || opp[(int64_t)a * nv + b] != -1) { free(opp); return -1; }
      opp[(int64_t)a * nv + b] = c;
    }
  int nb = 0;
  for (int a = 0; a < nv; ++a)
    for (int b = a + 1; b < nv; ++b) {
      int f = opp[(int64_t)a * nv + b] != -1, r = opp[(int64_t)b * nv + a] != -1;
      if (f != r) { free(opp); return -1; }
      nb += f;
    }
  S->rbcs = realloc(S->rbcs, (S->n_rbc + 1) * sizeof(orc_rbc));
  orc_rbc *R = &S->rbcs[S->n_rbc];
  memset(R, 0, sizeof *R);
  R->first_id = S->n;
  R->nv = nv; R->ntri = ntri; R->nbond = nb; R->ndih = nb; R->rp = *rp;
  R->tri = malloc(3 * ntri * sizeof(int32_t));
  memcpy(R->tri, tri, 3 * ntri * sizeof(int32_t));
  R->bond = malloc(2 * nb * sizeof(int32_t));
  R->dih = malloc(4 * nb * sizeof(int32_t));
  R->h0 = malloc(nb * sizeof(double));
  R->kp = malloc(nb * sizeof(double));
  R->A0t = malloc(ntri * sizeof(double));
  append(S, nv, verts, vel, NULL, mtype, conc, S->n_rbc + 1);
  double *r = malloc(3 * nv * sizeof *r);
  unwrap_rbc(S, R, r);
  int q = 0;
  for (int a = 0; a < nv; ++a)
    for (int b = a + 1; b < nv; ++b) {
      if (opp[(int64_t)a * nv + b] == -1) continue;
      R->bond[2 * q] = a; R->bond[2 * q + 1] = b;
      /* triangle with a->b is (c,a,b) = (v1,v2,v3); triangle with b->a is (d,b,a) = (v4,v3,v2) */
      R->dih[4 * q] = opp[(int64_t)a * nv + b];
      R->dih[4 * q + 1] = a;
      R->dih[4 * q + 2] = b;
      R->dih[4 * q + 3] = opp[(int64_t)b * nv + a];
      double d[3] = {r[3 * a] - r[3 * b], r[3 * a + 1] - r[3 * b + 1], r[3 * a + 2] - r[3 * b + 2]};
      double h0 = sqrt(dot(d, d));
      R->h0[q] = h0;
      R->kp[q] = wlc_force(S->P.kBT, rp->p, 1.0 / rp->x0) * pow(h0, rp->m);
      ++q;
    }
  R->A0 = 0.0;
  for (int t = 0; t < ntri; ++t) {
    double Vt;
    tri_area_volume(&r[3 * tri[3 * t]], &r[3 * tri[3 * t + 1]], &r[3 * tri[3 * t + 2]], &R->A0t[t], &Vt, NULL);
    R->A0 += R->A0t[t];
  }
  R->V0 = pow(R->A0, 1.5) * rp->VR_over_AR32;
  free(r); free(opp);
  return S->n_rbc++;
}

void orc_set_params(orc_sim *S, const orc_params *P) { S->P = *P; S->have_forces = 0; }
void orc_set_brute(orc_sim *S, int32_t on) { S->use_brute = on; S->have_forces = 0; }
void orc_set_lagged_area_volume(orc_sim *S, int32_t on) { S->lag_av = on; S->have_forces = 0; }
int64_t orc_n(const orc_sim *S) { return S->n; }
int64_t orc_step_count(const orc_sim *S) { return S->step; }

void orc_set_state(orc_sim *S, const double *x, const double *v, const double *C) {
  if (x) memcpy(S->x, x, 3 * S->n * sizeof(double));
  if (v) memcpy(S->v, v, 3 * S->n * sizeof(double));
  if (C) memcpy(S->C, C, (size_t)S->P.n_species * S->n * sizeof(double));
  S->have_forces = 0;
  S->lag_valid = 0;
}

/* force = pair + bonded (without the body term); any pointer may be NULL */
void orc_get_state(orc_sim *S, double *x, double *v, double *C, double *F_pair, double *F_bonded, double *Q) {
  if ((F_pair || F_bonded || Q) && !S->have_forces) orc_compute_forces(S, S->step);
  int ns = S->P.n_species;
  if (x) memcpy(x, S->x, 3 * S->n * sizeof(double));
  if (v) memcpy(v, S->v, 3 * S->n * sizeof(double));
  if (C) memcpy(C, S->C, (size_t)ns * S->n * sizeof(double));
  if (F_pair) memcpy(F_pair, S->F, 3 * S->n * sizeof(double));
  if (F_bonded) memcpy(F_bonded, S->Fb, 3 * S->n * sizeof(double));
  if (Q) memcpy(Q, S->Q, (size_t)ns * S->n * sizeof(double));
}

void orc_get_census_totals(const orc_sim *S, int64_t out[3]) {
  out[0] = S->n_cand; out[1] = S->n_cc; out[2] = S->n_c;
}

void orc_get_rbc_stats(const orc_sim *S, double *area, double *volume, double *A0, double *V0) {
  for (int m = 0; m < S->n_rbc; ++m) {
    if (area) area[m] = S->rbcs[m].area;
    if (volume) volume[m] = S->rbcs[m].volume;
    if (A0) A0[m] = S->rbcs[m].A0;
    if (V0) V0[m] = S->rbcs[m].V0;
  }
}

int32_t orc_rbc_topology(const orc_sim *S, int32_t m, int32_t *nbond, int32_t *bond, int32_t *dih, double *h0,
                         double *kp, double *A0t) {
  const orc_rbc *R = &S->rbcs[m];
  *nbond = R->nbond;
  if (bond) memcpy(bond, R->bond, 2 * R->nbond * sizeof(int32_t));
  if (dih) memcpy(dih, R->dih, 4 * R->ndih * sizeof(int32_t));
  if (h0) memcpy(h0, R->h0, R->nbond * sizeof(double));
  if (kp) memcpy(kp, R->kp, R->nbond * sizeof(double));
  if (A0t) memcpy(A0t, R->A0t, R->ntri * sizeof(double));
  return R->ntri;
}

void orc_destroy(orc_sim *S) {
  if (!S) return;
  for (int m = 0; m < S->n_rbc; ++m) {
    orc_rbc *R = &S->rbcs[m];
    free(R->tri); free(R->bond); free(R->dih); free(R->h0); free(R->kp); free(R->A0t);
  }
  free(S->rbcs); free(S->x); free(S->v); free(S->C); free(S->F); free(S->Fb); free(S->g); free(S->Q);
  free(S->type); free(S->rbc); free(S);
}

/* ------------------------------------------------------------------------------------------
 * Binning rule of the bit-exact indexing test.  Defined in
 * fp32: n_a = floor(L_a / r_cc) (double, from the fp32 parameter values), inv_a = (float)(n_a / L_a),
 * x_w = x (+-L if outside [0,L)), c_a = min(n_a - 1, (int)floorf(x_w * inv_a)), one rounded multiply.
 * ------------------------------------------------------------------------------------------ */
void orc_bin_fp32(const float box[3], float r_cc, int64_t n, const float *pos, int32_t *cell_xyz, int32_t ncell[3]) {
  float inv[3];
  for (int a = 0; a < 3; ++a) {
    ncell[a] = (int32_t)floor((double)box[a] / (double)r_cc);
    inv[a] = (float)((double)ncell[a] / (double)box[a]);
  }
  for (int64_t i = 0; i < n; ++i)
    for (int a = 0; a < 3; ++a) {
      volatile float x = pos[3 * i + a];
      if (x >= box[a]) x = x - box[a];
      if (x < 0.0f) x = x + box[a];
      volatile float t = x * inv[a]; /* volatile: forbid contraction / excess precision */
      int32_t c = (int32_t)floorf(t);
      if (c > ncell[a] - 1) c = ncell[a] - 1;
      if (c < 0) c = 0;
      cell_xyz[3 * i + a] = c;
    }
}

/* Neighbour census from the CURRENT positions (exact fp64 arithmetic on whatever was loaded): per
 * particle the number of neighbours within r_c and r_cc, the XOR of their ids, and the smallest
 * |r - cutoff| over all candidate pairs (so a test can set aside borderline pairs).  Same-membrane
 * pairs are excluded exactly as in the force sum. */
void orc_neighbor_census(orc_sim *S, int32_t *n_rc, int32_t *n_rcc, uint32_t *xor_rc, uint32_t *xor_rcc,
                         double *margin) {
  const orc_params *P = &S->P;
  int64_t n = S->n;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    int32_t a = 0, b = 0; uint32_t xa = 0, xb = 0; double mg = 1e30;
    for (int64_t j = 0; j < n; ++j) {
      if (j == i || same_membrane(S, i, j)) continue;
      double d[3];
      for (int k = 0; k < 3; ++k) d[k] = min_image(S->x[3 * i + k] - S->x[3 * j + k], P->box[k]);
      double r2 = dot(d, d);
      double rmax = P->r_c > P->r_cc ? P->r_c : P->r_cc;
      if (r2 > 4.0 * rmax * rmax) continue; /* far beyond both cutoffs: irrelevant to counts and margin */
      double r = sqrt(r2);
      if (r2 >= 1e-12) {
        if (r < P->r_c) { ++a; xa ^= (uint32_t)j; }
        if (r < P->r_cc) { ++b; xb ^= (uint32_t)j; }
      }
      if (fabs(r - P->r_c) < mg) mg = fabs(r - P->r_c);
      if (fabs(r - P->r_cc) < mg) mg = fabs(r - P->r_cc);
    }
    n_rc[i] = a; n_rcc[i] = b; xor_rc[i] = xa; xor_rcc[i] = xb; margin[i] = mg;
  }
}

int32_t orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_threads(int32_t n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}
