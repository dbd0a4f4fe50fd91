/*
 * md_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the short-range MD hot path of
 * arXiv 1009.4330 (Trott, Winterfeld, Crozier) computes.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it.  It shares no code with the CUDA path
 * (paper_1009_4330_b200/csrc) and neither includes the other.
 *
 * Nature of the method: neighbor lists, cell binning,
 * thread-/block-per-atom kernels and spatial sorting are EXACT accelerations;
 * they reach the result of the plain definition up to summation order.  So
 * the oracle is the plain definition:
 *
 *   neighbor set  P = { {i,j} : i != j, |mi(x_i - x_j)|^2 < (rc+skin)^2 }
 *                 mi(d) = d - L*nearbyint(d/L) per component (minimum image;
 *                 what a periodic box means, "short range force")
 *   LJ 12-6       u(r) = 4 eps [(s/r)^12 - (s/r)^6], r^2 < rc^2, plain
 *                 truncation (App. A "lj/cut"; reading s2, s3)
 *   EAM           E = sum_i F(rho_i) + 1/2 sum_ij phi(r_ij), rho_i = sum_j rho(r_ij)
 *                 (App. A, refs 11,12; the functional form is
 *                 BASELINE.json cfg 4: phi = A exp(-p(r/r0-1)),
 *                 rho = exp(-q(r/r0-1)), F = -B sqrt(rho); reading s12, s13)
 *   tabulated EAM (SURVEY.md 8(f)-2 "then tabulated/spline EAM (what the paper's EAM run actually used)"; App. A
 *                 L260; reading s26): rho(r), phi(r) on a uniform grid r_k = k dr and F(rho) on rho_k = k drho, each
 *                 interpolated by the cubic Hermite polynomial of its interval with node slopes from centred differences
 *                 (4th order inside, 2nd order next to the ends, one-sided at the ends); the force uses the DERIVATIVE OF
 *                 THE INTERPOLANT, so it is the exact gradient of the interpolated energy.  Same E and F_i as analytic EAM.
 *   Buckingham + cutoff Coulomb (App. A, the "silicate (cutoff)" workload, LAMMPS
 *                 style buck/coul/cut named there): per type pair (a,b)
 *                 u(r) = A_ab exp(-r/rho_ab) - C_ab / r^6 + k q_a q_b / r,  r^2 < rc^2, plain truncation of all three
 *                 terms at one cutoff; charges per TYPE (the paper's silicate has one charge per species).
 *   NVE           velocity Verlet ("NVE ... integrators"):
 *                 v += dt/2 f/m ftm2v; x += dt v; f = F(x); v += dt/2 f/m ftm2v
 *   NVT           ("NVE, NVT, and NPT integrators"; reading s25) one Nose-Hoover
 *                 thermostat: dv/dt = f/m - xi v, dxi/dt = G = (2 KE - g kT)/Q, deta/dt = xi, Q = g kT tau^2,
 *                 g = 3N - 3, integrated by the symmetric splitting  TH(dt/2) kick drift force kick TH(dt/2)  with
 *                 TH(h): xi += h/2 G(KE); s = exp(-xi h); v *= s; KE *= s^2; eta += xi h; xi += h/2 G(KE).
 *                 Conserved: H = KE + PE + Q xi^2 / 2 + g kT eta.
 *   neighbor list loop of PAPER.md L88-104 (TpA pseudo-code): for each i, for
 *                 jj < numneigh[i]: j = neighbors[i][jj]; cutoff test (L159);
 *                 ftmp += pair force; f[i] = ftmp      -- a FULL list.
 *   rebuild rule  rebuild iff max_i |x_i - x0_i|^2 > (skin/2)^2 (reading s4).
 *
 * Two independent routes are given for every quantity: an O(N^2) brute-force
 * double loop (the definition itself) and an O(N) cell-grid + Verlet-list route
 * (what the timed CPU baseline runs).  tests/ pins the brute-force route to
 * closed forms and checks the list route against it.
 *
 * Pins (tests/test_oracle_*.py): analytic LJ pair values, fcc lattice sums by
 * direct lattice-vector enumeration, finite-difference forces and virial,
 * Newton's third law, time reversal, dt^2 energy-error scaling, brute force
 * vs list route.  No function here is "parity unpinned".
 *
 * Layout: positions/velocities/forces are N x 3 AoS doubles.  Virial order is
 * xx,yy,zz,xy,xz,yz with W_ab = sum_{i<j} D_a f_b, D = mi(x_i-x_j), f = force
 * on i from j.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PAIR_LJ 1
#define ORC_PAIR_EAM 2
#define ORC_PAIR_BUCK_COUL 3
#define ORC_PAIR_EAM_TAB 4

typedef struct {
  int style;        /* ORC_PAIR_LJ, ORC_PAIR_EAM or ORC_PAIR_BUCK_COUL */
  double p[5];      /* LJ: eps, sigma ; EAM: A, p, B, q, r0 ; BUCK_COUL: k (the Coulomb constant, e.g. 14.399645 eV A / e^2) */
  double rc;
  /* ORC_PAIR_BUCK_COUL only (NULL / 0 otherwise) */
  const int32_t* type;   /* [N] type of every atom, 0..ntypes-1 */
  int ntypes;
  const double* coef;    /* [ntypes][ntypes][3]: A, rho, C of the type pair (symmetric) */
  const double* qtype;   /* [ntypes] charge of a type */
  /* ORC_PAIR_EAM_TAB only: tables on uniform grids starting at 0 */
  int nr, nrho;
  double dr, drho;
  const double* tab_rho;  /* [nr]  rho(k dr) */
  const double* tab_phi;  /* [nr]  phi(k dr) */
  const double* tab_F;    /* [nrho] F(k drho) */
} orc_pair;
#define IS_EAM(P) ((P)->style == ORC_PAIR_EAM || (P)->style == ORC_PAIR_EAM_TAB)

int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

static double min_image(double d, double L) { return d - L * nearbyint(d / L); }

/* ---- pair functions ------------------------------------------------------ */

/* LJ 12-6: returns u(r) and fpair = -(1/r) du/dr, so that F_i = fpair * D. */
static void lj_pair(const orc_pair* P, double r2, double* u, double* fpair) {
  double eps = P->p[0], sigma = P->p[1];
  double s2 = sigma * sigma / r2;
  double s6 = s2 * s2 * s2;
  *u = 4.0 * eps * (s6 * s6 - s6);
  *fpair = 24.0 * eps * (2.0 * s6 * s6 - s6) / r2;
}

/* Buckingham + cutoff Coulomb for the type pair (ta, tb): u and fpair = -(1/r) du/dr.
 * du/dr = -(A/rho) exp(-r/rho) + 6 C / r^7 - k qa qb / r^2. */
static void buck_coul_pair(const orc_pair* P, int ta, int tb, double r2, double* u, double* fpair) {
  const double* c = P->coef + 3 * ((size_t)ta * P->ntypes + tb);
  double A = c[0], rho = c[1], C = c[2], kqq = P->p[0] * P->qtype[ta] * P->qtype[tb];
  double r = sqrt(r2), r6 = r2 * r2 * r2;
  double ex = A * exp(-r / rho);
  *u = ex - C / r6 + kqq / r;
  *fpair = (ex / rho - 6.0 * C / (r6 * r) + kqq / r2) / r;
}

/* the pairwise (non-EAM) styles: one term of atoms i and j */
static void lj_pair(const orc_pair* P, double r2, double* u, double* fpair);
static void pairwise(const orc_pair* P, int64_t i, int64_t j, double r2, double* u, double* fpair) {
  if (P->style == ORC_PAIR_BUCK_COUL) buck_coul_pair(P, P->type[i], P->type[j], r2, u, fpair);
  else lj_pair(P, r2, u, fpair);
}

/* Tabulated functions (header; reading s26): node slope by centred differences, cubic Hermite inside the interval.
 * Returns the value, *dy the derivative with respect to x. */
static double tab_slope(const double* y, int n, double h, int k) {
  if (k <= 0) return (y[1] - y[0]) / h;
  if (k >= n - 1) return (y[n - 1] - y[n - 2]) / h;
  if (k == 1 || k == n - 2) return (y[k + 1] - y[k - 1]) / (2.0 * h);
  return (y[k - 2] - 8.0 * y[k - 1] + 8.0 * y[k + 1] - y[k + 2]) / (12.0 * h);
}
static double tab_eval(const double* y, int n, double h, double x, double* dy) {
  int k = (int)floor(x / h);
  if (k < 0) k = 0;
  if (k > n - 2) k = n - 2;
  double u = x / h - (double)k;
  double y0 = y[k], D = y[k + 1] - y[k], m0 = h * tab_slope(y, n, h, k), m1 = h * tab_slope(y, n, h, k + 1);
  double c2 = 3.0 * D - 2.0 * m0 - m1, c3 = -2.0 * D + m0 + m1;
  if (dy) *dy = (m0 + u * (2.0 * c2 + 3.0 * c3 * u)) / h;
  return y0 + u * (m0 + u * (c2 + c3 * u));
}

/* EAM pieces (BASELINE.json cfg 4); the tabulated style evaluates its tables instead. */
static double eam_phi(const orc_pair* P, double r) {
  if (P->style == ORC_PAIR_EAM_TAB) return tab_eval(P->tab_phi, P->nr, P->dr, r, NULL);
  return P->p[0] * exp(-P->p[1] * (r / P->p[4] - 1.0));
}
static double eam_dphi(const orc_pair* P, double r) {
  if (P->style == ORC_PAIR_EAM_TAB) { double d; tab_eval(P->tab_phi, P->nr, P->dr, r, &d); return d; }
  return -(P->p[1] / P->p[4]) * eam_phi(P, r);
}
static double eam_rho(const orc_pair* P, double r) {
  if (P->style == ORC_PAIR_EAM_TAB) return tab_eval(P->tab_rho, P->nr, P->dr, r, NULL);
  return exp(-P->p[3] * (r / P->p[4] - 1.0));
}
static double eam_drho(const orc_pair* P, double r) {
  if (P->style == ORC_PAIR_EAM_TAB) { double d; tab_eval(P->tab_rho, P->nr, P->dr, r, &d); return d; }
  return -(P->p[3] / P->p[4]) * eam_rho(P, r);
}
static double eam_F(const orc_pair* P, double rho) {
  if (P->style == ORC_PAIR_EAM_TAB) return tab_eval(P->tab_F, P->nrho, P->drho, rho, NULL);
  return rho > 0.0 ? -P->p[2] * sqrt(rho) : 0.0;
}
/* F'(0) := 0 (reading s13) */
static double eam_dF(const orc_pair* P, double rho) {
  if (P->style == ORC_PAIR_EAM_TAB) { double d; tab_eval(P->tab_F, P->nrho, P->drho, rho, &d); return d; }
  return rho > 0.0 ? -P->p[2] / (2.0 * sqrt(rho)) : 0.0;
}

static void zero(double* a, int64_t n) { for (int64_t k = 0; k < n; ++k) a[k] = 0.0; }

static void add_virial(double* W, const double D[3], double fp) {
  W[0] += D[0] * D[0] * fp; W[1] += D[1] * D[1] * fp; W[2] += D[2] * D[2] * fp;
  W[3] += D[0] * D[1] * fp; W[4] += D[0] * D[2] * fp; W[5] += D[1] * D[2] * fp;
}

/* ---- O(N^2) brute force: the definition itself ---------------------------- */

/* All unordered pairs i<j with |mi(x_i-x_j)|^2 < rcut^2.  Returns the number
 * found; writes at most cap of them.  r2out may be NULL. */
int64_t orc_pairs_brute(int64_t N, const double* x, const double* box, double rcut,
                        int32_t* pi, int32_t* pj, double* r2out, int64_t cap) {
  int64_t n = 0;
  double rc2 = rcut * rcut;
  for (int64_t i = 0; i < N; ++i)
    for (int64_t j = i + 1; j < N; ++j) {
      double r2 = 0.0;
      for (int a = 0; a < 3; ++a) { double d = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += d * d; }
      if (r2 < rc2) {
        if (n < cap) { pi[n] = (int32_t)i; pj[n] = (int32_t)j; if (r2out) r2out[n] = r2; }
        ++n;
      }
    }
  return n;
}

/* Forces f[N*3], energy E, virial W[6], number of in-cutoff pairs, by the
 * double loop over i<j.  rho_out (EAM only) may be NULL. */
void orc_forces_brute(int64_t N, const double* x, const double* box, const orc_pair* P,
                      double* f, double* E, double* W, int64_t* npairs, double* rho_out) {
  double rc2 = P->rc * P->rc, e = 0.0, w[6] = {0, 0, 0, 0, 0, 0};
  int64_t np = 0;
  zero(f, 3 * N);
  if (!IS_EAM(P)) {
    for (int64_t i = 0; i < N; ++i)
      for (int64_t j = i + 1; j < N; ++j) {
        double D[3], r2 = 0.0;
        for (int a = 0; a < 3; ++a) { D[a] = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += D[a] * D[a]; }
        if (r2 < rc2) {
          double u, fp;
          pairwise(P, i, j, r2, &u, &fp);
          for (int a = 0; a < 3; ++a) { f[3 * i + a] += fp * D[a]; f[3 * j + a] -= fp * D[a]; }
          e += u; add_virial(w, D, fp); ++np;
        }
      }
  } else {
    double* rho = (double*)calloc(N > 0 ? (size_t)N : 1, sizeof(double));
    for (int64_t i = 0; i < N; ++i)
      for (int64_t j = i + 1; j < N; ++j) {
        double r2 = 0.0;
        for (int a = 0; a < 3; ++a) { double d = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += d * d; }
        if (r2 < rc2) { double r = sqrt(r2), g = eam_rho(P, r); rho[i] += g; rho[j] += g; }
      }
    for (int64_t i = 0; i < N; ++i) e += eam_F(P, rho[i]);
    for (int64_t i = 0; i < N; ++i)
      for (int64_t j = i + 1; j < N; ++j) {
        double D[3], r2 = 0.0;
        for (int a = 0; a < 3; ++a) { D[a] = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += D[a] * D[a]; }
        if (r2 < rc2) {
          double r = sqrt(r2);
          /* F_i = -sum_j [ (F'(rho_i)+F'(rho_j)) rho'(r) + phi'(r) ] D / r */
          double fp = -((eam_dF(P, rho[i]) + eam_dF(P, rho[j])) * eam_drho(P, r) + eam_dphi(P, r)) / r;
          for (int a = 0; a < 3; ++a) { f[3 * i + a] += fp * D[a]; f[3 * j + a] -= fp * D[a]; }
          e += eam_phi(P, r); add_virial(w, D, fp); ++np;
        }
      }
    if (rho_out) memcpy(rho_out, rho, (size_t)N * sizeof(double));
    free(rho);
  }
  if (E) *E = e;
  if (W) memcpy(W, w, sizeof w);
  if (npairs) *npairs = np;
}

/* Force on (and per-atom energy share of) a few sampled atoms, each by a full
 * O(N) scan over every other atom: usable at any N.  e_out[s] is the atom's
 * share: 1/2 sum_j u (LJ) or F(rho_i) + 1/2 sum_j phi (EAM). */
void orc_forces_sample(int64_t N, const double* x, const double* box, const orc_pair* P,
                       int64_t ns, const int64_t* ids, double* f_out, double* e_out) {
  double rc2 = P->rc * P->rc;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t s = 0; s < ns; ++s) {
    int64_t i = ids[s];
    double fi[3] = {0, 0, 0}, e = 0.0;
    if (!IS_EAM(P)) {
      for (int64_t j = 0; j < N; ++j) {
        if (j == i) continue;
        double D[3], r2 = 0.0;
        for (int a = 0; a < 3; ++a) { D[a] = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += D[a] * D[a]; }
        if (r2 < rc2) { double u, fp; pairwise(P, i, j, r2, &u, &fp); for (int a = 0; a < 3; ++a) fi[a] += fp * D[a]; e += 0.5 * u; }
      }
    } else {
      double rho_i = 0.0;
      for (int64_t j = 0; j < N; ++j) {
        if (j == i) continue;
        double r2 = 0.0;
        for (int a = 0; a < 3; ++a) { double d = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += d * d; }
        if (r2 < rc2) rho_i += eam_rho(P, sqrt(r2));
      }
      e = eam_F(P, rho_i);
      for (int64_t j = 0; j < N; ++j) {
        if (j == i) continue;
        double D[3], r2 = 0.0;
        for (int a = 0; a < 3; ++a) { D[a] = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += D[a] * D[a]; }
        if (r2 < rc2) {
          double rho_j = 0.0;
          for (int64_t k = 0; k < N; ++k) {
            if (k == j) continue;
            double q2 = 0.0;
            for (int a = 0; a < 3; ++a) { double d = min_image(x[3 * j + a] - x[3 * k + a], box[a]); q2 += d * d; }
            if (q2 < rc2) rho_j += eam_rho(P, sqrt(q2));
          }
          double r = sqrt(r2);
          double fp = -((eam_dF(P, rho_i) + eam_dF(P, rho_j)) * eam_drho(P, r) + eam_dphi(P, r)) / r;
          for (int a = 0; a < 3; ++a) fi[a] += fp * D[a];
          e += 0.5 * eam_phi(P, r);
        }
      }
    }
    for (int a = 0; a < 3; ++a) f_out[3 * s + a] = fi[a];
    if (e_out) e_out[s] = e;
  }
}

/* Neighbors of a few sampled atoms by a full scan; row s gets at most stride
 * ids (ascending); count[s] is the true count. */
void orc_neighbors_sample(int64_t N, const double* x, const double* box, double rcut,
                          int64_t ns, const int64_t* ids, int32_t* count, int32_t* neigh, int64_t stride) {
  double rc2 = rcut * rcut;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t s = 0; s < ns; ++s) {
    int64_t i = ids[s];
    int32_t n = 0;
    for (int64_t j = 0; j < N; ++j) {
      if (j == i) continue;
      double r2 = 0.0;
      for (int a = 0; a < 3; ++a) { double d = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += d * d; }
      if (r2 < rc2) { if (n < stride) neigh[s * stride + n] = (int32_t)j; ++n; }
    }
    count[s] = n;
  }
}

/* ---- O(N) route: cell grid + full Verlet list ----------- */

typedef struct {
  int64_t N;
  int64_t* start;   /* N+1 row offsets (CSR) */
  int32_t* idx;     /* neighbor ids */
  int64_t cap;
} orc_list;

void orc_list_free(orc_list* l) { if (l) { free(l->start); free(l->idx); free(l); } }
int64_t orc_list_total(const orc_list* l) { return l->start[l->N]; }
void orc_list_export(const orc_list* l, int64_t* start, int32_t* idx) {
  memcpy(start, l->start, (size_t)(l->N + 1) * sizeof(int64_t));
  memcpy(idx, l->idx, (size_t)l->start[l->N] * sizeof(int32_t));
}

/* Full list: every j != i with |mi(x_i-x_j)|^2 < rl^2, found through a grid of
 * cells of edge >= rl (27-cell stencil, periodic).  Needs box >= 3 rl per
 * dimension (reading s19); returns NULL otherwise.  Positions need not be
 * wrapped: the cell index wraps them. */
orc_list* orc_list_build(int64_t N, const double* x, const double* box, double rl) {
  int nc[3];
  for (int a = 0; a < 3; ++a) { nc[a] = (int)floor(box[a] / rl); if (nc[a] < 3) return NULL; }
  int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
  int64_t* head = (int64_t*)malloc((size_t)(ncell + 1) * sizeof(int64_t));
  int64_t* cell_of = (int64_t*)malloc((size_t)N * sizeof(int64_t));
  int64_t* order = (int64_t*)malloc((size_t)N * sizeof(int64_t));
  for (int64_t c = 0; c <= ncell; ++c) head[c] = 0;
  for (int64_t i = 0; i < N; ++i) {
    int ci[3];
    for (int a = 0; a < 3; ++a) {
      double xw = x[3 * i + a] - box[a] * floor(x[3 * i + a] / box[a]);
      ci[a] = (int)floor(xw / box[a] * nc[a]);
      if (ci[a] >= nc[a]) ci[a] = nc[a] - 1;
      if (ci[a] < 0) ci[a] = 0;
    }
    cell_of[i] = ((int64_t)ci[2] * nc[1] + ci[1]) * nc[0] + ci[0];
    head[cell_of[i] + 1]++;
  }
  for (int64_t c = 0; c < ncell; ++c) head[c + 1] += head[c];
  {
    int64_t* fill = (int64_t*)malloc((size_t)ncell * sizeof(int64_t));
    memcpy(fill, head, (size_t)ncell * sizeof(int64_t));
    for (int64_t i = 0; i < N; ++i) order[fill[cell_of[i]]++] = i;
    free(fill);
  }
  orc_list* l = (orc_list*)malloc(sizeof(orc_list));
  l->N = N;
  l->start = (int64_t*)malloc((size_t)(N + 1) * sizeof(int64_t));
  int32_t* cnt = (int32_t*)malloc((size_t)N * sizeof(int32_t));
  double rl2 = rl * rl;
  for (int pass = 0; pass < 2; ++pass) {
    if (pass == 1) {
      l->start[0] = 0;
      for (int64_t i = 0; i < N; ++i) l->start[i + 1] = l->start[i] + cnt[i];
      l->cap = l->start[N];
      l->idx = (int32_t*)malloc((size_t)(l->cap > 0 ? l->cap : 1) * sizeof(int32_t));
    }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i) {
      int64_t c = cell_of[i];
      int cx = (int)(c % nc[0]), cy = (int)((c / nc[0]) % nc[1]), cz = (int)(c / ((int64_t)nc[0] * nc[1]));
      int32_t n = 0;
      for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
          for (int dx = -1; dx <= 1; ++dx) {
            int ox = (cx + dx + nc[0]) % nc[0], oy = (cy + dy + nc[1]) % nc[1], oz = (cz + dz + nc[2]) % nc[2];
            int64_t oc = ((int64_t)oz * nc[1] + oy) * nc[0] + ox;
            for (int64_t k = head[oc]; k < head[oc + 1]; ++k) {
              int64_t j = order[k];
              if (j == i) continue;
              double r2 = 0.0;
              for (int a = 0; a < 3; ++a) { double d = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += d * d; }
              if (r2 < rl2) { if (pass == 1) l->idx[l->start[i] + n] = (int32_t)j; ++n; }
            }
          }
      cnt[i] = n;
    }
  }
  free(cnt); free(head); free(cell_of); free(order);
  return l;
}

/* Forces through the full list: the loop of PAPER.md L88-104, one row per atom,
 * writes only f[i].  Each pair is visited twice, so energy and virial take 1/2. */
void orc_forces_list(int64_t N, const double* x, const double* box, const orc_pair* P, const orc_list* l,
                     double* f, double* E, double* W, int64_t* npairs, double* rho_out) {
  double rc2 = P->rc * P->rc, e = 0.0, w0 = 0, w1 = 0, w2 = 0, w3 = 0, w4 = 0, w5 = 0;
  int64_t np2 = 0;
  double* dF = NULL;
  if (IS_EAM(P)) {
    double* rho = (double*)malloc((size_t)N * sizeof(double));
    dF = (double*)malloc((size_t)N * sizeof(double));
#pragma omp parallel for schedule(static) reduction(+ : e)
    for (int64_t i = 0; i < N; ++i) {
      double r_i = 0.0;
      for (int64_t k = l->start[i]; k < l->start[i + 1]; ++k) {
        int64_t j = l->idx[k];
        double r2 = 0.0;
        for (int a = 0; a < 3; ++a) { double d = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += d * d; }
        if (r2 < rc2) r_i += eam_rho(P, sqrt(r2));
      }
      rho[i] = r_i; dF[i] = eam_dF(P, r_i); e += eam_F(P, r_i);
    }
    if (rho_out) memcpy(rho_out, rho, (size_t)N * sizeof(double));
    free(rho);
  }
#pragma omp parallel for schedule(static) reduction(+ : e, w0, w1, w2, w3, w4, w5, np2)
  for (int64_t i = 0; i < N; ++i) {
    double ftmp[3] = {0, 0, 0};
    for (int64_t k = l->start[i]; k < l->start[i + 1]; ++k) {
      int64_t j = l->idx[k];
      double D[3], r2 = 0.0;
      for (int a = 0; a < 3; ++a) { D[a] = min_image(x[3 * i + a] - x[3 * j + a], box[a]); r2 += D[a] * D[a]; }
      if (r2 < rc2) {
        double u, fp;
        if (!IS_EAM(P)) pairwise(P, i, j, r2, &u, &fp);
        else { double r = sqrt(r2); u = eam_phi(P, r); fp = -((dF[i] + dF[j]) * eam_drho(P, r) + eam_dphi(P, r)) / r; }
        for (int a = 0; a < 3; ++a) ftmp[a] += fp * D[a];
        e += 0.5 * u;
        w0 += 0.5 * D[0] * D[0] * fp; w1 += 0.5 * D[1] * D[1] * fp; w2 += 0.5 * D[2] * D[2] * fp;
        w3 += 0.5 * D[0] * D[1] * fp; w4 += 0.5 * D[0] * D[2] * fp; w5 += 0.5 * D[1] * D[2] * fp;
        ++np2;
      }
    }
    for (int a = 0; a < 3; ++a) f[3 * i + a] = ftmp[a];
  }
  free(dF);
  if (E) *E = e;
  if (W) { W[0] = w0; W[1] = w1; W[2] = w2; W[3] = w3; W[4] = w4; W[5] = w5; }
  if (npairs) *npairs = np2 / 2;
}

/* ---- velocity-Verlet NVE with displacement-triggered rebuilds -------------- */

/* Advances x, v in place by nsteps.  mass is per atom.  f holds F(x) of the
 * final positions on return.  pe_trace/ke_trace (nsteps+1 entries, may be NULL)
 * receive potential and kinetic energy at steps 0..nsteps (ke = 1/2 sum m v^2
 * mvv2e).  Returns the number of list builds (including the first), or -1 if
 * the box is too small. */
int64_t orc_run_nve(int64_t N, double* x, double* v, double* f, const double* box, const double* mass,
                    const orc_pair* P, double skin, double dt, int64_t nsteps, double ftm2v, double mvv2e,
                    double* pe_trace, double* ke_trace) {
  double rl = P->rc + skin, trigger = 0.25 * skin * skin;
  double* x0 = (double*)malloc((size_t)(3 * N) * sizeof(double));
  for (int64_t i = 0; i < N; ++i)
    for (int a = 0; a < 3; ++a) x[3 * i + a] -= box[a] * floor(x[3 * i + a] / box[a]);
  orc_list* l = orc_list_build(N, x, box, rl);
  if (!l) { free(x0); return -1; }
  memcpy(x0, x, (size_t)(3 * N) * sizeof(double));
  int64_t nbuild = 1;
  double pe;
  orc_forces_list(N, x, box, P, l, f, &pe, NULL, NULL, NULL);
  for (int64_t step = 0;; ++step) {
    if (pe_trace) pe_trace[step] = pe;
    if (ke_trace) {
      double ke = 0.0;
      for (int64_t i = 0; i < N; ++i) ke += 0.5 * mass[i] * (v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2]);
      ke_trace[step] = ke * mvv2e;
    }
    if (step == nsteps) break;
    double dmax = 0.0;
#pragma omp parallel for schedule(static) reduction(max : dmax)
    for (int64_t i = 0; i < N; ++i) {
      double dtf = 0.5 * dt * ftm2v / mass[i], d2 = 0.0;
      for (int a = 0; a < 3; ++a) {
        v[3 * i + a] += dtf * f[3 * i + a];
        x[3 * i + a] += dt * v[3 * i + a];
        double d = x[3 * i + a] - x0[3 * i + a];
        d2 += d * d;
      }
      if (d2 > dmax) dmax = d2;
    }
    if (dmax > trigger) {
      for (int64_t i = 0; i < N; ++i)
        for (int a = 0; a < 3; ++a) x[3 * i + a] -= box[a] * floor(x[3 * i + a] / box[a]);
      orc_list_free(l);
      l = orc_list_build(N, x, box, rl);
      memcpy(x0, x, (size_t)(3 * N) * sizeof(double));
      ++nbuild;
    }
    orc_forces_list(N, x, box, P, l, f, (pe_trace ? &pe : NULL), NULL, NULL, NULL);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i) {
      double dtf = 0.5 * dt * ftm2v / mass[i];
      for (int a = 0; a < 3; ++a) v[3 * i + a] += dtf * f[3 * i + a];
    }
  }
  orc_list_free(l);
  free(x0);
  return nbuild;
}

/* ---- NVT: velocity Verlet with one Nose-Hoover thermostat (header comment; reading s25) ------------------ */

static double kinetic(int64_t N, const double* v, const double* mass, double mvv2e) {
  double ke = 0.0;
  for (int64_t i = 0; i < N; ++i) ke += 0.5 * mass[i] * (v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2]);
  return ke * mvv2e;
}

/* TH(h): returns the velocity scale factor; updates xi, eta and KE */
static double thermostat_half(double* xi, double* eta, double* ke, double h, double gkT, double Q) {
  *xi += 0.5 * h * (2.0 * *ke - gkT) / Q;
  double sc = exp(-*xi * h);
  *ke *= sc * sc;
  *eta += *xi * h;
  *xi += 0.5 * h * (2.0 * *ke - gkT) / Q;
  return sc;
}

/* nsteps of NVT from (x, v) with thermostat state thermo[2] = {xi, eta} (in/out).  kT and tau in the caller's energy
 * and time units.  h_trace[nsteps+1] (may be NULL): the conserved quantity at every whole step.  Returns the number of
 * list builds, -1 if the box is too small.  Same list route and rebuild rule as orc_run_nve. */
int64_t orc_run_nvt(int64_t N, double* x, double* v, double* f, const double* box, const double* mass,
                    const orc_pair* P, double skin, double dt, int64_t nsteps, double ftm2v, double mvv2e,
                    double kT, double tau, double* thermo, double* h_trace, double* ke_trace) {
  double rl = P->rc + skin, trigger = 0.25 * skin * skin;
  double gkT = (3.0 * (double)N - 3.0) * kT, Q = gkT * tau * tau;
  double* x0 = (double*)malloc((size_t)(3 * N) * sizeof(double));
  for (int64_t i = 0; i < N; ++i)
    for (int a = 0; a < 3; ++a) x[3 * i + a] -= box[a] * floor(x[3 * i + a] / box[a]);
  orc_list* l = orc_list_build(N, x, box, rl);
  if (!l) { free(x0); return -1; }
  memcpy(x0, x, (size_t)(3 * N) * sizeof(double));
  int64_t nbuild = 1;
  double pe, xi = thermo[0], eta = thermo[1];
  orc_forces_list(N, x, box, P, l, f, &pe, NULL, NULL, NULL);
  for (int64_t step = 0;; ++step) {
    double ke = kinetic(N, v, mass, mvv2e);
    if (h_trace) h_trace[step] = ke + pe + 0.5 * Q * xi * xi + gkT * eta;
    if (ke_trace) ke_trace[step] = ke;
    if (step == nsteps) break;
    double sc = thermostat_half(&xi, &eta, &ke, 0.5 * dt, gkT, Q);
    double dmax = 0.0;
    for (int64_t i = 0; i < N; ++i) {
      double dtf = 0.5 * dt * ftm2v / mass[i], d2 = 0.0;
      for (int a = 0; a < 3; ++a) {
        v[3 * i + a] = sc * v[3 * i + a] + dtf * f[3 * i + a];
        x[3 * i + a] += dt * v[3 * i + a];
        double d = x[3 * i + a] - x0[3 * i + a];
        d2 += d * d;
      }
      if (d2 > dmax) dmax = d2;
    }
    if (dmax > trigger) {
      for (int64_t i = 0; i < N; ++i)
        for (int a = 0; a < 3; ++a) x[3 * i + a] -= box[a] * floor(x[3 * i + a] / box[a]);
      orc_list_free(l);
      l = orc_list_build(N, x, box, rl);
      memcpy(x0, x, (size_t)(3 * N) * sizeof(double));
      ++nbuild;
    }
    orc_forces_list(N, x, box, P, l, f, &pe, NULL, NULL, NULL);
    for (int64_t i = 0; i < N; ++i) {
      double dtf = 0.5 * dt * ftm2v / mass[i];
      for (int a = 0; a < 3; ++a) v[3 * i + a] += dtf * f[3 * i + a];
    }
    ke = kinetic(N, v, mass, mvv2e);
    sc = thermostat_half(&xi, &eta, &ke, 0.5 * dt, gkT, Q);
    for (int64_t i = 0; i < 3 * N; ++i) v[i] *= sc;
  }
  thermo[0] = xi; thermo[1] = eta;
  orc_list_free(l);
  free(x0);
  return nbuild;
}
