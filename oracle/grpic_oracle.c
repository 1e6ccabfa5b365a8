/*
 * grpic_oracle.c — TEST INFRASTRUCTURE. NOT PART OF THE PRODUCT PATH.
 *
 * Plain, slow, scalar FP64 CPU statement of the per-particle GRPIC step of
 * arxiv/paper_2511_17701 ("Entity II: General Relativistic Module"), written
 * from the paper's equations only.  P:n below = PAPER.md line n.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code
 * with the CUDA path under paper_2511_17701_b200/csrc (no common header,
 * helper, table or constant generator).
 *
 * What it computes, in the paper's order (Sec. 3.1 steps 1-11):
 *   orc_metric        Kerr-Schild 3+1 quantities in the code basis
 *   orc_dmetric       analytic derivatives d/dx1, d/dx2
 *   orc_*_tetrad      orthonormal-frame transforms
 *   orc_interp        Yee-staggered D,B -> particle (reading R-S4)
 *   orc_boris_half    tetrad-frame Boris half push                     P:230, P:182 (Eq. 19)
 *   orc_geodesic_u    Eq. 26-27, n_iter fixed-point iterations
 *   orc_geodesic_x    Eq. 28-29, n_iter fixed-point iterations
 *   phi update        Eq. 30
 *   particle BCs      axis reflection, radial removal
 *   orc_deposit       conformal charge-conserving deposit (R-S10)
 *
 * Readings of silent/garbled passages are listed in DESIGN.md ("Readings").
 * Parity pins live in tests/test_oracle_*.py.  Functions whose *scheme choice*
 * has no independent pin (the paper defers to "paper I"):
 *   orc_interp   — parity unpinned as to the choice among first-order schemes
 *                  (pinned: exactness on constant/linear fields, partition of
 *                  unity, continuity across faces);
 *   orc_deposit  — parity unpinned as to the choice among charge-conserving
 *                  schemes (pinned: discrete continuity Eq. 32/34, first
 *                  moments, one-cell hand formula for J^1, J^2, and the four
 *                  node weights of J^3 of Eq. 36 written out by hand for a path
 *                  inside one cell and for one across a face).
 */
#define _USE_MATH_DEFINES
#ifndef _GNU_SOURCE
#define _GNU_SOURCE
#endif
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Operation count of this statement of the method: the same source compiled as C++ with -DORC_COUNT
 * runs on a counting stand-in for `double` (oracle/orc_count.hpp); ORC_STAGE marks the stage the operations that
 * follow belong to.  In the normal build the marks vanish and nothing else changes. */
#ifdef ORC_COUNT
#include "orc_count.hpp"
#define double orc_cnt
#else
#define ORC_STAGE(s) ((void)0)
#endif
enum { ORC_ST_INTERP = 0, ORC_ST_METRIC, ORC_ST_EM, ORC_ST_ULOOP, ORC_ST_XLOOP, ORC_ST_BC, ORC_ST_DEPOSIT, ORC_ST_OTHER };

typedef struct {
  int32_t n1, n2, ng;    /* N_r, N_theta, ghost width          */
  int32_t n_iter;        /* fixed iteration count of Eq. 26-29        */
  double a;              /* spin, r_g = M = 1                          */
  double r_min, r_max;   /* radial extent; log-r map A.3 with r0=0,h0=0 */
  double small_angle;    /* SMALL_ANGLE_GR                            */
  double r0;             /* radial offset of A.3: xi = log(r - r0)    */
  double h0;             /* polar stretch of A.3; 0 = uniform     */
  int32_t linear_r;      /* 1: spherical Kerr-Schild of A.2, r uniform in x1 (r0 unused) */
  double mass;           /* M in units of r_g: 1 everywhere in the paper's GR runs; 0 with a = 0 is the flat
                            spherical metric kerr_schild_0 of A.1: z = 0, alpha = 1, beta = 0          */
} orc_grid;

typedef struct {
  double r, th, sth, cth;
  double Sigma, Delta, A, z;
  double s1, s2;                     /* dr/dx1 = dxi*(r-r0), dtheta/dx2 = deta*dtheta/deta */
  double alpha, beta1;               /* lapse, shift beta^1 (code basis)      */
  double hu11, hu22, hu33, hu13;     /* h^{ij}                                */
  double hd11, hd22, hd33, hd13;     /* h_{ij}                                */
  double sqrt_h;
  double dls2;                       /* d ln(s2)/dx2: non-zero only with the polar stretch h0 (A.3) */
} orc_metric_t;

typedef struct {                     /* [0] = d/dx1, [1] = d/dx2              */
  double hu11[2], hu22[2], hu33[2], hu13[2], alpha[2], beta1[2];
} orc_dmetric_t;

static double orc_dxi(const orc_grid* g) { return log((g->r_max - g->r0) / (g->r_min - g->r0)) / g->n1; }
/* d ln(s1)/dx1: dxi for s1 = dxi e^xi (A.3), 0 for the constant s1 = dr of A.2 */
static double orc_dls1(const orc_grid* g) { return g->linear_r ? 0.0 : orc_dxi(g); }
static double orc_dr(const orc_grid* g) { return (g->r_max - g->r_min) / g->n1; }
static double orc_deta(const orc_grid* g) { return M_PI / g->n2; }

/* P:820-823 (A.3): xi = log(r - r0) uniform in x1;  eta = x2*deta uniform in x2 and
 *   theta = eta + 2 h0 eta (pi - 2 eta)(pi - eta)/pi^2,
 *   dtheta/deta = 1 + 2 h0 + 12 h0 (eta/pi)(eta/pi - 1)   (P:823 prints "12h" for 12 h0).
 * All five BASELINE configs have r0 = 0, h0 = 0.
 * theta used in any metric evaluation is kept away from the axis. */
static double orc_theta_of_eta(const orc_grid* g, double eta) {
  return eta + 2.0 * g->h0 * eta * (M_PI - 2.0 * eta) * (M_PI - eta) / (M_PI * M_PI);
}
static double orc_dtheta_deta(const orc_grid* g, double eta) {
  return 1.0 + 2.0 * g->h0 + 12.0 * g->h0 * (eta / M_PI) * (eta / M_PI - 1.0);
}
static void orc_coords(const orc_grid* g, double x1, double x2, double* r, double* th) {
  *r = g->linear_r ? g->r_min + x1 * orc_dr(g) : g->r0 + exp(log(g->r_min - g->r0) + x1 * orc_dxi(g));
  double t = orc_theta_of_eta(g, x2 * orc_deta(g));
  if (t < g->small_angle) t = g->small_angle;
  if (t > M_PI - g->small_angle) t = M_PI - g->small_angle;
  *th = t;
}

/* P:739-750 (A1-A2, lapse/shift) in the code basis of A.3 with
 * dxi*e^xi = s1, deta*(dtheta/deta) = s2, dphi = 1. */
void orc_metric(const orc_grid* g, double x1, double x2, orc_metric_t* m) {
  double r, th;
  orc_coords(g, x1, x2, &r, &th);
  const double a = g->a, M = g->mass;
  m->r = r; m->th = th;
  m->sth = sin(th); m->cth = cos(th);
  const double s2th = m->sth * m->sth;
  m->Sigma = r * r + a * a * m->cth * m->cth;
  m->Delta = r * r - 2.0 * M * r + a * a;
  m->A = (r * r + a * a) * (r * r + a * a) - a * a * m->Delta * s2th;
  m->z = 2.0 * M * r / m->Sigma;
  m->s1 = g->linear_r ? orc_dr(g) : orc_dxi(g) * (r - g->r0);
  m->s2 = orc_deta(g) * orc_dtheta_deta(g, x2 * orc_deta(g));
  {
    const double eta = x2 * orc_deta(g);
    m->dls2 = orc_deta(g) * (12.0 * g->h0 / M_PI) * (2.0 * eta / M_PI - 1.0) / orc_dtheta_deta(g, eta);
  }
  m->alpha = 1.0 / sqrt(1.0 + m->z);
  m->beta1 = m->z / (1.0 + m->z) / m->s1;
  m->hu11 = m->A / (m->Sigma * (m->Sigma + 2.0 * M * r)) / (m->s1 * m->s1);
  m->hu22 = 1.0 / m->Sigma / (m->s2 * m->s2);
  m->hu33 = 1.0 / (m->Sigma * s2th);
  m->hu13 = a / m->Sigma / m->s1;
  m->hd11 = m->s1 * m->s1 * (1.0 + m->z);
  m->hd22 = m->s2 * m->s2 * m->Sigma;
  m->hd33 = m->A * s2th / m->Sigma;
  m->hd13 = -m->s1 * a * (1.0 + m->z) * s2th;
  m->sqrt_h = m->s1 * m->s2 * m->Sigma * m->sth / m->alpha;
}

/* P:816 (A.2) with dr -> s1, dtheta -> s2, plus the A.3 terms that come from
 * s1 = dxi*e^xi depending on x1 (legible entries of P:842) and, with the polar
 * stretch, from s2 depending on x2 (h^22 ~ 1/s2^2: the entry P:842 omits).  Corrections to the
 * printed text (DESIGN.md R-S2): d_theta Sigma from P:774; sign of d_xi alpha
 * as in A.2. */
void orc_dmetric(const orc_grid* g, const orc_metric_t* m, orc_dmetric_t* d) {
  const double a = g->a, M = g->mass, r = m->r, S = m->Sigma, A = m->A;   /* M = 1: the printed A.2 list */
  const double s1 = m->s1, s2 = m->s2, dxi = orc_dls1(g);   /* the A.3 extras vanish on the A.2 map */
  const double sth = m->sth, cth = m->cth, s2th = sth * sth;
  const double d1S = 2.0 * r * s1;
  const double d2S = -2.0 * a * a * sth * cth * s2;
  const double d1D = 2.0 * (r - M) * s1;
  const double d1A = 4.0 * r * s1 * (r * r + a * a) - a * a * s2th * d1D;
  const double d2A = -2.0 * a * a * sth * cth * m->Delta * s2;
  const double den = S * S * (S + 2.0 * M * r) * (S + 2.0 * M * r);

  d->hu11[0] = (S * (S + 2.0 * M * r) * d1A - 2.0 * A * (M * r * d1S + S * (d1S + M * s1))) / den / (s1 * s1)
               - 2.0 * dxi * m->hu11;
  d->hu11[1] = (S * (S + 2.0 * M * r) * d2A - 2.0 * A * d2S * (M * r + S)) / den / (s1 * s1);
  d->hu22[0] = -d1S / (S * S) / (s2 * s2);
  d->hu22[1] = -d2S / (S * S) / (s2 * s2) - 2.0 * m->dls2 * m->hu22;   /* A.3: s2 depends on x2 */
  d->hu33[0] = -d1S / (S * S * s2th);
  d->hu33[1] = -2.0 * cth * s2 / (S * S * sth * s2th) * (S - a * a * s2th);
  d->hu13[0] = -a / s1 * d1S / (S * S) - dxi * m->hu13;
  d->hu13[1] = -a / s1 * d2S / (S * S);
  d->beta1[0] = 2.0 * M / s1 * (s1 * S - r * d1S) / ((S + 2.0 * M * r) * (S + 2.0 * M * r)) - dxi * m->beta1;
  d->beta1[1] = -2.0 * M / s1 * r * d2S / (S * S * (1.0 + m->z) * (1.0 + m->z));
  const double al3 = m->alpha * m->alpha * m->alpha;
  d->alpha[0] = -M * (s1 * S - r * d1S) / (S * S) * al3;
  d->alpha[1] = M * r * d2S / (S * S) * al3;
}

/* Tetrads, matrix form of P:754 (the explicit inverse formulas at P:766/770
 * drop square roots; DESIGN.md R-S3). */
void orc_cntrv_to_tetrad(const orc_metric_t* m, const double A[3], double Ah[3]) {
  Ah[0] = A[0] / sqrt(m->hu11);
  Ah[1] = sqrt(m->hd22) * A[1];
  Ah[2] = m->hd13 / sqrt(m->hd33) * A[0] + sqrt(m->hd33) * A[2];
}
void orc_cov_to_tetrad(const orc_metric_t* m, const double u[3], double uh[3]) {
  uh[0] = sqrt(m->hu11) * (u[0] - m->hd13 / m->hd33 * u[2]);
  uh[1] = u[1] / sqrt(m->hd22);
  uh[2] = u[2] / sqrt(m->hd33);
}
void orc_tetrad_to_cov(const orc_metric_t* m, const double uh[3], double u[3]) {
  u[0] = uh[0] / sqrt(m->hu11) + m->hd13 / sqrt(m->hd33) * uh[2];
  u[1] = sqrt(m->hd22) * uh[1];
  u[2] = sqrt(m->hd33) * uh[2];
}
void orc_tetrad_to_cntrv(const orc_metric_t* m, const double Ah[3], double A[3]) {
  A[0] = sqrt(m->hu11) * Ah[0];
  A[1] = Ah[1] / sqrt(m->hd22);
  A[2] = -m->hd13 * sqrt(m->hu11) / m->hd33 * Ah[0] + Ah[2] / sqrt(m->hd33);
}

/* Eq. 20: FIDO-measured energy. eps = 1 massive, 0 massless. */
static double orc_gamma(const orc_metric_t* m, const double u[3], double eps) {
  return sqrt(eps + m->hu11 * u[0] * u[0] + m->hu22 * u[1] * u[1] + m->hu33 * u[2] * u[2]
              + 2.0 * m->hu13 * u[0] * u[2]);
}

/* ------------------------------------------------------------------------
 * Field interpolation, step 2.  Reading R-S4: first-order shape in
 * two stages — (i) every staggered component is brought to the four corner
 * nodes of the particle's cell by averaging its nearest samples along each
 * half-offset axis; (ii) bilinear in (dx1,dx2).  Storage (Eq. 40-41 locations,
 * P:388-402), index [i1+G][i2+G], i2 fastest:
 *   D1(i+1/2,j) D2(i,j+1/2) D3(i,j)   B1(i,j+1/2) B2(i+1/2,j) B3(i+1/2,j+1/2)
 * ---------------------------------------------------------------------- */
typedef struct { const double *D1, *D2, *D3, *B1, *B2, *B3; } orc_fields;

static double f_at(const orc_grid* g, const double* F, int i, int j) {
  const int64_t ld = g->n2 + 2 * g->ng;
  return F[(int64_t)(i + g->ng) * ld + (j + g->ng)];
}
/* node value of a component staggered by half a cell along axis 1 only */
static double node_h1(const orc_grid* g, const double* F, int i, int j) {
  return 0.5 * (f_at(g, F, i - 1, j) + f_at(g, F, i, j));
}
static double node_h2(const orc_grid* g, const double* F, int i, int j) {
  return 0.5 * (f_at(g, F, i, j - 1) + f_at(g, F, i, j));
}
static double node_h12(const orc_grid* g, const double* F, int i, int j) {
  return 0.25 * (f_at(g, F, i - 1, j - 1) + f_at(g, F, i - 1, j) + f_at(g, F, i, j - 1) + f_at(g, F, i, j));
}
static double node_00(const orc_grid* g, const double* F, int i, int j) { return f_at(g, F, i, j); }

typedef double (*node_fn)(const orc_grid*, const double*, int, int);
static double bilinear(const orc_grid* g, const double* F, node_fn nf, int i, int j, double dx1, double dx2) {
  const double c00 = nf(g, F, i, j), c10 = nf(g, F, i + 1, j);
  const double c01 = nf(g, F, i, j + 1), c11 = nf(g, F, i + 1, j + 1);
  const double lo = c00 * (1.0 - dx1) + c10 * dx1;
  const double hi = c01 * (1.0 - dx1) + c11 * dx1;
  return lo * (1.0 - dx2) + hi * dx2;
}
void orc_interp(const orc_grid* g, const orc_fields* F, int i1, int i2, double dx1, double dx2,
                double D[3], double B[3]) {
  D[0] = bilinear(g, F->D1, node_h1, i1, i2, dx1, dx2);
  D[1] = bilinear(g, F->D2, node_h2, i1, i2, dx1, dx2);
  D[2] = bilinear(g, F->D3, node_00, i1, i2, dx1, dx2);
  B[0] = bilinear(g, F->B1, node_h2, i1, i2, dx1, dx2);
  B[1] = bilinear(g, F->B2, node_h1, i1, i2, dx1, dx2);
  B[2] = bilinear(g, F->B3, node_h12, i1, i2, dx1, dx2);
}

/* ------------------------------------------------------------------------
 * EM half push (steps 3-5 / 7-9): Boris rotation in the tetrad
 * frame over dt/2.  Reading R-S5: coefficient c = (q/m) * alpha * dt/4 — the
 * lapse multiplies the whole Lorentz force in Eq. 19.
 * ---------------------------------------------------------------------- */
static void orc_boris_half(const double Dh[3], const double Bh[3], double c, double uh[3]) {
  double um[3], t[3], s[3], up[3], upl[3];
  for (int k = 0; k < 3; ++k) um[k] = uh[k] + c * Dh[k];
  const double gm = sqrt(1.0 + um[0] * um[0] + um[1] * um[1] + um[2] * um[2]);
  for (int k = 0; k < 3; ++k) t[k] = c * Bh[k] / gm;
  const double t2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
  for (int k = 0; k < 3; ++k) s[k] = 2.0 * t[k] / (1.0 + t2);
  up[0] = um[0] + (um[1] * t[2] - um[2] * t[1]);
  up[1] = um[1] + (um[2] * t[0] - um[0] * t[2]);
  up[2] = um[2] + (um[0] * t[1] - um[1] * t[0]);
  upl[0] = um[0] + (up[1] * s[2] - up[2] * s[1]);
  upl[1] = um[1] + (up[2] * s[0] - up[0] * s[2]);
  upl[2] = um[2] + (up[0] * s[1] - up[1] * s[0]);
  for (int k = 0; k < 3; ++k) uh[k] = upl[k] + c * Dh[k];
}

/* Eq. 26-27: metric and derivatives frozen at x^(n);
 * exactly n_iter applications of the map, first guess u~ = u*; u_3 untouched. */
static void orc_geodesic_u(const orc_metric_t* m, const orc_dmetric_t* d, double eps, double dt,
                           int n_iter, double u[3]) {
  const double us[3] = {u[0], u[1], u[2]};
  double ut[3] = {u[0], u[1], u[2]};
  for (int it = 0; it < n_iter; ++it) {
    double ub[3];
    for (int k = 0; k < 3; ++k) ub[k] = 0.5 * (us[k] + ut[k]);
    const double gam = orc_gamma(m, ub, eps);
    const double u0 = gam / m->alpha;
    for (int i = 0; i < 2; ++i) {
      ut[i] = us[i] + dt * (-m->alpha * u0 * d->alpha[i] + ub[0] * d->beta1[i]
                            - 1.0 / (2.0 * u0) * (d->hu11[i] * ub[0] * ub[0] + d->hu22[i] * ub[1] * ub[1]
                                                  + d->hu33[i] * ub[2] * ub[2]
                                                  + 2.0 * d->hu13[i] * ub[0] * ub[2]));
    }
    ut[2] = us[2];
  }
  u[0] = ut[0]; u[1] = ut[1]; u[2] = ut[2];
}

/* Eq. 28-29, in displacement space del = x~ - x^(n): all metric
 * coefficients, alpha, beta^1 (and gamma, reading R-S7) at the midpoint.
 * Returns d(phi)/dt of Eq. 30 evaluated at x_m = x^(n) + del/2. */
static double orc_geodesic_x(const orc_grid* g, double x1n, double x2n, const double u[3], double eps,
                             double dt, double del[2]) {
  del[0] = 0.0; del[1] = 0.0;
  orc_metric_t m;
  for (int it = 0; it < g->n_iter; ++it) {
    orc_metric(g, x1n + 0.5 * del[0], x2n + 0.5 * del[1], &m);
    const double u0 = orc_gamma(&m, u, eps) / m.alpha;
    del[0] = dt * ((m.hu11 * u[0] + m.hu13 * u[2]) / u0 - m.beta1);
    del[1] = dt * (m.hu22 * u[1] / u0);
  }
  orc_metric(g, x1n + 0.5 * del[0], x2n + 0.5 * del[1], &m);
  const double u0 = orc_gamma(&m, u, eps) / m.alpha;
  return (m.hu13 * u[0] + m.hu33 * u[2]) / u0;
}

/* Particle columns (SoA), as the C ABI of the product lays them out. */
typedef struct {
  int64_t n;
  int32_t *i1, *i2; double *dx1, *dx2;
  double *u1, *u2, *u3;
  double *phi;                               /* may be NULL */
  int32_t *i1_prev, *i2_prev; double *dx1_prev, *dx2_prev;
  const double* weight; uint8_t* tag;        /* 1 alive, 0 dead */
  double q_over_m, charge; int32_t massive;
} orc_particles;

/* Optional diagnostic output (no effect on any result): the raw displacement (del1, del2) of Eq. 28-29
 * before renormalisation and reflection, one entry per particle.  The parity tests use it to evaluate
 * the conditioning of phi for particles whose midpoint grazes the polar axis. */
static double* orc_diag_del1 = NULL;
static double* orc_diag_del2 = NULL;
void orc_set_diag(double* del1, double* del2) { orc_diag_del1 = del1; orc_diag_del2 = del2; }

/* Whole per-particle update with the fields at the particle given (Dp,Bp,
 * contravariant code basis).  Steps 1, 3-11 of P:264-311 and the BCs of
 * P:465-467 (reading R-S9). Returns 0 alive, 1 absorbed inside, 2 absorbed outside. */
static int orc_push_core(const orc_grid* g, orc_particles* p, int64_t k, const double Dp[3],
                         const double Bp[3], double dt) {
  const double eps = p->massive ? 1.0 : 0.0;
  const int em = (p->q_over_m != 0.0) && p->massive;
  /* 1. save previous location */
  p->i1_prev[k] = p->i1[k]; p->i2_prev[k] = p->i2[k];
  p->dx1_prev[k] = p->dx1[k]; p->dx2_prev[k] = p->dx2[k];
  const double x1n = (double)p->i1[k] + p->dx1[k];
  const double x2n = (double)p->i2[k] + p->dx2[k];
  double u[3] = {p->u1[k], p->u2[k], p->u3[k]};

  ORC_STAGE(ORC_ST_METRIC);
  orc_metric_t m; orc_dmetric_t d;
  orc_metric(g, x1n, x2n, &m);
  orc_dmetric(g, &m, &d);

  ORC_STAGE(ORC_ST_EM);
  double Dh[3] = {0, 0, 0}, Bh[3] = {0, 0, 0}, uh[3];
  const double c = p->q_over_m * m.alpha * dt * 0.25;
  if (em) {
    orc_cntrv_to_tetrad(&m, Dp, Dh);                           /* 3 */
    orc_cntrv_to_tetrad(&m, Bp, Bh);
    orc_cov_to_tetrad(&m, u, uh);
    orc_boris_half(Dh, Bh, c, uh);                             /* 4 */
    orc_tetrad_to_cov(&m, uh, u);                              /* 5 */
  }
  ORC_STAGE(ORC_ST_ULOOP);
  orc_geodesic_u(&m, &d, eps, dt, g->n_iter, u);               /* 6 */
  ORC_STAGE(ORC_ST_EM);
  if (em) {
    orc_cov_to_tetrad(&m, u, uh);                              /* 7 */
    orc_boris_half(Dh, Bh, c, uh);                             /* 8 */
    orc_tetrad_to_cov(&m, uh, u);                              /* 9 */
  }
  ORC_STAGE(ORC_ST_XLOOP);
  double del[2];
  const double dphidt = orc_geodesic_x(g, x1n, x2n, u, eps, dt, del);   /* 10 */
  if (orc_diag_del1) { orc_diag_del1[k] = del[0]; orc_diag_del2[k] = del[1]; }
  if (p->phi) p->phi[k] += dt * dphidt;                        /* 11 */
  ORC_STAGE(ORC_ST_BC);

  /* renormalise to (cell, displacement in [0,1)) */
  int32_t i1 = p->i1[k], i2 = p->i2[k];
  double t1 = p->dx1[k] + del[0], t2 = p->dx2[k] + del[1];
  double f1 = floor(t1), f2 = floor(t2);
  i1 += (int32_t)f1; i2 += (int32_t)f2;
  double dx1 = t1 - f1, dx2 = t2 - f2;
  if (dx1 >= 1.0) { dx1 = 0.0; i1 += 1; }
  if (dx2 >= 1.0) { dx2 = 0.0; i2 += 1; }
  /* axis reflection */
  if (i2 < 0 || i2 >= g->n2) {
    i2 = (i2 < 0) ? 0 : g->n2 - 1;
    dx2 = 1.0 - dx2;
    if (dx2 >= 1.0) dx2 = nextafter(1.0, 0.0);
    u[1] = -u[1];
  }
  p->i1[k] = i1; p->i2[k] = i2; p->dx1[k] = dx1; p->dx2[k] = dx2;
  p->u1[k] = u[0]; p->u2[k] = u[1]; p->u3[k] = u[2];
  /* radial removal */
  if (i1 < 0) { p->tag[k] = 0; return 1; }
  if (i1 >= g->n1) { p->tag[k] = 0; return 2; }
  return 0;
}

/* counters: [0] alive after, [1] absorbed inside, [2] absorbed outside */
void orc_push(const orc_grid* g, orc_particles* p, const orc_fields* F, double dt, int64_t counters[3]) {
  int64_t c0 = 0, c1 = 0, c2 = 0;
  const int em = (p->q_over_m != 0.0) && p->massive;
#pragma omp parallel for schedule(static) reduction(+ : c0, c1, c2) if (p->n > 4096)
  for (int64_t k = 0; k < p->n; ++k) {
    if (!p->tag[k]) continue;
    double Dp[3] = {0, 0, 0}, Bp[3] = {0, 0, 0};
    ORC_STAGE(ORC_ST_INTERP);
    if (em) orc_interp(g, F, p->i1[k], p->i2[k], p->dx1[k], p->dx2[k], Dp, Bp);   /* 2 */
    const int r = orc_push_core(g, p, k, Dp, Bp, dt);
    c0 += (r == 0); c1 += (r == 1); c2 += (r == 2);
  }
  if (counters) { counters[0] = c0; counters[1] = c1; counters[2] = c2; }
}

/* Same update with D,B at the particle supplied by the caller (arrays [n][3]):
 * used by the pins that isolate the pusher from the interpolation. */
void orc_push_given_fields(const orc_grid* g, orc_particles* p, const double* Dp, const double* Bp, double dt) {
  for (int64_t k = 0; k < p->n; ++k) {
    if (!p->tag[k]) continue;
    orc_push_core(g, p, k, Dp + 3 * k, Bp + 3 * k, dt);
  }
}

/* ------------------------------------------------------------------------
 * Deposit.  Reading R-S10: first-order shape, two-segment
 * ("zigzag") charge-conserving path split, relay point per axis
 *   x_r = min(min(ia,ib)+1, max(max(ia,ib), (xa+xb)/2));
 * J^3 = q w (alpha/gamma) u^3 (Eq. 36) at the midpoint of the deposited path,
 * theta clamped, each segment carrying half, bilinear on nodes.
 * Path = (prev) -> (current, after BCs); dead particles deposit nothing;
 * a particle that moved more than one cell along an axis is counted in
 * *n_overstep and skipped.  J arrays are ACCUMULATED into.
 * ---------------------------------------------------------------------- */
typedef struct { double *J1, *J2, *J3; } orc_current;

static void orc_deposit_one(const orc_grid* g, const orc_particles* p, int64_t k, double dt,
                            double* J1, double* J2, double* J3, int64_t* overstep) {
  ORC_STAGE(ORC_ST_DEPOSIT);
  const int64_t ld = g->n2 + 2 * g->ng;
  const int ia = p->i1_prev[k], ja = p->i2_prev[k], ib = p->i1[k], jb = p->i2[k];
  const int di = ib - ia, dj = jb - ja;
  if (di > 1 || di < -1 || dj > 1 || dj < -1) { (*overstep)++; return; }
  /* positions relative to the node (ia, ja) */
  const double xa = p->dx1_prev[k], ya = p->dx2_prev[k];
  const double xb = (double)di + p->dx1[k], yb = (double)dj + p->dx2[k];
  const double xr = fmin((double)(di < 0 ? di : 0) + 1.0, fmax((double)(di > 0 ? di : 0), 0.5 * (xa + xb)));
  const double yr = fmin((double)(dj < 0 ? dj : 0) + 1.0, fmax((double)(dj > 0 ? dj : 0), 0.5 * (ya + yb)));
  const double qw = p->charge * p->weight[k];
  const double c = qw / dt;

  /* out-of-plane velocity at the midpoint of the deposited path (Eq. 36) */
  orc_metric_t m;
  orc_metric(g, (double)ia + 0.5 * (xa + xb), (double)ja + 0.5 * (ya + yb), &m);
  const double u[3] = {p->u1[k], p->u2[k], p->u3[k]};
  const double gam = orc_gamma(&m, u, p->massive ? 1.0 : 0.0);
  const double v3 = m.alpha / gam * (m.hu13 * u[0] + m.hu33 * u[2]);

  const double sx[3] = {xa, xr, xb}, sy[3] = {ya, yr, yb};
  const int ci[2] = {ia, ib}, cj[2] = {ja, jb};
  const int oi[2] = {0, di}, oj[2] = {0, dj};
  for (int s = 0; s < 2; ++s) {
    const double F1 = c * (sx[s + 1] - sx[s]);
    const double F2 = c * (sy[s + 1] - sy[s]);
    const double W1 = 0.5 * (sx[s] + sx[s + 1]) - (double)oi[s];
    const double W2 = 0.5 * (sy[s] + sy[s + 1]) - (double)oj[s];
    const int64_t o = (int64_t)(ci[s] + g->ng) * ld + (cj[s] + g->ng);
    J1[o] += F1 * (1.0 - W2);
    J1[o + 1] += F1 * W2;
    J2[o] += F2 * (1.0 - W1);
    J2[o + ld] += F2 * W1;
    const double F3 = 0.5 * qw * v3;
    J3[o] += F3 * (1.0 - W1) * (1.0 - W2);
    J3[o + ld] += F3 * W1 * (1.0 - W2);
    J3[o + 1] += F3 * (1.0 - W1) * W2;
    J3[o + ld + 1] += F3 * W1 * W2;
  }
}

void orc_deposit(const orc_grid* g, const orc_particles* p, double dt, orc_current* J, int64_t* n_overstep) {
  int64_t over = 0;
  if (p->charge == 0.0) { if (n_overstep) *n_overstep = 0; return; }
  const int64_t ncell = (int64_t)(g->n1 + 2 * g->ng) * (g->n2 + 2 * g->ng);
#ifdef _OPENMP
  const int nt = omp_get_max_threads();
#else
  const int nt = 1;
#endif
  if (nt == 1 || p->n <= 4096) {
    for (int64_t k = 0; k < p->n; ++k)
      if (p->tag[k]) orc_deposit_one(g, p, k, dt, J->J1, J->J2, J->J3, &over);
  } else {
    /* thread-private J over static contiguous particle ranges, reduced in thread order */
    double* priv = (double*)calloc((size_t)nt * 3 * ncell, sizeof(double));
    int64_t* ov = (int64_t*)calloc((size_t)nt, sizeof(int64_t));
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
      const int t = omp_get_thread_num();
#else
      const int t = 0;
#endif
      const int64_t lo = p->n * t / nt, hi = p->n * (t + 1) / nt;
      double* b = priv + (size_t)t * 3 * ncell;
      for (int64_t k = lo; k < hi; ++k)
        if (p->tag[k]) orc_deposit_one(g, p, k, dt, b, b + ncell, b + 2 * ncell, &ov[t]);
    }
    for (int t = 0; t < nt; ++t) {
      const double* b = priv + (size_t)t * 3 * ncell;
      for (int64_t c = 0; c < ncell; ++c) {
        J->J1[c] += b[c]; J->J2[c] += b[ncell + c]; J->J3[c] += b[2 * ncell + c];
      }
      over += ov[t];
    }
    free(priv); free(ov);
  }
  if (n_overstep) *n_overstep = over;
}

/* vectorised accessors for the Python tests */
void orc_metric_many(const orc_grid* g, int64_t n, const double* x1, const double* x2, orc_metric_t* m,
                     orc_dmetric_t* d) {
  for (int64_t k = 0; k < n; ++k) {
    orc_metric(g, x1[k], x2[k], &m[k]);
    if (d) orc_dmetric(g, &m[k], &d[k]);
  }
}
void orc_interp_many(const orc_grid* g, const orc_fields* F, int64_t n, const int32_t* i1, const int32_t* i2,
                     const double* dx1, const double* dx2, double* D, double* B) {
  for (int64_t k = 0; k < n; ++k) orc_interp(g, F, i1[k], i2[k], dx1[k], dx2[k], D + 3 * k, B + 3 * k);
}
int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* ========================================================================
 * Field-solver half: auxiliary fields Eq. 38/42-44,
 * Faraday Eq. 40, Ampere Eq. 41 with the polar-axis
 * update of D^1 Eq. 45 (polar area P:792-794).
 * Plain loops over the mesh; arrays [n1+2G][n2+2G] as above; ghost ROWS (i < 0,
 * i >= n1) of the inputs are the caller's, ghost COLUMNS beyond the
 * axes are not read.  Rows updated: every row whose x1-stencils lie inside the
 * arrays (aux: array rows 1..rows-2; Faraday/Ampere: array rows 2..rows-3).
 * Readings (DESIGN.md R-F*): Eq. 44 is garbled in the text; every <.> is the
 * two-point volume-weighted average along x1 of Eq. 43, written with
 * sqrt(h~) = sqrt(h)/sin(theta) so that the axis rows are regular.
 * The metric here is NOT clamped at the axis (sin(theta) = 0 there, exactly).
 * ====================================================================== */
typedef struct { double alpha, h11, h22, h33, h13, sqh_t, beta1, sth; } orc_fm;   /* sqh_t = sqrt(h)/sin(theta) */

static void orc_field_metric(const orc_grid* g, double x1, double x2, orc_fm* f) {
  orc_grid gg = *g;
  gg.small_angle = 0.0;
  orc_metric_t m;
  orc_metric(&gg, x1, x2, &m);
  /* exactly on the axes sin(theta) must be exactly 0 (x2 = 0) or the rounded sin(pi) made 0 (x2 = n2) */
  double sth = m.sth;
  if (x2 == 0.0 || x2 == (double)g->n2) sth = 0.0;
  const double s2th = sth * sth;
  f->alpha = m.alpha;
  f->h11 = m.hd11;
  f->h22 = m.hd22;
  f->h33 = m.A * s2th / m.Sigma;
  f->h13 = -m.s1 * g->a * (1.0 + m.z) * s2th;
  f->sqh_t = m.s1 * m.s2 * m.Sigma / m.alpha;
  f->beta1 = m.beta1;
  f->sth = sth;
}

#define ORC_AT(F, a1, a2) (F)[(int64_t)(a1) * ld + (a2)]

/* E_i at the D^i locations, H_i at the B^i locations (Eq. 42).  Any output pointer may be NULL. */
void orc_aux_fields(const orc_grid* g, const orc_fields* F, double* E1, double* E2, double* E3,
                    double* H1, double* H2, double* H3) {
  const int G = g->ng, rows = g->n1 + 2 * G;
  const int64_t ld = g->n2 + 2 * G;
  for (int a1 = 1; a1 < rows - 1; ++a1) {
    const double i = (double)(a1 - G);
    for (int j = 0; j <= g->n2; ++j) {
      const int a2 = j + G;
      const double x2 = (double)j;
      orc_fm c, l, r, cl, cr;   /* centre and the two x1-neighbours of each interpolation */
      /* ---- locations with integer j: E1 (i+1/2,j), E3 (i,j), H2 (i+1/2,j) ---- */
      orc_field_metric(g, i + 0.5, x2, &c);
      orc_field_metric(g, i, x2, &l);
      orc_field_metric(g, i + 1.0, x2, &r);
      if (E1) {
        const double avg = (l.sqh_t * l.h13 * ORC_AT(F->D3, a1, a2) + r.sqh_t * r.h13 * ORC_AT(F->D3, a1 + 1, a2))
                           / (2.0 * c.sqh_t);
        ORC_AT(E1, a1, a2) = c.alpha * (c.h11 * ORC_AT(F->D1, a1, a2) + avg);
      }
      if (H2) {
        const double avg = 0.5 * (l.sqh_t * l.sth * l.beta1 * ORC_AT(F->D3, a1, a2)
                                  + r.sqh_t * r.sth * r.beta1 * ORC_AT(F->D3, a1 + 1, a2));
        ORC_AT(H2, a1, a2) = c.alpha * c.h22 * ORC_AT(F->B2, a1, a2) + avg;
      }
      if (E3) {
        orc_field_metric(g, i - 0.5, x2, &cl);
        const double a13 = (cl.sqh_t * cl.h13 * ORC_AT(F->D1, a1 - 1, a2) + c.sqh_t * c.h13 * ORC_AT(F->D1, a1, a2))
                           / (2.0 * l.sqh_t);
        const double ab = 0.5 * (cl.sqh_t * cl.sth * cl.beta1 * ORC_AT(F->B2, a1 - 1, a2)
                                 + c.sqh_t * c.sth * c.beta1 * ORC_AT(F->B2, a1, a2));
        ORC_AT(E3, a1, a2) = l.alpha * (l.h33 * ORC_AT(F->D3, a1, a2) + a13) + ab;
      }
      if (j == g->n2) continue;
      /* ---- locations with half-integer j: E2 (i,j+1/2), H1 (i,j+1/2), H3 (i+1/2,j+1/2) ---- */
      orc_field_metric(g, i, x2 + 0.5, &c);
      orc_field_metric(g, i - 0.5, x2 + 0.5, &cl);
      orc_field_metric(g, i + 0.5, x2 + 0.5, &cr);
      if (E2) {
        const double ab = 0.5 * (cl.sqh_t * cl.sth * cl.beta1 * ORC_AT(F->B3, a1 - 1, a2)
                                 + cr.sqh_t * cr.sth * cr.beta1 * ORC_AT(F->B3, a1, a2));
        ORC_AT(E2, a1, a2) = c.alpha * c.h22 * ORC_AT(F->D2, a1, a2) - ab;
      }
      if (H1) {
        const double a13 = (cl.sqh_t * cl.h13 * ORC_AT(F->B3, a1 - 1, a2) + cr.sqh_t * cr.h13 * ORC_AT(F->B3, a1, a2))
                           / (2.0 * c.sqh_t);
        ORC_AT(H1, a1, a2) = c.alpha * (c.h11 * ORC_AT(F->B1, a1, a2) + a13);
      }
      if (H3) {
        orc_field_metric(g, i + 1.0, x2 + 0.5, &r);
        const double a13 = (c.sqh_t * c.h13 * ORC_AT(F->B1, a1, a2) + r.sqh_t * r.h13 * ORC_AT(F->B1, a1 + 1, a2))
                           / (2.0 * cr.sqh_t);
        const double ab = 0.5 * (c.sqh_t * c.sth * c.beta1 * ORC_AT(F->D2, a1, a2)
                                 + r.sqh_t * r.sth * r.beta1 * ORC_AT(F->D2, a1 + 1, a2));
        ORC_AT(H3, a1, a2) = cr.alpha * (cr.h33 * ORC_AT(F->B3, a1, a2) + a13) - ab;
      }
    }
  }
}

static double orc_sqrt_h(const orc_grid* g, double x1, double x2) {
  orc_fm f;
  orc_field_metric(g, x1, x2, &f);
  return f.sqh_t * f.sth;
}

/* Eq. 40: B^i -= dt e^{ijk} d_j E_k with 1/sqrt(h) at the component's own location.
 * B^2 on the two axes is not evolved. */
void orc_faraday(const orc_grid* g, double* B1, double* B2, double* B3, const double* E1, const double* E2,
                 const double* E3, double dt) {
  const int G = g->ng, rows = g->n1 + 2 * G;
  const int64_t ld = g->n2 + 2 * G;
  for (int a1 = 2; a1 < rows - 2; ++a1) {
    const double i = (double)(a1 - G);
    for (int j = 0; j < g->n2; ++j) {
      const int a2 = j + G;
      ORC_AT(B1, a1, a2) -= dt * (ORC_AT(E3, a1, a2 + 1) - ORC_AT(E3, a1, a2)) / orc_sqrt_h(g, i, j + 0.5);
      if (j > 0)
        ORC_AT(B2, a1, a2) += dt * (ORC_AT(E3, a1 + 1, a2) - ORC_AT(E3, a1, a2)) / orc_sqrt_h(g, i + 0.5, (double)j);
      ORC_AT(B3, a1, a2) -= dt * ((ORC_AT(E2, a1 + 1, a2) - ORC_AT(E2, a1, a2))
                                  - (ORC_AT(E1, a1, a2 + 1) - ORC_AT(E1, a1, a2))) / orc_sqrt_h(g, i + 0.5, j + 0.5);
    }
  }
}

/* Polar area with a half-cell radius around the axis (P:792-794 for A.1, P:810-812 for A.2; the A.3 form follows with
 * dr -> s1 and the stretched theta): A_{i+1/2} = int_0^{1/2} sqrt(h) dx2 = s1 (r^2+a^2) sqrt(1 + 2Mr/(r^2+a^2)) (1 - cos theta(1/2)) */
static double orc_polar_area(const orc_grid* g, double x1) {
  orc_grid gg = *g;
  gg.small_angle = 0.0;
  orc_metric_t m;
  orc_metric(&gg, x1, 0.5, &m);
  const double q = m.r * m.r + g->a * g->a;
  return m.s1 * q * sqrt(1.0 + 2.0 * g->mass * m.r / q) * (1.0 - cos(m.th));
}

/* Eq. 41: D^i += dt (e^{ijk} d_j H_k - kJ J^i)/sqrt(h), J = deposited conformal currents (may be NULL),
 * kJ = 4 pi in the paper's Gaussian form.  On the axes D^3 is not evolved and D^1 takes the integral form Eq. 45:
 * D^1 += dt (+-H_3 of the neighbouring half cell - (kJ/2) J^1)/A_{i+1/2}, sign + at theta = 0 and - at theta = pi
 * (the circulation around the polar cap reverses; reading R-F2). */
void orc_ampere(const orc_grid* g, double* D1, double* D2, double* D3, const double* H1, const double* H2,
                const double* H3, const double* J1, const double* J2, const double* J3, double kJ, double dt) {
  const int G = g->ng, rows = g->n1 + 2 * G;
  const int64_t ld = g->n2 + 2 * G;
  for (int a1 = 2; a1 < rows - 2; ++a1) {
    const double i = (double)(a1 - G);
    for (int j = 0; j <= g->n2; ++j) {
      const int a2 = j + G;
      const double j1 = J1 ? ORC_AT(J1, a1, a2) : 0.0;
      if (j == 0)
        ORC_AT(D1, a1, a2) += dt * (ORC_AT(H3, a1, a2) - 0.5 * kJ * j1) / orc_polar_area(g, i + 0.5);
      else if (j == g->n2)
        ORC_AT(D1, a1, a2) += dt * (-ORC_AT(H3, a1, a2 - 1) - 0.5 * kJ * j1) / orc_polar_area(g, i + 0.5);
      else
        ORC_AT(D1, a1, a2) += dt * ((ORC_AT(H3, a1, a2) - ORC_AT(H3, a1, a2 - 1)) - kJ * j1) / orc_sqrt_h(g, i + 0.5, (double)j);
      if (j == g->n2) continue;
      const double j2 = J2 ? ORC_AT(J2, a1, a2) : 0.0;
      ORC_AT(D2, a1, a2) += dt * (-(ORC_AT(H3, a1, a2) - ORC_AT(H3, a1 - 1, a2)) - kJ * j2) / orc_sqrt_h(g, i, j + 0.5);
      if (j > 0) {
        const double j3 = J3 ? ORC_AT(J3, a1, a2) : 0.0;
        ORC_AT(D3, a1, a2) += dt * ((ORC_AT(H2, a1, a2) - ORC_AT(H2, a1 - 1, a2))
                                    - (ORC_AT(H1, a1, a2) - ORC_AT(H1, a1, a2 - 1)) - kJ * j3) / orc_sqrt_h(g, i, (double)j);
      }
    }
  }
}

#ifdef ORC_COUNT
/* One push + deposit of every alive particle on the counting type, single thread; out[stage][kind] receives the
 * totals (layout ORC_N_STAGES x ORC_N_KINDS of orc_count.hpp), *n_particles the number of particles counted. */
extern "C" void orc_count_step(const orc_grid* g, orc_particles* p, const orc_fields* F, orc_current* J, const double* dt,
                               int64_t* out, int64_t* n_particles) {
  for (int s = 0; s < ORC_N_STAGES; ++s)
    for (int k = 0; k < ORC_N_KINDS; ++k) orc_counts[s][k] = 0;
  const int em = (p->q_over_m != 0.0) && p->massive;
  int64_t n = 0, over = 0;
  ORC_STAGE(ORC_ST_OTHER);
  for (int64_t k = 0; k < p->n; ++k) {
    if (!p->tag[k]) continue;
    ++n;
    double Dp[3] = {0, 0, 0}, Bp[3] = {0, 0, 0};
    ORC_STAGE(ORC_ST_INTERP);
    if (em) orc_interp(g, F, p->i1[k], p->i2[k], p->dx1[k], p->dx2[k], Dp, Bp);
    orc_push_core(g, p, k, Dp, Bp, *dt);
    if (p->tag[k] && p->charge != 0.0) orc_deposit_one(g, p, k, *dt, J->J1, J->J2, J->J3, &over);
    ORC_STAGE(ORC_ST_OTHER);
  }
  for (int s = 0; s < ORC_N_STAGES; ++s)
    for (int k = 0; k < ORC_N_KINDS; ++k) out[s * ORC_N_KINDS + k] = orc_counts[s][k];
  *n_particles = n;
}
#endif
