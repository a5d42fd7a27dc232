/* vlbm_oracle.c — CPU ORACLE (test infrastructure only; see vlbm_oracle.h).
 *
 * Plain, slow, per-cell restatement of the vectorial LBM step of arxiv/paper_2606_00641:
 *   Eq.2  PAPER.md:78   f_{k,i}(x + c_i, t+1) = f_{k,i} + Omega^C + Omega^S
 *   Eq.3  PAPER.md:84   f^eq_{k,i} = w_i (Q_k + c_i . Phi_k / c_s^2)
 *   Eq.4  PAPER.md:90   Q_k = sum_i f_{k,i},  Phi_k = sum_i f_{k,i} c_i
 *   Eq.5  PAPER.md:98   D = (tau - 1/2) c_s^2
 *   Eq.8  PAPER.md:128  p = (gamma-1)(E - rho|u|^2/2 - |B|^2/2)
 *   Eq.11 PAPER.md:142  ideal-MHD Q and Phi
 *   Eq.12 PAPER.md:148  Powell source S = -(div B)(0, B, u.B, u)
 *   Eq.13-14 PAPER.md:160-162  homogenised solid: u^ = d u + (1-d) u^B, B^ likewise
 *   PAPER.md:154        static boundaries: Dirichlet (value defined) / Neumann (value from the
 *                       next cell along the discrete normal, new equilibrium assigned)
 * Stored state = post-collision populations g; one step = pull, moments, source, blend, flux,
 * BGK collide + direct injection, store.  fp64 throughout.
 * Compile: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC.
 */
#include "vlbm_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define MAXK 26
#define MAXDIP 4
#define NBODY 14          /* body integrals, oracle_body_read */
#define ACCW (MAXK + NBODY) /* per-row accumulator: source log | body integrals */
#define MAXQ 19

/* ---- lattice tables (A2): rest; +x,-x,+y,-y,+z,-z; diagonals (+,+),(-,-),(+,-),(-,+) per plane
 * xy, xz, yz.  Weights are the Gauss-Hermite ones of the textbook lattices, c_s^2 = 1/3.
 * D2Q5 / D3Q7 (the paper's own lattices): rest weight 1/3 resp. 1/4, which is
 * what sum_i w_i c_ia c_ib = c_s^2 delta_ab with c_s^2 = 1/3 resp. 1/4 forces. ---- */
typedef struct { int D, Q; int c[MAXQ][3]; double w[MAXQ]; double cs2; } lattice_t;

static int lattice_make(int id, lattice_t *L)
{
  static const int c19[19][3] = {
    {0,0,0},
    {1,0,0},{-1,0,0},{0,1,0},{0,-1,0},{0,0,1},{0,0,-1},
    {1,1,0},{-1,-1,0},{1,-1,0},{-1,1,0},
    {1,0,1},{-1,0,-1},{1,0,-1},{-1,0,1},
    {0,1,1},{0,-1,-1},{0,1,-1},{0,-1,1} };
  static const int c9[9][3] = {
    {0,0,0},{1,0,0},{-1,0,0},{0,1,0},{0,-1,0},{1,1,0},{-1,-1,0},{1,-1,0},{-1,1,0} };
  memset(L, 0, sizeof *L);
  int i;
  switch (id) {
  case ORC_D1Q3:
    L->D = 1; L->Q = 3; L->cs2 = 1.0 / 3.0;
    L->c[1][0] = 1; L->c[2][0] = -1;
    L->w[0] = 2.0 / 3.0; L->w[1] = L->w[2] = 1.0 / 6.0;
    return 0;
  case ORC_D2Q9:
    L->D = 2; L->Q = 9; L->cs2 = 1.0 / 3.0;
    memcpy(L->c, c9, sizeof c9);
    L->w[0] = 4.0 / 9.0;
    for (i = 1; i < 5; i++) L->w[i] = 1.0 / 9.0;
    for (i = 5; i < 9; i++) L->w[i] = 1.0 / 36.0;
    return 0;
  case ORC_D3Q19:
    L->D = 3; L->Q = 19; L->cs2 = 1.0 / 3.0;
    memcpy(L->c, c19, sizeof c19);
    L->w[0] = 1.0 / 3.0;
    for (i = 1; i < 7; i++) L->w[i] = 1.0 / 18.0;
    for (i = 7; i < 19; i++) L->w[i] = 1.0 / 36.0;
    return 0;
  case ORC_D2Q5:
    L->D = 2; L->Q = 5; L->cs2 = 1.0 / 3.0;
    memcpy(L->c, c9, 5 * sizeof c9[0]);
    L->w[0] = 1.0 / 3.0;
    for (i = 1; i < 5; i++) L->w[i] = 1.0 / 6.0;
    return 0;
  case ORC_D3Q7:
    L->D = 3; L->Q = 7; L->cs2 = 1.0 / 4.0;
    memcpy(L->c, c19, 7 * sizeof c19[0]);
    L->w[0] = 1.0 / 4.0;
    for (i = 1; i < 7; i++) L->w[i] = 1.0 / 8.0;
    return 0;
  }
  return -1;
}

int oracle_lattice(int lattice, int *D, int *Q, int *c, double *w, double *cs2)
{
  lattice_t L;
  if (lattice_make(lattice, &L)) return -1;
  *D = L.D; *Q = L.Q; *cs2 = L.cs2;
  for (int i = 0; i < L.Q; i++) { w[i] = L.w[i]; for (int a = 0; a < 3; a++) c[3 * i + a] = L.c[i][a]; }
  return 0;
}

static int is_ideal(int scheme) { return scheme == ORC_IDEAL || scheme == ORC_IDEAL_DIVB || scheme == ORC_RESIST || scheme == ORC_FULL; }   /* first 8 variables (rho, m, E, B) */
static int num_vars(int scheme, int D)
{
  if (scheme == ORC_IDEAL) return 8;
  if (scheme == ORC_IDEAL_DIVB) return 9;
  if (scheme == ORC_RESIST) return 8 + 3 * D;       /* + G_ab = tau_M d_a B_b, a < D, b < 3, index 8 + 3 a + b */
  if (scheme == ORC_FULL) return 8 + 6 * D;         /* + H_ab = tau_M d_a u_b, index 8 + 3 D + 3 a + b */
  return 1 + 2 * D;
}

int oracle_num_vars(const oracle_params *p)
{
  lattice_t L;
  if (lattice_make(p->lattice, &L)) return -1;
  return num_vars(p->scheme, L.D);
}
int oracle_num_dirs(const oracle_params *p)
{
  lattice_t L;
  if (lattice_make(p->lattice, &L)) return -1;
  return L.Q;
}

static int g_threads = 0;
void oracle_set_threads(int n) { g_threads = n; }
int oracle_get_threads(void)
{
#ifdef _OPENMP
  return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
  return 1;
#endif
}

/* ---- fluxes Phi_k,alpha(Q), alpha over the D lattice axes ---- */
/* IDEAL: Eq.11 PAPER.md:142 with the EOS Eq.8; magnetic pressure |B|^2/2.
 * INCRES (A3): P carries kinematic pressure, dP/dt + c0^2 div u = 0; momentum flux u u + (P + B^2/2) I - B B;
 * induction flux u B - B u. */
static void flux_eval(const oracle_params *prm, int D, const double *Q, double Phi[MAXK][3])
{
  const int scheme = prm->scheme;
  const double gamma = prm->gamma, c0sq = prm->c0sq;
  int a, b;
  if (is_ideal(scheme)) {
    double rho = Q[0], E = Q[4];
    const double *m = Q + 1, *B = Q + 5;
    double u[3];
    for (b = 0; b < 3; b++) u[b] = m[b] / rho;
    double B2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
    double mu = m[0] * u[0] + m[1] * u[1] + m[2] * u[2];
    double p = (gamma - 1.0) * (E - 0.5 * mu - 0.5 * B2);
    double pt = p + 0.5 * B2;
    double uB = u[0] * B[0] + u[1] * B[1] + u[2] * B[2];
    for (a = 0; a < D; a++) {
      Phi[0][a] = m[a];
      for (b = 0; b < 3; b++) Phi[1 + b][a] = m[b] * u[a] + (a == b ? pt : 0.0) - B[b] * B[a];
      Phi[4][a] = (E + pt) * u[a] - B[a] * uB;
      for (b = 0; b < 3; b++) Phi[5 + b][a] = u[a] * B[b] - B[a] * u[b];
      /* Eq.10 PAPER.md:136 traced: the relaxation variable D = tr G has the flux D u - B */
      if (scheme == ORC_IDEAL_DIVB) Phi[8][a] = Q[8] * u[a] - B[a];
    }
    if (scheme == ORC_RESIST || scheme == ORC_FULL) {
      /* dissipative system, PAPER.md:122 with the transported gradients of Eq.9-10 PAPER.md:132-136 (A22):
       *   g_cb = G_cb / tau_M ~ d_c B_b;  current j = curl B: j_e = eps_ecb g_cb (c < D);
       *   Phi_{B_b},a -= eta g_ab;  Phi_E,a += eta (j x B)_a;  Phi_{G_cb},a = G_cb u_a - delta_ca B_b */
      const double *Gv = Q + 8;
      const double eta = prm->eta, itm = 1.0 / prm->tau_relax;
      double g[3][3], j[3], jxB[3];
      int c;
      for (c = 0; c < 3; c++) for (b = 0; b < 3; b++) g[c][b] = c < D ? Gv[3 * c + b] * itm : 0.0;
      j[0] = g[1][2] - g[2][1];
      j[1] = g[2][0] - g[0][2];
      j[2] = g[0][1] - g[1][0];
      jxB[0] = j[1] * B[2] - j[2] * B[1];
      jxB[1] = j[2] * B[0] - j[0] * B[2];
      jxB[2] = j[0] * B[1] - j[1] * B[0];
      for (a = 0; a < D; a++) {
        Phi[4][a] += eta * jxB[a];
        for (b = 0; b < 3; b++) Phi[5 + b][a] -= eta * g[a][b];
        for (c = 0; c < D; c++) for (b = 0; b < 3; b++) Phi[8 + 3 * c + b][a] = Gv[3 * c + b] * u[a] - (c == a ? B[b] : 0.0);
      }
    }
    if (scheme == ORC_FULL) {
      /* viscous stress as transported variables (PAPER.md:132 Eq.9, :138 "a similar expansion logic is applied to the viscous
       * stress tensor"; reading A23): H_cb = tau_M d_c u_b with flux H_cb u_a - delta_ca u_b (Eq.10 with B -> u);
       *   h = H / tau_M ~ grad u;  sigma_ab = mu (h_ab + h_ba - 2/3 delta_ab tr h)   (Newtonian, mu = prm->nu);
       *   Phi_{m_b},a -= sigma_ab;  Phi_E,a -= u_b sigma_ab   (the -tau and -u.tau of PAPER.md:122; q = 0) */
      const double *Hv = Q + 8 + 3 * D;
      const double mu = prm->nu, itm = 1.0 / prm->tau_relax;
      double h[3][3], sig[3][3], trh = 0.0;
      int c;
      for (c = 0; c < 3; c++) for (b = 0; b < 3; b++) h[c][b] = c < D ? Hv[3 * c + b] * itm : 0.0;
      for (c = 0; c < 3; c++) trh += h[c][c];
      for (c = 0; c < 3; c++) for (b = 0; b < 3; b++) sig[c][b] = mu * (h[c][b] + h[b][c] - (c == b ? 2.0 / 3.0 * trh : 0.0));
      for (a = 0; a < D; a++) {
        double us = 0.0;
        for (b = 0; b < 3; b++) { Phi[1 + b][a] -= sig[a][b]; us += u[b] * sig[a][b]; }
        Phi[4][a] -= us;
        for (c = 0; c < D; c++) for (b = 0; b < 3; b++) Phi[8 + 3 * D + 3 * c + b][a] = Hv[3 * c + b] * u[a] - (c == a ? u[b] : 0.0);
      }
    }
  } else {
    double P = Q[0];
    const double *u = Q + 1, *B = Q + 1 + D;
    double B2 = 0.0;
    for (b = 0; b < D; b++) B2 += B[b] * B[b];
    double pt = P + 0.5 * B2;
    for (a = 0; a < D; a++) {
      Phi[0][a] = c0sq * u[a];
      for (b = 0; b < D; b++) Phi[1 + b][a] = u[b] * u[a] + (a == b ? pt : 0.0) - B[b] * B[a];
      for (b = 0; b < D; b++) Phi[1 + D + b][a] = u[a] * B[b] - B[a] * u[b];
    }
  }
}

/* Eq.3 */
static double feq_eval(const lattice_t *L, int i, double Qk, const double *Phik)
{
  double cPhi = 0.0;
  for (int a = 0; a < L->D; a++) cPhi += (double)L->c[i][a] * Phik[a];
  return L->w[i] * (Qk + cPhi / L->cs2);
}

int oracle_flux(const oracle_params *p, const double *Qv, double *Phi)
{
  lattice_t L;
  if (lattice_make(p->lattice, &L)) return -1;
  int K = num_vars(p->scheme, L.D);
  double F[MAXK][3];
  memset(F, 0, sizeof F);
  flux_eval(p, L.D, Qv, F);
  for (int k = 0; k < K; k++) for (int a = 0; a < 3; a++) Phi[3 * k + a] = a < L.D ? F[k][a] : 0.0;
  return 0;
}

int oracle_equilibrium(const oracle_params *p, const double *Qv, double *feq)
{
  lattice_t L;
  if (lattice_make(p->lattice, &L)) return -1;
  int K = num_vars(p->scheme, L.D);
  double F[MAXK][3];
  memset(F, 0, sizeof F);
  flux_eval(p, L.D, Qv, F);
  for (int k = 0; k < K; k++)
    for (int i = 0; i < L.Q; i++) feq[k * L.Q + i] = feq_eval(&L, i, Qv[k], F[k]);
  return 0;
}

/* ---- current-dependent resistivity (eta(j) = eta0 (1 + (j/j_c)^2); reading A20) ----
 * The B sets relax with a cell-local tau_B = 1/2 + eta(j)/c_s^2 (Eq.5).  The current comes from the antisymmetric part
 * of the non-equilibrium first moment of the B sets, N_ab = sum_i c_ia f_{B_b,i} - Phi_{B_b,a} ~ -tau_B c_s^2 d_a B_b:
 *   a2 := sum_{a<b} (N_ab - N_ba)^2 / c_s^4 = (tau_B |j|)^2.
 * tau_B then solves  tau = tau0 + e0 a2 / (j_c^2 tau^2),  tau0 = 1/2 + e0, e0 = eta0/c_s^2:  the cubic
 *   g(tau) = tau^3 - tau0 tau^2 - c = 0,  c = e0 a2 / j_c^2 >= 0,
 * whose only root >= tau0 is found by NEWTON_ITERS Newton steps from tau0 + cbrt(c) (g >= 0 there, g convex increasing). */
#define NEWTON_ITERS 6
static double tau_of_current(double tau0, double e0, double a2, double jc)
{
  double c = e0 * a2 / (jc * jc);
  double t = tau0 + cbrt(c);
  for (int it = 0; it < NEWTON_ITERS; it++) {
    double g = (t - tau0) * t * t - c;
    double dg = t * (3.0 * t - 2.0 * tau0);
    t = t - g / dg;
  }
  return t;
}

double oracle_tau_of_current(double tau0, double e0, double a2, double jc) { return tau_of_current(tau0, e0, a2, jc); }

/* ---- state ---- */
struct oracle {
  oracle_params p;
  lattice_t L;
  int K;
  long N;
  double omega[MAXK];  /* 1/tau_k */
  double tauB;         /* tau of the magnetic sets (all equal, A7) */
  int iB;              /* index of B_x in Q */
  int iU;              /* index of the first momentum / velocity component */
  double *g[2];        /* A/B population arrays [K][Q][N] */
  int cur;
  unsigned char *mask; /* [N] */
  double *Bsolid;      /* [3][N] or NULL */
  double usolid[3];
  int has_sphere;
  double sph_c0[3], sph_R, sph_u[3], sph_m[3], sph_Bs;
  long sph_t0;         /* step count at which the centre was sph_c0 */
  double sph_om[3];    /* angular velocity Omega of the body (rad per step): u^B(x) = u_s + Omega x r, dipole axis co-rotates */
  double sph_eps;      /* width eps_h of the linear porosity ramp across the sphere surface (Eq.15-16), 0 = sharp */
  int n_dip;           /* dipole ensemble of the sphere ("four independent, shifted, and smoothed magnetic dipoles"): */
  double dip_off[MAXDIP][3], dip_m[MAXDIP][3], dip_Bs[MAXDIP], dip_core[MAXDIP];   /* body-frame offset, axis, strength, core radius */
  double obs_om[3], obs_c[3];   /* masked bodies: u^B(x) = usolid + obs_om x (x - obs_c) */
  double *dfield;      /* lattice porosity d in [0,1] per cell (Eq.15), or NULL: d from the mask (SOLID -> 0) */
  long t;              /* steps done so far */
  double srclog[MAXK];
  double body[NBODY];  /* body integrals accumulated over the steps since the last reset (A21) */
  double body_ref[3];  /* torque reference point of masked bodies; an analytic sphere uses its own centre */
};

static long cell_index(const oracle_t *o, int x, int y, int z)
{
  return ((long)z * o->p.ny + y) * o->p.nx + x;
}
static double *pop(const oracle_t *o, double *g, int k, int i) { return g + ((long)k * o->L.Q + i) * o->N; }

int oracle_create(const oracle_params *p, const unsigned char *cell_mask, oracle_t **out)
{
  lattice_t L;
  *out = NULL;
  if (lattice_make(p->lattice, &L)) return -1;
  if (p->scheme != ORC_IDEAL && p->scheme != ORC_INCRES && p->scheme != ORC_IDEAL_DIVB && p->scheme != ORC_RESIST && p->scheme != ORC_FULL) return -1;
  if ((p->scheme == ORC_IDEAL_DIVB || p->scheme == ORC_RESIST || p->scheme == ORC_FULL) && !(p->tau_relax > 0.0)) return -1;
  if ((p->scheme == ORC_RESIST || p->scheme == ORC_FULL) && !(p->eta >= 0.0)) return -1;
  if (p->scheme == ORC_FULL && !(p->nu >= 0.0)) return -1;
  if (p->eta_jc != 0.0 && !(p->scheme == ORC_INCRES && p->eta_jc > 0.0)) return -1;
  if (p->nx < 1 || p->ny < 1 || p->nz < 1) return -1;
  if (L.D < 2 && p->ny != 1) return -1;
  if (L.D < 3 && p->nz != 1) return -1;
  const int n[3] = { p->nx, p->ny, p->nz };
  for (int a = 0; a < L.D; a++) {
    int lo = p->bc[2 * a], hi = p->bc[2 * a + 1];
    if (lo < 0 || lo > 2 || hi < 0 || hi > 2) return -1;
    if ((lo == ORC_BC_PERIODIC) != (hi == ORC_BC_PERIODIC)) return -1;
    if (lo != ORC_BC_PERIODIC && n[a] < 3) return -1;                     /* A9 needs an inward neighbour */
  }
  oracle_t *o = (oracle_t *)calloc(1, sizeof *o);
  if (!o) return -2;
  o->p = *p; o->L = L;
  o->K = num_vars(p->scheme, L.D);
  o->N = (long)p->nx * p->ny * p->nz;
  o->iU = 1;
  o->iB = is_ideal(p->scheme) ? 5 : 1 + L.D;
  int nvec = is_ideal(p->scheme) ? 3 : L.D;
  double tau[MAXK] = { 0 };
  for (int k = 0; k < o->K; k++) tau[k] = p->tau[k];
  /* Eq.5: tau = 1/2 + D / c_s^2 for the sets that carry a physical diffusivity (A3) */
  /* FULL carries nu (the shear viscosity mu) in the flux like eta: tau_u stays the stabilisation parameter */
  if (p->nu > 0.0 && p->scheme != ORC_FULL) {
    for (int b = 0; b < nvec; b++) tau[o->iU + b] = 0.5 + p->nu / L.cs2;
    if (p->scheme == ORC_INCRES) tau[0] = 0.5 + p->nu / L.cs2;
  }
  /* RESIST carries eta in the flux (-eta grad B): tau_B stays the stabilisation parameter */
  if (p->eta > 0.0 && p->scheme != ORC_RESIST && p->scheme != ORC_FULL) for (int b = 0; b < nvec; b++) tau[o->iB + b] = 0.5 + p->eta / L.cs2;
  for (int k = 0; k < o->K; k++) {
    if (!(tau[k] > 0.5)) { free(o); return -1; }
    o->omega[k] = 1.0 / tau[k];
  }
  o->tauB = tau[o->iB];
  for (int b = 1; b < nvec; b++) if (tau[o->iB + b] != o->tauB) { free(o); return -1; }   /* A7 */
  if (is_ideal(p->scheme) && !(p->gamma > 1.0)) { free(o); return -1; }
  size_t bytes = (size_t)o->K * L.Q * o->N * sizeof(double);
  o->g[0] = (double *)calloc(1, bytes);
  o->g[1] = (double *)calloc(1, bytes);
  o->mask = (unsigned char *)calloc(1, (size_t)o->N);
  if (!o->g[0] || !o->g[1] || !o->mask) { oracle_destroy(o); return -2; }
  if (cell_mask) memcpy(o->mask, cell_mask, (size_t)o->N);
  *out = o;
  return 0;
}

void oracle_destroy(oracle_t *o)
{
  if (!o) return;
  free(o->g[0]); free(o->g[1]); free(o->mask); free(o->Bsolid); free(o->dfield); free(o);
}

int oracle_set_obstacle(oracle_t *o, const unsigned char *mask, const double u_solid[3], const double *B_solid)
{
  if (!o || !mask) return -1;
  memcpy(o->mask, mask, (size_t)o->N);
  for (int a = 0; a < 3; a++) o->usolid[a] = u_solid ? u_solid[a] : 0.0;
  free(o->Bsolid); o->Bsolid = NULL;
  if (B_solid) {
    o->Bsolid = (double *)malloc(3 * (size_t)o->N * sizeof(double));
    if (!o->Bsolid) return -2;
    memcpy(o->Bsolid, B_solid, 3 * (size_t)o->N * sizeof(double));
  }
  return 0;
}

int oracle_set_sphere(oracle_t *o, const double centre[3], double radius, const double u_solid[3],
                      const double dipole_dir[3], double B_surface)
{
  if (!o || !(radius > 0.0)) return -1;
  o->has_sphere = 1;
  for (int a = 0; a < 3; a++) {
    o->sph_c0[a] = centre[a];   /* A12: centre before the next step; before step t it is c0 + (t - t0) u^B */
    o->sph_u[a] = u_solid[a]; o->sph_m[a] = dipole_dir[a];
  }
  o->sph_R = radius; o->sph_Bs = B_surface; o->sph_t0 = o->t;
  /* A12: one centred dipole capped at R/2 */
  o->n_dip = 1;
  for (int a = 0; a < 3; a++) { o->dip_off[0][a] = 0.0; o->dip_m[0][a] = dipole_dir[a]; }
  o->dip_Bs[0] = B_surface; o->dip_core[0] = 0.5 * radius;
  return 0;
}

/* ensemble of n <= 4 shifted, smoothed dipoles in the body frame; replaces the single dipole of set_sphere:
 *   B^B(x) = sum_j 1/2 Bs_j (R / max(|r_j|, core_j))^3 [3 (m_j.r^_j) r^_j - m_j],  r_j = x - c(t) - Rot(t) off_j,  m_j -> Rot(t) m_j */
int oracle_set_sphere_dipoles(oracle_t *o, int n, const double *offset, const double *dir, const double *B_surface, const double *core)
{
  if (!o || !o->has_sphere || n < 1 || n > MAXDIP || !offset || !dir || !B_surface || !core) return -1;
  for (int j = 0; j < n; j++) {
    if (!(core[j] > 0.0)) return -1;
    for (int a = 0; a < 3; a++) { o->dip_off[j][a] = offset[3 * j + a]; o->dip_m[j][a] = dir[3 * j + a]; }
    o->dip_Bs[j] = B_surface[j]; o->dip_core[j] = core[j];
  }
  o->n_dip = n;
  return 0;
}

/* rigid rotation of the masked / porosity body about `centre`: u^B(x) = u_solid + omega x (x - centre) */
int oracle_set_obstacle_rotation(oracle_t *o, const double omega[3], const double centre[3])
{
  if (!o || !omega || !centre) return -1;
  for (int a = 0; a < 3; a++) { o->obs_om[a] = omega[a]; o->obs_c[a] = centre[a]; }
  return 0;
}

int oracle_set_porosity(oracle_t *o, const double *d_field)
{
  if (!o) return -1;
  free(o->dfield); o->dfield = NULL;
  if (d_field) {
    o->dfield = (double *)malloc((size_t)o->N * sizeof(double));
    if (!o->dfield) return -2;
    for (long n = 0; n < o->N; n++) { if (!(d_field[n] >= 0.0 && d_field[n] <= 1.0)) return -1; o->dfield[n] = d_field[n]; }
  }
  return 0;
}

int oracle_set_sphere_rotation(oracle_t *o, const double omega[3])
{
  if (!o || !omega) return -1;
  for (int a = 0; a < 3; a++) o->sph_om[a] = omega[a];
  return 0;
}

int oracle_set_sphere_width(oracle_t *o, double eps)
{
  if (!o || !(eps >= 0.0)) return -1;
  o->sph_eps = eps;
  return 0;
}

/* Eq.3: g = f^eq(Q) from the given macroscopic fields */
int oracle_init(oracle_t *o, const double *fields)
{
  if (!o || !fields) return -1;
  const int K = o->K, Qn = o->L.Q;
  for (long n = 0; n < o->N; n++) {
    double Qv[MAXK], Phi[MAXK][3];
    for (int k = 0; k < K; k++) Qv[k] = fields[(long)k * o->N + n];
    memset(Phi, 0, sizeof Phi);
    flux_eval(&o->p, o->L.D, Qv, Phi);
    for (int k = 0; k < K; k++)
      for (int i = 0; i < Qn; i++) {
        double v = feq_eval(&o->L, i, Qv[k], Phi[k]);
        pop(o, o->g[0], k, i)[n] = v;
        pop(o, o->g[1], k, i)[n] = v;
      }
  }
  o->cur = 0; o->t = 0; o->sph_t0 = 0;
  memset(o->srclog, 0, sizeof o->srclog);
  memset(o->body, 0, sizeof o->body);
  return 0;
}

int oracle_get_populations(oracle_t *o, double *g_out)
{
  memcpy(g_out, o->g[o->cur], (size_t)o->K * o->L.Q * o->N * sizeof(double));
  return 0;
}
int oracle_set_populations(oracle_t *o, const double *g_in)
{
  memcpy(o->g[o->cur], g_in, (size_t)o->K * o->L.Q * o->N * sizeof(double));
  return 0;
}
int oracle_source_log(oracle_t *o, double *acc)
{
  for (int k = 0; k < o->K; k++) acc[k] = o->srclog[k];
  return 0;
}

/* ---- body integrals (A21) ----
 * The blend of Eq.13-14 injects dQh = Q^ - Q into the fluid at every cell with d < 1 (A8); what the fluid receives the body
 * gives.  Summed over those cells and accumulated over steps, r = x - (sphere centre at this step, else body_ref):
 *   [0..2] F = - sum dQh_m            momentum the fluid hands to the body per step (aerodynamic + Maxwell)
 *   [3..5] T = - sum r x dQh_m        its moment about the reference point
 *   [6]    W = - sum dQh_E            energy handed to the body (IDEAL; 0 for INCRES)
 *   [7..9] I =   sum dQh_B            magnetic field injected into the fluid
 *   [10..12]     sum (1-d) B          volume integral of the fluid's pre-blend B over the body (flux x length)
 *   [13]         sum (1-d)            body volume in cells
 * INCRES: the velocity sets stand for momentum (rho = 1). */
int oracle_body_read(oracle_t *o, double *out, int reset)
{
  if (!o) return -1;
  if (out) for (int j = 0; j < NBODY; j++) out[j] = o->body[j];
  if (reset) memset(o->body, 0, sizeof o->body);
  return 0;
}
int oracle_set_body_reference(oracle_t *o, const double ref[3])
{
  if (!o || !ref) return -1;
  for (int a = 0; a < 3; a++) o->body_ref[a] = ref[a];
  return 0;
}

/* ---- solid state at a cell (A8, A11, A12; Eq.15-16) ----
 * returns the lattice porosity d in [0,1]; fills uB[3], BB[3] when d < 1.
 * Sphere, c(t) = c0 + (t - t0) u^B, x the integer cell coordinates:
 *   sharp (eps = 0): d = 0 iff |x - c|^2 <= R^2;
 *   ramp  (eps > 0): d = clamp(phi/eps + 1/2, 0, 1), phi = |x - c| - R the signed distance (Eq.15 with the linear
 *                    profile Eq.16; eps_b read as eps_h, A14).
 * dipole B^B(r) = 1/2 B_s (R / max(|r|, R/2))^3 [3 (m.r^) r^ - m], r^ = r/|r| (0 at r = 0).
 * Mask / porosity field: d = dfield[n] if given, else 0 for SOLID cells; u^B uniform, B^B per cell. */
/* v rotated about the axis Omega by the angle |Omega| dt (Rodrigues); v itself when Omega = 0 */
static void rotate_about(const double om[3], double dt, const double v[3], double out[3])
{
  double om2 = om[0] * om[0] + om[1] * om[1] + om[2] * om[2];
  out[0] = v[0]; out[1] = v[1]; out[2] = v[2];
  if (om2 > 0.0) {
    double omn = sqrt(om2), th = omn * dt, cth = cos(th), sth = sin(th);
    double e[3] = { om[0] / omn, om[1] / omn, om[2] / omn };
    double ev = e[0] * v[0] + e[1] * v[1] + e[2] * v[2];
    double ex[3] = { e[1] * v[2] - e[2] * v[1], e[2] * v[0] - e[0] * v[2], e[0] * v[1] - e[1] * v[0] };
    for (int a = 0; a < 3; a++) out[a] = v[a] * cth + ex[a] * sth + e[a] * ev * (1.0 - cth);
  }
}

static double solid_state(const oracle_t *o, int x, int y, int z, long n, double uB[3], double BB[3])
{
  if (o->has_sphere) {
    double dt = (double)(o->t - o->sph_t0);
    double r[3], xi[3] = { (double)x, (double)y, (double)z };
    double r2 = 0.0;
    for (int a = 0; a < 3; a++) {
      double c = o->sph_c0[a] + dt * o->sph_u[a];
      r[a] = a < o->L.D ? xi[a] - c : 0.0;
      r2 = r2 + r[a] * r[a];
    }
    double rn = sqrt(r2);
    double d;
    if (o->sph_eps > 0.0) {
      d = (rn - o->sph_R) / o->sph_eps + 0.5;
      if (d < 0.0) d = 0.0;
      if (d > 1.0) d = 1.0;
    } else {
      d = r2 <= o->sph_R * o->sph_R ? 0.0 : 1.0;
    }
    if (d < 1.0) {
      BB[0] = BB[1] = BB[2] = 0.0;
      for (int j = 0; j < o->n_dip; j++) {
        /* offset and axis at this step: body-frame vectors rotated about Omega by |Omega| (t - t0) */
        double mt[3], ot[3], rj[3], rj2 = 0.0;
        rotate_about(o->sph_om, dt, o->dip_m[j], mt);
        rotate_about(o->sph_om, dt, o->dip_off[j], ot);
        for (int a = 0; a < 3; a++) { rj[a] = a < o->L.D ? r[a] - ot[a] : 0.0; rj2 = rj2 + rj[a] * rj[a]; }
        double rjn = sqrt(rj2);
        double rc = rjn > o->dip_core[j] ? rjn : o->dip_core[j];
        double q = o->sph_R / rc;
        double amp = 0.5 * o->dip_Bs[j] * (q * q * q);
        double rh[3], mr = 0.0;
        for (int a = 0; a < 3; a++) { rh[a] = rjn > 0.0 ? rj[a] / rjn : 0.0; mr += mt[a] * rh[a]; }
        for (int a = 0; a < 3; a++) BB[a] += amp * (3.0 * mr * rh[a] - mt[a]);
      }
      /* rigid body: u^B = u_s + Omega x r ("rotated around a ... tilt vector") */
      uB[0] = o->sph_u[0] + (o->sph_om[1] * r[2] - o->sph_om[2] * r[1]);
      uB[1] = o->sph_u[1] + (o->sph_om[2] * r[0] - o->sph_om[0] * r[2]);
      uB[2] = o->sph_u[2] + (o->sph_om[0] * r[1] - o->sph_om[1] * r[0]);
      return d;
    }
  }
  double d = 1.0;
  if (o->dfield) d = o->dfield[n];
  else if (o->mask[n] == ORC_CELL_SOLID) d = 0.0;
  if (d < 1.0) {
    double xi[3] = { (double)x, (double)y, (double)z }, r[3];
    for (int a = 0; a < 3; a++) r[a] = a < o->L.D ? xi[a] - o->obs_c[a] : 0.0;
    uB[0] = o->usolid[0] + (o->obs_om[1] * r[2] - o->obs_om[2] * r[1]);
    uB[1] = o->usolid[1] + (o->obs_om[2] * r[0] - o->obs_om[0] * r[2]);
    uB[2] = o->usolid[2] + (o->obs_om[0] * r[1] - o->obs_om[1] * r[0]);
    for (int a = 0; a < 3; a++) BB[a] = o->Bsolid ? o->Bsolid[(long)a * o->N + n] : 0.0;
  }
  return d;
}

/* ---- one cell of one step ---- */
static void cell_update(const oracle_t *o, const double *src, double *dst, int x, int y, int z, double *srcacc)
{
  const lattice_t *L = &o->L;
  const int K = o->K, Qn = L->Q, D = L->D;
  const int nn[3] = { o->p.nx, o->p.ny, o->p.nz };
  const int xi[3] = { x, y, z };
  const long n = cell_index(o, x, y, z);
  const long N = o->N;
  int k, i, a, b;

  /* frozen: mask FROZEN or on an INFLOW face (A10): g' = g */
  int frozen = o->mask[n] == ORC_CELL_FROZEN;
  for (a = 0; a < D; a++) {
    if (xi[a] == 0 && o->p.bc[2 * a] == ORC_BC_INFLOW) frozen = 1;
    if (xi[a] == nn[a] - 1 && o->p.bc[2 * a + 1] == ORC_BC_INFLOW) frozen = 1;
  }
  if (frozen) {
    for (k = 0; k < K; k++) for (i = 0; i < Qn; i++) dst[((long)k * Qn + i) * N + n] = src[((long)k * Qn + i) * N + n];
    return;
  }

  /* 1. pull  f[k][i] = g[k][i](x - c_i); periodic wrap; A9 substitution when the source is outside */
  double f[MAXK][MAXQ];
  int have_nb = 0;
  double Qnb[MAXK], Phinb[MAXK][3];
  for (i = 0; i < Qn; i++) {
    int s[3] = { x, y, z }, outside = 0;
    for (a = 0; a < D; a++) {
      s[a] = xi[a] - L->c[i][a];
      if (s[a] < 0) { if (o->p.bc[2 * a] == ORC_BC_PERIODIC) s[a] += nn[a]; else outside = 1; }
      else if (s[a] >= nn[a]) { if (o->p.bc[2 * a + 1] == ORC_BC_PERIODIC) s[a] -= nn[a]; else outside = 1; }
    }
    if (!outside) {
      long ns = cell_index(o, s[0], s[1], s[2]);
      for (k = 0; k < K; k++) f[k][i] = src[((long)k * Qn + i) * N + ns];
    } else {
      if (!have_nb) {
        /* A9 / PAPER.md:154: take the state of the next cell along the inward discrete normal */
        int q[3] = { x, y, z };
        for (a = 0; a < D; a++) {
          if (xi[a] == 0 && o->p.bc[2 * a] != ORC_BC_PERIODIC) q[a] = xi[a] + 1;
          if (xi[a] == nn[a] - 1 && o->p.bc[2 * a + 1] != ORC_BC_PERIODIC) q[a] = xi[a] - 1;
        }
        long nb = cell_index(o, q[0], q[1], q[2]);
        for (k = 0; k < K; k++) {
          double sum = 0.0;
          for (int j = 0; j < Qn; j++) sum += src[((long)k * Qn + j) * N + nb];
          Qnb[k] = sum;
        }
        memset(Phinb, 0, sizeof Phinb);
        flux_eval(&o->p, D, Qnb, Phinb);
        have_nb = 1;
      }
      for (k = 0; k < K; k++) f[k][i] = feq_eval(L, i, Qnb[k], Phinb[k]);
    }
  }

  /* 2. zeroth moments (Eq.4), sums in index order */
  double Qv[MAXK];
  for (k = 0; k < K; k++) { double sum = 0.0; for (i = 0; i < Qn; i++) sum += f[k][i]; Qv[k] = sum; }

  /* 3. local div B estimate (A6): delta = - tr Pi_B / (tau_B c_s^2) */
  double tr = 0.0;
  for (b = 0; b < D; b++) for (i = 0; i < Qn; i++) tr += (double)L->c[i][b] * f[o->iB + b][i];
  /* A20: cell-local tau_B from the current (INCRES with eta_jc > 0) */
  double tauB = o->tauB;
  if (o->p.scheme == ORC_INCRES && o->p.eta_jc > 0.0) {
    double Phieq[MAXK][3], Pi[3][3], a2 = 0.0;
    memset(Phieq, 0, sizeof Phieq);
    flux_eval(&o->p, D, Qv, Phieq);
    for (a = 0; a < D; a++) for (b = 0; b < D; b++) {
      double m = 0.0;
      for (i = 0; i < Qn; i++) m += (double)L->c[i][a] * f[o->iB + b][i];
      Pi[a][b] = m - Phieq[o->iB + b][a];
    }
    for (a = 0; a < D; a++) for (b = a + 1; b < D; b++) { double w2 = Pi[a][b] - Pi[b][a]; a2 += w2 * w2; }
    a2 /= L->cs2 * L->cs2;
    tauB = tau_of_current(o->tauB, o->tauB - 0.5, a2, o->p.eta_jc);
  }
  double delta = -tr / (tauB * L->cs2);
  /* IDEAL_DIVB: div B from the relaxation variable instead, D ~ tau_M div B (Eq.7) */
  if (o->p.scheme == ORC_IDEAL_DIVB) delta = Qv[8] / o->p.tau_relax;
  /* RESIST: div B = tr g = sum_a G_aa / tau_M */
  if (o->p.scheme == ORC_RESIST || o->p.scheme == ORC_FULL) {
    delta = 0.0;
    for (a = 0; a < D; a++) delta += Qv[8 + 3 * a + a] / o->p.tau_relax;
  }

  /* 4. Powell source (Eq.12), direct injection (A5) */
  double S[MAXK];
  for (k = 0; k < K; k++) S[k] = 0.0;
  double kd = o->p.powell * delta;
  if (is_ideal(o->p.scheme)) {
    double u[3], uBdot = 0.0;
    for (b = 0; b < 3; b++) { u[b] = Qv[1 + b] / Qv[0]; uBdot += u[b] * Qv[5 + b]; }
    for (b = 0; b < 3; b++) { S[1 + b] = -kd * Qv[5 + b]; S[5 + b] = -kd * u[b]; }
    S[4] = -kd * uBdot;
    if (o->p.scheme == ORC_IDEAL_DIVB) S[8] = -Qv[8] / o->p.tau_relax;      /* relaxation source of Eq.6 */
    if (o->p.scheme == ORC_RESIST || o->p.scheme == ORC_FULL) for (k = 8; k < K; k++) S[k] = -Qv[k] / o->p.tau_relax;
  } else {
    for (b = 0; b < D; b++) { S[1 + b] = -kd * Qv[1 + D + b]; S[1 + D + b] = -kd * Qv[1 + b]; }
  }

  /* 5. homogenised solid (Eq.13-14, A8): Q^ and the shift dQh = Q^ - Q; source scaled by d */
  double Qh[MAXK], dQh[MAXK];
  for (k = 0; k < K; k++) { Qh[k] = Qv[k]; dQh[k] = 0.0; }
  double uSol[3], BSol[3];
  double d = solid_state(o, x, y, z, n, uSol, BSol);
  if (d < 1.0) {
    if (is_ideal(o->p.scheme)) {
      double rho = Qv[0], u[3], uh[3], Bh[3], mu = 0.0, B2 = 0.0, uh2 = 0.0, Bh2 = 0.0;
      for (b = 0; b < 3; b++) {
        u[b] = Qv[1 + b] / rho;
        mu += Qv[1 + b] * u[b];
        B2 += Qv[5 + b] * Qv[5 + b];
      }
      double p = (o->p.gamma - 1.0) * (Qv[4] - 0.5 * mu - 0.5 * B2);
      for (b = 0; b < 3; b++) {
        uh[b] = d * u[b] + (1.0 - d) * uSol[b];
        Bh[b] = d * Qv[5 + b] + (1.0 - d) * BSol[b];
        uh2 += uh[b] * uh[b];
        Bh2 += Bh[b] * Bh[b];
      }
      for (b = 0; b < 3; b++) { Qh[1 + b] = rho * uh[b]; Qh[5 + b] = Bh[b]; }
      Qh[4] = p / (o->p.gamma - 1.0) + 0.5 * rho * uh2 + 0.5 * Bh2;
    } else {
      for (b = 0; b < D; b++) {
        Qh[1 + b] = d * Qv[1 + b] + (1.0 - d) * uSol[b];
        Qh[1 + D + b] = d * Qv[1 + D + b] + (1.0 - d) * BSol[b];
      }
    }
    /* the Powell rows are scaled by the porosity (A8); the relaxation of D is intrinsic and is not */
    for (k = 0; k < K; k++) { dQh[k] = Qh[k] - Qv[k]; if (k < 8 || !is_ideal(o->p.scheme)) S[k] *= d; }
    if (srcacc) {   /* body integrals (A21) */
      double *bd = srcacc + MAXK;
      const int nvec = is_ideal(o->p.scheme) ? 3 : D;
      double r[3] = { 0.0, 0.0, 0.0 }, Fm[3] = { 0.0, 0.0, 0.0 };
      for (a = 0; a < D; a++) {
        double ref = o->has_sphere ? o->sph_c0[a] + (double)(o->t - o->sph_t0) * o->sph_u[a] : o->body_ref[a];
        r[a] = (double)xi[a] - ref;
      }
      for (b = 0; b < nvec; b++) {
        Fm[b] = -dQh[o->iU + b];
        bd[b] += Fm[b];
        bd[7 + b] += dQh[o->iB + b];
        bd[10 + b] += (1.0 - d) * Qv[o->iB + b];
      }
      bd[3] += r[1] * Fm[2] - r[2] * Fm[1];
      bd[4] += r[2] * Fm[0] - r[0] * Fm[2];
      bd[5] += r[0] * Fm[1] - r[1] * Fm[0];
      if (is_ideal(o->p.scheme)) bd[6] += -dQh[4];
      bd[13] += 1.0 - d;
    }
  }
  if (srcacc) for (k = 0; k < K; k++) srcacc[k] += S[k];

  /* 6. flux of the (blended) state (Eq.11) */
  double Phi[MAXK][3];
  memset(Phi, 0, sizeof Phi);
  flux_eval(&o->p, D, Qh, Phi);

  /* 7./8. BGK + direct injection (Eq.2-3), store */
  for (k = 0; k < K; k++)
    for (i = 0; i < Qn; i++) {
      double feq = feq_eval(L, i, Qv[k], Phi[k]);
      double om = (k >= o->iB && k < o->iB + (is_ideal(o->p.scheme) ? 3 : D) && tauB != o->tauB) ? 1.0 / tauB : o->omega[k];
      dst[((long)k * Qn + i) * N + n] = f[k][i] + om * (feq - f[k][i]) + L->w[i] * (dQh[k] + S[k]);
    }
}

int oracle_step(oracle_t *o, int n_steps)
{
  if (!o || n_steps < 0) return -1;
  const int nx = o->p.nx, ny = o->p.ny, nz = o->p.nz;
  const long rows = (long)ny * nz;
  double *rowacc = (double *)calloc((size_t)rows * ACCW, sizeof(double));
  if (!rowacc) return -2;
  for (int s = 0; s < n_steps; s++) {
    const double *src = o->g[o->cur];
    double *dst = o->g[1 - o->cur];
    memset(rowacc, 0, (size_t)rows * ACCW * sizeof(double));
    if (rows >= 4) {
#pragma omp parallel for schedule(static) num_threads(oracle_get_threads())
      for (long r = 0; r < rows; r++) {
        int z = (int)(r / ny), y = (int)(r % ny);
        for (int x = 0; x < nx; x++) cell_update(o, src, dst, x, y, z, rowacc + r * ACCW);
      }
    } else {
      /* 1D / thin domains: parallelise over x, source log kept serial-free by per-cell slots */
      double *cellacc = (double *)calloc((size_t)o->N * ACCW, sizeof(double));
      if (!cellacc) { free(rowacc); return -2; }
#pragma omp parallel for schedule(static) num_threads(oracle_get_threads())
      for (long n = 0; n < o->N; n++) {
        int x = (int)(n % nx), y = (int)((n / nx) % ny), z = (int)(n / ((long)nx * ny));
        cell_update(o, src, dst, x, y, z, cellacc + n * ACCW);
      }
      for (long n = 0; n < o->N; n++) for (int k = 0; k < ACCW; k++) rowacc[k] += cellacc[n * ACCW + k];
      free(cellacc);
    }
    for (long r = 0; r < rows; r++) {
      for (int k = 0; k < o->K; k++) o->srclog[k] += rowacc[r * ACCW + k];
      for (int j = 0; j < NBODY; j++) o->body[j] += rowacc[r * ACCW + MAXK + j];
    }
    o->cur = 1 - o->cur;
    o->t += 1;
  }
  free(rowacc);
  return 0;
}

/* ---- moments and diagnostics of the stored populations (Eq.4) ----
 * diag = [ sum_x Q_k (K) | sum_x |Q_k| (K) | max_x |Q_k| (K) | max|div_h B|, min rho, min p, flag ]
 * div_h B(x) = sum_i w_i c_i . B(x + c_i) / c_s^2 (P4), neighbour index wrapped on periodic axes and
 * clamped on the others.  flag: +1 if any non-finite value, +2 if any rho <= 0.
 * INCRES: "min rho" slot = 1 (constant density), "min p" slot = min P. */
int oracle_moments(oracle_t *o, double *fields_out, double *diag_out)
{
  if (!o) return -1;
  const lattice_t *L = &o->L;
  const int K = o->K, Qn = L->Q, D = L->D;
  const long N = o->N;
  const double *g = o->g[o->cur];
  double *F = fields_out;
  double *tmp = NULL;
  if (!F) { tmp = (double *)malloc((size_t)K * N * sizeof(double)); if (!tmp) return -2; F = tmp; }
  for (int k = 0; k < K; k++)
    for (long n = 0; n < N; n++) {
      double sum = 0.0;
      for (int i = 0; i < Qn; i++) sum += g[((long)k * Qn + i) * N + n];
      F[(long)k * N + n] = sum;
    }
  if (diag_out) {
    const int nn[3] = { o->p.nx, o->p.ny, o->p.nz };
    int flag_nan = 0, flag_rho = 0;
    for (int k = 0; k < K; k++) {
      double s = 0.0, sa = 0.0, mx = 0.0;
      for (long n = 0; n < N; n++) {
        double v = F[(long)k * N + n];
        if (!isfinite(v)) flag_nan = 1;
        s += v; sa += fabs(v);
        if (fabs(v) > mx) mx = fabs(v);
      }
      diag_out[k] = s; diag_out[K + k] = sa; diag_out[2 * K + k] = mx;
    }
    double maxdiv = 0.0, minrho = INFINITY, minp = INFINITY;
    for (int z = 0; z < nn[2]; z++) for (int y = 0; y < nn[1]; y++) for (int x = 0; x < nn[0]; x++) {
      const int xi[3] = { x, y, z };
      long n = cell_index(o, x, y, z);
      double div = 0.0;
      for (int i = 0; i < Qn; i++) {
        int q[3] = { x, y, z };
        for (int a = 0; a < D; a++) {
          q[a] = xi[a] + L->c[i][a];
          if (q[a] < 0) q[a] = o->p.bc[2 * a] == ORC_BC_PERIODIC ? q[a] + nn[a] : 0;
          else if (q[a] >= nn[a]) q[a] = o->p.bc[2 * a + 1] == ORC_BC_PERIODIC ? q[a] - nn[a] : nn[a] - 1;
        }
        long nq = cell_index(o, q[0], q[1], q[2]);
        double cB = 0.0;
        for (int a = 0; a < D; a++) cB += (double)L->c[i][a] * F[(long)(o->iB + a) * N + nq];
        div += L->w[i] * cB;
      }
      div /= L->cs2;
      if (fabs(div) > maxdiv) maxdiv = fabs(div);
      if (is_ideal(o->p.scheme)) {
        double rho = F[n], mu = 0.0, B2 = 0.0;
        for (int b = 0; b < 3; b++) {
          double m = F[(long)(1 + b) * N + n], B = F[(long)(5 + b) * N + n];
          mu += m * (m / rho); B2 += B * B;
        }
        double p = (o->p.gamma - 1.0) * (F[4 * N + n] - 0.5 * mu - 0.5 * B2);
        if (rho < minrho) minrho = rho;
        if (p < minp) minp = p;
        if (!(rho > 0.0)) flag_rho = 1;
      } else {
        if (F[n] < minp) minp = F[n];
        minrho = 1.0;
      }
    }
    diag_out[3 * K] = maxdiv; diag_out[3 * K + 1] = minrho; diag_out[3 * K + 2] = minp;
    diag_out[3 * K + 3] = (double)(flag_nan + 2 * flag_rho);
  }
  free(tmp);
  return 0;
}
