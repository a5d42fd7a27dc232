/* vlbm_oracle.h — CPU ORACLE for the vectorial lattice Boltzmann MHD step.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this.  The CUDA product path shares no code, header, table or
 * helper with this file and never calls it.
 *
 * What it is: the algorithm of arxiv/paper_2606_00641 written out step by step, per cell, in fp64,
 * in the paper's order and notation (§2.2 Eq.2-5, §2.3 Eq.8, Eq.11, Eq.12, §2.4 Eq.13-14),
 * with the readings A1-A15 of SURVEY.md §8c-2 / DESIGN.md §3 where the paper is silent.
 * No blocking, fusion or reordering; A/B population arrays; OpenMP on the cell loop only.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1 equilibrium moments, P2 uniform invariance,
 * P3 conservation, P4 div B, P5/P5b linear waves (closed form + exact Fourier symbol), P6 numpy
 * brute force, P7 symmetries, P8 hydrodynamic limits, P9 obstacle, P10 boundaries, P12 body integrals (tests/test_oracle_body.py).
 * Parity unpinned: absolute accuracy against the paper's figures (data not available) and the
 * readings A3, A6, A8-A12 themselves (choices, not facts of the paper) — see DESIGN.md §3.
 */
#ifndef VLBM_ORACLE_H
#define VLBM_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_D1Q3 = 1, ORC_D2Q9 = 2, ORC_D3Q19 = 3, ORC_D2Q5 = 4, ORC_D3Q7 = 5 };
enum { ORC_IDEAL = 0, ORC_INCRES = 1, ORC_IDEAL_DIVB = 2, ORC_RESIST = 3, ORC_FULL = 4 };
enum { ORC_BC_PERIODIC = 0, ORC_BC_ZEROGRAD = 1, ORC_BC_INFLOW = 2 };
enum { ORC_CELL_FLUID = 0, ORC_CELL_FROZEN = 1, ORC_CELL_SOLID = 2 };

typedef struct {
  int scheme;      /* ORC_IDEAL: Q = (rho, m_x, m_y, m_z, E, B_x, B_y, B_z), K = 8 in every dimension
                      ORC_INCRES: Q = (P, u_1..u_D, B_1..B_D), K = 1 + 2 D                  (A2, A3)
                      ORC_IDEAL_DIVB: IDEAL + D = tr G, K = 9             (A19)
                      ORC_RESIST: IDEAL + G_ab = tau_M d_a B_b (a < D, b < 3; index 8 + 3a + b), K = 8 + 3 D, resistive
                                  fluxes -eta grad B and eta j x B from G (Eq.9-10)  (A22)
                      ORC_FULL: RESIST + H_ab = tau_M d_a u_b (index 8 + 3 D + 3a + b), K = 8 + 6 D: the full dissipative system of
                                PAPER.md:122 with the viscous stress -tau, -u.tau from H (Eq.9)          (A23) */
  int lattice;     /* ORC_D1Q3 / D2Q9 / D3Q19 (A2); D2Q5 / D3Q7 are the paper's own */
  int nx, ny, nz;  /* unused dims = 1 */
  double gamma;    /* IDEAL: adiabatic index, Eq.8 */
  double c0sq;     /* INCRES: artificial sound speed squared (A3) */
  double nu, eta;  /* if > 0: tau of the velocity / magnetic sets := 1/2 + D / c_s^2 (Eq.5);
                      ORC_RESIST, ORC_FULL: eta is the magnetic diffusivity of the flux terms instead and leaves tau alone;
                      ORC_FULL: nu is the shear viscosity mu of the flux terms likewise */
  double tau[32];  /* per variable, > 1/2, variable order of `scheme` */
  double tau_relax; /* IDEAL_DIVB, RESIST, FULL: relaxation time tau_M of the gradient variables (Eq.6), lattice units, > 0 */
  double eta_jc;   /* INCRES: critical current j_c of eta(j) = eta0 (1 + (j/j_c)^2), lattice units; 0 = constant eta */
  double powell;   /* kappa: 0 = off, 1 = Eq.12 */
  int bc[6];       /* xmin, xmax, ymin, ymax, zmin, zmax */
} oracle_params;

typedef struct oracle oracle_t;

int  oracle_num_vars(const oracle_params *p);      /* K */
int  oracle_num_dirs(const oracle_params *p);      /* Q */

int  oracle_create(const oracle_params *p, const unsigned char *cell_mask /* [N] or NULL */, oracle_t **out);
void oracle_destroy(oracle_t *o);
int  oracle_init(oracle_t *o, const double *fields /* [K][nz][ny][nx] */);
int  oracle_step(oracle_t *o, int n_steps);
/* diag_out[3K+4] = sum Q_k | sum |Q_k| | max |Q_k| | max|div_h B|, min rho, min p, flag */
int  oracle_moments(oracle_t *o, double *fields_out /* [K][N] or NULL */, double *diag_out /* or NULL */);
int  oracle_set_obstacle(oracle_t *o, const unsigned char *mask /* [N] */, const double u_solid[3],
                         const double *B_solid /* [3][N] or NULL (-> 0) */);
int  oracle_set_sphere(oracle_t *o, const double centre[3], double radius, const double u_solid[3],
                       const double dipole_dir[3], double B_surface);

/* fractional porosity (Eq.15-16): per-cell d in [0,1] for the masked solid (NULL = back to the mask),
 * linear ramp of width eps across the sphere surface (0 = sharp) */
int  oracle_set_porosity(oracle_t *o, const double *d_field /* [N] or NULL */);
int  oracle_set_sphere_width(oracle_t *o, double eps);
/* rigid rotation of the sphere: u^B(x) = u_solid + omega x (x - c), dipole axis rotates with the body */
int  oracle_set_sphere_rotation(oracle_t *o, const double omega[3]);

/* ensemble of n <= 4 shifted, smoothed dipoles fixed in the body frame of the sphere, replacing the single
 * dipole of oracle_set_sphere: offset[n][3] from the centre, dir[n][3], B_surface[n], core[n] (cap radius, > 0) */
int  oracle_set_sphere_dipoles(oracle_t *o, int n, const double *offset, const double *dir, const double *B_surface,
                               const double *core);
/* masked / porosity bodies: u^B(x) = u_solid + omega x (x - centre) */
int  oracle_set_obstacle_rotation(oracle_t *o, const double omega[3], const double centre[3]);

/* body integrals (A21), accumulated over the steps since init or the last reset:
 * out[14] = F[3] | T[3] | W | I_B[3] | sum (1-d) B [3] | sum (1-d);  see vlbm_oracle.c */
int  oracle_body_read(oracle_t *o, double *out /* [14] or NULL */, int reset);
int  oracle_set_body_reference(oracle_t *o, const double ref[3]);   /* torque reference of masked bodies (default 0) */

/* test hooks */
double oracle_tau_of_current(double tau0, double e0, double a2, double jc);
int  oracle_get_populations(oracle_t *o, double *g_out /* [K][Q][N] */);
int  oracle_set_populations(oracle_t *o, const double *g_in /* [K][Q][N] */);
int  oracle_source_log(oracle_t *o, double *acc /* [K]: accumulated sum_x d*S_k over all steps so far */);
int  oracle_lattice(int lattice, int *D, int *Q, int *c /* [Q][3] */, double *w /* [Q] */, double *cs2);
int  oracle_flux(const oracle_params *p, const double *Qv /* [K] */, double *Phi /* [K][3] */);
int  oracle_equilibrium(const oracle_params *p, const double *Qv /* [K] */, double *feq /* [K][Q] */);
void oracle_set_threads(int n);   /* 0 = OpenMP default */
int  oracle_get_threads(void);

#ifdef __cplusplus
}
#endif
#endif
