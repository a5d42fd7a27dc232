/* oracle_sanitize_main.c — drives oracle/vlbm_oracle.c through every scheme, lattice and boundary kind on small grids,
 * with a mask, a porosity field, a moving, spinning sphere with a dipole ensemble, body integrals and population I/O.
 * Built by tests/test_oracle_sanitize.py with gcc -fsanitize=address,undefined -fno-sanitize-recover and run once: an
 * out-of-bounds index, a use after free, a leak, signed overflow or a misaligned access in the oracle fails the test.
 * Test infrastructure; prints "ok <checksum>". */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../oracle/vlbm_oracle.h"

static unsigned long long rng_state = 88172645463325252ULL;
static double urand(void) {
  rng_state ^= rng_state << 13; rng_state ^= rng_state >> 7; rng_state ^= rng_state << 17;
  return (double)(rng_state >> 11) / 9007199254740992.0;
}

static double run_case(int scheme, int lattice, int nx, int ny, int nz, const int bc[6], int with_body) {
  oracle_params p;
  memset(&p, 0, sizeof p);
  p.scheme = scheme; p.lattice = lattice; p.nx = nx; p.ny = ny; p.nz = nz;
  p.gamma = 5.0 / 3.0; p.c0sq = 1.0 / 36.0; p.powell = 1.0; p.tau_relax = 3.0;
  if (scheme == ORC_RESIST || scheme == ORC_FULL) p.eta = 0.01;
  if (scheme == ORC_FULL) p.nu = 0.01;
  for (int k = 0; k < 32; k++) p.tau[k] = 0.7;
  for (int j = 0; j < 6; j++) p.bc[j] = bc[j];
  const int K = oracle_num_vars(&p), Q = oracle_num_dirs(&p);
  const int D = lattice == ORC_D1Q3 ? 1 : ((lattice == ORC_D2Q9 || lattice == ORC_D2Q5) ? 2 : 3);
  const size_t N = (size_t)nx * ny * nz;
  unsigned char *mask = (unsigned char *)calloc(N, 1);
  double *F = (double *)calloc((size_t)K * N, sizeof(double));
  double *out = (double *)malloc((size_t)K * N * sizeof(double));
  double *g = (double *)malloc((size_t)K * Q * N * sizeof(double));
  double *dfield = (double *)malloc(N * sizeof(double));
  double *Bs = (double *)malloc(3 * N * sizeof(double));
  double diag[3 * 32 + 4];
  for (size_t n = 0; n < N; n++) {
    if (with_body && urand() < 0.05) mask[n] = ORC_CELL_SOLID;
    if (with_body && urand() < 0.02) mask[n] = ORC_CELL_FROZEN;
    dfield[n] = urand();
    for (int c = 0; c < 3; c++) Bs[(size_t)c * N + n] = 0.05 * (urand() - 0.5);
    if (scheme == ORC_INCRES) {
      for (int k = 1; k < K; k++) F[(size_t)k * N + n] = 0.03 * (urand() - 0.5);
    } else {
      const double rho = 1.0 + 0.1 * urand(), pr = 0.05 + 0.01 * urand();
      double u[3], B[3], u2 = 0, B2 = 0;
      for (int c = 0; c < 3; c++) { u[c] = 0.05 * (urand() - 0.5); B[c] = 0.05 * (urand() - 0.5); u2 += u[c] * u[c]; B2 += B[c] * B[c]; }
      F[n] = rho;
      for (int c = 0; c < 3; c++) { F[(size_t)(1 + c) * N + n] = rho * u[c]; F[(size_t)(5 + c) * N + n] = B[c]; }
      F[(size_t)4 * N + n] = pr / (p.gamma - 1.0) + 0.5 * rho * u2 + 0.5 * B2;
      for (int k = 8; k < K; k++) F[(size_t)k * N + n] = 0.01 * (urand() - 0.5);
    }
  }
  oracle_t *o = NULL;
  if (oracle_create(&p, with_body ? mask : NULL, &o) != 0 || !o) { fprintf(stderr, "create failed\n"); exit(2); }
  if (with_body) {
    const double us[3] = {0.02, -0.01, 0.01}, om[3] = {0.0, 0.0, 0.01}, cen[3] = {nx / 2.0, ny / 2.0, nz / 2.0};
    oracle_set_obstacle(o, mask, us, Bs);
    oracle_set_obstacle_rotation(o, om, cen);
    if (with_body > 1) oracle_set_porosity(o, dfield);
    if (D >= 2 && scheme != ORC_INCRES) {
      const double sc[3] = {nx / 3.0, ny / 2.0, nz / 2.0}, su[3] = {-0.25, 0.0, 0.0}, m[3] = {0.3, -0.5, 0.8};
      const double off[2][3] = {{1.0, 0.0, 0.0}, {0.0, -1.0, 0.5}}, dir[2][3] = {{0, 0, 1}, {1, 0, 0}}, bs[2] = {0.03, 0.02}, core[2] = {1.5, 1.0};
      oracle_set_sphere(o, sc, 3.0, su, m, 0.03);
      oracle_set_sphere_width(o, 1.5);
      oracle_set_sphere_rotation(o, om);
      oracle_set_sphere_dipoles(o, 2, &off[0][0], &dir[0][0], bs, core);
    }
    const double ref[3] = {1.0, 2.0, 3.0};
    oracle_set_body_reference(o, ref);
  }
  oracle_init(o, F);
  oracle_step(o, 3);
  oracle_get_populations(o, g);
  oracle_set_populations(o, g);
  oracle_step(o, 2);
  oracle_moments(o, out, diag);
  double body[14], acc[32];
  oracle_body_read(o, body, 1);
  oracle_source_log(o, acc);
  double sum = diag[0] + body[13];
  for (int k = 0; k < K; k++) sum += out[(size_t)k * N + N / 2] + acc[k];
  oracle_destroy(o);
  free(mask); free(F); free(out); free(g); free(dfield); free(Bs);
  return sum;
}

int main(void) {
  const int lattices[5] = {ORC_D1Q3, ORC_D2Q9, ORC_D3Q19, ORC_D2Q5, ORC_D3Q7};
  const int dims[5] = {1, 2, 3, 2, 3};
  const int schemes[5] = {ORC_IDEAL, ORC_INCRES, ORC_IDEAL_DIVB, ORC_RESIST, ORC_FULL};
  double sum = 0.0;
  for (int li = 0; li < 5; li++)
    for (int si = 0; si < 5; si++)
      for (int variant = 0; variant < 3; variant++) {
        const int D = dims[li];
        const int nx = 13, ny = D > 1 ? 7 : 1, nz = D > 2 ? 5 : 1;
        int bc[6] = {0, 0, 0, 0, 0, 0};
        if (variant == 1) { bc[0] = ORC_BC_INFLOW; bc[1] = ORC_BC_ZEROGRAD; }
        if (variant == 2) for (int a = 0; a < D; a++) { bc[2 * a] = ORC_BC_ZEROGRAD; bc[2 * a + 1] = ORC_BC_ZEROGRAD; }
        sum += run_case(schemes[si], lattices[li], nx, ny, nz, bc, variant);
      }
  /* eta(j) on INCRES */
  {
    oracle_params p;
    memset(&p, 0, sizeof p);
    p.scheme = ORC_INCRES; p.lattice = ORC_D2Q9; p.nx = 9; p.ny = 8; p.nz = 1; p.c0sq = 1.0 / 36.0; p.eta_jc = 0.02; p.powell = 1.0;
    for (int k = 0; k < 32; k++) p.tau[k] = 0.6;
    oracle_t *o = NULL;
    if (oracle_create(&p, NULL, &o) != 0) return 2;
    double F[5 * 72];
    for (int j = 0; j < 5 * 72; j++) F[j] = j < 72 ? 0.0 : 0.03 * (urand() - 0.5);
    oracle_init(o, F);
    oracle_step(o, 4);
    double dg[3 * 5 + 4];
    oracle_moments(o, NULL, dg);
    sum += dg[1] + oracle_tau_of_current(0.6, 0.1 / 3.0, 0.3, 0.02);
    oracle_destroy(o);
  }
  if (!isfinite(sum)) { fprintf(stderr, "non-finite checksum\n"); return 3; }
  printf("ok %.17g\n", sum);
  return 0;
}
