/* lbmhd.h — C ABI of the B200-native vectorial lattice Boltzmann step for MHD.
 *
 * Implements the data-parallel hot path of arxiv/paper_2606_00641: every transported
 * variable k carries its own population set f_{k,i}; one step is
 *     f_{k,i}(x + c_i, t+1) = f_{k,i} + Omega^C + Omega^S                      (Eq.2)
 * with the linear equilibrium f^eq_{k,i} = w_i (Q_k + c_i.Phi_k / c_s^2)       (Eq.3),
 * moments Q_k = sum_i f_{k,i}                                                  (Eq.4),
 * BGK collision and direct-injection source, the ideal-MHD flux and EOS
 * (Eq.11, Eq.8), the Powell source (Eq.12), equilibrium-based
 * static boundaries and homogenised moving solids (Eq.13-14).
 * Where the paper is silent the readings A1-A15 of DESIGN.md §3 apply.
 *
 * Conventions
 *  - Everything is in lattice units (dx = dt = 1, c_i in {-1,0,1}^D); the caller scales (A1).
 *  - Macroscopic fields are fp64 SoA [K][nz][ny][nx], x fastest, at this boundary in both precisions.
 *    IDEAL: K = 8 in every dimension, order rho, m_x, m_y, m_z, E, B_x, B_y, B_z.
 *    INCRES: K = 1 + 2D, order P, u_1..u_D, B_1..B_D (P = kinematic pressure carrier, A3).
 *    IDEAL_DIVB: K = 9, the IDEAL order followed by D.
 *    RESIST: K = 8 + 3 D, the IDEAL order followed by G_ab, a-major (variable 8 + 3 a + b).
 *    FULL: K = 8 + 6 D, the RESIST order followed by H_ab, a-major (variable 8 + 3 D + 3 a + b).
 *  - Direction order: rest; +x,-x,+y,-y,+z,-z; diagonals (+,+),(-,-),(+,-),(-,+) per plane xy, xz, yz.
 *  - Every pointer argument says whether it is a HOST or a DEVICE pointer.  The caller owns every
 *    buffer it passes, including `workspace` (device memory, e.g. a torch tensor): the library never
 *    allocates or frees device memory and keeps no host pointer after a call returns.
 *  - All work is enqueued on `stream`; calls that return data to HOST memory synchronise that stream.
 *  - No call throws or aborts.  Return value 0 = success, < 0 = error code below; the text of the last
 *    error (per thread) is available from lbmhd_last_error().
 *  - There is no CPU fallback: without a CUDA device every call that needs one returns LBMHD_ECUDA.
 */
#ifndef LBMHD_H
#define LBMHD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbmhd lbmhd_t;

enum { LBMHD_D1Q3 = 1, LBMHD_D2Q9 = 2, LBMHD_D3Q19 = 3,
       LBMHD_D2Q5 = 4, LBMHD_D3Q7 = 5 /* the paper's own lattices; D3Q7 has c_s^2 = 1/4 */ };
enum { LBMHD_IDEAL = 0, LBMHD_INCRES = 1,
       LBMHD_IDEAL_DIVB = 2 /* IDEAL + the paper's local gradient evolution in traced form: a 9th set
                               D = tr G with flux D u - B and source -D/tau_relax; div B in Eq.12 := D/tau_relax */,
       LBMHD_RESIST = 3 /* dissipative MHD with the magnetic gradients transported (Eq.9-10 PAPER.md:132-136;
                           DESIGN.md A22): IDEAL + G_ab ~ tau_relax d_a B_b (a < D lattice axes, b < 3), flux G (x) u - I (x) B,
                           source -G/tau_relax; induction flux - eta G/tau_relax, energy flux + eta j x B with j = curl B
                           from G; div B in Eq.12 := tr G / tau_relax.  No viscous stress, no heat flux */,
       LBMHD_FULL = 4 /* the full dissipative system of PAPER.md:122 (Eq.9; A23): RESIST + the velocity
                         gradients H_ab ~ tau_relax d_a u_b transported the same way (flux H (x) u - I (x) u, source -H/tau_relax);
                         Newtonian stress sigma = nu (h + h^T - 2/3 tr h I), h = H/tau_relax, enters the momentum flux as -sigma and
                         the energy flux as -u.sigma.  Heat flux q = 0 */ };
enum { LBMHD_BC_PERIODIC = 0, LBMHD_BC_ZEROGRAD = 1, LBMHD_BC_INFLOW = 2,
       LBMHD_BC_HALO = 3 /* slab decomposition, slowest lattice axis only: the plane on this face is a ghost plane */ };
enum { LBMHD_CELL_FLUID = 0, LBMHD_CELL_FROZEN = 1, LBMHD_CELL_SOLID = 2 };
enum { LBMHD_STREAM_AB = 0, LBMHD_STREAM_INPLACE = 1 };
enum {
  LBMHD_OK = 0,
  LBMHD_EINVAL = -1,   /* bad lattice / dims / tau <= 1/2 / NULL / inconsistent boundary kinds */
  LBMHD_ENOMEM = -2,   /* workspace too small or misaligned */
  LBMHD_ECUDA = -3,    /* CUDA error (sticky), text in lbmhd_last_error() */
  LBMHD_ENUMERIC = -4  /* lbmhd_moments saw NaN/Inf or rho <= 0 (p < 0 alone is not an error) */
};

typedef struct {
  int    scheme;        /* LBMHD_IDEAL | LBMHD_INCRES | LBMHD_IDEAL_DIVB | LBMHD_RESIST | LBMHD_FULL */
  int    lattice;       /* LBMHD_D1Q3 | LBMHD_D2Q9 | LBMHD_D3Q19 | LBMHD_D2Q5 | LBMHD_D3Q7 */
  int    precision;     /* 64 (fp64 populations and arithmetic) or 32 (fp32 populations and arithmetic) */
  int    nx, ny, nz;    /* unused dims = 1 */
  double gamma;         /* IDEAL: adiabatic index, Eq.8 */
  double c0sq;          /* INCRES: artificial sound speed squared (A3) */
  double nu, eta;       /* if > 0: tau of the velocity (and P) / magnetic sets := 1/2 + D/c_s^2, Eq.5 PAPER.md:98.
                           RESIST, FULL: eta (>= 0) is the magnetic diffusivity of the flux terms instead and leaves tau alone;
                           FULL: nu (>= 0) is the shear viscosity mu of the flux terms likewise */
  double tau[32];       /* per variable (first K <= 26 used), > 1/2, order of `scheme`; all magnetic sets must share one value (A7) */
  double tau_relax;     /* IDEAL_DIVB, RESIST, FULL: relaxation time tau_M of the gradient variables (Eq.6), lattice units, > 0 */
  double eta_jc;        /* INCRES: critical current j_c of eta(j) = eta0 (1 + (j/j_c)^2) (eta0 from `eta` or tau),
                           lattice units; 0 = constant resistivity */
  double powell;        /* kappa: 0 = off, 1 = Eq.12 */
  int    bc[6];         /* xmin, xmax, ymin, ymax, zmin, zmax; periodic must be paired per axis */
  int    halo_offset;   /* slab decomposition: global index of local plane 0 along the slowest lattice axis (0 otherwise);
                           only the analytic sphere looks at it */
  int    streaming;     /* LBMHD_STREAM_AB (two population copies) | LBMHD_STREAM_INPLACE (one copy, AA pattern:
                           same results; a FROZEN cell is re-emitted as f^eq of its moments, which is what it holds
                           after lbmhd_init; host-pointer population I/O needs LBMHD_STREAM_AB) */
  int    device;        /* CUDA device ordinal */
  void  *stream;        /* cudaStream_t to enqueue on (0 = default stream) */
  void  *workspace;     /* DEVICE pointer, 256-byte aligned, >= lbmhd_workspace_bytes() (or _min()) bytes */
  size_t workspace_bytes;
} lbmhd_params;

/* K (number of population sets) and Q (directions) for the scheme/lattice in *p; < 0 on bad input. */
int lbmhd_num_vars(const lbmhd_params *p);
int lbmhd_num_dirs(const lbmhd_params *p);

/* Device bytes the handle needs: populations (1 or 2 copies of K*Q planes), cell mask, moments scratch, reduction scratch and,
 * last, the per-cell solid field B_solid (3 N fp64) and porosity field (N fp64).  lbmhd_workspace_bytes_min leaves that
 * optional tail out: a handle created on such a workspace refuses lbmhd_set_obstacle(B_solid != NULL) and
 * lbmhd_set_porosity with LBMHD_ENOMEM and is otherwise identical (config 5: 0.8 GB less).  0 on bad input.  Needs no device. */
size_t lbmhd_workspace_bytes(const lbmhd_params *p);
size_t lbmhd_workspace_bytes_min(const lbmhd_params *p);

/* Validates *p, lays the workspace out, uploads `cell_mask` (HOST uint8 [N], values LBMHD_CELL_*, or
 * NULL = all FLUID).  Cells on a face whose kind is LBMHD_BC_INFLOW are FROZEN whatever the mask says (A10). */
int lbmhd_create(const lbmhd_params *p, const unsigned char *cell_mask, lbmhd_t **out);

/* Frees the handle only (never the workspace). */
void lbmhd_destroy(lbmhd_t *h);

/* g_{k,i} = f^eq_{k,i}(Q) (Eq.3) from `fields` = fp64 [K][N]; HOST pointer if on_device == 0 (copied
 * synchronously through the moments scratch), DEVICE pointer otherwise.  Resets the step counter. */
int lbmhd_init(lbmhd_t *h, const double *fields, int on_device);

/* n_steps >= 0 applications of the fused update (pull-stream, moments, div-B estimate, Powell source,
 * solid blend, flux, BGK + injection, store: DESIGN.md §2), asynchronous on the stream.  A sphere set
 * by lbmhd_set_sphere advances its centre by u_solid per step.  On small lattices (launch-latency bound: BASELINE configs
 * 1 and 2) a call with n_steps >= 2 runs all its steps in ONE cooperative launch (LBMHD_PATH_PERSIST);
 * larger lattices launch one kernel per step.  The results do not depend on which. */
int lbmhd_step(lbmhd_t *h, int n_steps);

/* Q_k(x) = sum_i g_{k,i}(x) of the stored populations into fields_out (fp64 [K][N], NULL to skip) and the
 * diagnostics into diag_out (3K+4 doubles, NULL to skip):
 *   [0,K) sum_x Q_k | [K,2K) sum_x |Q_k| | [2K,3K) max_x |Q_k| | max_x |div_h B|, min rho, min p, flag
 * div_h B = sum_i w_i c_i.B(x + c_i)/c_s^2 (neighbour wrapped on periodic axes, clamped otherwise);
 * flag = 1*(non-finite seen) + 2*(rho <= 0 seen).  INCRES: "min rho" = 1, "min p" = min P.
 * Both pointers are HOST (on_device == 0: the call synchronises) or both DEVICE.
 * Returns LBMHD_ENUMERIC if flag != 0 and the outputs are HOST pointers (outputs are still written). */
int lbmhd_moments(lbmhd_t *h, double *fields_out, double *diag_out, int on_device);

/* Masked solid (A8, A11): cells with mask == LBMHD_CELL_SOLID take u^B = u_solid (HOST double[3]) and
 * B^B from B_solid (fp64 [3][N], NULL = 0); FROZEN cells keep their populations.  mask / B_solid are HOST
 * or DEVICE pointers according to on_device.  Replaces the mask given at create. */
int lbmhd_set_obstacle(lbmhd_t *h, const unsigned char *mask, const double u_solid[3],
                       const double *B_solid, int on_device);

/* Analytic moving sphere with a capped dipole (A12); all arguments HOST.  `centre` is the centre before
 * the next step; before step t it is centre + (t - t_now) u_solid.  A cell is solid iff
 * |x - c|^2 <= radius^2 with x the integer cell coordinates.  radius <= 0 removes the sphere. */
int lbmhd_set_sphere(lbmhd_t *h, const double centre[3], double radius, const double u_solid[3],
                     const double dipole_dir[3], double B_surface);

/* Fractional lattice porosity (Eq.15-16).  lbmhd_set_porosity: d in [0,1] per cell (fp64 [N], HOST or
 * DEVICE per on_device; NULL = back to the mask) for the masked solid: u^ = d u + (1-d) u_solid, B^ likewise (Eq.13-14),
 * u_solid / B_solid as given to lbmhd_set_obstacle.  lbmhd_set_sphere_width: linear ramp d = clamp(phi/eps + 1/2, 0, 1)
 * of width eps (cells) across the sphere surface, phi the signed distance; eps = 0 (default) is the sharp sphere. */
int lbmhd_set_porosity(lbmhd_t *h, const double *d_field, int on_device);
int lbmhd_set_sphere_width(lbmhd_t *h, double eps);

/* Rigid rotation of the sphere: u^B(x) = u_solid + omega x (x - c), omega HOST double[3] in radians per
 * step; the dipole axis rotates with the body about omega, counted from the step lbmhd_set_sphere was called at. */
int lbmhd_set_sphere_rotation(lbmhd_t *h, const double omega[3]);

/* Slab decomposition along the slowest lattice axis (z in 3D, y in 2D), one slab per GPU (the paper's own runs use
 * two GPUs).  A face of kind LBMHD_BC_HALO carries a ghost plane: its cells are never updated or counted here,
 * owned cells pull from them.  The caller moves the crossing populations between neighbouring slabs:
 *   lbmhd_halo_pack(h, side, what, buf)    plane on `side` (0 low, 1 high) -> DEVICE buf
 *   lbmhd_halo_unpack(h, side, what, buf)  DEVICE buf (packed by the neighbour on its opposite side) -> plane on `side`
 * `what`:
 *   LBMHD_HALO_CROSSING  pack reads the owned plane next to the ghost, the directions that leave through the face (5 of 19 on
 *                        D3Q19); unpack writes them into the ghost plane.  A/B streaming: before EVERY step.  In place: before
 *                        every pull-push step (even step count since lbmhd_init / lbmhd_set_populations).
 *   LBMHD_HALO_FULL      the same planes, all Q directions (A/B only; before lbmhd_moments so that div_h B sees the neighbour's
 *                        field — or exchange the ghost planes of the FIELDS and call lbmhd_diagnostics, which works in both
 *                        streaming modes).
 *   LBMHD_HALO_RETURN    in place only, after every pull-push step and before the local step that follows: the boundary cells
 *                        pushed their outgoing populations into the ghost plane; pack reads them there, unpack writes them
 *                        into the neighbour's owned plane next to its ghost (the slots its local step reads).
 * Buffer layout [K][ndir][plane], element type = `precision`, lbmhd_halo_bytes(h, what) bytes.  All calls are asynchronous on
 * the handle's stream; the _on variants run on `stream` instead and, with next_copy != 0, act on the population copy the
 * step IN PROGRESS writes (see lbmhd_step_part), so that the exchange overlaps the interior update. */
enum { LBMHD_HALO_CROSSING = 0, LBMHD_HALO_FULL = 1, LBMHD_HALO_RETURN = 2 };
size_t lbmhd_halo_bytes(const lbmhd_t *h, int what);
int lbmhd_halo_pack(lbmhd_t *h, int side, int what, void *buf);
int lbmhd_halo_unpack(lbmhd_t *h, int side, int what, const void *buf);
int lbmhd_halo_pack_on(lbmhd_t *h, int side, int what, void *buf, int next_copy, void *stream);
int lbmhd_halo_unpack_on(lbmhd_t *h, int side, int what, const void *buf, int next_copy, void *stream);

/* One step in pieces: the fused update of lbmhd_step restricted to the planes [plane_lo, plane_hi) of the slowest lattice
 * axis (local indices, ghost planes included in the count; an empty range launches nothing).  The pieces of one step must
 * cover every owned plane exactly once; the call with last != 0 completes the step (flips the copies / the in-place layout,
 * advances the step counter and the body).  Meant for slabs: update the two planes next to the ghosts first, start their
 * exchange with lbmhd_halo_*_on(next_copy = 1) on another stream, update the interior planes meanwhile.
 * Every piece reads only the state before the step, so the result is identical to one lbmhd_step(h, 1). */
int lbmhd_step_part(lbmhd_t *h, int plane_lo, int plane_hi, int last);

/* The diagnostics of lbmhd_moments (same 3K+4 slots) computed from a DEVICE fields array [K][N] the caller provides — e.g. the
 * output of lbmhd_moments(on_device) after the ghost planes of the FIELDS were refreshed from the neighbouring slabs.
 * diag_out HOST (synchronises, returns LBMHD_ENUMERIC on a flag) or DEVICE per on_device. */
int lbmhd_diagnostics(lbmhd_t *h, const double *fields, double *diag_out, int on_device);

/* Dipole ensemble of the sphere ("an analytical ensemble of four independent, shifted, and smoothed magnetic
 * dipoles"): replaces the single dipole of lbmhd_set_sphere (call that first) by n in 1..4 dipoles fixed in the body frame,
 *   B^B(x) = sum_j 1/2 B_surface[j] (R / max(|r_j|, core[j]))^3 [3 (m_j.r^_j) r^_j - m_j],  r_j = x - c(t) - Rot(t) offset[j],
 * m_j = Rot(t) dir[j], Rot(t) the rotation of lbmhd_set_sphere_rotation since the sphere was set.  HOST arrays offset[n][3],
 * dir[n][3] (used as given, not normalised), B_surface[n], core[n] (> 0, the smoothing radius); copied. */
int lbmhd_set_sphere_dipoles(lbmhd_t *h, int n, const double *offset, const double *dir, const double *B_surface,
                             const double *core);

/* Rigid rotation of the masked / porosity body: u^B(x) = u_solid + omega x (x - centre), global cell
 * coordinates, HOST [3] each, lattice units (radians per step).  The mask itself is the caller's: re-voxelise and pass it
 * with lbmhd_set_obstacle / lbmhd_set_porosity (device pointers keep that asynchronous) as the body turns. */
int lbmhd_set_obstacle_rotation(lbmhd_t *h, const double omega[3], const double centre[3]);

/* Body integrals ("per-timestep surface integrals of net magnetic flux, forces, torques,
 * electromagnetic work"; the paper prints no formulas: DESIGN.md reading A21 takes them from what the blend of
 * Eq.13-14 hands over).  While enabled every lbmhd_step adds, over the cells with d < 1,
 *   out[0..2]   F = - sum dQh_m         momentum the fluid gives the body per step (aerodynamic + Maxwell)
 *   out[3..5]   T = - sum r x dQh_m     its moment about the sphere centre (analytic sphere) or `ref` (masked bodies)
 *   out[6]      W = - sum dQh_E         energy given to the body (0 for INCRES)
 *   out[7..9]       sum dQh_B           magnetic field injected into the fluid
 *   out[10..12]     sum (1-d) B         volume integral of the fluid's B over the body (flux x length)
 *   out[13]         sum (1-d)           body volume in cells
 * in lattice units (INCRES: the velocity sets stand for momentum).  lbmhd_body_enable zeroes the accumulator (so does
 * lbmhd_init); `ref` HOST [3] or NULL (0,0,0), global cell coordinates.  lbmhd_body_read copies the 14 fp64 sums to
 * HOST (synchronises) or DEVICE (stays asynchronous on the stream) memory, then zeroes them if `reset`: one read per
 * step gives the per-step series.  The order of the additions across thread blocks is not fixed (atomics). */
int lbmhd_body_enable(lbmhd_t *h, int enable, const double ref[3]);
int lbmhd_body_read(lbmhd_t *h, double *out, int reset, int on_device);

/* Raw population access (checkpoint / tests): fp64 [K][Q][N] at this boundary in both precisions, in
 * canonical (k, i, cell) order whatever the streaming layout.  HOST or DEVICE pointer per on_device. */
int lbmhd_get_populations(lbmhd_t *h, double *g_out, int on_device);
int lbmhd_set_populations(lbmhd_t *h, const double *g_in, int on_device);

/* Counters: time steps done since init; kernels launched by this handle since create. */
long long lbmhd_steps_done(const lbmhd_t *h);
long long lbmhd_launch_count(const lbmhd_t *h);

/* Which step kernel the last lbmhd_step launch used: LBMHD_PATH_ONE one cell per thread, LBMHD_PATH_MULTI
 * several cells per thread on interior tiles, LBMHD_PATH_CLUSTER variable rows split over a 2-CTA cluster, LBMHD_PATH_TMA
 * the TMA-staged persistent kernel, LBMHD_PATH_PERSIST many steps in one cooperative launch; -1 before the first step or for
 * a NULL handle.  The choice is made per lattice, scheme, precision, grid size and step count; every path computes the same
 * update.  Environment variables read by lbmhd_create (test and measurement knobs, never needed for correct use):
 * LBMHD_PAIR=0 one cell per thread everywhere; LBMHD_MULTI=1 the multi-cell kernel on small grids too; LBMHD_CLUSTER=0 no
 * cluster split; LBMHD_PATH=tma the TMA-staged kernel (fp64 / fp32, A/B only); LBMHD_PERSIST=0 one launch per step
 * everywhere, =2 the cooperative many-step launch whatever the grid size; LBMHD_PERSIST_WAVES=n its size threshold (tiles <=
 * n x co-resident blocks); LBMHD_EDGE_MULTI=0 / 1 the x-face cells outside / inside the multi-cell tiles
 * (where that kernel variant is compiled); LBMHD_CELL=1 the cell-per-thread kernel on the short lattices
 * (off by default: measured slower), =2 that kernel on small grids too; LBMHD_PDL=0 plain launches instead of
 * programmatic dependent launches of the one-cell and multi-cell step kernels; LBMHD_RESIDENT=0 no
 * register-resident many-step kernel on 1D lattices. */
enum { LBMHD_PATH_ONE = 0, LBMHD_PATH_MULTI = 1, LBMHD_PATH_CLUSTER = 2, LBMHD_PATH_TMA = 3, LBMHD_PATH_PERSIST = 4,
       LBMHD_PATH_CELL = 5 /* one thread per cell, all K sets in its registers: the short lattices D1Q3 / D2Q5 / D3Q7 */,
       LBMHD_PATH_RESIDENT = 6 /* 1D lattices of <= 1024 cells, n >= 2 steps in one launch: populations resident in registers, one cluster */ };
int lbmhd_step_path(const lbmhd_t *h);

/* Measured-bandwidth probe (BabelStream-style copy b[i] = a[i] over n fp64 elements, the paper's roofline
 * denominator is such a measurement).  a, b DEVICE pointers; enqueues `reps` launches. */
int lbmhd_copy_probe(const double *a, double *b, size_t n, int reps, void *stream);

/* Its companion: BabelStream-style triad a[i] = b[i] + s * c[i] over n fp64 elements (two reads and one write per
 * element: 24 n bytes per launch), the second probe SURVEY.md:546-549 asks for beside the copy.  DEVICE pointers. */
int lbmhd_triad_probe(double *a, const double *b, const double *c, double s, size_t n, int reps, void *stream);

/* The same diagnostics with NO device allocation, NO handle and NO workspace, for callers that cannot allocate: code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc (csrc/lbmhd_noalloc.cu).  The per-block partials
 * of the two-stage reduction live in one file-scope device array of 1184 x 82 doubles = 776 704 bytes that every GPU which
 * loads the library holds until the process exits; the call itself allocates nothing.
 *   scheme, lattice, nx, ny, nz, bc[6] (HOST), gamma   as in lbmhd_params (bc: periodic faces wrap div_h B, the others clamp;
 *                                                       LBMHD_BC_HALO faces are ghost planes and are not counted)
 *   fields    DEVICE fp64 [K][N]  (input, e.g. written by lbmhd_moments(on_device))
 *   diag_out  DEVICE fp64 [3K+4]  (output, the slots of lbmhd_moments)
 *   device, stream   CUDA device ordinal and cudaStream_t; the two kernels are enqueued on `stream`, nothing synchronises.
 * Limit: nx * ny * nz <= LBMHD_STATIC_DIAG_MAX_CELLS, else LBMHD_ENOMEM with a message (use lbmhd_diagnostics).
 * Set-up: the first call on a device looks the array's device address up (cudaGetSymbolAddress); calling with fields == NULL
 * and diag_out == NULL does only that — do it once per device before capturing a graph.
 * Sharing: all calls on a device use the one array.  A call writes every slot it reads, so nothing carries over from the
 * previous call; calls that OVERLAP on the GPU (two streams, two unordered host threads) race on it — serialise them.
 * The result is bit-identical to lbmhd_diagnostics / lbmhd_moments on the same fields (same kernels, same block count). */
#define LBMHD_STATIC_DIAG_MAX_CELLS (1ull << 30)
int lbmhd_diagnostics_static(int scheme, int lattice, int nx, int ny, int nz, const int bc[6], double gamma,
                             const double *fields, double *diag_out, int device, void *stream);

/* Text of the last error on this thread ("" if none). */
const char *lbmhd_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LBMHD_H */
