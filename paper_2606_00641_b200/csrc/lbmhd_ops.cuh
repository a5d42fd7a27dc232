// lbmhd_ops.cuh — kernel dispatch: Ops<LAT, SCHEME, real> launches the kernels of lbmhd_kernels.cuh / lbmhd_tma.cuh for one
// (lattice, scheme, precision); table_for collects the entry points of a scheme group.  Included by lbmhd_inst.cu only.
#pragma once
#include <math.h>
#include <string.h>

#include "lbmhd_host.h"
#include "lbmhd_kernels.cuh"
#include "lbmhd_tma.cuh"
#include "lbmhd_resident.cuh"

namespace lbh {

using namespace lbk;

template <int LAT, int SCHEME, typename real> struct Ops {
  using L = Lattice<LAT>;
  static constexpr int Q = L::Q, K = Vars<SCHEME, L::D>::K;
  static constexpr int TXAUX = K > 16 ? 32 : 64;   // x-tile of init / moments (TXAUX * K threads <= 1024)
  // Launch bound (min blocks/SM) of the step kernels: the largest count whose register cap still holds the lean
  // interior path of this lattice (measured: D3Q19 72-80 registers, D2Q9 58, D3Q7 54, D2Q5 50, D1Q3 44), so that small
  // blocks (INCRES: 32 x 5 threads) do not leave the SM at 20 warps.  DESIGN.md §5.1.
  static constexpr int minb_for(int threads, int need) {
    int best = 1;
    for (int m = 1; m <= 16; m++)
      if (m * threads <= 2048 && (65536 / (m * threads)) / 8 * 8 >= need) best = m;
    return best;
  }
  static constexpr int REGS_NEED = Q > 9 ? 72 : (Q > 7 ? 64 : (Q > 3 ? 56 : 48));
  static constexpr int MINB = minb_for(32 * K, REGS_NEED);

  static real *pops(lbmhd_t *h, int which) { return (real *)(h->ws + h->L.off_pop[which]); }

  static dim3 grid(const lbmhd_t *h, int tx) { return dim3((h->p.nx + tx - 1) / tx, h->p.ny, h->p.nz); }

  // One launch over all tiles; the tile class (interior / x-edge / general) is chosen per block.
  // One cell per thread: A/B, or in place the pull-push step from layout P0 and the local step from P1.
  // grid over the planes [lo, hi) of the slowest lattice axis (the whole lattice: 0 .. n)
  static dim3 grid_planes(const lbmhd_t *h, int gx, int lo, int hi) {
    return L::D == 3 ? dim3(gx, h->p.ny, hi - lo) : (L::D == 2 ? dim3(gx, hi - lo, 1) : dim3(gx, 1, 1));
  }
  // A step kernel launched so that it may be scheduled while the previous kernel of the stream drains (programmatic dependent
  // launch; the kernel's pdl_enter() is the matching wait).  What precedes it in the stream need not be a step kernel: a
  // predecessor that never releases its dependents does so when it ends, which is the plain stream order.
  template <typename... P, typename... A> static cudaError_t launch_pdl(lbmhd_t *h, void (*kern)(P...), dim3 g, dim3 b, A... args) {
    if (!h->pdl) {
      kern<<<g, b, 0, h->stream>>>(args...);
      return cudaGetLastError();
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = g;
    cfg.blockDim = b;
    cfg.dynamicSmemBytes = 0;
    cfg.stream = h->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, args...);
  }
  static cudaError_t launch_step_one(lbmhd_t *h, const StepArgs<real> &a, int lo, int hi) {
    constexpr int TX = 32;
    const dim3 g = grid_planes(h, (h->p.nx + TX - 1) / TX, lo, hi), b(TX, K);
    const Region all{0, 1, 0, 1, 0, 1};
    cudaError_t e;
    if (h->p.streaming != LBMHD_STREAM_INPLACE) e = launch_pdl(h, step_kernel<LAT, SCHEME, real, TX, MINB, 0, ST_AB>, g, b, a, all, 0);
    else if (h->parity == 0) e = launch_pdl(h, step_kernel<LAT, SCHEME, real, TX, MINB, 0, ST_PP>, g, b, a, all, 0);
    else e = launch_pdl(h, step_kernel<LAT, SCHEME, real, TX, MINB, 0, ST_LOC>, g, b, a, all, 0);
    h->launches += 1;
    return e;
  }

  // several cells per thread on interior tiles (lbmhd_kernels.cuh, step_kernel_multi): NC-wide vector accesses need nx % NC == 0
  // NC = cells per thread: the widest of {NCMAX, NCMAX/2, .., 2} whose register need (NC*Q population registers + 36..52)
  // still lets two blocks share an SM, so that one block's loads overlap the other's arithmetic; a block that is alone on
  // its SM anyway (K = 17 rows) loses nothing.  Measured on B200: fp64 NC = 2 lifts config 5 from 0.955
  // to 0.975 of the copy bandwidth, D2Q5 0.76 -> 0.98; fp32 NC = 4 on D3Q19 / D2Q9 does not pay (scalar x-shifted loads).
  static constexpr int NCMAX = sizeof(real) == 8 ? 2 : (Q <= 7 ? 4 : 2);
#ifndef LBMHD_MULTI_REGS_EXTRA32
#define LBMHD_MULTI_REGS_EXTRA32 0      // measurement knob: more registers for the fp32 multi-cell kernels (fewer blocks per SM)
#endif
  static constexpr int regs_need_multi(int nc) {
    const int pops = nc * Q * (int)sizeof(real) / 4 + (sizeof(real) == 4 ? LBMHD_MULTI_REGS_EXTRA32 : 0);
    return (pops + (pops > 64 ? 52 : 36) + 7) / 8 * 8;        // D3Q19 fp64 x 2 cells: 76 + 52 = 128 (measured: no spills at 128, slower at 96)
  }
  static constexpr int pick_nc() {
    for (int nc = NCMAX; nc >= 2; nc /= 2)
      if (minb_for(32 * K, regs_need_multi(nc)) >= 2 || (MINB == 1 && regs_need_multi(nc) <= (65536 / (32 * K)) / 8 * 8)) return nc;
    return 1;
  }
  static constexpr int NC = pick_nc();
  static constexpr int VW = NC * (int)sizeof(real) >= 16 ? 16 / (int)sizeof(real) : NC;       // nx must be a multiple (vector alignment of rows)
  static constexpr int MINB_M = minb_for(32 * K, regs_need_multi(NC));
  // small grids keep one cell per thread: fewer, larger blocks lose to wave quantisation (config 2: 0.87 vs 0.81)
  static bool multi_pays(const lbmhd_t *h) {
    const long long blocks = (long long)((h->p.nx + 32 * NC - 1) / (32 * NC) + 1) * h->p.ny * h->p.nz;
    return h->multi_force || blocks >= 16LL * h->num_sms * MINB_M;
  }
  // Rows made of whole multi-cell tiles, the end tiles holding the face cells (step_kernel_multi<.., EDGE = true>), whenever nx is
  // a multiple of the tile width: measured faster in 20 of 22 cases (fp32 on config 5 in place 0.785 -> 0.877,
  // D3Q7 fp32 0.63 -> 0.75; the one loss: RESIST on config 4 in place 0.944 -> 0.920).  LBMHD_EDGE_MULTI=0 turns it off.
  static constexpr bool EDGE_COMPILED = NC > 1;
  static constexpr bool EDGE_DEFAULT = true;
  template <bool EDGE> static cudaError_t launch_multi_t(lbmhd_t *h, const StepArgs<real> &a, int lo, int hi) {
    constexpr int W = 32 * NC;
    const int xbase = EDGE ? 0 : 32;
    const int nm = EDGE ? h->p.nx / W : (h->p.nx >= 64 + W ? (h->p.nx - 64) / W : 0);      // multi-cell tiles at x0 = xbase + W j
    const int ntail = EDGE ? 0 : (h->p.nx - (32 + W * nm) + 31) / 32;                       // 32-cell tiles after them (>= 0)
    const dim3 g = grid_planes(h, EDGE ? nm : nm + 1 + (ntail > 0 ? ntail : 0), lo, hi), b(32, K);
    const bool inplace = h->p.streaming == LBMHD_STREAM_INPLACE;
    cudaError_t e;
    if (!inplace) e = launch_pdl(h, step_kernel_multi<LAT, SCHEME, real, NC, MINB_M, ST_AB, EDGE>, g, b, a, nm, xbase);
    else if (h->parity == 0) e = launch_pdl(h, step_kernel_multi<LAT, SCHEME, real, NC, MINB_M, ST_PP, EDGE>, g, b, a, nm, xbase);
    else e = launch_pdl(h, step_kernel_multi<LAT, SCHEME, real, NC, MINB_M, ST_LOC, EDGE>, g, b, a, nm, xbase);
    h->launches += 1;
    return e;
  }
  static cudaError_t launch_step_multi(lbmhd_t *h, const StepArgs<real> &a, int lo, int hi) {
    if constexpr (NC > 1) {
      if constexpr (EDGE_COMPILED) {
        const bool want = h->edge_multi < 0 ? EDGE_DEFAULT : h->edge_multi != 0;
        if (want && h->p.nx % (32 * NC) == 0 && h->p.nx >= 2 * 32 * NC) return launch_multi_t<true>(h, a, lo, hi);
      }
      return launch_multi_t<false>(h, a, lo, hi);
    } else {
      return cudaErrorInvalidValue;
    }
  }

  // one thread per cell on the short lattices (lbmhd_kernels.cuh, step_kernel_cell): K * Q populations in one thread's registers
  static constexpr bool CELL_OK = Q <= 7 && K <= 9;
  static constexpr int cell_wx() {      // tile width: 32 x the smallest divisor >= 2 of K (a 1D lattice: the whole block in one row)
    int g = 2;
    while (g < K && K % g != 0) g++;
    return L::D == 1 ? 32 * K : 32 * g;
  }
  static constexpr int WXC = cell_wx();
  static constexpr int RYC = 32 * K / WXC;
  static constexpr int regs_need_cell() { return (K * Q * (int)sizeof(real) / 4 + 48 + 7) / 8 * 8; }
  static constexpr int MINB_C = minb_for(32 * K, regs_need_cell());
  static bool cell_pays(const lbmhd_t *h) {
    if (h->p.nx < 64 + WXC) return false;
    const long long blocks = (long long)((h->p.nx - 64) / WXC + 2) * ((h->p.ny + RYC - 1) / RYC) * h->p.nz;
    return h->cell_force || blocks >= 8LL * h->num_sms * MINB_C;
  }
  static cudaError_t launch_step_cell(lbmhd_t *h, const StepArgs<real> &a, int lo, int hi) {
    if constexpr (CELL_OK) {
      const int nc = (h->p.nx - 64) / WXC;                                 // cell tiles at x0 = 32 + WXC j, all interior in x
      const int ntail = (h->p.nx - (32 + WXC * nc) + 31) / 32;             // 32-cell pieces after them
      const int gx = nc + 1 + ntail;
      const dim3 g = L::D == 3 ? dim3(gx, (h->p.ny + RYC - 1) / RYC, hi - lo) : (L::D == 2 ? dim3(gx, (hi - lo + RYC - 1) / RYC, 1) : dim3(gx, 1, 1));
      const dim3 b(32, K);
      const bool inplace = h->p.streaming == LBMHD_STREAM_INPLACE;
      if (!inplace) step_kernel_cell<LAT, SCHEME, real, WXC, MINB_C, ST_AB><<<g, b, 0, h->stream>>>(a, nc);
      else if (h->parity == 0) step_kernel_cell<LAT, SCHEME, real, WXC, MINB_C, ST_PP><<<g, b, 0, h->stream>>>(a, nc);
      else step_kernel_cell<LAT, SCHEME, real, WXC, MINB_C, ST_LOC><<<g, b, 0, h->stream>>>(a, nc);
      h->launches += 1;
      return cudaGetLastError();
    } else {
      return cudaErrorInvalidValue;
    }
  }

  // The rows of a tile split over a 2-CTA cluster (lbmhd_kernels.cuh, Share / ShareAsync): compiled for the schemes with gradient
  // sets on D3Q19 in fp64 (measured slower on D3Q7 and in fp32); the default is where it was measured to pay, LBMHD_CLUSTER=0 / 1 overrides.
  static constexpr bool CLUSTER_COMPILED = has_G(SCHEME) && Q > 9 && sizeof(real) == 8;
  static constexpr bool CLUSTER_DEFAULT = SCHEME == kResist && Q > 9 && sizeof(real) == 8;
  static constexpr int KH = (K + 1) / 2;
  static constexpr int MINB_CL = minb_for(32 * KH, REGS_NEED);
  static cudaError_t launch_step_cluster(lbmhd_t *h, const StepArgs<real> &a, int lo, int hi) {
    const dim3 g = grid_planes(h, 2 * ((h->p.nx + 31) / 32), lo, hi), b(32, KH);
    if (h->p.streaming != LBMHD_STREAM_INPLACE) step_kernel_cl<LAT, SCHEME, real, MINB_CL, ST_AB><<<g, b, 0, h->stream>>>(a);
    else if (h->parity == 0) step_kernel_cl<LAT, SCHEME, real, MINB_CL, ST_PP><<<g, b, 0, h->stream>>>(a);
    else step_kernel_cl<LAT, SCHEME, real, MINB_CL, ST_LOC><<<g, b, 0, h->stream>>>(a);
    h->launches += 1;
    return cudaGetLastError();
  }

  static cudaError_t launch_step_tma(lbmhd_t *h, const StepArgs<real> &a) {
    using C = TmaCfg<LAT, SCHEME, real, kTmaTX, kTmaStages>;
    auto kern = step_kernel_tma<LAT, SCHEME, real, kTmaTX, kTmaStages>;
    if (!h->tma_attr_set) {      // the attribute is per device: tracked per handle (a handle is bound to one device)
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
      if (e != cudaSuccess) return e;
      h->tma_attr_set = true;
    }
    const int tiles_x = (h->p.nx + kTmaTX - 1) / kTmaTX;
    const long long n_rows = (long long)h->p.ny * h->p.nz;                 // < 2^31 - SMs checked at create
    const int grid = (int)(n_rows < (long long)h->num_sms ? n_rows : (long long)h->num_sms);
    kern<<<grid, C::THREADS, C::SMEM_BYTES, h->stream>>>(a, h->tmap[h->cur][0], h->tmap[h->cur][1], tiles_x, (int)n_rows);
    h->launches += 1;
    return cudaGetLastError();
  }

  // the step-independent part of the kernel arguments
  static void make_args(const lbmhd_t *h, StepArgs<real> &a) {
    memset(&a, 0, sizeof a);
    a.pstride = h->L.pstride;
    a.nx = h->p.nx; a.ny = h->p.ny; a.nz = h->p.nz;
    for (int j = 0; j < 6; j++) a.bc[j] = h->p.bc[j];
    for (int k = 0; k < K; k++) { a.omega[k] = (real)(1.0 / h->tau[k]); a.tau[k] = (real)h->tau[k]; }
    a.inv_tauB_cs2 = (real)(1.0 / (h->tau[h->g.iB] * h->g.cs2));
    a.kappa = (real)h->p.powell; a.gamma = (real)h->p.gamma; a.c0sq = (real)h->p.c0sq;
    a.inv_tau_relax = h->p.tau_relax > 0.0 ? (real)(1.0 / h->p.tau_relax) : real(0);
    a.etaj_inv_jc2 = h->p.eta_jc > 0.0 ? (real)(1.0 / (h->p.eta_jc * h->p.eta_jc)) : real(0);
    a.eta = has_G(SCHEME) ? (real)h->p.eta : real(0);
    a.mu = SCHEME == kFull ? (real)h->p.nu : real(0);
    a.tauB0 = (real)h->tau[h->g.iB];
    a.mask = h->have_mask ? (const unsigned char *)(h->ws + h->L.off_mask) : nullptr;
    a.Bsolid = h->have_bsolid ? (const double *)(h->ws + h->L.off_bsolid) : nullptr;
    a.dfield = h->have_dfield ? (const double *)(h->ws + h->L.off_dfield) : nullptr;
    for (int c = 0; c < 3; c++) { a.usolid[c] = h->usolid[c]; a.obs_om[c] = h->obs_om[c]; a.obs_c[c] = h->obs_c[c]; }
    {
      const long long es = (long long)sizeof(real);
      for (int i = 0; i < Q; i++) {
        const long long shift = lat_c<L>(i, 0) + (long long)lat_c<L>(i, 1) * h->p.nx + (long long)lat_c<L>(i, 2) * h->p.nx * h->p.ny;
        a.ld_off[i] = ((long long)i * (long long)h->L.pstride - shift) * es;
        a.st_off[i] = (long long)i * (long long)h->L.pstride * es;
      }
    }
    a.kplane = (long long)Q * (long long)h->L.pstride * (long long)sizeof(real);
    a.hoff = h->p.halo_offset;
    a.body = h->body_on ? (double *)(h->ws + h->L.off_body) : nullptr;
    for (int c = 0; c < 3; c++) a.body_ref[c] = h->body_ref[c];
    a.has_sphere = h->has_sphere ? 1 : 0;
    if (h->has_sphere) {
      a.sph_R = h->sph_R;
      a.sph_R2 = h->sph_R * h->sph_R;
      a.sph_eps = h->sph_eps;
      a.sph_touch2 = h->sph_eps > 0.0 ? (h->sph_R + 0.5 * h->sph_eps) * (h->sph_R + 0.5 * h->sph_eps) : a.sph_R2;
      a.n_dip = h->n_dip;
      for (int j = 0; j < h->n_dip; j++) { a.dip_Bs[j] = h->dip_Bs[j]; a.dip_core[j] = h->dip_core[j]; }
      for (int c = 0; c < 3; c++) { a.sph_u[c] = h->sph_u[c]; a.sph_om[c] = h->sph_om[c]; }
    }
  }

  // the part that changes every step: population copies, published moment arrays, the body's position
  static void step_args(const lbmhd_t *h, StepArgs<real> &a) {
    const bool inplace = h->p.streaming == LBMHD_STREAM_INPLACE;
    a.src = pops(const_cast<lbmhd_t *>(h), h->cur);
    a.dst = pops(const_cast<lbmhd_t *>(h), inplace ? h->cur : 1 - h->cur);
    if (inplace) {
      a.M_cur = (const double *)(h->ws + h->L.off_M[h->mcur]);
      a.M_next = (double *)(h->ws + h->L.off_M[1 - h->mcur]);
    }
    if (h->has_sphere) {
      // A12: centre before step t is c0 + (t - t0) u^B; product and sum rounded separately, like the oracle
      const volatile double dt = (double)(h->t - h->sph_t0);
      for (int c = 0; c < 3; c++) {
        const volatile double prod = dt * h->sph_u[c];
        a.sph_c[c] = h->sph_c0[c] + prod;
      }
      // body-frame offsets and axes of the dipoles at this step: Rodrigues rotation about Omega by |Omega| (t - t0)
      const double om2 = h->sph_om[0] * h->sph_om[0] + h->sph_om[1] * h->sph_om[1] + h->sph_om[2] * h->sph_om[2];
      for (int j = 0; j < h->n_dip; j++)
        for (int which = 0; which < 2; which++) {
          const double *v = which ? h->dip_off[j] : h->dip_m[j];
          double *out = which ? a.dip_off[j] : a.dip_m[j];
          for (int c = 0; c < 3; c++) out[c] = v[c];
          if (om2 > 0.0) {
            const double omn = sqrt(om2), th = omn * dt, cth = cos(th), sth = sin(th);
            const double e[3] = {h->sph_om[0] / omn, h->sph_om[1] / omn, h->sph_om[2] / omn};
            const double ev = e[0] * v[0] + e[1] * v[1] + e[2] * v[2];
            const double ex[3] = {e[1] * v[2] - e[2] * v[1], e[2] * v[0] - e[0] * v[2], e[0] * v[1] - e[1] * v[0]};
            for (int c = 0; c < 3; c++) out[c] = v[c] * cth + ex[c] * sth + e[c] * ev * (1.0 - cth);
          }
        }
    }
  }

  // one launch of the step kernel chosen for this lattice, scheme, precision and grid over the planes
  // [lo, hi) of the slowest lattice axis
  static int launch(lbmhd_t *h, StepArgs<real> &a, int lo, int hi) {
    a.row0 = lo;
    a.row1 = hi;
    cudaError_t e;
    bool launched = false;
    if constexpr (CLUSTER_COMPILED) {
      const bool want = h->cluster < 0 ? CLUSTER_DEFAULT : h->cluster != 0;
      if (want && h->p.eta_jc == 0.0) { e = launch_step_cluster(h, a, lo, hi); launched = true; h->last_path = LBMHD_PATH_CLUSTER; }
    }
    if (launched) {}
    else if (h->use_tma) { e = launch_step_tma(h, a); h->last_path = LBMHD_PATH_TMA; }
    else if (CELL_OK && h->cell && h->pair && cell_pays(h)) { e = launch_step_cell(h, a, lo, hi); h->last_path = LBMHD_PATH_CELL; }
    else if (NC > 1 && h->pair && h->p.nx % VW == 0 && multi_pays(h)) { e = launch_step_multi(h, a, lo, hi); h->last_path = LBMHD_PATH_MULTI; }
    else { e = launch_step_one(h, a, lo, hi); h->last_path = LBMHD_PATH_ONE; }
    if (e != cudaSuccess) return fail(LBMHD_ECUDA, "step kernel launch: %s", cudaGetErrorString(e));
    return LBMHD_OK;
  }

  static void advance(lbmhd_t *h) {
    if (h->p.streaming == LBMHD_STREAM_INPLACE) { h->parity ^= 1; h->mcur ^= 1; }
    else h->cur = 1 - h->cur;
    h->t += 1;
  }

  static int n_planes(const lbmhd_t *h) { return L::D == 3 ? h->p.nz : (L::D == 2 ? h->p.ny : 1); }

  // ---- many steps in one cooperative launch (lbmhd_kernels.cuh, step_kernel_persist) --------------
  static constexpr int MINB_P = minb_for(32 * K, REGS_NEED + 8);
  template <bool INPLACE> static int persist_capacity(const lbmhd_t *h) {
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, step_kernel_persist<LAT, SCHEME, real, MINB_P, INPLACE>, 32 * K, 0) != cudaSuccess)
      return 0;
    return per_sm * h->num_sms;
  }
  // Taken when the caller asks for several steps at once on a lattice small enough that launch latency and the fill and drain
  // of every launch show (measured: DESIGN.md §5.7), never for slabs (their ghost planes change between steps) or a body
  // whose dipoles rotate (the host turns them every step).
  static bool persist_allowed(const lbmhd_t *h, int n_steps) {
    if (!h->persist || n_steps < 2 || h->use_tma) return false;
    const int D1 = L::D - 1;
    if (L::D >= 2 && (h->p.bc[2 * D1] == LBMHD_BC_HALO || h->p.bc[2 * D1 + 1] == LBMHD_BC_HALO)) return false;
    if (h->has_sphere && (h->sph_om[0] != 0.0 || h->sph_om[1] != 0.0 || h->sph_om[2] != 0.0)) return false;
    return true;
  }
  template <bool INPLACE> static void persist_args(lbmhd_t *h, PersistArgs<real> &p, int n_steps) {
    memset(&p, 0, sizeof p);
    p.n_steps = n_steps;
    p.inplace = INPLACE ? 1 : 0;
    p.parity0 = h->parity;
    p.pop[0] = pops(h, h->cur);
    p.pop[1] = pops(h, INPLACE ? h->cur : 1 - h->cur);
    if (INPLACE) {
      p.M[0] = (double *)(h->ws + h->L.off_M[h->mcur]);
      p.M[1] = (double *)(h->ws + h->L.off_M[1 - h->mcur]);
    }
    p.t_rel0 = h->t - h->sph_t0;
    for (int c = 0; c < 3; c++) p.sph_c0[c] = h->sph_c0[c];
    p.tiles_x = (h->p.nx + 31) / 32;
    p.n_tiles = (long long)p.tiles_x * h->p.ny * h->p.nz;
  }
  template <bool INPLACE> static int launch_persist(lbmhd_t *h, StepArgs<real> &a, int n_steps, int capacity) {
    PersistArgs<real> p;
    persist_args<INPLACE>(h, p, n_steps);
    a.row0 = 0;
    a.row1 = n_planes(h);
    const long long want = p.n_tiles < (long long)capacity ? p.n_tiles : (long long)capacity;
    void *params[2] = {(void *)&a, (void *)&p};
    cudaError_t e = cudaLaunchCooperativeKernel((const void *)step_kernel_persist<LAT, SCHEME, real, MINB_P, INPLACE>,
                                                dim3((unsigned)want), dim3(32, K), params, 0, h->stream);
    if (e != cudaSuccess) return fail(LBMHD_ECUDA, "cooperative step kernel launch: %s", cudaGetErrorString(e));
    h->launches += 1;
    h->last_path = LBMHD_PATH_PERSIST;
    for (int s = 0; s < n_steps; s++) advance(h);
    return LBMHD_OK;
  }
  // ---- many steps of a 1D lattice with the populations resident in registers (lbmhd_resident.cuh) --------------
  // One cluster of <= 16 CTAs of TXR cells (TXR = 32 or 64: nx <= 1024), fluid cells only, no body; in place from either layout
  // for any number of steps.  A zero-gradient face and its inward neighbour share a CTA.
  template <int TXR> static bool resident_fits(const lbmhd_t *h) {
    const int nx = h->p.nx, ncta = (nx + TXR - 1) / TXR;
    if (TXR * K > 1024 || ncta > 16) return false;
    const bool periodic = h->p.bc[0] == LBMHD_BC_PERIODIC;
    return periodic || (nx - 1) % TXR != 0;
  }
  static bool resident_allowed(const lbmhd_t *h) {
    if constexpr (L::D != 1) return false;
    if (!h->resident || h->use_tma) return false;
    if (h->have_mask || h->have_dfield || h->body_on || h->has_sphere || h->p.nx < 3) return false;
    if ((h->p.bc[0] == LBMHD_BC_PERIODIC) != (h->p.bc[1] == LBMHD_BC_PERIODIC)) return false;
    if (h->p.bc[0] == LBMHD_BC_HALO || h->p.bc[1] == LBMHD_BC_HALO) return false;
    return resident_fits<32>(h) || resident_fits<64>(h);
  }
  // returns LBMHD_OK and *done = true if the steps were run; *done = false (nothing launched) when no cluster of that size can be
  // co-scheduled on this device
  template <int TXR, bool INPLACE> static int launch_resident_t(lbmhd_t *h, StepArgs<real> &a, int n_steps, bool *done) {
    *done = false;
    if constexpr (L::D == 1) {
      auto kern = step_kernel_resident<LAT, SCHEME, real, TXR, INPLACE>;
      ResidentArgs<real> p;
      memset(&p, 0, sizeof p);
      p.n_steps = n_steps;
      p.ncta = (h->p.nx + TXR - 1) / TXR;
      p.pop_in = pops(h, h->cur);
      p.pop_out = pops(h, INPLACE ? h->cur : (h->cur + n_steps) & 1);
      if (INPLACE) {
        p.layout_in = h->parity;
        p.layout_out = (h->parity + n_steps) & 1;
        p.M_in = (const double *)(h->ws + h->L.off_M[h->mcur]);
        p.M_out[0] = (double *)(h->ws + h->L.off_M[0]);
        p.M_out[1] = (double *)(h->ws + h->L.off_M[1]);
      }
      if (p.ncta > 8 && cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
        cudaGetLastError();
        return LBMHD_OK;
      }
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)p.ncta);
      cfg.blockDim = dim3(TXR, K);
      cfg.stream = h->stream;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = (unsigned)p.ncta;
      at[0].val.clusterDim.y = 1;
      at[0].val.clusterDim.z = 1;
      cfg.attrs = at;
      cfg.numAttrs = 1;
      int nclusters = 0;
      if (cudaOccupancyMaxActiveClusters(&nclusters, kern, &cfg) != cudaSuccess || nclusters < 1) {
        cudaGetLastError();
        return LBMHD_OK;
      }
      a.row0 = 0;
      a.row1 = 1;
      cudaError_t e = cudaLaunchKernelEx(&cfg, kern, a, p);
      if (e != cudaSuccess) return fail(LBMHD_ECUDA, "resident step kernel launch: %s", cudaGetErrorString(e));
      h->launches += 1;
      h->last_path = LBMHD_PATH_RESIDENT;
      for (int s = 0; s < n_steps; s++) advance(h);
      *done = true;
    }
    return LBMHD_OK;
  }
  static int launch_resident(lbmhd_t *h, StepArgs<real> &a, int n_steps, bool *done) {
    const bool inplace = h->p.streaming == LBMHD_STREAM_INPLACE;
    if (resident_fits<32>(h)) return inplace ? launch_resident_t<32, true>(h, a, n_steps, done) : launch_resident_t<32, false>(h, a, n_steps, done);
    return inplace ? launch_resident_t<64, true>(h, a, n_steps, done) : launch_resident_t<64, false>(h, a, n_steps, done);
  }
  static int step(lbmhd_t *h, int n_steps) {
    StepArgs<real> a;
    make_args(h, a);
    const bool inplace = h->p.streaming == LBMHD_STREAM_INPLACE;
    if (n_steps >= 2 && resident_allowed(h)) {
      step_args(h, a);
      bool done = false;
      if (int rc = launch_resident(h, a, n_steps, &done)) return rc;
      if (done) return LBMHD_OK;
    }
    if (persist_allowed(h, n_steps)) {
      const long long n_tiles = (long long)((h->p.nx + 31) / 32) * h->p.ny * h->p.nz;
      const int cap = inplace ? persist_capacity<true>(h) : persist_capacity<false>(h);
      if (cap > 0 && (h->persist_force || n_tiles <= (long long)h->persist_waves * cap)) {
        step_args(h, a);
        return inplace ? launch_persist<true>(h, a, n_steps, cap) : launch_persist<false>(h, a, n_steps, cap);
      }
    }
    for (int s = 0; s < n_steps; s++) {
      step_args(h, a);
      if (int rc = launch(h, a, 0, n_planes(h))) return rc;
      advance(h);
    }
    return LBMHD_OK;
  }

  // one step in pieces (slab overlap): the planes [lo, hi) of the slowest lattice axis; `last` completes the step
  static int step_part(lbmhd_t *h, int lo, int hi, int last) {
    StepArgs<real> a;
    make_args(h, a);
    step_args(h, a);
    if (hi > lo)
      if (int rc = launch(h, a, lo, hi)) return rc;
    if (last) advance(h);
    return LBMHD_OK;
  }

  static int init(lbmhd_t *h, const double *fields_dev) {
    init_kernel<LAT, SCHEME, real, TXAUX><<<grid(h, TXAUX), dim3(TXAUX, K), 0, h->stream>>>(
        fields_dev, pops(h, 0), h->L.pstride, h->p.nx, h->p.ny, h->p.nz, (real)h->p.gamma, (real)h->p.c0sq,
        has_G(SCHEME) ? (real)h->p.eta : real(0), SCHEME == kFull ? (real)h->p.nu : real(0), h->p.tau_relax > 0.0 ? (real)(1.0 / h->p.tau_relax) : real(0));
    CUDA_TRY(cudaGetLastError());
    h->launches += 1;
    h->parity = 0;
    return refresh_published(h);
  }

  static int moments(lbmhd_t *h, double *fields_dev) {
    if (h->p.streaming == LBMHD_STREAM_INPLACE && h->parity == 1)
      moments_p1_kernel<LAT, SCHEME, real, TXAUX><<<grid(h, TXAUX), dim3(TXAUX, K), 0, h->stream>>>(
          pops(h, h->cur), h->L.pstride, fields_dev, h->p.nx, h->p.ny, h->p.nz, h->p.bc[0], h->p.bc[2], h->p.bc[4]);
    else
      moments_kernel<LAT, SCHEME, real, TXAUX><<<grid(h, TXAUX), dim3(TXAUX, K), 0, h->stream>>>(
          pops(h, h->cur), h->L.pstride, fields_dev, h->p.nx, h->p.ny, h->p.nz);
    CUDA_TRY(cudaGetLastError());
    h->launches += 1;
    return LBMHD_OK;
  }

  // in place: (re)publish the moments of every cell in both M arrays — after init, set_populations, set_obstacle
  static int refresh_published(lbmhd_t *h) {
    if (h->p.streaming != LBMHD_STREAM_INPLACE) return LBMHD_OK;
    double *m0 = (double *)(h->ws + h->L.off_M[0]), *m1 = (double *)(h->ws + h->L.off_M[1]);
    if (int rc = moments(h, m0)) return rc;
    CUDA_TRY(cudaMemcpyAsync(m1, m0, (size_t)K * h->N * 8, cudaMemcpyDeviceToDevice, h->stream));
    h->mcur = 0;
    return LBMHD_OK;
  }

  static int diag(lbmhd_t *h, const double *fields_dev, double *diag_dev) {
    size_t want = (h->N + kDiagThreads - 1) / kDiagThreads;
    const int nb = (int)(want < (size_t)kMaxDiagBlocks ? want : (size_t)kMaxDiagBlocks);
    double *partial = (double *)(h->ws + h->L.off_partial);
    diag_partial_kernel<LAT, SCHEME><<<nb, kDiagThreads, 0, h->stream>>>(fields_dev, partial, h->p.nx, h->p.ny, h->p.nz,
                                                                          h->p.bc[0], h->p.bc[2], h->p.bc[4], h->p.gamma,
                                                                          h->g.D >= 2 && h->p.bc[2 * (h->g.D - 1)] == LBMHD_BC_HALO,
                                                                          h->g.D >= 2 && h->p.bc[2 * (h->g.D - 1) + 1] == LBMHD_BC_HALO);
    CUDA_TRY(cudaGetLastError());
    diag_final_kernel<<<1, kDiagThreads, 0, h->stream>>>(partial, nb, K, diag_dev);
    CUDA_TRY(cudaGetLastError());
    h->launches += 2;
    return LBMHD_OK;
  }

  // directions whose component along the slowest lattice axis equals `sign` (all directions if sign == 0)
  static int halo_dirs(int sign, int *dirs) {
    int n = 0;
    for (int i = 0; i < Q; i++)
      if (sign == 0 || lat_c<L>(i, L::D - 1) == sign)      // entry: dir | (c_x + 1) << 8 | (c_y + 1) << 10 (in-plane components)
        dirs[n++] = i | ((lat_c<L>(i, 0) + 1) << 8) | (((L::D == 3 ? lat_c<L>(i, 1) : 0) + 1) << 10);
    return n;
  }

  static int pops_export(lbmhd_t *h, double *out_dev) {
    if (h->p.streaming == LBMHD_STREAM_INPLACE && h->parity == 1)
      pops_export_p1_kernel<LAT, real><<<1184, 256, 0, h->stream>>>(pops(h, h->cur), h->L.pstride, out_dev, h->p.nx, h->p.ny, h->p.nz,
                                                                    K * Q, h->p.bc[0], h->p.bc[2], h->p.bc[4]);
    else
      pops_export_kernel<real><<<1184, 256, 0, h->stream>>>(pops(h, h->cur), h->L.pstride, out_dev, h->N, K * Q);
    CUDA_TRY(cudaGetLastError());
    h->launches += 1;
    return LBMHD_OK;
  }
  static int pops_import(lbmhd_t *h, const double *in_dev) {
    pops_import_kernel<real><<<1184, 256, 0, h->stream>>>(in_dev, pops(h, h->cur), h->L.pstride, h->N, K * Q);
    CUDA_TRY(cudaGetLastError());
    h->launches += 1;
    h->parity = 0;                      // canonical order is layout P0
    return refresh_published(h);
  }
};

template <int LAT, int SCHEME, typename real> OpTable make_table() {
  using O = Ops<LAT, SCHEME, real>;
  return OpTable{O::step, O::step_part, O::init, O::moments, O::diag, O::pops_export, O::pops_import, O::refresh_published, O::halo_dirs};
}

// GROUP 0: the schemes without gradient tensors (IDEAL, INCRES, IDEAL_DIVB); GROUP 1: RESIST, FULL.  One translation unit per
// (lattice, precision, group): 20 units of similar weight compile in parallel (build.py).
template <int LAT, typename real, int GROUP> OpTable table_for(int scheme) {
  if constexpr (GROUP == 0) {
    if (scheme == LBMHD_IDEAL) return make_table<LAT, kIdeal, real>();
    if (scheme == LBMHD_IDEAL_DIVB) return make_table<LAT, kIdealD, real>();
    return make_table<LAT, kIncres, real>();
  } else {
    if (scheme == LBMHD_RESIST) return make_table<LAT, kResist, real>();
    return make_table<LAT, kFull, real>();
  }
}

}  // namespace lbh
