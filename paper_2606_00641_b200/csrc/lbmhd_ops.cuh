// lbmhd_ops.cuh — kernel dispatch: Ops<LAT, SCHEME, real> launches the kernels of lbmhd_kernels.cuh / lbmhd_tma.cuh for one
// (lattice, scheme, precision); table_for collects its entry points.  Included by lbmhd_inst.cu only.
#pragma once
#include <math.h>
#include <string.h>

#include "lbmhd_host.h"
#include "lbmhd_kernels.cuh"
#include "lbmhd_tma.cuh"

namespace lbh {

using namespace lbk;

template <int LAT, int SCHEME, typename real> struct Ops {
  using L = Lattice<LAT>;
  static constexpr int Q = L::Q, K = Vars<SCHEME, L::D>::K;
  static constexpr int TXAUX = K > 16 ? 32 : 64;   // x-tile of init / moments (TXAUX * K threads <= 1024)
  // launch bound of the step kernels of kResist (K = 11 / 14 / 17 variable rows per block): registers, not threads, limit it
  static constexpr int MINB_R = K >= 17 ? 1 : 2;

  static real *pops(lbmhd_t *h, int which) { return (real *)(h->ws + h->L.off_pop[which]); }

  static dim3 grid(const lbmhd_t *h, int tx) { return dim3((h->p.nx + tx - 1) / tx, h->p.ny, h->p.nz); }

  // One launch over all tiles (small grids, masked obstacles), or the split form: a lean interior launch plus
  // general launches over the x-edge columns, the y/z-edge rows and the sphere's bounding box.
  // in place: pull-push step from layout P0, local step from layout P1
  template <int MINB> static cudaError_t launch_step_inplace(lbmhd_t *h, const StepArgs<real> &a) {
    constexpr int TX = 32;
    const dim3 g((h->p.nx + TX - 1) / TX, h->p.ny, h->p.nz), b(TX, K);
    if (h->parity == 0) step_kernel<LAT, SCHEME, real, TX, MINB, 0, ST_PP><<<g, b, 0, h->stream>>>(a, Region{0, 1, 0, 1, 0, 1}, 0);
    else step_kernel<LAT, SCHEME, real, TX, MINB, 0, ST_LOC><<<g, b, 0, h->stream>>>(a, Region{0, 1, 0, 1, 0, 1}, 0);
    h->launches += 1;
    return cudaGetLastError();
  }

  // fp32: two cells per thread (64-cell tiles); needs an even nx for the 8-byte alignment of the float2 accesses
  template <int MINB> static cudaError_t launch_step_pair(lbmhd_t *h, const StepArgs<real> &a) {
    if constexpr (sizeof(real) == 4) {
      const int npair = h->p.nx >= 128 ? (h->p.nx - 64) / 64 : 0;      // pair tiles at x0 = 32 + 64 j, all interior in x
      const int ntail = (h->p.nx - (32 + 64 * npair) + 31) / 32;         // 32-cell tiles after the pair tiles (>= 0)
      const dim3 g(npair + 1 + (ntail > 0 ? ntail : 0), h->p.ny, h->p.nz), b(32, K);
      const bool inplace = h->p.streaming == LBMHD_STREAM_INPLACE;
      if (!inplace) step_kernel_pair<LAT, SCHEME, MINB, ST_AB><<<g, b, 0, h->stream>>>(a, npair);
      else if (h->parity == 0) step_kernel_pair<LAT, SCHEME, MINB, ST_PP><<<g, b, 0, h->stream>>>(a, npair);
      else step_kernel_pair<LAT, SCHEME, MINB, ST_LOC><<<g, b, 0, h->stream>>>(a, npair);
      h->launches += 1;
      return cudaGetLastError();
    } else {
      return cudaErrorInvalidValue;
    }
  }

  template <int TX, int MINB> static cudaError_t launch_step_whole(lbmhd_t *h, const StepArgs<real> &a) {
    step_kernel<LAT, SCHEME, real, TX, MINB, 0, ST_AB><<<dim3((h->p.nx + TX - 1) / TX, h->p.ny, h->p.nz), dim3(TX, K), 0, h->stream>>>(
        a, Region{0, 1, 0, 1, 0, 1}, 0);
    h->launches += 1;
    return cudaGetLastError();
  }

  template <int TX, int MINB> static cudaError_t launch_step(lbmhd_t *h, const StepArgs<real> &a) {
    constexpr int D = L::D;
    const int nx = h->p.nx, ny = h->p.ny, nz = h->p.nz;
    const int tiles_x = (nx + TX - 1) / TX;
    const dim3 block(TX, K);
    const bool split = h->split && !h->have_mask && tiles_x >= 3 && (D < 2 || ny >= 3) && (D < 3 || nz >= 3);
    if (!split) {
      step_kernel<LAT, SCHEME, real, TX, MINB, 0, ST_AB><<<dim3(tiles_x, ny, nz), block, 0, h->stream>>>(a, Region{0, 1, 0, 1, 0, 1}, 0);
      h->launches += 1;
      return cudaGetLastError();
    }
    const int iy0 = D > 1 ? 1 : 0, iny = D > 1 ? ny - 2 : 1;
    const int iz0 = D > 2 ? 1 : 0, inz = D > 2 ? nz - 2 : 1;
    // interior tiles (x-edge tiles excluded even when their cells are interior: they need wrap or face handling)
    step_kernel<LAT, SCHEME, real, TX, MINB, 1, ST_AB><<<dim3(tiles_x - 2, iny, inz), block, 0, h->stream>>>(a, Region{1, 1, iy0, 1, iz0, 1}, 0);
    // x-edge columns, all rows
    step_kernel<LAT, SCHEME, real, TX, 2, 2, ST_AB><<<dim3(2, ny, nz), block, 0, h->stream>>>(a, Region{0, tiles_x - 1, 0, 1, 0, 1}, 0);
    h->launches += 2;
    if (D > 1) {   // y-edge rows of the remaining columns
      step_kernel<LAT, SCHEME, real, TX, 2, 2, ST_AB><<<dim3(tiles_x - 2, 2, nz), block, 0, h->stream>>>(a, Region{1, 1, 0, ny - 1, 0, 1}, 0);
      h->launches += 1;
    }
    if (D > 2) {   // z-edge planes of what is left
      step_kernel<LAT, SCHEME, real, TX, 2, 2, ST_AB><<<dim3(tiles_x - 2, ny - 2, 2), block, 0, h->stream>>>(a, Region{1, 1, 1, 1, 0, nz - 1}, 0);
      h->launches += 1;
    }
    if (a.has_sphere) {   // interior-positioned tiles inside the sphere's bounding box
      const double R = a.sph_R + 0.5 * a.sph_eps + 1.0;
      int bx_lo = (int)floor((a.sph_c[0] - R) / TX), bx_hi = (int)floor((a.sph_c[0] + R) / TX);
      int y_lo = D > 1 ? (int)floor(a.sph_c[1] - R) : 0, y_hi = D > 1 ? (int)ceil(a.sph_c[1] + R) : 0;
      int z_lo = D > 2 ? (int)floor(a.sph_c[2] - R) : 0, z_hi = D > 2 ? (int)ceil(a.sph_c[2] + R) : 0;
      bx_lo = bx_lo < 1 ? 1 : bx_lo; bx_hi = bx_hi > tiles_x - 2 ? tiles_x - 2 : bx_hi;
      y_lo = y_lo < iy0 ? iy0 : y_lo; y_hi = y_hi > iy0 + iny - 1 ? iy0 + iny - 1 : y_hi;
      z_lo = z_lo < iz0 ? iz0 : z_lo; z_hi = z_hi > iz0 + inz - 1 ? iz0 + inz - 1 : z_hi;
      if (bx_lo <= bx_hi && y_lo <= y_hi && z_lo <= z_hi) {
        step_kernel<LAT, SCHEME, real, TX, 2, 2, ST_AB><<<dim3(bx_hi - bx_lo + 1, y_hi - y_lo + 1, z_hi - z_lo + 1), block, 0, h->stream>>>(
            a, Region{bx_lo, 1, y_lo, 1, z_lo, 1}, 1);
        h->launches += 1;
      }
    }
    return cudaGetLastError();
  }

  static cudaError_t launch_step_tma(lbmhd_t *h, const StepArgs<real> &a) {
    using C = TmaCfg<LAT, SCHEME, real, kTmaTX, kTmaStages>;
    auto kern = step_kernel_tma<LAT, SCHEME, real, kTmaTX, kTmaStages>;
    static bool attr_set = false;
    if (!attr_set) {
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
      if (e != cudaSuccess) return e;
      attr_set = true;
    }
    const int tiles_x = (h->p.nx + kTmaTX - 1) / kTmaTX;
    const long long n_rows = (long long)h->p.ny * h->p.nz;                 // < 2^31 - SMs checked at create
    const int grid = (int)(n_rows < (long long)h->num_sms ? n_rows : (long long)h->num_sms);
    kern<<<grid, C::THREADS, C::SMEM_BYTES, h->stream>>>(a, h->tmap[h->cur][0], h->tmap[h->cur][1], tiles_x, (int)n_rows);
    h->launches += 1;
    return cudaGetLastError();
  }

  static int step(lbmhd_t *h, int n_steps) {
    StepArgs<real> a;
    memset(&a, 0, sizeof a);
    a.pstride = h->L.pstride;
    a.nx = h->p.nx; a.ny = h->p.ny; a.nz = h->p.nz;
    for (int j = 0; j < 6; j++) a.bc[j] = h->p.bc[j];
    for (int k = 0; k < K; k++) a.omega[k] = (real)(1.0 / h->tau[k]);
    a.inv_tauB_cs2 = (real)(1.0 / (h->tau[h->g.iB] * h->g.cs2));
    a.kappa = (real)h->p.powell; a.gamma = (real)h->p.gamma; a.c0sq = (real)h->p.c0sq;
    a.inv_tau_relax = h->p.tau_relax > 0.0 ? (real)(1.0 / h->p.tau_relax) : real(0);
    a.etaj_inv_jc2 = h->p.eta_jc > 0.0 ? (real)(1.0 / (h->p.eta_jc * h->p.eta_jc)) : real(0);
    a.eta = SCHEME == kResist ? (real)h->p.eta : real(0);
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
      for (int c = 0; c < 3; c++) a.sph_u[c] = h->sph_u[c];
    }
    for (int s = 0; s < n_steps; s++) {
      const bool inplace = h->p.streaming == LBMHD_STREAM_INPLACE;
      a.src = pops(h, h->cur);
      a.dst = pops(h, inplace ? h->cur : 1 - h->cur);
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
          a.sph_om[c] = h->sph_om[c];
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
      cudaError_t e;
      if constexpr (SCHEME == kResist) {     // one launch configuration: one-cell kernels, one launch over all tiles
        e = inplace ? launch_step_inplace<MINB_R>(h, a) : launch_step_whole<32, MINB_R>(h, a);
      } else {
        if (sizeof(real) == 4 && h->pair) e = h->minb == 2 ? launch_step_pair<2>(h, a) : (h->minb == 4 ? launch_step_pair<4>(h, a) : launch_step_pair<3>(h, a));
        else if (inplace) e = h->minb == 4 ? launch_step_inplace<4>(h, a) : launch_step_inplace<3>(h, a);
        else if (h->use_tma) e = launch_step_tma(h, a);
        else switch (h->tx * 10 + h->minb) {
          case 322: e = launch_step_whole<32, 2>(h, a); break;
          case 323: e = launch_step<32, 3>(h, a); break;          // split launches exist for the two default bounds only
          case 324: e = launch_step<32, 4>(h, a); break;
          default: e = launch_step<32, 3>(h, a); break;
        }
      }
      if (e != cudaSuccess) return fail(LBMHD_ECUDA, "step kernel launch: %s", cudaGetErrorString(e));
      if (inplace) { h->parity ^= 1; h->mcur ^= 1; }
      else h->cur = 1 - h->cur;
      h->t += 1;
    }
    return LBMHD_OK;
  }

  static int init(lbmhd_t *h, const double *fields_dev) {
    init_kernel<LAT, SCHEME, real, TXAUX><<<grid(h, TXAUX), dim3(TXAUX, K), 0, h->stream>>>(
        fields_dev, pops(h, 0), h->L.pstride, h->p.nx, h->p.ny, h->p.nz, (real)h->p.gamma, (real)h->p.c0sq,
        SCHEME == kResist ? (real)h->p.eta : real(0), h->p.tau_relax > 0.0 ? (real)(1.0 / h->p.tau_relax) : real(0));
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
      if (sign == 0 || lat_c<L>(i, L::D - 1) == sign) dirs[n++] = i;
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
  return OpTable{O::step, O::init, O::moments, O::diag, O::pops_export, O::pops_import, O::refresh_published, O::halo_dirs};
}

template <int LAT, typename real> OpTable table_for(int scheme) {
  if (scheme == LBMHD_IDEAL) return make_table<LAT, kIdeal, real>();
  if (scheme == LBMHD_IDEAL_DIVB) return make_table<LAT, kIdealD, real>();
  if (scheme == LBMHD_RESIST) return make_table<LAT, kResist, real>();
  return make_table<LAT, kIncres, real>();
}

}  // namespace lbh
