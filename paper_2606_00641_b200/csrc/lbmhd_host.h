// lbmhd_host.h — what the host-side translation units of the library share: the handle behind lbmhd_t, the workspace
// layout, the per-(lattice, scheme, precision) operation table and the error helpers.  Private to csrc/.
// The kernel templates are instantiated in lbmhd_inst.cu, once per (lattice, precision) and in parallel; lbmhd_api.cu
// holds the C entry points and dispatches through OpTable.
#pragma once
#include "../../include/lbmhd.h"

#include <cuda.h>
#include <cuda_runtime.h>
#include <stddef.h>

namespace lbh {

int fail(int code, const char *fmt, ...);      // records the message lbmhd_last_error returns (thread-local), returns code

#define CUDA_TRY(expr)                                                                              \
  do {                                                                                              \
    cudaError_t e_ = (expr);                                                                        \
    if (e_ != cudaSuccess) return ::lbh::fail(LBMHD_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_));      \
  } while (0)
struct Geometry {
  int D, Q, K, NV, iU, iB;
  double cs2;
};

constexpr int kMaxDiagBlocks = 1184;   // 8 x 148 SMs
constexpr int kBodyInts = 14;          // lbmhd_body_read
constexpr int kTmaTX = 32, kTmaStages = 5;

struct Layout {
  size_t pstride;        // elements per population plane (N rounded up to 32)
  size_t pop_bytes;      // one population copy
  size_t off_pop[2], off_fields, off_M[2], off_mask, off_bsolid, off_dfield, off_partial, off_diag, off_dirs, off_body, total_min, total;
};

}  // namespace lbh

struct lbmhd {
  lbmhd_params p;
  lbh::Geometry g;
  lbh::Layout L;
  size_t N;
  double tau[32];
  cudaStream_t stream;
  char *ws;
  int cur;               // A/B: which population copy holds the current state (in place: always 0)
  int parity;            // in place: 0 = layout P0 (g_j(x) at (x, j)), 1 = layout P1 (after a pull-push step)
  int mcur;              // in place: which M array holds the moments published by the last step
  long long t;           // steps done since init
  long long launches;
  int last_path;         // LBMHD_PATH_* of the last step launch, -1 before the first
  bool have_mask, have_bsolid, have_dfield;
  bool have_solid_store; // the workspace holds the optional tail (B_solid, porosity field)
  bool dirs_uploaded[3]; // halo direction lists present on the device
  bool body_on;          // body integrals accumulate during the steps
  double body_ref[3];
  double usolid[3];
  bool has_sphere;
  double sph_c0[3], sph_R, sph_u[3], sph_eps, sph_om[3];
  int n_dip;             // dipole ensemble in the body frame (lbmhd_set_sphere: one centred dipole capped at R/2)
  double dip_off[4][3], dip_m[4][3], dip_Bs[4], dip_core[4];
  double obs_om[3], obs_c[3];   // rigid rotation of masked bodies
  long long sph_t0;
  bool multi_force;      // LBMHD_MULTI=1: take the multi-cell kernel on small grids too (tests)
  int cluster;           // variable rows of a tile split over a 2-CTA cluster: -1 = where measured to pay, 0 / 1 = LBMHD_CLUSTER
  bool pair;             // several cells per thread on interior tiles (fp32; fp64 on the short lattices); LBMHD_PAIR=0 turns it off
  int edge_multi;        // rows of whole multi-cell tiles with the face cells inside the end tiles: -1 = where measured to pay, 0 / 1 = LBMHD_EDGE_MULTI
  bool resident;         // 1D lattices: many steps with the populations resident in registers, one cluster (LBMHD_RESIDENT=0 turns it off)
  bool pdl;              // step kernels launched as programmatic dependents of the previous kernel in the stream (LBMHD_PDL=0 turns it off)
  bool cell;             // one thread per cell on the short lattices (off by default; LBMHD_CELL=1 turns it on)
  bool cell_force;       // LBMHD_CELL=2: on small grids too (tests)
  bool persist;          // many steps of a small lattice in one cooperative launch (LBMHD_PERSIST=0 turns it off)
  bool persist_force;    // LBMHD_PERSIST=2: take it whatever the lattice size (tests, measurements)
  int persist_waves;     // taken when tiles <= persist_waves x co-resident blocks (LBMHD_PERSIST_WAVES)
  bool use_tma;          // TMA-staged persistent step kernel (needs nx * sizeof(real) % 16 == 0)
  bool tma_attr_set;     // its dynamic shared memory attribute has been set on this handle's device
  int num_sms;
  CUtensorMap tmap[2][2];   // [copy][0: tile-wide box, 1: box 16 bytes wider] 5D views (x, y, z, i, k) of the populations
};

namespace lbh {

struct OpTable {
  int (*step)(lbmhd_t *, int);
  int (*step_part)(lbmhd_t *, int, int, int);
  int (*init)(lbmhd_t *, const double *);
  int (*moments)(lbmhd_t *, double *);
  int (*diag)(lbmhd_t *, const double *, double *);
  int (*pops_export)(lbmhd_t *, double *);
  int (*pops_import)(lbmhd_t *, const double *);
  int (*refresh_published)(lbmhd_t *);
  int (*halo_dirs)(int, int *);
};

// defined by lbmhd_inst.cu, one translation unit per (lattice, precision, scheme group: 0 = IDEAL / INCRES / IDEAL_DIVB, 1 = RESIST / FULL)
#define LBH_DECLARE_TABLES(P, G) \
  OpTable ops_table_1_##P##_g##G(int scheme); OpTable ops_table_2_##P##_g##G(int scheme); OpTable ops_table_3_##P##_g##G(int scheme); \
  OpTable ops_table_4_##P##_g##G(int scheme); OpTable ops_table_5_##P##_g##G(int scheme);
LBH_DECLARE_TABLES(64, 0)
LBH_DECLARE_TABLES(64, 1)
LBH_DECLARE_TABLES(32, 0)
LBH_DECLARE_TABLES(32, 1)
#undef LBH_DECLARE_TABLES

inline int use_device(const lbmhd_t *h) {
  CUDA_TRY(cudaSetDevice(h->p.device));
  return LBMHD_OK;
}

}  // namespace lbh
