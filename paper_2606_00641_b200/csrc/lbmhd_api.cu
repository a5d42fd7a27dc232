// lbmhd_api.cu — host side of the C ABI declared in include/lbmhd.h: validation, workspace layout, the step-independent
// entry points, dispatch on (lattice, scheme, precision) through lbh::OpTable.  No torch types, no device allocation:
// the caller owns the workspace.  There is no CPU fallback anywhere in this file.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <string>

#include "lbmhd_host.h"
#include "lbmhd_kernels.cuh"      // halo_plane_kernel, copy_probe_kernel, triad_probe_kernel

using namespace lbk;
using namespace lbh;

namespace {
thread_local std::string g_err;
}

int lbh::fail(int code, const char *fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}

namespace {

bool geometry(int scheme, int lattice, Geometry *g) {
  if (scheme != LBMHD_IDEAL && scheme != LBMHD_INCRES && scheme != LBMHD_IDEAL_DIVB && scheme != LBMHD_RESIST && scheme != LBMHD_FULL) return false;
  g->cs2 = 1.0 / 3.0;
  switch (lattice) {
    case LBMHD_D1Q3: g->D = 1; g->Q = 3; break;
    case LBMHD_D2Q9: g->D = 2; g->Q = 9; break;
    case LBMHD_D3Q19: g->D = 3; g->Q = 19; break;
    case LBMHD_D2Q5: g->D = 2; g->Q = 5; break;
    case LBMHD_D3Q7: g->D = 3; g->Q = 7; g->cs2 = 0.25; break;
    default: return false;
  }
  const bool ideal = scheme != LBMHD_INCRES;
  g->K = scheme == LBMHD_IDEAL ? 8 : (scheme == LBMHD_IDEAL_DIVB ? 9 : (scheme == LBMHD_RESIST ? 8 + 3 * g->D : (scheme == LBMHD_FULL ? 8 + 6 * g->D : 1 + 2 * g->D)));
  g->NV = ideal ? 3 : g->D;
  g->iU = 1;
  g->iB = ideal ? 5 : 1 + g->D;
  return true;
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
bool layout(const lbmhd_params *p, const Geometry &g, Layout *L) {
  if (p->nx < 1 || p->ny < 1 || p->nz < 1) return false;
  if (p->precision != 64 && p->precision != 32) return false;
  const size_t N = (size_t)p->nx * p->ny * p->nz;
  const size_t es = p->precision == 64 ? 8 : 4;
  L->pstride = align_up(N, 32);
  L->pop_bytes = align_up((size_t)g.K * g.Q * L->pstride * es, 256);
  size_t off = 0;
  L->off_pop[0] = off; off += L->pop_bytes;
  L->off_pop[1] = off; off += p->streaming == LBMHD_STREAM_AB ? L->pop_bytes : 0;
  L->off_fields = off; off += align_up((size_t)g.K * N * 8, 256);
  // in place: two ping-pong arrays of published post-collision moments (Q^nb of face cells, state of frozen cells)
  L->off_M[0] = off; off += p->streaming == LBMHD_STREAM_INPLACE ? align_up((size_t)g.K * N * 8, 256) : 0;
  L->off_M[1] = off; off += p->streaming == LBMHD_STREAM_INPLACE ? align_up((size_t)g.K * N * 8, 256) : 0;
  L->off_mask = off; off += align_up(N, 256);
  L->off_partial = off; off += align_up((size_t)kMaxDiagBlocks * (3 * g.K + 4) * 8, 256);
  L->off_diag = off; off += 256;
  L->off_dirs = off; off += 1024;      // direction lists of the halo pack kernels (8 x 32 ints)
  L->off_body = off; off += 256;       // body integrals accumulator (14 doubles)
  L->total_min = off;                  // everything a run without a per-cell solid field / porosity needs
  L->off_bsolid = off; off += align_up(3 * N * 8, 256);     // optional tail: lbmhd_set_obstacle(B_solid), lbmhd_set_porosity
  L->off_dfield = off; off += align_up(N * 8, 256);
  L->total = off;
  return true;
}

}  // namespace

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 5D view of one population copy: x, y, z, direction i, variable k; box = [K][1][1][1][kTmaTX]
int make_tensor_maps(lbmhd *h) {
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn)
    return fail(LBMHD_ECUDA, "cuTensorMapEncodeTiled is not available from the driver");
  const size_t es = h->p.precision == 64 ? 8 : 4;
  const cuuint64_t dims[5] = {(cuuint64_t)h->p.nx, (cuuint64_t)h->p.ny, (cuuint64_t)h->p.nz, (cuuint64_t)h->g.Q, (cuuint64_t)h->g.K};
  const cuuint64_t strides[4] = {(cuuint64_t)h->p.nx * es, (cuuint64_t)h->p.nx * h->p.ny * es, (cuuint64_t)h->L.pstride * es,
                                 (cuuint64_t)h->L.pstride * h->g.Q * es};
  const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  for (int b = 0; b < 4; b++) {
    const cuuint32_t box[5] = {(cuuint32_t)(kTmaTX + (b & 1) * (16 / es)), 1, 1, 1, (cuuint32_t)h->g.K};
    CUresult r = ((EncodeTiledFn)fn)(&h->tmap[b >> 1][b & 1], es == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5,
                                     h->ws + h->L.off_pop[b >> 1], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(LBMHD_ECUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
  }
  return LBMHD_OK;
}

}  // namespace

extern "C" {

const char *lbmhd_last_error(void) { return g_err.c_str(); }

int lbmhd_num_vars(const lbmhd_params *p) {
  Geometry g;
  if (!p || !geometry(p->scheme, p->lattice, &g)) return LBMHD_EINVAL;
  return g.K;
}
int lbmhd_num_dirs(const lbmhd_params *p) {
  Geometry g;
  if (!p || !geometry(p->scheme, p->lattice, &g)) return LBMHD_EINVAL;
  return g.Q;
}

size_t lbmhd_workspace_bytes(const lbmhd_params *p) {
  Geometry g;
  Layout L;
  if (!p || !geometry(p->scheme, p->lattice, &g) || !layout(p, g, &L)) return 0;
  return L.total;
}
size_t lbmhd_workspace_bytes_min(const lbmhd_params *p) {
  Geometry g;
  Layout L;
  if (!p || !geometry(p->scheme, p->lattice, &g) || !layout(p, g, &L)) return 0;
  return L.total_min;
}

void lbmhd_destroy(lbmhd_t *h) { delete h; }

long long lbmhd_steps_done(const lbmhd_t *h) { return h ? h->t : -1; }
long long lbmhd_launch_count(const lbmhd_t *h) { return h ? h->launches : -1; }
int lbmhd_step_path(const lbmhd_t *h) { return h ? h->last_path : -1; }

int lbmhd_create(const lbmhd_params *p, const unsigned char *cell_mask, lbmhd_t **out) {
  if (!out) return fail(LBMHD_EINVAL, "out is NULL");
  *out = nullptr;
  if (!p) return fail(LBMHD_EINVAL, "params is NULL");
  Geometry g;
  if (!geometry(p->scheme, p->lattice, &g)) return fail(LBMHD_EINVAL, "unknown scheme %d or lattice %d", p->scheme, p->lattice);
  Layout L;
  if (!layout(p, g, &L)) return fail(LBMHD_EINVAL, "bad dims %d x %d x %d or precision %d", p->nx, p->ny, p->nz, p->precision);
  if (p->streaming != LBMHD_STREAM_AB && p->streaming != LBMHD_STREAM_INPLACE)
    return fail(LBMHD_EINVAL, "unknown streaming mode %d", p->streaming);
  if (g.D < 2 && p->ny != 1) return fail(LBMHD_EINVAL, "ny must be 1 on a 1D lattice");
  if (g.D < 3 && p->nz != 1) return fail(LBMHD_EINVAL, "nz must be 1 on a 1D/2D lattice");
  if ((size_t)p->ny > 65535 || (size_t)p->nz > 65535) return fail(LBMHD_EINVAL, "ny, nz must be <= 65535");
  if ((unsigned long long)g.Q * L.pstride >= (1ull << 32))
    return fail(LBMHD_EINVAL, "grid too large: Q * cells must stay below 2^32 (32-bit plane offsets in the kernels)");
  const int nn[3] = {p->nx, p->ny, p->nz};
  for (int a = 0; a < g.D; a++) {
    const int lo = p->bc[2 * a], hi = p->bc[2 * a + 1];
    const int top = (a == g.D - 1 && g.D >= 2) ? LBMHD_BC_HALO : LBMHD_BC_INFLOW;
    if (lo < 0 || lo > top || hi < 0 || hi > top)
      return fail(LBMHD_EINVAL, "bad boundary kind on axis %d (HALO: slowest lattice axis, D >= 2)", a);
    if ((lo == LBMHD_BC_HALO || hi == LBMHD_BC_HALO) && nn[a] < 4) return fail(LBMHD_EINVAL, "a slab needs >= 4 planes (ghosts included)");
    if ((lo == LBMHD_BC_PERIODIC) != (hi == LBMHD_BC_PERIODIC)) return fail(LBMHD_EINVAL, "periodic must be paired on axis %d", a);
    if (lo != LBMHD_BC_PERIODIC && nn[a] < 3) return fail(LBMHD_EINVAL, "non-periodic axis %d needs >= 3 cells", a);
  }
  lbmhd_t *h = new lbmhd_t();
  h->p = *p; h->g = g; h->L = L;
  h->N = (size_t)p->nx * p->ny * p->nz;
  for (int k = 0; k < g.K; k++) h->tau[k] = p->tau[k];
  const double cs2 = g.cs2;
  if (p->nu > 0.0 && p->scheme != LBMHD_FULL) {    // Eq.5; FULL carries nu (the shear viscosity) in the flux
    for (int b = 0; b < g.NV; b++) h->tau[g.iU + b] = 0.5 + p->nu / cs2;
    if (p->scheme == LBMHD_INCRES) h->tau[0] = 0.5 + p->nu / cs2;
  }
  if (p->eta > 0.0 && p->scheme != LBMHD_RESIST && p->scheme != LBMHD_FULL)      // RESIST, FULL carry eta in the flux; tau_B stays the stabilisation parameter
    for (int b = 0; b < g.NV; b++) h->tau[g.iB + b] = 0.5 + p->eta / cs2;
  for (int k = 0; k < g.K; k++)
    if (!(h->tau[k] > 0.5)) { delete h; return fail(LBMHD_EINVAL, "tau[%d] = %g must be > 1/2", k, p->tau[k]); }
  for (int b = 1; b < g.NV; b++)
    if (h->tau[g.iB + b] != h->tau[g.iB]) { delete h; return fail(LBMHD_EINVAL, "all magnetic sets must share one tau (A7)"); }
  if (p->scheme != LBMHD_INCRES && !(p->gamma > 1.0)) { delete h; return fail(LBMHD_EINVAL, "gamma must be > 1"); }
  if ((p->scheme == LBMHD_IDEAL_DIVB || p->scheme == LBMHD_RESIST || p->scheme == LBMHD_FULL) && !(p->tau_relax > 0.0)) { delete h; return fail(LBMHD_EINVAL, "tau_relax must be > 0"); }
  if ((p->scheme == LBMHD_RESIST || p->scheme == LBMHD_FULL) && !(p->eta >= 0.0)) { delete h; return fail(LBMHD_EINVAL, "eta must be >= 0"); }
  if (p->scheme == LBMHD_FULL && !(p->nu >= 0.0)) { delete h; return fail(LBMHD_EINVAL, "nu must be >= 0"); }
  if (p->eta_jc != 0.0 && !(p->scheme == LBMHD_INCRES && p->eta_jc > 0.0)) { delete h; return fail(LBMHD_EINVAL, "eta_jc needs the INCRES scheme and must be > 0"); }
  if (!p->workspace) { delete h; return fail(LBMHD_EINVAL, "workspace is NULL"); }
  if (((uintptr_t)p->workspace & 255) != 0) { delete h; return fail(LBMHD_ENOMEM, "workspace must be 256-byte aligned"); }
  if (p->workspace_bytes < L.total_min) {
    delete h;
    return fail(LBMHD_ENOMEM, "workspace has %zu bytes, need %zu (%zu with per-cell solid fields)", p->workspace_bytes, L.total_min, L.total);
  }
  h->have_solid_store = p->workspace_bytes >= L.total;
  h->ws = (char *)p->workspace;
  h->stream = (cudaStream_t)p->stream;
  cudaError_t e = cudaSetDevice(p->device);
  if (e != cudaSuccess) { delete h; return fail(LBMHD_ECUDA, "cudaSetDevice(%d): %s", p->device, cudaGetErrorString(e)); }
  {
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p->device);
    if (e != cudaSuccess) { delete h; return fail(LBMHD_ECUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e)); }
    h->num_sms = sms;
    h->pair = p->eta_jc == 0.0;      // several cells per thread where the lattice has a multi-cell kernel; eta(j): one-cell kernels
    if (const char *e3 = getenv("LBMHD_PAIR")) h->pair = h->pair && atoi(e3) != 0;
    h->cluster = -1;
    if (const char *e4 = getenv("LBMHD_CLUSTER")) h->cluster = atoi(e4) != 0 ? 1 : 0;
    h->last_path = -1;
    h->edge_multi = -1;
    if (const char *e10 = getenv("LBMHD_EDGE_MULTI")) h->edge_multi = atoi(e10) != 0 ? 1 : 0;
    h->resident = true;
    if (const char *e12 = getenv("LBMHD_RESIDENT")) h->resident = atoi(e12) != 0;
    h->pdl = true;
    if (const char *e11 = getenv("LBMHD_PDL")) h->pdl = atoi(e11) != 0;
    h->cell = false;      // measured slower than the multi-cell kernel on B200 in all but one case: opt-in
    h->cell_force = false;
    if (const char *e8 = getenv("LBMHD_CELL")) { h->cell = atoi(e8) != 0; h->cell_force = atoi(e8) == 2; }
    h->persist = true;
    h->persist_force = false;
    h->persist_waves = 2;
    if (const char *e6 = getenv("LBMHD_PERSIST")) { h->persist = atoi(e6) != 0; h->persist_force = atoi(e6) == 2; }
    if (const char *e7 = getenv("LBMHD_PERSIST_WAVES")) h->persist_waves = atoi(e7);
    h->multi_force = false;
    if (const char *e5 = getenv("LBMHD_MULTI")) h->multi_force = atoi(e5) != 0;
    const char *path = getenv("LBMHD_PATH");      // tuning knob: "plain" forces the register-pull kernel
    const size_t es = p->precision == 64 ? 8 : 4;
    const long long tiles = (long long)((p->nx + kTmaTX - 1) / kTmaTX) * p->ny * p->nz;
    const bool halo = g.D >= 2 && (p->bc[2 * (g.D - 1)] == LBMHD_BC_HALO || p->bc[2 * (g.D - 1) + 1] == LBMHD_BC_HALO);
    h->use_tma = !halo && p->scheme != LBMHD_RESIST && p->scheme != LBMHD_FULL && p->streaming == LBMHD_STREAM_AB && path && strcmp(path, "tma") == 0 && ((size_t)p->nx * es) % 16 == 0 && tiles < 2000000000LL;
    if (h->use_tma) {
      const int rc = make_tensor_maps(h);
      if (rc) { delete h; return rc; }
    }
  }
  h->have_mask = cell_mask != nullptr;
  if (cell_mask) {
    e = cudaMemcpyAsync(h->ws + L.off_mask, cell_mask, h->N, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) { delete h; return fail(LBMHD_ECUDA, "mask upload: %s", cudaGetErrorString(e)); }
  }
  *out = h;
  return LBMHD_OK;
}

}  // extern "C"

namespace {

OpTable pick(const lbmhd_t *h) {
  const bool f64 = h->p.precision == 64;
  const int sc = h->p.scheme;
  const bool grp = sc == LBMHD_RESIST || sc == LBMHD_FULL;      // scheme group of the translation units (lbmhd_inst.cu)
  switch (h->p.lattice) {
#define LBH_PICK(LATID) (grp ? (f64 ? ops_table_##LATID##_64_g1(sc) : ops_table_##LATID##_32_g1(sc)) : (f64 ? ops_table_##LATID##_64_g0(sc) : ops_table_##LATID##_32_g0(sc)))
    case LBMHD_D1Q3: return LBH_PICK(1);
    case LBMHD_D2Q9: return LBH_PICK(2);
    case LBMHD_D2Q5: return LBH_PICK(4);
    case LBMHD_D3Q7: return LBH_PICK(5);
    default: return LBH_PICK(3);
#undef LBH_PICK
  }
}

}  // namespace

extern "C" {

int lbmhd_init(lbmhd_t *h, const double *fields, int on_device) {
  if (!h || !fields) return fail(LBMHD_EINVAL, "NULL argument");
  if (int rc = use_device(h)) return rc;
  const double *src = fields;
  if (!on_device) {
    double *scratch = (double *)(h->ws + h->L.off_fields);
    CUDA_TRY(cudaMemcpyAsync(scratch, fields, (size_t)h->g.K * h->N * 8, cudaMemcpyHostToDevice, h->stream));
    src = scratch;
  }
  h->cur = 0; h->t = 0; h->sph_t0 = 0;
  CUDA_TRY(cudaMemsetAsync(h->ws + h->L.off_body, 0, kBodyInts * 8, h->stream));
  const int rc = pick(h).init(h, src);
  if (rc) return rc;
  if (!on_device) CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LBMHD_OK;
}

int lbmhd_step(lbmhd_t *h, int n_steps) {
  if (!h || n_steps < 0) return fail(LBMHD_EINVAL, "bad handle or n_steps");
  if (int rc = use_device(h)) return rc;
  return pick(h).step(h, n_steps);
}

int lbmhd_step_part(lbmhd_t *h, int plane_lo, int plane_hi, int last) {
  if (!h) return fail(LBMHD_EINVAL, "NULL handle");
  const int nH = h->g.D == 3 ? h->p.nz : (h->g.D == 2 ? h->p.ny : 1);
  if (plane_lo < 0 || plane_hi > nH || plane_lo > plane_hi) return fail(LBMHD_EINVAL, "bad plane range [%d, %d) of %d", plane_lo, plane_hi, nH);
  if (int rc = use_device(h)) return rc;
  return pick(h).step_part(h, plane_lo, plane_hi, last);
}

int lbmhd_diagnostics(lbmhd_t *h, const double *fields, double *diag_out, int on_device) {
  if (!h || !fields || !diag_out) return fail(LBMHD_EINVAL, "NULL argument");
  if (int rc = use_device(h)) return rc;
  const int nd = 3 * h->g.K + 4;
  double *ddev = on_device ? diag_out : (double *)(h->ws + h->L.off_diag);
  if (int rc = pick(h).diag(h, fields, ddev)) return rc;
  if (on_device) return LBMHD_OK;
  CUDA_TRY(cudaMemcpyAsync(diag_out, ddev, nd * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (diag_out[nd - 1] != 0.0) return fail(LBMHD_ENUMERIC, "non-finite value or rho <= 0 seen (flag %g)", diag_out[nd - 1]);
  return LBMHD_OK;
}

int lbmhd_moments(lbmhd_t *h, double *fields_out, double *diag_out, int on_device) {
  if (!h) return fail(LBMHD_EINVAL, "NULL handle");
  if (int rc = use_device(h)) return rc;
  const OpTable op = pick(h);
  const size_t fbytes = (size_t)h->g.K * h->N * 8;
  const int nd = 3 * h->g.K + 4;
  double *fdev = (on_device && fields_out) ? fields_out : (double *)(h->ws + h->L.off_fields);
  if (int rc = op.moments(h, fdev)) return rc;
  double *ddev = (double *)(h->ws + h->L.off_diag);
  if (diag_out) {
    if (on_device) ddev = diag_out;
    if (int rc = op.diag(h, fdev, ddev)) return rc;
  }
  if (on_device) return LBMHD_OK;
  if (fields_out) CUDA_TRY(cudaMemcpyAsync(fields_out, fdev, fbytes, cudaMemcpyDeviceToHost, h->stream));
  if (diag_out) CUDA_TRY(cudaMemcpyAsync(diag_out, ddev, nd * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (diag_out && diag_out[nd - 1] != 0.0)
    return fail(LBMHD_ENUMERIC, "non-finite value or rho <= 0 seen (flag %g)", diag_out[nd - 1]);
  return LBMHD_OK;
}

int lbmhd_set_obstacle(lbmhd_t *h, const unsigned char *mask, const double u_solid[3], const double *B_solid, int on_device) {
  if (!h || !mask) return fail(LBMHD_EINVAL, "NULL argument");
  if (int rc = use_device(h)) return rc;
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  CUDA_TRY(cudaMemcpyAsync(h->ws + h->L.off_mask, mask, h->N, kind, h->stream));
  if (B_solid && !h->have_solid_store) return fail(LBMHD_ENOMEM, "workspace was sized with lbmhd_workspace_bytes_min: no room for B_solid");
  h->have_mask = true;
  h->have_bsolid = B_solid != nullptr;
  if (B_solid) CUDA_TRY(cudaMemcpyAsync(h->ws + h->L.off_bsolid, B_solid, 3 * h->N * 8, kind, h->stream));
  for (int c = 0; c < 3; c++) h->usolid[c] = u_solid ? u_solid[c] : 0.0;
  if (int rc = pick(h).refresh_published(h)) return rc;      // in place: newly FROZEN cells keep their current moments
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LBMHD_OK;
}

int lbmhd_set_sphere(lbmhd_t *h, const double centre[3], double radius, const double u_solid[3],
                     const double dipole_dir[3], double B_surface) {
  if (!h) return fail(LBMHD_EINVAL, "NULL handle");
  if (!(radius > 0.0)) { h->has_sphere = false; return LBMHD_OK; }
  if (!centre || !u_solid || !dipole_dir) return fail(LBMHD_EINVAL, "NULL argument");
  h->has_sphere = true;
  for (int c = 0; c < 3; c++) { h->sph_c0[c] = centre[c]; h->sph_u[c] = u_solid[c]; }
  h->sph_R = radius; h->sph_t0 = h->t;
  h->n_dip = 1;                                  // A12: one centred dipole capped at R/2
  for (int c = 0; c < 3; c++) { h->dip_off[0][c] = 0.0; h->dip_m[0][c] = dipole_dir[c]; }
  h->dip_Bs[0] = B_surface; h->dip_core[0] = 0.5 * radius;
  return LBMHD_OK;
}

int lbmhd_set_porosity(lbmhd_t *h, const double *d_field, int on_device) {
  if (!h) return fail(LBMHD_EINVAL, "NULL handle");
  if (int rc = use_device(h)) return rc;
  if (!d_field) { h->have_dfield = false; return LBMHD_OK; }
  if (!h->have_solid_store) return fail(LBMHD_ENOMEM, "workspace was sized with lbmhd_workspace_bytes_min: no room for the porosity field");
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  CUDA_TRY(cudaMemcpyAsync(h->ws + h->L.off_dfield, d_field, h->N * 8, kind, h->stream));
  if (!h->have_mask) {       // the kernels route tiles to the general path on "a mask exists"
    CUDA_TRY(cudaMemsetAsync(h->ws + h->L.off_mask, 0, h->N, h->stream));
    h->have_mask = true;
  }
  h->have_dfield = true;
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LBMHD_OK;
}

int lbmhd_set_sphere_dipoles(lbmhd_t *h, int n, const double *offset, const double *dir, const double *B_surface, const double *core) {
  if (!h || !offset || !dir || !B_surface || !core) return fail(LBMHD_EINVAL, "NULL argument");
  if (!h->has_sphere) return fail(LBMHD_EINVAL, "lbmhd_set_sphere first");
  if (n < 1 || n > 4) return fail(LBMHD_EINVAL, "1 to 4 dipoles, got %d", n);
  for (int j = 0; j < n; j++)
    if (!(core[j] > 0.0)) return fail(LBMHD_EINVAL, "core radius of dipole %d must be > 0", j);
  for (int j = 0; j < n; j++) {
    for (int c = 0; c < 3; c++) { h->dip_off[j][c] = offset[3 * j + c]; h->dip_m[j][c] = dir[3 * j + c]; }
    h->dip_Bs[j] = B_surface[j]; h->dip_core[j] = core[j];
  }
  h->n_dip = n;
  return LBMHD_OK;
}

int lbmhd_set_obstacle_rotation(lbmhd_t *h, const double omega[3], const double centre[3]) {
  if (!h || !omega || !centre) return fail(LBMHD_EINVAL, "NULL argument");
  for (int c = 0; c < 3; c++) { h->obs_om[c] = omega[c]; h->obs_c[c] = centre[c]; }
  return LBMHD_OK;
}

int lbmhd_body_enable(lbmhd_t *h, int enable, const double ref[3]) {
  if (!h) return fail(LBMHD_EINVAL, "NULL handle");
  if (int rc = use_device(h)) return rc;
  h->body_on = enable != 0;
  for (int c = 0; c < 3; c++) h->body_ref[c] = ref ? ref[c] : 0.0;
  CUDA_TRY(cudaMemsetAsync(h->ws + h->L.off_body, 0, kBodyInts * 8, h->stream));
  return LBMHD_OK;
}

int lbmhd_body_read(lbmhd_t *h, double *out, int reset, int on_device) {
  if (!h) return fail(LBMHD_EINVAL, "NULL handle");
  if (!h->body_on) return fail(LBMHD_EINVAL, "body integrals are not enabled (lbmhd_body_enable)");
  if (int rc = use_device(h)) return rc;
  if (out) CUDA_TRY(cudaMemcpyAsync(out, h->ws + h->L.off_body, kBodyInts * 8, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                                    h->stream));
  if (reset) CUDA_TRY(cudaMemsetAsync(h->ws + h->L.off_body, 0, kBodyInts * 8, h->stream));
  if (out && !on_device) CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LBMHD_OK;
}

int lbmhd_set_sphere_rotation(lbmhd_t *h, const double omega[3]) {
  if (!h || !omega) return fail(LBMHD_EINVAL, "NULL argument");
  for (int c = 0; c < 3; c++) h->sph_om[c] = omega[c];
  return LBMHD_OK;
}

int lbmhd_set_sphere_width(lbmhd_t *h, double eps) {
  if (!h || !(eps >= 0.0)) return fail(LBMHD_EINVAL, "bad handle or width");
  h->sph_eps = eps;
  return LBMHD_OK;
}

// ---- slab halo exchange: side 0 = low face of the slowest lattice axis, 1 = high face -----------------
static int halo_dir_list(const lbmhd_t *h, int sign, int *dirs) {      // directions with c_H == sign (all if sign == 0)
  return pick(h).halo_dirs(sign, dirs);
}

size_t lbmhd_halo_bytes(const lbmhd_t *h, int what) {
  if (!h || h->g.D < 2) return 0;
  int dirs[32];
  const int nd = halo_dir_list(h, what == LBMHD_HALO_FULL ? 0 : 1, dirs);
  const size_t plane = h->g.D == 3 ? (size_t)h->p.nx * h->p.ny : (size_t)h->p.nx;
  return (size_t)h->g.K * nd * plane * (h->p.precision == 64 ? 8 : 4);
}

// LBMHD_HALO_CROSSING  pack: the owned plane next to the ghost, directions that leave through that face (the neighbour pulls
//                      them); unpack: the ghost plane itself, directions that enter through that face.
// LBMHD_HALO_FULL      the same planes, all Q directions.
// LBMHD_HALO_RETURN    in place, after a pull-push step: this slab's boundary cells pushed g'_j (c_j leaving through the face)
//                      into the ghost plane, at slot opp(j); those values belong in the NEIGHBOUR's owned plane next to its
//                      ghost, same slots.  pack: the ghost plane, directions that enter through that face (the slots written);
//                      unpack: the owned plane next to the ghost, directions that leave through that face.
static int halo_move(lbmhd_t *h, int side, int what, void *buf, bool pack, int next_copy, cudaStream_t stream) {
  if (!h || !buf || side < 0 || side > 1 || what < 0 || what > 2) return fail(LBMHD_EINVAL, "bad argument");
  if (h->g.D < 2) return fail(LBMHD_EINVAL, "halo exchange needs D >= 2");
  const bool inplace = h->p.streaming == LBMHD_STREAM_INPLACE;
  if (what == LBMHD_HALO_RETURN && !inplace) return fail(LBMHD_EINVAL, "LBMHD_HALO_RETURN is the in-place exchange");
  if (what == LBMHD_HALO_FULL && inplace) return fail(LBMHD_EINVAL, "LBMHD_HALO_FULL needs A/B streaming (in place: exchange fields, lbmhd_diagnostics)");
  if (int rc = use_device(h)) return rc;
  const int nH = h->g.D == 3 ? h->p.nz : h->p.ny;
  const size_t plane = h->g.D == 3 ? (size_t)h->p.nx * h->p.ny : (size_t)h->p.nx;
  const bool ret = what == LBMHD_HALO_RETURN;
  const bool from_owned = pack != ret;          // crossing / full: pack reads the owned plane, unpack writes the ghost; return: the reverse
  const int sign = what == LBMHD_HALO_FULL ? 0 : (from_owned ? (side == 0 ? -1 : 1) : (side == 0 ? 1 : -1));
  const int hidx = from_owned ? (side == 0 ? 1 : nH - 2) : (side == 0 ? 0 : nH - 1);
  int dirs[32];
  const int nd = halo_dir_list(h, sign, dirs);
  // one list slot per (kind, sign): the lists are constant, but each call uploads its own so that no call depends on another
  int *ddev = (int *)(h->ws + h->L.off_dirs) + 32 * (what == LBMHD_HALO_FULL ? 2 : (sign > 0 ? 1 : 0));
  if (!h->dirs_uploaded[what == LBMHD_HALO_FULL ? 2 : (sign > 0 ? 1 : 0)]) {
    CUDA_TRY(cudaMemcpyAsync(ddev, dirs, nd * sizeof(int), cudaMemcpyHostToDevice, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));      // once per handle and list: later calls may run on another stream
    h->dirs_uploaded[what == LBMHD_HALO_FULL ? 2 : (sign > 0 ? 1 : 0)] = true;
  }
  const size_t total = (size_t)h->g.K * nd * plane;
  const int blocks = (int)((total + 255) / 256 < 1184 ? (total + 255) / 256 : 1184);
  char *pops = h->ws + h->L.off_pop[inplace ? 0 : (next_copy ? 1 - h->cur : h->cur)];
  // LBMHD_HALO_RETURN, unpack: skip the slots nobody pushed (the pusher would lie outside a non-periodic in-plane face)
  const int fx = (ret && !pack && h->p.bc[0] != LBMHD_BC_PERIODIC) ? 1 : 0;
  const int fy = (ret && !pack && h->g.D == 3 && h->p.bc[2] != LBMHD_BC_PERIODIC) ? 1 : 0;
  const int pny = h->g.D == 3 ? h->p.ny : 1;
  if (h->p.precision == 64) {
    if (pack) halo_plane_kernel<double, true><<<blocks, 256, 0, stream>>>((double *)pops, h->L.pstride, (double *)buf, plane, (size_t)hidx * plane, h->g.K, h->g.Q, nd, ddev, h->p.nx, pny, fx, fy);
    else halo_plane_kernel<double, false><<<blocks, 256, 0, stream>>>((double *)pops, h->L.pstride, (double *)buf, plane, (size_t)hidx * plane, h->g.K, h->g.Q, nd, ddev, h->p.nx, pny, fx, fy);
  } else {
    if (pack) halo_plane_kernel<float, true><<<blocks, 256, 0, stream>>>((float *)pops, h->L.pstride, (float *)buf, plane, (size_t)hidx * plane, h->g.K, h->g.Q, nd, ddev, h->p.nx, pny, fx, fy);
    else halo_plane_kernel<float, false><<<blocks, 256, 0, stream>>>((float *)pops, h->L.pstride, (float *)buf, plane, (size_t)hidx * plane, h->g.K, h->g.Q, nd, ddev, h->p.nx, pny, fx, fy);
  }
  CUDA_TRY(cudaGetLastError());
  h->launches += 1;
  return LBMHD_OK;
}

int lbmhd_halo_pack(lbmhd_t *h, int side, int what, void *buf) { return halo_move(h, side, what, buf, true, 0, h ? h->stream : 0); }
int lbmhd_halo_unpack(lbmhd_t *h, int side, int what, const void *buf) { return halo_move(h, side, what, (void *)buf, false, 0, h ? h->stream : 0); }
int lbmhd_halo_pack_on(lbmhd_t *h, int side, int what, void *buf, int next_copy, void *stream) {
  return halo_move(h, side, what, buf, true, next_copy, (cudaStream_t)stream);
}
int lbmhd_halo_unpack_on(lbmhd_t *h, int side, int what, const void *buf, int next_copy, void *stream) {
  return halo_move(h, side, what, (void *)buf, false, next_copy, (cudaStream_t)stream);
}

static int pops_io(lbmhd_t *h, double *out, const double *in, int on_device) {
  if (!h || (!out && !in)) return fail(LBMHD_EINVAL, "NULL argument");
  if (int rc = use_device(h)) return rc;
  const OpTable op = pick(h);
  const size_t bytes = (size_t)h->g.K * h->g.Q * h->N * 8;
  if (on_device) return out ? op.pops_export(h, out) : op.pops_import(h, in);
  // host path: stage through the not-current population copy when it is large enough (fp64 A/B), plane by plane otherwise
  if (h->p.precision != 64 || h->p.streaming != LBMHD_STREAM_AB)
    return fail(LBMHD_EINVAL, "host population I/O needs precision 64 and A/B streaming (use device pointers otherwise)");
  double *stage = (double *)(h->ws + h->L.off_pop[1 - h->cur]);
  if (bytes > h->L.pop_bytes) return fail(LBMHD_ENOMEM, "staging buffer too small");
  if (out) {
    if (int rc = op.pops_export(h, stage)) return rc;
    CUDA_TRY(cudaMemcpyAsync(out, stage, bytes, cudaMemcpyDeviceToHost, h->stream));
  } else {
    CUDA_TRY(cudaMemcpyAsync(stage, in, bytes, cudaMemcpyHostToDevice, h->stream));
    if (int rc = op.pops_import(h, stage)) return rc;
  }
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LBMHD_OK;
}

int lbmhd_get_populations(lbmhd_t *h, double *g_out, int on_device) { return pops_io(h, g_out, nullptr, on_device); }
int lbmhd_set_populations(lbmhd_t *h, const double *g_in, int on_device) { return pops_io(h, nullptr, g_in, on_device); }

int lbmhd_copy_probe(const double *a, double *b, size_t n, int reps, void *stream) {
  if (!a || !b || reps < 0) return fail(LBMHD_EINVAL, "bad argument");
  for (int r = 0; r < reps; r++) {
    copy_probe_kernel<<<148 * 8, 256, 0, (cudaStream_t)stream>>>((const double2 *)a, (double2 *)b, n / 2);
    CUDA_TRY(cudaGetLastError());
  }
  return LBMHD_OK;
}

int lbmhd_triad_probe(double *a, const double *b, const double *c, double s, size_t n, int reps, void *stream) {
  if (!a || !b || !c || reps < 0) return fail(LBMHD_EINVAL, "bad argument");
  for (int r = 0; r < reps; r++) {
    triad_probe_kernel<<<148 * 8, 256, 0, (cudaStream_t)stream>>>((double2 *)a, (const double2 *)b, (const double2 *)c, s, n / 2);
    CUDA_TRY(cudaGetLastError());
  }
  return LBMHD_OK;
}

}  // extern "C"
