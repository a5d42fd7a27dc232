// lbmhd_noalloc.cu — lbmhd_diagnostics_static: the conservation diagnostics (S9b, Eq.4 PAPER.md:90 summed over the lattice)
// for callers that cannot allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  It needs no lbmhd handle and no workspace.
//
// The two-stage reduction (diag_partial_kernel -> diag_final_kernel, lbmhd_kernels.cuh) needs scratch for the per-block
// partials.  Every other path keeps it in the caller's workspace; here it lives in ONE file-scope device array of a fixed size,
// kStaticScratchBytes = 1184 blocks x 82 slots x 8 bytes = 776 704 bytes, which every GPU that loads the library holds until
// the process exits.  In host code the array's NAME is a host-side stand-in, not a device address: the address the kernels get
// is taken once per device, with that device current, by cudaGetSymbolAddress below.
//
// Sharing: every call on a device uses the same array.  A call writes every slot it later reads (each of its nb blocks stores
// all 3K+4 of its partials before the fold reads nb x (3K+4) slots), so nothing has to be cleared between calls and stale
// contents of an earlier, larger call are never read.  Two calls that OVERLAP on the GPU (different streams, or different
// host threads without ordering) race on the array: callers serialise them.
#include <mutex>

#include "lbmhd_host.h"
#include "lbmhd_kernels.cuh"

using namespace lbk;
using namespace lbh;

namespace {

constexpr int kStaticMaxK = 26;                                       // FULL on a 3D lattice
constexpr int kStaticSlots = 3 * kStaticMaxK + 4;                     // 82
constexpr size_t kStaticScratchDoubles = (size_t)kMaxDiagBlocks * kStaticSlots;
constexpr size_t kStaticScratchBytes = kStaticScratchDoubles * sizeof(double);
static_assert(kStaticScratchBytes == 776704, "the size stated in include/lbmhd.h and README.md");
constexpr unsigned long long kStaticMaxCells = LBMHD_STATIC_DIAG_MAX_CELLS;      // stated limit of the entry point (config 5 has 2.5e7)
constexpr int kMaxDevices = 64;

static __device__ __align__(256) double g_diag_scratch[kStaticScratchDoubles];

std::mutex g_mu;
double *g_scratch_ptr[kMaxDevices];      // device address of g_diag_scratch on each device, nullptr until set up there

// once per device, with that device current: the device address of the scratch array
int scratch_for(int device, double **out) {
  if (device < 0 || device >= kMaxDevices) return fail(LBMHD_EINVAL, "device ordinal %d out of range", device);
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_ptr[device]) {
    double *ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_diag_scratch);
    if (e != cudaSuccess || !ptr) return fail(LBMHD_ECUDA, "cudaGetSymbolAddress(g_diag_scratch) on device %d: %s", device, cudaGetErrorString(e));
    g_scratch_ptr[device] = ptr;
  }
  *out = g_scratch_ptr[device];
  return LBMHD_OK;
}

template <int LAT, int SCHEME>
cudaError_t launch_diag(const double *fields, double *partial, int nb, int nx, int ny, int nz, const int bc[6], double gamma, double *diag_out,
                        cudaStream_t stream) {
  constexpr int D = Lattice<LAT>::D, K = Vars<SCHEME, D>::K;
  const int ghost_lo = D >= 2 && bc[2 * (D - 1)] == BC_HALO, ghost_hi = D >= 2 && bc[2 * (D - 1) + 1] == BC_HALO;
  diag_partial_kernel<LAT, SCHEME><<<nb, kDiagThreads, 0, stream>>>(fields, partial, nx, ny, nz, bc[0], bc[2], bc[4], gamma, ghost_lo, ghost_hi);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  diag_final_kernel<<<1, kDiagThreads, 0, stream>>>(partial, nb, K, diag_out);
  return cudaGetLastError();
}

template <int LAT>
cudaError_t launch_scheme(int scheme, const double *fields, double *partial, int nb, int nx, int ny, int nz, const int bc[6], double gamma,
                          double *diag_out, cudaStream_t stream) {
  switch (scheme) {
    case LBMHD_IDEAL: return launch_diag<LAT, kIdeal>(fields, partial, nb, nx, ny, nz, bc, gamma, diag_out, stream);
    case LBMHD_INCRES: return launch_diag<LAT, kIncres>(fields, partial, nb, nx, ny, nz, bc, gamma, diag_out, stream);
    case LBMHD_IDEAL_DIVB: return launch_diag<LAT, kIdealD>(fields, partial, nb, nx, ny, nz, bc, gamma, diag_out, stream);
    case LBMHD_RESIST: return launch_diag<LAT, kResist>(fields, partial, nb, nx, ny, nz, bc, gamma, diag_out, stream);
    default: return launch_diag<LAT, kFull>(fields, partial, nb, nx, ny, nz, bc, gamma, diag_out, stream);
  }
}

}  // namespace

extern "C" {

int lbmhd_diagnostics_static(int scheme, int lattice, int nx, int ny, int nz, const int bc[6], double gamma, const double *fields,
                             double *diag_out, int device, void *stream) {
  if (scheme != LBMHD_IDEAL && scheme != LBMHD_INCRES && scheme != LBMHD_IDEAL_DIVB && scheme != LBMHD_RESIST && scheme != LBMHD_FULL)
    return fail(LBMHD_EINVAL, "unknown scheme %d", scheme);
  if (lattice < LBMHD_D1Q3 || lattice > LBMHD_D3Q7) return fail(LBMHD_EINVAL, "unknown lattice %d", lattice);
  const int D = lattice == LBMHD_D1Q3 ? 1 : ((lattice == LBMHD_D2Q9 || lattice == LBMHD_D2Q5) ? 2 : 3);
  if (!bc) return fail(LBMHD_EINVAL, "bc is NULL");
  if (nx < 1 || ny < 1 || nz < 1 || (D < 2 && ny != 1) || (D < 3 && nz != 1)) return fail(LBMHD_EINVAL, "bad dims %d x %d x %d for a %dD lattice", nx, ny, nz, D);
  const unsigned long long N = (unsigned long long)nx * (unsigned long long)ny * (unsigned long long)nz;
  if (N > kStaticMaxCells)
    return fail(LBMHD_ENOMEM, "lbmhd_diagnostics_static handles at most %llu cells, got %llu (use lbmhd_diagnostics with a workspace)", kStaticMaxCells, N);
  CUDA_TRY(cudaSetDevice(device));
  double *partial = nullptr;
  if (int rc = scratch_for(device, &partial)) return rc;
  if (!fields && !diag_out) return LBMHD_OK;      // set-up only: the address is now known for this device
  if (!fields || !diag_out) return fail(LBMHD_EINVAL, "fields and diag_out must both be given (or both NULL for set-up only)");
  const unsigned long long want = (N + kDiagThreads - 1) / kDiagThreads;
  const int nb = (int)(want < (unsigned long long)kMaxDiagBlocks ? want : (unsigned long long)kMaxDiagBlocks);      // as lbmhd_moments does
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e;
  switch (lattice) {
    case LBMHD_D1Q3: e = launch_scheme<1>(scheme, fields, partial, nb, nx, ny, nz, bc, gamma, diag_out, st); break;
    case LBMHD_D2Q9: e = launch_scheme<2>(scheme, fields, partial, nb, nx, ny, nz, bc, gamma, diag_out, st); break;
    case LBMHD_D3Q19: e = launch_scheme<3>(scheme, fields, partial, nb, nx, ny, nz, bc, gamma, diag_out, st); break;
    case LBMHD_D2Q5: e = launch_scheme<4>(scheme, fields, partial, nb, nx, ny, nz, bc, gamma, diag_out, st); break;
    default: e = launch_scheme<5>(scheme, fields, partial, nb, nx, ny, nz, bc, gamma, diag_out, st); break;
  }
  if (e != cudaSuccess) return fail(LBMHD_ECUDA, "diagnostics kernel launch: %s", cudaGetErrorString(e));
  return LBMHD_OK;
}

}  // extern "C"
