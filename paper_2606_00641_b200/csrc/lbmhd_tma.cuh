// lbmhd_tma.cuh — TMA-staged persistent variant of the fused step kernel for sm_100a.
//
// Why: with plain pulls every in-flight byte is pinned to a register of a resident warp, and the fp64
// D3Q19 kernel (19 populations + addresses per thread) tops out at 24 warps/SM: ncu shows 54-62 % DRAM
// utilisation with long-scoreboard stalls dominating.  Here the pull is done by the TMA unit instead:
// one producer thread per CTA issues Q tensor copies per tile (cp.async.bulk.tensor.5d), each moving the
// [K][TXT] box of direction i for all K sets with the lattice shift -c_i applied in the box COORDINATES
// (so misaligned x-shifts, and out-of-domain rows, cost nothing: TMA zero-fills what is outside).  The
// boxes land in a ring of NSTAGE shared-memory stages guarded by mbarriers, so ~(NSTAGE-1) tiles
// (~150 KB per SM) are in flight regardless of how many registers the math needs.  Two consumer groups
// of TXT*K threads alternate over the tiles: read their Q populations from shared memory, release the
// stage at once, then run the same finish_cell() as the plain kernel and store straight to global.
//
// TMA box starts must be 16-byte aligned (a box starting at an odd fp64 x faults with "illegal instruction"),
// so directions with c_x != 0 load an aligned window PAD = 16/sizeof(real) elements wider than the tile
// (start x0 - PAD for c_x = +1, x0 for c_x = -1) and the consumer reads it at a one-element offset.
//
// Population tensor as TMA sees it (fastest first): x (nx), y (ny), z (nz), i (Q), k (K).
#pragma once
#include <cuda.h>

#include "lbmhd_kernels.cuh"

namespace lbk {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_5d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2, int c3,
                                            int c4) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
      : "memory");
}

template <int LAT, int SCHEME, typename real, int TXT, int NSTAGE> struct TmaCfg {
  using L = Lattice<LAT>;
  static constexpr int Q = L::Q, D = L::D, K = Vars<SCHEME, L::D>::K;
  static constexpr int PAD = 16 / (int)sizeof(real);       // elements per 16 bytes
  static constexpr int GROUP = TXT * K;                    // consumer threads per group
  static constexpr int NGROUP = 2;
  static constexpr int THREADS = NGROUP * GROUP + 32;      // + one producer warp
  __host__ __device__ static constexpr int width(int i) { return L::cx(i) == 0 ? TXT : TXT + PAD; }
  __host__ __device__ static constexpr size_t box_bytes(int i) { return (size_t)K * width(i) * sizeof(real); }
  __host__ __device__ static constexpr size_t slot_bytes(int i) { return (box_bytes(i) + 127) / 128 * 128; }
  __host__ __device__ static constexpr size_t slot_off(int i) {      // byte offset of direction i inside a stage
    size_t o = 0;
    for (int j = 0; j < i; j++) o += slot_bytes(j);
    return o;
  }
  __host__ __device__ static constexpr size_t tx_bytes() {           // bytes TMA delivers per stage
    size_t o = 0;
    for (int j = 0; j < Q; j++) o += box_bytes(j);
    return o;
  }
  static constexpr size_t STAGE_BYTES = slot_off(Q);
  static constexpr size_t OFF_SQ = (size_t)NSTAGE * STAGE_BYTES;
  static constexpr size_t OFF_STR = OFF_SQ + (size_t)NGROUP * K * TXT * sizeof(real);
  static constexpr size_t OFF_BAR = OFF_STR + (size_t)NGROUP * D * D * TXT * sizeof(real);
  static constexpr size_t SMEM_BYTES = OFF_BAR + 2 * NSTAGE * sizeof(uint64_t) + 128;   // + alignment slack
};

template <int LAT, int SCHEME, typename real, int TXT, int NSTAGE>
__global__ void __launch_bounds__(TmaCfg<LAT, SCHEME, real, TXT, NSTAGE>::THREADS, 1)
step_kernel_tma(const __grid_constant__ StepArgs<real> a, const __grid_constant__ CUtensorMap map_tile, const __grid_constant__ CUtensorMap map_wide,
                int tiles_x, int n_rows) {
  using C = TmaCfg<LAT, SCHEME, real, TXT, NSTAGE>;
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q, K = C::K;
  // no static shared memory in this kernel, so the dynamic window starts at shared offset 0 (checked below);
  // no integer round trip on the pointer, so every access below stays an LDS/STS (not a generic LD/ST)
  extern __shared__ __align__(1024) unsigned char smem[];
  uint64_t *full = (uint64_t *)(smem + C::OFF_BAR);
  uint64_t *empty = full + NSTAGE;

  const int tid = threadIdx.x;
  const int nx = a.nx, ny = a.ny, nz = a.nz;
  if (tid == 0) {
    if ((smem_u32(smem) & 127u) != 0) __trap();
#pragma unroll
    for (int s = 0; s < NSTAGE; s++) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], C::GROUP / 32);      // one arrival per consumer warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const bool npy = D > 1 && a.bc[2] != BC_PERIODIC, npz = D > 2 && a.bc[4] != BC_PERIODIC;
  const bool npx = a.bc[0] != BC_PERIODIC;

  if (tid >= C::NGROUP * C::GROUP) {
    // ---------------- producer warp: one elected lane feeds the ring ----------------
    if (tid == C::NGROUP * C::GROUP) {
      // work unit = one (y, z) row, rows dealt round-robin to the CTAs; a CTA walks the tiles_x tiles of its row
      // in order, so every CTA gets the same mix of face tiles and interior tiles and streams whole rows
      int row = (int)blockIdx.x;
      int y = row % ny, z = row / ny, bx = 0;
      const int dy = (int)(gridDim.x % ny), dz = (int)(gridDim.x / ny);
      int s = 0;
      uint32_t ph = 0;
      while (row < n_rows) {
        mbar_wait(&empty[s], ph ^ 1u);
        mbar_expect_tx(&full[s], (uint32_t)C::tx_bytes());
        unsigned char *dst = smem + (size_t)s * C::STAGE_BYTES;
#pragma unroll
        for (int i = 0; i < Q; i++) {
          int sy = y - L::cy(i), sz = z - L::cz(i);
          if (!npy && D > 1) sy = sy < 0 ? ny - 1 : (sy >= ny ? 0 : sy);
          if (!npz && D > 2) sz = sz < 0 ? nz - 1 : (sz >= nz ? 0 : sz);
          // aligned window: c_x = +1 needs x0-1.. -> start x0-PAD; c_x = -1 needs ..x0+TXT -> start x0, PAD wider
          const int c0 = L::cx(i) == 1 ? bx * TXT - C::PAD : bx * TXT;
          tma_load_5d(dst + C::slot_off(i), L::cx(i) == 0 ? &map_tile : &map_wide, &full[s], c0, sy, sz, i, 0);
        }
        if (++s == NSTAGE) { s = 0; ph ^= 1u; }
        if (++bx == tiles_x) {
          bx = 0; row += (int)gridDim.x; y += dy; z += dz;
          if (y >= ny) { y -= ny; z += 1; }
        }
      }
    }
    return;
  }

  // ---------------- consumers: group g takes this CTA's tiles j = g, g + 2, ... ----------------
  const int g = tid / C::GROUP;
  const int lt = tid - g * C::GROUP;
  const int tx = lt % TXT, k = lt / TXT;
  real(*sQ)[TXT] = (real(*)[TXT])(smem + C::OFF_SQ + (size_t)g * K * TXT * sizeof(real));
  real(*sTr)[TXT] = (real(*)[TXT])(smem + C::OFF_STR + (size_t)g * D * D * TXT * sizeof(real));
  const uint32_t ps = (uint32_t)a.pstride;
  const real *__restrict__ srck = a.src + (size_t)k * Q * a.pstride;
  real *__restrict__ dstk = a.dst + (size_t)k * Q * a.pstride;
  auto gsync = [g] {
    if (g == 0) asm volatile("bar.sync 1, %0;" ::"n"(C::GROUP) : "memory");
    else asm volatile("bar.sync 2, %0;" ::"n"(C::GROUP) : "memory");
  };
  const Share<real, TXT, false, decltype(gsync)> sh{sQ, sTr, nullptr, nullptr, nullptr, nullptr, gsync};

  // this group's tiles: the CTA's tile sequence (rows blockIdx.x, + gridDim.x, ...; tiles_x tiles per row) taken
  // alternately by the two groups; (row, bx, y, z), stage and phase are kept incrementally
  int row = (int)blockIdx.x, bx = g;
  int y = row % ny, z = row / ny;
  const int dy = (int)(gridDim.x % ny), dz = (int)(gridDim.x / ny);
  int s = g % NSTAGE;
  uint32_t ph = (uint32_t)((g / NSTAGE) & 1);
  for (;;) {
    while (bx >= tiles_x) {
      bx -= tiles_x; row += (int)gridDim.x; y += dy; z += dz;
      if (y >= ny) { y -= ny; z += 1; }
    }
    if (row >= n_rows) break;
    const int x = bx * TXT + tx;
    const bool active = x < nx;
    const uint32_t n = ((uint32_t)z * ny + y) * nx + (active ? x : 0);
    const bool x_lo = x == 0, x_hi = x == nx - 1;
    const bool y_lo = D > 1 && y == 0, y_hi = D > 1 && y == ny - 1;
    const bool z_lo = D > 2 && z == 0, z_hi = D > 2 && z == nz - 1;
    const bool edge_x = bx == 0 || bx == tiles_x - 1;
    // tile-uniform classification: the interior fluid tile takes the lean path
    const bool touches_face = (npy && (y_lo || y_hi)) || (npz && (z_lo || z_hi)) || (npx && edge_x);
    const bool special = touches_face || a.mask != nullptr || sphere_may_touch<real, D>(a, bx * TXT, TXT, y, z);

    bool frozen = false;
    if (special && active) {
      frozen = (a.mask != nullptr && a.mask[n] == CELL_FROZEN) || (x_lo && a.bc[0] == BC_INFLOW) ||
               (x_hi && a.bc[1] == BC_INFLOW) || (y_lo && a.bc[2] == BC_INFLOW) || (y_hi && a.bc[3] == BC_INFLOW) ||
               (z_lo && a.bc[4] == BC_INFLOW) || (z_hi && a.bc[5] == BC_INFLOW);
      if (frozen) {
#pragma unroll
        for (int i = 0; i < Q; i++) dstk[(uint32_t)i * ps + n] = srck[(uint32_t)i * ps + n];
      }
    }
    const bool work = active && !frozen;

    // S1: the pulled populations are already in the stage; take them and hand the stage back at once
    mbar_wait(&full[s], ph);
    const unsigned char *st = smem + (size_t)s * C::STAGE_BYTES;
    real f[Q];
#pragma unroll
    for (int i = 0; i < Q; i++) {
      const int off = L::cx(i) == 1 ? C::PAD - 1 : (L::cx(i) == -1 ? 1 : 0);
      f[i] = ((const real *)(st + C::slot_off(i)))[k * C::width(i) + tx + off];
    }
    __syncwarp();
    if ((lt & 31) == 0) mbar_arrive(&empty[s]);

    // periodic x: the one element TMA zero-filled beyond a row end comes from the other end of the row
    if (!npx && edge_x && work && (x_lo || x_hi)) {
      const int ym = y_lo ? ny - 1 : y - 1, yp = y_hi ? 0 : y + 1;
      const int zm = z_lo ? nz - 1 : z - 1, zp = z_hi ? 0 : z + 1;
#pragma unroll
      for (int i = 0; i < Q; i++) {
        const int cx = L::cx(i), cy = L::cy(i), cz = L::cz(i);
        if ((cx == 1 && x_lo) || (cx == -1 && x_hi)) {
          const int sx = cx == 1 ? nx - 1 : 0;
          const int sy = cy == 1 ? ym : (cy == -1 ? yp : y);
          const int sz = cz == 1 ? zm : (cz == -1 ? zp : z);
          const bool outside = (cy == 1 && npy && y_lo) || (cy == -1 && npy && y_hi) || (cz == 1 && npz && z_lo) ||
                               (cz == -1 && npz && z_hi);
          if (!outside) f[i] = srck[(uint32_t)i * ps + ((uint32_t)sz * ny + sy) * nx + sx];
        }
      }
    }
    if (!work) {
#pragma unroll
      for (int i = 0; i < Q; i++) f[i] = real(0);
    }
    const StoreOwn<real> sto{reinterpret_cast<char *>(dstk + n), a.st_off};
    if (!special) {
      CellCtx c{tx, k, x, y, z, n, work, false, false, false, false, false, false, false};
      finish_cell<LAT, SCHEME, real, TXT, false, false, ST_AB>(a, c, f, sto, sh);
    } else {
      CellCtx c{tx, k, x, y, z, n, work, npx && x_lo, npx && x_hi, npy && y_lo, npy && y_hi, npz && z_lo, npz && z_hi, false};
      finish_cell<LAT, SCHEME, real, TXT, true, true, ST_AB>(a, c, f, sto, sh);
    }
    gsync();      // sQ / sTr are reused by this group's next tile
    s += 2;
    if (s >= NSTAGE) { s -= NSTAGE; ph ^= 1u; }
    bx += 2;
  }
}

}  // namespace lbk
