// lbmhd_resident.cuh — many steps of a 1D lattice with the populations RESIDENT IN REGISTERS.
//
// Config 1 (BASELINE: 800 cells of D1Q3, 8 sets) is 0.15 MB: a step is not bound by HBM but by the dependent chain
// load -> moment -> barrier -> flux -> store -> fence -> grid barrier of step_kernel_persist (2.9 us per step, of which the global
// round trips and the GPU-scope fence before the grid barrier are the larger part).  Here the lattice is split over ONE
// thread-block cluster (<= 16 CTAs of TXR cells x K rows); every thread keeps the Q populations of its (cell, row) in registers
// for all n steps, the pull along x is an exchange through shared memory, and the two populations per row that cross a CTA
// boundary travel through distributed shared memory with st.async, which signals the receiver's mbarrier by byte count
// (complete_tx): no global access, no fence and no grid barrier inside the loop.
//
//   per step:  [stream]  own c_x = +-1 populations -> sG[buffer][dir][row][1 + cell]; the CTA's end cells also send theirs into the
//                        neighbour CTA's halo slots (0 and na + 1); block barrier + mbarrier wait; f_i(x) = g_i(x - c_i)
//              [faces]   A9-A11 as in run_tile: periodic = the wrap neighbour delivers the halo; INFLOW = the face cell keeps its
//                        populations; ZEROGRAD = the outside direction takes f^eq of the inward neighbour's state Q^nb
//                        (A/B: the sum of its stored populations; in place: its published moment Q_k + inj)
//              [collide] finish_cell (S2-S8: the same code every other step kernel runs), its store policy writing registers
//
// Flow control: a CTA sends halo(s + 1) only after it has received halo(s) from both neighbours, so a CTA is never more than one
// step ahead of a neighbour: two halo buffers and two mbarriers, used alternately, are enough (the j-th use of a barrier waits for
// phase parity j & 1).  A cluster barrier after the mbarrier initialisation makes every CTA resident before anything is sent;
// one before the exit keeps every CTA alive until nothing more can arrive.
//
// Layouts: the resident state is g_i(x), the post-collision population of direction i at cell x.  A/B and layout P0 of the in-place
// scheme store it at (slot i, cell x); layout P1 (after a pull-push step) at (slot opp(i), cell x + c_i), wrapped on a periodic
// axis, and parked at (slot i, cell x) when x + c_i is outside a non-periodic face (StorePPEdge).  The kernel reads either layout
// and writes the one the step count leads to, so any n from any parity is one launch; in place it also leaves the published
// moments M of its last step behind.
#pragma once
#include "lbmhd_kernels.cuh"

namespace lbk {

template <typename real> struct ResidentArgs {
  int n_steps;
  int ncta;              // CTAs of the one cluster = ceil(nx / TXR)
  const real *pop_in;    // the copy the first step reads
  real *pop_out;         // the copy the last step's result belongs in (A/B: copy (cur + n) & 1; in place: the single copy)
  int layout_in, layout_out;   // in place: 0 = P0, 1 = P1 (A/B: 0)
  const double *M_in;    // in place: the published moments the first step reads (M_cur)
  double *M_out[2];      // in place: both published-moment arrays take the last step's moments
};

template <typename real, int Q> struct StoreRegs {
  real *g;
  __device__ __forceinline__ void put(int i, real v) const { g[i] = v; }
};

template <class L> __host__ __device__ constexpr int dir_with_cx(int cx) {
  for (int i = 0; i < L::Q; i++)
    if (L::cx(i) == cx) return i;
  return -1;
}

__device__ __forceinline__ void mbar_init(unsigned long long *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(cl_smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(cl_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, uint32_t parity) {
  const uint32_t b = cl_smem_u32(bar);
  uint32_t ok;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok)
                 : "r"(b), "r"(parity)
                 : "memory");
  } while (!ok);
}

template <int LAT, int SCHEME, typename real, int TXR, bool INPLACE>
__global__ void __launch_bounds__(TXR * Vars<SCHEME, Lattice<LAT>::D>::K, 1)
step_kernel_resident(const __grid_constant__ StepArgs<real> a0, const __grid_constant__ ResidentArgs<real> p) {
  using L = Lattice<LAT>;
  static_assert(L::D == 1, "one-dimensional lattices");
  constexpr int D = 1, Q = L::Q, K = Vars<SCHEME, D>::K;
  constexpr int STREAM = INPLACE ? ST_LOC : ST_AB;      // finish_cell: ST_LOC publishes Q_k + inj through M_next
  constexpr int ip = dir_with_cx<L>(1), im = dir_with_cx<L>(-1);
  static_assert(ip > 0 && im > 0 && Q == 3, "D1Q3");
  __shared__ real sQ[K][TXR];
  __shared__ real sTr[D * D][TXR];
  __shared__ real sNb[K];
  __shared__ real sG[2][2][K][TXR + 2];      // [buffer][0: c_x = +1, 1: c_x = -1][row][1 + cell]; slots 0 and na + 1 are the halo
  __shared__ real sS[2][K];                  // state of the inward neighbour of the low / high face
  __shared__ double sM[INPLACE ? K : 1][TXR];
  __shared__ StepArgs<real> sa;
  __shared__ __align__(8) unsigned long long mbar[2];
  static_assert(sizeof(StepArgs<real>) % 4 == 0, "word copy");

  const int tx = threadIdx.x, k = threadIdx.y, tid = k * TXR + tx;
  const int nx = a0.nx, rank = (int)blockIdx.x, ncta = p.ncta;
  const int x0 = rank * TXR, x = x0 + tx;
  const int na = nx - x0 < TXR ? nx - x0 : TXR;      // cells of this CTA
  const bool active = tx < na;
  const bool periodic = a0.bc[0] == BC_PERIODIC;
  const bool face_lo = active && !periodic && x == 0, face_hi = active && !periodic && x == nx - 1;
  const bool frozen = (face_lo && a0.bc[0] == BC_INFLOW) || (face_hi && a0.bc[1] == BC_INFLOW);
  const bool zg_lo = face_lo && a0.bc[0] == BC_ZEROGRAD, zg_hi = face_hi && a0.bc[1] == BC_ZEROGRAD;
  const bool nb_lo = active && !periodic && a0.bc[0] == BC_ZEROGRAD && x == 1;            // publishes Q^nb for the low face
  const bool nb_hi = active && !periodic && a0.bc[1] == BC_ZEROGRAD && x == nx - 2;
  const int left = rank > 0 ? rank - 1 : (periodic ? ncta - 1 : -1);
  const int right = rank < ncta - 1 ? rank + 1 : (periodic ? 0 : -1);
  const uint32_t expect = (uint32_t)((left >= 0 ? 1 : 0) + (right >= 0 ? 1 : 0)) * (uint32_t)(K * sizeof(real));

  {      // the arguments finish_cell sees: M_next = this CTA's sM[K][TXR] (index k * (nx ny nz) + n with nx := TXR, n := tx)
    const uint32_t *src = reinterpret_cast<const uint32_t *>(&a0);
    uint32_t *dst = reinterpret_cast<uint32_t *>(&sa);
    for (int j = tid; j < (int)(sizeof(StepArgs<real>) / 4); j += TXR * K) dst[j] = src[j];
  }
  if (tid == 0) {
    mbar_init(&mbar[0], 1);
    mbar_init(&mbar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
    sa.nx = TXR;
    sa.ny = 1;
    sa.nz = 1;
    sa.M_cur = nullptr;
    sa.M_next = INPLACE ? &sM[0][0] : nullptr;
  }
  cluster_arrive_release();
  cluster_wait_acquire();

  // where this thread's crossing populations go in the neighbour CTAs (shared::cluster addresses)
  const int na_left = left == ncta - 1 ? nx - left * TXR : TXR;
  const uint32_t sG0 = cl_smem_u32(&sG[0][0][0][0]), bar0 = cl_smem_u32(&mbar[0]);
  const bool send_r = active && tx == na - 1 && right >= 0, send_l = tx == 0 && left >= 0;
  uint32_t rG = 0, rbar = 0, slot = 0;
  if (send_r) { rG = cl_mapa(sG0, (uint32_t)right); rbar = cl_mapa(bar0, (uint32_t)right); slot = (uint32_t)((0 * K + k) * (TXR + 2) + 0); }
  uint32_t lG = 0, lbar = 0, lslot = 0;
  if (send_l) { lG = cl_mapa(sG0, (uint32_t)left); lbar = cl_mapa(bar0, (uint32_t)left); lslot = (uint32_t)((1 * K + k) * (TXR + 2) + na_left + 1); }
  constexpr uint32_t BUF = (uint32_t)(2 * K * (TXR + 2));      // elements per buffer

  // (slot, cell) of g_i(x) in layout P0 / P1
  auto where = [&](int i, int layout, int &slot_i, int &cell) {
    slot_i = i;
    cell = x;
    if (layout != 0 && L::cx(i) != 0) {
      int xs = x + L::cx(i);
      if (periodic) xs = xs < 0 ? xs + nx : (xs >= nx ? xs - nx : xs);
      if (xs >= 0 && xs < nx) { slot_i = opp(i); cell = xs; }
    }
  };
  real g[Q], f[Q];
#pragma unroll
  for (int i = 0; i < Q; i++) {
    int si, xc;
    where(i, INPLACE ? p.layout_in : 0, si, xc);
    g[i] = active ? p.pop_in[((size_t)k * Q + si) * a0.pstride + xc] : real(0);
  }
  real pub = real(0);      // in place: this cell's published moment Q_k + inj of the previous step
  if (INPLACE && (nb_lo || nb_hi)) pub = (real)p.M_in[(size_t)k * nx + x];
  const Share<real, TXR, false> sh{sQ, sTr, sNb, nullptr, nullptr, nullptr, SyncBlock{}};

  for (int s = 0; s < p.n_steps; s++) {
    const uint32_t b = (uint32_t)(s & 1);
    // ---- stream: f_i(x) = g_i(x - c_i) ----
    if (active) {      // (an inactive thread's slot na + 1 .. is the halo the wrap neighbour delivers into)
      sG[b][0][k][tx + 1] = g[ip];
      sG[b][1][k][tx + 1] = g[im];
    }
    if (send_r) cl_st_async(rG + (b * BUF + slot) * (uint32_t)sizeof(real), g[ip], rbar + b * 8u);
    if (send_l) cl_st_async(lG + (b * BUF + lslot) * (uint32_t)sizeof(real), g[im], lbar + b * 8u);
    if (nb_lo || nb_hi) {
      // A/B: the stored populations of the neighbour summed as the x-edge tile does (butterfly over lanes 0 .. 2: (g0 + g2) + g1)
      const real v = INPLACE ? pub : (g[0] + g[2]) + g[1];
      if (nb_lo) sS[0][k] = v;
      if (nb_hi) sS[1][k] = v;
    }
    if (expect != 0 && tid == 0) mbar_expect_tx(&mbar[b], expect);
    __syncthreads();
    if (expect != 0) mbar_wait(&mbar[b], (uint32_t)((s >> 1) & 1));
    f[0] = g[0];
    f[ip] = sG[b][0][k][tx];
    f[im] = sG[b][1][k][tx + 2];
    if (zg_lo || zg_hi) {
      real Qnb[K], Phi[3];
#pragma unroll
      for (int l = 0; l < K; l++) Qnb[l] = sS[zg_lo ? 0 : 1][l];
      const real Qnbk = pick<K, real>(Qnb, k);
      flux_row<SCHEME, D, real>(k, Qnb, Qnbk, a0.gamma, a0.c0sq, a0.eta, a0.mu, a0.inv_tau_relax, Phi);
      const int i = zg_lo ? ip : im;
      const real cPhi = real(zg_lo ? 1 : -1) * Phi[0] + real(0) * Phi[1] + real(0) * Phi[2];
      const real v = real(L::w(ip)) * (Qnbk + real(L::inv_cs2) * cPhi);
      if (i == ip) f[ip] = v;
      else f[im] = v;
    }
    // ---- collide (S2-S8) into registers; a frozen face cell keeps its populations ----
    real gn[Q];
#pragma unroll
    for (int i = 0; i < Q; i++) gn[i] = g[i];
    const CellCtx c{tx, k, x, 0, 0, (uint32_t)tx, active && !frozen, false, false, false, false, false, false, true};
    const StoreRegs<real, Q> st{gn};
    finish_cell<LAT, SCHEME, real, TXR, false, false, STREAM>(sa, c, f, st, sh);
#pragma unroll
    for (int i = 0; i < Q; i++) g[i] = active ? gn[i] : real(0);
    if (INPLACE && active && !frozen) pub = (real)sM[k][tx];
  }

  if (active) {
#pragma unroll
    for (int i = 0; i < Q; i++) {
      int si, xc;
      where(i, INPLACE ? p.layout_out : 0, si, xc);
      p.pop_out[((size_t)k * Q + si) * a0.pstride + xc] = g[i];
    }
    if (INPLACE && !frozen && p.n_steps > 0) {
      p.M_out[0][(size_t)k * nx + x] = (double)pub;
      p.M_out[1][(size_t)k * nx + x] = (double)pub;
    }
  }
  cluster_arrive_release();      // nobody exits while a neighbour may still deliver into it
  cluster_wait_acquire();
}

}  // namespace lbk
