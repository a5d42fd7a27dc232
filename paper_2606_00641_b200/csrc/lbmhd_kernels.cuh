// lbmhd_kernels.cuh — CUDA kernels of the fused VLBM step for sm_100a.
//
// Mapping: ONE THREAD PER (CELL, VARIABLE).  A block owns TX consecutive x-cells of one (y, z) row and
// all K population sets: blockDim = (TX, K), so every warp is 32 consecutive x of ONE variable k and
// each of its Q loads / Q stores is one fully coalesced 32*sizeof(real) row segment of plane (k, i).
// A thread keeps only its own Q populations in registers (19 fp64 for D3Q19) — the 8 x 19 = 152 fp64
// of a D3Q19 cell do not fit one thread's 255 registers.  The only coupling between the K sets of a
// cell is the K zeroth moments plus tr Pi_B; they go through (K+1)*TX reals of shared memory and one
// __syncthreads().  The per-variable branches below are warp-uniform (k = threadIdx.y).
//
// DRAM traffic per cell update = K*Q loads + K*Q stores, each population read exactly once (pull
// scheme: population (k,i) at x - c_i is read only by cell x).  Shifts in x misalign a warp's 256-byte
// segment by one element; the straddled 32-byte sector is re-read from L2/L1, not from DRAM.
#pragma once
#include <cooperative_groups.h>
#include <cooperative_groups/reduce.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "lbmhd_lattice.cuh"

namespace lbk {

enum { BC_PERIODIC = 0, BC_ZEROGRAD = 1, BC_INFLOW = 2, BC_HALO = 3 };
enum { CELL_FLUID = 0, CELL_FROZEN = 1, CELL_SOLID = 2 };

template <typename real> struct StepArgs {
  const real *src;              // populations read (plane (k,i) at (k*Q+i)*pstride)
  real *dst;                    // populations written
  size_t pstride;               // elements between planes
  int nx, ny, nz;
  int bc[6];
  real omega[26];               // 1 / tau_k (K <= 26)
  real tau[26];                 // tau_k (fp32 collide: inj / omega without a division)
  real inv_tauB_cs2;            // 1 / (tau_B c_s^2)
  real kappa, gamma, c0sq;
  real inv_tau_relax;           // kIdealD, kResist: 1 / tau_M of the relaxation variables (Eq.6)
  real eta;                     // kResist, kFull: magnetic diffusivity of the flux terms -eta grad B, eta j x B
  real mu;                      // kFull: shear viscosity of the flux terms -sigma, -u.sigma
  real etaj_inv_jc2;            // kIncres: 1 / j_c^2 of eta(j) = eta0 (1 + (j/j_c)^2), 0 = constant eta
  real tauB0;                   // tau of the magnetic sets at zero current
  const unsigned char *mask;    // [N] or nullptr
  const double *Bsolid;         // [3][N] or nullptr
  const double *dfield;         // lattice porosity d in [0,1] per cell (Eq.15) or nullptr: d from the mask (SOLID -> 0)
  double usolid[3];
  long long ld_off[19];         // bytes from a cell's own slot in plane (k,0) to its pull source in plane (k,i), no wrap:
                                //   (i*pstride - (c_x + c_y nx + c_z nx ny)) * sizeof(real)
  long long st_off[19];         // i * pstride * sizeof(real)
  const double *M_cur;          // in-place modes: post-collision moments [K][N] published last step (and the constant
                                //   state of frozen cells); nullptr in A/B mode
  double *M_next;               // in-place modes: moments published by this step
  int hoff;                     // slab decomposition: global index of local plane 0 along the slowest lattice axis
  int row0, row1;               // planes [row0, row1) of the slowest lattice axis this launch covers (lbmhd_step_part: a plane range)
  long long kplane;             // Q * pstride * sizeof(real): bytes from plane (k, i) to plane (k + 1, i)
  int has_sphere;
  double sph_c[3], sph_R, sph_R2, sph_u[3];
  double sph_om[3];             // angular velocity of the body: u^B = sph_u + sph_om x r
  int n_dip;                    // dipole ensemble of the sphere, offsets and axes already rotated by the host
  double dip_off[4][3], dip_m[4][3], dip_Bs[4], dip_core[4];
  double obs_om[3], obs_c[3];   // masked bodies: u^B = usolid + obs_om x (x - obs_c)
  double sph_eps, sph_touch2;   // width of the linear porosity ramp (Eq.15-16), 0 = sharp; (R + eps/2)^2
  double *body;                 // body integrals accumulator [14] (A21) or nullptr = off
  double body_ref[3];           // torque reference of masked bodies; an analytic sphere uses its centre
};

// ---- homogenised solid state at a cell (Eq.13-16; A8, A11, A12) ----------
// Returns the lattice porosity d in [0,1] and fills uS, BS when d < 1.  The sharp-sphere decision
// |x - c|^2 <= R^2 is taken in fp64 with separately rounded products and sums, the order the oracle uses,
// so both sides agree on the integer outcome; the ramp d = clamp(phi/eps + 1/2, 0, 1) is continuous.
template <typename real, int D>
__device__ __forceinline__ double solid_state(const StepArgs<real> &a, int x, int y, int z, size_t n, double uS[3],
                                              double BS[3]) {
  if (a.has_sphere) {
    double r[3];
    r[0] = __dsub_rn((double)x, a.sph_c[0]);
    r[1] = D > 1 ? __dsub_rn((double)(y + (D == 2 ? a.hoff : 0)), a.sph_c[1]) : 0.0;
    r[2] = D > 2 ? __dsub_rn((double)(z + a.hoff), a.sph_c[2]) : 0.0;
    double r2 = __dmul_rn(r[0], r[0]);
    r2 = __dadd_rn(r2, __dmul_rn(r[1], r[1]));
    r2 = __dadd_rn(r2, __dmul_rn(r[2], r[2]));
    if (r2 <= a.sph_touch2) {
      const double rn = sqrt(r2);
      double d;
      if (a.sph_eps > 0.0) d = fmin(fmax((rn - a.sph_R) / a.sph_eps + 0.5, 0.0), 1.0);
      else d = r2 <= a.sph_R2 ? 0.0 : 1.0;
      if (d < 1.0) {
        BS[0] = BS[1] = BS[2] = 0.0;
        for (int j = 0; j < a.n_dip; j++) {     // 1/2 Bs_j (R / max(|r_j|, core_j))^3 [3 (m_j.r^_j) r^_j - m_j]
          double rj[3], rj2 = 0.0;
#pragma unroll
          for (int c = 0; c < 3; c++) {
            rj[c] = c < D ? r[c] - a.dip_off[j][c] : 0.0;
            rj2 = rj2 + rj[c] * rj[c];
          }
          const double rjn = sqrt(rj2);
          const double rc = rjn > a.dip_core[j] ? rjn : a.dip_core[j];
          const double q = a.sph_R / rc;
          const double amp = 0.5 * a.dip_Bs[j] * (q * q * q);
          double rh[3], mr = 0.0;
#pragma unroll
          for (int c = 0; c < 3; c++) {
            rh[c] = rjn > 0.0 ? rj[c] / rjn : 0.0;
            mr += a.dip_m[j][c] * rh[c];
          }
#pragma unroll
          for (int c = 0; c < 3; c++) BS[c] += amp * (3.0 * mr * rh[c] - a.dip_m[j][c]);
        }
        uS[0] = a.sph_u[0] + (a.sph_om[1] * r[2] - a.sph_om[2] * r[1]);
        uS[1] = a.sph_u[1] + (a.sph_om[2] * r[0] - a.sph_om[0] * r[2]);
        uS[2] = a.sph_u[2] + (a.sph_om[0] * r[1] - a.sph_om[1] * r[0]);
        return d;
      }
    }
  }
  double d = 1.0;
  if (a.dfield != nullptr) d = a.dfield[n];
  else if (a.mask != nullptr && a.mask[n] == CELL_SOLID) d = 0.0;
  if (d < 1.0) {
    const double rx = (double)x - a.obs_c[0];
    const double ry = D > 1 ? (double)(y + (D == 2 ? a.hoff : 0)) - a.obs_c[1] : 0.0;
    const double rz = D > 2 ? (double)(z + a.hoff) - a.obs_c[2] : 0.0;
    uS[0] = a.usolid[0] + (a.obs_om[1] * rz - a.obs_om[2] * ry);
    uS[1] = a.usolid[1] + (a.obs_om[2] * rx - a.obs_om[0] * rz);
    uS[2] = a.usolid[2] + (a.obs_om[0] * ry - a.obs_om[1] * rx);
#pragma unroll
    for (int c = 0; c < 3; c++) BS[c] = a.Bsolid != nullptr ? a.Bsolid[(size_t)c * ((size_t)a.nx * a.ny * a.nz) + n] : 0.0;
  }
  return d;
}

// register-array element by a runtime (warp-uniform) index without spilling the array to local memory
template <int K, typename real> __device__ __forceinline__ real pick(const real *v, int k) {
  real r = v[0];
#pragma unroll
  for (int l = 1; l < K; l++)
    if (k == l) r = v[l];
  return r;
}

// ---- S2: zeroth moment Q_k = sum_i f_i (Eq.4) ---------------------------------------------------------------
// fp64: index order, the order of the oracle.  fp32: the rounding error d of this sum re-enters the populations as w_i omega d
// (Eq.2-3) and so lands, amplified by omega ~ 2, in the conserved sum itself every step: it is the largest single source of
// fp32 drift (config 4, 100 steps: 1.2e-5 on rho with the index-order sum).  So fp32 adds the small populations first —
// diagonal directions (w = 1/36), then axis directions, the rest population (the largest) last — with two accumulators per
// weight class: the same Q - 1 additions, shorter dependency chains, partial sums that stay small until the last two adds.
// two_sum: s = fl(a + b) and e with a + b = s + e exactly (Knuth); no multiplication, so nothing here can be contracted.
template <typename real> __device__ __forceinline__ void two_sum(real a, real b, real &s, real &e) {
  s = a + b;
  const real bb = s - a;
  e = (a - (s - bb)) + (b - bb);
}

// lo (fp32 only; 0 in fp64): what the last two additions of the sum rounded away, Q_k = result + lo to second order.
template <class L, typename real, class FA> __device__ __forceinline__ real moment_sum(const FA &f, real &lo) {
  constexpr int Q = L::Q;
  // Every accumulator starts with its first term: `0 + x` is not x for x = -0, so the compiler keeps that addition (ncu on D2Q5
  // fp32: 7 of the 23 FADD per cell of this function and the collide were additions of zero).  The values are the same.
  if constexpr (sizeof(real) == 8) {
    real s = f[0];
#pragma unroll
    for (int i = 1; i < Q; i++) s += f[i];
    lo = real(0);
    return s;
  } else {
    // (D3Q19 keeps the zero-initialised accumulators: measured 2.5 % faster there, config 5 fp32 A/B 0.905 against 0.882 —
    // the kernel is at its register cap and the other form schedules worse; the short lattices gain 2-4 % from FIRST)
    constexpr bool FIRST = Q <= 9;
    real d0 = real(0), d1 = real(0), a0 = real(0), a1 = real(0);
    int nd = 0, na = 0;      // (compile-time after unrolling: which accumulators exist and hold a term)
#pragma unroll
    for (int i = 1; i < Q; i++) {
      const int c2 = L::cx(i) * L::cx(i) + L::cy(i) * L::cy(i) + L::cz(i) * L::cz(i);
      if (c2 > 1) {
        if (nd & 1) d1 = (FIRST && nd < 2) ? f[i] : d1 + f[i];
        else d0 = (FIRST && nd < 2) ? f[i] : d0 + f[i];
        nd++;
      } else {
        if (na & 1) a1 = (FIRST && na < 2) ? f[i] : a1 + f[i];
        else a0 = (FIRST && na < 2) ? f[i] : a0 + f[i];
        na++;
      }
    }
    const real dd = (!FIRST || nd > 1) ? d0 + d1 : d0, aa = (!FIRST || na > 1) ? a0 + a1 : a0;
    const bool both = !FIRST || (nd > 0 && na > 0);
    real s1, e1 = real(0), hi, e2;
    if (both) two_sum<real>(dd, aa, s1, e1);
    else s1 = nd > 0 ? dd : aa;
    two_sum<real>(s1, f[0], hi, e2);
    lo = both ? e1 + e2 : e2;
    return hi;
  }
}
template <class L, typename real, class FA> __device__ __forceinline__ real moment_sum(const FA &f) {
  real lo;
  return moment_sum<L, real>(f, lo);
}

// ---- S7 BGK + direct injection (Eq.2-3, A5), the populations of one (cell, variable) ------------------------
//   g'_i = f_i + w [ w_i (Q_k + c_i.Phi/c_s^2) - f_i ] + w_i inj          (w = omega_k)
// fp64: evaluated as (1 - w) f_i + w_i [w Q_k + inj] + w_i c_i.(3 w Phi): 52 instructions per thread on D3Q19.
// fp32: that form rounds w Q_k + inj and w_i [..] to 6e-8 of Q_k, and those roundings — like the one of the moment sum — land
// in sum_i g'_i, i.e. in the conserved quantity, every step (config 4, 100 steps: 1.2e-5 .. 2.4e-5 on rho and B_y).  Here the
// relaxation acts on the DEVIATION e_i = w_i Qe - f_i + w_i c_i.Phi/c_s^2, a small number whose rounding is small in absolute
// terms, with Qe = fl(Q_k + inj / w); what the additions that formed Q_k and Qe rounded away (lo, err: error-free
// transformations) is handed to the rest population, so that sum_i g'_i = Q_k + inj up to the rounding of the Q stores
// themselves.  Same instruction count per population (one FFMA instead of the FMUL).
template <class L, typename real> struct Collide {
  Collide() = default;
  real om, a0, a1, P0, P1, P2;      // fp64: a0 = 1 - w, a1 = w Q_k + inj, P = 3 w Phi | fp32: a0 = Qe, a1 = lo + err, P = 3 Phi
  __device__ __forceinline__ Collide(real om_, real tau, real Qk, real lo, real inj, const real (&Phi)[3]) : om(om_) {
    if constexpr (sizeof(real) == 8) {
      a0 = real(1) - om;
      a1 = om * Qk + inj;
      P0 = real(L::inv_cs2) * om * Phi[0]; P1 = real(L::inv_cs2) * om * Phi[1]; P2 = real(L::inv_cs2) * om * Phi[2];
    } else {
      real err;
      two_sum<real>(Qk, inj * tau, a0, err);
      a1 = lo + err;
      P0 = real(L::inv_cs2) * Phi[0]; P1 = real(L::inv_cs2) * Phi[1]; P2 = real(L::inv_cs2) * Phi[2];
    }
  }
  // out(i, f) == f: a frozen cell that goes through the tile's update unchanged
  __device__ __forceinline__ void identity() {
    if constexpr (sizeof(real) == 8) { a0 = real(1); a1 = real(0); }
    else { om = real(0); a0 = real(0); a1 = real(0); }
    P0 = P1 = P2 = real(0);
  }
  __device__ __forceinline__ real out(int i, real fi) const {
    if constexpr (sizeof(real) == 8) {
      real t = real(L::w(i)) * a1;
      if (L::cx(i) != 0) t = fma(real(L::cx(i) * L::w(i)), P0, t);
      if (L::cy(i) != 0) t = fma(real(L::cy(i) * L::w(i)), P1, t);
      if (L::cz(i) != 0) t = fma(real(L::cz(i) * L::w(i)), P2, t);
      return fma(fi, a0, t);
    } else {
      real e = fma(real(L::w(i)), a0, -fi);
      if (L::cx(i) != 0) e = fma(real(L::cx(i) * L::w(i)), P0, e);
      if (L::cy(i) != 0) e = fma(real(L::cy(i) * L::w(i)), P1, e);
      if (L::cz(i) != 0) e = fma(real(L::cz(i) * L::w(i)), P2, e);
      if (i == 0) e += a1;
      return fma(om, e, fi);
    }
  }
};

// ---- flux row of variable k: Phi_k,alpha(Qh), alpha < D (Eq.11, Eq.8; A3) -------
// Qh is the (possibly solid-blended) state: an array in registers or a column of the shared exchange array (QCol) — the
// rows read only the entries they need (a gradient row of RESIST / FULL needs 5 of the 17 / 26).  `own` = Qh[k].
// k is warp-uniform, so the branches do not diverge.
// Calls f(integral_constant<int, k>) for the run-time row k in [LO, HI) by bisection (k is warp-uniform: no divergence), so
// that the flux / source code of a row is compiled with k known: no selects, no unused terms.
template <int LO, int HI, class F> __device__ __forceinline__ void dispatch_row(int k, F &&f) {
  if constexpr (HI - LO == 1) {
    f(std::integral_constant<int, LO>{});
  } else {
    constexpr int MID = (LO + HI) / 2;
    if (k < MID) dispatch_row<LO, MID>(k, f);
    else dispatch_row<MID, HI>(k, f);
  }
}

template <int I> __device__ __forceinline__ constexpr int row_of(std::integral_constant<int, I>) { return I; }
__device__ __forceinline__ constexpr int row_of(int k) { return k; }

template <typename real, int TX> struct QCol {
  real (*s)[TX];
  int tx;
  __device__ __forceinline__ real operator[](int l) const { return s[l][tx]; }
};
template <class QA, typename real> __device__ __forceinline__ real pick3(const QA &Q, int base, int b) {
  return b == 0 ? Q[base] : (b == 1 ? Q[base + 1] : Q[base + 2]);
}

template <int SCHEME, int D, typename real, class QA>
__device__ __forceinline__ void flux_row(int k, const QA &Qh, real own, real gamma, real c0sq, real eta, real visc, real itm, real Phi[3]) {
  Phi[0] = Phi[1] = Phi[2] = real(0);
  if (is_ideal(SCHEME)) {
    if (k == 0) {
#pragma unroll
      for (int a = 0; a < D; a++) Phi[a] = Qh[1 + a];
      return;
    }
    const real ir = real(1) / Qh[0];
    const real m[3] = {Qh[1], Qh[2], Qh[3]};
    const real u[3] = {m[0] * ir, m[1] * ir, m[2] * ir};
    if (SCHEME == kIdealD && k == 8) {   // relaxation variable D = tr G: D u - B (Eq.10, traced)
#pragma unroll
      for (int a = 0; a < D; a++) Phi[a] = own * u[a] - Qh[5 + a];
      return;
    }
    if (has_G(SCHEME) && k >= 8) {   // G_cb: G_cb u_a - delta_ca B_b (Eq.10); kFull H_cb: H_cb u_a - delta_ca u_b
      const bool isH = SCHEME == kFull && k >= 8 + 3 * D;
      const int kk = k - 8 - (isH ? 3 * D : 0);
      const int c = kk / 3, b = kk - 3 * c;
      const real Vb = isH ? (b == 0 ? u[0] : (b == 1 ? u[1] : u[2])) : pick3<QA, real>(Qh, 5, b);
#pragma unroll
      for (int a = 0; a < D; a++) Phi[a] = own * u[a] - (a == c ? Vb : real(0));
      return;
    }
    const real B[3] = {Qh[5], Qh[6], Qh[7]};
    if (k >= 5) {   // induction: u_a B_b - B_a u_b  (kResist, kFull: - eta g_ab, g = G / tau_M ~ grad B)
      const int b = k - 5;
      const real Bb = b == 0 ? B[0] : (b == 1 ? B[1] : B[2]);
      const real ub = b == 0 ? u[0] : (b == 1 ? u[1] : u[2]);
#pragma unroll
      for (int a = 0; a < D; a++) Phi[a] = u[a] * Bb - B[a] * ub;
      if (has_G(SCHEME)) {
#pragma unroll
        for (int a = 0; a < D; a++) Phi[a] -= eta * (pick3<QA, real>(Qh, 8 + 3 * a, b) * itm);
      }
      return;
    }
    const real E = Qh[4];
    const real B2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
    const real mu = m[0] * u[0] + m[1] * u[1] + m[2] * u[2];
    const real p = (gamma - real(1)) * (E - real(0.5) * mu - real(0.5) * B2);
    const real pt = p + real(0.5) * B2;
    if (k == 4) {
      const real uB = u[0] * B[0] + u[1] * B[1] + u[2] * B[2];
#pragma unroll
      for (int a = 0; a < D; a++) Phi[a] = (E + pt) * u[a] - B[a] * uB;
      if (has_G(SCHEME)) {   // + eta (j x B)_a,  j = curl B: j_e = eps_ecb g_cb over the lattice axes c < D
        real g[3][3];
#pragma unroll
        for (int c = 0; c < 3; c++)
#pragma unroll
          for (int b = 0; b < 3; b++) g[c][b] = c < D ? Qh[8 + 3 * (c < D ? c : 0) + b] * itm : real(0);
        const real j0 = g[1][2] - g[2][1], j1 = g[2][0] - g[0][2], j2 = g[0][1] - g[1][0];
        const real jxB[3] = {j1 * B[2] - j2 * B[1], j2 * B[0] - j0 * B[2], j0 * B[1] - j1 * B[0]};
#pragma unroll
        for (int a = 0; a < D; a++) Phi[a] += eta * jxB[a];
      }
      if (SCHEME == kFull) {   // - u_b sigma_ab,  sigma = mu (h + h^T - 2/3 tr h I),  h = H / tau_M ~ grad u (A23)
        real h[3][3];
#pragma unroll
        for (int c = 0; c < 3; c++)
#pragma unroll
          for (int b = 0; b < 3; b++) h[c][b] = c < D ? Qh[8 + 3 * D + 3 * (c < D ? c : 0) + b] * itm : real(0);
        const real trh = h[0][0] + h[1][1] + h[2][2];
#pragma unroll
        for (int a = 0; a < D; a++) {
          real us = real(0);
#pragma unroll
          for (int b = 0; b < 3; b++) us += u[b] * (visc * (h[a][b] + h[b][a] - (a == b ? real(2.0 / 3.0) * trh : real(0))));
          Phi[a] -= us;
        }
      }
      return;
    }
    const int b = k - 1;   // momentum: m_b u_a + pt delta_ab - B_b B_a  (kFull: - sigma_ab)
    const real mb = b == 0 ? m[0] : (b == 1 ? m[1] : m[2]);
    const real Bb = b == 0 ? B[0] : (b == 1 ? B[1] : B[2]);
#pragma unroll
    for (int a = 0; a < D; a++) Phi[a] = mb * u[a] + (a == b ? pt : real(0)) - Bb * B[a];
    if (SCHEME == kFull) {
      real trh = real(0);
#pragma unroll
      for (int c = 0; c < D; c++) trh += Qh[8 + 3 * D + 3 * c + c] * itm;
#pragma unroll
      for (int a = 0; a < D; a++) {
        // h_ab = H_ab / tau_M (a < D), h_ba = H_ba / tau_M if b < D else 0
        const real hab = pick3<QA, real>(Qh, 8 + 3 * D + 3 * a, b) * itm;
        real hba = real(0);
#pragma unroll
        for (int c = 0; c < D; c++)
          if (b == c) hba = Qh[8 + 3 * D + 3 * c + a] * itm;
        Phi[a] -= visc * (hab + hba - (a == b ? real(2.0 / 3.0) * trh : real(0)));
      }
    }
  } else {
    if (k == 0) {
#pragma unroll
      for (int a = 0; a < D; a++) Phi[a] = c0sq * Qh[1 + a];
      return;
    }
    real u[D], B[D];
#pragma unroll
    for (int c = 0; c < D; c++) { u[c] = Qh[1 + c]; B[c] = Qh[1 + D + c]; }
    if (k >= 1 + D) {
      const int b = k - 1 - D;
      real Bb = B[0], ub = u[0];
#pragma unroll
      for (int c = 1; c < D; c++)
        if (b == c) { Bb = B[c]; ub = u[c]; }
#pragma unroll
      for (int a = 0; a < D; a++) Phi[a] = u[a] * Bb - B[a] * ub;
      return;
    }
    real B2 = real(0);
#pragma unroll
    for (int c = 0; c < D; c++) B2 += B[c] * B[c];
    const real pt = Qh[0] + real(0.5) * B2;
    const int b = k - 1;
    real Bb = B[0], ub = u[0];
#pragma unroll
    for (int c = 1; c < D; c++)
      if (b == c) { Bb = B[c]; ub = u[c]; }
#pragma unroll
    for (int a = 0; a < D; a++) Phi[a] = ub * u[a] + (a == b ? pt : real(0)) - Bb * B[a];
  }
}

// ---- Powell source row S_k / (-kappa delta) (Eq.12): (0, B, u.B, u) resp. (0, B, u) ----------
template <int SCHEME, int D, typename real, class QA>
__device__ __forceinline__ real powell_row(int k, const QA &Qv) {
  if (k == 0) return real(0);
  if (is_ideal(SCHEME)) {
    if (has_relax(SCHEME) && k >= 8) return real(0);
    if (k <= 3) return pick3<QA, real>(Qv, 5, k - 1);
    const real ir = real(1) / Qv[0];
    if (k == 4) return (Qv[1] * Qv[5] + Qv[2] * Qv[6] + Qv[3] * Qv[7]) * ir;
    return pick3<QA, real>(Qv, 1, k - 5) * ir;
  } else {
    real r = real(0);
#pragma unroll
    for (int c = 0; c < D; c++) {
      if (k == 1 + c) r = Qv[1 + D + c];
      if (k == 1 + D + c) r = Qv[1 + c];
    }
    return r;
  }
}

// ---- blended state Q^ of a cell with porosity d < 1 (Eq.13-14, A8): rho and p kept, u^ = d u + (1-d) u^B, B^ likewise -----
template <int SCHEME, int D, typename real>
__device__ __forceinline__ void solid_blend(const real *Qv, real gamma, real d, const double uS[3], const double BS[3], real *Qh) {
  const real e = real(1) - d;
  if (has_relax(SCHEME)) {      // gradient variables are not blended
#pragma unroll
    for (int l = 8; l < Vars<SCHEME, D>::K; l++) Qh[l] = Qv[l];
  }
  if (is_ideal(SCHEME)) {
    const real rho = Qv[0];
    const real ir = real(1) / rho;
    const real mu = (Qv[1] * Qv[1] + Qv[2] * Qv[2] + Qv[3] * Qv[3]) * ir;
    const real B2 = Qv[5] * Qv[5] + Qv[6] * Qv[6] + Qv[7] * Qv[7];
    const real p = (gamma - real(1)) * (Qv[4] - real(0.5) * mu - real(0.5) * B2);
    real uh2 = real(0), Bh2 = real(0);
#pragma unroll
    for (int c = 0; c < 3; c++) {
      const real uh = d * (Qv[1 + c] * ir) + e * (real)uS[c], Bh = d * Qv[5 + c] + e * (real)BS[c];
      Qh[1 + c] = rho * uh;
      Qh[5 + c] = Bh;
      uh2 += uh * uh;
      Bh2 += Bh * Bh;
    }
    Qh[0] = rho;
    Qh[4] = p / (gamma - real(1)) + real(0.5) * rho * uh2 + real(0.5) * Bh2;
  } else {
    Qh[0] = Qv[0];
#pragma unroll
    for (int c = 0; c < D; c++) {
      Qh[1 + c] = d * Qv[1 + c] + e * (real)uS[c];
      Qh[1 + D + c] = d * Qv[1 + D + c] + e * (real)BS[c];
    }
  }
}

// ---- streaming layouts -------------------------------------------------------------------
// ST_AB   two population copies; step reads src, writes dst:            g'_j(x) -> dst (x, slot j)
// ST_PP   one copy, AA pattern, layout P0 -> P1 ("pull-push"): the cell reads f_i from (x - c_i, slot i), exactly
//         the A/B pull, and writes g'_j back into the location it read for the opposite direction:
//         g'_j(x) -> (x + c_j, slot opp(j)); if x + c_j is outside a non-periodic face, -> (x, slot j).
// ST_LOC  one copy, layout P1 -> P0 (local): f_i(x) is at (x, slot opp(i)); g'_j(x) -> (x, slot j).
// In both in-place steps a cell only touches locations no other cell touches, so there is no race.
enum { ST_AB = 0, ST_PP = 1, ST_LOC = 2 };

__host__ __device__ constexpr int opp(int i) { return i == 0 ? 0 : ((i & 1) ? i + 1 : i - 1); }

// per-cell context shared by the load front ends (plain pulls / TMA-staged pulls) and finish_cell
struct CellCtx {
  int tx, k, x, y, z;
  uint32_t n;                                   // cell index (N < 2^32 is checked at create)
  bool work;                                    // active and not frozen
  bool out_xm, out_xp, out_ym, out_yp, out_zm, out_zp;   // source x - c would be outside a non-periodic face
  bool writeM;                                  // in-place modes: publish this cell's post-collision moment (see M_next)
};

// ---- where result j of a cell goes --------------------------------------------------------------------------
// own slot: A/B (base in the dst copy) and ST_LOC (base in the single copy)
template <typename real> struct StoreOwn {
  char *base;                 // address of (k, 0, cell)
  const long long *st_off;
  __device__ __forceinline__ void put(int j, real v) const { *reinterpret_cast<real *>(base + st_off[j]) = v; }
};
// ST_PP, interior tile: the location read for direction opp(j)
template <typename real> struct StorePPInterior {
  char *base;
  const long long *ld_off;
  __device__ __forceinline__ void put(int j, real v) const { *reinterpret_cast<real *>(base + ld_off[opp(j)]) = v; }
};
// ST_PP, x-edge tile of an interior row: only the thread on the face differs (wrap, or own slot when outside)
template <class L, typename real> struct StorePPEdge {
  char *base;
  const long long *ld_off, *st_off;
  bool edge_lo, on_face, wrap;
  long long wrap_adj;
  __device__ __forceinline__ void put(int j, real v) const {
    const int i = opp(j);
    long long off = ld_off[i];
    if ((L::cx(i) == 1 || L::cx(i) == -1) && on_face && ((edge_lo && L::cx(i) == 1) || (!edge_lo && L::cx(i) == -1)))
      off = wrap ? off + wrap_adj : st_off[j];
    *reinterpret_cast<real *>(base + off) = v;
  }
};
// ST_PP, general tile: full index arithmetic with wrap and outside tests
template <class L, typename real> struct StorePPGeneral {
  real *basek;                // (k, 0, cell 0)
  uint32_t ps, n;
  int x, y, z, nx, ny, nz;
  bool npx, npy, npz;
  __device__ __forceinline__ void put(int j, real v) const {
    const int i = opp(j);
    int sx = x - L::cx(i), sy = y - L::cy(i), sz = z - L::cz(i);
    bool outside = false;
    if (sx < 0) { if (npx) outside = true; else sx += nx; } else if (sx >= nx) { if (npx) outside = true; else sx -= nx; }
    if (sy < 0) { if (npy) outside = true; else sy += ny; } else if (sy >= ny) { if (npy) outside = true; else sy -= ny; }
    if (sz < 0) { if (npz) outside = true; else sz += nz; } else if (sz >= nz) { if (npz) outside = true; else sz -= nz; }
    if (outside) basek[(uint32_t)j * ps + n] = v;
    else basek[(uint32_t)i * ps + ((uint32_t)sz * ny + sy) * nx + sx] = v;
  }
};

// Slab decomposition: the plane on a HALO face of the slowest lattice axis is a ghost plane owned by the
// neighbouring slab: it is never updated here (the caller refreshes it before every step) and its cells are pulled from
// like any other in-range cell.
template <typename real, int D>
__device__ __forceinline__ bool ghost_row(const StepArgs<real> &a, int y, int z) {
  if (D < 2) return false;
  const int hc = D == 3 ? z : y, hn = D == 3 ? a.nz : a.ny;
  return (hc == 0 && a.bc[2 * (D - 1)] == BC_HALO) || (hc == hn - 1 && a.bc[2 * (D - 1) + 1] == BC_HALO);
}

// Conservative, tile-uniform test: can the sphere touch cells [x0, x0+tx_cells) of row (y, z)?
template <typename real, int D>
__device__ __forceinline__ bool sphere_may_touch(const StepArgs<real> &a, int x0, int tx_cells, int y, int z) {
  if (!a.has_sphere) return false;
  const double lo = (double)x0 - a.sph_c[0], hi = a.sph_c[0] - (double)(x0 + tx_cells - 1);
  const double dx = fmax(0.0, fmax(lo, hi));
  const double dy = D > 1 ? (double)(y + (D == 2 ? a.hoff : 0)) - a.sph_c[1] : 0.0;
  const double dz = D > 2 ? (double)(z + a.hoff) - a.sph_c[2] : 0.0;
  return dx * dx + dy * dy + dz * dz <= a.sph_touch2 * (1.0 + 1e-9) + 1e-9;
}

// frozen cell in the in-place modes (A10): its populations are f^eq of its constant state, kept in M_cur
template <int LAT, int SCHEME, typename real, class Store>
__device__ __forceinline__ void frozen_rematerialise(const StepArgs<real> &a, int k, uint32_t n, const Store &store) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q, K = Vars<SCHEME, D>::K;
  const size_t N = (size_t)a.nx * a.ny * a.nz;
  real Qf[K], Phi[3];
#pragma unroll
  for (int l = 0; l < K; l++) Qf[l] = (real)a.M_cur[(size_t)l * N + n];
  const real Qfk = pick<K, real>(Qf, k);
  flux_row<SCHEME, D, real>(k, Qf, Qfk, a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
#pragma unroll
  for (int j = 0; j < Q; j++) {
    const real cPhi = real(L::cx(j)) * Phi[0] + real(L::cy(j)) * Phi[1] + real(L::cz(j)) * Phi[2];
    store.put(j, real(L::w(j)) * (Qfk + real(L::inv_cs2) * cPhi));
  }
}

// ---- body integrals (A21) ------------------------------------------------
// What the blend hands over at a cell with d < 1, summed over the body and accumulated over steps:
//   [0..2] F = -sum dQh_m | [3..5] T = -sum r x dQh_m | [6] W = -sum dQh_E | [7..9] sum dQh_B |
//   [10..12] sum (1-d) B | [13] sum (1-d).
// Thread (cell, k) owns dQh_k; k and so the slots are uniform over the lanes of a group: they reduce their values
// and one lane adds to the accumulator (solid cells are 0.2 % of config 5; fluid tiles never get here).
// One out-of-line copy for every kernel: the lanes that are here reduce up to three values and one lane adds them.
static __device__ __noinline__ void body_add(double *body, bool solid, int s0, double v0, int s1, double v1, int s2, double v2) {
  namespace cg = cooperative_groups;
  // the lanes that are here, grouped by slot: with 16-cell tiles a warp holds two variables (two slot sets)
  const cg::coalesced_group g = cg::labeled_partition(cg::coalesced_threads(), s0);
  if (!g.any(solid)) return;
  if (!solid) v0 = v1 = v2 = 0.0;
  const double t0 = cg::reduce(g, v0, cg::plus<double>());
  const double t1 = s1 >= 0 ? cg::reduce(g, v1, cg::plus<double>()) : 0.0;       // slots are warp-uniform (k is)
  const double t2 = s2 >= 0 ? cg::reduce(g, v2, cg::plus<double>()) : 0.0;
  if (g.thread_rank() == 0) {
    atomicAdd(body + s0, t0);
    if (s1 >= 0) atomicAdd(body + s1, t1);
    if (s2 >= 0) atomicAdd(body + s2, t2);
  }
}

template <int SCHEME, int D, typename real>
__device__ __forceinline__ void body_accumulate(const StepArgs<real> &a, const CellCtx &c, int k, bool solid, double dq, double d,
                                                double Qk) {
  constexpr int nvec = is_ideal(SCHEME) ? 3 : D;
  constexpr int iB = Vars<SCHEME, D>::iB;
  int s0 = -1, s1 = -1, s2 = -1;
  double v0 = 0.0, v1 = 0.0, v2 = 0.0;
  if (k == 0) {
    s0 = 13; v0 = 1.0 - d;
  } else if (k >= 1 && k < 1 + nvec) {
    const int b = k - 1;
    const double *ref = a.has_sphere ? a.sph_c : a.body_ref;
    const double rx = (double)c.x - ref[0];
    const double ry = D > 1 ? (double)(c.y + (D == 2 ? a.hoff : 0)) - ref[1] : 0.0;
    const double rz = D > 2 ? (double)(c.z + a.hoff) - ref[2] : 0.0;
    const double F = -dq;
    // (r x F)_{b+1} += r_{b+2} F_b,  (r x F)_{b+2} -= r_{b+1} F_b   (indices mod 3)
    s0 = b; v0 = F;
    s1 = 3 + (b + 1) % 3; v1 = (b == 0 ? rz : (b == 1 ? rx : ry)) * F;
    s2 = 3 + (b + 2) % 3; v2 = -(b == 0 ? ry : (b == 1 ? rz : rx)) * F;
  } else if (is_ideal(SCHEME) && k == 4) {
    s0 = 6; v0 = -dq;
  } else if (k >= iB && k < iB + nvec) {
    s0 = 7 + (k - iB); v0 = dq;
    s1 = 10 + (k - iB); v1 = (1.0 - d) * Qk;
  }
  if (s0 >= 0) body_add(a.body, solid, s0, v0, s1, v1, s2, v2);
}

// =====================================================================================================
// How the K variable rows of a tile exchange their moments.  The threads of a tile write the K zeroth moments
// (sQ), the first moments of the B sets (sTr) and, on a zero-gradient x face, the neighbour state (sNb) for
// each other and meet at a barrier.
//   CL = false  one CTA holds all K rows: shared memory + a block barrier (`Sync`: __syncthreads or a named barrier).
//   CL = true   a 2-CTA cluster splits the rows (RESIST: K = 11 / 14 / 17 rows in one block would leave an SM with
//               one or two blocks, i.e. no other block's loads in flight while one computes): each CTA keeps a full
//               copy of the arrays, every value is written into both copies (the partner's through distributed
//               shared memory) and the barrier is the cluster's (release / acquire, so the remote writes are
//               visible).  begin() waits for the start barrier the kernel arrived at on entry: the partner CTA is
//               resident before its shared memory is written.  All remote writes precede a barrier both CTAs
//               pass, so neither can exit while the other still writes into it.
// =====================================================================================================
struct SyncBlock {
  __device__ __forceinline__ void operator()() const { __syncthreads(); }
};
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_arrive_release() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait_acquire() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// The exchange of the lean tiles of the 2-CTA cluster kernel WITHOUT a fence: on sm_100a the release half of a
// cluster barrier is a GPU-scope MEMBAR (ncu: 5.0 of 24 stall cycles per issued instruction in step_kernel_cl).  Here every
// row-thread delivers its moment into the partner CTA's copy with st.async, which signals the partner's mbarrier by byte
// count (complete_tx): the partner waits for exactly the bytes its partner's rows deliver, and the data is visible to it when
// the wait returns.  One phase per kernel (a cluster owns one tile), so the parity is always 0.
__device__ __forceinline__ uint32_t cl_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t cl_mapa(uint32_t local_addr, uint32_t peer) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(peer));
  return r;
}
__device__ __forceinline__ void cl_st_async(uint32_t remote_addr, double v, uint32_t remote_bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];" ::"r"(remote_addr),
               "l"(__double_as_longlong(v)), "r"(remote_bar)
               : "memory");
}
__device__ __forceinline__ void cl_st_async(uint32_t remote_addr, float v, uint32_t remote_bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];" ::"r"(remote_addr),
               "r"(__float_as_uint(v)), "r"(remote_bar)
               : "memory");
}
template <typename real, int W> struct ShareAsync {
  real (*sQ)[W];
  real (*sTr)[W];
  real *sNb;
  uint32_t rQ, rbar;       // shared::cluster addresses of the partner's sQ[0][0] and of its mbarrier
  unsigned long long *bar; // this CTA's mbarrier
  uint32_t expect;         // bytes the partner's rows deliver
  __device__ __forceinline__ void begin() const { cluster_wait_acquire(); }      // start barrier: the partner is resident, its mbarrier initialised
  __device__ __forceinline__ void putQ(int l, int tx, real v) const {
    sQ[l][tx] = v;
    cl_st_async(rQ + (uint32_t)((l * W + tx) * (int)sizeof(real)), v, rbar);
  }
  __device__ __forceinline__ void putTr(int, int, real) const {}      // the schemes this kernel serves take div B from G
  __device__ __forceinline__ void putNb(int, real) const {}
  __device__ __forceinline__ void sync() const {
    const uint32_t b = cl_smem_u32(bar);
    if (threadIdx.x == 0 && threadIdx.y == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b), "r"(expect) : "memory");
    __syncthreads();      // this CTA's own rows
    uint32_t ok;
    do {
      asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }" : "=r"(ok) : "r"(b) : "memory");
    } while (!ok);
  }
};

template <typename real, int W, bool CL, class Sync = SyncBlock> struct Share {
  real (*sQ)[W];
  real (*sTr)[W];
  real *sNb;
  real (*rQ)[W];      // the partner CTA's copies (CL only)
  real (*rTr)[W];
  real *rNb;
  Sync sync_;
  uint32_t rQa = 0, rbar = 0, expect = 0;      // CL with the fence-free exchange (ShareAsync): see lean()
  unsigned long long *bar = nullptr;
  // the policy of the lean tiles (interior, fluid): the fence-free exchange where the kernel set it up, else this one
  __device__ __forceinline__ auto lean() const {
    if constexpr (CL) return ShareAsync<real, W>{sQ, sTr, sNb, rQa, rbar, bar, expect};
    else return *this;
  }
  __device__ __forceinline__ void begin() const {
    if (CL) cluster_wait_acquire();
  }
  __device__ __forceinline__ void putQ(int l, int tx, real v) const {
    sQ[l][tx] = v;
    if (CL) rQ[l][tx] = v;
  }
  __device__ __forceinline__ void putTr(int j, int tx, real v) const {
    sTr[j][tx] = v;
    if (CL) rTr[j][tx] = v;
  }
  __device__ __forceinline__ void putNb(int l, real v) const {
    sNb[l] = v;
    if (CL) rNb[l] = v;
  }
  __device__ __forceinline__ void sync() const {
    if (CL) {
      cluster_arrive_release();
      cluster_wait_acquire();
    } else {
      sync_();
    }
  }
  // the same arrays seen W2 cells wide (W2 <= W): the one-cell paths of the multi-cell kernels
  template <int W2> __device__ __forceinline__ Share<real, W2, CL, Sync> narrow() const {
    return Share<real, W2, CL, Sync>{reinterpret_cast<real(*)[W2]>(&sQ[0][0]), reinterpret_cast<real(*)[W2]>(&sTr[0][0]), sNb,
                                    reinterpret_cast<real(*)[W2]>(CL ? &rQ[0][0] : nullptr),
                                    reinterpret_cast<real(*)[W2]>(CL ? &rTr[0][0] : nullptr), rNb, sync_};
  }
};

// =====================================================================================================
// Everything after the pull: boundary substitution (A9), moments exchange, div-B estimate, Powell source,
// solid blend, flux, BGK + direct injection, store (DESIGN.md §2 steps S2-S8; Eq.2-4, 8, 11-14).
// `sh` (Share) holds the exchange arrays sQ[K][TX], sTr[D*D][TX] of the threads that call this together and their
// barrier.  BND / SOLID are tile-uniform: the interior fluid tile (both
// false) is the hot path and carries no boundary predicates, no mask or sphere test.  `store` says where
// result j goes (streaming layout); STREAM only selects where Q^nb comes from.
// =====================================================================================================
template <int LAT, int SCHEME, typename real, int TX, bool BND, bool SOLID, int STREAM, class FArr, class Store, class Sh>
__device__ __forceinline__ void finish_cell(const StepArgs<real> &a, const CellCtx &c, FArr &f, const Store &store, const Sh &sh) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q;
  using V = Vars<SCHEME, D>;
  constexpr int K = V::K, iB = V::iB;
  const int tx = c.tx, k = c.k;
  const bool work = c.work;

  if constexpr (BND) {
    // A9 / PAPER.md:154: directions whose source is outside take the equilibrium of the inward neighbour's state
    const bool cell_bnd = work && (c.out_xm || c.out_xp || c.out_ym || c.out_yp || c.out_zm || c.out_zp);
    if (cell_bnd) {
      const int qx = c.out_xm ? c.x + 1 : (c.out_xp ? c.x - 1 : c.x);
      const int qy = c.out_ym ? c.y + 1 : (c.out_yp ? c.y - 1 : c.y);
      const int qz = c.out_zm ? c.z + 1 : (c.out_zp ? c.z - 1 : c.z);
      const uint32_t nb = ((uint32_t)qz * a.ny + qy) * a.nx + qx;
      real s = real(0);
      if (STREAM == ST_AB) {      // stored populations of the neighbour, index order
        const uint32_t ps = (uint32_t)a.pstride;
        const real *__restrict__ srck = a.src + (size_t)k * Q * a.pstride;
#pragma unroll
        for (int j = 0; j < Q; j++) s += srck[(uint32_t)j * ps + nb];
      } else {                    // in place the neighbour's slots are in flux: it published its moment last step
        s = (real)a.M_cur[(size_t)k * ((size_t)a.nx * a.ny * a.nz) + nb];
      }
      sh.putQ(k, tx, s);
    }
    sh.sync();
    if (cell_bnd) {
      real Qnb[K], Phi[3];
#pragma unroll
      for (int l = 0; l < K; l++) Qnb[l] = sh.sQ[l][tx];
      const real Qnbk = pick<K, real>(Qnb, k);
      flux_row<SCHEME, D, real>(k, Qnb, Qnbk, a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
#pragma unroll
      for (int i = 0; i < Q; i++) {
        const int cx = L::cx(i), cy = L::cy(i), cz = L::cz(i);
        const bool outside = (cx == 1 && c.out_xm) || (cx == -1 && c.out_xp) || (cy == 1 && c.out_ym) ||
                             (cy == -1 && c.out_yp) || (cz == 1 && c.out_zm) || (cz == -1 && c.out_zp);
        const real cPhi = real(cx) * Phi[0] + real(cy) * Phi[1] + real(cz) * Phi[2];
        if (outside) f[i] = real(L::w(i)) * (Qnbk + real(L::inv_cs2) * cPhi);
      }
    }
    sh.sync();
  }

  // S2 zeroth moment of this set (index order) and S3 this set's share of tr Pi_B
  real Qlo;
  const real Qk = moment_sum<L, real>(f, Qlo);
  sh.putQ(k, tx, Qk);
  if (!has_relax(SCHEME) && k >= iB && k < iB + D) {      // A6 (the schemes with gradient sets take div B from them)
    const int b = k - iB;   // warp-uniform
    // first moment of this B set, Pi_{a,b} = sum_i c_ia f_i: the diagonal entry is its share of tr Pi_B (A6); the
    // resistive scheme keeps all D entries, their antisymmetric part gives the current (A20)
    real m[3] = {real(0), real(0), real(0)};
    if (SCHEME == kIncres || b == 0) {
#pragma unroll
      for (int i = 0; i < Q; i++)
        if (L::cx(i) != 0) m[0] += real(L::cx(i)) * f[i];
    }
    if (D > 1 && (SCHEME == kIncres || b == 1)) {
#pragma unroll
      for (int i = 0; i < Q; i++)
        if (L::cy(i) != 0) m[1] += real(L::cy(i)) * f[i];
    }
    if (D > 2 && (SCHEME == kIncres || b == 2)) {
#pragma unroll
      for (int i = 0; i < Q; i++)
        if (L::cz(i) != 0) m[2] += real(L::cz(i)) * f[i];
    }
#pragma unroll
    for (int al = 0; al < D; al++)
      if (SCHEME == kIncres || al == b) sh.putTr(b * D + al, tx, m[al]);
  }
  sh.sync();
  if (!work) return;

  // The schemes with gradient sets (K = 11 .. 26) read the exchanged moments where a row needs them (a gradient row needs
  // 5); the others keep the K moments in registers.
  constexpr bool LAZY = has_G(SCHEME);
  const QCol<real, TX> qc{sh.sQ, tx};
  [[maybe_unused]] real Qv[LAZY ? 1 : K];
  if constexpr (!LAZY) {
#pragma unroll
    for (int l = 0; l < K; l++) Qv[l] = sh.sQ[l][tx];
  }
  real tr = real(0);
  if constexpr (!has_relax(SCHEME)) {
    tr = sh.sTr[0][tx];
#pragma unroll
    for (int b = 1; b < D; b++) tr += sh.sTr[b * D + b][tx];
  }
  // A20: current-dependent resistivity -> cell-local tau_B (6 Newton steps on tau^3 - tau0 tau^2 - c = 0 from tau0 + cbrt(c))
  real inv_tauB_cs2 = a.inv_tauB_cs2;
  real omB = real(0);
  if constexpr (SCHEME == kIncres) if (a.etaj_inv_jc2 > real(0)) {
    real a2 = real(0);
#pragma unroll
    for (int al = 0; al < D; al++)
#pragma unroll
      for (int be = al + 1; be < D; be++) {
        // N_ab = Pi_ab - Phi_{B_b,a},  Phi_{B_b,a} = u_a B_b - B_a u_b  (antisymmetric in a <-> b)
        const real phi = Qv[1 + al] * Qv[1 + D + be] - Qv[1 + D + al] * Qv[1 + be];
        const real w2 = (sh.sTr[be * D + al][tx] - phi) - (sh.sTr[al * D + be][tx] + phi);
        a2 += w2 * w2;
      }
    a2 *= real(L::inv_cs2 * L::inv_cs2);
    const real tau0 = a.tauB0;
    const real cc = (tau0 - real(0.5)) * a2 * a.etaj_inv_jc2;
    real t = tau0 + cbrt(cc);
#pragma unroll
    for (int it = 0; it < 6; it++) t = t - ((t - tau0) * t * t - cc) / (t * (real(3) * t - real(2) * tau0));
    omB = real(1) / t;
    inv_tauB_cs2 = omB * real(L::inv_cs2);
  }
  // A6: local estimate from tr Pi_B; kIdealD: from the relaxation variable, D ~ tau_M div B (Eq.7)
  real delta;
  if constexpr (SCHEME == kIdealD) delta = Qv[K - 1] * a.inv_tau_relax;
  else if constexpr (has_G(SCHEME)) {         // div B = tr g = sum_a G_aa / tau_M (only the 8 Powell rows use it)
    delta = real(0);
    if (k < 8) {
#pragma unroll
      for (int al = 0; al < D; al++) delta += qc[8 + 3 * al + al] * a.inv_tau_relax;
    }
  } else delta = -tr * inv_tauB_cs2;

  // S4 Powell source, S5 solid blend (rare: own branch so the blended copy of the state costs no registers
  // on the fluid path), S6 flux row of this variable
  real Phi[3];
  real inj;
  bool solid = false;
  if constexpr (SOLID) {
    double uS[3], BS[3];
    const real d = (real)solid_state<real, D>(a, c.x, c.y, c.z, c.n, uS, BS);
    real dq = real(0);
    if (d < real(1)) {
      real Qh[K], Qs[K];
#pragma unroll
      for (int l = 0; l < K; l++) Qs[l] = LAZY ? sh.sQ[l][tx] : Qv[LAZY ? 0 : l];
      solid_blend<SCHEME, D, real>(Qs, a.gamma, d, uS, BS, Qh);
      const real Qhk = pick<K, real>(Qh, k);
      flux_row<SCHEME, D, real>(k, Qh, Qhk, a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
      // dQh plus the Powell source scaled by the porosity d (A8)
      dq = Qhk - Qk;
      inj = dq - d * (a.kappa * delta) * powell_row<SCHEME, D, real>(k, Qs);
      if (has_relax(SCHEME) && k >= 8) inj = -Qk * a.inv_tau_relax;      // relaxation source of Eq.6, not porosity-scaled
      solid = true;
    }
    if (a.body != nullptr) body_accumulate<SCHEME, D, real>(a, c, k, solid, (double)dq, (double)d, (double)Qk);
  }
  if (!solid) {
    if constexpr (LAZY) {
      flux_row<SCHEME, D, real>(k, qc, Qk, a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
      inj = k < 8 ? -(a.kappa * delta) * powell_row<SCHEME, D, real>(k, qc) : -Qk * a.inv_tau_relax;
    } else {
      flux_row<SCHEME, D, real>(k, Qv, Qk, a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
      inj = -(a.kappa * delta) * powell_row<SCHEME, D, real>(k, Qv);
      if (has_relax(SCHEME) && k >= 8) inj = -Qk * a.inv_tau_relax;        // relaxation source of Eq.6
    }
  }
  // in place: cells next to a non-periodic face publish their post-collision moment (sum_i g'_i = Q_k + inj)
  if (STREAM != ST_AB && c.writeM) a.M_next[(size_t)k * ((size_t)a.nx * a.ny * a.nz) + c.n] = (double)(Qk + inj);

  // S7 BGK + direct injection (Collide), S8 store
  const real om = (SCHEME == kIncres && omB > real(0) && k >= iB) ? omB : a.omega[k];
  const real tauk = (SCHEME == kIncres && omB > real(0) && k >= iB) ? real(1) / omB : a.tau[k];
  const Collide<L, real> col(om, tauk, Qk, Qlo, inj, Phi);
#pragma unroll
  for (int i = 0; i < Q; i++) store.put(i, col.out(i, f[i]));
}

// =====================================================================================================
// General tile (faces, periodic wrap, mask, sphere): register pulls with per-direction predicates, then
// finish_cell with boundary and solid handling compiled in.  Used by every step kernel for the tiles that are
// not interior; the TX*K threads of the tile call it together.
// =====================================================================================================
template <int LAT, int SCHEME, typename real, int TX, int STREAM, class Sh>
__device__ __forceinline__ void general_tile(const StepArgs<real> &a, int tx, int k, int x, int y, int z, const Sh &sh) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q;
  const int nx = a.nx, ny = a.ny, nz = a.nz;
  const bool active = x < nx;
  const uint32_t ps = (uint32_t)a.pstride;
  const uint32_t n = ((uint32_t)z * ny + y) * nx + (active ? x : 0);
  const real *__restrict__ srck = a.src + (size_t)k * Q * a.pstride;
  real *__restrict__ dstk = a.dst + (size_t)k * Q * a.pstride;       // ST_AB: the other copy; in place: the same copy
  const bool npx = a.bc[0] != BC_PERIODIC, npy = D > 1 && a.bc[2] != BC_PERIODIC, npz = D > 2 && a.bc[4] != BC_PERIODIC;
  const bool x_lo = x == 0, x_hi = x == nx - 1;
  const bool y_lo = D > 1 && y == 0, y_hi = D > 1 && y == ny - 1;
  const bool z_lo = D > 2 && z == 0, z_hi = D > 2 && z == nz - 1;
  const int xm = x_lo ? nx - 1 : x - 1, xp = x_hi ? 0 : x + 1;
  const int ym = y_lo ? ny - 1 : y - 1, yp = y_hi ? 0 : y + 1;
  const int zm = z_lo ? nz - 1 : z - 1, zp = z_hi ? 0 : z + 1;
  const StoreOwn<real> own{reinterpret_cast<char *>(dstk + n), a.st_off};
  const StorePPGeneral<L, real> pp{dstk, ps, n, x, y, z, nx, ny, nz, npx, npy, npz};

  // frozen cells keep their populations: mask FROZEN or on an INFLOW face (A10)
  bool frozen = false;
  if (active) {
    frozen = (a.mask != nullptr && a.mask[n] == CELL_FROZEN) || (x_lo && a.bc[0] == BC_INFLOW) ||
             (x_hi && a.bc[1] == BC_INFLOW) || (y_lo && a.bc[2] == BC_INFLOW) || (y_hi && a.bc[3] == BC_INFLOW) ||
             (z_lo && a.bc[4] == BC_INFLOW) || (z_hi && a.bc[5] == BC_INFLOW);
    if (frozen) {
      if (STREAM == ST_AB) {
#pragma unroll
        for (int i = 0; i < Q; i++) dstk[(uint32_t)i * ps + n] = srck[(uint32_t)i * ps + n];
      } else if (STREAM == ST_PP) {
        frozen_rematerialise<LAT, SCHEME, real>(a, k, n, pp);
      } else {
        frozen_rematerialise<LAT, SCHEME, real>(a, k, n, own);
      }
    }
  }
  const bool work = active && !frozen;
  const bool out_xm = npx && x_lo, out_xp = npx && x_hi;
  const bool out_ym = npy && y_lo, out_yp = npy && y_hi;
  const bool out_zm = npz && z_lo, out_zp = npz && z_hi;

  // S1 pull: f_i(x) = g_i(x - c_i), periodic wrap; sources outside a non-periodic face are filled in finish_cell
  real f[Q];
#pragma unroll
  for (int i = 0; i < Q; i++) {
    const int cx = L::cx(i), cy = L::cy(i), cz = L::cz(i);
    const int sx = cx == 1 ? xm : (cx == -1 ? xp : x);
    const int sy = cy == 1 ? ym : (cy == -1 ? yp : y);
    const int sz = cz == 1 ? zm : (cz == -1 ? zp : z);
    const bool outside = (cx == 1 && out_xm) || (cx == -1 && out_xp) || (cy == 1 && out_ym) || (cy == -1 && out_yp) ||
                         (cz == 1 && out_zm) || (cz == -1 && out_zp);
    const uint32_t at = STREAM == ST_LOC ? (uint32_t)opp(i) * ps + n : (uint32_t)i * ps + ((uint32_t)sz * ny + sy) * nx + sx;
    f[i] = (work && !outside) ? srck[at] : real(0);
  }
  CellCtx c{tx, k, x, y, z, n, work, out_xm, out_xp, out_ym, out_yp, out_zm, out_zp, true};
  sh.begin();
  if (STREAM == ST_PP) finish_cell<LAT, SCHEME, real, TX, true, true, STREAM>(a, c, f, pp, sh);
  else finish_cell<LAT, SCHEME, real, TX, true, true, STREAM>(a, c, f, own, sh);
}

// Which tiles a launch covers: block (bx, by, bz) -> tile (bx0 + bx*bxs, y0 + by*ys, z0 + bz*zs).
struct Region {
  int bx0, bxs, y0, ys, z0, zs;
};

// =====================================================================================================
// Fused step kernel: coalesced pulls into registers (S1) + finish_cell.  STREAM: ST_AB | ST_PP | ST_LOC.
// MODE 0: one launch over all tiles; interior tiles take the lean path, x-edge tiles of interior rows the lean
//         edge path, the others general_tile().
// MODE 1: interior tiles only (no general path compiled in); MODE 2: general tiles only, over a Region.
//         (split launches were measured slower; the modes remain for register-use checks.)
// =====================================================================================================
// One TX-cell tile of row (y, z) starting at x0: classification and the three paths (interior / x-edge / general).
// Called by all TX*K threads of a block together (it contains block barriers).
template <int LAT, int SCHEME, typename real, int TX, int MODE, int STREAM, class Sh>
__device__ __forceinline__ void run_tile(const StepArgs<real> &a, const int tx, const int k, const int x0, const int y, const int z,
                                         const int sphere_only, const Sh &sh) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q;
  using V = Vars<SCHEME, D>;
  constexpr int K = V::K;
  const int x = x0 + tx;
  const int nx = a.nx, ny = a.ny, nz = a.nz;
  if (ghost_row<real, D>(a, y, z)) {
    sh.begin();      // cluster: consume the start barrier the kernel arrived at
    return;
  }
  const bool npx = a.bc[0] != BC_PERIODIC, npy = D > 1 && a.bc[2] != BC_PERIODIC, npz = D > 2 && a.bc[4] != BC_PERIODIC;

  // block-uniform classification.  Interior tile: no face, no wrap in any direction, every thread active, no
  // mask, sphere out of reach -> the lean path: one base pointer per thread plus per-direction byte offsets
  // from the constant bank, no predicates.
  const bool row_inner = (D < 2 || (y >= 1 && y <= ny - 2)) && (D < 3 || (z >= 1 && z <= nz - 2));
  const bool inner_pos = x0 >= 1 && x0 + TX <= nx - 1 && row_inner;
  const bool touched = sphere_may_touch<real, D>(a, x0, TX, y, z);
  const bool interior = inner_pos && a.mask == nullptr && !touched;
  // in place: rows next to a non-periodic y/z face publish their moments (Q^nb of the face cells, A9)
  const bool rowM = STREAM != ST_AB && ((npy && (y == 1 || y == ny - 2)) || (npz && (z == 1 || z == nz - 2)));
  if ((MODE == 1 && !interior) || (MODE == 2 && sphere_only && !(inner_pos && touched))) {
    sh.begin();
    return;
  }
  if (MODE != 2 && interior) {
    const uint32_t n = ((uint32_t)z * ny + y) * nx + x;
    char *__restrict__ pb = reinterpret_cast<char *>(const_cast<real *>(a.src) + ((size_t)k * Q * a.pstride + n));
    real f[Q];
#pragma unroll
    for (int i = 0; i < Q; i++) f[i] = *reinterpret_cast<const real *>(pb + (STREAM == ST_LOC ? a.st_off[opp(i)] : a.ld_off[i]));
    const bool writeM = STREAM != ST_AB && (rowM || (npx && (x == 1 || x == nx - 2)));
    CellCtx c{tx, k, x, y, z, n, true, false, false, false, false, false, false, writeM};
    const auto shl = sh.lean();      // cluster kernel: the fence-free exchange (ShareAsync); every other kernel: sh itself
    shl.begin();
    if (STREAM == ST_AB) {
      const StoreOwn<real> st{reinterpret_cast<char *>(a.dst + ((size_t)k * Q * a.pstride + n)), a.st_off};
      finish_cell<LAT, SCHEME, real, TX, false, false, STREAM>(a, c, f, st, shl);
    } else if (STREAM == ST_PP) {
      const StorePPInterior<real> st{pb, a.ld_off};
      finish_cell<LAT, SCHEME, real, TX, false, false, STREAM>(a, c, f, st, shl);
    } else {
      const StoreOwn<real> st{pb, a.st_off};
      finish_cell<LAT, SCHEME, real, TX, false, false, STREAM>(a, c, f, st, shl);
    }
    return;
  }
  if (MODE == 1) return;      // (never reached: MODE 1 left above)

  // x-edge tile of an otherwise interior row (no mask, sphere out of reach, not both ends in one tile): lean
  // loads for every thread; only the thread ON the face differs (A9-A11):
  //   periodic x   its c_x != 0 sources come from the other end of the row (offset +- nx);
  //   INFLOW face  it is frozen: it re-stores its own populations (in place: f^eq of its constant state);
  //   ZEROGRAD     its outside directions take f^eq of the inward neighbour's state Q^nb.  A/B: the Q values
  //                g_j(nb) are fetched one per lane together with the pulls and summed by shuffles, so the
  //                face costs no second memory round trip.  In place: Q^nb was published in M_cur.
  const bool edge_lo = x0 == 0, edge_hi = x0 + TX >= nx;
  if (TX == 32 && row_inner && a.mask == nullptr && !touched && (edge_lo != edge_hi) && nx >= 3) {
    const bool active = x < nx;
    const int xe = active ? x : nx - 1;                      // inactive tail threads shadow the last cell, store nothing
    const uint32_t n = ((uint32_t)z * ny + y) * nx + xe;
    const bool on_face = active && (edge_lo ? x == 0 : x == nx - 1);
    const int bcf = edge_lo ? a.bc[0] : a.bc[1];
    const bool frozen = on_face && bcf == BC_INFLOW;
    const bool zg = on_face && bcf == BC_ZEROGRAD;
    const bool wrap = on_face && bcf == BC_PERIODIC;
    const long long wrap_adj = (long long)nx * (long long)sizeof(real) * (edge_lo ? 1 : -1);
    char *__restrict__ pb = reinterpret_cast<char *>(const_cast<real *>(a.src) + ((size_t)k * Q * a.pstride + n));
    real f[Q];
#pragma unroll
    for (int i = 0; i < Q; i++) {
      long long off;
      if (STREAM == ST_LOC) {
        off = a.st_off[opp(i)];
      } else {
        off = (STREAM == ST_AB && frozen) ? a.st_off[i] : a.ld_off[i];
        if ((edge_lo && L::cx(i) == 1) || (!edge_lo && L::cx(i) == -1)) off += wrap ? wrap_adj : 0;   // only these cross the face
      }
      f[i] = *reinterpret_cast<const real *>(pb + off);
    }
    const bool tile_zg = bcf == BC_ZEROGRAD;                 // tile-uniform
    sh.begin();
    if (tile_zg) {
      const uint32_t nb = ((uint32_t)z * ny + y) * nx + (edge_lo ? 1 : nx - 2);
      if (STREAM == ST_AB) {
        // lane j < Q fetches g_{k,j}(nb); butterfly sum -> Q^nb_k in every lane
        real v = tx < Q ? a.src[(size_t)k * Q * a.pstride + (size_t)tx * a.pstride + nb] : real(0);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (tx == 0) sh.putNb(k, v);
      } else {
        if (tx == 0) sh.putNb(k, (real)a.M_cur[(size_t)k * ((size_t)nx * ny * nz) + nb]);
      }
      sh.sync();
      if (zg) {
        real Qnb[K], Phi[3];
#pragma unroll
        for (int l = 0; l < K; l++) Qnb[l] = sh.sNb[l];
        const real Qnbk = pick<K, real>(Qnb, k);
        flux_row<SCHEME, D, real>(k, Qnb, Qnbk, a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
#pragma unroll
        for (int i = 0; i < Q; i++) {
          if ((edge_lo && L::cx(i) == 1) || (!edge_lo && L::cx(i) == -1)) {
            const real cPhi = real(L::cx(i)) * Phi[0] + real(L::cy(i)) * Phi[1] + real(L::cz(i)) * Phi[2];
            f[i] = real(L::w(i)) * (Qnbk + real(L::inv_cs2) * cPhi);
          }
        }
      }
    }
    CellCtx c{tx, k, x, y, z, n, active && !frozen, false, false, false, false, false, false, true};
    if (STREAM == ST_AB) {
      const StoreOwn<real> st{reinterpret_cast<char *>(a.dst + ((size_t)k * Q * a.pstride + n)), a.st_off};
      if (frozen) {
#pragma unroll
        for (int i = 0; i < Q; i++) st.put(i, f[i]);
      }
      finish_cell<LAT, SCHEME, real, TX, false, false, STREAM>(a, c, f, st, sh);
    } else if (STREAM == ST_PP) {
      const StorePPEdge<L, real> st{pb, a.ld_off, a.st_off, edge_lo, on_face, wrap, wrap_adj};
      if (frozen) frozen_rematerialise<LAT, SCHEME, real>(a, k, n, st);
      finish_cell<LAT, SCHEME, real, TX, false, false, STREAM>(a, c, f, st, sh);
    } else {
      const StoreOwn<real> st{pb, a.st_off};
      if (frozen) frozen_rematerialise<LAT, SCHEME, real>(a, k, n, st);
      finish_cell<LAT, SCHEME, real, TX, false, false, STREAM>(a, c, f, st, sh);
    }
    return;
  }
  general_tile<LAT, SCHEME, real, TX, STREAM>(a, tx, k, x, y, z, sh);
}

// Programmatic dependent launch (lbmhd_ops.cuh, launch_pdl): a step kernel launched with the stream-serialisation attribute may
// be scheduled while the previous step's last blocks are still running.  Every block first lets ITS dependent grid go
// (`launch_dependents`: the next step is released once all blocks of this one have started, so its blocks take the slots
// this step's blocks free), then waits until the grid it depends on has completed and its stores are visible (`wait`), before
// its first global access.  Launched without the attribute both instructions do nothing.
__device__ __forceinline__ void pdl_enter() {
  asm volatile("griddepcontrol.launch_dependents;");
  asm volatile("griddepcontrol.wait;" ::: "memory");
}

template <int LAT, int SCHEME, typename real, int TX, int MINB, int MODE, int STREAM>
__global__ void __launch_bounds__(TX * Vars<SCHEME, Lattice<LAT>::D>::K, MINB)
step_kernel(const __grid_constant__ StepArgs<real> a, const Region r, const int sphere_only) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, K = Vars<SCHEME, D>::K;
  pdl_enter();
  __shared__ real sQ[K][TX];
  __shared__ real sTr[D * D][TX];
  __shared__ real sNb[K];
  const Share<real, TX, false> sh{sQ, sTr, sNb, nullptr, nullptr, nullptr, SyncBlock{}};
  run_tile<LAT, SCHEME, real, TX, MODE, STREAM>(a, threadIdx.x, threadIdx.y, (r.bx0 + (int)blockIdx.x * r.bxs) * TX,
                                                r.y0 + (int)blockIdx.y * r.ys + (D == 2 ? a.row0 : 0),
                                                r.z0 + (int)blockIdx.z * r.zs + (D == 3 ? a.row0 : 0), sphere_only, sh);
}

// The same step with the K rows of a tile split over a 2-CTA cluster (Share<.., CL = true>): CTA `rank` owns rows
// rank*KH .. rank*KH + KH - 1 (KH = ceil(K/2)); for odd K the last warp of CTA 1 has no row and exits at once (exited
// threads count as arrived at the cluster barrier).  grid.x = 2 * tiles_x.
template <int LAT, int SCHEME, typename real, int MINB, int STREAM>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(32 * ((Vars<SCHEME, Lattice<LAT>::D>::K + 1) / 2), MINB)
step_kernel_cl(const __grid_constant__ StepArgs<real> a) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, K = Vars<SCHEME, D>::K, KH = (K + 1) / 2;
  __shared__ real sQ[K][32];
  __shared__ real sTr[D * D][32];
  __shared__ real sNb[K];
  __shared__ __align__(8) unsigned long long mbar;      // arrival of the partner's moments on the lean tiles (ShareAsync)
  static_assert(has_relax(SCHEME), "the fence-free exchange carries the zeroth moments only");
  const unsigned rank = blockIdx.x & 1u;
  const int k = (int)rank * KH + (int)threadIdx.y;
  if (k >= K) return;
  if (threadIdx.x == 0 && threadIdx.y == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(cl_smem_u32(&mbar)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  cluster_arrive_relaxed();      // start barrier; begin() waits for it: the partner is resident and its mbarrier initialised
  namespace cg = cooperative_groups;
  cg::cluster_group cl = cg::this_cluster();
  Share<real, 32, true> sh{sQ, sTr, sNb, cl.map_shared_rank(sQ, rank ^ 1u), cl.map_shared_rank(sTr, rank ^ 1u),
                           cl.map_shared_rank(sNb, rank ^ 1u), SyncBlock{}};
  sh.rQa = cl_mapa(cl_smem_u32(&sQ[0][0]), rank ^ 1u);
  sh.rbar = cl_mapa(cl_smem_u32(&mbar), rank ^ 1u);
  sh.bar = &mbar;
  sh.expect = (uint32_t)((rank == 0 ? K - KH : KH) * 32 * (int)sizeof(real));      // the partner's rows, 32 cells each
  run_tile<LAT, SCHEME, real, 32, 0, STREAM>(a, threadIdx.x, k, (int)(blockIdx.x >> 1) * 32, (int)blockIdx.y + (D == 2 ? a.row0 : 0),
                                             (int)blockIdx.z + (D == 3 ? a.row0 : 0), 0, sh);
}

// =====================================================================================================
// Several adjacent cells per thread.  With one cell per thread a warp moves 32*sizeof(real)
// bytes per load: 128 bytes in fp32, and only Q loads are in flight per thread, so the short lattices (D3Q7,
// D2Q5, D1Q3) and fp32 run out of bytes in flight long before the SM runs out of warps (measured: fp32
// D3Q19 4.9 TB/s, fp64 D3Q7 5.4, fp32 D3Q7 4.5 with one cell per thread).  Here a block owns 32*NC x-cells
// x K sets with the same 32 x K threads; thread tx holds cells x0 + NC tx .. x0 + NC tx + NC - 1: one
// NC-wide vector load (8 or 16 bytes) per direction without x-shift and one vector store per direction, NC
// scalar loads where the x-shift breaks the vector alignment.  Interior tiles only; every other tile is
// handed to run_tile() in 32-cell pieces.  Needs nx % NC == 0 (vector alignment of every row).
// =====================================================================================================
template <typename real, int NC> __device__ __forceinline__ void ldv(const char *p, real (&v)[NC]) {
  static_assert(NC == 2 || (NC * sizeof(real)) % 16 == 0, "vector width");
  if constexpr (NC * sizeof(real) == 8) {
    const float2 t = *reinterpret_cast<const float2 *>(p);
    v[0] = t.x; v[1] = t.y;
  } else if constexpr (sizeof(real) == 4) {
#pragma unroll
    for (int j = 0; j < NC / 4; j++) {
      const float4 t = *reinterpret_cast<const float4 *>(p + 16 * j);
      v[4 * j] = t.x; v[4 * j + 1] = t.y; v[4 * j + 2] = t.z; v[4 * j + 3] = t.w;
    }
  } else {
#pragma unroll
    for (int j = 0; j < NC / 2; j++) {
      const double2 t = *reinterpret_cast<const double2 *>(p + 16 * j);
      v[2 * j] = t.x; v[2 * j + 1] = t.y;
    }
  }
}
template <typename real, int NC> __device__ __forceinline__ void stv(char *p, const real (&v)[NC]) {
  if constexpr (NC * sizeof(real) == 8) {
    *reinterpret_cast<float2 *>(p) = make_float2(v[0], v[1]);
  } else if constexpr (sizeof(real) == 4) {
#pragma unroll
    for (int j = 0; j < NC / 4; j++) *reinterpret_cast<float4 *>(p + 16 * j) = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
  } else {
#pragma unroll
    for (int j = 0; j < NC / 2; j++) *reinterpret_cast<double2 *>(p + 16 * j) = make_double2(v[2 * j], v[2 * j + 1]);
  }
}

template <typename real, int NC> struct StoreMultiOwn {
  char *base;
  const long long *st_off;
  __device__ __forceinline__ void put(int j, const real (&v)[NC]) const { stv<real, NC>(base + st_off[j], v); }
};
// EDGE (step_kernel_multi<.., EDGE = true> only): `edge` = 1 / 2 when the tile holds the cell ON the x = 0 / x = nx - 1 face
// (lane 0's first cell / lane 31's last cell): its pushes across the face go to the other end of the row (periodic) or stay in
// the cell's own slot j; 0 for a tile that is interior in x.
template <class L, typename real, int NC, bool EDGE = false> struct StoreMultiPP {
  char *base;
  const long long *ld_off;
  int tx;
  const long long *st_off;      // EDGE only
  int edge;                     // EDGE only
  bool wrap;                    // EDGE only: periodic x
  long long wrap_adj;           // EDGE only: +- nx * sizeof(real)
  // fp32: a direction with an x-shift lands one cell beside the thread's aligned NC-vector.  Scalar stores there half-fill
  // 32-byte sectors (ncu: +14 % DRAM write bytes for fp32 in place).  Instead the value that crosses into the
  // neighbouring lane's vector travels by shuffle and every lane writes its own aligned vector; only the two ends of the
  // tile (lane 0 / lane 31) still store scalars.  All 32 lanes of the warp call put() together.
  static constexpr bool SHUFFLE = sizeof(real) == 4;
  // where the value of the cell at the low (c = 0 of lane 0) / high (c = NC - 1 of lane 31) end of the tile goes
  __device__ __forceinline__ char *end_target(int j, char *plain, int c, bool low_end) const {
    if constexpr (EDGE) {
      if (edge == (low_end ? 1 : 2)) return wrap ? plain + wrap_adj : base + st_off[j] + (long long)(c * sizeof(real));
    }
    return plain;
  }
  __device__ __forceinline__ void put(int j, const real (&v)[NC]) const {
    const int i = opp(j);
    if (L::cx(i) == 0) {
      stv<real, NC>(base + ld_off[i], v);
    } else if (!SHUFFLE) {
#pragma unroll
      for (int c = 0; c < NC; c++) {
        char *t = base + ld_off[i] + (long long)(c * sizeof(real));
        if (EDGE && c == 0 && L::cx(i) > 0 && tx == 0) t = end_target(j, t, 0, true);
        if (EDGE && c == NC - 1 && L::cx(i) < 0 && tx == 31) t = end_target(j, t, NC - 1, false);
        *reinterpret_cast<real *>(t) = v[c];
      }
    } else if (L::cx(i) < 0) {      // c_jx = +1: cell c goes to x + 1; the own vector is [left lane's last, v[0..NC-2]]
      char *a0 = base + ld_off[i];                       // where v[0] goes: one element right of the vector start
      const real left = __shfl_up_sync(0xffffffffu, v[NC - 1], 1);
      real w[NC];
      w[0] = left;
#pragma unroll
      for (int c = 1; c < NC; c++) w[c] = v[c - 1];
      if (tx > 0) {
        stv<real, NC>(a0 - (long long)sizeof(real), w);
      } else {
#pragma unroll
        for (int c = 0; c < NC - 1; c++) *reinterpret_cast<real *>(a0 + (long long)(c * sizeof(real))) = v[c];
      }
      if (tx == 31) *reinterpret_cast<real *>(end_target(j, a0 + (long long)((NC - 1) * sizeof(real)), NC - 1, false)) = v[NC - 1];
    } else {                        // c_jx = -1: cell c goes to x - 1; the own vector is [v[1..NC-1], right lane's first]
      char *a0 = base + ld_off[i];                       // where v[0] goes: one element left of the vector start
      const real right = __shfl_down_sync(0xffffffffu, v[0], 1);
      real w[NC];
#pragma unroll
      for (int c = 0; c < NC - 1; c++) w[c] = v[c + 1];
      w[NC - 1] = right;
      if (tx < 31) {
        stv<real, NC>(a0 + (long long)sizeof(real), w);
      } else {
#pragma unroll
        for (int c = 1; c < NC; c++) *reinterpret_cast<real *>(a0 + (long long)(c * sizeof(real))) = v[c];
      }
      if (tx == 0) *reinterpret_cast<real *>(end_target(j, a0, 0, true)) = v[0];
    }
  }
};

// Which cells of a multi-cell tile publish their post-collision moment (in-place modes, A9): every cell of a row next to a
// non-periodic y / z face (`row`), and the two cells at each end of a row whose x faces are not periodic.  `any`, `row`, `edge`
// and `npx` are block-uniform; `any` is false on the interior tiles of interior rows.
struct PubM {
  bool any, row, npx;
  int edge;      // EDGE tiles: 1 = the tile starts at x = 0, 2 = it ends at nx, 0 = neither
  int x, nx;     // first cell of this thread
};

// S2-S8 of NC fluid cells of an interior tile (no boundary, no solid, constant eta).  sQ / sTr rows are laid out
// [c][32] (cell c of lane tx at c*32 + tx): conflict-free scalar accesses.
// pass[c] (EDGE tiles only): cell c is a frozen face cell whose f already holds what it keeps / emits (A10): unchanged.
template <int LAT, int SCHEME, typename real, int NC, int STREAM, bool EDGE = false, class Store>
__device__ __forceinline__ void finish_multi(const StepArgs<real> &a, int tx, int k, uint32_t n, const PubM pm,
                                             const bool (&pass)[NC], real (&f)[NC][Lattice<LAT>::Q], const Store &store,
                                             real (*sQ)[32 * NC], real (*sTr)[32 * NC]) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q;
  using V = Vars<SCHEME, D>;
  constexpr int K = V::K, iB = V::iB;
  constexpr bool use_tr = !has_relax(SCHEME);       // A6; the schemes with gradient sets take div B from them
  real Qk[NC], Qlo[NC];
#pragma unroll
  for (int c = 0; c < NC; c++) {
    const real s = moment_sum<L, real>(f[c], Qlo[c]);
    Qk[c] = s;
    sQ[k][c * 32 + tx] = s;
  }
  if (use_tr && k >= iB && k < iB + D) {
    const int b = k - iB;
#pragma unroll
    for (int c = 0; c < NC; c++) {
      real t = real(0);
#pragma unroll
      for (int i = 0; i < Q; i++) {
        const int cb = lat_c<L>(i, 0) * (b == 0) + lat_c<L>(i, 1) * (b == 1) + lat_c<L>(i, 2) * (b == 2);
        if (lat_c<L>(i, 0) != 0 || lat_c<L>(i, 1) != 0 || lat_c<L>(i, 2) != 0) t += real(cb) * f[c][i];
      }
      sTr[b * D + b][c * 32 + tx] = t;
    }
  }
  __syncthreads();
  const real om = a.omega[k];
  real injv[NC], P[NC][3];
  // The flux / source code of the NC cells, with the row either a compile-time constant (one copy of the code per row, chosen
  // by dispatch_row: no selects, no unused terms, but K times the code) or the run-time k.  Measured on B200:
  // the constant-row form pays where the kernel is bound by instruction issue (fp32; fp64 on the short lattices; the 20 / 26
  // sets of FULL: +2 .. +6 %) and costs ~1 % where it is at the HBM roof (fp64 D3Q19 / D2Q9 with up to 17 sets); fp32 D3Q7 loses
  // to spills (0.75 -> 0.70).
  constexpr bool ROWCONST = sizeof(real) == 8 ? (Q <= 7 || K >= 20) : Q != 7;
  const auto cells = [&](auto kc) {
    const int KC = row_of(kc);      // == k
#pragma unroll
    for (int c = 0; c < NC; c++) {
      constexpr bool LAZY = has_G(SCHEME);      // read the exchanged moments where a row needs them (see finish_cell)
      const QCol<real, 32 * NC> qc{sQ, c * 32 + tx};
      [[maybe_unused]] real Qv[LAZY ? 1 : K];
      if constexpr (!LAZY) {
#pragma unroll
        for (int l = 0; l < K; l++) Qv[l] = sQ[l][c * 32 + tx];
      }
      real delta;
      if constexpr (SCHEME == kIdealD) {
        delta = Qv[K - 1] * a.inv_tau_relax;
      } else if constexpr (has_G(SCHEME)) {
        delta = real(0);
        if (KC < 8) {
#pragma unroll
          for (int al = 0; al < D; al++) delta += qc[8 + 3 * al + al] * a.inv_tau_relax;
        }
      } else {
        real tr = sTr[0][c * 32 + tx];
#pragma unroll
        for (int b = 1; b < D; b++) tr += sTr[b * D + b][c * 32 + tx];
        delta = -tr * a.inv_tauB_cs2;
      }
      real Phi[3];
      real inj;
      if constexpr (LAZY) {
        flux_row<SCHEME, D, real>(KC, qc, Qk[c], a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
        inj = KC < 8 ? -(a.kappa * delta) * powell_row<SCHEME, D, real>(KC, qc) : -Qk[c] * a.inv_tau_relax;
      } else {
        flux_row<SCHEME, D, real>(KC, Qv, Qk[c], a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
        inj = -(a.kappa * delta) * powell_row<SCHEME, D, real>(KC, Qv);
        if (has_relax(SCHEME) && KC >= 8) inj = -Qk[c] * a.inv_tau_relax;      // relaxation source of Eq.6
      }
      injv[c] = inj;
      P[c][0] = Phi[0]; P[c][1] = Phi[1]; P[c][2] = Phi[2];
    }
  };
  if constexpr (ROWCONST) dispatch_row<0, K>(k, cells);
  else cells(k);
  // in place: the cells next to a non-periodic face publish their post-collision moment (A9).  `anyM` is block-uniform and false
  // on the interior tiles of interior rows, which then pay one uniform branch for all of this.
  if (STREAM != ST_AB && pm.any) {
    auto put = [&](int c) { a.M_next[(size_t)k * ((size_t)a.nx * a.ny * a.nz) + n + c] = (double)(Qk[c] + injv[c]); };
    if (pm.row) {
#pragma unroll
      for (int c = 0; c < NC; c++)
        if (!(EDGE && pass[c])) put(c);
    } else if (EDGE) {      // cells x = 0, 1 are the first two of lane 0 in the tile at x = 0; x = nx - 2, nx - 1 the last two of lane 31
      if (pm.npx && pm.edge == 1 && tx == 0) {
        if (!pass[0]) put(0);
        put(1);
      } else if (pm.npx && pm.edge == 2 && tx == 31) {
        put(NC - 2);
        if (!pass[NC - 1]) put(NC - 1);
      }
    } else {
#pragma unroll
      for (int c = 0; c < NC; c++)
        if (pm.x + c == 1 || pm.x + c == pm.nx - 2) put(c);
    }
  }
  Collide<L, real> col[NC];
#pragma unroll
  for (int c = 0; c < NC; c++) {
    col[c] = Collide<L, real>(om, a.tau[k], Qk[c], Qlo[c], injv[c], P[c]);
    if (EDGE && pass[c]) col[c].identity();
  }
#pragma unroll
  for (int i = 0; i < Q; i++) {
    real out[NC];
#pragma unroll
    for (int c = 0; c < NC; c++) out[c] = col[c].out(i, f[c][i]);
    store.put(i, out);
  }
}

// Pulls of a multi-cell tile that holds the cell ON an x face of an otherwise interior row (no mask, sphere out of reach).
// Only the face cell (first cell of lane 0 in the tile at x = 0, last cell of lane 31 in the tile that ends at nx) differs
// from the interior tile (A9-A11), as in the 32-cell x-edge path of run_tile():
//   periodic x   its pulls across the face come from the other end of the row (its in-place pushes go there: StoreMultiPP);
//   ZEROGRAD     those pulls are replaced by f^eq of the inward neighbour's state Q^nb (A/B: its Q stored populations fetched
//                one per lane and summed by shuffles; in place: published in M_cur), exchanged through sNb: one more barrier;
//   INFLOW       the cell is frozen: f takes what it holds (A/B: its own stored populations; in place: f^eq of its constant
//                state in M_cur) and finish_multi passes it through unchanged.
template <int LAT, int SCHEME, typename real, int NC, int STREAM>
__device__ __forceinline__ void edge_multi_pull(const StepArgs<real> &a, const int tx, const int k, char *__restrict__ pb, const int y, const int z,
                                                const bool edge_lo, real (&f)[NC][Lattice<LAT>::Q], real *sNb) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q;
  constexpr int K = Vars<SCHEME, D>::K;
  const int nx = a.nx, ny = a.ny, nz = a.nz;
  const int bcf = edge_lo ? a.bc[0] : a.bc[1];
  const bool frozen = bcf == BC_INFLOW, zg = bcf == BC_ZEROGRAD, wrap = bcf == BC_PERIODIC;      // tile-uniform
  const bool face_thread = edge_lo ? tx == 0 : tx == 31;
  const long long wrap_adj = (long long)nx * (long long)sizeof(real) * (edge_lo ? 1 : -1);
#pragma unroll
  for (int i = 0; i < Q; i++) {
    if (STREAM == ST_LOC || L::cx(i) == 0) {
      real v[NC];
      ldv<real, NC>(pb + (STREAM == ST_LOC ? a.st_off[opp(i)] : a.ld_off[i]), v);
#pragma unroll
      for (int c = 0; c < NC; c++) f[c][i] = v[c];
    } else {
#pragma unroll
      for (int c = 0; c < NC; c++) {
        long long off = a.ld_off[i] + (long long)(c * sizeof(real));
        // the pull of the face cell that crosses the face: c_ix = +1 at x = 0 (first cell), c_ix = -1 at x = nx - 1 (last cell)
        const bool cross = face_thread && ((c == 0 && L::cx(i) > 0 && edge_lo) || (c == NC - 1 && L::cx(i) < 0 && !edge_lo));
        if (cross && wrap) off += wrap_adj;
        f[c][i] = (cross && !wrap) ? real(0) : *reinterpret_cast<const real *>(pb + off);
      }
    }
  }
  const uint32_t nrow = ((uint32_t)z * ny + y) * nx;
  if (frozen && face_thread) {
    const int cf = edge_lo ? 0 : NC - 1;
    if (STREAM == ST_AB) {      // the face cell's own stored populations
#pragma unroll
      for (int i = 0; i < Q; i++) {
        const real own = *reinterpret_cast<const real *>(pb + a.st_off[i] + (long long)(cf * sizeof(real)));
        if (edge_lo) f[0][i] = own;
        else f[NC - 1][i] = own;
      }
    } else {                    // in place its slots are in flux: f^eq of its constant state
      const size_t N = (size_t)nx * ny * nz;
      const uint32_t nface = nrow + (edge_lo ? 0 : nx - 1);
      real Qf[K], Phi[3];
#pragma unroll
      for (int l = 0; l < K; l++) Qf[l] = (real)a.M_cur[(size_t)l * N + nface];
      const real Qfk = pick<K, real>(Qf, k);
      flux_row<SCHEME, D, real>(k, Qf, Qfk, a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
#pragma unroll
      for (int i = 0; i < Q; i++) {
        const real cPhi = real(L::cx(i)) * Phi[0] + real(L::cy(i)) * Phi[1] + real(L::cz(i)) * Phi[2];
        const real fe = real(L::w(i)) * (Qfk + real(L::inv_cs2) * cPhi);
        if (edge_lo) f[0][i] = fe;
        else f[NC - 1][i] = fe;
      }
    }
  }
  if (zg) {
    const uint32_t nb = nrow + (edge_lo ? 1 : nx - 2);
    if (STREAM == ST_AB) {      // lane j < Q fetches g_{k,j}(nb); butterfly sum -> Q^nb_k in every lane
      real v = tx < Q ? a.src[(size_t)k * Q * a.pstride + (size_t)tx * a.pstride + nb] : real(0);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      if (tx == 0) sNb[k] = v;
    } else {
      if (tx == 0) sNb[k] = (real)a.M_cur[(size_t)k * ((size_t)nx * ny * nz) + nb];
    }
    __syncthreads();
    if (face_thread) {
      real Qnb[K], Phi[3];
#pragma unroll
      for (int l = 0; l < K; l++) Qnb[l] = sNb[l];
      const real Qnbk = pick<K, real>(Qnb, k);
      flux_row<SCHEME, D, real>(k, Qnb, Qnbk, a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
#pragma unroll
      for (int i = 0; i < Q; i++) {
        if (L::cx(i) != 0) {
          const real cPhi = real(L::cx(i)) * Phi[0] + real(L::cy(i)) * Phi[1] + real(L::cz(i)) * Phi[2];
          const real fe = real(L::w(i)) * (Qnbk + real(L::inv_cs2) * cPhi);
          if (L::cx(i) > 0 && edge_lo) f[0][i] = fe;
          if (L::cx(i) < 0 && !edge_lo) f[NC - 1][i] = fe;
        }
      }
    }
  }
}

// Row layout.  EDGE = false (any nx that is a multiple of the vector width): [32-cell edge tile][nmulti tiles of 32*NC cells]
// [rest in 32-cell tiles], one block each, so that the multi-cell tiles are all interior in x; blocks 0..nmulti-1 are those
// tiles, block nmulti the first edge tile; xbase = 32.  EDGE = true (nx a multiple of the tile width W = 32 NC, at least two
// tiles; xbase = 0): nmulti = nx / W multi-cell tiles cover the whole row, the first and the last hold the face cells
// (edge_multi_pull).  EDGE is a template parameter so that the kernels of the lattices / precisions where it does not pay
// are compiled exactly as without it.
template <int LAT, int SCHEME, typename real, int NC, int MINB, int STREAM, bool EDGE>
__global__ void __launch_bounds__(32 * Vars<SCHEME, Lattice<LAT>::D>::K, MINB)
step_kernel_multi(const __grid_constant__ StepArgs<real> a, const int nmulti, const int xbase) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q;
  using V = Vars<SCHEME, D>;
  constexpr int K = V::K, W = 32 * NC;
  __shared__ real sQ[K][W];
  __shared__ real sTr[D * D][W];
  __shared__ real sNb[K];
  const int tx = threadIdx.x, k = threadIdx.y;
  const int nx = a.nx, ny = a.ny, nz = a.nz;
  const int y = (int)blockIdx.y + (D == 2 ? a.row0 : 0), z = (int)blockIdx.z + (D == 3 ? a.row0 : 0);
  pdl_enter();
  if (ghost_row<real, D>(a, y, z)) return;
  const Share<real, 32, false> sh32{reinterpret_cast<real(*)[32]>(&sQ[0][0]), reinterpret_cast<real(*)[32]>(&sTr[0][0]), sNb,
                                    nullptr, nullptr, nullptr, SyncBlock{}};
  if ((int)blockIdx.x >= nmulti) {
    const int t = (int)blockIdx.x - nmulti;
    run_tile<LAT, SCHEME, real, 32, 0, STREAM>(a, tx, k, t == 0 ? 0 : 32 + W * nmulti + 32 * (t - 1), y, z, 0, sh32);
    return;
  }
  const int x0 = xbase + (int)blockIdx.x * W;
  const bool npx = a.bc[0] != BC_PERIODIC, npy = D > 1 && a.bc[2] != BC_PERIODIC, npz = D > 2 && a.bc[4] != BC_PERIODIC;
  const bool row_inner = (D < 2 || (y >= 1 && y <= ny - 2)) && (D < 3 || (z >= 1 && z <= nz - 2));
  const int edge = !EDGE ? 0 : (x0 == 0 ? 1 : (x0 + W >= nx ? 2 : 0));
  const bool lean = (EDGE || (x0 >= 1 && x0 + W <= nx - 1)) && row_inner && a.mask == nullptr && !sphere_may_touch<real, D>(a, x0, W, y, z);
  if (lean) {
    const int x = x0 + NC * tx;
    const uint32_t n = ((uint32_t)z * ny + y) * nx + x;
    char *__restrict__ pb = reinterpret_cast<char *>(const_cast<real *>(a.src) + ((size_t)k * Q * a.pstride + n));
    real f[NC][Q];
    if (!EDGE || edge == 0) {
#pragma unroll
      for (int i = 0; i < Q; i++) {
        if (STREAM == ST_LOC || L::cx(i) == 0) {
          real v[NC];
          ldv<real, NC>(pb + (STREAM == ST_LOC ? a.st_off[opp(i)] : a.ld_off[i]), v);
#pragma unroll
          for (int c = 0; c < NC; c++) f[c][i] = v[c];
        } else {
#pragma unroll
          for (int c = 0; c < NC; c++) f[c][i] = *reinterpret_cast<const real *>(pb + a.ld_off[i] + (long long)(c * sizeof(real)));
        }
      }
    } else {
      if constexpr (EDGE) edge_multi_pull<LAT, SCHEME, real, NC, STREAM>(a, tx, k, pb, y, z, edge == 1, f, sNb);
    }
    const bool rowM = STREAM != ST_AB && ((npy && (y == 1 || y == ny - 2)) || (npz && (z == 1 || z == nz - 2)));
    const bool frozen_face = EDGE && edge != 0 && (edge == 1 ? a.bc[0] : a.bc[1]) == BC_INFLOW;
    // block-uniform: does the tile hold a cell that publishes (x <= 1 or x >= nx - 2 on a non-periodic axis, or a row next to a face)
    const bool anyM = STREAM != ST_AB && (rowM || (npx && (x0 <= 1 || x0 + W >= nx - 1)));
    const PubM pm{anyM, rowM, npx, edge, x, nx};
    bool pass[NC];
#pragma unroll
    for (int c = 0; c < NC; c++) {
      // EDGE: the frozen face cell goes through unchanged and publishes nothing (its state is constant); the face cell of a
      // zero-gradient face publishes its moment like its neighbour does (every cell of an x-edge tile does in run_tile)
      pass[c] = frozen_face && ((edge == 1 && tx == 0 && c == 0) || (edge == 2 && tx == 31 && c == NC - 1));
    }
    if (STREAM == ST_AB) {
      const StoreMultiOwn<real, NC> st{reinterpret_cast<char *>(a.dst + ((size_t)k * Q * a.pstride + n)), a.st_off};
      finish_multi<LAT, SCHEME, real, NC, STREAM, EDGE>(a, tx, k, n, pm, pass, f, st, sQ, sTr);
    } else if (STREAM == ST_PP) {
      const StoreMultiPP<L, real, NC, EDGE> st{pb, a.ld_off, tx, a.st_off, edge, !npx,
                                               (long long)nx * (long long)sizeof(real) * (edge == 1 ? 1 : -1)};
      finish_multi<LAT, SCHEME, real, NC, STREAM, EDGE>(a, tx, k, n, pm, pass, f, st, sQ, sTr);
    } else {
      const StoreMultiOwn<real, NC> st{pb, a.st_off};
      finish_multi<LAT, SCHEME, real, NC, STREAM, EDGE>(a, tx, k, n, pm, pass, f, st, sQ, sTr);
    }
    return;
  }
  // anything else: the NC 32-cell pieces through the one-cell paths (they share sQ / sTr columns 0..31)
#pragma unroll 1
  for (int s = 0; s < NC; s++) {
    if (s) __syncthreads();
    if (x0 + 32 * s < nx) run_tile<LAT, SCHEME, real, 32, 0, STREAM>(a, tx, k, x0 + 32 * s, y, z, 0, sh32);
  }
}

// =====================================================================================================
// One thread per CELL on the short lattices: D2Q5 / D3Q7 / D1Q3 carry K*Q = 40 / 56 / 24 populations per
// cell, which fit one thread's registers in both precisions, so the mapping north_star names applies: the flux, the Powell
// source and the primitives (1/rho, u, p_tot, u.B) are evaluated ONCE per cell and shared by the K variable sets in registers
// (the paper's CSE lesson), with no shared memory and no barrier.  With one thread per (cell, variable)
// those lattices were bound by instruction issue (ncu: ~230 warp instructions per (cell, variable), K-fold repeated flux
// arithmetic).  A block keeps the 32 x K thread shape of the other kernels and owns RY = 32 K / WX rows of WX cells; each warp
// is 32 consecutive x of one row, so every access is a coalesced row segment of one plane.  Interior fluid tiles only:
// everything else (faces, wrap, mask, sphere, the 32-cell end pieces of a row) goes through run_tile() piece by piece.
// =====================================================================================================
template <int LAT, int SCHEME, typename real, int WX, int MINB, int STREAM>
__global__ void __launch_bounds__(32 * Vars<SCHEME, Lattice<LAT>::D>::K, MINB)
step_kernel_cell(const __grid_constant__ StepArgs<real> a, const int ncell) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q;
  using V = Vars<SCHEME, D>;
  constexpr int K = V::K, iB = V::iB, RY = 32 * K / WX;
  static_assert((32 * K) % WX == 0 && WX % 32 == 0 && (D > 1 || RY == 1), "tile shape");
  __shared__ real sQ[K][32];
  __shared__ real sTr[D * D][32];
  __shared__ real sNb[K];
  const Share<real, 32, false> sh32{sQ, sTr, sNb, nullptr, nullptr, nullptr, SyncBlock{}};
  const int tx = threadIdx.x, k = threadIdx.y;
  const int nx = a.nx, ny = a.ny, nz = a.nz;
  const int y0 = D == 1 ? 0 : (int)blockIdx.y * RY + (D == 2 ? a.row0 : 0);
  const int yend = D == 1 ? 1 : (D == 2 ? a.row1 : ny);
  const int z = D == 3 ? (int)blockIdx.z + a.row0 : 0;
  if ((int)blockIdx.x >= ncell) {      // 32-cell pieces: the tile at the x = 0 end and what follows the cell tiles
    const int t = (int)blockIdx.x - ncell;
    const int x0 = t == 0 ? 0 : 32 + WX * ncell + 32 * (t - 1);
#pragma unroll 1
    for (int r = 0; r < RY; r++) {
      if (y0 + r >= yend) break;
      if (r) __syncthreads();
      run_tile<LAT, SCHEME, real, 32, 0, STREAM>(a, tx, k, x0, y0 + r, z, 0, sh32);
    }
    return;
  }
  const int x0 = 32 + (int)blockIdx.x * WX;
  const bool npx = a.bc[0] != BC_PERIODIC, npy = D > 1 && a.bc[2] != BC_PERIODIC, npz = D > 2 && a.bc[4] != BC_PERIODIC;
  bool fast = a.mask == nullptr && x0 + WX <= nx - 1 && (D < 2 || (y0 >= 1 && y0 + RY - 1 <= ny - 2 && y0 + RY <= yend)) &&
              (D < 3 || (z >= 1 && z <= nz - 2));
  if (fast && a.has_sphere) {
#pragma unroll 1
    for (int r = 0; r < RY; r++) fast = fast && !sphere_may_touch<real, D>(a, x0, WX, y0 + r, z);
  }
  if (!fast) {
#pragma unroll 1
    for (int r = 0; r < RY; r++) {
      if (y0 + r >= yend) break;
#pragma unroll 1
      for (int p = 0; p < WX / 32; p++) {
        if (r || p) __syncthreads();
        if (x0 + 32 * p < nx) run_tile<LAT, SCHEME, real, 32, 0, STREAM>(a, tx, k, x0 + 32 * p, y0 + r, z, 0, sh32);
      }
    }
    return;
  }
  // ---- interior fluid tile: this thread owns one cell and all its K sets ----
  const int tid = k * 32 + tx;
  const int x = x0 + tid % WX, y = y0 + tid / WX;
  const uint32_t n = ((uint32_t)z * ny + y) * nx + x;
  char *__restrict__ pb = reinterpret_cast<char *>(const_cast<real *>(a.src) + n);
  real f[K][Q];
#pragma unroll
  for (int l = 0; l < K; l++)
#pragma unroll
    for (int i = 0; i < Q; i++)
      f[l][i] = *reinterpret_cast<const real *>(pb + (long long)l * a.kplane + (STREAM == ST_LOC ? a.st_off[opp(i)] : a.ld_off[i]));
  real Qv[K], Qlo[K];
#pragma unroll
  for (int l = 0; l < K; l++) {      // S2 zeroth moments
    Qv[l] = moment_sum<L, real>(f[l], Qlo[l]);
  }
  real delta;                        // S3 (A6) or the relaxation variable (A19)
  if constexpr (SCHEME == kIdealD) {
    delta = Qv[K - 1] * a.inv_tau_relax;
  } else {
    real tr = real(0);
#pragma unroll
    for (int b = 0; b < D; b++) {
      real m = real(0);
#pragma unroll
      for (int i = 0; i < Q; i++)
        if (lat_c<L>(i, b) != 0) m += real(lat_c<L>(i, b)) * f[iB + b][i];
      tr += m;
    }
    delta = -tr * a.inv_tauB_cs2;
  }
  const bool wM = STREAM != ST_AB && (((npy && (y == 1 || y == ny - 2)) || (npz && (z == 1 || z == nz - 2))) || (npx && x == nx - 2));
  char *__restrict__ ob = STREAM == ST_AB ? reinterpret_cast<char *>(a.dst + n) : pb;
#pragma unroll
  for (int l = 0; l < K; l++) {      // S4, S6-S8 row by row; the compiler shares 1/rho, u, p_tot, u.B across the rows
    real Phi[3];
    flux_row<SCHEME, D, real>(l, Qv, Qv[l], a.gamma, a.c0sq, a.eta, a.mu, a.inv_tau_relax, Phi);
    real inj = -(a.kappa * delta) * powell_row<SCHEME, D, real>(l, Qv);
    if (has_relax(SCHEME) && l >= 8) inj = -Qv[l] * a.inv_tau_relax;
    if (STREAM != ST_AB && wM) a.M_next[(size_t)l * ((size_t)nx * ny * nz) + n] = (double)(Qv[l] + inj);
    const Collide<L, real> col(a.omega[l], a.tau[l], Qv[l], Qlo[l], inj, Phi);
#pragma unroll
    for (int i = 0; i < Q; i++)
      *reinterpret_cast<real *>(ob + (long long)l * a.kplane + (STREAM == ST_PP ? a.ld_off[opp(i)] : a.st_off[i])) = col.out(i, f[l][i]);
  }
}

// =====================================================================================================
// Many steps in ONE launch: small lattices (config 1: 25 tiles, config 2: 8192) are bound by the
// launch-to-launch latency and by the fill and drain of every launch, not by HBM.  A cooperative grid of at most the
// co-resident block count loops over the tiles of a step (run_tile, the one-cell paths), meets at a grid barrier, flips the
// population copies (A/B) or the step type (in place) and goes on.  The per-step part of the arguments (copies, published
// moment arrays, sphere centre) lives in a shared-memory copy of StepArgs that thread 0 updates between steps.
// =====================================================================================================
template <typename real> struct PersistArgs {
  int n_steps;
  int inplace, parity0;         // in place: the first step is a pull-push step (parity 0) or a local step (1)
  real *pop[2];                 // A/B: pop[0] is read by the first step; in place: both the single copy
  double *M[2];                 // in place: M[0] is M_cur of the first step
  long long t_rel0;             // sphere: steps since lbmhd_set_sphere at the first step
  double sph_c0[3];             // sphere centre when it was set (A12: centre before step t is c0 + (t - t0) u)
  int tiles_x;
  long long n_tiles;            // tiles_x * ny * nz
};

template <int LAT, int SCHEME, typename real, int MINB, bool INPLACE>
__global__ void __launch_bounds__(32 * Vars<SCHEME, Lattice<LAT>::D>::K, MINB)
step_kernel_persist(const __grid_constant__ StepArgs<real> a0, const __grid_constant__ PersistArgs<real> p) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, K = Vars<SCHEME, D>::K;
  __shared__ real sQ[K][32];
  __shared__ real sTr[D * D][32];
  __shared__ real sNb[K];
  __shared__ StepArgs<real> sa;
  static_assert(sizeof(StepArgs<real>) % 4 == 0, "word copy");
  namespace cg = cooperative_groups;
  const int tid = threadIdx.y * 32 + threadIdx.x, nthr = 32 * K;
  {
    const uint32_t *src = reinterpret_cast<const uint32_t *>(&a0);
    uint32_t *dst = reinterpret_cast<uint32_t *>(&sa);
    for (int j = tid; j < (int)(sizeof(StepArgs<real>) / 4); j += nthr) dst[j] = src[j];
  }
  const Share<real, 32, false> sh{sQ, sTr, sNb, nullptr, nullptr, nullptr, SyncBlock{}};
  for (int s = 0; s < p.n_steps; s++) {
    __syncthreads();
    if (tid == 0) {
      sa.src = p.pop[s & 1];
      sa.dst = p.pop[(s & 1) ^ 1];
      sa.M_cur = INPLACE ? p.M[s & 1] : nullptr;
      sa.M_next = INPLACE ? p.M[(s & 1) ^ 1] : nullptr;
      if (a0.has_sphere) {
        const double dt = (double)(p.t_rel0 + s);
#pragma unroll
        for (int c = 0; c < 3; c++) sa.sph_c[c] = __dadd_rn(p.sph_c0[c], __dmul_rn(dt, a0.sph_u[c]));
      }
    }
    __syncthreads();
    const bool pullpush = INPLACE && (((p.parity0 + s) & 1) == 0);
    for (long long tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x) {
      const int bx = (int)(tile % p.tiles_x);
      const long long row = tile / p.tiles_x;
      const int y = (int)(row % a0.ny), z = (int)(row / a0.ny);
      if constexpr (!INPLACE) run_tile<LAT, SCHEME, real, 32, 0, ST_AB>(sa, threadIdx.x, threadIdx.y, bx * 32, y, z, 0, sh);
      else if (pullpush) run_tile<LAT, SCHEME, real, 32, 0, ST_PP>(sa, threadIdx.x, threadIdx.y, bx * 32, y, z, 0, sh);
      else run_tile<LAT, SCHEME, real, 32, 0, ST_LOC>(sa, threadIdx.x, threadIdx.y, bx * 32, y, z, 0, sh);
      __syncthreads();      // the exchange arrays are reused by the next tile
    }
    if (s + 1 < p.n_steps) cg::this_grid().sync();      // every store of this step is visible before any pull of the next
  }
}

// ---- S10 init: g_{k,i} = w_i (Q_k + c_i.Phi_k(Q)/c_s^2) (Eq.3) from fp64 fields [K][N] ---------
template <int LAT, int SCHEME, typename real, int TX>
__global__ void __launch_bounds__(TX * Vars<SCHEME, Lattice<LAT>::D>::K)
init_kernel(const double *__restrict__ fields, real *__restrict__ g, size_t pstride, int nx, int ny, int nz, real gamma,
            real c0sq, real eta, real mu, real itm) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q, K = Vars<SCHEME, D>::K;
  const int k = threadIdx.y;
  const int x = blockIdx.x * TX + threadIdx.x;
  if (x >= nx) return;
  const size_t N = (size_t)nx * ny * nz;
  const size_t n = ((size_t)blockIdx.z * ny + blockIdx.y) * nx + x;
  real Qv[K], Phi[3];
#pragma unroll
  for (int l = 0; l < K; l++) Qv[l] = (real)fields[(size_t)l * N + n];
  flux_row<SCHEME, D, real>(k, Qv, pick<K, real>(Qv, k), gamma, c0sq, eta, mu, itm, Phi);
  const real Qk = pick<K, real>(Qv, k);
  real *gk = g + (size_t)k * Q * pstride;
#pragma unroll
  for (int i = 0; i < Q; i++) {
    const real cPhi = real(L::cx(i)) * Phi[0] + real(L::cy(i)) * Phi[1] + real(L::cz(i)) * Phi[2];
    gk[(size_t)i * pstride + n] = real(L::w(i)) * (Qk + real(L::inv_cs2) * cPhi);
  }
}

// ---- S9a moments: Q_k(x) = sum_i g_{k,i}(x) (Eq.4), fp64 out [K][N] --------------------------
template <int LAT, int SCHEME, typename real, int TX>
__global__ void __launch_bounds__(TX * Vars<SCHEME, Lattice<LAT>::D>::K)
moments_kernel(const real *__restrict__ g, size_t pstride, double *__restrict__ out, int nx, int ny, int nz) {
  using L = Lattice<LAT>;
  constexpr int Q = L::Q;
  const int k = threadIdx.y;
  const int x = blockIdx.x * TX + threadIdx.x;
  if (x >= nx) return;
  const size_t N = (size_t)nx * ny * nz;
  const size_t n = ((size_t)blockIdx.z * ny + blockIdx.y) * nx + x;
  const real *gk = g + (size_t)k * Q * pstride;
  double s = 0.0;      // fp64 accumulation in both precisions: the output is fp64 and an fp32 sum would only add its own rounding
#pragma unroll
  for (int i = 0; i < Q; i++) s += (double)gk[(size_t)i * pstride + n];
  out[(size_t)k * N + n] = s;
}

// ---- in-place layout P1 (after a pull-push step): g_{k,j}(x) lives at (x + c_j, slot opp(j)), or at (x, slot j) when
// x + c_j is outside a non-periodic face.  Element fetch used by the P1 moments and export kernels. ----------------
template <class L, typename real>
__device__ __forceinline__ real p1_fetch(const real *__restrict__ gk, size_t pstride, int j, int x, int y, int z, int nx, int ny,
                                         int nz, bool npx, bool npy, bool npz) {
  int sx = x + lat_c<L>(j, 0), sy = y + lat_c<L>(j, 1), sz = z + lat_c<L>(j, 2);
  bool outside = false;
  if (sx < 0) { if (npx) outside = true; else sx += nx; } else if (sx >= nx) { if (npx) outside = true; else sx -= nx; }
  if (sy < 0) { if (npy) outside = true; else sy += ny; } else if (sy >= ny) { if (npy) outside = true; else sy -= ny; }
  if (sz < 0) { if (npz) outside = true; else sz += nz; } else if (sz >= nz) { if (npz) outside = true; else sz -= nz; }
  if (outside) return gk[(size_t)j * pstride + ((size_t)z * ny + y) * nx + x];
  return gk[(size_t)opp(j) * pstride + ((size_t)sz * ny + sy) * nx + sx];
}

template <int LAT, int SCHEME, typename real, int TX>
__global__ void __launch_bounds__(TX * Vars<SCHEME, Lattice<LAT>::D>::K)
moments_p1_kernel(const real *__restrict__ g, size_t pstride, double *__restrict__ out, int nx, int ny, int nz, int bc0, int bc2, int bc4) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q;
  const int k = threadIdx.y;
  const int x = blockIdx.x * TX + threadIdx.x, y = blockIdx.y, z = blockIdx.z;
  if (x >= nx) return;
  const size_t N = (size_t)nx * ny * nz;
  const size_t n = ((size_t)z * ny + y) * nx + x;
  const real *gk = g + (size_t)k * Q * pstride;
  const bool npx = bc0 != BC_PERIODIC, npy = D > 1 && bc2 != BC_PERIODIC, npz = D > 2 && bc4 != BC_PERIODIC;
  double s = 0.0;
#pragma unroll
  for (int j = 0; j < Q; j++) s += (double)p1_fetch<L, real>(gk, pstride, j, x, y, z, nx, ny, nz, npx, npy, npz);
  out[(size_t)k * N + n] = s;
}

template <int LAT, typename real>
__global__ void pops_export_p1_kernel(const real *__restrict__ g, size_t pstride, double *__restrict__ out, int nx, int ny, int nz,
                                      int planes, int bc0, int bc2, int bc4) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q;
  const size_t N = (size_t)nx * ny * nz, total = N * (size_t)planes;
  const bool npx = bc0 != BC_PERIODIC, npy = D > 1 && bc2 != BC_PERIODIC, npz = D > 2 && bc4 != BC_PERIODIC;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
    const size_t pl = e / N, n = e - pl * N;
    const int k = (int)(pl / Q), j = (int)(pl % Q);
    const int x = (int)(n % nx), y = (int)((n / nx) % ny), z = (int)(n / ((size_t)nx * ny));
    out[e] = (double)p1_fetch<L, real>(g + (size_t)k * Q * pstride, pstride, j, x, y, z, nx, ny, nz, npx, npy, npz);
  }
}

// ---- S9b diagnostics: two-stage deterministic reduction with warp shuffles --------------------------------
// slots: [0,K) sum | [K,2K) sum|.| | [2K,3K) max|.| | 3K max|div_h B| | 3K+1 min rho | 3K+2 min p | 3K+3 flag
constexpr int kDiagThreads = 256;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ double warp_min(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// kind: 0 sum, 1 max, 2 min.  Result valid in thread 0.
template <int KIND> __device__ __forceinline__ double block_reduce(double v, double *sm) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  v = KIND == 0 ? warp_sum(v) : (KIND == 1 ? warp_max(v) : warp_min(v));
  __syncthreads();
  if (lane == 0) sm[wid] = v;
  __syncthreads();
  if (wid == 0) {
    const int nw = blockDim.x >> 5;
    v = lane < nw ? sm[lane] : (KIND == 0 ? 0.0 : (KIND == 1 ? -INFINITY : INFINITY));
    v = KIND == 0 ? warp_sum(v) : (KIND == 1 ? warp_max(v) : warp_min(v));
  }
  return v;
}

template <int LAT, int SCHEME>
__global__ void __launch_bounds__(kDiagThreads)
diag_partial_kernel(const double *__restrict__ F, double *__restrict__ partial, int nx, int ny, int nz, int bc0, int bc2,
                    int bc4, double gamma, int ghost_lo, int ghost_hi) {
  using L = Lattice<LAT>;
  constexpr int D = L::D, Q = L::Q, K = Vars<SCHEME, D>::K, iB = Vars<SCHEME, D>::iB;
  __shared__ double sm[32];
  const size_t N = (size_t)nx * ny * nz;
  double sum[K], asum[K], mx[K];
#pragma unroll
  for (int l = 0; l < K; l++) { sum[l] = 0.0; asum[l] = 0.0; mx[l] = 0.0; }
  double maxdiv = 0.0, minrho = INFINITY, minp = INFINITY, flag_nan = 0.0, flag_rho = 0.0;
  const bool per[3] = {bc0 == BC_PERIODIC, bc2 == BC_PERIODIC, bc4 == BC_PERIODIC};
  const int nn[3] = {nx, ny, nz};
  for (size_t n = (size_t)blockIdx.x * blockDim.x + threadIdx.x; n < N; n += (size_t)gridDim.x * blockDim.x) {
    const int x = (int)(n % nx), y = (int)((n / nx) % ny), z = (int)(n / ((size_t)nx * ny));
    const int xi[3] = {x, y, z};
    if (D >= 2) {      // ghost planes of a slab belong to the neighbour: not counted
      const int hc = D == 3 ? z : y, hn = D == 3 ? nz : ny;
      if ((ghost_lo && hc == 0) || (ghost_hi && hc == hn - 1)) continue;
    }
    double v[K];
#pragma unroll
    for (int l = 0; l < K; l++) {
      v[l] = F[(size_t)l * N + n];
      if (!isfinite(v[l])) flag_nan = 1.0;
      sum[l] += v[l];
      asum[l] += fabs(v[l]);
      mx[l] = fmax(mx[l], fabs(v[l]));
    }
    double div = 0.0;
#pragma unroll
    for (int i = 1; i < Q; i++) {
      int q[3] = {x, y, z};
#pragma unroll
      for (int c = 0; c < D; c++) {
        q[c] = xi[c] + lat_c<L>(i, c);
        if (q[c] < 0) q[c] = per[c] ? q[c] + nn[c] : 0;
        else if (q[c] >= nn[c]) q[c] = per[c] ? q[c] - nn[c] : nn[c] - 1;
      }
      const size_t nq = ((size_t)q[2] * ny + q[1]) * nx + q[0];
      double cB = 0.0;
#pragma unroll
      for (int c = 0; c < D; c++)
        if (lat_c<L>(i, c) != 0) cB += (double)lat_c<L>(i, c) * F[(size_t)(iB + c) * N + nq];
      div += L::w(i) * cB;
    }
    div *= L::inv_cs2;
    maxdiv = fmax(maxdiv, fabs(div));
    if (is_ideal(SCHEME)) {
      const double rho = v[0];
      const double mu = (v[1] * v[1] + v[2] * v[2] + v[3] * v[3]) / rho;
      const double B2 = v[5] * v[5] + v[6] * v[6] + v[7] * v[7];
      const double p = (gamma - 1.0) * (v[4] - 0.5 * mu - 0.5 * B2);
      minrho = fmin(minrho, rho);
      minp = fmin(minp, p);
      if (!(rho > 0.0)) flag_rho = 1.0;
    } else {
      minp = fmin(minp, v[0]);
      minrho = 1.0;
    }
  }
  double *out = partial + (size_t)blockIdx.x * (3 * K + 4);
#pragma unroll
  for (int l = 0; l < K; l++) {
    double r = block_reduce<0>(sum[l], sm);
    if (threadIdx.x == 0) out[l] = r;
    r = block_reduce<0>(asum[l], sm);
    if (threadIdx.x == 0) out[K + l] = r;
    r = block_reduce<1>(mx[l], sm);
    if (threadIdx.x == 0) out[2 * K + l] = r;
  }
  double r = block_reduce<1>(maxdiv, sm);
  if (threadIdx.x == 0) out[3 * K] = r;
  r = block_reduce<2>(minrho, sm);
  if (threadIdx.x == 0) out[3 * K + 1] = r;
  r = block_reduce<2>(minp, sm);
  if (threadIdx.x == 0) out[3 * K + 2] = r;
  r = block_reduce<1>(flag_nan, sm);
  const double r2 = block_reduce<1>(flag_rho, sm);
  if (threadIdx.x == 0) out[3 * K + 3] = r + 2.0 * r2;
}

// stage 2: one block folds the per-block partials in block order (deterministic).  The flag slot is a bit mask
// (1 = non-finite seen, 2 = rho <= 0 seen): its two bits fold separately (OR), so NaN in one block and rho <= 0 in
// another give 3.
static __global__ void __launch_bounds__(kDiagThreads)
diag_final_kernel(const double *__restrict__ partial, int nblocks, int K, double *__restrict__ out) {
  __shared__ double sm[32];
  const int nslots = 3 * K + 4;
  for (int s = 0; s < nslots - 1; s++) {
    const int kind = s < 2 * K ? 0 : (s < 3 * K + 1 ? 1 : 2);
    double v = kind == 0 ? 0.0 : (kind == 1 ? -INFINITY : INFINITY);
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) {
      const double p = partial[(size_t)b * nslots + s];
      v = kind == 0 ? v + p : (kind == 1 ? fmax(v, p) : fmin(v, p));
    }
    double r = kind == 0 ? block_reduce<0>(v, sm) : (kind == 1 ? block_reduce<1>(v, sm) : block_reduce<2>(v, sm));
    if (threadIdx.x == 0) out[s] = r;
  }
  double f_nan = 0.0, f_rho = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += blockDim.x) {
    const int bits = (int)partial[(size_t)b * nslots + nslots - 1];
    if (bits & 1) f_nan = 1.0;
    if (bits & 2) f_rho = 1.0;
  }
  f_nan = block_reduce<1>(f_nan, sm);
  f_rho = block_reduce<1>(f_rho, sm);
  if (threadIdx.x == 0) out[nslots - 1] = f_nan + 2.0 * f_rho;
}

// ---- population import / export: canonical fp64 [K*Q][N] <-> internal real planes with pstride ------------
template <typename real>
__global__ void pops_export_kernel(const real *__restrict__ g, size_t pstride, double *__restrict__ out, size_t N, int planes) {
  const size_t total = N * (size_t)planes;
  for (size_t j = (size_t)blockIdx.x * blockDim.x + threadIdx.x; j < total; j += (size_t)gridDim.x * blockDim.x) {
    const size_t pl = j / N, n = j - pl * N;
    out[j] = (double)g[pl * pstride + n];
  }
}
template <typename real>
__global__ void pops_import_kernel(const double *__restrict__ in, real *__restrict__ g, size_t pstride, size_t N, int planes) {
  const size_t total = N * (size_t)planes;
  for (size_t j = (size_t)blockIdx.x * blockDim.x + threadIdx.x; j < total; j += (size_t)gridDim.x * blockDim.x) {
    const size_t pl = j / N, n = j - pl * N;
    g[pl * pstride + n] = (real)in[j];
  }
}

// ---- slab halo: pack the populations of one plane of the slowest axis (the listed directions, all K sets) into a
// contiguous buffer [K][ndir][plane cells], or write such a buffer into a plane.  A list entry is the direction index plus
// its in-plane components: dir | (c_x + 1) << 8 | (c_y + 1) << 10.
// filt_x / filt_y (unpack of LBMHD_HALO_RETURN only): slot s of plane cell (x, y) was pushed by the cell at (x + c_sx,
// y + c_sy) of the neighbouring slab's plane; where that cell would lie outside a non-periodic face nobody pushed, the
// buffer holds no value for it, and the destination keeps what its own cell left there (a population that could not be
// pushed out of the domain stays in its own slot). ------------------------------
template <typename real, bool PACK>
__global__ void halo_plane_kernel(real *__restrict__ g, size_t pstride, real *__restrict__ buf, size_t plane_cells, size_t plane_first,
                                  int K, int Q, int ndir, const int *__restrict__ dirs, int nx, int ny, int filt_x, int filt_y) {
  const size_t total = (size_t)K * ndir * plane_cells;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
    const size_t c = e % plane_cells, kd = e / plane_cells;
    const int d = (int)(kd % ndir), k = (int)(kd / ndir);
    const int entry = dirs[d], dir = entry & 255;
    if (!PACK && (filt_x | filt_y)) {
      const int x = (int)(c % nx), y = (int)(c / nx);
      const int px = x + ((entry >> 8) & 3) - 1, py = y + ((entry >> 10) & 3) - 1;
      if ((filt_x && (px < 0 || px >= nx)) || (filt_y && (py < 0 || py >= ny))) continue;
    }
    real *slot = g + ((size_t)k * Q + dir) * pstride + plane_first + c;
    if (PACK) buf[e] = *slot;
    else *slot = buf[e];
  }
}

// ---- bandwidth probe: BabelStream-style copy, 2 fp64 per thread per iteration ----------------
static __global__ void __launch_bounds__(256) copy_probe_kernel(const double2 *__restrict__ a, double2 *__restrict__ b, size_t n2) {
  for (size_t j = (size_t)blockIdx.x * blockDim.x + threadIdx.x; j < n2; j += (size_t)gridDim.x * blockDim.x) b[j] = a[j];
}

static __global__ void __launch_bounds__(256) triad_probe_kernel(double2 *__restrict__ a, const double2 *__restrict__ b,
                                                                const double2 *__restrict__ c, double s, size_t n2) {
  for (size_t j = (size_t)blockIdx.x * blockDim.x + threadIdx.x; j < n2; j += (size_t)gridDim.x * blockDim.x) {
    const double2 bv = b[j], cv = c[j];
    a[j] = make_double2(fma(s, cv.x, bv.x), fma(s, cv.y, bv.y));
  }
}

}  // namespace lbk
