// lbmhd_lattice.cuh — compile-time lattice tables for the CUDA path (A2).
// Direction order: rest; +x,-x,+y,-y,+z,-z; diagonals (+,+),(-,-),(+,-),(-,+) per plane xy, xz, yz.
// Gauss-Hermite weights, c_s^2 = 1/3 on all three lattices.  Every accessor is constexpr
// and is only ever called with a compile-time index inside fully unrolled loops, so no table lives in
// memory: the velocities become immediate offsets and the weights immediate fp constants.
#pragma once

namespace lbk {

template <int LAT> struct Lattice;

template <> struct Lattice<1> {   // D1Q3
  static constexpr int D = 1, Q = 3;
  static constexpr double inv_cs2 = 3.0;
  __host__ __device__ static constexpr int cx(int i) { return i == 1 ? 1 : (i == 2 ? -1 : 0); }
  __host__ __device__ static constexpr int cy(int) { return 0; }
  __host__ __device__ static constexpr int cz(int) { return 0; }
  __host__ __device__ static constexpr double w(int i) { return i == 0 ? 2.0 / 3.0 : 1.0 / 6.0; }
};

template <> struct Lattice<2> {   // D2Q9
  static constexpr int D = 2, Q = 9;
  static constexpr double inv_cs2 = 3.0;
  __host__ __device__ static constexpr int cx(int i) {
    constexpr int t[9] = {0, 1, -1, 0, 0, 1, -1, 1, -1};
    return t[i];
  }
  __host__ __device__ static constexpr int cy(int i) {
    constexpr int t[9] = {0, 0, 0, 1, -1, 1, -1, -1, 1};
    return t[i];
  }
  __host__ __device__ static constexpr int cz(int) { return 0; }
  __host__ __device__ static constexpr double w(int i) { return i == 0 ? 4.0 / 9.0 : (i < 5 ? 1.0 / 9.0 : 1.0 / 36.0); }
};

template <> struct Lattice<3> {   // D3Q19
  static constexpr int D = 3, Q = 19;
  static constexpr double inv_cs2 = 3.0;
  __host__ __device__ static constexpr int cx(int i) {
    constexpr int t[19] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
    return t[i];
  }
  __host__ __device__ static constexpr int cy(int i) {
    constexpr int t[19] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
    return t[i];
  }
  __host__ __device__ static constexpr int cz(int i) {
    constexpr int t[19] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
    return t[i];
  }
  __host__ __device__ static constexpr double w(int i) { return i == 0 ? 1.0 / 3.0 : (i < 7 ? 1.0 / 18.0 : 1.0 / 36.0); }
};

// The paper's own lattices (PAPER.md:183 D2Q5 in all validation cases, :300 D3Q7 in the showcase): axis directions only.
// Rest weight and c_s^2 follow from sum_i w_i = 1 and sum_i w_i c_ia c_ib = c_s^2 delta_ab with the textbook choice
// c_s^2 = 1/3 (D2Q5: w = 1/3, 1/6) resp. c_s^2 = 1/4 (D3Q7: w = 1/4, 1/8).
template <> struct Lattice<4> {   // D2Q5
  static constexpr int D = 2, Q = 5;
  static constexpr double inv_cs2 = 3.0;
  __host__ __device__ static constexpr int cx(int i) { return i == 1 ? 1 : (i == 2 ? -1 : 0); }
  __host__ __device__ static constexpr int cy(int i) { return i == 3 ? 1 : (i == 4 ? -1 : 0); }
  __host__ __device__ static constexpr int cz(int) { return 0; }
  __host__ __device__ static constexpr double w(int i) { return i == 0 ? 1.0 / 3.0 : 1.0 / 6.0; }
};

template <> struct Lattice<5> {   // D3Q7
  static constexpr int D = 3, Q = 7;
  static constexpr double inv_cs2 = 4.0;
  __host__ __device__ static constexpr int cx(int i) { return i == 1 ? 1 : (i == 2 ? -1 : 0); }
  __host__ __device__ static constexpr int cy(int i) { return i == 3 ? 1 : (i == 4 ? -1 : 0); }
  __host__ __device__ static constexpr int cz(int i) { return i == 5 ? 1 : (i == 6 ? -1 : 0); }
  __host__ __device__ static constexpr double w(int i) { return i == 0 ? 1.0 / 4.0 : 1.0 / 8.0; }
};

template <class L> __host__ __device__ constexpr int lat_c(int i, int axis) {
  return axis == 0 ? L::cx(i) : (axis == 1 ? L::cy(i) : L::cz(i));
}

// kIdealD: ideal MHD plus the traced gradient-relaxation variable D = tr G (A19), K = 9
// kResist: ideal MHD plus the transported gradients G_ab = tau_M d_a B_b (a < D, b < 3; variable 8 + 3a + b) with the
//          resistive fluxes taken from them (Eq.9-10; A22), K = 8 + 3 D
// kFull:   kResist plus the transported velocity gradients H_ab = tau_M d_a u_b (variable 8 + 3 D + 3a + b) with the viscous
//          stress -sigma, -u.sigma taken from them: the full dissipative system (A23), K = 8 + 6 D
constexpr int kIdeal = 0, kIncres = 1, kIdealD = 2, kResist = 3, kFull = 4;
__host__ __device__ constexpr bool has_G(int scheme) { return scheme == kResist || scheme == kFull; }   // carries G_ab at 8 + 3a + b
__host__ __device__ constexpr bool is_ideal(int scheme) { return scheme != kIncres; }          // first 8 variables (rho, m, E, B)
__host__ __device__ constexpr bool has_relax(int scheme) { return scheme == kIdealD || scheme == kResist || scheme == kFull; }   // variables >= 8 relax
template <int SCHEME, int D> struct Vars {
  static constexpr int K = SCHEME == kIdeal ? 8 : (SCHEME == kIdealD ? 9 : (SCHEME == kResist ? 8 + 3 * D : (SCHEME == kFull ? 8 + 6 * D : 1 + 2 * D)));
  static constexpr int NV = is_ideal(SCHEME) ? 3 : D;      // vector components carried
  static constexpr int iU = 1;                             // first momentum / velocity component
  static constexpr int iB = is_ideal(SCHEME) ? 5 : 1 + D;  // first magnetic component
};

}  // namespace lbk
