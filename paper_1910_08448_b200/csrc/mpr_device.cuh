// mpr_device.cuh -- per-site arithmetic of the MPR conditional hybrid sweep, shared by the
// plain (one launch per colour pass) and the tiled (TMA + shared memory) kernels so that both
// give bit-identical spins.  Compiled with --fmad=false: every fused multiply-add below is
// written out, so the rounding sequence does not depend on the inlining context.
//
// Spin representation.  H = -J sum cos[q(phi_i - phi_j)] (Eq. 2)
// depends on the spins only through the unit vectors u_i = (cos q phi_i, sin q phi_i):
// cos[q(phi_i - phi_j)] = u_i . u_j.  With q = 1/2 and phi in [0, 2pi], q phi lies in [0, pi],
// i.e. the upper half circle s >= 0, and phi = 2 atan2(s, c).  The library stores u_i; the
// local field of a site is F = (A, B) = sum_j u_j over its existing neighbours.
//   Metropolis (R7):  phi' = phi + Delta  <=>  u' = rot(q Delta) u;  phi' in [0, 2pi] <=> s' >= 0;
//       dE = -(u' - u).F = 2 sd (sd P - cd Q),  sd = sin(q Delta/2), cd = cos(q Delta/2),
//       P = u.F, Q = c B - s A  (cancellation-free form of the cos differences).
//   Over-relaxation (R5):  q phi' = 2 Phi - q phi, Phi = atan2(B, A)  <=>  u' = 2 (u.F) F/|F|^2 - u,
//       in range <=> s' >= 0 (B >= 0 always, so q phi' lies in [-pi, 2pi]).
//   Quench (R8):  phi = Phi/q  <=>  u = F/|F|.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mpr {

enum { MODE_DP = 0, MODE_SP = 1, MODE_SP_PRECISE = 2, MODE_SP_INTRINSIC = 3 };
enum { PASS_INIT = 0, PASS_MET = 1 };  // Philox counter word 2 (R9)
enum { KIND_MET = 0, KIND_OR = 1, KIND_QUENCH = 2 };

template <int MODE> struct Traits;
template <> struct Traits<MODE_DP>           { using real = double; using vec = double2; };
template <> struct Traits<MODE_SP>           { using real = double; using vec = float2;  };
template <> struct Traits<MODE_SP_PRECISE>   { using real = float;  using vec = float2;  };
template <> struct Traits<MODE_SP_INTRINSIC> { using real = float;  using vec = float2;  };

// ---- Philox4x32-10 (Salmon et al., SC'11), restated.  counter (c0..c3), key (k0, k1).
// R9: counter = (site, sweep, pass, trial), key = (seed lo, seed hi).
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
    const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += W0; k1 += W1;
  }
  return make_uint4(c0, c1, c2, c3);
}

// 53-bit uniform in [0,1): 27 high bits of a, 26 high bits of b (exact in double).
__device__ __forceinline__ double u53(uint32_t a, uint32_t b) {
  const double hi = static_cast<double>(a >> 5);
  const double lo = static_cast<double>(b >> 6);
  return (hi * 67108864.0 + lo) * (1.0 / 9007199254740992.0);
}
// 24-bit uniform in (0,1), bin centres (float modes; judged statistically).
__device__ __forceinline__ float u24(uint32_t a) {
  return (static_cast<float>(a >> 8) + 0.5f) * (1.0f / 16777216.0f);
}

// ---- function-precision policies (X_F) -----------------------------------
template <int MODE> struct Fn;
template <> struct Fn<MODE_DP> {
  static __device__ __forceinline__ void sincos_(double x, double* s, double* c) { sincos(x, s, c); }
  static __device__ __forceinline__ double exp_(double x) { return exp(x); }
  static __device__ __forceinline__ double div_(double a, double b) { return a / b; }
  static __device__ __forceinline__ double rsqrt_(double x) { return 1.0 / sqrt(x); }
  static __device__ __forceinline__ double atan2_(double y, double x) { return atan2(y, x); }
};
template <> struct Fn<MODE_SP> : Fn<MODE_DP> {};
template <> struct Fn<MODE_SP_PRECISE> {
  static __device__ __forceinline__ void sincos_(float x, float* s, float* c) { sincosf(x, s, c); }
  static __device__ __forceinline__ float exp_(float x) { return expf(x); }
  static __device__ __forceinline__ float div_(float a, float b) { return a / b; }
  static __device__ __forceinline__ float rsqrt_(float x) { return 1.0f / sqrtf(x); }
  static __device__ __forceinline__ float atan2_(float y, float x) { return atan2f(y, x); }
};
template <> struct Fn<MODE_SP_INTRINSIC> {
  static __device__ __forceinline__ void sincos_(float x, float* s, float* c) {
    *s = __sinf(x); *c = __cosf(x);
  }
  static __device__ __forceinline__ float exp_(float x) { return __expf(x); }
  static __device__ __forceinline__ float div_(float a, float b) { return __fdividef(a, b); }
  static __device__ __forceinline__ float rsqrt_(float x) { return rsqrtf(x); }
  static __device__ __forceinline__ float atan2_(float y, float x) { return atan2f(y, x); }
};

__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }

// Run-time constants of a chain, in the arithmetic type of the mode.
template <typename R> struct ChainConst {
  R delta;     // R7 proposal half-width min(pi, 4 sqrt(T/(4 J q^2)))
  R inv_T;     // 1/T
  uint32_t k0, k1, trial;
};

// Local field from the four neighbours in the fixed order left, right, up, down; a missing
// neighbour (open boundaries, R2) contributes exactly 0.
template <typename R>
__device__ __forceinline__ void local_field(R lc, R ls, R rc, R rs, R uc, R us, R dc, R ds,
                                            bool hl, bool hr, bool hu, bool hd, R* A, R* B) {
  const R z = R(0);
  R a = hl ? lc : z, b = hl ? ls : z;
  a = a + (hr ? rc : z); b = b + (hr ? rs : z);
  a = a + (hu ? uc : z); b = b + (hu ? us : z);
  a = a + (hd ? dc : z); b = b + (hd ? ds : z);
  *A = a; *B = b;
}

// Metropolis move of one free site (R7, R10).  Returns true when accepted.
template <int MODE>
__device__ __forceinline__ bool met_update(typename Traits<MODE>::real* c, typename Traits<MODE>::real* s,
                                           typename Traits<MODE>::real A, typename Traits<MODE>::real B,
                                           uint32_t site, uint32_t sweep,
                                           const ChainConst<typename Traits<MODE>::real>& k) {
  using R = typename Traits<MODE>::real;
  const uint4 r = philox4x32_10(site, sweep, PASS_MET, k.trial, k.k0, k.k1);
  R t, u2;
  if constexpr (sizeof(R) == 8) {
    t = fma_(R(2), R(u53(r.x, r.y)), R(-1));     // 2 u1 - 1 (exact)
    u2 = R(u53(r.z, r.w));
  } else {
    t = fma_(R(2), R(u24(r.x)), R(-1));
    u2 = R(u24(r.z));
  }
  const R h = R(0.25) * (k.delta * t);           // q Delta / 2
  R sd, cd;
  Fn<MODE>::sincos_(h, &sd, &cd);
  const R s2 = R(2) * (sd * cd);                 // sin(q Delta)
  const R c2m1 = R(-2) * (sd * sd);              // cos(q Delta) - 1
  const R c0 = *c, s0 = *s;
  const R cn = fma_(c0, c2m1, c0) - s0 * s2;     // c cos - s sin
  const R sn = fma_(s0, c2m1, s0) + c0 * s2;     // s cos + c sin
  const R P = fma_(c0, A, s0 * B);               // u.F
  const R Q = fma_(c0, B, -(s0 * A));            // c B - s A
  const R dE = (R(2) * sd) * fma_(sd, P, -(cd * Q));
  const bool ok = (sn >= R(0)) && (u2 < Fn<MODE>::exp_(-(dE * k.inv_T)));
  if (ok) { *c = cn; *s = sn; }
  return ok;
}

// Over-relaxation move (R5): reflect u about the local field; keep it iff it stays on the
// upper half circle.  One Newton step towards |u| = 1 stops the rounding drift of the norm.
template <int MODE>
__device__ __forceinline__ void or_update(typename Traits<MODE>::real* c, typename Traits<MODE>::real* s,
                                          typename Traits<MODE>::real A, typename Traits<MODE>::real B) {
  using R = typename Traits<MODE>::real;
  const R R2 = fma_(A, A, B * B);
  if (R2 == R(0)) return;
  const R c0 = *c, s0 = *s;
  const R P = fma_(c0, A, s0 * B);
  const R t = Fn<MODE>::div_(R(2) * P, R2);
  R cn = fma_(t, A, -c0);
  R sn = fma_(t, B, -s0);
  if (!(sn >= R(0))) return;
  const R f = fma_(R(-0.5), fma_(cn, cn, sn * sn), R(1.5));
  cn = cn * f; sn = sn * f;
  *c = cn; *s = sn;
}

// Quench move (R8): the minimiser of the local energy, u = F/|F|.
template <int MODE>
__device__ __forceinline__ void quench_update(typename Traits<MODE>::real* c, typename Traits<MODE>::real* s,
                                              typename Traits<MODE>::real A, typename Traits<MODE>::real B) {
  using R = typename Traits<MODE>::real;
  const R R2 = fma_(A, A, B * B);
  if (R2 == R(0)) return;
  const R inv = Fn<MODE>::rsqrt_(R2);
  *c = A * inv; *s = B * inv;
}

// phi = 2 atan2(s, c) in [0, 2pi] (s >= 0).
template <int MODE>
__device__ __forceinline__ double spin_angle(typename Traits<MODE>::real c, typename Traits<MODE>::real s) {
  return 2.0 * static_cast<double>(Fn<MODE>::atan2_(s, c));
}

// Column pair of the left/right neighbours in the other colour plane: a site of colour col
// in row y sits at x = 2 j + ((y + col) & 1); its left neighbour is column j - 1 + par, its
// right neighbour column j + par, par = (y + col) & 1.
__device__ __forceinline__ int x_parity(int y, int col) { return (y + col) & 1; }

}  // namespace mpr
