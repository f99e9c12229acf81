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
    const uint64_t p0 = static_cast<uint64_t>(M0) * c0;   // one IMAD.WIDE.U32 gives hi and lo
    const uint64_t p1 = static_cast<uint64_t>(M1) * c2;
    const uint32_t hi0 = static_cast<uint32_t>(p0 >> 32), lo0 = static_cast<uint32_t>(p0);
    const uint32_t hi1 = static_cast<uint32_t>(p1 >> 32), lo1 = static_cast<uint32_t>(p1);
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
// Float modes (R9, judged statistically): the proposal offset is the word read as a signed integer,
// converted with round-to-nearest (24-bit mantissa) -- a symmetric uniform on [-2^31, 2^31] whose
// scale 2^-31 is folded into ChainConst::hscale; the acceptance uniform is the word converted as
// an unsigned integer, u2 = float(w) 2^-32 in [0, 1].  One conversion instruction each.
__device__ __forceinline__ float sym_word(uint32_t a) { return static_cast<float>(static_cast<int32_t>(a)); }
__device__ __forceinline__ float pos_word(uint32_t a) { return static_cast<float>(a); }

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
  // the MUFU.EX2 that __expf(x) = ex2(x log2 e) ends in, with the scale folded by the caller
  static __device__ __forceinline__ float ex2_(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
  }
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
  R hscale;    // float modes: q Delta / 2 = hscale * float(int32 word) = (delta / 4) 2^-31 word
  R xscale;    // SP_INTRINSIC: -log2(e) / T, so that exp(-dE / T) 2^32 = ex2(dE * xscale + 32)
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

// Random words of the Metropolis move at a site (R9).  Double-arithmetic modes (DP, SP): one
// Philox block per site, counter word 0 = the site's row-major index; all four words are used
// (two 53-bit uniforms), exactly as in the oracle.  Float-arithmetic modes: one block per PAIR of
// sites of the same colour and row whose plane columns are (2m, 2m + 1); counter word 0 = the index
// of the first site of the pair (pair_site); that site takes words (0, 2), the other one (1, 3).
struct MetWords { uint32_t p, q, a, b; };   // proposal (p [, q]) and acceptance (a [, b]) words

template <int MODE>
__device__ __forceinline__ void met_words_pair(uint32_t pair_site, uint32_t sweep,
                                               const ChainConst<typename Traits<MODE>::real>& k,
                                               MetWords* w0, MetWords* w1) {
  if constexpr (sizeof(typename Traits<MODE>::real) == 8) {
    const uint4 r0 = philox4x32_10(pair_site, sweep, PASS_MET, k.trial, k.k0, k.k1);
    const uint4 r1 = philox4x32_10(pair_site + 2u, sweep, PASS_MET, k.trial, k.k0, k.k1);
    *w0 = MetWords{r0.x, r0.y, r0.z, r0.w};
    *w1 = MetWords{r1.x, r1.y, r1.z, r1.w};
  } else {
    const uint4 r = philox4x32_10(pair_site, sweep, PASS_MET, k.trial, k.k0, k.k1);
    *w0 = MetWords{r.x, 0u, r.z, 0u};
    *w1 = MetWords{r.y, 0u, r.w, 0u};
  }
}

// Metropolis move of one site (R7, R10), written without branches: the new spin is kept iff the
// site is free, the proposal stays in range (s' >= 0) and the acceptance test passes.  Returns
// true when the move was accepted.
template <int MODE>
__device__ __forceinline__ bool met_update(typename Traits<MODE>::real* c, typename Traits<MODE>::real* s,
                                           typename Traits<MODE>::real A, typename Traits<MODE>::real B,
                                           const MetWords& w, bool is_free,
                                           const ChainConst<typename Traits<MODE>::real>& k) {
  using R = typename Traits<MODE>::real;
  R h;                                           // q Delta / 2
  if constexpr (sizeof(R) == 8) {
    const R t = fma_(R(2), R(u53(w.p, w.q)), R(-1));   // 2 u1 - 1 (exact)
    h = R(0.25) * (k.delta * t);
  } else {
    h = k.hscale * sym_word(w.p);
  }
  R sd, cd;
  Fn<MODE>::sincos_(h, &sd, &cd);
  const R ts = sd + sd;
  const R s2 = ts * cd;                          // sin(q Delta)
  const R c2m1 = -(ts * sd);                     // cos(q Delta) - 1
  const R c0 = *c, s0 = *s;
  const R cn = fma_(-s0, s2, fma_(c0, c2m1, c0));   // c cos - s sin
  const R sn = fma_(c0, s2, fma_(s0, c2m1, s0));    // s cos + c sin
  const R P = fma_(c0, A, s0 * B);               // u.F
  const R Q = fma_(c0, B, -(s0 * A));            // c B - s A
  const R dE = ts * fma_(sd, P, -(cd * Q));
  bool acc;
  if constexpr (sizeof(R) == 8) {
    acc = R(u53(w.a, w.b)) < Fn<MODE>::exp_(-(dE * k.inv_T));
  } else if constexpr (MODE == MODE_SP_INTRINSIC) {
    acc = pos_word(w.a) < Fn<MODE>::ex2_(fma_(dE, k.xscale, R(32)));   // = __expf(-dE/T) 2^32: one FFMA + MUFU.EX2
  } else {
    acc = pos_word(w.a) * R(2.3283064365386963e-10) < Fn<MODE>::exp_(-(dE * k.inv_T));
  }
  const bool ok = is_free && (sn >= R(0)) && acc;
  *c = ok ? cn : c0;
  *s = ok ? sn : s0;
  return ok;
}

// Over-relaxation move (R5): reflect u about the local field; keep it iff the site is free, F != 0
// and u' stays on the upper half circle.  One Newton step towards |u| = 1 stops the rounding
// drift of the norm.  Branch-free.
template <int MODE>
__device__ __forceinline__ void or_update(typename Traits<MODE>::real* c, typename Traits<MODE>::real* s,
                                          typename Traits<MODE>::real A, typename Traits<MODE>::real B,
                                          bool is_free) {
  using R = typename Traits<MODE>::real;
  const R R2 = fma_(A, A, B * B);
  const R c0 = *c, s0 = *s;
  const R P = fma_(c0, A, s0 * B);
  const R t = Fn<MODE>::div_(P + P, R2);
  R cn = fma_(t, A, -c0);
  R sn = fma_(t, B, -s0);
  const bool ok = is_free && (R2 != R(0)) && (sn >= R(0));
  const R f = fma_(R(-0.5), fma_(cn, cn, sn * sn), R(1.5));
  cn = cn * f; sn = sn * f;
  *c = ok ? cn : c0;
  *s = ok ? sn : s0;
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
