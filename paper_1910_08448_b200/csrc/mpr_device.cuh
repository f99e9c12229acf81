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
#include <cuda_fp16.h>

namespace mpr {

enum { MODE_DP = 0, MODE_SP = 1, MODE_SP_PRECISE = 2, MODE_SP_INTRINSIC = 3, MODE_DS = 4, MODE_HP = 5 };   // DS: double storage, float intrinsics (paper D.S)
enum { PASS_INIT = 0, PASS_MET = 1 };  // Philox counter word 2 (R9)
enum { KIND_MET = 0, KIND_OR = 1, KIND_QUENCH = 2, KIND_MO = 3 };   // MO: Metropolis then over-relaxation in one visit (R4b)

template <int MODE> struct Traits;
template <> struct Traits<MODE_DP>           { using real = double; using vec = double2; };
template <> struct Traits<MODE_SP>           { using real = double; using vec = float2;  };
template <> struct Traits<MODE_SP_PRECISE>   { using real = float;  using vec = float2;  };
template <> struct Traits<MODE_SP_INTRINSIC> { using real = float;  using vec = float2;  };
template <> struct Traits<MODE_DS>           { using real = float;  using vec = double2; };
// half-precision storage (the paper's outlook): (c, s) as two fp16, arithmetic as in SP_INTRINSIC
struct alignas(4) hvec2 { __half x, y; };
template <> struct Traits<MODE_HP>           { using real = float;  using vec = hvec2;   };
__device__ __forceinline__ double to_double(double v) { return v; }
__device__ __forceinline__ double to_double(float v) { return static_cast<double>(v); }
__device__ __forceinline__ double to_double(__half v) { return static_cast<double>(__half2float(v)); }
// CUtensorMapDataType of a storage scalar (cuda.h: FLOAT16 = 6, FLOAT32 = 7, FLOAT64 = 8)
template <typename S> struct TmaType;
template <> struct TmaType<double> { static constexpr int value = 8; };
template <> struct TmaType<float>  { static constexpr int value = 7; };
template <> struct TmaType<__half> { static constexpr int value = 6; };

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

// The same with the ten round keys (k0 + r W0, k1 + r W1) precomputed by the host and passed as
// kernel parameters: each xor reads its key straight from the constant bank -- no key
// registers, no key additions in the inner loop.
struct PhiloxKeys { uint32_t a[10], b[10]; };
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const PhiloxKeys& rk) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = static_cast<uint64_t>(M0) * c0;
    const uint64_t p1 = static_cast<uint64_t>(M1) * c2;
    const uint32_t hi0 = static_cast<uint32_t>(p0 >> 32), lo0 = static_cast<uint32_t>(p0);
    const uint32_t hi1 = static_cast<uint32_t>(p1 >> 32), lo1 = static_cast<uint32_t>(p1);
    const uint32_t n0 = hi1 ^ c1 ^ rk.a[r];
    const uint32_t n2 = hi0 ^ c3 ^ rk.b[r];
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
  }
  return make_uint4(c0, c1, c2, c3);
}

// 53-bit uniform in [0,1): 27 high bits of a, 26 high bits of b (exact in double).
__device__ __forceinline__ double u53(uint32_t a, uint32_t b) {
  const double hi = static_cast<double>(a >> 5);
  const double lo = static_cast<double>(b >> 6);
  return (hi * 67108864.0 + lo) * (1.0 / 9007199254740992.0);
}
// Float modes (R9, judged statistically): ONE 32-bit word per site carries both random numbers of its move.
//   proposal   top 12 bits k:  f = 1 + (k + 1/2) / 4096 in [1, 2), built in the mantissa (no conversion);
//              q Delta / 2 = hscale (f - 3/2): 4096 equidistant offsets, exactly symmetric about 0
//   acceptance low 20 bits m, converted exactly:  accept iff m < exp(-dE/T) 2^20
__device__ __forceinline__ float prop_word(uint32_t w) { return __uint_as_float(((w >> 9) & 0x007FF800u) | 0x3F800400u); }
__device__ __forceinline__ float acc_word(uint32_t w) { return static_cast<float>(w & 0x000FFFFFu); }

// ---- double-precision sin/cos/exp on the ranges the Metropolis move needs ---------------------
// The library sincos(double) / exp(double) are written for any argument: Cody-Waite reduction,
// quadrant logic, a Payne-Hanek slow path behind a branch, and coefficients that the compiler
// rebuilds from immediates at every use (ncu, DP sweep kernel: UMOV 13.7 % of all executed
// instructions, BRA/BSSY/BSYNC 4.3 % of the instructions and 13 % of the stall samples, real
// DFMA/DMUL/DADD only 32 %).  The move calls them on fixed, small ranges:
//   sincos(q Delta / 2):  |q Delta / 2| = |Delta| / 4 <= delta / 4 <= pi / 4   (R7: delta <= pi, q = 1/2)
//   exp(-dE / T) is compared with u2 in [0, 1): only arguments <= 0 decide anything.
// So both are branch-free Taylor polynomials whose coefficients +-1/n! (exact quotients of integers
// below 2^53, correctly rounded by the host compiler) sit in constant memory and enter each DFMA
// as a constant-bank operand.  Truncation errors are below half an ulp: sin stops at x^17
// (next term (pi/4)^19 / 19! = 8e-20), cos at x^16 ((pi/4)^18 / 18! = 2e-18), exp at r^13 with
// |r| <= ln 2 / 2 (r^14 / 14! = 4e-18).
static __constant__ double kSinC[8] = {-1.0 / 6.0, 1.0 / 120.0, -1.0 / 5040.0, 1.0 / 362880.0, -1.0 / 39916800.0,
                                1.0 / 6227020800.0, -1.0 / 1307674368000.0, 1.0 / 355687428096000.0};
static __constant__ double kCosC[8] = {-1.0 / 2.0, 1.0 / 24.0, -1.0 / 720.0, 1.0 / 40320.0, -1.0 / 3628800.0,
                                1.0 / 479001600.0, -1.0 / 87178291200.0, 1.0 / 20922789888000.0};
static __constant__ double kExpC[12] = {1.0 / 2.0, 1.0 / 6.0, 1.0 / 24.0, 1.0 / 120.0, 1.0 / 720.0, 1.0 / 5040.0,
                                 1.0 / 40320.0, 1.0 / 362880.0, 1.0 / 3628800.0, 1.0 / 39916800.0,
                                 1.0 / 479001600.0, 1.0 / 6227020800.0};

// sin and cos of x, |x| <= pi/4 (no range reduction: the caller guarantees the range), from the first NC coefficients
template <int NC>
__device__ __forceinline__ void sincos_taylor(double x, double* s, double* c) {
  const double z = x * x;
  double ps = kSinC[NC - 1], pc = kCosC[NC - 1];
#pragma unroll
  for (int i = NC - 2; i >= 0; --i) { ps = fma(ps, z, kSinC[i]); pc = fma(pc, z, kCosC[i]); }
  *s = fma(x * z, ps, x);        // x + x^3 (S1 + S2 z + ...)
  *c = fma(z, pc, 1.0);          // 1 + z (C1 + C2 z + ...)
}
__device__ __forceinline__ void sincos_quarter(double x, double* s, double* c) { sincos_taylor<8>(x, s, c); }
// The proposal half-angle is bounded by q delta / 2, which shrinks with sqrt(T) (R7): at the temperatures the method
// infers (1e-3 .. 1e-1) most of the 8 + 8 coefficients above multiply powers of x below half an ulp.  `terms` (4, 6 or 8;
// the same for every thread of a launch, chosen on the host by sincos_terms_for) selects a shorter Horner chain whose
// truncation error is still below 2^-54 relative:
//   4 coefficients (sin to x^9, cos to x^8):   |x| <= 0.10   (x^10 / 10! < 2.8e-17, x^11 / 11! < 2.6e-19 x)
//   6 coefficients (sin to x^13, cos to x^12): |x| <= 0.40   (x^14 / 14! < 3.1e-17, x^15 / 15! < 8.3e-19 x)
__device__ __forceinline__ void sincos_quarter_terms(double x, int terms, double* s, double* c) {
  if (terms == 4) sincos_taylor<4>(x, s, c);
  else if (terms == 6) sincos_taylor<6>(x, s, c);
  else sincos_taylor<8>(x, s, c);
}
inline int sincos_terms_for(double max_abs_x) { return max_abs_x <= 0.10 ? 4 : max_abs_x <= 0.40 ? 6 : 8; }

// exp(min(y, 0)): for y >= 0 the result is exactly 1, which exceeds every u2 in [0, 1) -- the same
// decision as "accept if dE <= 0".  y = k ln 2 + r, |r| <= ln 2 / 2; 2^k is applied as two exact
// power-of-two factors 2^(k >> 1) 2^(k - (k >> 1)), both normal for k >= -1075, so that results in
// the subnormal range are rounded once, by the last multiplication.  Below -745.2 the result is 0.
__device__ __forceinline__ double exp_nonpos(double y) {
  y = fmin(y, 0.0);
  const double yc = fmax(y, -745.2);
  const double t = fma(yc, 1.4426950408889634, 6755399441055744.0);   // rint(y log2 e) in the low word
  const int k = __double2loint(t);
  const double kd = t - 6755399441055744.0;
  double r = fma(kd, -0.6931471805599453, yc);                        // ln 2, high part
  r = fma(kd, -2.3190468138462996e-17, r);                            // ln 2, low part
  double p = kExpC[11];
#pragma unroll
  for (int i = 10; i >= 0; --i) p = fma(p, r, kExpC[i]);
  p = fma(r * r, p, r) + 1.0;                                         // 1 + r + r^2 (1/2 + r/6 + ...)
  const int k1 = k >> 1, k2 = k - k1;
  p = p * __hiloint2double((k1 + 1023) << 20, 0);
  p = p * __hiloint2double((k2 + 1023) << 20, 0);
  return y < -745.2 ? 0.0 : p;
}

// The Metropolis decision of the double-arithmetic modes, u2 < exp(min(x, 0)) with x = -dE/T and u2 = u53(wa, wb), taken
// EXACTLY as the double evaluation takes it, but without evaluating the double exponential unless it matters:
//   * 2^y, y = x log2 e, from one MUFU.EX2 in float: ef = 2^y (1 + d), |d| < 6e-6 for y >= -120 (argument rounding
//     |y| 2^-24 ln 2 <= 5e-6, ex2.approx 2^-22);
//   * u2 bracketed by its top 24 bits: u_lo <= u2 < u_hi = u_lo + 2^-24, both exact floats;
//   * u_hi <= ef (1 - 2^-15)  =>  u2 < exp(x): accept;   u_lo >= ef (1 + 2^-15)  =>  u2 > exp(x): reject;
//     y < -120: exp(x) < 2^-119 < 2^-24 <= u_lo unless u_lo = 0: reject;
//   * anything else (probability ~3e-5 per move; also NaN) falls through to the double evaluation, out of line.
// The decision is the one `u53(wa, wb) < exp_nonpos(x)` gives, always; what is saved is the ~25 FP64-pipe
// instructions of exp_nonpos and u53 per move, a fifth of the FP64 work of a DP / SP hybrid sweep (the FP64 pipe is
// what binds those modes on B200).
static __device__ __noinline__ bool metropolis_accept_slow(uint32_t wa, uint32_t wb, double x) {
  return u53(wa, wb) < exp_nonpos(x);
}
// `fast` (tests only): set to false when the decision went through the double evaluation
__device__ __forceinline__ bool metropolis_accept_exact(uint32_t wa, uint32_t wb, double mdE, double inv_T, double log2e_over_T,
                                                        bool* fast = nullptr) {
  const float yf = __double2float_rn(mdE * log2e_over_T);
  float ef;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ef) : "f"(yf));
  const float u_lo = static_cast<float>(wa >> 8) * 5.9604644775390625e-08f;      // k 2^-24, exact
  const float u_hi = u_lo + 5.9604644775390625e-08f;                            // (k + 1) 2^-24, exact
  const bool in_range = yf >= -120.0f, tiny = yf < -120.0f;                      // NaN: neither
  if (in_range && u_hi <= ef * 0.999969482421875f) return true;                  // 1 - 2^-15
  if ((in_range && u_lo >= ef * 1.000030517578125f) || (tiny && u_lo > 0.0f)) return false;   // 1 + 2^-15
  if (fast) *fast = false;
  return metropolis_accept_slow(wa, wb, mdE * inv_T);
}

// ---- function-precision policies (X_F) -----------------------------------
template <int MODE> struct Fn;
template <> struct Fn<MODE_DP> {
  static __device__ __forceinline__ void sincos_(double x, double* s, double* c) { sincos_quarter(x, s, c); }
  static __device__ __forceinline__ double exp_(double x) { return exp_nonpos(x); }
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
  // a * rcp.approx(b): the MUFU.RCP at the heart of __fdividef, without its rescaling of huge / tiny
  // divisors (|F|^2 lies in {0} U [~1e-14, 16]; F = 0 is rejected by the caller)
  static __device__ __forceinline__ float div_(float a, float b) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(b));
    return a * r;
  }
  static __device__ __forceinline__ float rsqrt_(float x) { return rsqrtf(x); }
  // atan2(y, x) for y >= 0 (the upper half circle the spins live on), in the spirit of the other intrinsics of
  // this mode: octant reduction to r = min / max in [0, 1] by one MUFU.RCP, atan(r) = r P(r^2) with a degree-7
  // polynomial (Chebyshev interpolation of atan(sqrt z) / sqrt z on [0, 1], computed for this file; max error
  // 1.7e-7 rad in float evaluation), two selects to undo the reduction.  ~16 instructions against ~40 of atan2f.
  static __device__ __forceinline__ float atan2_(float y, float x) {
    const float ax = fabsf(x);
    const float a = fminf(y, ax), b = fmaxf(y, ax);
    float rb;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rb) : "f"(b));
    const float r = a * rb, z = r * r;
    float p = -0.004668773151934147f;
    p = fmaf(p, z, 0.02416618913412094f);
    p = fmaf(p, z, -0.0593671016395092f);
    p = fmaf(p, z, 0.09906096756458282f);
    p = fmaf(p, z, -0.14016585052013397f);
    p = fmaf(p, z, 0.19969235360622406f);
    p = fmaf(p, z, -0.33331960439682007f);
    p = fmaf(p, z, 0.9999998807907104f);
    float t = p * r;
    t = y > ax ? 1.5707963267948966f - t : t;
    return x < 0.0f ? 3.1415926535897931f - t : t;
  }
};

template <> struct Fn<MODE_DS> : Fn<MODE_SP_INTRINSIC> {};
template <> struct Fn<MODE_HP> : Fn<MODE_SP_INTRINSIC> {};
template <int MODE> struct IsIntrinsic { static constexpr bool value = MODE == MODE_SP_INTRINSIC || MODE == MODE_DS || MODE == MODE_HP; };

__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }

// Run-time constants of a chain, in the arithmetic type of the mode.
template <typename R> struct ChainConst {
  R delta;     // R7 proposal half-width min(pi, 4 sqrt(T/(4 J q^2)))
  R inv_T;     // 1/T
  R hscale;    // float modes: q Delta / 2 = hscale (f - 3/2), f = prop_word in [1, 2): hscale = delta / 2
  R hoff;      //              = fma(f, hscale, hoff), hoff = -3/2 hscale
  R qhalf;     // q / 2 (double-arithmetic proposal: q Delta / 2 = qhalf * delta * (2 u1 - 1)); 1/4 for q = 1/2
  R bq_c, bq_s;  // general q only (GENQ): the end of the allowed arc, (cos 2 pi q, sin 2 pi q): phi <= 2 pi <=> u x b >= 0
  R xscale;    // log2(e) / T.  SP_INTRINSIC: exp(-dE / T) 2^20 = ex2(-dE * xscale + 20); double modes: metropolis_accept_exact
  uint32_t k0, k1, trial;
  int sc_terms;    // double modes: Taylor coefficients the proposal's sin / cos need at this delta (sincos_quarter_terms)
  PhiloxKeys rk;   // round keys of (k0, k1)
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

// ---- per-site energy term of S5 (R3, R13): sum over the existing neighbours j of cos[q(phi - phi_j)] ----
// Double arithmetic (DP, SP): u . F with F = sum_j u_j, as Eq. 2 reads in the unit-vector form.
// Float arithmetic (SP_PRECISE, SP_INTRINSIC): the same quantity per bond as 1 - |u - u_j|^2 / 2.
// u . u_j = |u||u_j| cos(theta) carries the norm error of the stored float vectors and the
// rounding of a value near 1 (measured on the B200: a constant +2.1e-8 .. +2.6e-8 in e at L = 16384,
// T = 1.1e-3, i.e. ~3 standard errors of e there), whereas |u - u_j|^2 = (|u|^2 + |u_j|^2)/2 x
// 2 (1 - cos(theta)) up to second order: the same errors now multiply the small thermal part only.
// A missing neighbour (open boundary, R2) and an out-of-grid padding site are the zero vector in
// both kernels; a real spin is never (0, 0).  Neighbour order l, r, u, d; the bond terms are float
// (the mode's arithmetic), the count is exact and the combination is done in double (R13).
template <typename R>
__device__ __forceinline__ double site_energy_term(R c, R s, R lc, R ls, R rc, R rs, R uc, R us, R dc, R ds) {
  if constexpr (sizeof(R) == 8) {
    const R A = ((lc + rc) + uc) + dc, B = ((ls + rs) + us) + ds;
    return static_cast<double>(fma_(c, A, s * B));
  } else {
    const R z = R(0);
    const bool me = (c != z) || (s != z);
    const bool hl = (lc != z) || (ls != z), hr = (rc != z) || (rs != z);
    const bool hu = (uc != z) || (us != z), hd = (dc != z) || (ds != z);
    R ec, es;
    ec = c - lc; es = s - ls; const R tl = fma_(ec, ec, es * es);
    ec = c - rc; es = s - rs; const R tr = fma_(ec, ec, es * es);
    ec = c - uc; es = s - us; const R tu = fma_(ec, ec, es * es);
    ec = c - dc; es = s - ds; const R td = fma_(ec, ec, es * es);
    R t = hl ? tl : z;
    t = t + (hr ? tr : z);
    t = t + (hu ? tu : z);
    t = t + (hd ? td : z);
    const int n = static_cast<int>(hl) + static_cast<int>(hr) + static_cast<int>(hu) + static_cast<int>(hd);
    return me ? static_cast<double>(n) - 0.5 * static_cast<double>(t) : 0.0;
  }
}

// ---- two-lane arithmetic -----------------------------------------------------------------
// Every move is written once, for TWO sites at a time (lanes a, b).  In the float modes the two
// lanes are the halves of one 64-bit register and every add / mul / fma is ONE packed sm_100
// instruction (add/mul/fma.rn.f32x2 -> SASS FADD2 / FMUL2 / FFMA2: half the issue slots of the
// scalar form, same IEEE round-to-nearest result per lane).  In the double modes a lane is a
// double and the ops are the scalar ones.  The PLAIN path calls the same functions with its one
// site in both lanes, which is what keeps PLAIN and TILED bit-identical.
template <typename R> struct Two;
template <> struct Two<double> { double a, b; };
template <> struct Two<float>  { unsigned long long v; };

__device__ __forceinline__ Two<double> mk2(double a, double b) { return Two<double>{a, b}; }
__device__ __forceinline__ Two<float> mk2(float a, float b) {
  Two<float> r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(a), "f"(b));
  return r;
}
__device__ __forceinline__ void un2(const Two<double>& x, double* a, double* b) { *a = x.a; *b = x.b; }
__device__ __forceinline__ void un2(const Two<float>& x, float* a, float* b) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(*a), "=f"(*b) : "l"(x.v));
}
__device__ __forceinline__ Two<double> add2(const Two<double>& x, const Two<double>& y) { return {x.a + y.a, x.b + y.b}; }
__device__ __forceinline__ Two<double> mul2(const Two<double>& x, const Two<double>& y) { return {x.a * y.a, x.b * y.b}; }
__device__ __forceinline__ Two<double> fma2(const Two<double>& x, const Two<double>& y, const Two<double>& z) {
  return {fma(x.a, y.a, z.a), fma(x.b, y.b, z.b)};
}
__device__ __forceinline__ Two<float> add2(const Two<float>& x, const Two<float>& y) {
  Two<float> r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(x.v), "l"(y.v));
  return r;
}
__device__ __forceinline__ Two<float> mul2(const Two<float>& x, const Two<float>& y) {
  Two<float> r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(x.v), "l"(y.v));
  return r;
}
__device__ __forceinline__ Two<float> fma2(const Two<float>& x, const Two<float>& y, const Two<float>& z) {
  Two<float> r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(x.v), "l"(y.v), "l"(z.v));
  return r;
}
template <typename R> __device__ __forceinline__ Two<R> bc2(R k) { return mk2(k, k); }

// Random words of the Metropolis move at a site (R9).  Double-arithmetic modes (DP, SP): one Philox block per
// site, counter word 0 = the site's row-major index; all four words are used (two 53-bit uniforms): the R9
// reading in full.  Float-arithmetic modes: one block per QUAD of sites of the same colour -- plane columns
// (2m, 2m + 1) in the rows (2k, 2k + 1); counter word 0 = the index of the site in row 2k, column 2m (quad_site);
// the sites take the words 0, 1 (row 2k: columns 2m, 2m + 1) and 2, 3 (row 2k + 1), one word each.
struct MetWords { uint32_t p, q, a, b; };   // proposal (p [, q]) and acceptance (a [, b]) words

// float modes: the four words of a quad
template <int MODE>
__device__ __forceinline__ uint4 met_words_quad(uint32_t quad_site, uint32_t sweep,
                                                const ChainConst<typename Traits<MODE>::real>& k) {
  return philox4x32_10(quad_site, sweep, PASS_MET, k.trial, k.rk);
}
// row_odd: the row of the two sites is 2k + 1.  pair_site = index of the first of the two sites in ITS row; the
// float modes derive the quad's key from it (the first site of the even row lies one row up and, the x-parity
// of a colour alternating from row to row, one column to the left or right).
template <int MODE>
__device__ __forceinline__ void met_words_pair(uint32_t pair_site, uint32_t sweep, uint32_t L, int par, bool row_odd,
                                               const ChainConst<typename Traits<MODE>::real>& k,
                                               MetWords* w0, MetWords* w1) {
  if constexpr (sizeof(typename Traits<MODE>::real) == 8) {
    const uint4 r0 = philox4x32_10(pair_site, sweep, PASS_MET, k.trial, k.rk);
    const uint4 r1 = philox4x32_10(pair_site + 2u, sweep, PASS_MET, k.trial, k.rk);
    *w0 = MetWords{r0.x, r0.y, r0.z, r0.w};
    *w1 = MetWords{r1.x, r1.y, r1.z, r1.w};
  } else {
    // even row: the pair's first site is the quad's key.  odd row: same plane columns one row up, where the
    // x-parity is the other one: x_even = x - par + (1 - par)
    const uint32_t quad_site = row_odd ? pair_site - L + 1u - 2u * static_cast<uint32_t>(par) : pair_site;
    const uint4 r = met_words_quad<MODE>(quad_site, sweep, k);
    const uint32_t wa = row_odd ? r.z : r.x, wb = row_odd ? r.w : r.y;
    *w0 = MetWords{wa, 0u, wa, 0u};
    *w1 = MetWords{wb, 0u, wb, 0u};
  }
}

// Metropolis move (R7, R10) of two sites at once, branch-free.  Lane x keeps its new spin iff the
// site is free, the proposal stays in range (s' >= 0) and the acceptance test passes; ok[x] tells.
//   sd = sin(q Delta/2), cd = cos(q Delta/2);  sin(q Delta) = 2 sd cd,  cos(q Delta) - 1 = -2 sd^2
//   u' = rot(q Delta) u;  P = u.F;  -Q = s A - c B;  dE = 2 sd (sd P - cd Q)
// GENQ: q < 1/2 (q in (0, 1/2]).  q phi then runs over [0, 2 pi q], an arc shorter than the half circle: besides
// s >= 0 (phi >= 0) a spin must satisfy u x b = c b_s - s b_c >= 0 (phi <= 2 pi), b the end of the arc.  For q = 1/2 that
// second test IS s >= 0, and the kernels of the fused paths are compiled without it.
template <int MODE, bool GENQ = false>
__device__ __forceinline__ void met_update2(Two<typename Traits<MODE>::real> c, Two<typename Traits<MODE>::real> s,
                                            Two<typename Traits<MODE>::real> A, Two<typename Traits<MODE>::real> B,
                                            const MetWords& wa, const MetWords& wb, bool free_a, bool free_b,
                                            const ChainConst<typename Traits<MODE>::real>& k,
                                            typename Traits<MODE>::real out[4] /* ca, cb, sa, sb */, bool ok[2]) {
  using R = typename Traits<MODE>::real;
  Two<R> h;                                      // q Delta / 2
  if constexpr (sizeof(R) == 8) {
    const R ta = fma_(R(2), R(u53(wa.p, wa.q)), R(-1));   // 2 u1 - 1 (exact)
    const R tb = fma_(R(2), R(u53(wb.p, wb.q)), R(-1));
    h = mul2(bc2(k.qhalf), mul2(bc2(k.delta), mk2(ta, tb)));
  } else {
    h = fma2(mk2(prop_word(wa.p), prop_word(wb.p)), bc2(k.hscale), bc2(k.hoff));
  }
  R ha, hb, sda, cda, sdb, cdb;
  un2(h, &ha, &hb);
  if constexpr (sizeof(R) == 8) {
    sincos_quarter_terms(ha, k.sc_terms, &sda, &cda);
    sincos_quarter_terms(hb, k.sc_terms, &sdb, &cdb);
  } else {
    Fn<MODE>::sincos_(ha, &sda, &cda);
    Fn<MODE>::sincos_(hb, &sdb, &cdb);
  }
  const Two<R> sd = mk2(sda, sdb), cd = mk2(cda, cdb);
  const Two<R> ts = add2(sd, sd);                // 2 sd
  const Two<R> nts = mul2(sd, bc2(R(-2)));       // -2 sd
  const Two<R> ps2 = mul2(ts, cd);               // sin(q Delta)
  const Two<R> ns2 = mul2(nts, cd);              // -sin(q Delta)
  const Two<R> c2m1 = mul2(nts, sd);             // cos(q Delta) - 1
  // u' - u = (rot(q Delta) - 1) u:  dc = c (cos - 1) - s sin,  ds = s (cos - 1) + c sin
  const Two<R> dc = fma2(c, c2m1, mul2(s, ns2));
  const Two<R> ds = fma2(s, c2m1, mul2(c, ps2));
  const Two<R> cn = add2(c, dc), sn = add2(s, ds);
  const Two<R> mdE = fma2(ds, B, mul2(dc, A));   // -dE = (u' - u) . F
  R c0a, c0b, s0a, s0b, cna, cnb, sna, snb;
  un2(c, &c0a, &c0b); un2(s, &s0a, &s0b); un2(cn, &cna, &cnb); un2(sn, &sna, &snb);
  bool acc_a, acc_b;
  if constexpr (sizeof(R) == 8) {
    R ea, eb;
    un2(mdE, &ea, &eb);
    acc_a = metropolis_accept_exact(wa.a, wa.b, ea, k.inv_T, k.xscale);
    acc_b = metropolis_accept_exact(wb.a, wb.b, eb, k.inv_T, k.xscale);
  } else if constexpr (IsIntrinsic<MODE>::value) {
    R xa, xb;                                    // exp(-dE/T) 2^20 = ex2(-dE xscale + 20): one FFMA2 + 2 MUFU.EX2
    un2(fma2(mdE, bc2(k.xscale), bc2(R(20))), &xa, &xb);
    acc_a = acc_word(wa.a) < Fn<MODE>::ex2_(xa);
    acc_b = acc_word(wb.a) < Fn<MODE>::ex2_(xb);
  } else {
    R xa, xb, ua, ub;
    un2(mul2(mdE, bc2(k.inv_T)), &xa, &xb);
    un2(mul2(mk2(acc_word(wa.a), acc_word(wb.a)), bc2(R(9.5367431640625e-07))), &ua, &ub);   // m 2^-20, exact
    acc_a = ua < Fn<MODE>::exp_(xa);
    acc_b = ub < Fn<MODE>::exp_(xb);
  }
  bool in_a = sna >= R(0), in_b = snb >= R(0);
  if constexpr (GENQ) {
    in_a = in_a && (fma_(cna, k.bq_s, -(sna * k.bq_c)) >= R(0));
    in_b = in_b && (fma_(cnb, k.bq_s, -(snb * k.bq_c)) >= R(0));
  }
  const bool oka = free_a && in_a && acc_a;
  const bool okb = free_b && in_b && acc_b;
  out[0] = oka ? cna : c0a; out[2] = oka ? sna : s0a;
  out[1] = okb ? cnb : c0b; out[3] = okb ? snb : s0b;
  ok[0] = oka; ok[1] = okb;
}

// Over-relaxation move (R5) of two sites at once: reflect u about the local field, u' = t F - u,
// t = 2 (u.F)/|F|^2; keep it iff the site is free, F != 0 and u' stays on the upper half circle.
// One Newton step towards |u'| = 1 stops the rounding drift of the norm.  Computed as
// m = u - t F = -u' and -f, so that no negation is needed: u' f = m (-f).
template <int MODE, bool GENQ = false>
__device__ __forceinline__ void or_update2(Two<typename Traits<MODE>::real> c, Two<typename Traits<MODE>::real> s,
                                           Two<typename Traits<MODE>::real> A, Two<typename Traits<MODE>::real> B,
                                           bool free_a, bool free_b,
                                           typename Traits<MODE>::real out[4] /* ca, cb, sa, sb */,
                                           const ChainConst<typename Traits<MODE>::real>* kq = nullptr) {
  using R = typename Traits<MODE>::real;
  const Two<R> F2 = fma2(A, A, mul2(B, B));
  const Two<R> P = fma2(c, A, mul2(s, B));
  const Two<R> nPP = mul2(P, bc2(R(-2)));
  R f2a, f2b, na, nb;
  un2(F2, &f2a, &f2b);
  un2(nPP, &na, &nb);
  const Two<R> nt = mk2(Fn<MODE>::div_(na, f2a), Fn<MODE>::div_(nb, f2b));   // -t
  const Two<R> mc = fma2(nt, A, c);              // -c'
  const Two<R> ms = fma2(nt, B, s);              // -s'
  const Two<R> nf = fma2(bc2(R(0.5)), fma2(mc, mc, mul2(ms, ms)), bc2(R(-1.5)));   // -(1.5 - |u'|^2 / 2)
  const Two<R> co = mul2(mc, nf), so = mul2(ms, nf);
  R c0a, c0b, s0a, s0b, msa, msb, coa, cob, soa, sob;
  un2(c, &c0a, &c0b); un2(s, &s0a, &s0b); un2(ms, &msa, &msb); un2(co, &coa, &cob); un2(so, &soa, &sob);
  // F = 0 (no field: nothing to reflect about) needs no test of its own: t = -2 P / 0 is inf or NaN, t F - u is NaN
  // (inf x 0), and NaN <= 0 is false -- the spin stays.  (void)f2a keeps the name for readers of the formula above.
  (void)f2a; (void)f2b;
  bool oka = free_a && (msa <= R(0));
  bool okb = free_b && (msb <= R(0));
  if constexpr (GENQ) {
    oka = oka && (fma_(coa, kq->bq_s, -(soa * kq->bq_c)) >= R(0));
    okb = okb && (fma_(cob, kq->bq_s, -(sob * kq->bq_c)) >= R(0));
  }
  out[0] = oka ? coa : c0a; out[2] = oka ? soa : s0a;
  out[1] = okb ? cob : c0b; out[3] = okb ? sob : s0b;
}

// Quench move (R8): the minimiser of the local energy, u = F/|F|.
template <int MODE, bool GENQ = false>
__device__ __forceinline__ void quench_update(typename Traits<MODE>::real* c, typename Traits<MODE>::real* s,
                                              typename Traits<MODE>::real A, typename Traits<MODE>::real B,
                                              const ChainConst<typename Traits<MODE>::real>* kq = nullptr) {
  using R = typename Traits<MODE>::real;
  const R R2 = fma_(A, A, B * B);
  if (R2 == R(0)) return;
  const R inv = Fn<MODE>::rsqrt_(R2);
  R cn = A * inv, sn = B * inv;
  if constexpr (GENQ) {                       // Phi / q > 2 pi: clipped to the end of the arc (R8)
    if (fma_(cn, kq->bq_s, -(sn * kq->bq_c)) < R(0)) { cn = kq->bq_c; sn = kq->bq_s; }
  }
  *c = cn; *s = sn;
}

// Quench move of two sites at once (same per-lane operations as quench_update).
template <int MODE>
__device__ __forceinline__ void quench_update2(Two<typename Traits<MODE>::real> c, Two<typename Traits<MODE>::real> s,
                                               Two<typename Traits<MODE>::real> A, Two<typename Traits<MODE>::real> B,
                                               bool free_a, bool free_b,
                                               typename Traits<MODE>::real out[4] /* ca, cb, sa, sb */) {
  using R = typename Traits<MODE>::real;
  R f2a, f2b, c0a, c0b, s0a, s0b, coa, cob, soa, sob;
  un2(fma2(A, A, mul2(B, B)), &f2a, &f2b);
  const Two<R> inv = mk2(Fn<MODE>::rsqrt_(f2a), Fn<MODE>::rsqrt_(f2b));
  un2(mul2(A, inv), &coa, &cob); un2(mul2(B, inv), &soa, &sob);
  un2(c, &c0a, &c0b); un2(s, &s0a, &s0b);
  const bool oka = free_a && (f2a != R(0)), okb = free_b && (f2b != R(0));
  out[0] = oka ? coa : c0a; out[2] = oka ? soa : s0a;
  out[1] = okb ? cob : c0b; out[3] = okb ? sob : s0b;
}

// phi = atan2(s, c) / q in [0, 2pi] (s >= 0); inv_q = 2 for q = 1/2.
template <int MODE>
__device__ __forceinline__ double spin_angle(typename Traits<MODE>::real c, typename Traits<MODE>::real s, double inv_q = 2.0) {
  return inv_q * static_cast<double>(Fn<MODE>::atan2_(s, c));
}

// Column pair of the left/right neighbours in the other colour plane: a site of colour col
// in row y sits at x = 2 j + ((y + col) & 1); its left neighbour is column j - 1 + par, its
// right neighbour column j + par, par = (y + col) & 1.
__device__ __forceinline__ int x_parity(int y, int col) { return (y + col) & 1; }

}  // namespace mpr
