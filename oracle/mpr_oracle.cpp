// oracle/mpr_oracle.cpp
//
// TEST INFRASTRUCTURE, NOT THE PRODUCT.  Plain, slow, single-file CPU statement of
// the MPR conditional hybrid Monte-Carlo prediction path of arxiv/paper_1910_08448
// (PAPER.md), in double precision throughout, with its own Philox4x32-10.  It shares
// no code, header, table or helper with the CUDA library (paper_1910_08448_b200/csrc);
// only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load it.
//
// What follows the paper and what is a reading of it (DESIGN.md section 3 lists every
// reading, R1..R17):
//   * Hamiltonian  H = -J sum_<ij> cos[q (phi_i - phi_j)],  phi in [0, 2pi],
//     q in (0, 1/2]                                  PAPER.md:27-29 (Eq. 2); q = 1/2, J = 1.
//   * "maps the measured data onto spins"            PAPER.md:13 (sec. 1)    -> orc_map  (R1)
//   * "temperature ... needs to be inferred from the incomplete data"
//                                                    PAPER.md:31 (sec. 2)    -> estimate (R6)
//   * "conditional Monte Carlo simulation, in which only the spins at the prediction
//     locations are allowed to change ... hybrid algorithm"
//                                                    PAPER.md:31 (sec. 2)    -> sweeps   (R4,R5,R7)
//   * "averaging over multiple configurations in equilibrium"
//                                                    PAPER.md:31 (sec. 2)    -> run      (R15)
//   * specific energy e = <H>/L^2                    PAPER.md:35 (sec. 2)    -> energy   (R3)
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): ground state e = -2J; i.i.d.-uniform
// e = -8J/pi^2; bond sum vs brute force; over-relaxation energy invariance and involution;
// single-site Metropolis and hybrid histograms vs the exact conditional density (chi^2);
// two-free-site system vs 2-D quadrature; T->0 limit; equipartition slope; Philox vs the
// CUDA toolkit's curand_Philox4x32_10 host path; mapping round trip.
// "parity unpinned" (no value in the paper to compare with): the T-matching procedure
// (R6), the quench initialisation (R8), open boundaries (R2), the prediction values / MAE.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fopenmp -shared -fPIC (oracle/mpr_oracle.py).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr double kQDefault = 0.5;   // PAPER.md:27, q in (0,1/2]; north_star fixes q = 1/2 (orc_set_q: any q of the range)
constexpr double kJ = 1.0;   // PAPER.md:27, exchange constant
// 2*pi rounded to double; the closed upper end of the spin range.
const double kTwoPi = 2.0 * 3.14159265358979323846264338327950288;

enum Status {
  OK = 0, ERR_INVALID_ARG = -1, ERR_NO_MEASURED = -2, ERR_DEGENERATE_RANGE = -3,
  ERR_NONFINITE = -4, ERR_WORKSPACE = -5, ERR_NOT_READY = -6, ERR_NO_ROOT = -7
};

enum PassId : uint32_t { PASS_INIT = 0, PASS_MET = 1 };

// ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), restated -----------------
// counter (c0..c3), key (k0,k1); 10 rounds; key bumped by the Weyl constants between
// rounds.  R9: counter = (site, sweep, pass, trial), key = (seed lo, seed hi).
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = static_cast<uint64_t>(M0) * c0;
    const uint64_t p1 = static_cast<uint64_t>(M1) * c2;
    const uint32_t hi0 = static_cast<uint32_t>(p0 >> 32), lo0 = static_cast<uint32_t>(p0);
    const uint32_t hi1 = static_cast<uint32_t>(p1 >> 32), lo1 = static_cast<uint32_t>(p1);
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// 53-bit uniform in [0,1) from two 32-bit words: 27 high bits of a, 26 high bits of b.
double u53(uint32_t a, uint32_t b) {
  const double hi = static_cast<double>(a >> 5);   // < 2^27
  const double lo = static_cast<double>(b >> 6);   // < 2^26
  return (hi * 67108864.0 + lo) * (1.0 / 9007199254740992.0);
}

struct Oracle {
  int L = 0;                    // columns (x)
  int H = 0;                    // rows (y); == L unless the grid is rectangular (orc_create_rect)
  std::vector<double> z;        // input values, row-major s = y*L + x
  std::vector<uint8_t> mask;    // 1 = prediction ("free") site, 0 = measured
  std::vector<double> phi;      // spins
  std::vector<double> acc;      // running sum of phi at free sites over measurement sweeps
  std::vector<double> series;   // e_n of the last run
  double zmin = 0.0, zmax = kTwoPi;
  uint64_t seed = 0;
  uint32_t trial = 0;
  uint64_t sweep = 0;           // hybrid sweeps done since the last chain reset
  uint64_t accepted = 0, attempted = 0;
  double T = -1.0;
  int n_quench = 32;            // R8
  double q = kQDefault;
  int schedule = 0;             // 0 = R4 (MET c0, MET c1, OR c0, OR c1), 1 = R4b site-fused (MET c0, OR c0, MET c1, OR c1)
  int threads = 1;
  long n_acc = 0;
  int est_trials = 0;

  size_t N() const { return static_cast<size_t>(L) * H; }
};

// Neighbour list of (x,y) in the fixed order left, right, up, down; open boundaries (R2).
inline int neighbours(int L, int H, int x, int y, size_t nb[4]) {
  int n = 0;
  const size_t s = static_cast<size_t>(y) * L + x;
  if (x > 0)     nb[n++] = s - 1;
  if (x < L - 1) nb[n++] = s + 1;
  if (y > 0)     nb[n++] = s - L;
  if (y < H - 1) nb[n++] = s + L;
  return n;
}

// E_loc(phi_s) = -J sum_j cos(q (phi_s - phi_j))  (the part of Eq. 2 that contains site s)
double local_energy(const Oracle& o, int x, int y, double phi_s) {
  size_t nb[4];
  const int n = neighbours(o.L, o.H, x, y, nb);
  double sum = 0.0;
  for (int k = 0; k < n; ++k) sum += std::cos(o.q * (phi_s - o.phi[nb[k]]));
  return -kJ * sum;
}

// R7: proposal half-width delta = min(pi, 4 sqrt(T / (4 J q^2))).
double proposal_width(double T, double q = kQDefault) {
  const double d = 4.0 * std::sqrt(T / (4.0 * kJ * q * q));
  const double pi = 0.5 * kTwoPi;
  return d < pi ? d : pi;
}

// O2 / R8 first half: free spins i.i.d. uniform on [0, 2pi) from Philox (pass = INIT).
void init_random(Oracle& o, uint32_t trial) {
  const uint32_t key[2] = {static_cast<uint32_t>(o.seed), static_cast<uint32_t>(o.seed >> 32)};
  const long long n = static_cast<long long>(o.N());
#pragma omp parallel for schedule(static) num_threads(o.threads)
  for (long long s = 0; s < n; ++s) {
    if (!o.mask[s]) continue;
    const uint32_t ctr[4] = {static_cast<uint32_t>(s), 0u, PASS_INIT, trial};
    uint32_t r[4];
    philox4x32_10(ctr, key, r);
    o.phi[s] = kTwoPi * u53(r[0], r[1]);
  }
}

// Metropolis pass over the free sites of colour c = (x+y)&1 at sweep n (O3 MET, R7, R10).
void met_pass(Oracle& o, int c, uint64_t n) {
  const int L = o.L;
  const double T = o.T, delta = proposal_width(o.T, o.q);
  const double kQ = o.q;
  const uint32_t key[2] = {static_cast<uint32_t>(o.seed), static_cast<uint32_t>(o.seed >> 32)};
  uint64_t acc = 0, att = 0;
#pragma omp parallel for schedule(static) reduction(+ : acc, att) num_threads(o.threads)
  for (int y = 0; y < o.H; ++y) {
    for (int x = (y + c) & 1; x < L; x += 2) {
      const size_t s = static_cast<size_t>(y) * L + x;
      if (!o.mask[s]) continue;
      const uint32_t ctr[4] = {static_cast<uint32_t>(s), static_cast<uint32_t>(n), PASS_MET, o.trial};
      uint32_t r[4];
      philox4x32_10(ctr, key, r);
      const double u1 = u53(r[0], r[1]);
      const double u2 = u53(r[2], r[3]);
      ++att;
      const double phi_old = o.phi[s];
      const double phi_new = phi_old + delta * (2.0 * u1 - 1.0);
      if (phi_new < 0.0 || phi_new > kTwoPi) continue;            // outside [0,2pi]: reject
      size_t nb[4];
      const int nn = neighbours(L, o.H, x, y, nb);
      double diff = 0.0;
      for (int k = 0; k < nn; ++k) {
        const double pj = o.phi[nb[k]];
        diff += std::cos(kQ * (phi_new - pj)) - std::cos(kQ * (phi_old - pj));
      }
      const double dE = -kJ * diff;
      if (dE <= 0.0 || u2 < std::exp(-dE / T)) {
        o.phi[s] = phi_new;
        ++acc;
      }
    }
  }
  o.accepted += acc;
  o.attempted += att;
}

// Neighbour field of a site: A = sum_j cos(q phi_j), B = sum_j sin(q phi_j).
inline void field(const Oracle& o, int x, int y, double& A, double& B) {
  size_t nb[4];
  const int nn = neighbours(o.L, o.H, x, y, nb);
  A = 0.0; B = 0.0;
  const double kQ = o.q;
  for (int k = 0; k < nn; ++k) {
    A += std::cos(kQ * o.phi[nb[k]]);
    B += std::sin(kQ * o.phi[nb[k]]);
  }
}

// Over-relaxation pass (O3 OR, R5): reflect q*phi about the local-field angle Phi;
// E_loc = -J R cos(q phi - Phi) is unchanged.  Out of [0,2pi] -> leave the spin alone.
void or_pass(Oracle& o, int c) {
  const int L = o.L;
  const double kQ = o.q;
#pragma omp parallel for schedule(static) num_threads(o.threads)
  for (int y = 0; y < o.H; ++y) {
    for (int x = (y + c) & 1; x < L; x += 2) {
      const size_t s = static_cast<size_t>(y) * L + x;
      if (!o.mask[s]) continue;
      double A, B;
      field(o, x, y, A, B);
      if (A == 0.0 && B == 0.0) continue;
      const double Phi = std::atan2(B, A);
      const double phi_new = (2.0 * Phi) / kQ - o.phi[s];
      if (phi_new >= 0.0 && phi_new <= kTwoPi) o.phi[s] = phi_new;
    }
  }
}

// Quench pass (R8 second half): put the spin at the minimum of its local energy,
// phi = Phi / q, clipped to [0, 2pi].  Deterministic; never raises H.
void quench_pass(Oracle& o, int c) {
  const int L = o.L;
  const double kQ = o.q;
#pragma omp parallel for schedule(static) num_threads(o.threads)
  for (int y = 0; y < o.H; ++y) {
    for (int x = (y + c) & 1; x < L; x += 2) {
      const size_t s = static_cast<size_t>(y) * L + x;
      if (!o.mask[s]) continue;
      double A, B;
      field(o, x, y, A, B);
      if (A == 0.0 && B == 0.0) continue;
      double phi_new = std::atan2(B, A) / kQ;
      if (phi_new < 0.0) phi_new = 0.0;
      if (phi_new > kTwoPi) phi_new = kTwoPi;
      o.phi[s] = phi_new;
    }
  }
}

// R4: one hybrid sweep = Metropolis colour 0, colour 1, then over-relaxation colour 0, 1.
// R4b (site-fused order): the same four passes as MET c0, OR c0, MET c1, OR c1.  Both moves of a site read only the
// other colour, so doing a colour's over-relaxation pass right after its Metropolis pass is the same as giving every
// site of the colour its Metropolis move and at once its over-relaxation move -- which is how the CUDA path runs it.
void hybrid_sweep(Oracle& o) {
  o.sweep += 1;
  if (o.schedule == 0) {
    met_pass(o, 0, o.sweep);
    met_pass(o, 1, o.sweep);
    or_pass(o, 0);
    or_pass(o, 1);
  } else {
    met_pass(o, 0, o.sweep);
    or_pass(o, 0);
    met_pass(o, 1, o.sweep);
    or_pass(o, 1);
  }
}

void reset_chain(Oracle& o, uint32_t trial) {
  o.trial = trial;
  o.sweep = 0;
  o.accepted = o.attempted = 0;
  init_random(o, trial);
  for (int k = 0; k < o.n_quench; ++k) { quench_pass(o, 0); quench_pass(o, 1); }
  std::fill(o.acc.begin(), o.acc.end(), 0.0);
  o.n_acc = 0;
  o.series.clear();
}

// H = -J sum over right and down bonds of cos(q (phi_s - phi_t)), open boundaries;
// e = 2 H / N_b with N_b = Lx (Ly - 1) + Ly (Lx - 1) bonds, 2 L (L-1) on the paper's square grid (R3).  Neumaier-compensated sum.
void energy(const Oracle& o, double* H_out, double* e_out) {
  const int L = o.L;
  const double kQ = o.q;
  double sum = 0.0, comp = 0.0;
  auto add = [&](double v) {
    const double t = sum + v;
    if (std::fabs(sum) >= std::fabs(v)) comp += (sum - t) + v; else comp += (v - t) + sum;
    sum = t;
  };
  for (int y = 0; y < o.H; ++y)
    for (int x = 0; x < L; ++x) {
      const size_t s = static_cast<size_t>(y) * L + x;
      if (x < L - 1) add(std::cos(kQ * (o.phi[s] - o.phi[s + 1])));
      if (y < o.H - 1) add(std::cos(kQ * (o.phi[s] - o.phi[s + L])));
    }
  const double H = -kJ * (sum + comp);
  const double nb = static_cast<double>(L) * (o.H - 1.0) + static_cast<double>(o.H) * (L - 1.0);   // 2 L (L - 1) on a square grid
  if (H_out) *H_out = H;
  if (e_out) *e_out = 2.0 * H / nb;
}

// O1: sample energy over nearest-neighbour pairs with both ends measured, same normalisation.
int sample_energy(const Oracle& o, double* es, long long* nsp) {
  const int L = o.L;
  const double kQ = o.q;
  double sum = 0.0;
  long long cnt = 0;
  for (int y = 0; y < o.H; ++y)
    for (int x = 0; x < L; ++x) {
      const size_t s = static_cast<size_t>(y) * L + x;
      if (o.mask[s]) continue;
      if (x < L - 1 && !o.mask[s + 1]) { sum += std::cos(kQ * (o.phi[s] - o.phi[s + 1])); ++cnt; }
      if (y < o.H - 1 && !o.mask[s + L]) { sum += std::cos(kQ * (o.phi[s] - o.phi[s + L])); ++cnt; }
    }
  if (nsp) *nsp = cnt;
  if (cnt == 0) return ERR_NO_MEASURED;
  if (es) *es = -2.0 * kJ * sum / static_cast<double>(cnt);
  return OK;
}

// Mean and binned standard error of a series (R16): 10 equal bins if n >= 20, else
// bins of one sample; unbiased variance of the bin means / number of bins.
void mean_stderr(const std::vector<double>& v, double* mean, double* se) {
  const size_t n = v.size();
  double m = 0.0;
  for (double x : v) m += x;
  m = n ? m / static_cast<double>(n) : std::numeric_limits<double>::quiet_NaN();
  double s = 0.0;
  if (n >= 2) {
    const size_t nb = n >= 20 ? 10 : n;
    const size_t len = n / nb;
    std::vector<double> bm(nb, 0.0);
    double bmean = 0.0;
    for (size_t b = 0; b < nb; ++b) {
      for (size_t k = 0; k < len; ++k) bm[b] += v[b * len + k];
      bm[b] /= static_cast<double>(len);
      bmean += bm[b];
    }
    bmean /= static_cast<double>(nb);
    double var = 0.0;
    for (size_t b = 0; b < nb; ++b) var += (bm[b] - bmean) * (bm[b] - bmean);
    var /= static_cast<double>(nb - 1);
    s = std::sqrt(var / static_cast<double>(nb));
  }
  if (mean) *mean = m;
  if (se) *se = s;
}

// n_eq equilibration sweeps, then n_meas sweeps each followed by O4 (energy sample and
// accumulation of phi at the free sites).  Continues the current chain.
void run_sweeps(Oracle& o, int n_eq, int n_meas) {
  for (int k = 0; k < n_eq; ++k) hybrid_sweep(o);
  o.series.clear();
  for (int k = 0; k < n_meas; ++k) {
    hybrid_sweep(o);
    double e;
    energy(o, nullptr, &e);
    o.series.push_back(e);
    for (size_t s = 0; s < o.N(); ++s)
      if (o.mask[s]) o.acc[s] += o.phi[s];
    o.n_acc += 1;
  }
}

constexpr int kTrialEq = 200, kTrialMeas = 50, kMaxIllinois = 20;

// One temperature trial of R6: fresh chain (trial index in the Philox counter), short run.
void trial_energy(Oracle& o, double T, double* e, double* se) {
  o.est_trials += 1;
  o.T = T;
  reset_chain(o, static_cast<uint32_t>(o.est_trials));
  run_sweeps(o, kTrialEq, kTrialMeas);
  mean_stderr(o.series, e, se);
}

// R6: conditional energy matching.  Find T with e_cond(T) = e_s by bracketing on
// [1e-4, 1] (expanded by decades within [1e-6, 1e2]) and Illinois regula falsi.
// `trial(T, &e, &se)` runs one temperature trial; the search itself never looks at the chain,
// so a test can hand it a synthetic e(T) (orc_debug_match_temperature) and follow the
// iterates by hand.
template <typename Trial>
int match_temperature(double es, Trial&& trial, double* T_hat) {
  double T_lo = 1e-4, T_hi = 1.0, g_lo, g_hi, e, se;
  bool have_hi = false;
  trial(T_lo, &e, &se);
  g_lo = e - es;
  while (g_lo > 0.0) {
    if (T_lo <= 1.5e-6) return ERR_NO_ROOT;
    T_hi = T_lo; g_hi = g_lo; have_hi = true;
    T_lo /= 10.0;
    trial(T_lo, &e, &se);
    g_lo = e - es;
  }
  if (!have_hi) {
    trial(T_hi, &e, &se);
    g_hi = e - es;
    while (g_hi < 0.0) {
      if (T_hi >= 0.99e2) return ERR_NO_ROOT;
      T_lo = T_hi; g_lo = g_hi;
      T_hi *= 10.0;
      trial(T_hi, &e, &se);
      g_hi = e - es;
    }
  }
  double T_new = T_hi, T_prev = T_hi;
  int last_side = 0;   // -1: last replaced lo, +1: last replaced hi
  for (int it = 0; it < kMaxIllinois; ++it) {
    T_new = T_hi - g_hi * (T_hi - T_lo) / (g_hi - g_lo);
    if (!(T_new > T_lo && T_new < T_hi)) T_new = 0.5 * (T_lo + T_hi);
    trial(T_new, &e, &se);
    const double g = e - es;
    if (std::fabs(g) <= 2.0 * se) break;
    if (g < 0.0) {
      T_lo = T_new; g_lo = g;
      if (last_side == -1) g_hi *= 0.5;
      last_side = -1;
    } else {
      T_hi = T_new; g_hi = g;
      if (last_side == +1) g_lo *= 0.5;
      last_side = +1;
    }
    if (it > 0 && std::fabs(T_new - T_prev) / T_new < 0.01) break;
    T_prev = T_new;
  }
  if (T_hat) *T_hat = T_new;
  return OK;
}

int estimate_temperature(Oracle& o, double* T_hat, double* e_sample) {
  double es = 0.0;
  long long nsp = 0;
  const int st = sample_energy(o, &es, &nsp);
  if (st != OK) return st;
  if (e_sample) *e_sample = es;
  o.est_trials = 0;
  double T_found = 0.0;
  const int sr = match_temperature(es, [&](double T, double* e, double* se) { trial_energy(o, T, e, se); }, &T_found);
  if (sr != OK) return sr;
  o.T = T_found;
  reset_chain(o, 0);
  if (T_hat) *T_hat = T_found;
  return OK;
}

}  // namespace

extern "C" {

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  philox4x32_10(ctr, key, out);
}
double orc_u53(uint32_t a, uint32_t b) { return u53(a, b); }
double orc_proposal_width(double T) { return proposal_width(T); }
double orc_proposal_width_q(double T, double q) { return proposal_width(T, q); }
void orc_mean_stderr(const double* v, long n, double* mean, double* se) {
  std::vector<double> w(v, v + n);
  mean_stderr(w, mean, se);
}

// O0 (R1): phi = 2pi (z - zmin)/(zmax - zmin), min/max over the measured sample.
// mask[s] = 1 -> prediction site (value never read).  Returns a handle or null + status.
static void* create_impl(int L, int H, const double* values, const uint8_t* mask, int* status, bool reset);
void* orc_create(int L, const double* values, const uint8_t* mask, int* status) {
  return create_impl(L, L, values, mask, status, true);
}
// Rectangular grid of Lx columns and Ly rows (row-major, s = y Lx + x): nothing in the method depends on the
// grid being square (nearest neighbours on a regular grid); only the bond count of R3 changes.
void* orc_create_rect(int Lx, int Ly, const double* values, const uint8_t* mask, int* status) {
  return create_impl(Lx, Ly, values, mask, status, true);
}
void* orc_create_rect_deferred(int Lx, int Ly, const double* values, const uint8_t* mask, int* status) {
  return create_impl(Lx, Ly, values, mask, status, false);
}
// Same map, but the chain is NOT initialised: the caller sets threads / seed / quench count first and
// then calls orc_configure, so that a large grid pays for one R8 initialisation (on all threads)
// instead of three single-threaded ones.
void* orc_create_deferred(int L, const double* values, const uint8_t* mask, int* status) {
  return create_impl(L, L, values, mask, status, false);
}
static void* create_impl(int L, int H, const double* values, const uint8_t* mask, int* status, bool reset) {
  auto fail = [&](int code) -> void* { if (status) *status = code; return nullptr; };
  if (L < 1 || H < 1 || static_cast<long long>(L) * H < 2 || (L == H && L < 2) || !values || !mask) return fail(ERR_INVALID_ARG);
  Oracle* o = new Oracle;
  o->L = L; o->H = H;
  const size_t N = o->N();
  o->z.assign(values, values + N);
  o->mask.assign(mask, mask + N);
  o->phi.assign(N, 0.0);
  o->acc.assign(N, 0.0);
  double zmin = std::numeric_limits<double>::infinity(), zmax = -zmin;
  size_t n_meas = 0;
  for (size_t s = 0; s < N; ++s) {
    if (mask[s]) continue;
    if (!std::isfinite(values[s])) { delete o; return fail(ERR_NONFINITE); }
    ++n_meas;
    if (values[s] < zmin) zmin = values[s];
    if (values[s] > zmax) zmax = values[s];
  }
  if (n_meas == 0) { delete o; return fail(ERR_NO_MEASURED); }
  if (!(zmax > zmin)) { delete o; return fail(ERR_DEGENERATE_RANGE); }
  o->zmin = zmin; o->zmax = zmax;
  for (size_t s = 0; s < N; ++s)
    if (!mask[s]) o->phi[s] = kTwoPi * ((values[s] - zmin) / (zmax - zmin));
  if (reset) reset_chain(*o, 0);
  if (status) *status = OK;
  return o;
}

// Pins only: take the spins as given (identity map, zmin = 0, zmax = 2pi); no chain reset.
void* orc_create_from_phi_rect(int L, int H, const double* phi, const uint8_t* mask);
void* orc_create_from_phi(int L, const double* phi, const uint8_t* mask) {
  if (L < 2) return nullptr;
  return orc_create_from_phi_rect(L, L, phi, mask);
}
void* orc_create_from_phi_rect(int L, int H, const double* phi, const uint8_t* mask) {
  if (L < 1 || H < 1 || static_cast<long long>(L) * H < 2 || !phi || !mask) return nullptr;
  Oracle* o = new Oracle;
  o->L = L; o->H = H;
  const size_t N = o->N();
  o->z.assign(phi, phi + N);
  o->mask.assign(mask, mask + N);
  o->phi.assign(phi, phi + N);
  o->acc.assign(N, 0.0);
  o->zmin = 0.0; o->zmax = kTwoPi;
  return o;
}

void orc_destroy(void* h) { delete static_cast<Oracle*>(h); }

int orc_set_seed(void* h, uint64_t seed) {
  Oracle& o = *static_cast<Oracle*>(h);
  o.seed = seed;
  reset_chain(o, 0);
  return OK;
}
int orc_set_temperature(void* h, double T) {
  if (!(T > 0.0) || !std::isfinite(T)) return ERR_INVALID_ARG;
  static_cast<Oracle*>(h)->T = T;
  return OK;
}
int orc_set_quench(void* h, int n) {
  if (n < 0) return ERR_INVALID_ARG;
  Oracle& o = *static_cast<Oracle*>(h);
  o.n_quench = n;
  reset_chain(o, 0);
  return OK;
}
int orc_configure(void* h, uint64_t seed, int n_quench) {
  if (n_quench < 0) return ERR_INVALID_ARG;
  Oracle& o = *static_cast<Oracle*>(h);
  o.seed = seed;
  o.n_quench = n_quench;
  reset_chain(o, 0);
  return OK;
}
// q in (0, 1/2].  The spins (angles) do not depend on q; the chain is restarted.
int orc_set_q(void* h, double q) {
  if (!(q > 0.0) || q > 0.5) return ERR_INVALID_ARG;
  Oracle& o = *static_cast<Oracle*>(h);
  o.q = q;
  reset_chain(o, 0);
  return OK;
}
int orc_set_schedule(void* h, int schedule) {
  if (schedule != 0 && schedule != 1) return ERR_INVALID_ARG;
  static_cast<Oracle*>(h)->schedule = schedule;
  return OK;
}
int orc_set_threads(void* h, int n) {
  if (n < 1) return ERR_INVALID_ARG;
  static_cast<Oracle*>(h)->threads = n;
  return OK;
}
int orc_threads_available(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_reset_chain(void* h, uint32_t trial) { reset_chain(*static_cast<Oracle*>(h), trial); }
void orc_init_random(void* h, uint32_t trial) {
  Oracle& o = *static_cast<Oracle*>(h);
  o.trial = trial;
  init_random(o, trial);
}
void orc_get_range(void* h, double* zmin, double* zmax) {
  Oracle& o = *static_cast<Oracle*>(h);
  *zmin = o.zmin; *zmax = o.zmax;
}

int orc_met_pass(void* h, int c, uint64_t n) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (!(o.T > 0.0)) return ERR_NOT_READY;
  met_pass(o, c & 1, n);
  return OK;
}
void orc_or_pass(void* h, int c) { or_pass(*static_cast<Oracle*>(h), c & 1); }
void orc_quench_pass(void* h, int c) { quench_pass(*static_cast<Oracle*>(h), c & 1); }
int orc_hybrid_sweeps(void* h, int n) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (!(o.T > 0.0)) return ERR_NOT_READY;
  for (int k = 0; k < n; ++k) hybrid_sweep(o);
  return OK;
}

// Pins: run n sweeps and record phi at the listed sites after every sweep.
// kind 0: Metropolis-only sweeps (colour 0 then 1); kind 1: hybrid sweeps.
int orc_trace(void* h, long n, int kind, const int64_t* sites, int n_sites, double* out) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (!(o.T > 0.0)) return ERR_NOT_READY;
  for (long k = 0; k < n; ++k) {
    if (kind == 0) {
      o.sweep += 1;
      met_pass(o, 0, o.sweep);
      met_pass(o, 1, o.sweep);
    } else {
      hybrid_sweep(o);
    }
    for (int i = 0; i < n_sites; ++i) out[k * n_sites + i] = o.phi[sites[i]];
  }
  return OK;
}

// Pins: run n hybrid sweeps and record e after every sweep.
int orc_trace_energy(void* h, long n, double* out) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (!(o.T > 0.0)) return ERR_NOT_READY;
  for (long k = 0; k < n; ++k) {
    hybrid_sweep(o);
    energy(o, nullptr, &out[k]);
  }
  return OK;
}

void orc_energy(void* h, double* H, double* e) { energy(*static_cast<Oracle*>(h), H, e); }
int orc_sample_energy(void* h, double* es, long long* nsp) {
  return sample_energy(*static_cast<Oracle*>(h), es, nsp);
}
double orc_local_energy(void* h, int x, int y, double phi_s) {
  return local_energy(*static_cast<Oracle*>(h), x, y, phi_s);
}

void orc_get_state(void* h, double* phi) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(phi, o.phi.data(), o.N() * sizeof(double));
}
void orc_set_state(void* h, const double* phi) {
  Oracle& o = *static_cast<Oracle*>(h);
  std::memcpy(o.phi.data(), phi, o.N() * sizeof(double));
}
void orc_get_counters(void* h, uint64_t* accepted, uint64_t* attempted, uint64_t* sweep) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (accepted) *accepted = o.accepted;
  if (attempted) *attempted = o.attempted;
  if (sweep) *sweep = o.sweep;
}

// O3-O5: continue the chain for n_eq + n_meas hybrid sweeps; prediction = back-mapped mean
// of phi over all measurement sweeps since the last chain reset; measured sites return
// their input value.  e_mean / e_stderr over this call's n_meas energies.
int orc_run(void* h, int n_eq, int n_meas, double* pred, double* e_mean, double* e_stderr) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (n_eq < 0 || n_meas < 0) return ERR_INVALID_ARG;
  if (!(o.T > 0.0)) return ERR_NOT_READY;
  run_sweeps(o, n_eq, n_meas);
  mean_stderr(o.series, e_mean, e_stderr);
  if (pred) {
    for (size_t s = 0; s < o.N(); ++s) {
      if (!o.mask[s]) { pred[s] = o.z[s]; continue; }
      if (o.n_acc == 0) { pred[s] = std::numeric_limits<double>::quiet_NaN(); continue; }
      const double frac = o.acc[s] / (kTwoPi * static_cast<double>(o.n_acc));
      pred[s] = o.zmin + (o.zmax - o.zmin) * frac;
    }
  }
  return OK;
}
long orc_get_series(void* h, double* out, long cap) {
  Oracle& o = *static_cast<Oracle*>(h);
  const long n = static_cast<long>(o.series.size());
  for (long k = 0; k < n && k < cap; ++k) out[k] = o.series[k];
  return n;
}

int orc_estimate_temperature(void* h, double* T_hat, double* e_sample, int* n_trials) {
  Oracle& o = *static_cast<Oracle*>(h);
  const int st = estimate_temperature(o, T_hat, e_sample);
  if (n_trials) *n_trials = o.est_trials;
  return st;
}

// Pins: the R6 search on a caller-supplied e(T) (no chain involved).  trial(T, index, &e, &se, user).
int orc_debug_match_temperature(double e_sample, int (*trial)(double, int, double*, double*, void*), void* user,
                                double* T_hat, int* n_trials) {
  int n = 0;
  const int st = match_temperature(e_sample, [&](double T, double* e, double* se) { trial(T, ++n, e, se, user); }, T_hat);
  if (n_trials) *n_trials = n;
  return st;
}

// One temperature trial exactly as the estimator runs it (for the monotonicity pin).
int orc_trial_energy(void* h, double T, int trial_index, double* e, double* se) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (!(T > 0.0)) return ERR_INVALID_ARG;
  o.est_trials = trial_index - 1;
  trial_energy(o, T, e, se);
  return OK;
}

}  // extern "C"
