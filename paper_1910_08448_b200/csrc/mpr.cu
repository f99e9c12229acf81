// mpr.cu -- host side of libmpr.so: the C ABI declared in include/mpr.h, workspace carving,
// launch logic of both kernel paths, the temperature-matching loop (R6) and the binned error
// (R16).  No torch types, no device allocation, no CPU fallback.
#include "../../include/mpr.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <new>
#include <string>
#include <vector>

#include <cuda.h>
#include <cuda_runtime.h>

#include "mpr_device.cuh"
#include "mpr_host_math.hpp"
#include "mpr_plain.cuh"
#include "mpr_tiled.cuh"
#include "mpr_strip.cuh"

using namespace mpr;

namespace {

constexpr double kQDefault = 0.5;   // PAPER.md:27, q in (0, 1/2]; north_star fixes q = 1/2 (mpr_set_q: any q of the range)
constexpr double kJ = 1.0;
constexpr int kMaxL = 32768;
constexpr int kPartials = 1 << 18;       // doubles
constexpr int kSeriesCap = 1 << 16;      // energy samples per mpr_run
constexpr int kAcceptSlots = 1024;
constexpr int kTrialEq = 200, kTrialMeas = 50;   // R6: sweeps of one temperature trial

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
// N_b of R3: nearest-neighbour bonds of an open L x H grid, 2 L (L - 1) on the paper's square one
// the side of the square grid with as many sites (what the AUTO thresholds, tuned on square grids, go by)
double grid_side(const Geom& g) { return std::sqrt(static_cast<double>(g.L) * g.H); }
double bond_count(const Geom& g) {
  return static_cast<double>(g.L) * (g.H - 1.0) + static_cast<double>(g.H) * (g.L - 1.0);
}

struct Layout {
  Geom g;
  size_t off_state[2], off_acc, off_bits, off_smask[2], off_list[2], off_rows, off_part, off_series, off_slots, off_scal, total;
};

Layout make_layout(int L, int H) {      // L columns, H rows
  Layout lo;
  lo.g.L = L;
  lo.g.H = H;
  lo.g.site0 = 0u;
  lo.g.own0 = 0;
  lo.g.own1 = H;
  lo.g.peer_rows = 0;
  lo.g.peer_dst[0] = lo.g.peer_dst[1] = nullptr;
  lo.g.peer_plane[0] = lo.g.peer_plane[1] = 0;
  lo.g.peer_row_off[0] = lo.g.peer_row_off[1] = 0;
  lo.g.Wp = static_cast<int>(align_up(static_cast<size_t>((L + 1) / 2), 16));
  lo.g.Wm = (lo.g.Wp + 31) / 32;
  lo.g.Wb = lo.g.Wm + kBitPadLeft + kBitPadRight;
  lo.g.Hb = H + kBitPadTop + kBitPadBot;
  lo.g.plane = static_cast<size_t>(H) * lo.g.Wp;
  lo.g.energy_single = 0;
  lo.g.q = kQDefault;
  size_t o = 0;
  const size_t state_bytes = 2 * lo.g.plane * sizeof(double2);
  lo.off_state[0] = o; o = align_up(o + state_bytes, 256);
  lo.off_state[1] = o; o = align_up(o + state_bytes, 256);
  lo.off_acc = o;      o = align_up(o + 2 * lo.g.plane * sizeof(double), 256);
  lo.off_bits = o;     o = align_up(o + static_cast<size_t>(2) * lo.g.Hb * lo.g.Wb * sizeof(uint32_t), 256);
  for (int hl = 1; hl <= 2; ++hl) {
    lo.off_smask[hl - 1] = o;
    o = align_up(o + strip_mask_words(lo.g, hl) * sizeof(uint32_t), 256);
  }
  for (int col = 0; col < 2; ++col) {                 // compacted prediction-site lists (LIST path), worst case: all free
    lo.off_list[col] = o;
    o = align_up(o + lo.g.plane * sizeof(uint32_t), 256);
  }
  lo.off_rows = o;     o = align_up(o + static_cast<size_t>(4) * H * sizeof(uint32_t) + 64, 256);   // row counts, offsets, totals
  lo.off_part = o;     o = align_up(o + kPartials * sizeof(double), 256);
  lo.off_series = o;   o = align_up(o + kSeriesCap * sizeof(double), 256);
  lo.off_slots = o;    o = align_up(o + kAcceptSlots * sizeof(unsigned long long), 256);
  lo.off_scal = o;     o = align_up(o + 64 * sizeof(double), 256);
  lo.total = o;
  return lo;
}

}  // namespace

struct mpr_ctx {
  Layout lo;
  const double* d_values = nullptr;
  const uint8_t* d_mask = nullptr;
  char* ws = nullptr;
  cudaStream_t stream = nullptr;
  int mode = MPR_DP;
  int path = MPR_PATH_AUTO;
  int schedule = MPR_SCHEDULE_R4;
  int fused = 0;               // hybrid sweeps per launch; 0 = chosen by auto_fused()
  int n_quench = 32;
  uint64_t seed = 0;
  uint32_t trial = 0;
  uint64_t sweep = 0;
  uint64_t attempted = 0;
  long long n_acc = 0;
  int cur = 0;                 // which state buffer holds the chain
  // timing of the equilibration phase of the last mpr_run (mpr_get_run_timing): two events on the
  // ctx stream, created on first use, destroyed with the ctx
  cudaEvent_t ev_eq[2] = {nullptr, nullptr};
  double last_eq_ms = -1.0;
  long long last_eq_launches = 0, last_eq_sweeps = 0;
  double T = -1.0;
  double zmin = 0.0, zmax = 0.0;
  double e_sample = 0.0;
  long long n_pairs = 0;
  long long n_free = 0;          // prediction sites of the rows that count (all rows; a slab: its own rows)
  double pair_sum = 0.0;         // sum of cos over the measured pairs behind e_sample (mpr_sample_energy_parts)
  double nb_norm = 0.0;          // bonds the energy is normalised by: bond_count(g), or the whole grid's for a slab
  bool slab = false;
  bool expect_slab = false;    // created by mpr_create_slab: unusable until mpr_set_slab, local sample may be empty / constant
  // peer mode (mpr_set_peers): the neighbour slabs' contexts (same process) and the number of strip launches made so
  // far, by which a launch finds the buffer its neighbour's launch of the same number writes
  mpr_ctx* peer[2] = {nullptr, nullptr};
  int slab_row0 = 0;           // global row of local row 0 (mpr_set_slab)
  long long strip_epoch = 0;
  uint32_t n_list[2] = {0u, 0u};     // prediction sites per colour (lengths of the LIST path's lists)
  uint64_t launches = 0;
  std::vector<double> series;
  bool stale = true;     // the chain has to be (re)initialised before its next use (ensure_chain)
  std::string err;
  TiledPlan tiled;
  StripPlan strip;

  void* state(int b) const { return ws + lo.off_state[b]; }
  double* acc() const { return reinterpret_cast<double*>(ws + lo.off_acc); }
  uint32_t* bits_base() const { return reinterpret_cast<uint32_t*>(ws + lo.off_bits); }
  // word 0 of row 0 of colour 0 inside the padded bitmaps (mpr_plain.cuh)
  uint32_t* bits() const { return bits_base() + static_cast<size_t>(kBitPadTop) * lo.g.Wb + kBitPadLeft; }
  uint32_t* list(int col) const { return reinterpret_cast<uint32_t*>(ws + lo.off_list[col]); }
  uint32_t* rows() const { return reinterpret_cast<uint32_t*>(ws + lo.off_rows); }
  uint32_t* smask(int hl) const { return reinterpret_cast<uint32_t*>(ws + lo.off_smask[hl - 1]); }
  double* part() const { return reinterpret_cast<double*>(ws + lo.off_part); }
  double* dseries() const { return reinterpret_cast<double*>(ws + lo.off_series); }
  unsigned long long* slots() const { return reinterpret_cast<unsigned long long*>(ws + lo.off_slots); }
  double* scal() const { return reinterpret_cast<double*>(ws + lo.off_scal); }
};

namespace {

int fail(mpr_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}
#define CUDA_OK(ctx, expr)                                                                         \
  do {                                                                                             \
    cudaError_t e_ = (expr);                                                                       \
    if (e_ != cudaSuccess)                                                                         \
      return fail(ctx, MPR_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));          \
  } while (0)
#define LAUNCH_OK(ctx)                                                                             \
  do {                                                                                             \
    (ctx)->launches += 1;                                                                          \
    cudaError_t e_ = cudaGetLastError();                                                           \
    if (e_ != cudaSuccess) return fail(ctx, MPR_ERR_CUDA, std::string("launch: ") + cudaGetErrorString(e_)); \
  } while (0)
#define TRY(expr)                                                                                  \
  do {                                                                                             \
    int st_ = (expr);                                                                              \
    if (st_ != MPR_OK) return st_;                                                                 \
  } while (0)

// R7: proposal half-width delta = min(pi, 4 sqrt(T / (4 J q^2))).
double proposal_width(double T, double q = kQDefault) {
  const double d = 4.0 * std::sqrt(T / (4.0 * kJ * q * q));
  const double pi = 3.14159265358979323846264338327950288;
  return d < pi ? d : pi;
}

template <typename R>
ChainConst<R> chain_const(const mpr_ctx* c) {
  ChainConst<R> k;
  const double T = c->T > 0.0 ? c->T : 1.0;
  const double q = c->lo.g.q;
  k.delta = static_cast<R>(proposal_width(T, q));
  k.qhalf = static_cast<R>(0.5 * q);
  k.bq_c = static_cast<R>(std::cos(6.283185307179586476925286766559 * q));
  k.bq_s = static_cast<R>(std::sin(6.283185307179586476925286766559 * q));
  k.inv_T = static_cast<R>(1.0 / T);
  k.hscale = static_cast<R>(q * proposal_width(T, q));      // q Delta / 2 = q delta (f - 3/2)
  if (sizeof(R) == 4) {
    // the two lowest mantissa bits cleared: 3/2 hscale is then exact in float and the 4096 proposal offsets
    // fma(f, hscale, hoff) are exactly symmetric about 0 (delta itself is a free parameter, R7)
    float hs = static_cast<float>(k.hscale);
    uint32_t bits;
    std::memcpy(&bits, &hs, sizeof(bits));
    bits &= ~3u;
    std::memcpy(&hs, &bits, sizeof(bits));
    k.hscale = static_cast<R>(hs);
  }
  k.hoff = static_cast<R>(-1.5) * k.hscale;
  k.xscale = static_cast<R>(1.4426950408889634074 / T);
  k.sc_terms = sincos_terms_for(0.5 * q * proposal_width(T, q));      // |q Delta / 2| <= q delta / 2
  k.k0 = static_cast<uint32_t>(c->seed);
  k.k1 = static_cast<uint32_t>(c->seed >> 32);
  k.trial = c->trial;
  for (int r = 0; r < 10; ++r) {
    k.rk.a[r] = k.k0 + static_cast<uint32_t>(r) * 0x9E3779B9u;
    k.rk.b[r] = k.k1 + static_cast<uint32_t>(r) * 0xBB67AE85u;
  }
  return k;
}

// Mean and binned standard error of a series (R16): mpr_host_math.hpp.
void mean_stderr(const std::vector<double>& v, double* mean, double* se) {
  const mpr_host::SeriesStats st = mpr_host::series_stats(v.data(), v.size());
  if (mean) *mean = st.mean;
  if (se) *se = st.stderr_;
}

// ---- mode dispatch ---------------------------------------------------------------------------
template <int MODE, bool GENQ> int plain_pass_q(mpr_ctx* c, int kind, int col, uint64_t sweep) {
  using R = typename Traits<MODE>::real;
  using V = typename Traits<MODE>::vec;
  const Geom& g = c->lo.g;
  dim3 block(128), grid((g.Wp + 127) / 128, g.H);
  V* st = static_cast<V*>(c->state(c->cur));
  const ChainConst<R> k = chain_const<R>(c);
  const uint32_t sw = static_cast<uint32_t>(sweep);
  if (kind == KIND_MET)
    plain_pass_kernel<MODE, KIND_MET, GENQ><<<grid, block, 0, c->stream>>>(st, c->bits(), g, col, sw, k, c->slots());
  else if (kind == KIND_MO)
    plain_pass_kernel<MODE, KIND_MO, GENQ><<<grid, block, 0, c->stream>>>(st, c->bits(), g, col, sw, k, c->slots());
  else if (kind == KIND_OR)
    plain_pass_kernel<MODE, KIND_OR, GENQ><<<grid, block, 0, c->stream>>>(st, c->bits(), g, col, sw, k, c->slots());
  else
    plain_pass_kernel<MODE, KIND_QUENCH, GENQ><<<grid, block, 0, c->stream>>>(st, c->bits(), g, col, sw, k, c->slots());
  LAUNCH_OK(c);
  return MPR_OK;
}
// q = 1/2 (the default) runs the kernels without the second range test; any other q the general ones
template <int MODE> int plain_pass(mpr_ctx* c, int kind, int col, uint64_t sweep) {
  return c->lo.g.q == kQDefault ? plain_pass_q<MODE, false>(c, kind, col, sweep) : plain_pass_q<MODE, true>(c, kind, col, sweep);
}

template <int MODE, bool GENQ> int list_pass_q(mpr_ctx* c, int kind, int col, uint64_t sweep) {
  using R = typename Traits<MODE>::real;
  using V = typename Traits<MODE>::vec;
  const Geom& g = c->lo.g;
  const uint32_t n = c->n_list[col];
  if (n == 0) return MPR_OK;
  const unsigned grid = (n + 127u) / 128u;
  V* st = static_cast<V*>(c->state(c->cur));
  const ChainConst<R> k = chain_const<R>(c);
  const uint32_t sw = static_cast<uint32_t>(sweep);
  if (kind == KIND_MET)
    list_pass_kernel<MODE, KIND_MET, GENQ><<<grid, 128, 0, c->stream>>>(st, c->list(col), n, g, col, sw, k, c->slots());
  else if (kind == KIND_MO)
    list_pass_kernel<MODE, KIND_MO, GENQ><<<grid, 128, 0, c->stream>>>(st, c->list(col), n, g, col, sw, k, c->slots());
  else if (kind == KIND_OR)
    list_pass_kernel<MODE, KIND_OR, GENQ><<<grid, 128, 0, c->stream>>>(st, c->list(col), n, g, col, sw, k, c->slots());
  else
    list_pass_kernel<MODE, KIND_QUENCH, GENQ><<<grid, 128, 0, c->stream>>>(st, c->list(col), n, g, col, sw, k, c->slots());
  LAUNCH_OK(c);
  return MPR_OK;
}
template <int MODE> int list_pass(mpr_ctx* c, int kind, int col, uint64_t sweep) {
  return c->lo.g.q == kQDefault ? list_pass_q<MODE, false>(c, kind, col, sweep) : list_pass_q<MODE, true>(c, kind, col, sweep);
}

template <int MODE> int init_chain(mpr_ctx* c) {
  using V = typename Traits<MODE>::vec;
  const Geom& g = c->lo.g;
  dim3 block(128), grid((g.Wp + 127) / 128, g.H, 2);
  init_chain_kernel<MODE><<<grid, block, 0, c->stream>>>(c->d_values, c->d_mask, g, c->zmin, c->zmax,
                                                         static_cast<uint32_t>(c->seed),
                                                         static_cast<uint32_t>(c->seed >> 32), c->trial,
                                                         static_cast<V*>(c->state(c->cur)));
  LAUNCH_OK(c);
  return MPR_OK;
}

// Energy of the current state into d_out[0] (e = 2H/N_b when `as_e`, else H).
template <int MODE> int plain_energy(mpr_ctx* c, double* d_out, bool as_e) {
  using V = typename Traits<MODE>::vec;
  const Geom& g = c->lo.g;
  const int nblk = g.H < 2048 ? g.H : 2048;
  plain_energy_kernel<MODE><<<nblk, 256, 0, c->stream>>>(static_cast<const V*>(c->state(c->cur)), g, c->part());
  LAUNCH_OK(c);
  const double nb = c->nb_norm;
  final_sum_kernel<<<1, 1024, 0, c->stream>>>(c->part(), nblk, as_e ? -kJ * 2.0 / nb : -kJ, d_out, g.energy_single);
  LAUNCH_OK(c);
  return MPR_OK;
}

template <int MODE> int plain_accumulate(mpr_ctx* c) {
  using V = typename Traits<MODE>::vec;
  const Geom& g = c->lo.g;
  dim3 block(128), grid((g.Wp + 127) / 128, g.H, 2);
  plain_accumulate_kernel<MODE><<<grid, block, 0, c->stream>>>(static_cast<const V*>(c->state(c->cur)), c->bits(),
                                                               g, c->acc());
  LAUNCH_OK(c);
  return MPR_OK;
}

template <int MODE> int get_state(mpr_ctx* c, double* d_phi) {
  using V = typename Traits<MODE>::vec;
  const Geom& g = c->lo.g;
  dim3 block(128), grid((g.L + 127) / 128, g.H);
  get_state_kernel<MODE><<<grid, block, 0, c->stream>>>(static_cast<const V*>(c->state(c->cur)), g, d_phi);
  LAUNCH_OK(c);
  return MPR_OK;
}

template <int MODE> int set_state(mpr_ctx* c, const double* d_phi) {
  using V = typename Traits<MODE>::vec;
  const Geom& g = c->lo.g;
  dim3 block(128), grid((g.Wp + 127) / 128, g.H, 2);
  set_state_kernel<MODE><<<grid, block, 0, c->stream>>>(d_phi, g, c->bits(), static_cast<V*>(c->state(c->cur)));
  LAUNCH_OK(c);
  return MPR_OK;
}

// k hybrid sweeps of the tiled path (k <= fused depth), with the energy sample and the
// accumulation of phi after the last one when `measure`; d_e receives e_n.
template <int MODE> int tiled_sweeps(mpr_ctx* c, int k, int measure, double* d_e) {
  using R = typename Traits<MODE>::real;
  const Geom& g = c->lo.g;
  int ntiles = 0;
  const int st = tiled_launch<MODE>(c->tiled, g, c->state(c->cur), c->state(1 - c->cur), c->bits(), c->acc(),
                                    c->part(), c->slots(), chain_const<R>(c), static_cast<uint32_t>(c->sweep + 1), k,
                                    measure, c->stream, &ntiles, kPartials);
  if (st != 0) return fail(c, MPR_ERR_CUDA, std::string("tiled launch: ") + tiled_error(st));
  c->launches += 1;
  c->cur = 1 - c->cur;
  if (measure == 1 || measure == 2) {
    const double nb = c->nb_norm;
    final_sum_kernel<<<1, 1024, 0, c->stream>>>(c->part(), ntiles, -kJ * 2.0 / nb, d_e, g.energy_single);
    LAUNCH_OK(c);
  }
  return MPR_OK;
}

// One launch of the STRIP path: k sweeps of the current schedule (prog = PROG_R4 / PROG_FUSED) or two quench double
// passes (PROG_QUENCH, k = 2); `measure` as in tiled_sweeps.
template <int MODE> int strip_sweeps(mpr_ctx* c, int prog, int k, int measure, double* d_e) {
  using R = typename Traits<MODE>::real;
  Geom g = c->lo.g;
  if (g.peer_rows) {
    // the buffer the neighbour's launch number `strip_epoch` writes: the other one if it has not been launched yet,
    // its current one if it already has
    for (int d = 0; d < 2; ++d) {
      const mpr_ctx* p = c->peer[d];
      g.peer_dst[d] = nullptr;
      if (!p) continue;
      if (p->strip_epoch != c->strip_epoch && p->strip_epoch != c->strip_epoch + 1)
        return fail(c, MPR_ERR_INVALID_ARG, "peer mode: the slabs are out of step (every slab makes the same calls in turn)");
      if (p->mode != c->mode || !p->ws) return fail(c, MPR_ERR_INVALID_ARG, "peer mode: neighbour in another mode or without workspace");
      g.peer_dst[d] = p->state(p->strip_epoch == c->strip_epoch ? 1 - p->cur : p->cur);
      g.peer_plane[d] = static_cast<long long>(p->lo.g.plane);
      g.peer_row_off[d] = c->slab_row0 - p->slab_row0;
    }
  }
  const ChainConst<R> kc = chain_const<R>(c);
  int nblocks = 0;
  StripArgs a{&c->strip, &c->tiled, g, c->cur, c->state(c->cur), c->state(1 - c->cur), {c->smask(1), c->smask(2)}, c->acc(), c->part(),
              c->slots(), &kc, static_cast<uint32_t>(c->sweep + 1), prog, k, measure, c->stream, &nblocks, kPartials};
  const int st = MODE == MODE_DP ? strip_launch_mode0(a) : MODE == MODE_SP ? strip_launch_mode1(a)
                 : MODE == MODE_SP_PRECISE ? strip_launch_mode2(a) : MODE == MODE_DS ? strip_launch_mode4(a)
                 : MODE == MODE_HP ? strip_launch_mode5(a) : strip_launch_mode3(a);
  if (st != 0) return fail(c, MPR_ERR_CUDA, std::string("strip launch: ") + tiled_error(st));
  c->launches += 1;
  c->cur = 1 - c->cur;
  c->strip_epoch += 1;
  if (measure == 1 || measure == 2) {
    const double nb = c->nb_norm;
    final_sum_kernel<<<1, 1024, 0, c->stream>>>(c->part(), nblocks, -kJ * 2.0 / nb, d_e, g.energy_single);
    LAUNCH_OK(c);
  }
  return MPR_OK;
}

#define DISPATCH(c, call)                                                     \
  ((c)->mode == MPR_DP           ? call<MODE_DP>                              \
   : (c)->mode == MPR_SP         ? call<MODE_SP>                              \
   : (c)->mode == MPR_SP_PRECISE ? call<MODE_SP_PRECISE>                      \
                                 : call<MODE_SP_INTRINSIC>)

int eff_path(const mpr_ctx* c);

int do_list_pass(mpr_ctx* c, int kind, int col, uint64_t sweep) {
  switch (c->mode) {
    case MPR_DP: return list_pass<MODE_DP>(c, kind, col, sweep);
    case MPR_SP: return list_pass<MODE_SP>(c, kind, col, sweep);
    case MPR_SP_PRECISE: return list_pass<MODE_SP_PRECISE>(c, kind, col, sweep);
    case MPR_DS_INTRINSIC: return list_pass<MODE_DS>(c, kind, col, sweep);
    case MPR_HP: return list_pass<MODE_HP>(c, kind, col, sweep);
    default: return list_pass<MODE_SP_INTRINSIC>(c, kind, col, sweep);
  }
}
int do_pass(mpr_ctx* c, int kind, int col, uint64_t sweep) {
  if (eff_path(c) == MPR_PATH_LIST) return do_list_pass(c, kind, col, sweep);
  switch (c->mode) {
    case MPR_DP: return plain_pass<MODE_DP>(c, kind, col, sweep);
    case MPR_SP: return plain_pass<MODE_SP>(c, kind, col, sweep);
    case MPR_SP_PRECISE: return plain_pass<MODE_SP_PRECISE>(c, kind, col, sweep);
    case MPR_DS_INTRINSIC: return plain_pass<MODE_DS>(c, kind, col, sweep);
    case MPR_HP: return plain_pass<MODE_HP>(c, kind, col, sweep);
    default: return plain_pass<MODE_SP_INTRINSIC>(c, kind, col, sweep);
  }
}
int do_init(mpr_ctx* c) {
  switch (c->mode) {
    case MPR_DP: return init_chain<MODE_DP>(c);
    case MPR_SP: return init_chain<MODE_SP>(c);
    case MPR_SP_PRECISE: return init_chain<MODE_SP_PRECISE>(c);
    case MPR_DS_INTRINSIC: return init_chain<MODE_DS>(c);
    case MPR_HP: return init_chain<MODE_HP>(c);
    default: return init_chain<MODE_SP_INTRINSIC>(c);
  }
}
int do_energy(mpr_ctx* c, double* d_out, bool as_e) {
  switch (c->mode) {
    case MPR_DP: return plain_energy<MODE_DP>(c, d_out, as_e);
    case MPR_SP: return plain_energy<MODE_SP>(c, d_out, as_e);
    case MPR_SP_PRECISE: return plain_energy<MODE_SP_PRECISE>(c, d_out, as_e);
    case MPR_DS_INTRINSIC: return plain_energy<MODE_DS>(c, d_out, as_e);
    case MPR_HP: return plain_energy<MODE_HP>(c, d_out, as_e);
    default: return plain_energy<MODE_SP_INTRINSIC>(c, d_out, as_e);
  }
}
int do_accumulate(mpr_ctx* c) {
  switch (c->mode) {
    case MPR_DP: return plain_accumulate<MODE_DP>(c);
    case MPR_SP: return plain_accumulate<MODE_SP>(c);
    case MPR_SP_PRECISE: return plain_accumulate<MODE_SP_PRECISE>(c);
    case MPR_DS_INTRINSIC: return plain_accumulate<MODE_DS>(c);
    case MPR_HP: return plain_accumulate<MODE_HP>(c);
    default: return plain_accumulate<MODE_SP_INTRINSIC>(c);
  }
}
int do_tiled(mpr_ctx* c, int k, int measure, double* d_e) {
  switch (c->mode) {
    case MPR_DP: return tiled_sweeps<MODE_DP>(c, k, measure, d_e);
    case MPR_SP: return tiled_sweeps<MODE_SP>(c, k, measure, d_e);
    case MPR_SP_PRECISE: return tiled_sweeps<MODE_SP_PRECISE>(c, k, measure, d_e);
    case MPR_DS_INTRINSIC: return tiled_sweeps<MODE_DS>(c, k, measure, d_e);
    case MPR_HP: return tiled_sweeps<MODE_HP>(c, k, measure, d_e);
    default: return tiled_sweeps<MODE_SP_INTRINSIC>(c, k, measure, d_e);
  }
}

int do_strip(mpr_ctx* c, int prog, int k, int measure, double* d_e) {
  switch (c->mode) {
    case MPR_DP: return strip_sweeps<MODE_DP>(c, prog, k, measure, d_e);
    case MPR_SP: return strip_sweeps<MODE_SP>(c, prog, k, measure, d_e);
    case MPR_SP_PRECISE: return strip_sweeps<MODE_SP_PRECISE>(c, prog, k, measure, d_e);
    case MPR_DS_INTRINSIC: return strip_sweeps<MODE_DS>(c, prog, k, measure, d_e);
    case MPR_HP: return strip_sweeps<MODE_HP>(c, prog, k, measure, d_e);
    default: return strip_sweeps<MODE_SP_INTRINSIC>(c, prog, k, measure, d_e);
  }
}

// MPR_PATH_AUTO: the path measured fastest for the case at hand (B200, bench.py --path, profiles/): the STRIP
// kernels in SP_INTRINSIC on grids large enough to give every warp a long run of rows, and for the site-fused
// schedule (which the TILED kernels do not carry); the TILED kernels otherwise (double arithmetic and the
// library sincosf / expf of SP_PRECISE need more registers per update chain than four interleaved chains leave).
int eff_path(const mpr_ctx* c) {
  if (c->lo.g.peer_rows) return MPR_PATH_STRIP;      // peer mode lives in the strip kernels (mpr_set_peers checks the rest)
  // q < 1/2 (mpr_set_q): the general range test lives in the per-pass kernels only
  if (c->lo.g.q != kQDefault) return c->path == MPR_PATH_LIST ? MPR_PATH_LIST : MPR_PATH_PLAIN;
  // half-precision storage: the TILED kernel's tile origins (60 tx - 2 plane columns) are not 16-byte aligned at
  // 4 bytes per column, which the TMA unit requires; the STRIP kernels carry two halo lanes for it and take over
  if (c->mode == MPR_HP) {
    if (c->path == MPR_PATH_PLAIN || c->path == MPR_PATH_LIST) return c->path;
    if (c->path == MPR_PATH_AUTO && grid_side(c->lo.g) < 4096) return MPR_PATH_PLAIN;
    return MPR_PATH_STRIP;
  }
  if (c->path != MPR_PATH_AUTO) return c->path;
  if (c->schedule == MPR_SCHEDULE_SITE_FUSED) {
    // small, sparsely masked grids: the compacted lists win (config 3, f = 0.33, L2-resident: 0.021 against 0.025 ms)
    const double f = static_cast<double>(c->n_free) / (static_cast<double>(c->lo.g.L) * c->lo.g.H);
    return (f < 0.5 && grid_side(c->lo.g) <= 4096) ? MPR_PATH_LIST : MPR_PATH_STRIP;
  }
  return (c->mode == MPR_SP_INTRINSIC && grid_side(c->lo.g) >= 4096) ? MPR_PATH_STRIP : MPR_PATH_TILED;
}

// `left` quench double passes (colour 0, colour 1): the tiled kernel runs them 2 k at a time (k <= 2,
// halo 4 k), the strip kernel two per launch, an odd remainder goes through the plain kernels -- same moves, same order
int quench_passes(mpr_ctx* c, int left) {
  const int path = eff_path(c);
  if (c->lo.g.peer_rows && (left & 1))
    return fail(c, MPR_ERR_INVALID_ARG, "peer mode: quench double passes come two per launch (an even number)");
  if (path == MPR_PATH_TILED) {
    while (left >= 2) {
      const int k = left / 2 < 2 ? left / 2 : 2;
      TRY(do_tiled(c, k, kTiledQuench, nullptr));
      left -= 2 * k;
    }
  } else if (path == MPR_PATH_STRIP) {
    for (; left >= 2; left -= 2) TRY(do_strip(c, PROG_QUENCH, 2, 0, nullptr));     // two double passes per launch
  }
  for (; left > 0; --left) {
    TRY(do_pass(c, KIND_QUENCH, 0, 0));
    TRY(do_pass(c, KIND_QUENCH, 1, 0));
  }
  return MPR_OK;
}

// R8: uniform initial spins, then n_quench x (quench colour 0, quench colour 1); everything
// that belongs to the chain is cleared.
int reset_chain(mpr_ctx* c, uint32_t trial) {
  if (!c->ws) return fail(c, MPR_ERR_WORKSPACE, "no workspace attached (mpr_set_workspace)");
  c->stale = false;
  c->trial = trial;
  c->sweep = 0;
  c->attempted = 0;
  c->n_acc = 0;
  c->series.clear();
  TRY(do_init(c));
  TRY(quench_passes(c, c->n_quench));
  CUDA_OK(c, cudaMemsetAsync(c->slots(), 0, kAcceptSlots * sizeof(unsigned long long), c->stream));
  const size_t n = 2 * c->lo.g.plane;
  clear_acc_kernel<<<1184, 256, 0, c->stream>>>(c->acc(), n);
  LAUNCH_OK(c);
  return MPR_OK;
}

// Setters only mark the chain stale; the reset (init + quench passes, R8) runs once, when the
// chain is next used -- mpr_create followed by mpr_set_precision pays for one reset, not two.
void mark_stale(mpr_ctx* c) {
  c->stale = true;
  c->trial = 0;
  c->sweep = 0;
  c->attempted = 0;
  c->n_acc = 0;
  c->series.clear();
}
int ensure_chain(mpr_ctx* c) {
  if (!c->ws) return fail(c, MPR_ERR_WORKSPACE, "no workspace attached (mpr_set_workspace)");
  if (c->expect_slab && !c->slab) return fail(c, MPR_ERR_NOT_READY, "created by mpr_create_slab: mpr_set_slab first");
  return c->stale ? reset_chain(c, 0) : MPR_OK;
}

// Hybrid sweeps per launch when the caller has not fixed them (mpr_set_fused_sweeps(0), the default).  Small grids are
// bound by the latency of a launch whose few tiles each run their passes back to back, so several sweeps per launch
// (halo 4 k) pay until the redundant halo work outweighs it.  Measured on B200, tiled kernel, us per sweep at
// k = 1 / 2 / 4 -- float arithmetic: L = 64: 10.3 / 8.2 / 7.2, 512: 12.3 / 8.7 / 7.2, 1024: 12.3 / 9.2 / 12.3,
// 1536: 18.5 / 14.4 / 18.0, 2048: 24.8 / 26.2 / 29.0; double arithmetic: 256: 20.5 / 17.8 / 16.4, 512: 20.5 / 17.8 / 22.6,
// 1024: 28.7 / 35.9 / 50.1.  The result does not depend on k.
// Not chosen automatically, but measured: the strip kernel of the headline mode with TWO sweeps per launch
// (mpr_set_fused_sweeps(2): 8 stages, 8 warps per SM) is slower than one per launch when timed alone (1.066 against 0.99 ms
// per sweep at L = 16384) yet moves half the DRAM bytes per sweep, draws less power and is not clocked down by this
// pool's 1000 W cap in a long run (1965 against 1680 MHz): 1.068 against 1.101 ms per sweep inside bench.py's step.  A
// property of the box's power limit, not of the kernel: the default stays one sweep per launch.
int auto_fused(const mpr_ctx* c, int path, int n) {
  (void)n;
  if (path != MPR_PATH_TILED) return 1;
  const double side = grid_side(c->lo.g);
  const bool dbl = c->mode == MPR_DP || c->mode == MPR_SP;
  if (dbl) return side <= 256.0 ? 4 : side <= 512.0 ? 2 : 1;
  return side <= 512.0 ? 4 : side <= 1536.0 ? 2 : 1;
}

// measure: 0 = sweeps only, 1 = + energy sample per sweep, 2 = + accumulation of phi.
// n hybrid sweeps (R4); with `measure`, each is followed by the energy sample into
// dseries[first_slot + i] and the accumulation of phi.
int hybrid_sweeps(mpr_ctx* c, int n, int measure, int first_slot) {
  if (n <= 0) return MPR_OK;
  if (!(c->T > 0.0)) return fail(c, MPR_ERR_NOT_READY, "temperature not set");
  TRY(ensure_chain(c));
  const int path = eff_path(c);
  if (path == MPR_PATH_PLAIN || path == MPR_PATH_LIST) {
    for (int i = 0; i < n; ++i) {
      const uint64_t sw = c->sweep + 1;
      if (c->schedule == MPR_SCHEDULE_SITE_FUSED) {      // R4b
        TRY(do_pass(c, KIND_MO, 0, sw));
        TRY(do_pass(c, KIND_MO, 1, sw));
      } else {                                            // R4
        TRY(do_pass(c, KIND_MET, 0, sw));
        TRY(do_pass(c, KIND_MET, 1, sw));
        TRY(do_pass(c, KIND_OR, 0, sw));
        TRY(do_pass(c, KIND_OR, 1, sw));
      }
      c->sweep = sw;
      c->attempted += static_cast<uint64_t>(c->n_free);
      if (measure) {
        TRY(do_energy(c, c->dseries() + first_slot + i, true));
        if (measure == 2) {
          TRY(do_accumulate(c));
          c->n_acc += 1;
        }
      }
    }
    return MPR_OK;
  }
  if (path == MPR_PATH_TILED && c->schedule != MPR_SCHEDULE_R4)
    return fail(c, MPR_ERR_INVALID_ARG, "the site-fused schedule runs on the STRIP and PLAIN paths");
  const int fused = c->fused > 0 ? c->fused : auto_fused(c, path, n);
  int done = 0;
  while (done < n) {
    // measurement needs the state after every sweep: one sweep per launch there
    int k = measure ? 1 : (n - done < fused ? n - done : fused);
    double* d_e = measure ? c->dseries() + first_slot + done : nullptr;
    if (path == MPR_PATH_STRIP) {
      if (k > 2) k = 2;                                   // the strip pipeline carries at most two sweeps
      if (c->lo.g.peer_rows) k = 1;                       // peer mode: the halo lasts one sweep, refreshed by every launch
      TRY(do_strip(c, c->schedule == MPR_SCHEDULE_SITE_FUSED ? PROG_FUSED : PROG_R4, k, measure, d_e));
    } else {
      TRY(do_tiled(c, k, measure, d_e));
    }
    c->sweep += static_cast<uint64_t>(k);
    c->attempted += static_cast<uint64_t>(k) * static_cast<uint64_t>(c->n_free);
    if (measure == 2) c->n_acc += 1;
    done += k;
  }
  return MPR_OK;
}

int fetch_series(mpr_ctx* c, int n) {
  c->series.assign(static_cast<size_t>(n), 0.0);
  if (n > 0)
    CUDA_OK(c, cudaMemcpyAsync(c->series.data(), c->dseries(), n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CUDA_OK(c, cudaStreamSynchronize(c->stream));
  return MPR_OK;
}

// One temperature trial of R6: fresh chain with the trial index in the Philox counter.
int trial_energy(mpr_ctx* c, int* est_trials, double T, double* e, double* se) {
  *est_trials += 1;
  c->T = T;
  TRY(reset_chain(c, static_cast<uint32_t>(*est_trials)));
  TRY(hybrid_sweeps(c, kTrialEq, 0, 0));
  TRY(hybrid_sweeps(c, kTrialMeas, 1, 0));   // energy only: a trial's phi average is never used
  TRY(fetch_series(c, kTrialMeas));
  mean_stderr(c->series, e, se);
  return MPR_OK;
}

int setup(mpr_ctx* c) {
  const Geom& g = c->lo.g;
  const size_t N = static_cast<size_t>(g.L) * g.H;
  // R1: range of the measured sample
  const int nblk = 1024;
  sample_range_kernel<<<nblk, 256, 0, c->stream>>>(c->d_values, c->d_mask, N, c->part());
  LAUNCH_OK(c);
  sample_range_final_kernel<<<1, 32, 0, c->stream>>>(c->part(), nblk, c->scal());
  LAUNCH_OK(c);
  double h[4];
  CUDA_OK(c, cudaMemcpyAsync(h, c->scal(), sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  CUDA_OK(c, cudaStreamSynchronize(c->stream));
  if (h[3] != 0.0) return fail(c, MPR_ERR_NONFINITE, "non-finite value at a measured site");
  if (c->expect_slab && (h[2] == 0.0 || !(h[1] > h[0]))) {
    // the rows of a slab may hold no measured site, or one value only: the range that counts is the whole grid's,
    // which mpr_set_slab brings (a placeholder until then)
    h[0] = 0.0;
    h[1] = 1.0;
  } else {
    if (h[2] == 0.0) return fail(c, MPR_ERR_NO_MEASURED, "no measured site");
    if (!(h[1] > h[0])) return fail(c, MPR_ERR_DEGENERATE_RANGE, "z_max == z_min over the measured sample");
  }
  c->zmin = h[0];
  c->zmax = h[1];
  // R6: sample energy
  sample_energy_kernel<<<nblk, 256, 0, c->stream>>>(c->d_values, c->d_mask, g.L, g.H, g.own0, g.own1, c->zmin, c->zmax, c->part(), g.q);
  LAUNCH_OK(c);
  pair_final_kernel<<<1, 32, 0, c->stream>>>(c->part(), nblk, c->scal());
  LAUNCH_OK(c);
  // mask bitmaps and the number of prediction sites
  const size_t nwords = static_cast<size_t>(2) * g.Hb * g.Wb;
  const int mblk = static_cast<int>((nwords + 255) / 256);
  if (mblk > kPartials) return fail(c, MPR_ERR_INVALID_ARG, "grid too large");
  double* cnt_part = c->part() + 2 * nblk;
  pack_mask_kernel<<<mblk, 256, 0, c->stream>>>(c->d_mask, g, c->bits_base(), cnt_part);
  LAUNCH_OK(c);
  final_sum_kernel<<<1, 1024, 0, c->stream>>>(cnt_part, mblk, 1.0, c->scal() + 2);
  LAUNCH_OK(c);
  // the same bits in strip order, for the STRIP path (mpr_strip.cuh)
  for (int hl = 1; hl <= 2; ++hl) {
    CUDA_OK(c, strip_mask_build(c->d_mask, g, hl, c->smask(hl), c->stream));
    c->launches += 1;
  }
  // compacted per-colour lists of the prediction sites, for the LIST path (mpr_plain.cuh)
  {
    uint32_t* row_count = c->rows();
    uint32_t* row_off = row_count + 2 * static_cast<size_t>(g.H);
    uint32_t* totals = row_off + 2 * static_cast<size_t>(g.H);
    list_row_count_kernel<<<dim3(g.H, 2), 128, 0, c->stream>>>(c->bits(), g, row_count);
    LAUNCH_OK(c);
    list_row_scan_kernel<<<1, 1024, 0, c->stream>>>(row_count, g.H, row_off, totals);
    LAUNCH_OK(c);
    list_fill_kernel<<<dim3((g.H + 3) / 4, 2), 128, 0, c->stream>>>(c->bits(), g, row_off, c->list(0), c->list(1));
    LAUNCH_OK(c);
    CUDA_OK(c, cudaMemcpyAsync(c->n_list, totals, sizeof(c->n_list), cudaMemcpyDeviceToHost, c->stream));
  }
  double h2[3];
  CUDA_OK(c, cudaMemcpyAsync(h2, c->scal(), sizeof(h2), cudaMemcpyDeviceToHost, c->stream));
  CUDA_OK(c, cudaStreamSynchronize(c->stream));
  c->n_pairs = static_cast<long long>(h2[1]);
  c->pair_sum = h2[0];
  if (!c->slab) c->nb_norm = bond_count(g);
  c->e_sample = c->n_pairs > 0 ? -2.0 * kJ * h2[0] / h2[1] : std::numeric_limits<double>::quiet_NaN();
  c->n_free = static_cast<long long>(h2[2]);
  return MPR_OK;
}

}  // namespace

// =============================================================================================
extern "C" {

const char* mpr_status_string(int status) {
  switch (status) {
    case MPR_OK: return "ok";
    case MPR_ERR_INVALID_ARG: return "invalid argument";
    case MPR_ERR_NO_MEASURED: return "no measured site / pair";
    case MPR_ERR_DEGENERATE_RANGE: return "degenerate value range";
    case MPR_ERR_NONFINITE: return "non-finite measured value";
    case MPR_ERR_WORKSPACE: return "workspace null, misaligned or too small";
    case MPR_ERR_NOT_READY: return "temperature not set";
    case MPR_ERR_NO_ROOT: return "sample energy not bracketed by e(T)";
    case MPR_ERR_CUDA: return "CUDA error";
    default: return "unknown status";
  }
}

const char* mpr_last_error(const mpr_ctx* ctx) { return ctx ? ctx->err.c_str() : ""; }

// a grid is valid when both sides are in [1, kMaxL], it has at least two sites, and its Philox site index fits 32 bits
static bool valid_shape(int Lx, int Ly) {
  return Lx >= 1 && Ly >= 1 && Lx <= kMaxL && Ly <= kMaxL && static_cast<long long>(Lx) * Ly >= 2 &&
         static_cast<long long>(Lx) * Ly <= (1ll << 32);
}

int mpr_workspace_bytes_rect(int Lx, int Ly, size_t* bytes) {
  if (!valid_shape(Lx, Ly) || !bytes) return MPR_ERR_INVALID_ARG;
  *bytes = make_layout(Lx, Ly).total;
  return MPR_OK;
}
int mpr_workspace_bytes(int L, size_t* bytes) {
  if (L < 2) return MPR_ERR_INVALID_ARG;
  return mpr_workspace_bytes_rect(L, L, bytes);
}

int mpr_create(mpr_ctx** out, int L, const double* d_values, const uint8_t* d_mask, void* d_workspace,
               size_t workspace_bytes, void* cuda_stream) {
  if (!out) return MPR_ERR_INVALID_ARG;
  *out = nullptr;
  if (L < 2) return MPR_ERR_INVALID_ARG;
  return mpr_create_rect(out, L, L, d_values, d_mask, d_workspace, workspace_bytes, cuda_stream);
}

static int create_impl(mpr_ctx** out, int Lx, int Ly, const double* d_values, const uint8_t* d_mask, void* d_workspace,
                       size_t workspace_bytes, void* cuda_stream, bool expect_slab);
int mpr_create_rect(mpr_ctx** out, int Lx, int Ly, const double* d_values, const uint8_t* d_mask, void* d_workspace,
                    size_t workspace_bytes, void* cuda_stream) {
  return create_impl(out, Lx, Ly, d_values, d_mask, d_workspace, workspace_bytes, cuda_stream, false);
}
int mpr_create_slab(mpr_ctx** out, int Lx, int Ly, const double* d_values, const uint8_t* d_mask, void* d_workspace,
                    size_t workspace_bytes, void* cuda_stream) {
  return create_impl(out, Lx, Ly, d_values, d_mask, d_workspace, workspace_bytes, cuda_stream, true);
}
static int create_impl(mpr_ctx** out, int Lx, int Ly, const double* d_values, const uint8_t* d_mask, void* d_workspace,
                       size_t workspace_bytes, void* cuda_stream, bool expect_slab) {
  if (!out) return MPR_ERR_INVALID_ARG;
  *out = nullptr;
  if (!valid_shape(Lx, Ly) || !d_values || !d_mask) return MPR_ERR_INVALID_ARG;
  const Layout lo = make_layout(Lx, Ly);
  const bool with_ws = d_workspace || workspace_bytes;
  if (with_ws && (!d_workspace || (reinterpret_cast<uintptr_t>(d_workspace) & 255u) || workspace_bytes < lo.total))
    return MPR_ERR_WORKSPACE;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return MPR_ERR_CUDA;
  mpr_ctx* c = new (std::nothrow) mpr_ctx;
  if (!c) return MPR_ERR_INVALID_ARG;
  c->lo = lo;
  c->d_values = d_values;
  c->d_mask = d_mask;
  c->stream = static_cast<cudaStream_t>(cuda_stream);
  c->expect_slab = expect_slab;
  // SURVEY 8(b) form: create(L, values, mask) first, mpr_set_workspace / mpr_set_stream afterwards
  if (with_ws) {
    const int st = mpr_set_workspace(c, d_workspace, workspace_bytes);
    if (st != MPR_OK) { delete c; return st; }
  }
  *out = c;
  return MPR_OK;
}

int mpr_set_workspace(mpr_ctx* c, void* d_workspace, size_t workspace_bytes) {
  if (!c) return MPR_ERR_INVALID_ARG;
  if (!d_workspace || (reinterpret_cast<uintptr_t>(d_workspace) & 255u) || workspace_bytes < c->lo.total)
    return fail(c, MPR_ERR_WORKSPACE, "workspace null, misaligned or too small");
  if (c->ws) CUDA_OK(c, cudaStreamSynchronize(c->stream));   // nothing of ours still runs on the old one
  c->ws = static_cast<char*>(d_workspace);
  int st = setup(c);
  if (st == MPR_OK) {
    const int ts = tiled_plan_init(&c->tiled, c->lo.g);
    if (ts != 0) st = fail(c, MPR_ERR_CUDA, std::string("tiled plan: ") + tiled_error(ts));
  }
  if (st != MPR_OK) { c->ws = nullptr; return st; }
  mark_stale(c);
  return MPR_OK;
}

int mpr_set_stream(mpr_ctx* c, void* cuda_stream) {
  if (!c) return MPR_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  if (s == c->stream) return MPR_OK;
  // work already enqueued on the old stream must be finished before the new one touches the state
  if (c->ws) CUDA_OK(c, cudaStreamSynchronize(c->stream));
  c->stream = s;
  return MPR_OK;
}

void mpr_destroy(mpr_ctx* ctx) {
  if (!ctx) return;
  for (cudaEvent_t e : ctx->ev_eq)
    if (e) cudaEventDestroy(e);
  delete ctx;
}

int mpr_set_precision(mpr_ctx* c, mpr_precision mode) {
  if (!c || mode < MPR_DP || mode > MPR_HP) return fail(c, MPR_ERR_INVALID_ARG, "bad mode");
  c->mode = mode;
  mark_stale(c);
  return MPR_OK;
}
int mpr_set_q(mpr_ctx* c, double q) {
  if (!c || !(q > 0.0) || q > 0.5) return fail(c, MPR_ERR_INVALID_ARG, "q must lie in (0, 1/2]");
  c->lo.g.q = q;
  if (c->ws) TRY(setup(c));       // the sample energy of R6 depends on q
  mark_stale(c);
  return MPR_OK;
}
int mpr_set_energy_precision(mpr_ctx* c, int single) {
  if (!c || (single != 0 && single != 1)) return fail(c, MPR_ERR_INVALID_ARG, "energy precision: 0 (double) or 1 (single)");
  c->lo.g.energy_single = single;     // only the measuring arithmetic changes: the chain is left alone
  return MPR_OK;
}
int mpr_set_precision_triple(mpr_ctx* c, const char* xs_xe_xf) {
  if (!c || !xs_xe_xf || std::strlen(xs_xe_xf) != 3) return fail(c, MPR_ERR_INVALID_ARG, "triple: three letters, D or S");
  for (int i = 0; i < 3; ++i)
    if (xs_xe_xf[i] != 'D' && xs_xe_xf[i] != 'S') return fail(c, MPR_ERR_INVALID_ARG, "triple: three letters, D or S");
  const bool s_single = xs_xe_xf[0] == 'S', e_single = xs_xe_xf[1] == 'S', f_single = xs_xe_xf[2] == 'S';
  const mpr_precision mode = f_single ? (s_single ? MPR_SP_INTRINSIC : MPR_DS_INTRINSIC) : (s_single ? MPR_SP : MPR_DP);
  TRY(mpr_set_precision(c, mode));
  return mpr_set_energy_precision(c, e_single ? 1 : 0);
}
int mpr_set_seed(mpr_ctx* c, uint64_t seed) {
  if (!c) return MPR_ERR_INVALID_ARG;
  c->seed = seed;
  mark_stale(c);
  return MPR_OK;
}
int mpr_set_temperature(mpr_ctx* c, double T) {
  if (!c || !(T > 0.0) || !std::isfinite(T)) return fail(c, MPR_ERR_INVALID_ARG, "T must be finite and > 0");
  c->T = T;
  return MPR_OK;
}
int mpr_set_quench(mpr_ctx* c, int n) {
  if (!c || n < 0) return fail(c, MPR_ERR_INVALID_ARG, "n_quench < 0");
  c->n_quench = n;
  mark_stale(c);
  return MPR_OK;
}
int mpr_set_path(mpr_ctx* c, mpr_path path) {
  if (!c || (path != MPR_PATH_TILED && path != MPR_PATH_PLAIN && path != MPR_PATH_STRIP && path != MPR_PATH_AUTO &&
             path != MPR_PATH_LIST))
    return fail(c, MPR_ERR_INVALID_ARG, "bad path");
  c->path = path;
  return MPR_OK;
}
int mpr_set_schedule(mpr_ctx* c, mpr_schedule schedule) {
  if (!c || (schedule != MPR_SCHEDULE_R4 && schedule != MPR_SCHEDULE_SITE_FUSED))
    return fail(c, MPR_ERR_INVALID_ARG, "bad schedule");
  c->schedule = schedule;     // the chain continues: both orders are valid Markov kernels for the same density
  return MPR_OK;
}
int mpr_set_fused_sweeps(mpr_ctx* c, int k) {
  if (!c || k < 0 || k > tiled_max_fused()) return fail(c, MPR_ERR_INVALID_ARG, "fused depth out of range");
  c->fused = k;
  return MPR_OK;
}
int mpr_reset_chain(mpr_ctx* c, uint32_t trial) {
  if (!c) return MPR_ERR_INVALID_ARG;
  return reset_chain(c, trial);
}

int mpr_estimate_temperature(mpr_ctx* c, double* T_hat, double* e_sample, int* n_trials) {
  if (!c) return MPR_ERR_INVALID_ARG;
  if (!c->ws) return fail(c, MPR_ERR_WORKSPACE, "no workspace attached (mpr_set_workspace)");
  if (c->n_pairs == 0) return fail(c, MPR_ERR_NO_MEASURED, "no measured nearest-neighbour pair");
  if (e_sample) *e_sample = c->e_sample;
  // R6 steps 1-5: the search itself is mpr_host::TemperatureMatcher; this loop only runs the trial
  // chains it asks for (trial i = fresh chain with i in Philox counter word 3, 200 + 50 sweeps).
  const double T_before = c->T;
  mpr_host::TemperatureMatcher search;
  int trials = 0, st = MPR_OK;
  while (st == MPR_OK && search.want_trial()) {
    double e = 0.0, se = 0.0;
    st = trial_energy(c, &trials, search.T(), &e, &se);
    if (st == MPR_OK) search.report(e - c->e_sample, se);
  }
  if (n_trials) *n_trials = trials;
  if (st == MPR_OK && search.outcome() != mpr_host::TemperatureMatcher::FOUND)
    st = fail(c, MPR_ERR_NO_ROOT, search.outcome() == mpr_host::TemperatureMatcher::NO_ROOT_BELOW
                                      ? "e_sample below e(T) for every T >= 1e-6"
                                      : "e_sample above e(T) for every T <= 1e2");
  if (st != MPR_OK) {
    // a failed estimate leaves no trial temperature behind: T as before the call, chain to be rebuilt
    c->T = T_before;
    mark_stale(c);
    return st;
  }
  c->T = search.result();
  TRY(reset_chain(c, 0));
  if (T_hat) *T_hat = c->T;
  return MPR_OK;
}

int mpr_sweep(mpr_ctx* c, int n) {
  if (!c || n < 0) return fail(c, MPR_ERR_INVALID_ARG, "n < 0");
  return hybrid_sweeps(c, n, 0, 0);
}

int mpr_pass(mpr_ctx* c, int kind, int colour, uint64_t sweep) {
  if (!c || kind < 0 || kind > 3) return fail(c, MPR_ERR_INVALID_ARG, "bad pass kind");
  if ((kind == KIND_MET || kind == KIND_MO) && !(c->T > 0.0)) return fail(c, MPR_ERR_NOT_READY, "temperature not set");
  TRY(ensure_chain(c));
  return do_pass(c, kind, colour & 1, sweep);
}

int mpr_run(mpr_ctx* c, int n_eq, int n_meas, double* d_pred, double* e_mean, double* e_stderr) {
  if (!c || n_eq < 0 || n_meas < 0 || n_meas > kSeriesCap) return fail(c, MPR_ERR_INVALID_ARG, "bad sweep counts");
  if (!(c->T > 0.0)) return fail(c, MPR_ERR_NOT_READY, "temperature not set");
  TRY(ensure_chain(c));
  for (cudaEvent_t& e : c->ev_eq)
    if (!e) CUDA_OK(c, cudaEventCreate(&e));
  const uint64_t launches0 = c->launches;
  CUDA_OK(c, cudaEventRecord(c->ev_eq[0], c->stream));      // after the chain reset, if one was due
  TRY(hybrid_sweeps(c, n_eq, 0, 0));
  CUDA_OK(c, cudaEventRecord(c->ev_eq[1], c->stream));
  const long long eq_launches = static_cast<long long>(c->launches - launches0);
  TRY(hybrid_sweeps(c, n_meas, 2, 0));
  if (d_pred) {
    const Geom& g = c->lo.g;
    dim3 block(128), grid((g.L + 127) / 128, g.H);
    predict_kernel<<<grid, block, 0, c->stream>>>(c->d_values, c->d_mask, g, c->acc(), c->zmin, c->zmax, c->n_acc,
                                                  d_pred);
    LAUNCH_OK(c);
  }
  TRY(fetch_series(c, n_meas));
  mean_stderr(c->series, e_mean, e_stderr);
  CUDA_OK(c, cudaEventSynchronize(c->ev_eq[1]));
  float ms = 0.0f;
  CUDA_OK(c, cudaEventElapsedTime(&ms, c->ev_eq[0], c->ev_eq[1]));
  c->last_eq_ms = n_eq > 0 ? static_cast<double>(ms) : 0.0;   // two adjacent events are a few us apart, not 0
  c->last_eq_launches = eq_launches;
  c->last_eq_sweeps = n_eq;
  return MPR_OK;
}

int mpr_get_run_timing(mpr_ctx* c, double* eq_ms, int64_t* eq_launches, int64_t* eq_sweeps) {
  if (!c) return MPR_ERR_INVALID_ARG;
  if (c->last_eq_ms < 0.0) return fail(c, MPR_ERR_NOT_READY, "no mpr_run yet");
  if (eq_ms) *eq_ms = c->last_eq_ms;
  if (eq_launches) *eq_launches = c->last_eq_launches;
  if (eq_sweeps) *eq_sweeps = c->last_eq_sweeps;
  return MPR_OK;
}

int mpr_get_state(mpr_ctx* c, double* d_phi) {
  if (!c || !d_phi) return fail(c, MPR_ERR_INVALID_ARG, "null pointer");
  TRY(ensure_chain(c));
  switch (c->mode) {
    case MPR_DP: return get_state<MODE_DP>(c, d_phi);
    case MPR_SP: return get_state<MODE_SP>(c, d_phi);
    case MPR_SP_PRECISE: return get_state<MODE_SP_PRECISE>(c, d_phi);
    case MPR_DS_INTRINSIC: return get_state<MODE_DS>(c, d_phi);
    case MPR_HP: return get_state<MODE_HP>(c, d_phi);
    default: return get_state<MODE_SP_INTRINSIC>(c, d_phi);
  }
}
int mpr_set_state(mpr_ctx* c, const double* d_phi) {
  if (!c || !d_phi) return fail(c, MPR_ERR_INVALID_ARG, "null pointer");
  TRY(ensure_chain(c));
  switch (c->mode) {
    case MPR_DP: return set_state<MODE_DP>(c, d_phi);
    case MPR_SP: return set_state<MODE_SP>(c, d_phi);
    case MPR_SP_PRECISE: return set_state<MODE_SP_PRECISE>(c, d_phi);
    case MPR_DS_INTRINSIC: return set_state<MODE_DS>(c, d_phi);
    case MPR_HP: return set_state<MODE_HP>(c, d_phi);
    default: return set_state<MODE_SP_INTRINSIC>(c, d_phi);
  }
}

int mpr_energy(mpr_ctx* c, double* H, double* e) {
  if (!c) return MPR_ERR_INVALID_ARG;
  TRY(ensure_chain(c));
  TRY(do_energy(c, c->scal() + 8, false));
  double h = 0.0;
  CUDA_OK(c, cudaMemcpyAsync(&h, c->scal() + 8, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CUDA_OK(c, cudaStreamSynchronize(c->stream));
  const double nb = c->nb_norm;
  if (H) *H = h;
  if (e) *e = c->lo.g.energy_single ? static_cast<double>(2.0f * static_cast<float>(h) / static_cast<float>(nb))
                                    : 2.0 * h / nb;
  return MPR_OK;
}

int mpr_sample_energy(mpr_ctx* c, double* e_sample, int64_t* n_pairs) {
  if (!c) return MPR_ERR_INVALID_ARG;
  if (!c->ws) return fail(c, MPR_ERR_WORKSPACE, "no workspace attached (mpr_set_workspace)");
  if (n_pairs) *n_pairs = c->n_pairs;
  if (c->n_pairs == 0) return fail(c, MPR_ERR_NO_MEASURED, "no measured nearest-neighbour pair");
  if (e_sample) *e_sample = c->e_sample;
  return MPR_OK;
}

int mpr_sample_energy_parts(mpr_ctx* c, double* cos_sum, int64_t* n_pairs) {
  if (!c) return MPR_ERR_INVALID_ARG;
  if (!c->ws) return fail(c, MPR_ERR_WORKSPACE, "no workspace attached (mpr_set_workspace)");
  if (cos_sum) *cos_sum = c->pair_sum;
  if (n_pairs) *n_pairs = c->n_pairs;
  return MPR_OK;
}

// ---- slabs of a larger grid ----------------------------------------------------
static size_t spin_bytes(int mode) { return mode == MPR_HP ? 4 : (mode == MPR_DP || mode == MPR_DS_INTRINSIC) ? 16 : 8; }

int mpr_set_slab(mpr_ctx* c, int global_row0, int own_begin, int own_end, double z_min, double z_max, double global_bonds) {
  if (!c) return MPR_ERR_INVALID_ARG;
  if (!c->ws) return fail(c, MPR_ERR_WORKSPACE, "no workspace attached (mpr_set_workspace)");
  Geom& g = c->lo.g;
  if (global_row0 < 0 || (global_row0 & 1) || own_begin < 0 || own_end > g.H || own_begin >= own_end || !(z_max > z_min) ||
      !std::isfinite(z_min) || !std::isfinite(z_max) || !(global_bonds >= 1.0) ||
      (static_cast<long long>(global_row0) + g.H) * g.L > (1ll << 32))
    return fail(c, MPR_ERR_INVALID_ARG, "slab: first row even and >= 0, 0 <= own_begin < own_end <= rows, z_max > z_min");
  CUDA_OK(c, cudaStreamSynchronize(c->stream));
  c->slab_row0 = global_row0;
  g.site0 = static_cast<uint32_t>(static_cast<long long>(global_row0) * g.L);
  g.own0 = own_begin;
  g.own1 = own_end;
  c->zmin = z_min;
  c->zmax = z_max;
  c->nb_norm = global_bonds;
  c->slab = true;
  // the measured pairs to the right of and below the slab's own rows, in the whole sample's range
  const int nblk = 1024;
  sample_energy_kernel<<<nblk, 256, 0, c->stream>>>(c->d_values, c->d_mask, g.L, g.H, g.own0, g.own1, c->zmin, c->zmax, c->part(), g.q);
  LAUNCH_OK(c);
  pair_final_kernel<<<1, 32, 0, c->stream>>>(c->part(), nblk, c->scal());
  LAUNCH_OK(c);
  double h2[2];
  CUDA_OK(c, cudaMemcpyAsync(h2, c->scal(), sizeof(h2), cudaMemcpyDeviceToHost, c->stream));
  // prediction sites of the own rows (the per-row counts the LIST set-up left in the workspace)
  std::vector<uint32_t> rc(static_cast<size_t>(2) * g.H);
  CUDA_OK(c, cudaMemcpyAsync(rc.data(), c->rows(), rc.size() * sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
  CUDA_OK(c, cudaStreamSynchronize(c->stream));
  c->pair_sum = h2[0];
  c->n_pairs = static_cast<long long>(h2[1]);
  c->e_sample = c->n_pairs > 0 ? -2.0 * kJ * h2[0] / h2[1] : std::numeric_limits<double>::quiet_NaN();
  long long nf = 0;
  for (int col = 0; col < 2; ++col)
    for (int y = own_begin; y < own_end; ++y) nf += rc[static_cast<size_t>(col) * g.H + y];
  c->n_free = nf;
  mark_stale(c);
  return MPR_OK;
}

int mpr_set_peers(mpr_ctx* c, mpr_ctx* up, mpr_ctx* down) {
  if (!c) return MPR_ERR_INVALID_ARG;
  Geom& g = c->lo.g;
  if (!up && !down) {                       // leave peer mode
    g.peer_rows = 0;
    c->peer[0] = c->peer[1] = nullptr;
    return MPR_OK;
  }
  if (!c->slab) return fail(c, MPR_ERR_INVALID_ARG, "peer mode: mpr_set_slab first");
  if (g.q != kQDefault) return fail(c, MPR_ERR_INVALID_ARG, "peer mode runs on the strip kernels: q = 1/2 only");
  constexpr int kPeerRows = 4;              // one launch (a hybrid sweep, or two quench double passes) spoils 4 halo rows
  mpr_ctx* ps[2] = {up, down};
  for (int d = 0; d < 2; ++d) {
    const mpr_ctx* p = ps[d];
    if (!p) continue;
    if (p == c || !p->slab || p->lo.g.L != g.L || p->mode != c->mode)
      return fail(c, MPR_ERR_INVALID_ARG, "peer mode: neighbours are slabs of the same grid and mode");
    // the neighbour's halo must be exactly the rows this slab sends: kPeerRows rows beyond its own rows, on my side
    const int my_first = c->slab_row0 + g.own0, my_last = c->slab_row0 + g.own1;         // global own rows [first, last)
    const int p_first = p->slab_row0 + p->lo.g.own0, p_last = p->slab_row0 + p->lo.g.own1;
    const bool ok = d == 0 ? (p_last == my_first && p->lo.g.H - p->lo.g.own1 == kPeerRows && g.own0 == kPeerRows)
                           : (p_first == my_last && p->lo.g.own0 == kPeerRows && g.H - g.own1 == kPeerRows);
    if (!ok) return fail(c, MPR_ERR_INVALID_ARG, "peer mode: adjacent slabs with a halo of exactly 4 rows");
  }
  if ((!up && g.own0 != 0) || (!down && g.own1 != g.H))
    return fail(c, MPR_ERR_INVALID_ARG, "peer mode: a slab with halo rows on a side needs the neighbour of that side");
  if (g.own1 - g.own0 < 2 * kPeerRows) return fail(c, MPR_ERR_INVALID_ARG, "peer mode: a slab owns at least 8 rows");
  c->peer[0] = up;
  c->peer[1] = down;
  g.peer_rows = kPeerRows;
  c->strip_epoch = 0;
  mark_stale(c);
  return MPR_OK;
}

int mpr_rows_bytes(mpr_ctx* c, int n_rows, size_t* bytes) {
  if (!c || !bytes || n_rows < 0 || n_rows > c->lo.g.H) return MPR_ERR_INVALID_ARG;
  *bytes = static_cast<size_t>(2) * n_rows * c->lo.g.Wp * spin_bytes(c->mode);
  return MPR_OK;
}

static int copy_rows(mpr_ctx* c, int row_begin, int n_rows, void* d_buf, bool out) {
  if (!c || !d_buf) return fail(c, MPR_ERR_INVALID_ARG, "null pointer");
  const Geom& g = c->lo.g;
  if (row_begin < 0 || n_rows < 0 || row_begin + n_rows > g.H) return fail(c, MPR_ERR_INVALID_ARG, "rows outside the grid");
  TRY(ensure_chain(c));
  const size_t sb = spin_bytes(c->mode), row_b = static_cast<size_t>(g.Wp) * sb, chunk = row_b * n_rows;
  char* st = static_cast<char*>(c->state(c->cur));
  for (int col = 0; col < 2 && n_rows > 0; ++col) {
    char* in_state = st + (static_cast<size_t>(col) * g.plane + static_cast<size_t>(row_begin) * g.Wp) * sb;
    char* in_buf = static_cast<char*>(d_buf) + col * chunk;
    CUDA_OK(c, cudaMemcpyAsync(out ? in_buf : in_state, out ? in_state : in_buf, chunk, cudaMemcpyDeviceToDevice, c->stream));
  }
  return MPR_OK;
}
int mpr_export_rows(mpr_ctx* c, int row_begin, int n_rows, void* d_out) { return copy_rows(c, row_begin, n_rows, d_out, true); }
int mpr_import_rows(mpr_ctx* c, int row_begin, int n_rows, const void* d_in) {
  return copy_rows(c, row_begin, n_rows, const_cast<void*>(d_in), false);
}

int mpr_advance(mpr_ctx* c, int n_sweeps, int measure, int first_slot) {
  if (!c || n_sweeps < 0 || measure < 0 || measure > 2 || first_slot < 0 ||
      (measure && static_cast<long long>(first_slot) + n_sweeps > kSeriesCap))
    return fail(c, MPR_ERR_INVALID_ARG, "bad sweep count, measure flag or series slot");
  return hybrid_sweeps(c, n_sweeps, measure, first_slot);
}

int mpr_quench(mpr_ctx* c, int n_double_passes) {
  if (!c || n_double_passes < 0) return fail(c, MPR_ERR_INVALID_ARG, "negative pass count");
  TRY(ensure_chain(c));
  return quench_passes(c, n_double_passes);
}

int mpr_fetch_series(mpr_ctx* c, int n, double* h_out) {
  if (!c || n < 0 || n > kSeriesCap || (n > 0 && !h_out)) return fail(c, MPR_ERR_INVALID_ARG, "bad series length");
  if (!c->ws) return fail(c, MPR_ERR_WORKSPACE, "no workspace attached (mpr_set_workspace)");
  TRY(fetch_series(c, n));
  for (int i = 0; i < n; ++i) h_out[i] = c->series[static_cast<size_t>(i)];
  return MPR_OK;
}

int mpr_predict(mpr_ctx* c, double* d_pred) {
  if (!c || !d_pred) return fail(c, MPR_ERR_INVALID_ARG, "null pointer");
  TRY(ensure_chain(c));
  const Geom& g = c->lo.g;
  dim3 block(128), grid((g.L + 127) / 128, g.H);
  predict_kernel<<<grid, block, 0, c->stream>>>(c->d_values, c->d_mask, g, c->acc(), c->zmin, c->zmax, c->n_acc, d_pred);
  LAUNCH_OK(c);
  return MPR_OK;
}

int mpr_get_counters(mpr_ctx* c, uint64_t* accepted, uint64_t* attempted, uint64_t* sweeps) {
  if (!c) return MPR_ERR_INVALID_ARG;
  TRY(ensure_chain(c));
  unsigned long long h[kAcceptSlots];
  CUDA_OK(c, cudaMemcpyAsync(h, c->slots(), sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  CUDA_OK(c, cudaStreamSynchronize(c->stream));
  unsigned long long a = 0;
  for (int i = 0; i < kAcceptSlots; ++i) a += h[i];
  if (accepted) *accepted = a;
  if (attempted) *attempted = c->attempted;
  if (sweeps) *sweeps = c->sweep;
  return MPR_OK;
}

int64_t mpr_get_energy_series(mpr_ctx* c, double* out, int64_t cap) {
  if (!c) return MPR_ERR_INVALID_ARG;
  const int64_t n = static_cast<int64_t>(c->series.size());
  for (int64_t k = 0; out && k < n && k < cap; ++k) out[k] = c->series[k];
  return n;
}

int mpr_get_info(mpr_ctx* c, double* z_min, double* z_max, int64_t* n_free, double* T) {
  if (!c) return MPR_ERR_INVALID_ARG;
  if (!c->ws) return fail(c, MPR_ERR_WORKSPACE, "no workspace attached (mpr_set_workspace)");
  if (z_min) *z_min = c->zmin;
  if (z_max) *z_max = c->zmax;
  if (n_free) *n_free = c->n_free;
  if (T) *T = c->T;
  return MPR_OK;
}

int mpr_get_launch_stats(mpr_ctx* c, uint64_t* launches) {
  if (!c || !launches) return MPR_ERR_INVALID_ARG;
  *launches = c->launches;
  return MPR_OK;
}

int mpr_workspace_bytes_host_rect(int Lx, int Ly, size_t* bytes) {
  size_t b = 0;
  const int st = mpr_workspace_bytes_rect(Lx, Ly, &b);
  if (st != MPR_OK) return st;
  const size_t N = static_cast<size_t>(Lx) * Ly;
  *bytes = b + align_up(N * sizeof(double), 256) * 2 + align_up(N, 256);
  return MPR_OK;
}
int mpr_workspace_bytes_host(int L, size_t* bytes) {
  if (L < 2) return MPR_ERR_INVALID_ARG;
  return mpr_workspace_bytes_host_rect(L, L, bytes);
}

int mpr_predict_host(int L, const double* h_values, const uint8_t* h_mask, mpr_precision mode, uint64_t seed, double T,
                     int n_eq, int n_meas, void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                     double* h_pred, double* e_mean, double* e_stderr, double* T_used, uint64_t* launches) {
  if (L < 2) return MPR_ERR_INVALID_ARG;
  return mpr_predict_host_rect(L, L, h_values, h_mask, mode, seed, T, n_eq, n_meas, d_workspace, workspace_bytes, cuda_stream,
                               h_pred, e_mean, e_stderr, T_used, launches);
}

int mpr_predict_host_rect(int Lx, int Ly, const double* h_values, const uint8_t* h_mask, mpr_precision mode, uint64_t seed,
                          double T, int n_eq, int n_meas, void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                          double* h_pred, double* e_mean, double* e_stderr, double* T_used, uint64_t* launches) {
  size_t need = 0, core = 0;
  if (mpr_workspace_bytes_host_rect(Lx, Ly, &need) != MPR_OK || !h_values || !h_mask) return MPR_ERR_INVALID_ARG;
  mpr_workspace_bytes_rect(Lx, Ly, &core);
  if (!d_workspace || (reinterpret_cast<uintptr_t>(d_workspace) & 255u) || workspace_bytes < need)
    return MPR_ERR_WORKSPACE;
  const size_t N = static_cast<size_t>(Lx) * Ly;
  char* base = static_cast<char*>(d_workspace) + core;
  double* d_values = reinterpret_cast<double*>(base);
  double* d_pred = reinterpret_cast<double*>(base + align_up(N * sizeof(double), 256));
  uint8_t* d_mask = reinterpret_cast<uint8_t*>(base + 2 * align_up(N * sizeof(double), 256));
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  if (cudaMemcpyAsync(d_values, h_values, N * sizeof(double), cudaMemcpyHostToDevice, s) != cudaSuccess ||
      cudaMemcpyAsync(d_mask, h_mask, N, cudaMemcpyHostToDevice, s) != cudaSuccess)
    return MPR_ERR_CUDA;
  mpr_ctx* c = nullptr;
  int st = mpr_create_rect(&c, Lx, Ly, d_values, d_mask, d_workspace, core, cuda_stream);
  if (st != MPR_OK) return st;
  st = mpr_set_precision(c, mode);
  if (st != MPR_OK) { mpr_destroy(c); return st; }
  c->seed = seed;
  if (T > 0.0) {
    c->T = T;
    st = reset_chain(c, 0);
  } else {
    st = mpr_estimate_temperature(c, nullptr, nullptr, nullptr);
  }
  if (st == MPR_OK) st = mpr_run(c, n_eq, n_meas, h_pred ? d_pred : nullptr, e_mean, e_stderr);
  if (st == MPR_OK && h_pred) {
    if (cudaMemcpyAsync(h_pred, d_pred, N * sizeof(double), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaStreamSynchronize(s) != cudaSuccess)
      st = MPR_ERR_CUDA;
  }
  if (T_used) *T_used = c->T;
  if (launches) *launches = c->launches;
  mpr_destroy(c);
  return st;
}

void mpr_debug_trial_lengths(int* n_eq, int* n_meas) {
  if (n_eq) *n_eq = kTrialEq;
  if (n_meas) *n_meas = kTrialMeas;
}
double mpr_debug_proposal_width(double T) { return proposal_width(T); }
double mpr_debug_proposal_width_q(double T, double q) { return proposal_width(T, q); }

int mpr_debug_series_stats(const double* h_series, int64_t n, double* mean, double* se) {
  if (n < 0 || (n > 0 && !h_series)) return MPR_ERR_INVALID_ARG;
  const mpr_host::SeriesStats st = mpr_host::series_stats(h_series, static_cast<size_t>(n));
  if (mean) *mean = st.mean;
  if (se) *se = st.stderr_;
  return MPR_OK;
}

int mpr_debug_match_temperature(double e_sample, mpr_trial_fn trial, void* user, double* T_hat, int* n_trials) {
  if (!trial) return MPR_ERR_INVALID_ARG;
  mpr_host::TemperatureMatcher search;
  while (search.want_trial()) {
    double e = 0.0, se = 0.0;
    if (trial(search.T(), search.trials() + 1, &e, &se, user) != 0) return MPR_ERR_INVALID_ARG;
    search.report(e - e_sample, se);
  }
  if (n_trials) *n_trials = search.trials();
  if (search.outcome() != mpr_host::TemperatureMatcher::FOUND) return MPR_ERR_NO_ROOT;
  if (T_hat) *T_hat = search.result();
  return MPR_OK;
}

int mpr_debug_philox(const uint32_t* d_ctr, const uint32_t key[2], uint32_t* d_out, int64_t n, void* cuda_stream) {
  if (!d_ctr || !key || !d_out || n < 0) return MPR_ERR_INVALID_ARG;
  if (n == 0) return MPR_OK;
  philox_debug_kernel<<<static_cast<unsigned>((n + 255) / 256), 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
      d_ctr, key[0], key[1], d_out, n);
  return cudaGetLastError() == cudaSuccess ? MPR_OK : MPR_ERR_CUDA;
}

int mpr_debug_accept(const uint32_t* d_words, const double* d_mdE, double T, uint8_t* d_out, int64_t n, void* cuda_stream) {
  if (!d_words || !d_mdE || !d_out || n < 0 || !(T > 0.0)) return MPR_ERR_INVALID_ARG;
  if (n == 0) return MPR_OK;
  accept_debug_kernel<<<static_cast<unsigned>((n + 255) / 256), 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
      d_words, d_mdE, T, d_out, n);
  return cudaGetLastError() == cudaSuccess ? MPR_OK : MPR_ERR_CUDA;
}

}  // extern "C"
