// mpr_tiled.cuh -- the TILED path: one launch runs k whole hybrid sweeps (4k colour passes, R4)
// on a tile of both colour planes staged in shared memory by one 3-D TMA load (tile + halo of
// 4k sites on every side, out-of-grid elements zero-filled by the TMA unit).  After pass p the
// sites closer than p to the edge of the staged region are stale; they are never stored: each
// CTA writes back only its interior (distance >= 4k), into the other state buffer (ping-pong,
// because neighbouring tiles read each other's interiors as halo).  Halo sites are recomputed
// by both tiles with the same Philox counters (logical site index) and the same instruction
// sequence, so the result is bit-identical to the PLAIN path for every k.
//
// Staged region: TH rows x 64 plane columns (= 128 sites wide) x 2 planes, dense [plane][row][col].
// Work item = one row of one colour: a warp covers its 64 columns, every thread a PAIR of adjacent
// columns (2 lane, 2 lane + 1), read and written as one 16-byte (float modes) or two 16-byte (DP)
// shared-memory accesses.  Warp w owns the rows w, w + NW, w + 2 NW, ... for the whole launch, so
//  * the x-parity of its rows in a colour pass is a per-warp constant (NW is even): the left/right
//    neighbour selection is compiled in (template PAR), no per-site selects;
//  * the mask bits of a thread's sites (RPW rows x 2 colours x 2 sites) are read once from the
//    global bitmaps into one 64-bit register -- no mask staging in shared memory;
//  * all grid-boundary handling is done by zero vectors: TMA zero-fills what lies outside the
//    tensor and the plane columns past the grid hold (0, 0), so a missing neighbour adds nothing to
//    the local field (same sum, same order as the PLAIN path's selects: bit-identical).
// Moves are branch-free (mpr_device.cuh); every lane computes, a site keeps its new spin iff it is
// free and the move is accepted.
#pragma once
#include <cuda.h>
#include "mpr_device.cuh"
#include "mpr_plain.cuh"

namespace mpr {

static_assert(TmaType<double>::value == CU_TENSOR_MAP_DATA_TYPE_FLOAT64 && TmaType<float>::value == CU_TENSOR_MAP_DATA_TYPE_FLOAT32 &&
              TmaType<__half>::value == CU_TENSOR_MAP_DATA_TYPE_FLOAT16, "TmaType mirrors cuda.h");

constexpr int kTileCols = 64;   // plane columns staged per tile (incl. halo)

template <int MODE> struct TileCfg;
// PAIR_SYNC: synchronise two colour passes by pairwise named barriers between neighbouring warps
// (neighbour_sync) instead of __syncthreads.  Chosen per mode from an A/B run on one B200 at a
// constant 1965 MHz (L = 16384, ms per hybrid sweep, __syncthreads -> pairwise, two runs each):
// DP 4.279 -> 4.221, SP 3.555 -> 3.531, SP_PRECISE 1.616 -> 1.570, but SP_INTRINSIC 1.229 -> 1.247
// (at its 80-register cap the barrier ids spill, and its barrier waits were already covered by the
// second resident CTA), so that mode keeps __syncthreads.
// UNROLL: rows of a warp per iteration of the pass loop (0 = all RPW rows).  Even, so the row
// parities stay compile-time.  Double arithmetic: 2 (measured again after the Metropolis decision filter freed
// registers: DP 6 rows 3.67 -> 4.31 ms, SP 4 rows 2.98 -> 3.00 ms).  Float
// arithmetic, A/B at 1965 MHz, ms per sweep, full unroll -> 4: SP_INTRINSIC 1.2266 -> 1.2199 (and half
// the code), SP_PRECISE 1.570 -> 1.630, so only SP_INTRINSIC takes 4.
template <> struct TileCfg<MODE_DP>           { static constexpr int TH = 48, NT = 256, UNROLL = 2; static constexpr bool PAIR_SYNC = true; };
template <> struct TileCfg<MODE_SP>           { static constexpr int TH = 96, NT = 256, UNROLL = 2; static constexpr bool PAIR_SYNC = true; };
template <> struct TileCfg<MODE_SP_PRECISE>   { static constexpr int TH = 96, NT = 512, UNROLL = 0; static constexpr bool PAIR_SYNC = true; };
template <> struct TileCfg<MODE_SP_INTRINSIC> { static constexpr int TH = 96, NT = 384, UNROLL = 4; static constexpr bool PAIR_SYNC = false; };
template <> struct TileCfg<MODE_DS>           { static constexpr int TH = 48, NT = 384, UNROLL = 4; static constexpr bool PAIR_SYNC = false; };
template <> struct TileCfg<MODE_HP>           { static constexpr int TH = 96, NT = 384, UNROLL = 4; static constexpr bool PAIR_SYNC = false; };

inline int tiled_max_fused() { return 4; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TiledPlan {
  EncodeTiledFn encode = nullptr;
  bool attr_set[6] = {false, false, false, false, false, false};
};

enum { TILED_OK = 0, TILED_NO_DRIVER = 1, TILED_ENCODE = 2, TILED_ATTR = 3, TILED_LAUNCH = 4, TILED_TOO_MANY = 5 };

// the CUDA error behind the last TILED_LAUNCH / TILED_ATTR (for the message of mpr_last_error)
inline cudaError_t& tiled_last_cuda_error() { static cudaError_t e = cudaSuccess; return e; }

inline const char* tiled_error(int st) {
  switch (st) {
    case TILED_OK: return "ok";
    case TILED_NO_DRIVER: return "cuTensorMapEncodeTiled not found in the driver";
    case TILED_ENCODE: return "cuTensorMapEncodeTiled failed";
    case TILED_ATTR: return "cudaFuncSetAttribute(max dynamic shared memory) failed";
    case TILED_LAUNCH: return cudaGetErrorString(tiled_last_cuda_error());
    case TILED_TOO_MANY: return "too many tiles for the partials buffer";
    default: return "unknown";
  }
}

inline int tiled_plan_init(TiledPlan* p, const Geom&) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn ||
      q != cudaDriverEntryPointSuccess)
    return TILED_NO_DRIVER;
  p->encode = reinterpret_cast<EncodeTiledFn>(fn);
  return TILED_OK;
}

// ---- PTX wrappers: mbarrier + TMA (cp.async.bulk.tensor -> SASS UTMALDG) -------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}

// neighbour exchange between adjacent lanes; fp16 values travel as floats (exact both ways)
template <typename S> __device__ __forceinline__ S lane_dn(S v) { return __shfl_down_sync(0xffffffffu, v, 1); }
template <typename S> __device__ __forceinline__ S lane_up(S v) { return __shfl_up_sync(0xffffffffu, v, 1); }
template <> __device__ __forceinline__ __half lane_dn<__half>(__half v) { return __float2half_rn(__shfl_down_sync(0xffffffffu, __half2float(v), 1)); }
template <> __device__ __forceinline__ __half lane_up<__half>(__half v) { return __float2half_rn(__shfl_up_sync(0xffffffffu, __half2float(v), 1)); }

template <int MODE> constexpr size_t tile_smem_bytes() {
  return sizeof(typename Traits<MODE>::vec) * (2 * TileCfg<MODE>::TH + 1) * kTileCols   // spins + one pad row
         + 64;                                                                            // mbarrier
}

// Storage unit (mpr_plain.cuh): the two sites of plane columns (2m, 2m + 1) as (c_a, c_b, s_a, s_b):
// one 128-bit access in the float-storage modes, two in DP; (ca, cb) and (sa, sb) land in
// adjacent registers, i.e. they ARE the two-lane operands of the packed arithmetic.
template <typename S> struct alignas(4 * sizeof(S)) Unit { S ca, cb, sa, sb; };
constexpr int kRowScalars = 2 * kTileCols;

template <int MODE> struct TileView {
  using S = decltype(Traits<MODE>::vec::x);
  static constexpr int TH = TileCfg<MODE>::TH;
  S* base;   // [2][TH][kRowScalars]
  // unit of columns (2 u, 2 u + 1) in row r of plane pl
  __device__ __forceinline__ S* unit(int pl, int r, int u) const { return base + (pl * TH + r) * kRowScalars + 4 * u; }
};

// Local fields of the two sites of a unit of colour-plane row r from the other plane's units of
// the same columns in rows r - 1 (up), r (mid), r + 1 (dn) and the one extra site `ex`.
// par = x-parity of the row for this colour: the left/right neighbours of column j are the other
// plane's columns (j - 1 + par, j + par), so besides mid one more site is needed: column jj - 1
// (par = 0; lane b of the previous unit) or jj + 2 (par = 1; lane a of the next unit).
// Sum order l, r, u, d, lanes = (site a, site b): one packed add per term in the float modes.
template <int MODE>
__device__ __forceinline__ void combine_fields(int par, const Unit<decltype(Traits<MODE>::vec::x)>& up,
                                               const Unit<decltype(Traits<MODE>::vec::x)>& mid,
                                               const Unit<decltype(Traits<MODE>::vec::x)>& dn,
                                               decltype(Traits<MODE>::vec::x) exc, decltype(Traits<MODE>::vec::x) exs,
                                               Two<typename Traits<MODE>::real>* A, Two<typename Traits<MODE>::real>* B) {
  using R = typename Traits<MODE>::real;
  const Two<R> midc = mk2(R(mid.ca), R(mid.cb)), mids = mk2(R(mid.sa), R(mid.sb));
  Two<R> a, b;
  if (par == 0) {                   // a: l = ex, r = mid.a     b: l = mid.a, r = mid.b
    a = add2(mk2(R(exc), R(mid.ca)), midc);
    b = add2(mk2(R(exs), R(mid.sa)), mids);
  } else {                          // a: l = mid.a, r = mid.b  b: l = mid.b, r = ex
    a = add2(midc, mk2(R(mid.cb), R(exc)));
    b = add2(mids, mk2(R(mid.sb), R(exs)));
  }
  a = add2(a, mk2(R(up.ca), R(up.cb))); b = add2(b, mk2(R(up.sa), R(up.sb)));
  a = add2(a, mk2(R(dn.ca), R(dn.cb))); b = add2(b, mk2(R(dn.sa), R(dn.sb)));
  *A = a; *B = b;
}

// One row of a colour pass: the unit at `own` (row r, x-parity `par`) from the register window
// (up, mid, dn) of the other plane.  The extra neighbour comes from the adjacent lane by warp
// shuffle (wrong at lanes 0 / 31, for sites that are stale anyway).  Returns inc x accepted moves.
template <int MODE, int KIND>
__device__ __forceinline__ int row_step(int par, decltype(Traits<MODE>::vec::x)* own,
                                        const Unit<decltype(Traits<MODE>::vec::x)>& up,
                                        const Unit<decltype(Traits<MODE>::vec::x)>& mid,
                                        const Unit<decltype(Traits<MODE>::vec::x)>& dn,
                                        bool fa, bool fb, int inc, uint32_t pair_site, uint32_t sweep, uint32_t L,
                                        bool row_odd, const ChainConst<typename Traits<MODE>::real>& kc) {
  using R = typename Traits<MODE>::real;
  using S = decltype(Traits<MODE>::vec::x);
  const S exc = par ? lane_dn(mid.ca) : lane_up(mid.cb);
  const S exs = par ? lane_dn(mid.sa) : lane_up(mid.sb);
  Two<R> A, B;
  combine_fields<MODE>(par, up, mid, dn, exc, exs, &A, &B);
  const Unit<S> me = *reinterpret_cast<const Unit<S>*>(own);
  const Two<R> c = mk2(R(me.ca), R(me.cb)), s = mk2(R(me.sa), R(me.sb));
  R o[4];
  int n = 0;
  if constexpr (KIND == KIND_MET) {
    MetWords w0, w1;
    met_words_pair<MODE>(pair_site, sweep, L, par, row_odd, kc, &w0, &w1);
    bool ok[2];
    met_update2<MODE>(c, s, A, B, w0, w1, fa, fb, kc, o, ok);
    if (ok[0]) n += inc;
    if (ok[1]) n += inc;
  } else if constexpr (KIND == KIND_OR) {
    or_update2<MODE>(c, s, A, B, fa, fb, o);
  } else {
    quench_update2<MODE>(c, s, A, B, fa, fb, o);
  }
  Unit<S> out;
  out.ca = static_cast<S>(o[0]); out.cb = static_cast<S>(o[1]);
  out.sa = static_cast<S>(o[2]); out.sb = static_cast<S>(o[3]);
  *reinterpret_cast<Unit<S>*>(own) = out;
  return n;
}

// Synchronisation between two colour passes.  In a pass warp w writes its own RPW rows of one plane
// and reads rows w RPW - 1 .. (w + 1) RPW of the other: the only warps it exchanges data with are
// w - 1 and w + 1, so it need not wait for the whole CTA.  Two rounds of PAIRWISE named barriers
// (bar.sync id, 64): round A pairs (0,1), (2,3), ..., round B pairs (1,2), (3,4), ...  The pairs of a
// round are disjoint, so every round resolves in parallel (no ripple from warp 0 upwards), and a
// warp that has passed both rounds knows that both neighbours have finished the pass -- their
// writes are visible to it (RAW) and their reads of its rows are done (WAR for the next pass).
// Warps may drift apart by one pass per warp of distance, which also spreads the Philox /
// arithmetic / MUFU phases of the resident warps over time.  Ids 1 .. NW - 1; id 0 stays
// __syncthreads.  NW is even and <= 16.
template <int NW>
__device__ __forceinline__ void neighbour_sync(int warp) {
  static_assert(NW % 2 == 0 && NW >= 2 && NW <= 16, "pair barriers use ids 1 .. NW - 1 of the 16 hardware barriers");
  asm volatile("bar.sync %0, 64;" ::"r"(1 + (warp >> 1)) : "memory");                       // A: (w, w ^ 1)
  if (warp > 0 && warp < NW - 1)                                                             // B: odd w with w + 1
    asm volatile("bar.sync %0, 64;" ::"r"(NW / 2 + ((warp + 1) >> 1)) : "memory");
}

template <int MODE>
__device__ __forceinline__ void pass_sync(int warp) {
  if constexpr (TileCfg<MODE>::PAIR_SYNC) neighbour_sync<TileCfg<MODE>::NT / 32>(warp);
  else __syncthreads();
}

// One colour pass over the RPW contiguous rows of this warp.  The other plane's rows slide through
// a register window: each row is read from shared memory once per pass (RPW + 2 reads for RPW
// rows instead of 3 RPW).  COL, KIND and the row parities are compile-time constants: the first
// row of every warp has x-parity COL (y0 and RPW are even).  EVERY row is computed in every pass,
// without a test: the rows and columns within p sites of the rim of the staged region are stale
// after pass p whatever is done to them (they are recomputed by the neighbouring tile, never
// stored and never counted), and leaving the tests out keeps the warp free of branches.
// cnt = bit i set iff the CTA owns row i of this warp and this thread's columns.
// Returns the number of accepted Metropolis moves at sites this CTA owns (its interior).
template <int MODE, int KIND, int COL>
__device__ __forceinline__ int pass_rows(const TileView<MODE>& t, uint32_t mcol, uint32_t cnt,
                                         uint32_t site_row0, uint32_t L, uint32_t sweep,
                                         const ChainConst<typename Traits<MODE>::real>& kc) {
  using S = decltype(Traits<MODE>::vec::x);
  constexpr int TH = TileCfg<MODE>::TH, NW = TileCfg<MODE>::NT / 32, RPW = TH / NW;
  constexpr int kOther = (COL ? -1 : 1) * TH * kRowScalars;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  S* own = t.unit(COL, warp * RPW, lane);
  // row -1 does not exist: warp 0 reads row 0 instead (used by row 0 only, which is always stale);
  // row TH of plane 1 is the pad row behind the tile
  Unit<S> up = *reinterpret_cast<const Unit<S>*>(own + kOther - (warp > 0 ? kRowScalars : 0));
  Unit<S> mid = *reinterpret_cast<const Unit<S>*>(own + kOther);
  const uint32_t site = site_row0 + static_cast<uint32_t>(warp * RPW) * L;
  int n_acc = 0;
  // keeps the bit tests where they are used (hoisted out of the sweep loop they cost 24 registers)
  asm volatile("" : "+r"(mcol), "+r"(cnt));
  // unrolled bodies rotate the window by register renaming; the depth is per mode (TileCfg::UNROLL)
  constexpr int kUnroll = TileCfg<MODE>::UNROLL == 0 ? RPW : TileCfg<MODE>::UNROLL;
  static_assert(kUnroll % 2 == 0 && RPW % kUnroll == 0, "row parities must be compile-time constants");
#pragma unroll kUnroll
  for (int i = 0; i < RPW; ++i) {
    const int par = (COL + i) & 1;
    // the last row of the last warp has no row below it inside the tile: in a colour-1 pass the address
    // one row further is row 0 of plane 1, which warp 0 is writing -- read the row itself instead (the
    // value only feeds row TH - 1, which is stale from the first pass on); in a colour-0 pass it is the
    // zero-filled pad row behind plane 1
    const int dn_row = (COL == 1 && i == RPW - 1 && warp == NW - 1) ? i : i + 1;
    const Unit<S> dn = *reinterpret_cast<const Unit<S>*>(own + kOther + dn_row * kRowScalars);
    n_acc += row_step<MODE, KIND>(par, own + i * kRowScalars, up, mid, dn, (mcol >> (2 * i)) & 1u,
                                  (mcol >> (2 * i + 1)) & 1u, (cnt >> i) & 1u,
                                  site + static_cast<uint32_t>(i) * L + static_cast<uint32_t>(par), sweep, L,
                                  (i & 1) != 0, kc);      // tile origin and RPW are even: row parity = i & 1
    up = mid;
    mid = dn;
  }
  return n_acc;
}

// MEASURE: 0 = sweeps only; 1 = + energy sample (temperature trials, R6); 2 = + accumulation of phi (R15);
// 3 (kTiledQuench) = no sweeps but 2 nsweeps quench double passes (R8), same halo bookkeeping
constexpr int kTiledQuench = 3;
template <int MODE, int MEASURE>
__global__ void __launch_bounds__(TileCfg<MODE>::NT, 2)
tiled_sweep_kernel(const __grid_constant__ CUtensorMap tmap, typename Traits<MODE>::vec* __restrict__ dst,
                   const uint32_t* __restrict__ bits, double* __restrict__ acc, double* __restrict__ part,
                   unsigned long long* __restrict__ accept_slots, Geom g,
                   ChainConst<typename Traits<MODE>::real> kc, uint32_t first_sweep, int nsweeps, int tiles_x) {
  using R = typename Traits<MODE>::real;
  using V = typename Traits<MODE>::vec;
  constexpr int TH = TileCfg<MODE>::TH, NT = TileCfg<MODE>::NT, NW = NT / 32, RPW = TH / NW;
  static_assert(TH % NW == 0 && RPW % 2 == 0 && RPW * 2 <= 32, "row ownership / mask register layout");
  static_assert(TH % 2 == 0, "y0 = ty (TH - 8 k) - 4 k must be even: the first row of a warp has x-parity = colour");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  using S = decltype(V::x);
  TileView<MODE> t{reinterpret_cast<S*>(smem_raw)};
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + sizeof(V) * (2 * TH + 1) * kTileCols);
  __shared__ double red[32];

  const int h = 4 * nsweeps, hc = 2 * nsweeps;
  const int IC = kTileCols - 2 * hc, IR = TH - 2 * h;
  const int tx = blockIdx.x % tiles_x, ty = blockIdx.x / tiles_x;
  const int j0 = tx * IC - hc, y0 = ty * IR - h;    // j0 is even: pairs are aligned in the global planes too
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int jj = 2 * lane;

  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    mbar_expect_tx(bar, static_cast<uint32_t>(sizeof(V) * 2 * TH * kTileCols));
    tma_load_3d(t.base, &tmap, bar, (sizeof(S) == 2 ? 1 : 2) * j0, y0, 0);
  }
  // pad row behind plane 1 (read as "row TH" by the last warp in colour-0 passes): the zero vector
  if (threadIdx.x < kRowScalars) t.base[2 * TH * kRowScalars + threadIdx.x] = S(0);
  // mask bits of this thread's sites, one register per colour: bit 2 i + {0, 1} of mreg[col] = site
  // (row warp RPW + i, colour col, column jj + {0, 1}) is a prediction site.  (j0 + jj) is even, so
  // both bits sit in one word of the bitmap.
  uint32_t mreg[2] = {0u, 0u};
  {
    // the bitmaps are padded with zero words: no bounds test (mpr_plain.cuh)
    const int j = j0 + jj;
    const int sh = j & 31;
    const uint32_t* bp = mask_word(bits, g, 0, y0 + warp * RPW, j >> 5);
    const size_t colour = static_cast<size_t>(g.Hb) * g.Wb;
#pragma unroll
    for (int i = 0; i < RPW; ++i) {
      mreg[0] |= ((__ldg(bp) >> sh) & 3u) << (2 * i);
      mreg[1] |= ((__ldg(bp + colour) >> sh) & 3u) << (2 * i);
      bp += g.Wb;
    }
  }
  const bool col_interior = jj >= hc && jj < kTileCols - hc;
  // Philox counter word 0 of the first site of this thread's pair in tile row 0, without the parity
  const uint32_t site_row0 = g.site0 + static_cast<uint32_t>(y0) * static_cast<uint32_t>(g.L) + static_cast<uint32_t>(2 * (j0 + jj));
  const uint32_t Lu = static_cast<uint32_t>(g.L);
  __syncthreads();          // mbarrier initialised before anyone polls it
  mbar_wait(bar, 0);

  // rows and columns this CTA owns (for the accepted-move count)
  uint32_t cnt = 0;
  if (col_interior) {
#pragma unroll
    for (int i = 0; i < RPW; ++i) {
      const int r = warp * RPW + i;
      if (r >= h && r < TH - h) cnt |= 1u << i;
    }
  }
  // the rows among them that enter the accepted-move count and the energy sum: all, unless the context is a slab of a
  // larger grid (then its own rows only, Geom::own0 / own1)
  uint32_t cnt_c = 0;
#pragma unroll
  for (int i = 0; i < RPW; ++i) {
    const int row = y0 + warp * RPW + i;
    if (((cnt >> i) & 1u) && row >= g.own0 && row < g.own1) cnt_c |= 1u << i;
  }
  int n_acc = 0;
#pragma unroll 1
  for (int sw = 0; sw < nsweeps; ++sw) {
    const uint32_t sweep = first_sweep + static_cast<uint32_t>(sw);
    if constexpr (MEASURE == kTiledQuench) {
#pragma unroll 1
      for (int d = 0; d < 2; ++d) {
        pass_rows<MODE, KIND_QUENCH, 0>(t, mreg[0], cnt, site_row0, Lu, sweep, kc);
        pass_sync<MODE>(warp);
        pass_rows<MODE, KIND_QUENCH, 1>(t, mreg[1], cnt, site_row0, Lu, sweep, kc);
        pass_sync<MODE>(warp);
      }
      continue;
    }
    n_acc += pass_rows<MODE, KIND_MET, 0>(t, mreg[0], cnt_c, site_row0, Lu, sweep, kc);
    pass_sync<MODE>(warp);
    n_acc += pass_rows<MODE, KIND_MET, 1>(t, mreg[1], cnt_c, site_row0, Lu, sweep, kc);
    pass_sync<MODE>(warp);
    pass_rows<MODE, KIND_OR, 0>(t, mreg[0], cnt, site_row0, Lu, sweep, kc);
    pass_sync<MODE>(warp);
    pass_rows<MODE, KIND_OR, 1>(t, mreg[1], cnt, site_row0, Lu, sweep, kc);
    pass_sync<MODE>(warp);
  }

  // interior -> other state buffer (+ energy sample and accumulation of phi when measuring).
  // cnt already says which rows of this warp and whether this thread's columns are owned; what
  // is left is the edge of the grid (rows >= H, plane columns >= Wp).  Unrolled: one pointer each
  // for shared and global memory plus immediate / strided offsets.
  double esum = 0.0;
  {
    const int j = j0 + jj;                                        // even
    const int row0 = y0 + warp * RPW;
    const int nrows = g.H - row0;                                 // rows i < nrows lie in the grid
    const uint32_t own_rows = j < g.Wp ? cnt : 0u;
    const long long g0 = static_cast<long long>(row0) * g.Wp + j; // never dereferenced for rows outside
    S* gp = reinterpret_cast<S*>(dst) + 2 * g0;
    const S* sp = t.unit(0, warp * RPW, lane);
    const size_t grow = 2 * static_cast<size_t>(g.Wp), gplane = 2 * g.plane;
    constexpr int kEpiUnroll = MEASURE == 2 ? 1 : RPW;   // the measuring variant carries two atan2 per unit: keep it rolled
#pragma unroll kEpiUnroll
    for (int i = 0; i < RPW; ++i) {
      if (((own_rows >> i) & 1u) && i < nrows) {
        const Unit<S> u0 = *reinterpret_cast<const Unit<S>*>(sp + i * kRowScalars);
        const Unit<S> u1 = *reinterpret_cast<const Unit<S>*>(sp + (TH + i) * kRowScalars);
        *reinterpret_cast<Unit<S>*>(gp + i * grow) = u0;
        *reinterpret_cast<Unit<S>*>(gp + i * grow + gplane) = u1;
        if ((MEASURE == 1 || MEASURE == 2) && ((cnt_c >> i) & 1u)) {
          // every bond has exactly one colour-1 end: H = -J sum over colour-1 sites of their
          // site_energy_term (mpr_device.cuh; the same function as plain_energy_kernel).  The
          // neighbours are the other plane's units of rows r - 1, r, r + 1 and one extra site:
          // x-parity par = 0: site a has (l, r) = (ex, mid.a), site b (mid.a, mid.b);
          // par = 1: site a (mid.a, mid.b), site b (mid.b, ex)  -- as in combine_fields
          const S* oth = sp + i * kRowScalars;
          const int par = (row0 + i + 1) & 1;
          const Unit<S> mid = *reinterpret_cast<const Unit<S>*>(oth);
          const Unit<S> up = *reinterpret_cast<const Unit<S>*>(oth - kRowScalars);
          const Unit<S> dn = *reinterpret_cast<const Unit<S>*>(oth + kRowScalars);
          const R exc = R(oth[par ? 4 : -3]), exs = R(oth[par ? 6 : -1]);
          const R alc = par ? R(mid.ca) : exc, als = par ? R(mid.sa) : exs;
          const R arc = par ? R(mid.cb) : R(mid.ca), ars = par ? R(mid.sb) : R(mid.sa);
          const R blc = par ? R(mid.cb) : R(mid.ca), bls = par ? R(mid.sb) : R(mid.sa);
          const R brc = par ? exc : R(mid.cb), brs = par ? exs : R(mid.sb);
          energy_add(esum, site_energy_term<R>(R(u1.ca), R(u1.sa), alc, als, arc, ars, R(up.ca), R(up.sa), R(dn.ca), R(dn.sa)),
                     g.energy_single);
          energy_add(esum, site_energy_term<R>(R(u1.cb), R(u1.sb), blc, bls, brc, brs, R(up.cb), R(up.sb), R(dn.cb), R(dn.sb)),
                     g.energy_single);
        }
        if constexpr (MEASURE == 2) {
#pragma unroll
          for (int pl = 0; pl < 2; ++pl) {
            const Unit<S>& me = pl ? u1 : u0;
            const uint32_t mm = (mreg[pl] >> (2 * i)) & 3u;
            if (mm) {
              double* ap = acc + (g0 + static_cast<long long>(i) * g.Wp + static_cast<long long>(pl) * g.plane);
              double2 a2 = *reinterpret_cast<const double2*>(ap);
              if (mm & 1u) a2.x += spin_angle<MODE>(R(me.ca), R(me.sa));
              if (mm & 2u) a2.y += spin_angle<MODE>(R(me.cb), R(me.sb));
              *reinterpret_cast<double2*>(ap) = a2;
            }
          }
        }
      }
    }
  }
  if constexpr (MEASURE == 1 || MEASURE == 2) {
    const double e = block_sum(esum, red, g.energy_single);
    if (threadIdx.x == 0) part[blockIdx.x] = e;
  }
  const double a = block_sum(static_cast<double>(n_acc), red);
  if (threadIdx.x == 0 && a > 0.0)
    atomicAdd(accept_slots + (blockIdx.x & 1023u), static_cast<unsigned long long>(a));
}

template <int MODE>
int tiled_encode(TiledPlan& plan, const Geom& g, void* src, CUtensorMap* map) {
  using V = typename Traits<MODE>::vec;
  // fp16 storage travels as 32-bit words (two halves each): the copy is the same bytes, and the plain FLOAT32 path
  // of the TMA unit is the one every other mode has proven
  constexpr bool kHalf = sizeof(decltype(V::x)) == 2;
  const cuuint64_t dims[3] = {static_cast<cuuint64_t>(kHalf ? 1 : 2) * g.Wp, static_cast<cuuint64_t>(g.H), 2};
  const cuuint64_t strides[2] = {static_cast<cuuint64_t>(g.Wp) * sizeof(V), static_cast<cuuint64_t>(g.plane) * sizeof(V)};
  const cuuint32_t box[3] = {(kHalf ? 1 : 2) * kTileCols, static_cast<cuuint32_t>(TileCfg<MODE>::TH), 2};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = plan.encode(map, kHalf ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : static_cast<CUtensorMapDataType>(TmaType<decltype(V::x)>::value), 3, src,
                                 dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? TILED_OK : TILED_ENCODE;
}

template <int MODE>
int tiled_launch(TiledPlan& plan, const Geom& g, void* src, void* dst, const uint32_t* bits, double* acc, double* part,
                 unsigned long long* slots, ChainConst<typename Traits<MODE>::real> kc, uint32_t first_sweep, int k,
                 int measure, cudaStream_t stream, int* ntiles_out, long long max_partials) {
  using V = typename Traits<MODE>::vec;
  constexpr int TH = TileCfg<MODE>::TH, NT = TileCfg<MODE>::NT;
  if (!plan.encode) return TILED_NO_DRIVER;
  CUtensorMap map;
  const int es = tiled_encode<MODE>(plan, g, src, &map);
  if (es != TILED_OK) return es;
  constexpr size_t smem = tile_smem_bytes<MODE>();
  if (!plan.attr_set[MODE]) {
    if (cudaFuncSetAttribute(tiled_sweep_kernel<MODE, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(smem)) != cudaSuccess ||
        cudaFuncSetAttribute(tiled_sweep_kernel<MODE, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(smem)) != cudaSuccess ||
        cudaFuncSetAttribute(tiled_sweep_kernel<MODE, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(smem)) != cudaSuccess ||
        cudaFuncSetAttribute(tiled_sweep_kernel<MODE, kTiledQuench>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(smem)) != cudaSuccess)
      return TILED_ATTR;
    plan.attr_set[MODE] = true;
  }
  const int IC = kTileCols - 4 * k, IR = TH - 8 * k;
  const int tiles_x = (g.Wp + IC - 1) / IC, tiles_y = (g.H + IR - 1) / IR;
  const long long ntiles = static_cast<long long>(tiles_x) * tiles_y;
  // only the measuring launches write one partial per tile (they always run at k = 1)
  if ((measure == 1 || measure == 2) && ntiles > max_partials) return TILED_TOO_MANY;
  if (ntiles > 0x7fffffffLL) return TILED_TOO_MANY;
  if (measure == kTiledQuench)
    tiled_sweep_kernel<MODE, kTiledQuench><<<static_cast<unsigned>(ntiles), NT, smem, stream>>>(
        map, static_cast<V*>(dst), bits, acc, part, slots, g, kc, first_sweep, k, tiles_x);
  else if (measure == 2)
    tiled_sweep_kernel<MODE, 2><<<static_cast<unsigned>(ntiles), NT, smem, stream>>>(
        map, static_cast<V*>(dst), bits, acc, part, slots, g, kc, first_sweep, k, tiles_x);
  else if (measure == 1)
    tiled_sweep_kernel<MODE, 1><<<static_cast<unsigned>(ntiles), NT, smem, stream>>>(
        map, static_cast<V*>(dst), bits, acc, part, slots, g, kc, first_sweep, k, tiles_x);
  else
    tiled_sweep_kernel<MODE, 0><<<static_cast<unsigned>(ntiles), NT, smem, stream>>>(
        map, static_cast<V*>(dst), bits, acc, part, slots, g, kc, first_sweep, k, tiles_x);
  if (const cudaError_t le = cudaGetLastError(); le != cudaSuccess) { tiled_last_cuda_error() = le; return TILED_LAUNCH; }
  *ntiles_out = static_cast<int>(ntiles);
  return TILED_OK;
}

}  // namespace mpr
