// mpr_tiled.cuh -- the TILED path: one launch runs k whole hybrid sweeps (4k colour passes, R4)
// on a tile of both colour planes staged in shared memory by one 3-D TMA load (tile + halo of
// 4k sites on every side, out-of-grid elements zero-filled by the TMA unit).  After pass p the
// sites closer than p to the edge of the staged region are stale; they are never stored: each
// CTA writes back only its interior (distance >= 4k), into the other state buffer (ping-pong,
// because neighbouring tiles read each other's interiors as halo).  Halo sites are recomputed
// by both tiles with the same Philox counters (logical site index) and the same instruction
// sequence, so the result is bit-identical to the PLAIN path for every k.
//
// Staged region: TH rows x 64 plane columns (= 128 sites wide) x 2 planes, dense [plane][row][col],
// so a warp reads 32 consecutive vec's of one row: conflict-free shared-memory wavefronts.
#pragma once
#include <cuda.h>
#include "mpr_device.cuh"
#include "mpr_plain.cuh"

namespace mpr {

constexpr int kTileCols = 64;   // plane columns staged per tile (incl. halo)

template <int MODE> struct TileCfg;
template <> struct TileCfg<MODE_DP>           { static constexpr int TH = 48, NT = 256; };
template <> struct TileCfg<MODE_SP>           { static constexpr int TH = 96, NT = 256; };
template <> struct TileCfg<MODE_SP_PRECISE>   { static constexpr int TH = 96, NT = 512; };
template <> struct TileCfg<MODE_SP_INTRINSIC> { static constexpr int TH = 96, NT = 512; };

inline int tiled_max_fused() { return 4; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TiledPlan {
  EncodeTiledFn encode = nullptr;
  bool attr_set[4] = {false, false, false, false};
};

enum { TILED_OK = 0, TILED_NO_DRIVER = 1, TILED_ENCODE = 2, TILED_ATTR = 3, TILED_LAUNCH = 4, TILED_TOO_MANY = 5 };

inline const char* tiled_error(int st) {
  switch (st) {
    case TILED_OK: return "ok";
    case TILED_NO_DRIVER: return "cuTensorMapEncodeTiled not found in the driver";
    case TILED_ENCODE: return "cuTensorMapEncodeTiled failed";
    case TILED_ATTR: return "cudaFuncSetAttribute(max dynamic shared memory) failed";
    case TILED_LAUNCH: return "kernel launch failed";
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

template <int MODE> constexpr size_t tile_smem_bytes() {
  return sizeof(typename Traits<MODE>::vec) * 2 * TileCfg<MODE>::TH * kTileCols   // spins
         + sizeof(uint32_t) * 2 * TileCfg<MODE>::TH * 2                             // mask words
         + 64;                                                                      // mbarrier + reduction scratch pad
}

template <int MODE, bool MEASURE>
__global__ void __launch_bounds__(TileCfg<MODE>::NT, 2)
tiled_sweep_kernel(const __grid_constant__ CUtensorMap tmap, typename Traits<MODE>::vec* __restrict__ dst,
                   const uint32_t* __restrict__ bits, double* __restrict__ acc, double* __restrict__ part,
                   unsigned long long* __restrict__ accept_slots, Geom g,
                   ChainConst<typename Traits<MODE>::real> kc, uint32_t first_sweep, int nsweeps, int tiles_x) {
  using R = typename Traits<MODE>::real;
  using V = typename Traits<MODE>::vec;
  constexpr int TH = TileCfg<MODE>::TH, NT = TileCfg<MODE>::NT, NW = NT / 32;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  V (*tile)[TH][kTileCols] = reinterpret_cast<V (*)[TH][kTileCols]>(smem_raw);
  uint32_t (*mb)[TH][2] = reinterpret_cast<uint32_t (*)[TH][2]>(smem_raw + sizeof(V) * 2 * TH * kTileCols);
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw + sizeof(V) * 2 * TH * kTileCols + sizeof(uint32_t) * 2 * TH * 2);
  __shared__ double red[32];

  const int h = 4 * nsweeps, hc = 2 * nsweeps;
  const int IC = kTileCols - 2 * hc, IR = TH - 2 * h;
  const int tx = blockIdx.x % tiles_x, ty = blockIdx.x / tiles_x;
  const int j0 = tx * IC - hc, y0 = ty * IR - h;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    mbar_expect_tx(bar, static_cast<uint32_t>(sizeof(V) * 2 * TH * kTileCols));
    tma_load_3d(&tile[0][0][0], &tmap, bar, 2 * j0, y0, 0);
  }
  // mask words of the staged region, re-aligned to the tile's first column
  for (int i = threadIdx.x; i < 2 * TH * 2; i += NT) {
    const int w = i & 1, r = (i >> 1) % TH, p = (i >> 1) / TH;
    const int y = y0 + r;
    uint32_t word = 0;
    if (y >= 0 && y < g.L) {
      const uint32_t* row = bits + (static_cast<size_t>(p) * g.L + y) * g.Wm;
      const int jb = j0 + 32 * w;
      const int wi = jb >> 5, sh = jb & 31;   // arithmetic shift: floor for negative jb
      const uint32_t lo = (wi >= 0 && wi < g.Wm) ? row[wi] : 0u;
      const uint32_t hi = (wi + 1 >= 0 && wi + 1 < g.Wm) ? row[wi + 1] : 0u;
      word = __funnelshift_r(lo, hi, sh);
    }
    mb[p][r][w] = word;
  }
  __syncthreads();
  mbar_wait(bar, 0);

  int n_acc = 0;
  for (int sw = 0; sw < nsweeps; ++sw) {
    const uint32_t sweep = first_sweep + static_cast<uint32_t>(sw);
#pragma unroll 1
    for (int pass = 0; pass < 4; ++pass) {
      const int col = pass & 1;
      const int p = 4 * sw + pass + 1;
      const int nitems = (TH - 2 * p) * 2;
      for (int item = warp; item < nitems; item += NW) {
        const int r = p + (item >> 1), half = item & 1;
        const int y = y0 + r;
        if (y < 0 || y >= g.L) continue;
        const int jj = half * 32 + lane;
        if (!((mb[col][r][half] >> lane) & 1u)) continue;
        const int par = x_parity(y, col);
        const int x = 2 * (j0 + jj) + par;
        const bool hl = x > 0, hr = x < g.L - 1, hu = y > 0, hd = y < g.L - 1;
        int jl = jj - 1 + par, jr = jj + par;
        jl = jl < 0 ? 0 : jl;
        jr = jr > kTileCols - 1 ? kTileCols - 1 : jr;
        const V l = tile[1 - col][r][jl];
        const V rr = tile[1 - col][r][jr];
        const V u = tile[1 - col][r - 1][jj];
        const V d = tile[1 - col][r + 1][jj];
        R A, B;
        local_field<R>(R(l.x), R(l.y), R(rr.x), R(rr.y), R(u.x), R(u.y), R(d.x), R(d.y), hl, hr, hu, hd, &A, &B);
        const V me = tile[col][r][jj];
        R c = R(me.x), s = R(me.y);
        if (pass < 2) {
          const bool ok = met_update<MODE>(&c, &s, A, B, static_cast<uint32_t>(y) * static_cast<uint32_t>(g.L) + x,
                                           sweep, kc);
          if (ok && r >= h && r < TH - h && jj >= hc && jj < kTileCols - hc) n_acc += 1;
        } else {
          or_update<MODE>(&c, &s, A, B);
        }
        V out;
        out.x = static_cast<decltype(out.x)>(c);
        out.y = static_cast<decltype(out.y)>(s);
        tile[col][r][jj] = out;
      }
      __syncthreads();
    }
  }

  // interior -> other state buffer (+ energy sample and accumulation of phi when measuring)
  double esum = 0.0;
  const int nint = IR * 2 * 2;   // rows x planes x halves
  for (int item = warp; item < nint; item += NW) {
    const int half = item & 1, pl = (item >> 1) & 1, r = h + (item >> 2);
    const int y = y0 + r;
    if (y >= g.L) continue;
    const int jj = half * 32 + lane;
    const int j = j0 + jj;
    if (jj < hc || jj >= kTileCols - hc || j >= g.Wp) continue;
    const V me = tile[pl][r][jj];
    const size_t gi = static_cast<size_t>(pl) * g.plane + static_cast<size_t>(y) * g.Wp + j;
    dst[gi] = me;
    if constexpr (MEASURE) {
      const int par = x_parity(y, pl);
      const int x = 2 * j + par;
      if (pl == 1 && x < g.L) {
        const bool hl = x > 0, hr = x < g.L - 1, hu = y > 0, hd = y < g.L - 1;
        const V l = tile[0][r][jj - 1 + par];
        const V rr = tile[0][r][jj + par];
        const V u = tile[0][r - 1][jj];
        const V d = tile[0][r + 1][jj];
        R A, B;
        local_field<R>(R(l.x), R(l.y), R(rr.x), R(rr.y), R(u.x), R(u.y), R(d.x), R(d.y), hl, hr, hu, hd, &A, &B);
        esum += static_cast<double>(fma_(R(me.x), A, R(me.y) * B));
      }
      if ((mb[pl][r][half] >> lane) & 1u) acc[gi] += spin_angle<MODE>(R(me.x), R(me.y));
    }
  }
  if constexpr (MEASURE) {
    const double e = block_sum(esum, red);
    if (threadIdx.x == 0) part[blockIdx.x] = e;
  }
  const double a = block_sum(static_cast<double>(n_acc), red);
  if (threadIdx.x == 0 && a > 0.0)
    atomicAdd(accept_slots + (blockIdx.x & 1023u), static_cast<unsigned long long>(a));
}

template <int MODE>
int tiled_encode(TiledPlan& plan, const Geom& g, void* src, CUtensorMap* map) {
  using V = typename Traits<MODE>::vec;
  constexpr bool f64 = sizeof(V) == 16;
  const cuuint64_t dims[3] = {static_cast<cuuint64_t>(2) * g.Wp, static_cast<cuuint64_t>(g.L), 2};
  const cuuint64_t strides[2] = {static_cast<cuuint64_t>(g.Wp) * sizeof(V), static_cast<cuuint64_t>(g.plane) * sizeof(V)};
  const cuuint32_t box[3] = {2 * kTileCols, static_cast<cuuint32_t>(TileCfg<MODE>::TH), 2};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = plan.encode(map, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, src,
                                 dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? TILED_OK : TILED_ENCODE;
}

template <int MODE>
int tiled_launch(TiledPlan& plan, const Geom& g, void* src, void* dst, const uint32_t* bits, double* acc, double* part,
                 unsigned long long* slots, ChainConst<typename Traits<MODE>::real> kc, uint32_t first_sweep, int k,
                 bool measure, cudaStream_t stream, int* ntiles_out) {
  using V = typename Traits<MODE>::vec;
  constexpr int TH = TileCfg<MODE>::TH, NT = TileCfg<MODE>::NT;
  if (!plan.encode) return TILED_NO_DRIVER;
  CUtensorMap map;
  const int es = tiled_encode<MODE>(plan, g, src, &map);
  if (es != TILED_OK) return es;
  constexpr size_t smem = tile_smem_bytes<MODE>();
  if (!plan.attr_set[MODE]) {
    if (cudaFuncSetAttribute(tiled_sweep_kernel<MODE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(smem)) != cudaSuccess ||
        cudaFuncSetAttribute(tiled_sweep_kernel<MODE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(smem)) != cudaSuccess)
      return TILED_ATTR;
    plan.attr_set[MODE] = true;
  }
  const int IC = kTileCols - 4 * k, IR = TH - 8 * k;
  const int tiles_x = (g.Wp + IC - 1) / IC, tiles_y = (g.L + IR - 1) / IR;
  const long long ntiles = static_cast<long long>(tiles_x) * tiles_y;
  if (ntiles > (1 << 18)) return TILED_TOO_MANY;
  if (measure)
    tiled_sweep_kernel<MODE, true><<<static_cast<unsigned>(ntiles), NT, smem, stream>>>(
        map, static_cast<V*>(dst), bits, acc, part, slots, g, kc, first_sweep, k, tiles_x);
  else
    tiled_sweep_kernel<MODE, false><<<static_cast<unsigned>(ntiles), NT, smem, stream>>>(
        map, static_cast<V*>(dst), bits, acc, part, slots, g, kc, first_sweep, k, tiles_x);
  if (cudaGetLastError() != cudaSuccess) return TILED_LAUNCH;
  *ntiles_out = static_cast<int>(ntiles);
  return TILED_OK;
}

}  // namespace mpr
