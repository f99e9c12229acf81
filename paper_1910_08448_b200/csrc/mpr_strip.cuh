// mpr_strip.cuh -- the STRIP path: every WARP owns a column strip of the grid (64 plane columns =
// 128 sites wide) over a segment of rows and streams the rows through a private ring in shared
// memory, with the colour passes of the launch running as a software pipeline down the rows:
//
//     stage p (p = 0 .. NS-1) works on row t - 2p at step t          (lag 2 rows per stage)
//
// Stage p + 1 at row r needs the rows r - 1 .. r + 1 as stage p left them; with a lag of two rows
// those were all finished in EARLIER steps, so the NS stages of one step are independent of each
// other: a warp carries NS independent dependency chains (two Metropolis + two over-relaxation
// updates in the R4 program) through every step, without any barrier -- a lane only ever touches
// its own column of the ring (left / right neighbours come by warp shuffle), so there is no
// CTA-wide and not even a warp-wide synchronisation in the data path.  Compared with the TILED
// path: no redundant halo ROWS (a segment pays 2 NS + 6 warm-up / drain rows once, the columns
// keep the 64 / (64 - NS) redundancy), no bulk-synchronous pass phases, results go from registers
// straight to global memory.
//
// Rows enter the ring in chunks of 4 rows x 2 colour planes by one 3-D TMA load per chunk
// (cp.async.bulk.tensor -> UTMALDG.3D, out-of-grid elements zero-filled) issued by lane 0 one
// chunk ahead of its use and awaited on a per-slot mbarrier.  The ring has just enough slots for
// the 2 NS + 1 live rows plus the chunk in flight.
//
// The per-site arithmetic is that of mpr_device.cuh, called with the same operands in the same
// order as the PLAIN kernels: the spins are bit-identical on all three paths.  Stale data: the
// sites within p of the left / right rim of the strip are wrong after stage p (their neighbour
// shuffle has no partner) and the rows above the first loaded one do not exist; none of them is
// ever stored to global memory or counted.
#pragma once
#include <cuda.h>
#include "mpr_device.cuh"
#include "mpr_plain.cuh"
#include "mpr_tiled.cuh"   // Unit, combine_fields, mbarrier / TMA wrappers

namespace mpr {

constexpr int kStripRB = 4;      // rows per TMA chunk
constexpr int kStripLag = 2;     // rows between consecutive pipeline stages

// What one launch does: the sequence of colour passes ("stages").
//   PROG_R4     k hybrid sweeps in the R4 order: MET c0, MET c1, OR c0, OR c1      NS = 4 k
//   PROG_FUSED  k hybrid sweeps in the site-fused order (R4b): [MET+OR] c0, [MET+OR] c1   NS = 2 k
//   PROG_QUENCH k quench double passes (R8): Q c0, Q c1                                  NS = 2 k
enum { PROG_R4 = 0, PROG_FUSED = 1, PROG_QUENCH = 2 };

template <int PROG, int K> struct StripProg {
  static constexpr int NS = PROG == PROG_R4 ? 4 * K : 2 * K;
  static __host__ __device__ constexpr int kind(int p) {
    return PROG == PROG_R4 ? ((p & 2) ? KIND_OR : KIND_MET) : PROG == PROG_FUSED ? KIND_MO : KIND_QUENCH;
  }
  static __host__ __device__ constexpr int sweep_off(int p) { return PROG == PROG_R4 ? p / 4 : PROG == PROG_FUSED ? p / 2 : 0; }
  static constexpr int SWEEPS = PROG == PROG_QUENCH ? 0 : K;
};

__host__ __device__ constexpr int strip_halo_lanes(int ns) { return (ns + 3) / 4; }            // stale lanes per side after ns stages
__host__ __device__ constexpr int strip_interior_cols(int ns) { return kTileCols - 4 * strip_halo_lanes(ns); }
__host__ __device__ constexpr int strip_slots(int ns) { return (2 * ns + 1 + kStripRB - 1) / kStripRB + 1; }
__host__ __device__ constexpr int strip_lead_rows(int ns) { return (ns + kStripRB - 1) / kStripRB * kStripRB; }   // rows loaded above a segment

// warps per CTA (one CTA per SM): as many as their rings fit into 216 KiB of shared memory, at most 12
// (the ring of a warp is 16 KiB with float storage and NS = 4, 32 KiB in DP)
template <int MODE, int NS> struct StripCfg {
  static constexpr int kRingBytes = strip_slots(NS) * 2 * kStripRB * 2 * kTileCols * static_cast<int>(sizeof(decltype(Traits<MODE>::vec::x)));
  static constexpr int kFit = (216 * 1024) / kRingBytes;
  static constexpr int NW = kFit < 12 ? kFit : 12;
};

struct StripGeom {
  int n_strips, n_seg, seg_rows;   // items = n_strips * n_seg, item -> (strip = item % n_strips, seg = item / n_strips)
  int n_items;
};

template <int MODE, int NS> constexpr size_t strip_smem_bytes() {
  using S = decltype(Traits<MODE>::vec::x);
  return static_cast<size_t>(StripCfg<MODE, NS>::NW) * strip_slots(NS) * (2 * kStripRB * kRowScalars * sizeof(S) + sizeof(uint64_t)) + 128;
}

__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// MEASURE: 0 = none; 1 = + energy sample after the last stage; 2 = + accumulation of phi (R15)
template <int MODE, int PROG, int K, int MEASURE>
__global__ void __launch_bounds__(StripCfg<MODE, StripProg<PROG, K>::NS>::NW * 32, 1)
strip_kernel(const __grid_constant__ CUtensorMap tmap, typename Traits<MODE>::vec* __restrict__ dst,
             const uint32_t* __restrict__ bits, double* __restrict__ acc, double* __restrict__ part,
             unsigned long long* __restrict__ accept_slots, Geom g, ChainConst<typename Traits<MODE>::real> kc,
             uint32_t first_sweep, StripGeom sg) {
  using R = typename Traits<MODE>::real;
  using V = typename Traits<MODE>::vec;
  using S = decltype(V::x);
  using P = StripProg<PROG, K>;
  constexpr int NS = P::NS, NW = StripCfg<MODE, NS>::NW, RB = kStripRB, LAG = kStripLag;
  constexpr int NSLOT = strip_slots(NS), HL = strip_halo_lanes(NS), IC = strip_interior_cols(NS);
  constexpr int CHUNK = 2 * RB * kRowScalars;          // scalars per chunk: [plane][row][128]
  constexpr int PLANE = RB * kRowScalars;
  static_assert(MEASURE == 0 || K == 1, "measuring launches carry one sweep");
  static_assert(LAG * (NS - 1) * 2 + 4 <= 32, "mask queue: 2 bits per row in a 32-bit register");

  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ double red[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  S* const ring = reinterpret_cast<S*>(smem_raw) + static_cast<size_t>(warp) * NSLOT * CHUNK;
  uint64_t* const bars = reinterpret_cast<uint64_t*>(smem_raw + static_cast<size_t>(NW) * NSLOT * CHUNK * sizeof(S)) + warp * NSLOT;

  const int item = blockIdx.x * NW + warp;
  int n_acc = 0;
  double esum = 0.0;
  if (item < sg.n_items) {
    const int strip = item % sg.n_strips, seg = item / sg.n_strips;
    const int j0 = strip * IC - 2 * HL;                       // plane column of lane 0 (even)
    const int yb = seg * sg.seg_rows;
    const int ye = min(g.L, yb + sg.seg_rows);
    const int t0 = yb - strip_lead_rows(NS);                  // first loaded row (multiple of 4 below yb, even)
    const int n_steps = ye - t0 + LAG * (NS - 1);             // the last stage finishes row ye - 1 in the last step
    const int n_iter = (n_steps + RB - 1) / RB;
    const int j = j0 + 2 * lane;
    const bool lane_ok = lane >= HL && lane < 32 - HL && j < g.Wp;

    if (lane == 0) {
#pragma unroll
      for (int k = 0; k < NSLOT; ++k) mbar_init(bars + k, 1);
    }
    __syncwarp();
    constexpr uint32_t kChunkBytes = CHUNK * sizeof(S);
    if (lane == 0) {                                          // chunk 0 -> slot 0
      mbar_expect_tx(bars, kChunkBytes);
      tma_load_3d(ring, &tmap, bars, 2 * j0, t0, 0);
    }
    // cb[k] = scalar offset (inside this warp's ring) of the chunk  i + 2 - NSLOT + k,  i.e. cb[NSLOT-1] holds
    // chunk i + 1 (in flight), cb[NSLOT-2] chunk i, cb[0] the oldest live one.  Chunk c lives in slot c % NSLOT.
    int cb[NSLOT];
#pragma unroll
    for (int k = 0; k < NSLOT; ++k) cb[k] = ((k + 2) % NSLOT) * CHUNK;    // iteration 0: chunk k + 2 - NSLOT
    int slot_next = 1 % NSLOT;                                // slot of chunk i + 1
    uint32_t phase_bits = 0;                                  // bit s = parity the next wait on slot s expects

    // mask bits: queue per colour, 2 bits per row, row t at bits 0..1, row t - d at bits 2d..2d+1
    uint32_t mq[2] = {0u, 0u};
    const int sh = j & 31;
    const uint32_t* bp = mask_word(bits, g, 0, t0, j >> 5);
    const size_t colour_words = static_cast<size_t>(g.Hb) * g.Wb;
    uint32_t nxt0 = (__ldg(bp) >> sh) & 3u, nxt1 = (__ldg(bp + colour_words) >> sh) & 3u;    // row t0

    const uint32_t Lu = static_cast<uint32_t>(g.L);
    uint32_t site_t = static_cast<uint32_t>(t0) * Lu + static_cast<uint32_t>(2 * j);         // Philox word 0 of row t, no parity
    // global pointers of this lane's unit in row t of plane 0 (dst / accumulator); never dereferenced outside the grid
    const long long g_t0 = static_cast<long long>(t0) * g.Wp + j;
    S* gp = reinterpret_cast<S*>(dst) + 2 * g_t0;
    double* ap = acc + g_t0;
    const long long grow = 2 * static_cast<long long>(g.Wp), gplane = 2 * static_cast<long long>(g.plane);

    mbar_wait(bars, 0);
    phase_bits ^= 1u;

#pragma unroll 1
    for (int i = 0; i < n_iter; ++i) {
      // prefetch chunk i + 1 into the slot whose old chunk (i + 1 - NSLOT) nobody reads any more
      __syncwarp();
      if (lane == 0) {
        fence_proxy_async_smem();
        mbar_expect_tx(bars + slot_next, kChunkBytes);
        tma_load_3d(ring + cb[NSLOT - 1], &tmap, bars + slot_next, 2 * j0, t0 + RB * (i + 1), 0);
      }
#pragma unroll
      for (int u = 0; u < RB; ++u) {
        if (u == RB - 1) {                                    // row 4 i + 4 (first of chunk i + 1) is read from here on
          mbar_wait(bars + slot_next, (phase_bits >> slot_next) & 1u);
          phase_bits ^= 1u << slot_next;
        }
        const int n = RB * i + u;                             // step number; row t = t0 + n
        const int t = t0 + n;
        // ---- mask bits of row t enter the queues; those of row t + 1 are fetched for the next step
        mq[0] = (mq[0] << 2) | nxt0;
        mq[1] = (mq[1] << 2) | nxt1;
        bp += g.Wb;
        nxt0 = (__ldg(bp) >> sh) & 3u;
        nxt1 = (__ldg(bp + colour_words) >> sh) & 3u;

        // ---- gather: own unit and local fields of every stage (all reads before any write of this step)
        Two<R> A[NS], B[NS], c[NS], s[NS];
        S* own[NS];
        Unit<S> nb_l[1], nb_m[1], nb_u[1], nb_d[1];           // float-mode energy: the last stage's neighbours
        S exc_last = S(0), exs_last = S(0);
#pragma unroll
        for (int p = 0; p < NS; ++p) {
          const int col = p & 1, par = (u + col) & 1;         // t0 and LAG are even: x-parity of row t - 2p is (u + col) & 1
          const int rel = u - LAG * p;                        // row relative to 4 i
          auto at = [&](int plane, int r) -> S* {
            const int q = (r >= 0) ? r / RB : -((-r + RB - 1) / RB);      // floor(r / RB)
            return ring + cb[NSLOT - 2 + q] + plane * PLANE + (r - q * RB) * kRowScalars + 4 * lane;
          };
          own[p] = at(col, rel);
          const Unit<S> up = *reinterpret_cast<const Unit<S>*>(at(1 - col, rel - 1));
          const Unit<S> mid = *reinterpret_cast<const Unit<S>*>(at(1 - col, rel));
          const Unit<S> dn = *reinterpret_cast<const Unit<S>*>(at(1 - col, rel + 1));
          const Unit<S> me = *reinterpret_cast<const Unit<S>*>(own[p]);
          const S exc = par ? __shfl_down_sync(0xffffffffu, mid.ca, 1) : __shfl_up_sync(0xffffffffu, mid.cb, 1);
          const S exs = par ? __shfl_down_sync(0xffffffffu, mid.sa, 1) : __shfl_up_sync(0xffffffffu, mid.sb, 1);
          combine_fields<MODE>(par, up, mid, dn, exc, exs, &A[p], &B[p]);
          c[p] = mk2(R(me.ca), R(me.cb));
          s[p] = mk2(R(me.sa), R(me.sb));
          if (MEASURE != 0 && sizeof(R) == 4 && p == NS - 1) {
            nb_u[0] = up; nb_m[0] = mid; nb_d[0] = dn; exc_last = exc; exs_last = exs;
          }
        }
        (void)nb_l;

        // ---- compute
        R o[NS][4];
#pragma unroll
        for (int p = 0; p < NS; ++p) {
          const int col = p & 1, par = (u + col) & 1;
          const uint32_t mbits = mq[col] >> (2 * LAG * p);
          const bool fa = mbits & 1u, fb = mbits & 2u;
          const int row = t - LAG * p;
          const bool counted = lane_ok && row >= yb && row < ye;
          constexpr int dummy = 0; (void)dummy;
          const int kind = P::kind(p);
          if (kind == KIND_MET || kind == KIND_MO) {
            const uint32_t pair_site = site_t - static_cast<uint32_t>(LAG * p) * Lu + static_cast<uint32_t>(par);
            MetWords w0, w1;
            met_words_pair<MODE>(pair_site, first_sweep + static_cast<uint32_t>(P::sweep_off(p)), kc, &w0, &w1);
            bool ok[2];
            met_update2<MODE>(c[p], s[p], A[p], B[p], w0, w1, fa, fb, kc, o[p], ok);
            if (counted) n_acc += static_cast<int>(ok[0]) + static_cast<int>(ok[1]);
            if (kind == KIND_MO) {
              R o2[4];
              or_update2<MODE>(mk2(o[p][0], o[p][1]), mk2(o[p][2], o[p][3]), A[p], B[p], fa, fb, o2);
              o[p][0] = o2[0]; o[p][1] = o2[1]; o[p][2] = o2[2]; o[p][3] = o2[3];
            }
          } else if (kind == KIND_OR) {
            or_update2<MODE>(c[p], s[p], A[p], B[p], fa, fb, o[p]);
          } else {
            quench_update2<MODE>(c[p], s[p], A[p], B[p], fa, fb, o[p]);
          }
        }

        // ---- scatter: ring (stages whose row is loaded), global memory (final stage of each colour, owned rows)
#pragma unroll
        for (int p = 0; p < NS; ++p) {
          const int col = p & 1;
          const int row = t - LAG * p;
          Unit<S> out;
          out.ca = static_cast<S>(o[p][0]); out.cb = static_cast<S>(o[p][1]);
          out.sa = static_cast<S>(o[p][2]); out.sb = static_cast<S>(o[p][3]);
          if (n >= LAG * p) *reinterpret_cast<Unit<S>*>(own[p]) = out;       // rows above t0 do not exist
          if (p >= NS - 2) {                                                   // last stage of this colour
            const bool owned = lane_ok && row >= yb && row < ye;
            if (owned) {
              *reinterpret_cast<Unit<S>*>(gp - (LAG * p) * grow + col * gplane) = out;
              if (MEASURE == 2) {
                const uint32_t mm = (mq[col] >> (2 * LAG * p)) & 3u;
                if (mm) {
                  double* a = ap - static_cast<long long>(LAG * p) * g.Wp + static_cast<long long>(col) * static_cast<long long>(g.plane);
                  double2 a2 = *reinterpret_cast<const double2*>(a);
                  if (mm & 1u) a2.x += spin_angle<MODE>(o[p][0], o[p][2]);
                  if (mm & 2u) a2.y += spin_angle<MODE>(o[p][1], o[p][3]);
                  *reinterpret_cast<double2*>(a) = a2;
                }
              }
              if (MEASURE != 0 && p == NS - 1) {
                // every bond has exactly one colour-1 end: H = -J sum over colour-1 sites of site_energy_term
                // with the final spins; the neighbours (colour 0) were final when this stage gathered them
                if constexpr (sizeof(R) == 8) {
                  R Aa, Ab, Ba, Bb;
                  un2(A[p], &Aa, &Ab); un2(B[p], &Ba, &Bb);
                  esum += static_cast<double>(fma_(o[p][0], Aa, o[p][2] * Ba));
                  esum += static_cast<double>(fma_(o[p][1], Ab, o[p][3] * Bb));
                } else {
                  const int par = (u + col) & 1;
                  const Unit<S>& mid = nb_m[0];
                  const R alc = par ? R(mid.ca) : R(exc_last), als = par ? R(mid.sa) : R(exs_last);
                  const R arc = par ? R(mid.cb) : R(mid.ca), ars = par ? R(mid.sb) : R(mid.sa);
                  const R blc = par ? R(mid.cb) : R(mid.ca), bls = par ? R(mid.sb) : R(mid.sa);
                  const R brc = par ? R(exc_last) : R(mid.cb), brs = par ? R(exs_last) : R(mid.sb);
                  esum += site_energy_term<R>(o[p][0], o[p][2], alc, als, arc, ars, R(nb_u[0].ca), R(nb_u[0].sa),
                                              R(nb_d[0].ca), R(nb_d[0].sa));
                  esum += site_energy_term<R>(o[p][1], o[p][3], blc, bls, brc, brs, R(nb_u[0].cb), R(nb_u[0].sb),
                                              R(nb_d[0].cb), R(nb_d[0].sb));
                }
              }
            }
          }
        }
        site_t += Lu;
        gp += grow;
        ap += g.Wp;
      }
      // rotate: the oldest chunk's slot receives chunk i + 2 in the next iteration
      const int freed = cb[0];
#pragma unroll
      for (int k = 0; k + 1 < NSLOT; ++k) cb[k] = cb[k + 1];
      cb[NSLOT - 1] = freed;
      slot_next = slot_next + 1 == NSLOT ? 0 : slot_next + 1;
    }
    // every chunk issued was awaited inside its iteration: nothing is in flight here
  }
  if constexpr (MEASURE != 0) {
    const double e = block_sum(esum, red);
    if (threadIdx.x == 0) part[blockIdx.x] = e;
  }
  if constexpr (PROG != PROG_QUENCH) {
    const double a = block_sum(static_cast<double>(n_acc), red);
    if (threadIdx.x == 0 && a > 0.0)
      atomicAdd(accept_slots + (blockIdx.x & 1023u), static_cast<unsigned long long>(a));
  }
}

// ---- host side -------------------------------------------------------------------------------
struct StripPlan {
  int sm_count = 0;
  bool attr_set[4] = {false, false, false, false};
  // tensor maps are encoded once per (state buffer, element width): the two buffers ping-pong
  CUtensorMap map[2][2];
  void* map_src[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};
};

template <int MODE>
int strip_encode(TiledPlan& tp, const Geom& g, void* src, CUtensorMap* map) {
  using V = typename Traits<MODE>::vec;
  constexpr bool f64 = sizeof(V) == 16;
  const cuuint64_t dims[3] = {static_cast<cuuint64_t>(2) * g.Wp, static_cast<cuuint64_t>(g.L), 2};
  const cuuint64_t strides[2] = {static_cast<cuuint64_t>(g.Wp) * sizeof(V), static_cast<cuuint64_t>(g.plane) * sizeof(V)};
  const cuuint32_t box[3] = {2 * kTileCols, static_cast<cuuint32_t>(kStripRB), 2};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = tp.encode(map, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, src,
                               dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                               CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? TILED_OK : TILED_ENCODE;
}

// Segments per strip: as many as fill the resident warps (sm_count * NW), but no shorter than the point where the
// warm-up / drain rows (2 NS + 6 per segment) would cost more than the idle warps they save.
inline StripGeom strip_geometry(const Geom& g, int ns, int nw, int sm_count) {
  StripGeom sg;
  const int ic = strip_interior_cols(ns);
  sg.n_strips = (g.Wp + ic - 1) / ic;
  const int slots = sm_count * nw;
  const int overhead = strip_lead_rows(ns) + kStripLag * (ns - 1) + 3;      // steps a segment runs beyond its own rows
  int best_seg = 1;
  double best_cost = 1e300;
  const int max_seg = (g.L + 7) / 8;
  for (int nseg = 1; nseg <= max_seg && static_cast<long long>(nseg) * sg.n_strips <= 4LL * slots; ++nseg) {
    const int rows = ((g.L + nseg - 1) / nseg + 3) / 4 * 4;
    const long long items = static_cast<long long>(sg.n_strips) * ((g.L + rows - 1) / rows);
    const long long waves = (items + slots - 1) / slots;
    // a wave with few warps per SM runs each warp faster, but not proportionally: model the per-step time as
    // 1 + 0.35 (w - 1) for w resident warps per SM (measured shape: issue-bound beyond ~4 warps per scheduler)
    const double per_sm = static_cast<double>(items) / waves / sm_count;
    const double w = per_sm < 1.0 ? 1.0 : per_sm;
    const double cost = static_cast<double>(waves) * (rows + overhead) * (1.0 + 0.35 * (w - 1.0));
    if (cost < best_cost) { best_cost = cost; best_seg = nseg; }
  }
  sg.seg_rows = ((g.L + best_seg - 1) / best_seg + 3) / 4 * 4;
  sg.n_seg = (g.L + sg.seg_rows - 1) / sg.seg_rows;
  sg.n_items = sg.n_strips * sg.n_seg;
  return sg;
}

template <int MODE, int PROG, int K, int MEASURE>
int strip_launch_one(StripPlan& plan, const CUtensorMap& map, const Geom& g, void* dst, const uint32_t* bits, double* acc,
                     double* part, unsigned long long* slots, const ChainConst<typename Traits<MODE>::real>& kc,
                     uint32_t first_sweep, cudaStream_t stream, int* nblocks_out, long long max_partials) {
  using V = typename Traits<MODE>::vec;
  constexpr int NS = StripProg<PROG, K>::NS, NW = StripCfg<MODE, NS>::NW;
  constexpr size_t smem = strip_smem_bytes<MODE, NS>();
  static bool attr_done = false;
  if (!attr_done) {
    if (cudaFuncSetAttribute(strip_kernel<MODE, PROG, K, MEASURE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(smem)) != cudaSuccess)
      return TILED_ATTR;
    attr_done = true;
  }
  const StripGeom sg = strip_geometry(g, NS, NW, plan.sm_count);
  const int nblocks = (sg.n_items + NW - 1) / NW;
  if (MEASURE != 0 && nblocks > max_partials) return TILED_TOO_MANY;
  strip_kernel<MODE, PROG, K, MEASURE><<<nblocks, NW * 32, smem, stream>>>(map, static_cast<V*>(dst), bits, acc, part, slots,
                                                                            g, kc, first_sweep, sg);
  if (cudaGetLastError() != cudaSuccess) return TILED_LAUNCH;
  *nblocks_out = nblocks;
  return TILED_OK;
}

// prog / k / measure -> instantiation.  Supported: R4 k = 1 (measure 0, 1, 2), R4 k = 2; FUSED k = 1 (measure 0, 1, 2),
// FUSED k = 2; QUENCH k = 2 (two double passes).  Returns TILED_LAUNCH for anything else.
template <int MODE>
int strip_launch(StripPlan& plan, TiledPlan& tp, const Geom& g, int src_index, void* src, void* dst, const uint32_t* bits,
                 double* acc, double* part, unsigned long long* slots, const ChainConst<typename Traits<MODE>::real>& kc,
                 uint32_t first_sweep, int prog, int k, int measure, cudaStream_t stream, int* nblocks_out,
                 long long max_partials) {
  if (!tp.encode) return TILED_NO_DRIVER;
  if (plan.sm_count == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&plan.sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || plan.sm_count <= 0)
      return TILED_ATTR;
  }
  constexpr int w = sizeof(typename Traits<MODE>::vec) == 16 ? 1 : 0;
  if (plan.map_src[src_index][w] != src) {
    const int es = strip_encode<MODE>(tp, g, src, &plan.map[src_index][w]);
    if (es != TILED_OK) return es;
    plan.map_src[src_index][w] = src;
  }
  const CUtensorMap& map = plan.map[src_index][w];
#define MPR_STRIP_CASE(PROG_, K_, M_)                                                                              \
  if (prog == PROG_ && k == K_ && measure == M_)                                                                   \
    return strip_launch_one<MODE, PROG_, K_, M_>(plan, map, g, dst, bits, acc, part, slots, kc, first_sweep, stream, \
                                                 nblocks_out, max_partials);
  MPR_STRIP_CASE(PROG_R4, 1, 0)
  MPR_STRIP_CASE(PROG_R4, 1, 1)
  MPR_STRIP_CASE(PROG_R4, 1, 2)
  MPR_STRIP_CASE(PROG_R4, 2, 0)
  MPR_STRIP_CASE(PROG_FUSED, 1, 0)
  MPR_STRIP_CASE(PROG_FUSED, 1, 1)
  MPR_STRIP_CASE(PROG_FUSED, 1, 2)
  MPR_STRIP_CASE(PROG_FUSED, 2, 0)
  MPR_STRIP_CASE(PROG_QUENCH, 2, 0)
#undef MPR_STRIP_CASE
  return TILED_LAUNCH;
}

// One non-template entry per precision mode, each defined in its own translation unit (mpr_strip_mode.cu compiled
// with -DMPR_STRIP_MODE=0..3) so that the instantiations build in parallel.
struct StripArgs {
  StripPlan* plan;
  TiledPlan* tp;
  Geom g;
  int src_index;
  void* src;
  void* dst;
  const uint32_t* bits;
  double* acc;
  double* part;
  unsigned long long* slots;
  const void* kc;            // ChainConst<real of the mode>
  uint32_t first_sweep;
  int prog, k, measure;
  cudaStream_t stream;
  int* nblocks_out;
  long long max_partials;
};
int strip_launch_mode0(const StripArgs& a);
int strip_launch_mode1(const StripArgs& a);
int strip_launch_mode2(const StripArgs& a);
int strip_launch_mode3(const StripArgs& a);

}  // namespace mpr
