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
#include <type_traits>
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
// Halo lanes of a MODE: the TMA unit wants every box row to start on a 16-byte boundary.  The first plane column of
// a strip is strip * (64 - 4 HL) - 2 HL; with 8 or 16 bytes per plane column (float / double storage) any HL does, with
// the 4 bytes of fp16 storage the column must be a multiple of 4, i.e. HL even: HP strips carry two halo lanes per side.
template <int MODE> __host__ __device__ constexpr int strip_mode_halo_lanes(int ns) {
  return (sizeof(decltype(Traits<MODE>::vec::x)) == 2 && strip_halo_lanes(ns) < 2) ? 2 : strip_halo_lanes(ns);
}
__host__ __device__ constexpr int strip_slots(int ns) { return (2 * ns + 1 + kStripRB - 1) / kStripRB + 1; }
__host__ __device__ constexpr int strip_lead_rows(int ns) { return (ns + kStripRB - 1) / kStripRB * kStripRB; }   // rows loaded above a segment

// warps per CTA (one CTA per SM): as many as their rings fit into 216 KiB of shared memory, at most 12 -- 168
// registers per thread, which the four interleaved update chains of a 4-stage program need -- or 16 for the
// 2-stage programs, whose two chains fit the 128 registers that leaves (measured at L = 16384, SP_INTRINSIC,
// site-fused schedule, one sweep per launch: 12 warps 1.07 ms, 16 warps 0.78 ms per sweep; a 4-stage program
// squeezed into 128 registers for 13 warps: 1.11 against 0.98 ms).  The ring of a warp is 16.5 KiB with float
// storage and NS = 4, 33 KiB in DP.
// Launches that accumulate phi (MEASURE == 2) add 2 KiB of accumulator staging per warp (kAccStageBytes) and may
// fill the 227 KiB of a CTA to the last KiB: 12 warps for NS = 4, 15 for NS = 2 with float storage.
constexpr int kAccStageBytes = 2 * 2 * 32 * 16;
template <int MODE, int NS, int MEASURE = 0> struct StripCfg {
  static constexpr int kRingBytes = strip_slots(NS) * (2 * kStripRB * 2 * kTileCols * static_cast<int>(sizeof(decltype(Traits<MODE>::vec::x))) + 128 + 8) +
                                    (MEASURE == 2 ? kAccStageBytes : 0);
  static constexpr int kFit = (MEASURE == 2 ? 232448 - 256 - 128 : 216 * 1024) / kRingBytes;
  static constexpr int kMax = (NS <= 2 && sizeof(typename Traits<MODE>::real) == 4) ? 16 : 12;
  static constexpr int NW = kFit < kMax ? kFit : kMax;
};

// Work distribution.  The rows of all strips are laid end to end (strip s occupies [s Lp, (s + 1) Lp), Lp = the number of rows rounded
// up to a multiple of 4) and cut into equal quotas of `quota` rows (a multiple of 4): warp w of the launch takes
// [w quota, (w + 1) quota).  A quota that crosses the end of a strip is worked off as two segments.  Warp w is warp
// slot w / gridDim.x of CTA w % gridDim.x, so that a launch with fewer warps than slots still uses every SM.
struct StripGeom {
  int n_strips, Lp, quota, n_warps;
  int n_mchunks;      // chunks per strip in the strip-ordered mask (strip_mask_chunks)
};

// Strip-ordered mask: for every strip and every chunk of 4 rows one 128-byte block, one 32-bit word per lane:
// bit 4 r + 2 c + k = site (row 4 chunk + r, colour c, plane column j0 + 2 lane + k) exists and is a prediction site.
// It travels into shared memory with the spins of the chunk (one 1-D bulk copy on the same mbarrier), so a lane gets
// the mask bits of 4 rows x 2 colours with one LDS and tests them with immediate bit masks.  Chunk index 0 is the
// chunk of rows -kStripMaskLead .. -kStripMaskLead + 3; rows outside the grid have no bits set.
constexpr int kStripMaskLead = 8;      // rows (two chunks) above the grid
constexpr int kStripMaskTail = 32;     // rows below it
__host__ __device__ constexpr int strip_mask_chunks(int L) { return ((L + 3) / 4 * 4 + kStripMaskLead + kStripMaskTail) / kStripRB; }

// Measuring launches that accumulate phi (MEASURE == 2) stage the accumulator words of the NEXT step through shared
// memory (cp.async, two buffers of 2 rows x 32 lanes x 16 bytes per warp): a whole step hides the DRAM latency
// without holding registers.
template <int MODE, int NS, int MEASURE = 0> constexpr size_t strip_smem_bytes() {
  using S = decltype(Traits<MODE>::vec::x);
  return static_cast<size_t>(StripCfg<MODE, NS, MEASURE>::NW) *
             (strip_slots(NS) * (2 * kStripRB * kRowScalars * sizeof(S) + 128 + sizeof(uint64_t)) + (MEASURE == 2 ? kAccStageBytes : 0)) + 128;
}

__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// Arming a slot's mbarrier publishes nothing (the data arrives through complete_tx and the waiter acquires): the
// default .release of mbarrier.arrive costs a MEMBAR.ALL.CTA that waits for the warp's global stores.
__device__ __forceinline__ void mbar_expect_tx_relaxed(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.relaxed.cta.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// One lane of the (converged) warp; unlike `lane == 0` the compiler knows the branch is taken by one thread of a
// uniform warp and issues the TMA instructions from uniform registers without a broadcast loop.
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n.reg .pred p;\nelect.sync _|p, 0xffffffff;\nselp.u32 %0, 1, 0, p;\n}\n" : "=r"(pred));
  return pred != 0u;
}
// 16-byte asynchronous copy global -> shared (SASS LDGSTS), skipped when `pred` is false; groups are per thread
__device__ __forceinline__ void cp_async_16(void* dst_smem, const void* src, bool pred) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %2, 0;\n@p cp.async.cg.shared.global [%0], [%1], 16;\n}\n"
               ::"r"(smem_u32(dst_smem)), "l"(src), "r"(static_cast<int>(pred)) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
// 1-D bulk copy global -> shared, completion counted on an mbarrier (SASS UBLKCP)
__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// MEASURE: 0 = none; 1 = + energy sample after the last stage; 2 = + accumulation of phi (R15)
template <int MODE, int PROG, int K, int MEASURE>
__global__ void __launch_bounds__(StripCfg<MODE, StripProg<PROG, K>::NS, MEASURE>::NW * 32, 1)
strip_kernel(const __grid_constant__ CUtensorMap tmap, typename Traits<MODE>::vec* __restrict__ dst,
             const uint32_t* __restrict__ smask, double* __restrict__ acc, double* __restrict__ part,
             unsigned long long* __restrict__ accept_slots, Geom g, ChainConst<typename Traits<MODE>::real> kc,
             uint32_t first_sweep, StripGeom sg) {
  using R = typename Traits<MODE>::real;
  using V = typename Traits<MODE>::vec;
  using S = decltype(V::x);
  using P = StripProg<PROG, K>;
  constexpr int NS = P::NS, NW = StripCfg<MODE, NS, MEASURE>::NW, RB = kStripRB, LAG = kStripLag;
  constexpr int NSLOT = strip_slots(NS), HL = strip_mode_halo_lanes<MODE>(NS), IC = kTileCols - 4 * HL;
  constexpr int LEAD = strip_lead_rows(NS);
  constexpr int CHUNK = 2 * RB * kRowScalars;          // scalars per chunk: [plane][row][128]
  constexpr int PLANE = RB * kRowScalars;
  constexpr uint32_t kSpinBytes = CHUNK * sizeof(S), kMaskBytes = 128, kChunkBytes = kSpinBytes + kMaskBytes;
  constexpr int NQ = (LAG * (NS - 1) + RB - 1) / RB + 1;     // mask words a lane holds: chunks i, i - 1, ..., i - NQ + 1
  static_assert(MEASURE == 0 || K == 1, "measuring launches carry one sweep");
  static_assert(LEAD <= kStripMaskLead, "the strip-ordered mask starts kStripMaskLead rows above the grid");

  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ double red[32];
  const int lane = threadIdx.x & 31;
  // the shuffle tells the compiler that the warp index is warp-uniform: everything derived from it (quota, strip,
  // row range, loop bounds) then lives in uniform registers and the loops are known not to diverge
  const int warp = __shfl_sync(0xffffffffu, static_cast<int>(threadIdx.x >> 5), 0);
  S* const ring = reinterpret_cast<S*>(smem_raw) + static_cast<size_t>(warp) * NSLOT * CHUNK;
  unsigned char* const after_rings = smem_raw + static_cast<size_t>(NW) * NSLOT * CHUNK * sizeof(S);
  uint32_t* const mring = reinterpret_cast<uint32_t*>(after_rings) + warp * NSLOT * 32;          // 128 B of mask per slot
  uint64_t* const bars = reinterpret_cast<uint64_t*>(after_rings + static_cast<size_t>(NW) * NSLOT * kMaskBytes) + warp * NSLOT;
  // accumulator staging (MEASURE == 2): [buffer = step parity][final stage 0 / 1][lane] double2
  double2* const astage = reinterpret_cast<double2*>(after_rings + ((static_cast<size_t>(NW) * NSLOT * (kMaskBytes + sizeof(uint64_t)) + 15) & ~size_t(15))) +
                          warp * (kAccStageBytes / 16) + lane;
  (void)astage;

  int n_acc = 0;
  // per-thread energy sum: X_E = D in `esum`, X_E = S (every partial sum a float) in `esum_f` -- the same values as
  // energy_add gives, without its per-term conversions both ways
  double esum = 0.0;
  float esum_f = 0.0f;
  auto energy_term = [&](double term) {
    if (g.energy_single) esum_f = esum_f + static_cast<float>(term); else esum = esum + term;
  };
  const int wg = warp * static_cast<int>(gridDim.x) + static_cast<int>(blockIdx.x);
  if (wg < sg.n_warps) {
    if (lane == 0) {
#pragma unroll
      for (int k = 0; k < NSLOT; ++k) mbar_init(bars + k, 1);
    }
    __syncwarp();
    uint32_t phase_bits = 0;                                  // bit s = parity the next wait on slot s expects
    const long long total = static_cast<long long>(sg.n_strips) * sg.Lp;
    long long q0 = static_cast<long long>(wg) * sg.quota;
    const long long q1 = min(total, q0 + sg.quota);
    const uint32_t Lu = static_cast<uint32_t>(g.L);
    const long long grow = 2 * static_cast<long long>(g.Wp), gplane = 2 * static_cast<long long>(g.plane);

#pragma unroll 1
    while (q0 < q1) {
      // ---- one segment: rows [yb, ye) of one strip
      const int strip = static_cast<int>(q0 / sg.Lp);
      const int yb = static_cast<int>(q0 - static_cast<long long>(strip) * sg.Lp);     // multiple of 4
      const int ye_pad = static_cast<int>(min(static_cast<long long>(sg.Lp), yb + (q1 - q0)));
      q0 += ye_pad - yb;
      const int ye = min(g.H, ye_pad);
      if (yb >= ye) continue;
      const int j0 = strip * IC - 2 * HL;                     // plane column of lane 0 (even)
      const int t0 = yb - LEAD;                               // first loaded row (a multiple of 4, so even)
      const int n_steps = ye - t0 + LAG * (NS - 1);           // the last stage finishes row ye - 1 in the last step
      const int n_iter = (n_steps + RB - 1) / RB;
      // iterations in which every stage works on an owned, loaded row in all four steps: no predicates needed
      // [cnt_b, cnt_e): the rows of the segment that enter the accepted-move count and the energy sum -- all of them,
      // unless the context is a slab of a larger grid (Geom::own0 / own1: its halo rows are updated and stored, not counted)
      const int cnt_b = max(yb, g.own0), cnt_e = min(ye, g.own1);
      // peer mode (Geom::peer_rows > 0): the own rows next to an inner edge are also stored into the neighbour slab; they
      // are left to the predicated iterations too.  [st_b, st_e): the rows this launch stores into its own buffer.
      const int fast_b = cnt_b + (g.peer_dst[0] ? g.peer_rows : 0), fast_e = cnt_e - (g.peer_dst[1] ? g.peer_rows : 0);
      const int st_b = g.peer_rows ? cnt_b : yb, st_e = g.peer_rows ? cnt_e : ye;
      const int i_lo = (fast_b - t0 + LAG * (NS - 1) + RB - 1) / RB;    // = (LEAD + LAG (NS - 1) + RB - 1) / RB when fast_b = yb
      const int i_hi = (max(fast_e, t0) - t0) / RB;                     // RB i + RB - 1 < fast_e - t0
      const int j = j0 + 2 * lane;
      const bool lane_ok = lane >= HL && lane < 32 - HL && j < g.Wp;
      int seg_acc = 0;

      __syncwarp();
      // this strip's mask blocks; block of the chunk whose first row is t0 + 4 c: index (t0 + lead) / 4 + c
      const uint32_t* const mblk = smask + (static_cast<size_t>(strip) * sg.n_mchunks + (t0 + kStripMaskLead) / RB) * 32;
      if (elect_one()) {                                      // chunk 0 -> slot 0
        fence_proxy_async_smem();
        mbar_expect_tx_relaxed(bars, kChunkBytes);
        tma_load_3d(ring, &tmap, bars, (sizeof(S) == 2 ? 1 : 2) * j0, t0, 0);
        bulk_load_1d(mring, mblk, kMaskBytes, bars);
      }
      // cb[k] = scalar offset (inside this warp's ring) of the chunk  i + 2 - NSLOT + k,  i.e. cb[NSLOT-1] holds
      // chunk i + 1 (in flight), cb[NSLOT-2] chunk i, cb[0] the oldest live one.  Chunk c lives in slot c % NSLOT.
      int cb[NSLOT];
#pragma unroll
      for (int k = 0; k < NSLOT; ++k) cb[k] = ((k + 2) % NSLOT) * CHUNK;    // iteration 0: chunk k + 2 - NSLOT
      int slot_next = 1 % NSLOT;                              // slot of chunk i + 1

      // mask words of the chunks i, i - 1, ... (cw[0] = chunk i); chunks above t0 were never loaded: no bits
      uint32_t cw[NQ];
#pragma unroll
      for (int k = 0; k < NQ; ++k) cw[k] = 0u;

      uint32_t site_t = g.site0 + static_cast<uint32_t>(t0) * Lu + static_cast<uint32_t>(2 * j);   // Philox word 0 of row t, no parity
      // global pointers of this lane's unit in row t of plane 0 (dst / accumulator); never dereferenced outside the grid
      const long long g_t0 = static_cast<long long>(t0) * g.Wp + j;
      S* gp = reinterpret_cast<S*>(dst) + 2 * g_t0;
      double* ap = acc + g_t0;

      mbar_wait(bars, phase_bits & 1u);
      phase_bits ^= 1u;

      // ---- one iteration = RB steps = the rows of one chunk entering the pipeline
      auto iteration = [&](int i, auto edge_tag) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        // prefetch chunk i + 1 into the slot whose old chunk (i + 1 - NSLOT) nobody reads any more
        __syncwarp();
        if (elect_one()) {
          fence_proxy_async_smem();
          mbar_expect_tx_relaxed(bars + slot_next, kChunkBytes);
          tma_load_3d(ring + cb[NSLOT - 1], &tmap, bars + slot_next, (sizeof(S) == 2 ? 1 : 2) * j0, t0 + RB * (i + 1), 0);
          bulk_load_1d(mring + slot_next * 32, mblk + static_cast<size_t>(i + 1) * 32, kMaskBytes, bars + slot_next);
        }
        // the mask word of chunk i (its slot is the one before slot_next; the chunk was awaited in iteration i - 1)
#pragma unroll
        for (int k = NQ - 1; k > 0; --k) cw[k] = cw[k - 1];
        cw[0] = mring[(slot_next == 0 ? NSLOT - 1 : slot_next - 1) * 32 + lane];
        uint32_t stash[NS][2];                                // second half of the Philox blocks (float modes)
        (void)stash;
#pragma unroll
        for (int u = 0; u < RB; ++u) {
          if (u == RB - 1) {                                  // row 4 i + 4 (first of chunk i + 1) is read from here on
            mbar_wait(bars + slot_next, (phase_bits >> slot_next) & 1u);
            phase_bits ^= 1u << slot_next;
          }
          const int n = RB * i + u;                           // step number; row t = t0 + n
          const int t = t0 + n;
          // ---- gather: own unit and local fields of every stage (all reads before any write of this step)
          Two<R> A[NS], B[NS], c[NS], s[NS];
          S* own[NS];
          Unit<S> nb_m, nb_u, nb_d;                           // float-mode energy: the last stage's neighbours
          S exc_last = S(0), exs_last = S(0);
#pragma unroll
          for (int p = 0; p < NS; ++p) {
            const int col = p & 1, par = (u + col) & 1;       // t0 and LAG are even: x-parity of row t - 2p is (u + col) & 1
            const int rel = u - LAG * p;                      // row relative to 4 i
            auto at = [&](int plane, int r) -> S* {
              const int q = (r >= 0) ? r / RB : -((-r + RB - 1) / RB);      // floor(r / RB)
              return ring + cb[NSLOT - 2 + q] + plane * PLANE + (r - q * RB) * kRowScalars + 4 * lane;
            };
            own[p] = at(col, rel);
            const Unit<S> up = *reinterpret_cast<const Unit<S>*>(at(1 - col, rel - 1));
            const Unit<S> mid = *reinterpret_cast<const Unit<S>*>(at(1 - col, rel));
            const Unit<S> dn = *reinterpret_cast<const Unit<S>*>(at(1 - col, rel + 1));
            const Unit<S> me = *reinterpret_cast<const Unit<S>*>(own[p]);
            const S exc = par ? lane_dn(mid.ca) : lane_up(mid.cb);
            const S exs = par ? lane_dn(mid.sa) : lane_up(mid.sb);
            combine_fields<MODE>(par, up, mid, dn, exc, exs, &A[p], &B[p]);
            c[p] = mk2(R(me.ca), R(me.cb));
            s[p] = mk2(R(me.sa), R(me.sb));
            if (MEASURE != 0 && sizeof(R) == 4 && p == NS - 1) {
              nb_u = up; nb_m = mid; nb_d = dn; exc_last = exc; exs_last = exs;
            }
          }

          // measuring launches: the accumulator words of the two rows that become final in the NEXT step are requested
          // now (cp.async into the other staging buffer); this step's words were requested one step ago
          if constexpr (MEASURE == 2) {
#pragma unroll
            for (int p = NS - 2; p < NS; ++p) {
              const int col = p & 1, row_next = t + 1 - LAG * p;
              cp_async_16(astage + (((u + 1) & 1) * 2 + (p - (NS - 2))) * 32,
                          ap + static_cast<long long>(1 - LAG * p) * g.Wp + static_cast<long long>(col) * static_cast<long long>(g.plane),
                          lane_ok && row_next >= yb && row_next < ye);
            }
            cp_async_commit();
          }

          // ---- compute
          R o[NS][4];
#pragma unroll
          for (int p = 0; p < NS; ++p) {
            const int col = p & 1, par = (u + col) & 1;
            // mask bits of row 4 i + u - 2 p: chunk i + mq (mq <= 0), row mr of it
            const int rel = u - LAG * p;
            const int mqk = (rel >= 0) ? 0 : (-rel + RB - 1) / RB;          // chunks back
            const int mr = rel + mqk * RB;
            const bool fa = (cw[mqk] & (1u << (4 * mr + 2 * col))) != 0u, fb = (cw[mqk] & (2u << (4 * mr + 2 * col))) != 0u;
            const int kind = P::kind(p);
            if (kind == KIND_MET || kind == KIND_MO) {
              const uint32_t pair_site = site_t - static_cast<uint32_t>(LAG * p) * Lu + static_cast<uint32_t>(par);
              MetWords w0, w1;
              const uint32_t sweep = first_sweep + static_cast<uint32_t>(P::sweep_off(p));
              if constexpr (sizeof(R) == 8) {
                met_words_pair<MODE>(pair_site, sweep, Lu, par, (u & 1) != 0, kc, &w0, &w1);
              } else {
                // float modes: one Philox block per quad (R9) -- computed in the even row (t0 is even, so that is an
                // even step), its second half kept for the odd row that follows in the next step
                if ((u & 1) == 0) {
                  const uint4 r = met_words_quad<MODE>(pair_site, sweep, kc);
                  w0 = MetWords{r.x, 0u, r.x, 0u};
                  w1 = MetWords{r.y, 0u, r.y, 0u};
                  stash[p][0] = r.z; stash[p][1] = r.w;
                } else {
                  w0 = MetWords{stash[p][0], 0u, stash[p][0], 0u};
                  w1 = MetWords{stash[p][1], 0u, stash[p][1], 0u};
                }
              }
              bool ok[2];
              met_update2<MODE>(c[p], s[p], A[p], B[p], w0, w1, fa, fb, kc, o[p], ok);
              // accepted moves are counted per lane; the lanes that do not own their columns are dropped at the end
              const int row = t - LAG * p;
              if (!EDGE || (row >= cnt_b && row < cnt_e)) seg_acc += static_cast<int>(ok[0]) + static_cast<int>(ok[1]);
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
            // rows above t0 do not exist; nobody reads the ring copy of the last stage's row (it is final: global only)
            if (p < NS - 1 && (!EDGE || n >= LAG * p)) *reinterpret_cast<Unit<S>*>(own[p]) = out;
            if (p >= NS - 2) {                                                            // last stage of this colour
              const bool owned = lane_ok && (!EDGE || (row >= st_b && row < st_e));
              if (owned) {
                *reinterpret_cast<Unit<S>*>(gp - (LAG * p) * grow + col * gplane) = out;
                if (EDGE && g.peer_rows) {       // peer mode: the rows next to an inner edge go to the neighbour's halo as well
#pragma unroll
                  for (int d = 0; d < 2; ++d) {
                    const bool send = d == 0 ? row < g.own0 + g.peer_rows : row >= g.own1 - g.peer_rows;
                    if (send && g.peer_dst[d])
                      *reinterpret_cast<Unit<S>*>(reinterpret_cast<S*>(g.peer_dst[d]) +
                          2 * (static_cast<long long>(row + g.peer_row_off[d]) * g.Wp + j + col * g.peer_plane[d])) = out;
                  }
                }
                if (MEASURE == 2) {
                  const int rel = u - LAG * p;
                  const int mqk = (rel >= 0) ? 0 : (-rel + RB - 1) / RB;
                  const uint32_t mm = (cw[mqk] >> (4 * (rel + mqk * RB) + 2 * col)) & 3u;
                  if (mm) {
                    double* a = ap - static_cast<long long>(LAG * p) * g.Wp + static_cast<long long>(col) * static_cast<long long>(g.plane);
                    cp_async_wait<1>();                       // everything but the group of the next step has landed
                    double2 a2 = astage[((u & 1) * 2 + (p - (NS - 2))) * 32];
                    // from the spins AS STORED (SP: rounded to float), like the other paths
                    if (mm & 1u) a2.x += spin_angle<MODE>(R(out.ca), R(out.sa));
                    if (mm & 2u) a2.y += spin_angle<MODE>(R(out.cb), R(out.sb));
                    *reinterpret_cast<double2*>(a) = a2;
                  }
                }
                if (MEASURE != 0 && p == NS - 1 && (!EDGE || (row >= cnt_b && row < cnt_e))) {
                  // every bond has exactly one colour-1 end: H = -J sum over colour-1 sites of site_energy_term
                  // with the final spins; the neighbours (colour 0) were final when this stage gathered them
                  if constexpr (sizeof(R) == 8) {
                    R Aa, Ab, Ba, Bb;
                    un2(A[p], &Aa, &Ab); un2(B[p], &Ba, &Bb);
                    energy_term(static_cast<double>(fma_(R(out.ca), Aa, R(out.sa) * Ba)));
                    energy_term(static_cast<double>(fma_(R(out.cb), Ab, R(out.sb) * Bb)));
                  } else {
                    const int par = (u + col) & 1;
                    const R alc = par ? R(nb_m.ca) : R(exc_last), als = par ? R(nb_m.sa) : R(exs_last);
                    const R arc = par ? R(nb_m.cb) : R(nb_m.ca), ars = par ? R(nb_m.sb) : R(nb_m.sa);
                    const R blc = par ? R(nb_m.cb) : R(nb_m.ca), bls = par ? R(nb_m.sb) : R(nb_m.sa);
                    const R brc = par ? R(exc_last) : R(nb_m.cb), brs = par ? R(exs_last) : R(nb_m.sb);
                    energy_term(site_energy_term<R>(R(out.ca), R(out.sa), alc, als, arc, ars, R(nb_u.ca), R(nb_u.sa),
                                                         R(nb_d.ca), R(nb_d.sa)));
                    energy_term(site_energy_term<R>(R(out.cb), R(out.sb), blc, bls, brc, brs, R(nb_u.cb), R(nb_u.sb),
                                                         R(nb_d.cb), R(nb_d.sb)));
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
      };

      int i = 0;
#pragma unroll 1
      for (; i < n_iter && i < i_lo; ++i) iteration(i, std::true_type{});
#pragma unroll 1
      for (; i < n_iter && i < i_hi; ++i) iteration(i, std::false_type{});
#pragma unroll 1
      for (; i < n_iter; ++i) iteration(i, std::true_type{});
      // every chunk issued was awaited inside its iteration: nothing is in flight here
      if (lane_ok) n_acc += seg_acc;
    }
  }
  if constexpr (MEASURE != 0) {
    const double e = block_sum(g.energy_single ? static_cast<double>(esum_f) : esum, red, g.energy_single);
    if (threadIdx.x == 0) part[blockIdx.x] = e;
  }
  if constexpr (PROG != PROG_QUENCH) {
    const double a = block_sum(static_cast<double>(n_acc), red);
    if (threadIdx.x == 0 && a > 0.0)
      atomicAdd(accept_slots + (blockIdx.x & 1023u), static_cast<unsigned long long>(a));
  }
}

// Strip-ordered mask for strips with `hl` halo lanes per side (see strip_mask_chunks): one thread per word.
static __global__ void pack_strip_mask_kernel(const uint8_t* __restrict__ mask, Geom g, int hl, int n_strips, int n_mchunks,
                                              uint32_t* __restrict__ out) {
  const long long w = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x;
  const long long nwords = static_cast<long long>(n_strips) * n_mchunks * 32;
  if (w >= nwords) return;
  const int lane = static_cast<int>(w & 31);
  const int chunk = static_cast<int>((w >> 5) % n_mchunks), strip = static_cast<int>((w >> 5) / n_mchunks);
  const int ic = kTileCols - 4 * hl;
  const int j = strip * ic - 2 * hl + 2 * lane;
  uint32_t word = 0;
  for (int r = 0; r < kStripRB; ++r) {
    const int y = chunk * kStripRB - kStripMaskLead + r;
    if (y < 0 || y >= g.H) continue;
    for (int c = 0; c < 2; ++c)
      for (int k = 0; k < 2; ++k) {
        const int jj = j + k;
        const int x = 2 * jj + x_parity(y, c);
        if (jj >= 0 && x < g.L && mask[static_cast<size_t>(y) * g.L + x]) word |= 1u << (4 * r + 2 * c + k);
      }
  }
  out[w] = word;
}
inline int strip_mask_strips(const Geom& g, int hl) { const int ic = kTileCols - 4 * hl; return (g.Wp + ic - 1) / ic; }
inline size_t strip_mask_words(const Geom& g, int hl) {
  return static_cast<size_t>(strip_mask_strips(g, hl)) * strip_mask_chunks(g.H) * 32;
}
inline cudaError_t strip_mask_build(const uint8_t* d_mask, const Geom& g, int hl, uint32_t* out, cudaStream_t stream) {
  const size_t n = strip_mask_words(g, hl);
  pack_strip_mask_kernel<<<static_cast<unsigned>((n + 255) / 256), 256, 0, stream>>>(d_mask, g, hl, strip_mask_strips(g, hl),
                                                                                     strip_mask_chunks(g.H), out);
  return cudaGetLastError();
}

// ---- host side -------------------------------------------------------------------------------
struct StripPlan {
  int sm_count = 0;
  // tensor maps are encoded once per (state buffer, element width): the two buffers ping-pong
  CUtensorMap map[2][3];
  void* map_src[2][3] = {{nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr}};
};

template <int MODE>
int strip_encode(TiledPlan& tp, const Geom& g, void* src, CUtensorMap* map) {
  using V = typename Traits<MODE>::vec;
  // fp16 storage travels as 32-bit words (two halves each): the copy is the same bytes, and the plain FLOAT32 path
  // of the TMA unit is the one every other mode has proven
  constexpr bool kHalf = sizeof(decltype(V::x)) == 2;
  const cuuint64_t dims[3] = {static_cast<cuuint64_t>(kHalf ? 1 : 2) * g.Wp, static_cast<cuuint64_t>(g.H), 2};
  const cuuint64_t strides[2] = {static_cast<cuuint64_t>(g.Wp) * sizeof(V), static_cast<cuuint64_t>(g.plane) * sizeof(V)};
  const cuuint32_t box[3] = {(kHalf ? 1 : 2) * kTileCols, static_cast<cuuint32_t>(kStripRB), 2};
  const cuuint32_t estr[3] = {1, 1, 1};
  // 64-byte promotion: a strip row (512 B at a 480-byte pitch) then drags in the least data it does not use
  // (128 B: 0.983 ms, 64 B: 0.970 ms, none: 0.983 ms per sweep at L = 16384)
  const CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_L2_64B;
  const CUresult r = tp.encode(map, kHalf ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : static_cast<CUtensorMapDataType>(TmaType<decltype(V::x)>::value), 3, src,
                               dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                               promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? TILED_OK : TILED_ENCODE;
}

// Rows per warp.  Preferred: every strip cut at the SAME rows into n_seg = floor(slots / n_strips) segments (the
// warps of neighbouring strips then work on the same rows at the same time and the columns they share are read
// from DRAM once and from L2 the second time) -- taken when that keeps at least 96 % of the warp slots busy.
// Otherwise the rows of all strips are laid end to end and cut into equal quotas, whatever the strip boundaries.
// Fewer warps than slots when a warp would get fewer than 8 rows (a warp pays LEAD + 2 (NS - 1) + 3 warm-up / drain
// steps per segment whatever its quota).
inline StripGeom strip_geometry(const Geom& g, int ns, int hl, int nw, int sm_count, int* nblocks) {
  StripGeom sg;
  (void)ns;
  const int ic = kTileCols - 4 * hl;
  sg.n_strips = (g.Wp + ic - 1) / ic;
  const int L4 = (g.H + 3) / 4 * 4;
  const long long slots = static_cast<long long>(sm_count) * nw;
  const long long n_seg = slots / sg.n_strips;
  const int seg_rows = n_seg > 0 ? static_cast<int>(((g.H + n_seg - 1) / n_seg + 3) / 4 * 4) : 0;
  if (n_seg > 0 && sg.n_strips * n_seg * 100 >= slots * 96 && seg_rows >= 8) {
    const int segs = (g.H + seg_rows - 1) / seg_rows;
    sg.Lp = segs * seg_rows;
    sg.quota = seg_rows;
    sg.n_warps = sg.n_strips * segs;
  } else {
    sg.Lp = L4;
    const long long total = static_cast<long long>(sg.n_strips) * sg.Lp;
    long long warps = total / 8 < slots ? total / 8 : slots;
    if (warps < 1) warps = 1;
    long long quota = (total + warps - 1) / warps;
    quota = (quota + 3) / 4 * 4;
    sg.quota = static_cast<int>(quota);
    sg.n_warps = static_cast<int>((total + quota - 1) / quota);
  }
  sg.n_mchunks = strip_mask_chunks(g.H);
  *nblocks = sg.n_warps < sm_count ? sg.n_warps : sm_count;
  return sg;
}

template <int MODE, int PROG, int K, int MEASURE>
int strip_launch_one(StripPlan& plan, const CUtensorMap& map, const Geom& g, void* dst, const uint32_t* const smask[2], double* acc,
                     double* part, unsigned long long* slots, const ChainConst<typename Traits<MODE>::real>& kc,
                     uint32_t first_sweep, cudaStream_t stream, int* nblocks_out, long long max_partials) {
  using V = typename Traits<MODE>::vec;
  constexpr int NS = StripProg<PROG, K>::NS, NW = StripCfg<MODE, NS, MEASURE>::NW;
  constexpr size_t smem = strip_smem_bytes<MODE, NS, MEASURE>();
  static_assert(smem <= 232448 - 256, "dynamic + static shared memory of one CTA");
  static bool attr_done = false;
  if (!attr_done) {
    if (cudaFuncSetAttribute(strip_kernel<MODE, PROG, K, MEASURE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(smem)) != cudaSuccess)
      return TILED_ATTR;
    attr_done = true;
  }
  int nblocks = 0;
  constexpr int HL = strip_mode_halo_lanes<MODE>(NS);
  const StripGeom sg = strip_geometry(g, NS, HL, NW, plan.sm_count, &nblocks);
  if (MEASURE != 0 && nblocks > max_partials) return TILED_TOO_MANY;
  strip_kernel<MODE, PROG, K, MEASURE><<<nblocks, NW * 32, smem, stream>>>(map, static_cast<V*>(dst), smask[HL - 1], acc, part, slots,
                                                                            g, kc, first_sweep, sg);
  if (const cudaError_t le = cudaGetLastError(); le != cudaSuccess) { tiled_last_cuda_error() = le; return TILED_LAUNCH; }
  *nblocks_out = nblocks;
  return TILED_OK;
}

// prog / k / measure -> instantiation.  Supported: R4 k = 1 (measure 0, 1, 2), R4 k = 2; FUSED k = 1 (measure 0, 1, 2),
// FUSED k = 2; QUENCH k = 2 (two double passes).  Returns TILED_LAUNCH for anything else.
template <int MODE>
int strip_launch(StripPlan& plan, TiledPlan& tp, const Geom& g, int src_index, void* src, void* dst, const uint32_t* const smask[2],
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
  constexpr int w = sizeof(typename Traits<MODE>::vec) == 16 ? 1 : sizeof(typename Traits<MODE>::vec) == 8 ? 0 : 2;
  if (plan.map_src[src_index][w] != src) {
    const int es = strip_encode<MODE>(tp, g, src, &plan.map[src_index][w]);
    if (es != TILED_OK) return es;
    plan.map_src[src_index][w] = src;
  }
  const CUtensorMap& map = plan.map[src_index][w];
#define MPR_STRIP_CASE(PROG_, K_, M_)                                                                              \
  if (prog == PROG_ && k == K_ && measure == M_) {                                                                 \
    return strip_launch_one<MODE, PROG_, K_, M_>(plan, map, g, dst, smask, acc, part, slots, kc, first_sweep,     \
                                                   stream, nblocks_out, max_partials);                             \
  }
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
  const uint32_t* smask[2];   // strip-ordered masks for 1 and 2 halo lanes per side (NS <= 4, NS = 8)
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
int strip_launch_mode4(const StripArgs& a);
int strip_launch_mode5(const StripArgs& a);

}  // namespace mpr
