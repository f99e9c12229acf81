// mpr_plain.cuh -- kernels that work directly on the global colour planes: set-up (R1 map,
// mask bitmaps, sample energy), chain initialisation (R8), one-launch-per-colour-pass updates
// (the PLAIN path, also the quench passes of R8), energy (R3), accumulation and back-map (R15).
//
// Layout.  Site (x, y) has colour (x + y) & 1 and lives in colour plane `col`
// at row y, column j = x >> 1; a plane is H rows of Wp columns (Wp = ceil(L/2) rounded up to 16; L columns, H rows,
// H = L on the paper's square grid),
// one spin (c, s) per site, stored PAIR-INTERLEAVED: the two sites of plane columns (2m, 2m + 1)
// share one unit of four scalars (c_2m, c_2m+1, s_2m, s_2m+1), so that the tiled kernel reads a pair
// with one 128-bit access whose register halves are already (site a, site b) lanes for the packed
// f32x2 arithmetic.  With idx = row offset + j (always of j's parity), c sits at scalar
// 2 idx - (j & 1) and s two scalars further (ld_spin / st_spin).  mask bit j of row y of plane col is 1 iff the site exists and is a
// prediction site; Wm 32-bit words per row.
#pragma once
#include "mpr_device.cuh"

namespace mpr {

struct Geom {
  int L, Wp, Wm;         // L = columns of the grid (x); rows: H below
  int Wb, Hb;            // padded bitmap: words per row, rows per colour
  size_t plane;          // elements per colour plane = H * Wp
  int H;                 // rows of the grid (y); == L unless created by mpr_create_rect
  // Slab of a larger grid (mpr_set_slab): the context holds rows [row0, row0 + H) of it.  The random
  // numbers are keyed on the GLOBAL site index (site0 = row0 * L is added to every local one), and only rows
  // [own0, own1) -- the rows this slab owns, the rest being halo -- enter the energy sums and the accepted-move count.
  uint32_t site0;        // 0 for a whole grid
  int own0, own1;        // [0, H) for a whole grid
  // Peer mode of a slab (mpr_set_peers; STRIP kernels only): a launch stores its OWN rows only, and the `peer_rows`
  // own rows next to each inner edge ALSO straight into the halo rows of the neighbour slab's destination buffer --
  // peer memory; on one GPU just another pointer, between GPUs a store over NVLink -- so that no copy launch follows.
  // peer_dst[d] (d = 0: the slab above, 1: below; null = none) is the neighbour's destination state buffer of this
  // launch, peer_plane[d] its plane size in units, peer_row_off[d] = (neighbour's local row) - (this slab's local row).
  int peer_rows;         // 0: not in peer mode
  void* peer_dst[2];
  long long peer_plane[2];
  int peer_row_off[2];
  double q;              // PAPER.md:27, q in (0, 1/2]; 1/2 unless mpr_set_q
  int energy_single;     // X_E of PAPER.md:35: 0 = energy sums in double (R13), 1 = the energy variable is a float
};

// The mask bitmaps are padded with zero words (kBitPadTop rows above, kBitPadBot below, kBitPadLeft
// words to the left, kBitPadRight to the right of every row), so that the tiled kernel can read
// the words of a whole staged region -- halo and out-of-grid part included -- without a bounds
// test.  `bits` always points at word 0 of row 0 of colour 0 INSIDE the padded array.
constexpr int kBitPadTop = 16, kBitPadBot = 96, kBitPadLeft = 1, kBitPadRight = 3;

__device__ __forceinline__ const uint32_t* mask_word(const uint32_t* __restrict__ bits, const Geom& g, int col, int y,
                                                     int wi) {
  return bits + (static_cast<long long>(col) * g.Hb + y) * g.Wb + wi;
}
__device__ __forceinline__ bool mask_bit(const uint32_t* __restrict__ bits, const Geom& g, int col, int y, int j) {
  return (*mask_word(bits, g, col, y, j >> 5) >> (j & 31)) & 1u;
}

// ---- pair-interleaved spin storage -----------------------------------------------------------
template <typename V> __device__ __forceinline__ V ld_spin(const V* base, long long idx) {
  using S = decltype(V::x);
  const S* p = reinterpret_cast<const S*>(base) + (2 * idx - (idx & 1));
  V v;
  v.x = p[0]; v.y = p[2];
  return v;
}
template <typename V> __device__ __forceinline__ void st_spin(V* base, long long idx, const V& v) {
  using S = decltype(V::x);
  S* p = reinterpret_cast<S*>(base) + (2 * idx - (idx & 1));
  p[0] = v.x; p[2] = v.y;
}

// ---- block reduction helpers (deterministic order) -------------------------------------
// X_E = S ("the system specific energy ... as 32-bit single precision"): with `single` every partial
// sum of the energy reduction is rounded to float, at every level -- thread, warp, block, grid.  energy_add is the
// per-thread step; the running value is kept in a double variable that then only ever holds floats.
__device__ __forceinline__ double sum_step(double a, double b, int single) {
  return single ? static_cast<double>(static_cast<float>(a) + static_cast<float>(b)) : a + b;
}
__device__ __forceinline__ void energy_add(double& sum, double term, int single) { sum = sum_step(sum, term, single); }
__device__ __forceinline__ double warp_sum(double v, int single = 0) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = sum_step(v, __shfl_down_sync(0xffffffffu, v, o), single);
  return v;
}
__device__ __forceinline__ double block_sum(double v, double* sh /* >= 32 */, int single = 0) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  v = warp_sum(v, single);
  __syncthreads();
  if (lane == 0) sh[w] = v;
  __syncthreads();
  double r = 0.0;
  if (w == 0) {
    r = lane < nw ? sh[lane] : 0.0;
    r = warp_sum(r, single);
  }
  return r;  // valid in thread 0
}

// out[0] = scale * sum(partials[0..n)), fixed order; one block.
static __global__ void final_sum_kernel(const double* __restrict__ partials, int n, double scale, double* out,
                                        int single = 0) {
  __shared__ double sh[32];
  double v = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) v = sum_step(v, partials[i], single);
  v = block_sum(v, sh, single);
  if (threadIdx.x == 0)
    out[0] = single ? static_cast<double>(static_cast<float>(scale) * static_cast<float>(v)) : scale * v;
}

// ---- set-up ---------------------------------------------------------------------------------
// Per-block partials of the measured sample: [0] min, [1] max, [2] count, [3] non-finite count.
static __global__ void sample_range_kernel(const double* __restrict__ z, const uint8_t* __restrict__ mask, size_t N,
                                    double* __restrict__ part /* 4 per block */) {
  double mn = INFINITY, mx = -INFINITY, cnt = 0.0, bad = 0.0;
  for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < N;
       i += static_cast<size_t>(gridDim.x) * blockDim.x) {
    if (mask[i]) continue;
    const double v = z[i];
    cnt += 1.0;
    if (!isfinite(v)) { bad += 1.0; continue; }
    mn = fmin(mn, v); mx = fmax(mx, v);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mn = fmin(mn, __shfl_down_sync(0xffffffffu, mn, o));
    mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
    cnt += __shfl_down_sync(0xffffffffu, cnt, o);
    bad += __shfl_down_sync(0xffffffffu, bad, o);
  }
  __shared__ double sh[4][32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if (lane == 0) { sh[0][w] = mn; sh[1][w] = mx; sh[2][w] = cnt; sh[3][w] = bad; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < nw; ++k) {
      mn = fmin(mn, sh[0][k]); mx = fmax(mx, sh[1][k]); cnt += sh[2][k]; bad += sh[3][k];
    }
    double* p = part + 4 * static_cast<size_t>(blockIdx.x);
    p[0] = mn; p[1] = mx; p[2] = cnt; p[3] = bad;
  }
}
static __global__ void sample_range_final_kernel(const double* __restrict__ part, int nblocks, double* out /* 4 */) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double mn = INFINITY, mx = -INFINITY, cnt = 0.0, bad = 0.0;
  for (int b = 0; b < nblocks; ++b) {
    mn = fmin(mn, part[4 * b]); mx = fmax(mx, part[4 * b + 1]); cnt += part[4 * b + 2]; bad += part[4 * b + 3];
  }
  out[0] = mn; out[1] = mx; out[2] = cnt; out[3] = bad;
}

// R1: phi = 2pi (z - zmin)/(zmax - zmin)
__device__ __forceinline__ double map_to_phi(double z, double zmin, double zmax) {
  return 6.283185307179586476925286766559 * ((z - zmin) / (zmax - zmin));
}

// R6 first half: e_s = -2J mean over measured nearest-neighbour pairs of cos[q(phi_s - phi_t)].
// Per-block partials: [0] sum of cos, [1] pair count.
static __global__ void sample_energy_kernel(const double* __restrict__ z, const uint8_t* __restrict__ mask, int L, int H, int own0, int own1,
                                     double zmin, double zmax, double* __restrict__ part /* 2 per block */, double q) {
  __shared__ double sh[32];
  double sum = 0.0, cnt = 0.0;
  const size_t N = static_cast<size_t>(L) * H;
  for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < N;
       i += static_cast<size_t>(gridDim.x) * blockDim.x) {
    if (mask[i]) continue;
    const int x = static_cast<int>(i % L), y = static_cast<int>(i / L);
    if (y < own0 || y >= own1) continue;      // a slab counts the bonds to the right of and below its own rows
    const double p = map_to_phi(z[i], zmin, zmax);
    if (x < L - 1 && !mask[i + 1]) { sum += cos(q * (p - map_to_phi(z[i + 1], zmin, zmax))); cnt += 1.0; }
    if (y < H - 1 && !mask[i + L]) { sum += cos(q * (p - map_to_phi(z[i + L], zmin, zmax))); cnt += 1.0; }
  }
  const double s = block_sum(sum, sh);
  const double c = block_sum(cnt, sh);
  if (threadIdx.x == 0) { part[2 * blockIdx.x] = s; part[2 * blockIdx.x + 1] = c; }
}
static __global__ void pair_final_kernel(const double* __restrict__ part, int nblocks, double* out /* 2 */) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double s = 0.0, c = 0.0;
  for (int b = 0; b < nblocks; ++b) { s += part[2 * b]; c += part[2 * b + 1]; }
  out[0] = s; out[1] = c;
}

// Mask bitmaps: one thread per 32-bit word of the PADDED arrays (`base` = their first word);
// per-block partial = number of set bits.
static __global__ void pack_mask_kernel(const uint8_t* __restrict__ mask, Geom g, uint32_t* __restrict__ base,
                                 double* __restrict__ part) {
  __shared__ double sh[32];
  const size_t nwords = static_cast<size_t>(2) * g.Hb * g.Wb;
  const size_t w = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x;
  double cnt = 0.0;
  if (w < nwords) {
    const int wi = static_cast<int>(w % g.Wb) - kBitPadLeft;
    const size_t row = w / g.Wb;
    const int y = static_cast<int>(row % g.Hb) - kBitPadTop, col = static_cast<int>(row / g.Hb);
    uint32_t word = 0;
    if (y >= 0 && y < g.H && wi >= 0 && wi < g.Wm) {
      const int par = x_parity(y, col);
      for (int b = 0; b < 32; ++b) {
        const int x = 2 * (32 * wi + b) + par;
        if (x < g.L && mask[static_cast<size_t>(y) * g.L + x]) word |= (1u << b);
      }
    }
    base[w] = word;
    cnt = static_cast<double>(__popc(word));
  }
  const double s = block_sum(cnt, sh);
  if (threadIdx.x == 0) part[blockIdx.x] = s;
}

// ---- chain initialisation (R1 for the measured sites, R8 first half for the free ones) ------
template <int MODE>
__global__ void init_chain_kernel(const double* __restrict__ z, const uint8_t* __restrict__ mask, Geom g,
                                  double zmin, double zmax, uint32_t k0, uint32_t k1, uint32_t trial,
                                  typename Traits<MODE>::vec* __restrict__ state) {
  using V = typename Traits<MODE>::vec;
  const int y = blockIdx.y, col = blockIdx.z;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= g.Wp) return;
  const int x = 2 * j + x_parity(y, col);
  V v;
  v.x = 0; v.y = 0;   // columns past the grid hold the zero vector: they add nothing to a local field
  if (x < g.L) {
    const size_t s = static_cast<size_t>(y) * g.L + x;
    double phi;
    if (mask[s]) {
      const uint4 r = philox4x32_10(g.site0 + static_cast<uint32_t>(s), 0u, PASS_INIT, trial, k0, k1);
      phi = 6.283185307179586476925286766559 * u53(r.x, r.y);
    } else {
      phi = map_to_phi(z[s], zmin, zmax);
    }
    double sn, cs;
    sincos(g.q * phi, &sn, &cs);
    if (sn < 0.0) sn = 0.0;
    // through the arithmetic type of the mode first: with double storage and float arithmetic (MODE_DS) a stored spin
    // must be a value the arithmetic can hand back unchanged, or the tiled kernels (which rewrite every site, moved or
    // not) would round the measured spins on their first pass
    using R = typename Traits<MODE>::real;
    v.x = static_cast<decltype(v.x)>(static_cast<R>(cs));
    v.y = static_cast<decltype(v.y)>(static_cast<R>(sn));
  }
  st_spin(state, static_cast<long long>(col) * g.plane + static_cast<long long>(y) * g.Wp + j, v);
}

// Overwrite the free spins from angles (tests, checkpoint restore).
template <int MODE>
__global__ void set_state_kernel(const double* __restrict__ phi, Geom g, const uint32_t* __restrict__ bits,
                                 typename Traits<MODE>::vec* __restrict__ state) {
  using V = typename Traits<MODE>::vec;
  const int y = blockIdx.y, col = blockIdx.z;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= g.Wp) return;
  if (!mask_bit(bits, g, col, y, j)) return;
  const int x = 2 * j + x_parity(y, col);
  double sn, cs;
  // angles outside [0, 2pi] are clamped to the nearer end: the stored vector is always a
  // unit vector on the upper half circle
  const double p = fmin(fmax(phi[static_cast<size_t>(y) * g.L + x], 0.0), 6.283185307179586476925286766559);
  sincos(g.q * p, &sn, &cs);
  if (sn < 0.0) { sn = 0.0; cs = cs < 0.0 ? -1.0 : 1.0; }
  V v;
  using R = typename Traits<MODE>::real;
  v.x = static_cast<decltype(v.x)>(static_cast<R>(cs));
  v.y = static_cast<decltype(v.y)>(static_cast<R>(sn));
  st_spin(state, static_cast<long long>(col) * g.plane + static_cast<long long>(y) * g.Wp + j, v);
}

template <int MODE>
__global__ void get_state_kernel(const typename Traits<MODE>::vec* __restrict__ state, Geom g,
                                 double* __restrict__ phi) {
  const int y = blockIdx.y;
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  if (x >= g.L) return;
  const int col = (x + y) & 1, j = x >> 1;
  const auto v = ld_spin(state, static_cast<long long>(col) * g.plane + static_cast<long long>(y) * g.Wp + j);
  phi[static_cast<size_t>(y) * g.L + x] = atan2(to_double(v.y), to_double(v.x)) / g.q;
}

// ---- one colour pass on the global planes -------------------------------------------------
// The move of ONE site (row y, plane column j of colour col), in place.  Shared by the kernel that visits every
// plane position and tests its mask bit (PLAIN) and the one that walks the compacted list of prediction sites
// (LIST): the same instructions on the same operands, hence the same spins.  Returns whether a Metropolis move
// was accepted.
template <int MODE, int KIND, bool GENQ = false>
__device__ __forceinline__ bool plain_site_update(typename Traits<MODE>::vec* __restrict__ state, const Geom& g, int col,
                                                  int y, int j, uint32_t sweep,
                                                  const ChainConst<typename Traits<MODE>::real>& k) {
  using R = typename Traits<MODE>::real;
  using V = typename Traits<MODE>::vec;
  bool accepted = false;
  const int par = x_parity(y, col);
  const int x = 2 * j + par;
  V* own = state + static_cast<size_t>(col) * g.plane + static_cast<size_t>(y) * g.Wp;
  const V* oth = state + static_cast<size_t>(1 - col) * g.plane + static_cast<size_t>(y) * g.Wp;
  const bool hl = x > 0, hr = x < g.L - 1, hu = y > 0, hd = y < g.H - 1;
  const int jl = j - 1 + par, jr = j + par;
  V zero; zero.x = 0; zero.y = 0;
  const V l = hl ? ld_spin(oth, jl) : zero;
  const V r = hr ? ld_spin(oth, jr) : zero;
  const V u = hu ? ld_spin(oth, j - g.Wp) : zero;
  const V d = hd ? ld_spin(oth, j + g.Wp) : zero;
  R A, B;
  local_field<R>(R(l.x), R(l.y), R(r.x), R(r.y), R(u.x), R(u.y), R(d.x), R(d.y), hl, hr, hu, hd, &A, &B);
  const V me = ld_spin(own, j);
  R c = R(me.x), s = R(me.y);
  if constexpr (KIND == KIND_MET || KIND == KIND_MO) {
    // R9: the quad (plane columns 2m, 2m + 1) x (rows 2k, 2k + 1) shares one Philox block in the float modes
    const uint32_t pair_site = g.site0 + static_cast<uint32_t>(y) * static_cast<uint32_t>(g.L) +
                               static_cast<uint32_t>(2 * (j & ~1) + par);
    MetWords w0, w1;
    met_words_pair<MODE>(pair_site, sweep, static_cast<uint32_t>(g.L), par, (y & 1) != 0, k, &w0, &w1);
    const MetWords w = (j & 1) ? w1 : w0;
    R o[4];
    bool ok[2];
    met_update2<MODE, GENQ>(bc2(c), bc2(s), bc2(A), bc2(B), w, w, true, true, k, o, ok);   // the site in both lanes
    c = o[0]; s = o[2];
    accepted = ok[0] && y >= g.own0 && y < g.own1;
    if constexpr (KIND == KIND_MO) {     // site-fused schedule (R4b): the over-relaxation move follows at once
      R o2[4];
      or_update2<MODE, GENQ>(bc2(c), bc2(s), bc2(A), bc2(B), true, true, o2, &k);
      c = o2[0]; s = o2[2];
    }
  } else if constexpr (KIND == KIND_OR) {
    R o[4];
    or_update2<MODE, GENQ>(bc2(c), bc2(s), bc2(A), bc2(B), true, true, o, &k);
    c = o[0]; s = o[2];
  } else {
    quench_update<MODE, GENQ>(&c, &s, A, B, &k);
  }
  V out;
  out.x = static_cast<decltype(out.x)>(c);
  out.y = static_cast<decltype(out.y)>(s);
  st_spin(own, j, out);
  return accepted;
}

template <int MODE, int KIND, bool GENQ = false>
__global__ void __launch_bounds__(128)
plain_pass_kernel(typename Traits<MODE>::vec* __restrict__ state, const uint32_t* __restrict__ bits, Geom g,
                  int col, uint32_t sweep, ChainConst<typename Traits<MODE>::real> k,
                  unsigned long long* __restrict__ accept_slots) {
  const int y = blockIdx.y;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  bool accepted = false;
  if (j < g.Wp && mask_bit(bits, g, col, y, j)) accepted = plain_site_update<MODE, KIND, GENQ>(state, g, col, y, j, sweep, k);
  if constexpr (KIND == KIND_MET || KIND == KIND_MO) {
    const int n = __syncthreads_count(accepted);
    if (threadIdx.x == 0 && n)
      atomicAdd(accept_slots + ((blockIdx.y * gridDim.x + blockIdx.x) & 1023u), static_cast<unsigned long long>(n));
  }
}

// ---- LIST path: the compacted per-colour lists of prediction sites (north_star (a)) ------------------------------
// list[col] holds the plane positions y * Wp + j of the prediction sites of colour col in row-major order, n[col]
// of them.  Built once per context from the mask bitmaps: per-row counts, an exclusive scan over the rows, then
// every row writes its positions.  A pass over a list does work proportional to the number of PREDICTION sites of
// the colour, whatever the masked fraction; neighbour reads are gathers from the global planes.
static __global__ void list_row_count_kernel(const uint32_t* __restrict__ bits, Geom g, uint32_t* __restrict__ row_count) {
  __shared__ double sh[32];
  const int y = blockIdx.x, col = blockIdx.y;
  double n = 0.0;
  for (int wi = threadIdx.x; wi < g.Wm; wi += blockDim.x) n += static_cast<double>(__popc(*mask_word(bits, g, col, y, wi)));
  const double s = block_sum(n, sh);
  if (threadIdx.x == 0) row_count[static_cast<size_t>(col) * g.H + y] = static_cast<uint32_t>(s);
}
// exclusive scan of the row counts of both colours (one block; L = number of ROWS <= 32768): row_off[col][y], total[col]
static __global__ void list_row_scan_kernel(const uint32_t* __restrict__ row_count, int L, uint32_t* __restrict__ row_off,
                                            uint32_t* __restrict__ total) {
  __shared__ uint32_t part[1024];
  for (int col = 0; col < 2; ++col) {
    const uint32_t* rc = row_count + static_cast<size_t>(col) * L;
    uint32_t* ro = row_off + static_cast<size_t>(col) * L;
    const int per = (L + blockDim.x - 1) / blockDim.x;
    const int lo = threadIdx.x * per, hi = min(L, lo + per);
    uint32_t s = 0;
    for (int y = lo; y < hi; ++y) s += rc[y];
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
      uint32_t run = 0;
      for (int t = 0; t < static_cast<int>(blockDim.x); ++t) { const uint32_t v = part[t]; part[t] = run; run += v; }
      total[col] = run;
    }
    __syncthreads();
    uint32_t run = part[threadIdx.x];
    for (int y = lo; y < hi; ++y) { ro[y] = run; run += rc[y]; }
    __syncthreads();
  }
}
// one warp per row: positions in increasing column order
static __global__ void list_fill_kernel(const uint32_t* __restrict__ bits, Geom g, const uint32_t* __restrict__ row_off,
                                        uint32_t* __restrict__ list0, uint32_t* __restrict__ list1) {
  const int y = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), col = blockIdx.y, lane = threadIdx.x & 31;
  if (y >= g.H) return;
  uint32_t* out = (col ? list1 : list0) + row_off[static_cast<size_t>(col) * g.H + y];
  uint32_t base = 0;
  for (int w0 = 0; w0 < g.Wm; w0 += 32) {
    const int wi = w0 + lane;
    const uint32_t word = wi < g.Wm ? *mask_word(bits, g, col, y, wi) : 0u;
    const uint32_t cnt = __popc(word);
    uint32_t incl = cnt;                                  // inclusive prefix of the counts over the warp
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += v;
    }
    uint32_t pos = base + incl - cnt;
    uint32_t rest = word;
    while (rest) {
      const int b = __ffs(rest) - 1;
      rest &= rest - 1;
      out[pos++] = static_cast<uint32_t>(y) * static_cast<uint32_t>(g.Wp) + static_cast<uint32_t>(32 * wi + b);
    }
    base += __shfl_sync(0xffffffffu, incl, 31);
  }
}

template <int MODE, int KIND, bool GENQ = false>
__global__ void __launch_bounds__(128)
list_pass_kernel(typename Traits<MODE>::vec* __restrict__ state, const uint32_t* __restrict__ list, uint32_t n, Geom g,
                 int col, uint32_t sweep, ChainConst<typename Traits<MODE>::real> k,
                 unsigned long long* __restrict__ accept_slots) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  bool accepted = false;
  if (i < n) {
    const uint32_t pos = list[i];
    const int y = static_cast<int>(pos / static_cast<uint32_t>(g.Wp)), j = static_cast<int>(pos % static_cast<uint32_t>(g.Wp));
    accepted = plain_site_update<MODE, KIND, GENQ>(state, g, col, y, j, sweep, k);
  }
  if constexpr (KIND == KIND_MET || KIND == KIND_MO) {
    const int m = __syncthreads_count(accepted);
    if (threadIdx.x == 0 && m) atomicAdd(accept_slots + (blockIdx.x & 1023u), static_cast<unsigned long long>(m));
  }
}

// ---- energy (R3): every bond has exactly one colour-1 end, so H = -J sum over colour-1
// sites of site_energy_term (mpr_device.cuh): u_s . F_s in the double-arithmetic modes, the
// per-bond form n - sum_j |u_s - u_j|^2 / 2 in the float-arithmetic modes.  Terms in the mode's
// arithmetic, sums in double (R13).  Missing neighbours are passed as the zero vector.
template <int MODE>
__global__ void __launch_bounds__(256)
plain_energy_kernel(const typename Traits<MODE>::vec* __restrict__ state, Geom g, double* __restrict__ part) {
  using R = typename Traits<MODE>::real;
  using V = typename Traits<MODE>::vec;
  __shared__ double sh[32];
  double sum = 0.0;
  const int col = 1;
  for (int y = g.own0 + blockIdx.x; y < g.own1; y += gridDim.x) {
    const int par = x_parity(y, col);
    const V* own = state + static_cast<size_t>(col) * g.plane + static_cast<size_t>(y) * g.Wp;
    const V* oth = state + static_cast<size_t>(1 - col) * g.plane + static_cast<size_t>(y) * g.Wp;
    for (int j = threadIdx.x; j < g.Wp; j += blockDim.x) {
      const int x = 2 * j + par;
      if (x >= g.L) continue;
      const bool hl = x > 0, hr = x < g.L - 1, hu = y > 0, hd = y < g.H - 1;
      V zero; zero.x = 0; zero.y = 0;
      const V l = hl ? ld_spin(oth, j - 1 + par) : zero;
      const V r = hr ? ld_spin(oth, j + par) : zero;
      const V u = hu ? ld_spin(oth, j - g.Wp) : zero;
      const V d = hd ? ld_spin(oth, j + g.Wp) : zero;
      const V me = ld_spin(own, j);
      energy_add(sum, site_energy_term<R>(R(me.x), R(me.y), R(l.x), R(l.y), R(r.x), R(r.y), R(u.x), R(u.y), R(d.x), R(d.y)),
                 g.energy_single);
    }
  }
  const double s = block_sum(sum, sh, g.energy_single);
  if (threadIdx.x == 0) part[blockIdx.x] = s;
}

// ---- accumulation of phi at the free sites (R15) and the back-map --------------------------
template <int MODE>
__global__ void plain_accumulate_kernel(const typename Traits<MODE>::vec* __restrict__ state,
                                        const uint32_t* __restrict__ bits, Geom g, double* __restrict__ acc) {
  using R = typename Traits<MODE>::real;
  const int y = blockIdx.y, col = blockIdx.z;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= g.Wp || !mask_bit(bits, g, col, y, j)) return;
  const size_t i = static_cast<size_t>(col) * g.plane + static_cast<size_t>(y) * g.Wp + j;
  const auto v = ld_spin(state, static_cast<long long>(i));
  acc[i] += spin_angle<MODE>(R(v.x), R(v.y), 1.0 / g.q);
}

static __global__ void clear_acc_kernel(double* __restrict__ acc, size_t n) {
  for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < n;
       i += static_cast<size_t>(gridDim.x) * blockDim.x)
    acc[i] = 0.0;
}

// pred = zmin + (zmax - zmin) * acc / (2pi n_acc) at prediction sites, the input value elsewhere.
static __global__ void predict_kernel(const double* __restrict__ z, const uint8_t* __restrict__ mask, Geom g,
                               const double* __restrict__ acc, double zmin, double zmax, long long n_acc,
                               double* __restrict__ pred) {
  const int y = blockIdx.y;
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  if (x >= g.L) return;
  const size_t s = static_cast<size_t>(y) * g.L + x;
  if (!mask[s]) { pred[s] = z[s]; return; }
  if (n_acc == 0) { pred[s] = __longlong_as_double(0x7ff8000000000000LL); return; }
  const int col = (x + y) & 1, j = x >> 1;
  const double a = acc[static_cast<size_t>(col) * g.plane + static_cast<size_t>(y) * g.Wp + j];
  const double frac = a / (6.283185307179586476925286766559 * static_cast<double>(n_acc));
  pred[s] = zmin + (zmax - zmin) * frac;
}

static __global__ void philox_debug_kernel(const uint32_t* __restrict__ ctr, uint32_t k0, uint32_t k1,
                                    uint32_t* __restrict__ out, long long n) {
  const long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x;
  if (i >= n) return;
  const uint4 r = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], k0, k1);
  out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

// out[i]: bit 0 = decision of metropolis_accept_exact, bit 1 = decision of the plain double evaluation
// u53(wa, wb) < exp_nonpos(mdE / T), bit 2 = the float filter decided alone
static __global__ void accept_debug_kernel(const uint32_t* __restrict__ w, const double* __restrict__ mdE, double T,
                                           uint8_t* __restrict__ out, long long n) {
  const long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x;
  if (i >= n) return;
  const double inv_T = 1.0 / T, xs = 1.4426950408889634074 / T;
  bool fast = true;
  const bool a = metropolis_accept_exact(w[2 * i], w[2 * i + 1], mdE[i], inv_T, xs, &fast);
  const bool b = u53(w[2 * i], w[2 * i + 1]) < exp_nonpos(mdE[i] * inv_T);
  out[i] = static_cast<uint8_t>((a ? 1 : 0) | (b ? 2 : 0) | (fast ? 4 : 0));
}

}  // namespace mpr
