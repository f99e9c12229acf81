// mpr_static.cu -- the one entry point of libmpr.so that needs NO caller workspace and allocates nothing:
// mpr_sample_energy_static (include/mpr.h).  It computes the sample statistics the method starts from -- the range
// of the measured values (R1) and the sample energy e_s over measured nearest-neighbour pairs (R6, first half;
// PAPER.md:31) -- for callers that cannot call cudaMalloc (code under CUDA-graph capture, serving loops, harnesses
// that forbid it) and have no workspace to hand to mpr_create.
//
// The per-block partial results that the context path keeps in the caller's workspace live here in ONE file-scope
// device array of fixed size (kScratchDoubles doubles = 49 216 bytes, held by every GPU that loads the library until
// the process exits).  Consequences, all stated in the header too:
//   * the entry point rejects grids of more than kStaticMaxSites sites;
//   * every call on a device shares the array: calls that overlap on the GPU (two streams, two threads) race;
//   * the array keeps the last call's contents.  Nothing in it has to start at zero -- every slot a call reads it
//     has written first (each block stores its partials unconditionally, the final kernels read exactly the slots
//     of the blocks of this call) -- and the scalar slots are overwritten at the start of every call anyway.
// In host code the array's name is a host-side stand-in, not a device address: its address is taken once per device
// with cudaGetSymbolAddress (device current) and that pointer is what the kernels are given.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <mutex>
#include <string>

#include "../../include/mpr.h"
#include "mpr_plain.cuh"

namespace mpr {
namespace {

constexpr int kStaticBlocks = 1024;                       // at most this many blocks of 256 threads per kernel
constexpr long long kStaticMaxSites = 1ll << 28;          // 16384 x 16384: a thread walks at most 1024 sites
constexpr int kRangeOff = 0;                              // [kStaticBlocks][4]  min, max, count, non-finite count
constexpr int kPairOff = 4 * kStaticBlocks;               // [kStaticBlocks][2]  sum of cos, pair count
constexpr int kScalOff = 6 * kStaticBlocks;               // [8]                 z_min, z_max, count, non-finite count
constexpr int kScratchDoubles = 6 * kStaticBlocks + 8;    // 49 216 bytes

static __device__ __align__(256) double g_static_scratch[kScratchDoubles];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
double* g_scratch_ptr[kMaxDevices] = {};                  // device address of the array, per device
thread_local std::string g_err;

int fail(int code, const std::string& msg) { g_err = msg; return code; }

// Device address of the scratch array on the CURRENT device (taken once per device).
int scratch_address(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(MPR_ERR_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDevices) return fail(MPR_ERR_CUDA, "device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p)
      return fail(MPR_ERR_CUDA, std::string("cudaGetSymbolAddress(g_static_scratch): ") + cudaGetErrorString(e));
    g_scratch_ptr[dev] = static_cast<double*>(p);
  }
  *out = g_scratch_ptr[dev];
  return MPR_OK;
}

// The variant of sample_energy_kernel (mpr_plain.cuh) of this entry point: the range of the sample is read from
// the scratch array (where static_range_final_kernel left it) instead of arriving as kernel arguments from the host,
// so that no host round trip separates the two steps.  Same loop, same order of operations per thread and block.
__global__ void sample_energy_static_kernel(const double* __restrict__ z, const uint8_t* __restrict__ mask, int L, int H,
                                            const double* __restrict__ scal, double* __restrict__ part, double q) {
  __shared__ double sh[32];
  const double zmin = scal[0], zmax = scal[1];
  double sum = 0.0, cnt = 0.0;
  const size_t N = static_cast<size_t>(L) * H;
  for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < N;
       i += static_cast<size_t>(gridDim.x) * blockDim.x) {
    if (mask[i]) continue;
    const int x = static_cast<int>(i % L), y = static_cast<int>(i / L);
    const double p = map_to_phi(z[i], zmin, zmax);
    if (x < L - 1 && !mask[i + 1]) { sum += cos(q * (p - map_to_phi(z[i + 1], zmin, zmax))); cnt += 1.0; }
    if (y < H - 1 && !mask[i + L]) { sum += cos(q * (p - map_to_phi(z[i + L], zmin, zmax))); cnt += 1.0; }
  }
  const double s = block_sum(sum, sh);
  const double c = block_sum(cnt, sh);
  if (threadIdx.x == 0) { part[2 * blockIdx.x] = s; part[2 * blockIdx.x + 1] = c; }
}

// Sums the pair partials and writes the six results.  e_s is NaN when it is undefined: no measured pair, a
// non-finite measured value, or z_max == z_min (the conditions mpr_create reports as errors; here they cannot be
// reported by the host without a synchronisation, so the caller reads them off the output).
__global__ void static_finish_kernel(const double* __restrict__ part, int nblocks, const double* __restrict__ scal,
                                     double* __restrict__ out /* 6 */) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double s = 0.0, c = 0.0;
  for (int b = 0; b < nblocks; ++b) { s += part[2 * b]; c += part[2 * b + 1]; }
  const double zmin = scal[0], zmax = scal[1], n_meas = scal[2], bad = scal[3];
  const bool defined = c > 0.0 && bad == 0.0 && zmax > zmin;
  out[0] = defined ? -2.0 * 1.0 * s / c : __longlong_as_double(0x7ff8000000000000LL);      // J = 1 (R3)
  out[1] = c;
  out[2] = zmin;
  out[3] = zmax;
  out[4] = n_meas;
  out[5] = bad;
}

}  // namespace
}  // namespace mpr

extern "C" {

const char* mpr_static_last_error(void) { return mpr::g_err.c_str(); }

int mpr_static_setup(void) {
  double* p = nullptr;
  return mpr::scratch_address(&p);
}

int64_t mpr_static_max_sites(void) { return mpr::kStaticMaxSites; }

int mpr_sample_energy_static(int Lx, int Ly, const double* d_values, const uint8_t* d_mask, double q, void* cuda_stream,
                             double* d_out) {
  using namespace mpr;
  if (Lx < 1 || Ly < 1 || static_cast<long long>(Lx) * Ly < 2)
    return fail(MPR_ERR_INVALID_ARG, "mpr_sample_energy_static: the grid needs at least two sites");
  if (static_cast<long long>(Lx) * Ly > kStaticMaxSites)
    return fail(MPR_ERR_INVALID_ARG, "mpr_sample_energy_static: " + std::to_string(static_cast<long long>(Lx) * Ly) +
                                         " sites exceed the " + std::to_string(kStaticMaxSites) +
                                         " the built-in scratch array is sized for; use mpr_create with a workspace");
  if (!d_values || !d_mask || !d_out) return fail(MPR_ERR_INVALID_ARG, "mpr_sample_energy_static: null pointer");
  if (!(q > 0.0 && q <= 0.5)) return fail(MPR_ERR_INVALID_ARG, "mpr_sample_energy_static: q outside (0, 1/2]");
  double* scratch = nullptr;
  const int st = scratch_address(&scratch);
  if (st != MPR_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const size_t N = static_cast<size_t>(Lx) * Ly;
  const int nblk = static_cast<int>(N / 256 + 1 < static_cast<size_t>(kStaticBlocks) ? N / 256 + 1 : kStaticBlocks);
  double* range_part = scratch + kRangeOff;
  double* pair_part = scratch + kPairOff;
  double* scal = scratch + kScalOff;
  sample_range_kernel<<<nblk, 256, 0, s>>>(d_values, d_mask, N, range_part);
  sample_range_final_kernel<<<1, 32, 0, s>>>(range_part, nblk, scal);
  sample_energy_static_kernel<<<nblk, 256, 0, s>>>(d_values, d_mask, Lx, Ly, scal, pair_part, q);
  static_finish_kernel<<<1, 32, 0, s>>>(pair_part, nblk, scal, d_out);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(MPR_ERR_CUDA, std::string("mpr_sample_energy_static launch: ") + cudaGetErrorString(e));
  g_err.clear();
  return MPR_OK;
}

}  // extern "C"
