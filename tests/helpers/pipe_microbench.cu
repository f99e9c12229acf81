// pipe_microbench.cu -- measured per-SM instruction throughputs of the sm_100a pipes the MPR sweep
// kernels run on, and L2 / HBM copy bandwidths.  Test-side program (bench.py --microbench builds and
// runs it; the numbers go into profiles/ and into bench.py's "alu" ceilings).  Nothing of the
// library is used here.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o pipe_microbench pipe_microbench.cu
//
// Every test: each thread runs ILP independent dependency chains of one instruction kind for ITER
// iterations; 148 x CTAS CTAs of 1024 threads (all resident at once); cycles = clock64() span of
// each CTA, averaged.  Reported: warp instructions per clock per SM (4 schedulers: 4.0 = one per
// scheduler and clock), so the figures do not depend on the SM clock of the day.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_)); exit(2); } } while (0)

constexpr int ITER = 1024;
constexpr int ILP = 8;

template <int KIND> struct Op;
// 0: FFMA (three register operands)
template <> struct Op<0> { static constexpr const char* name = "FFMA r,r,r";
  using T = float; static __device__ T init(int i) { return 1.0f + i; }
  static __device__ void step(T& x, T a, T b) { asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x) : "f"(a), "f"(b)); } };
// 1: FFMA2 (packed f32x2)
template <> struct Op<1> { static constexpr const char* name = "FFMA2 (fma.rn.f32x2)";
  using T = unsigned long long; static __device__ T init(int i) { return 0x3f8000003f800000ull + i; }
  static __device__ void step(T& x, T a, T b) { asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x) : "l"(a), "l"(b)); } };
// 2: FMUL2
template <> struct Op<2> { static constexpr const char* name = "FMUL2 (mul.rn.f32x2)";
  using T = unsigned long long; static __device__ T init(int i) { return 0x3f8000003f800000ull + i; }
  static __device__ void step(T& x, T a, T) { asm volatile("mul.rn.f32x2 %0, %0, %1;" : "+l"(x) : "l"(a)); } };
// 3: FADD2
template <> struct Op<3> { static constexpr const char* name = "FADD2 (add.rn.f32x2)";
  using T = unsigned long long; static __device__ T init(int i) { return 0x3f8000003f800000ull + i; }
  static __device__ void step(T& x, T a, T) { asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(x) : "l"(a)); } };
// 4: IMAD.WIDE.U32 (32 x 32 -> 64, the Philox multiply)
template <> struct Op<4> { static constexpr const char* name = "IMAD.WIDE.U32 (mul.wide.u32)";
  using T = unsigned long long; static __device__ T init(int i) { return 0x9E3779B97F4A7C15ull + i; }
  static __device__ void step(T& x, T, T) {
    asm volatile("{ .reg .b32 lo, hi; mov.b64 {lo, hi}, %0; xor.b32 lo, lo, hi; mul.wide.u32 %0, lo, 0xD2511F53; }" : "+l"(x)); } };
// 5: LOP3
template <> struct Op<5> { static constexpr const char* name = "LOP3 (3-input xor)";
  using T = unsigned; static __device__ T init(int i) { return 0x12345u + i; }
  static __device__ void step(T& x, T a, T b) { asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x) : "r"(a), "r"(b)); } };
// 6: MUFU.EX2
template <> struct Op<6> { static constexpr const char* name = "MUFU.EX2 (ex2.approx.ftz.f32)";
  using T = float; static __device__ T init(int i) { return -0.5f - i; }
  static __device__ void step(T& x, T, T) { asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x)); } };
// 7: MUFU.SIN
template <> struct Op<7> { static constexpr const char* name = "MUFU.SIN (sin.approx.ftz.f32: FMUL + MUFU)";
  using T = float; static __device__ T init(int i) { return 0.5f + i; }
  static __device__ void step(T& x, T, T) { asm volatile("sin.approx.ftz.f32 %0, %0;" : "+f"(x)); } };
// 8: MUFU.RCP
template <> struct Op<8> { static constexpr const char* name = "MUFU.RCP (rcp.approx.ftz.f32)";
  using T = float; static __device__ T init(int i) { return 1.5f + i; }
  static __device__ void step(T& x, T, T) { asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(x)); } };
// 9: DFMA
template <> struct Op<9> { static constexpr const char* name = "DFMA";
  using T = double; static __device__ T init(int i) { return 1.0 + i; }
  static __device__ void step(T& x, T a, T b) { asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(x) : "d"(a), "d"(b)); } };
// 10: FSETP + FSEL (compare and select, the accept / keep pattern)
template <> struct Op<10> { static constexpr const char* name = "FSETP + FSEL pair (2 instructions)";
  using T = float; static __device__ T init(int i) { return 1.0f + i; }
  static __device__ void step(T& x, T a, T b) {
    asm volatile("{ .reg .pred p; setp.ge.f32 p, %0, %1; selp.f32 %0, %2, %1, p; }" : "+f"(x) : "f"(a), "f"(b)); } };
// 11: I2F (int32 -> float, the random-word conversion)
template <> struct Op<11> { static constexpr const char* name = "I2FP.F32.S32 + F2I pair (2 instructions)";
  using T = int; static __device__ T init(int i) { return 12345 + i; }
  static __device__ void step(T& x, T, T) {
    asm volatile("{ .reg .f32 f; cvt.rn.f32.s32 f, %0; cvt.rzi.s32.f32 %0, f; }" : "+r"(x)); } };
// 12: SHFL
template <> struct Op<12> { static constexpr const char* name = "SHFL.UP";
  using T = unsigned; static __device__ T init(int i) { return 7u + i; }
  static __device__ void step(T& x, T, T) { asm volatile("shfl.sync.up.b32 %0, %0, 1, 0, 0xffffffff;" : "+r"(x)); } };
// 13: IMAD (32-bit low product + add)
template <> struct Op<13> { static constexpr const char* name = "IMAD (mad.lo.u32)";
  using T = unsigned; static __device__ T init(int i) { return 7u + i; }
  static __device__ void step(T& x, T a, T b) { asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x) : "r"(a), "r"(b)); } };
// 14: a whole Philox4x32-10 block, unrolled as the sweep kernel has it: 20 IMAD.WIDE + 20 LOP3
template <> struct Op<14> { static constexpr const char* name = "Philox4x32-10 block (20 IMAD.WIDE + 20 LOP3 = 40 instructions)";
  using T = uint4; static __device__ T init(int i) { return make_uint4(1 + i, 2, 3, 4); }
  static __device__ void step(T& c, T k, T) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
      const unsigned long long p0 = (unsigned long long)0xD2511F53u * c.x, p1 = (unsigned long long)0xCD9E8D57u * c.z;
      const unsigned n0 = (unsigned)(p1 >> 32) ^ c.y ^ k.x, n2 = (unsigned)(p0 >> 32) ^ c.w ^ k.y;
      c = make_uint4(n0, (unsigned)p1, n2, (unsigned)p0);
    }
  } };
// 15: FFMA2 and LOP3 interleaved 1:1 (two pipes at once)
struct MixState { unsigned long long v; unsigned z, pad; };
template <> struct Op<15> { static constexpr const char* name = "FFMA2 + LOP3 interleaved (2 instructions)";
  using T = MixState; static __device__ T init(int i) { return MixState{0x3f8000003f800000ull + i, 5u + i, 77u * i}; }
  static __device__ void step(T& c, T k, T) {
    asm volatile("fma.rn.f32x2 %0, %0, %1, %1;" : "+l"(c.v) : "l"(k.v));
    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(c.z) : "r"(k.z), "r"(k.pad)); } };
// 16: IMAD.WIDE and FFMA2 interleaved 1:1 (both on the FMA pipe?)
template <> struct Op<16> { static constexpr const char* name = "FFMA2 + IMAD.WIDE interleaved (2 instructions + 1 LOP3)";
  using T = MixState; static __device__ T init(int i) { return MixState{0x3f8000003f800000ull + i, 5u + i, 77u * i}; }
  static __device__ void step(T& c, T k, T) {
    asm volatile("fma.rn.f32x2 %0, %0, %1, %1;" : "+l"(c.v) : "l"(k.v));
    unsigned long long w = ((unsigned long long)c.pad << 32) | c.z;
    asm volatile("{ .reg .b32 lo, hi; mov.b64 {lo, hi}, %0; xor.b32 lo, lo, hi; mul.wide.u32 %0, lo, 0xD2511F53; }" : "+l"(w));
    c.z = (unsigned)w; c.pad = (unsigned)(w >> 32); } };
template <int KIND>
__global__ void __launch_bounds__(1024, 1) pipe_kernel(const unsigned long long* __restrict__ seed, unsigned long long* sink,
                                                        long long* cycles) {
  using T = typename Op<KIND>::T;
  T x[ILP];
#pragma unroll
  for (int i = 0; i < ILP; ++i) x[i] = Op<KIND>::init(i + threadIdx.x);
  T a, b;
  {  // opaque operands (loaded, so nothing folds)
    const unsigned long long s0 = seed[0], s1 = seed[1];
    if constexpr (sizeof(T) == 16) { a = *reinterpret_cast<const T*>(seed); b = a; }
    else if constexpr (sizeof(T) == 8) { a = *reinterpret_cast<const T*>(&s0); b = *reinterpret_cast<const T*>(&s1); }
    else { const unsigned u0 = (unsigned)s0, u1 = (unsigned)s1; a = *reinterpret_cast<const T*>(&u0); b = *reinterpret_cast<const T*>(&u1); }
  }
  __syncthreads();
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < ITER; ++it) {
#pragma unroll
    for (int i = 0; i < ILP; ++i) Op<KIND>::step(x[i], a, b);
  }
  const long long t1 = clock64();
  __syncthreads();
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
  unsigned long long acc = 0;
#pragma unroll
  for (int i = 0; i < ILP; ++i) {
    if constexpr (sizeof(T) == 16) { const uint4 q = *reinterpret_cast<uint4*>(&x[i]); acc += q.x + q.y + q.z + q.w; }
    else if constexpr (sizeof(T) == 8) acc += *reinterpret_cast<unsigned long long*>(&x[i]);
    else acc += *reinterpret_cast<unsigned*>(&x[i]);
  }
  if (acc == seed[3]) sink[0] = acc;      // run-time value: the chains cannot be folded away
}

template <int KIND>
void run_pipe(int nsm, unsigned long long* d_seed, unsigned long long* d_sink, long long* d_cyc, double inst_per_step) {
  const int grid = nsm;                       // one 1024-thread CTA per SM: 32 warps, 8 per scheduler
  pipe_kernel<KIND><<<grid, 1024>>>(d_seed, d_sink, d_cyc);
  CK(cudaDeviceSynchronize());
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  CK(cudaEventRecord(e0));
  pipe_kernel<KIND><<<grid, 1024>>>(d_seed, d_sink, d_cyc);
  CK(cudaEventRecord(e1));
  CK(cudaDeviceSynchronize());
  float ms = 0;
  CK(cudaEventElapsedTime(&ms, e0, e1));
  std::vector<long long> h(grid);
  CK(cudaMemcpy(h.data(), d_cyc, grid * sizeof(long long), cudaMemcpyDeviceToHost));
  double cyc = 0;
  for (long long c : h) cyc += (double)c;
  cyc /= grid;
  const double warp_inst = 32.0 * ITER * ILP * inst_per_step;    // per SM
  printf("{\"test\": \"%s\", \"warp_inst_per_clk_per_sm\": %.4f, \"cycles\": %.0f, \"ms\": %.4f, \"sm_mhz_effective\": %.0f}\n",
         Op<KIND>::name, warp_inst / cyc, cyc, ms, cyc / (ms * 1e3));
}

__global__ void copy_kernel(const float4* __restrict__ src, float4* __restrict__ dst, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

void run_copy(const char* name, size_t bytes, int reps) {
  float4 *a, *b;
  CK(cudaMalloc(&a, bytes)); CK(cudaMalloc(&b, bytes));
  CK(cudaMemset(a, 1, bytes)); CK(cudaMemset(b, 0, bytes));
  const size_t n = bytes / sizeof(float4);
  for (int i = 0; i < 3; ++i) copy_kernel<<<148 * 8, 512>>>(a, b, n);
  CK(cudaDeviceSynchronize());
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  float best = 1e30f;
  for (int r = 0; r < 5; ++r) {
    CK(cudaEventRecord(e0));
    for (int i = 0; i < reps; ++i) copy_kernel<<<148 * 8, 512>>>(a, b, n);
    CK(cudaEventRecord(e1));
    CK(cudaDeviceSynchronize());
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    if (ms < best) best = ms;
  }
  printf("{\"test\": \"%s\", \"bytes_per_buffer\": %zu, \"read_plus_write_gb_per_s\": %.1f}\n", name, bytes,
         2.0 * bytes * reps / (best * 1e-3) / 1e9);
  CK(cudaFree(a)); CK(cudaFree(b));
}

int main() {
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, 0));
  const int nsm = prop.multiProcessorCount;
  printf("{\"device\": \"%s\", \"sms\": %d, \"l2_bytes\": %d, \"iter\": %d, \"ilp\": %d, \"warps_per_sm\": 32}\n", prop.name, nsm,
         prop.l2CacheSize, ITER, ILP);
  unsigned long long *d_seed, *d_sink;
  long long* d_cyc;
  CK(cudaMalloc(&d_seed, 64)); CK(cudaMalloc(&d_sink, 64)); CK(cudaMalloc(&d_cyc, nsm * sizeof(long long)));
  const unsigned long long hs[4] = {0x3f7ff0003f7ff000ull, 0x3a8000003a800000ull, 0, 0x0123456789abcdefull};
  CK(cudaMemcpy(d_seed, hs, sizeof(hs), cudaMemcpyHostToDevice));
  run_pipe<0>(nsm, d_seed, d_sink, d_cyc, 1);
  run_pipe<1>(nsm, d_seed, d_sink, d_cyc, 1);
  run_pipe<2>(nsm, d_seed, d_sink, d_cyc, 1);
  run_pipe<3>(nsm, d_seed, d_sink, d_cyc, 1);
  run_pipe<4>(nsm, d_seed, d_sink, d_cyc, 2);     // xor (LOP3) + IMAD.WIDE
  run_pipe<5>(nsm, d_seed, d_sink, d_cyc, 1);
  run_pipe<6>(nsm, d_seed, d_sink, d_cyc, 1);
  run_pipe<7>(nsm, d_seed, d_sink, d_cyc, 2);
  run_pipe<8>(nsm, d_seed, d_sink, d_cyc, 1);
  run_pipe<9>(nsm, d_seed, d_sink, d_cyc, 1);
  run_pipe<10>(nsm, d_seed, d_sink, d_cyc, 2);
  run_pipe<11>(nsm, d_seed, d_sink, d_cyc, 2);
  run_pipe<12>(nsm, d_seed, d_sink, d_cyc, 1);
  run_pipe<13>(nsm, d_seed, d_sink, d_cyc, 1);
  run_pipe<14>(nsm, d_seed, d_sink, d_cyc, 40);
  run_pipe<15>(nsm, d_seed, d_sink, d_cyc, 2);
  run_pipe<16>(nsm, d_seed, d_sink, d_cyc, 3);
  run_copy("L2-resident copy (2 x 16 MiB)", (size_t)16 << 20, 200);
  run_copy("L2-resident copy (2 x 32 MiB)", (size_t)32 << 20, 100);
  run_copy("HBM copy (2 x 4 GiB)", (size_t)4 << 30, 3);
  return 0;
}
