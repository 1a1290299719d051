// das_convert: layout transform + cast (the paper's permute-and-convert pre-pass,
// PAPER.md:149, :200).
//
//   in : raw  [Q][M][K]    complex64 / float32, samples contiguous in k
//   out: conv [M][Q][Kp]   (mid, slope) table entries in storage precision (das_internal.cuh):
//          entry i <-> sample interval k = i - kPadLeft
//          mid_k = y_k/2 + y_k+1/2,  slope_k = y_k+1 - y_k   for 0 <= k <= K-2, else (0, 0)
//
// The only arithmetic is the optional scale, one add and one subtract in FP32, and the cast
// (round to nearest even for fp16; overflow gives +-inf).  Pure streaming, HBM-bound:
// 8 B read + 8 B (fp16) or 16 B (fp32) written per complex sample.  One thread produces 4
// consecutive entries of one (m, q) row from 5 consecutive samples, so a warp reads ~1 KiB of
// contiguous complex64 and writes 1 KiB (fp16) / 2 KiB (fp32) contiguous, with 16-byte stores.
#include "das_internal.cuh"

namespace das {

namespace {

__device__ __forceinline__ float2 ldg_stream(const float2* p) {
  float2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ float ldg_stream(const float* p) {
  float v;
  asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ float2 scaled(float2 v, float s) { return make_float2(v.x * s, v.y * s); }
__device__ __forceinline__ float scaled(float v, float s) { return v * s; }
__device__ __forceinline__ void zero(float2& v) { v = make_float2(0.f, 0.f); }
__device__ __forceinline__ void zero(float& v) { v = 0.f; }

// mid = a/2 + b/2 (each halving exact, one rounding), slope = b - a; no FMA contraction.
__device__ __forceinline__ float mid_of(float a, float b) { return __fadd_rn(__fmul_rn(a, 0.5f), __fmul_rn(b, 0.5f)); }
__device__ __forceinline__ float slope_of(float a, float b) { return __fadd_rn(b, -a); }

__device__ __forceinline__ unsigned pack_h2(float lo, float hi) {
  const __half2 h = __floats2half2_rn(lo, hi);
  return *reinterpret_cast<const unsigned*>(&h);
}

// one table entry from the two samples that bound its interval
__device__ __forceinline__ void make_entry(float4& e, float2 a, float2 b) {
  e = make_float4(mid_of(a.x, b.x), mid_of(a.y, b.y), slope_of(a.x, b.x), slope_of(a.y, b.y));
}
__device__ __forceinline__ void make_entry(uint2& e, float2 a, float2 b) {
  e = make_uint2(pack_h2(mid_of(a.x, b.x), mid_of(a.y, b.y)), pack_h2(slope_of(a.x, b.x), slope_of(a.y, b.y)));
}
__device__ __forceinline__ void make_entry(Fp8x4& e, float2 a, float2 b) {
  e.v = (unsigned)float2_to_fp8x2(mid_of(a.x, b.x), mid_of(a.y, b.y)) | ((unsigned)float2_to_fp8x2(slope_of(a.x, b.x), slope_of(a.y, b.y)) << 16);
}
__device__ __forceinline__ void make_entry(Fp8x2& e, float a, float b) { e.v = float2_to_fp8x2(mid_of(a, b), slope_of(a, b)); }
__device__ __forceinline__ void make_entry(float2& e, float a, float b) { e = make_float2(mid_of(a, b), slope_of(a, b)); }
__device__ __forceinline__ void make_entry(unsigned& e, float a, float b) { e = pack_h2(mid_of(a, b), slope_of(a, b)); }

constexpr int kThreads = 256;

template <typename Out, int EPT> struct alignas(EPT * sizeof(Out) >= 16 ? 16 : 8) Quad { Out e[EPT]; };

// In = float2 (IQ) or float (RF); Out = entry type: float4 / uint2 / Fp8x4 (IQ fp32 / fp16 / fp8),
// float2 / unsigned / Fp8x2 (RF); kEntriesPerThread entries (>= 16 bytes) per thread
template <typename In, typename Out, int kEntriesPerThread>
__global__ void __launch_bounds__(kThreads)
convert_kernel(const In* __restrict__ raw, Out* __restrict__ conv, int M, int Q, int K, int Kp,
               float scale) {
  const int chunks = Kp / kEntriesPerThread;                 // Kp is a multiple of 8
  const long long total = (long long)M * Q * chunks;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total;
       i += (long long)gridDim.x * blockDim.x) {
    const int ch = (int)(i % chunks);
    const long long row = i / chunks;                        // output row = m*Q + q
    const int q = (int)(row % Q);
    const int m = (int)(row / Q);
    const In* src = raw + ((long long)q * M + m) * K;
    const int k0 = ch * kEntriesPerThread - kPadLeft;        // first sample interval of this thread
    In y[kEntriesPerThread + 1];
#pragma unroll
    for (int j = 0; j <= kEntriesPerThread; ++j) {
      const int k = k0 + j;
      if (k >= 0 && k < K) y[j] = scaled(ldg_stream(src + k), scale); else zero(y[j]);
    }
    Quad<Out, kEntriesPerThread> out;
    In z;
    zero(z);
#pragma unroll
    for (int j = 0; j < kEntriesPerThread; ++j) {
      const int k = k0 + j;
      const bool ok = (k >= 0) && (k <= K - 2);              // both samples of the interval exist
      make_entry(out.e[j], ok ? y[j] : z, ok ? y[j + 1] : z);
    }
    *reinterpret_cast<Quad<Out, kEntriesPerThread>*>(conv + row * Kp + (long long)ch * kEntriesPerThread) = out;
  }
}

}  // namespace

cudaError_t launch_convert(const Params& P, const void* d_raw, void* d_conv, float scale,
                           cudaStream_t s) {
  const int ept = (!P.iq && P.fp8) ? 8 : 4;                  // RF fp8 entries are 2 bytes: 8 of them make 16
  const long long total = (long long)P.M * P.Q * (P.Kp / ept);
  long long blocks = (total + kThreads - 1) / kThreads;
  const long long cap = 148LL * 8 * 16;                     // grid-stride beyond 16 waves
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  dim3 grid((unsigned)blocks), block(kThreads);
  if (P.iq) {
    if (P.fp8)       convert_kernel<float2, Fp8x4, 4><<<grid, block, 0, s>>>((const float2*)d_raw, (Fp8x4*)d_conv, P.M, P.Q, P.K, P.Kp, scale);
    else if (P.fp16) convert_kernel<float2, uint2, 4><<<grid, block, 0, s>>>((const float2*)d_raw, (uint2*)d_conv, P.M, P.Q, P.K, P.Kp, scale);
    else             convert_kernel<float2, float4, 4><<<grid, block, 0, s>>>((const float2*)d_raw, (float4*)d_conv, P.M, P.Q, P.K, P.Kp, scale);
  } else {
    if (P.fp8)       convert_kernel<float, Fp8x2, 8><<<grid, block, 0, s>>>((const float*)d_raw, (Fp8x2*)d_conv, P.M, P.Q, P.K, P.Kp, scale);
    else if (P.fp16) convert_kernel<float, unsigned, 4><<<grid, block, 0, s>>>((const float*)d_raw, (unsigned*)d_conv, P.M, P.Q, P.K, P.Kp, scale);
    else             convert_kernel<float, float2, 4><<<grid, block, 0, s>>>((const float*)d_raw, (float2*)d_conv, P.M, P.Q, P.K, P.Kp, scale);
  }
  count_launch();
  return cudaGetLastError();
}

}  // namespace das
