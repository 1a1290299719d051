// Internal definitions shared by the translation units of libdas_b200.so.
// Nothing here is part of the C ABI (include/das.h) and nothing here is shared with oracle/.
#pragma once

#include <cuda_fp16.h>
#include <cuda_fp8.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "das.h"

namespace das {

// Device layout of the converted channel data (das_convert output), chosen by this build
// ("gather-friendly layout", BASELINE.json north_star; the paper's own [K][Q][M][B] batch-inner
// layout, needs a frame batch and does not apply to one frame per call):
//
//   conv[m][q][i], i in [0, Kp), entry i describes the sample interval k = i - kPadLeft:
//     mid_k   = (y_k + y_k+1) / 2          slope_k = y_k+1 - y_k          for 0 <= k <= K-2
//     (0, 0)                                                             otherwise
//   so that linear interpolation at t = k + a is ONE fused multiply-add per
//   component and ONE aligned load:  y[t] = mid_k + (a - 1/2) slope_k,  and samples outside
//   [0, K-2] (dropped terms) read as zero without a bounds test.
//   Kp = kPadLeft + round_up(K, 8) + kPadRight; both pads are at least the largest staged window.
//
// Entry type (mid, slope) in storage precision:
//   IQ fp32: float4 (mid.re, mid.im, slope.re, slope.im)   16 B
//   IQ fp16: 2 x __half2 (mid.re, mid.im | slope.re, slope.im) 8 B
//   RF fp32: float2 (mid, slope) 8 B            RF fp16: __half2 (mid, slope) 4 B
//   IQ fp8 : 4 x e4m3 (mid.re, mid.im, slope.re, slope.im) 4 B      RF fp8: 2 x e4m3 (mid, slope) 2 B
// Element-major so that the Q rows one receiver contributes to a voxel tile sit side by side;
// every row starts 16-byte aligned (Kp is a multiple of 8) for TMA bulk copies.
struct Fp8x4 { unsigned v; };            // IQ fp8 entry
struct Fp8x2 { unsigned short v; };      // RF fp8 entry
// e4m3 pair -> two floats (hardware conversion through half precision, exact)
__device__ __forceinline__ float2 fp8x2_to_float2(unsigned short v) {
  const __half2_raw h = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)v, __NV_E4M3);
  return __half22float2(*reinterpret_cast<const __half2*>(&h));
}
__device__ __forceinline__ unsigned short float2_to_fp8x2(float lo, float hi) {
  return (unsigned short)__nv_cvt_float2_to_fp8x2(make_float2(lo, hi), __NV_SATFINITE, __NV_E4M3);
}
// storage code of a plan: 0 fp32, 1 fp16, 2 fp8
__host__ __device__ inline int storage_code(int fp16, int fp8) { return fp8 ? 2 : (fp16 ? 1 : 0); }
constexpr int kPadLeft = 64;
constexpr int kPadRight = 64;
__host__ __device__ inline int padded_samples(int K) { return kPadLeft + ((K + 7) / 8) * 8 + kPadRight; }

struct TxDev {        // one transmit, device copy (double: the transmit delay is common to all
  int type;           // elements of a voxel, so its rounding error adds coherently)
  int pad;
  double vx, vy, vz;
  double t0;
};

struct Params {
  int M, Q, K, Kp;
  int nx, ny, nz;
  int iq;               // 1 = IQ (complex), 0 = RF
  int fp16;             // 1 = fp16 storage
  int fp8;              // 1 = fp8 (e4m3) storage
  int apod;             // 1 = f-number boxcar active
  int has_dir;          // 1 = per-element normals given
  const float* xs;      // device copies of the axis vectors
  const float* ys;
  const float* zs;
  const float4* elem;   // [M] (x, y, z, 0)
  const float4* edir;   // [M] (nx, ny, nz, 0) or nullptr
  const TxDev* tx;      // [Q]
  double c, fc, fs, t_start, fnum;
  // the paper's general interface (include/das.h); nullptr / 0 = off
  const float* tau_tab;       // [Q][N] transmit delays in seconds
  const float* wtx_tab;       // [Q][N] transmit weights with the observation lists folded in: 0 for a transmit a
                              // voxel does not list (such terms are skipped, not multiplied)
  const float4* vox;          // [N] voxel list (x, y, z, 0)
  int window;                 // das_window_t
  int interp;                 // das_interp_t
  float taper;                // Tukey taper fraction
};

// Transmit delay of (q, voxel n at (x, y, z)) in seconds, FP64: the table when the plan has one, else the
// delay model of the transmit (fn. 2, readings A1 / A2).
__device__ __forceinline__ double tx_tau(const Params& P, int q, long long n, double x, double y, double z) {
  if (P.tau_tab) return (double)__ldg(&P.tau_tab[(long long)q * ((long long)P.nx * P.ny * P.nz) + n]);
  const TxDev tx = P.tx[q];
  if (tx.type == DAS_TX_PLANE) return (x * tx.vx + y * tx.vy + z * tx.vz) / P.c + tx.t0;
  const double bx = x - tx.vx, by = y - tx.vy, bz = z - tx.vz;
  return sqrt(bx * bx + by * by + bz * bz) / P.c + tx.t0;
}
__device__ __forceinline__ float tx_weight(const Params& P, int q, long long n) {
  return P.wtx_tab ? __ldg(&P.wtx_tab[(long long)q * ((long long)P.nx * P.ny * P.nz) + n]) : 1.f;
}
// Receive window on the f-number cone as a function of u^2 = 4 f#^2 rho^2 / a^2 (u in [0, 1] inside the cone)
__device__ __forceinline__ float rx_window(int window, float taper, float u2) {
  if (window == DAS_WINDOW_BOXCAR) return 1.f;
  const float u = sqrtf(fminf(fmaxf(u2, 0.f), 1.f));
  if (window == DAS_WINDOW_HANN) return 0.5f + 0.5f * cospif(u);
  return u <= 1.f - taper ? 1.f : 0.5f + 0.5f * cospif((u - 1.f + taper) / taper);
}

// ---- kernels' host-side launchers (each returns the cudaError_t of its launch) -------------
cudaError_t launch_convert(const Params& P, const void* d_raw, void* d_conv, float scale,
                           cudaStream_t s);
cudaError_t launch_general(const Params& P, const void* d_conv, void* d_out, cudaStream_t s);
cudaError_t launch_count(const Params& P, unsigned long long* d_counters, cudaStream_t s);

struct TiledPlan;      // opaque to the API layer (das_tiled.cu)
// Returns nullptr and fills why[] if the geometry does not qualify for the tiled kernel.
TiledPlan* tiled_plan_create(const Params& P, const das_plan_desc_t& desc, int device,
                             char* why, size_t why_len, cudaError_t* cuda_err);
void tiled_plan_destroy(TiledPlan* tp);
cudaError_t launch_tiled(const TiledPlan* tp, const Params& P, const void* d_conv, void* d_out,
                         cudaStream_t s, int* n_launches);

void count_launch(unsigned long long n = 1);

// das_api.cu, for das_static.cu: the plan's device ordinal and the thread-local das_last_error() text
int plan_device(const das_plan* p);
void set_error_text(const char* msg);

}  // namespace das
