// Internal definitions shared by the translation units of libdas_b200.so.
// Nothing here is part of the C ABI (include/das.h) and nothing here is shared with oracle/.
#pragma once

#include <cuda_fp16.h>
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
// Element-major so that the Q rows one receiver contributes to a voxel tile sit side by side;
// every row starts 16-byte aligned (Kp is a multiple of 8) for TMA bulk copies.
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
  int apod;             // 1 = f-number boxcar active
  int has_dir;          // 1 = per-element normals given
  const float* xs;      // device copies of the axis vectors
  const float* ys;
  const float* zs;
  const float4* elem;   // [M] (x, y, z, 0)
  const float4* edir;   // [M] (nx, ny, nz, 0) or nullptr
  const TxDev* tx;      // [Q]
  double c, fc, fs, t_start, fnum;
};

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

}  // namespace das
