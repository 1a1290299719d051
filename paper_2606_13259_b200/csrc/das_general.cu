// General delay-and-sum kernel: one thread per voxel, any receiver positions and normals.
//
// This is the computation of the paper's Algorithm 1 with B = 1, except that
// the transmit delay is also computed in-kernel (BASELINE.json north_star) and the loops are
// swapped (receiver outer, transmit inner, in chunks of kQc transmits) so that the receive
// geometry is evaluated once per (m, n) instead of once per (q, m, n).  It is the fallback for
// geometries the tiled kernel does not take (non-planar arrays, tilted normals) and the
// reference point the tiled kernel is measured against; it is not the fast path.
//
// The channel data is read from the (mid, slope) table layout das_convert writes
// (das_internal.cuh): one aligned load per term.
//
// Precision: all geometry (delays, aperture test, sample coordinate, phase in cycles) is FP64,
// which B200 runs at half the FP32 rate; only the interpolation, rotation and accumulation are
// FP32.  The aperture test repeats the defining expression
// 4 f#^2 rho^2 <= a^2 with separately rounded FP64 operations so that a voxel/element pair on
// the edge of the cone is classified exactly as the definition does ("aperture edge").
#include "das_internal.cuh"

namespace das {

namespace {

constexpr int kQc = 8;          // transmits per pass: 8 complex FP32 accumulators + 8 FP64 tau_tx
constexpr int kThreads = 128;

// One (mid, slope) table entry of the device layout (das_internal.cuh), widened to FP32.
struct EntryF { float mid_re, mid_im, slope_re, slope_im; };
template <typename T> struct Sample;
template <> struct Sample<float4> {       // IQ fp32
  static __device__ __forceinline__ EntryF load(const float4* p) { const float4 v = __ldg(p); return {v.x, v.y, v.z, v.w}; }
};
template <> struct Sample<uint2> {        // IQ fp16: (half2 mid, half2 slope)
  static __device__ __forceinline__ EntryF load(const uint2* p) {
    const uint2 u = __ldg(p);
    const float2 m = __half22float2(*reinterpret_cast<const __half2*>(&u.x));
    const float2 s = __half22float2(*reinterpret_cast<const __half2*>(&u.y));
    return {m.x, m.y, s.x, s.y};
  }
};
template <> struct Sample<float2> {       // RF fp32
  static __device__ __forceinline__ EntryF load(const float2* p) { const float2 v = __ldg(p); return {v.x, 0.f, v.y, 0.f}; }
};
template <> struct Sample<unsigned> {     // RF fp16: half2 (mid, slope)
  static __device__ __forceinline__ EntryF load(const unsigned* p) {
    const unsigned u = __ldg(p);
    const float2 v = __half22float2(*reinterpret_cast<const __half2*>(&u));
    return {v.x, 0.f, v.y, 0.f};
  }
};

template <> struct Sample<Fp8x4> {        // IQ fp8: 4 x e4m3 (mid.re, mid.im, slope.re, slope.im)
  static __device__ __forceinline__ EntryF load(const Fp8x4* p) {
    const unsigned u = __ldg(reinterpret_cast<const unsigned*>(p));
    const float2 m = fp8x2_to_float2((unsigned short)(u & 0xffffu)), s = fp8x2_to_float2((unsigned short)(u >> 16));
    return {m.x, m.y, s.x, s.y};
  }
};
template <> struct Sample<Fp8x2> {        // RF fp8: 2 x e4m3 (mid, slope)
  static __device__ __forceinline__ EntryF load(const Fp8x2* p) {
    const float2 v = fp8x2_to_float2(__ldg(reinterpret_cast<const unsigned short*>(p)));
    return {v.x, 0.f, v.y, 0.f};
  }
};

template <bool IQ, typename T>
__global__ void __launch_bounds__(kThreads)
general_kernel(const Params P, const T* __restrict__ conv, void* __restrict__ out_v) {
  const long long N = (long long)P.nx * P.ny * P.nz;
  const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= N) return;
  const int iz = (int)(n % P.nz);
  const int iy = (int)((n / P.nz) % P.ny);
  const int ix = (int)(n / ((long long)P.nz * P.ny));
  double px, py, pz;
  if (P.vox) { const float4 v = __ldg(&P.vox[n]); px = (double)v.x; py = (double)v.y; pz = (double)v.z; }
  else { px = (double)P.xs[ix]; py = (double)P.ys[iy]; pz = (double)P.zs[iz]; }
  const double inv_c = 1.0 / P.c;
  const bool cubic = P.interp == DAS_INTERP_CUBIC;
  const double lim_lo = cubic ? 1.0 : 0.0, lim_hi = (double)(P.K - (cubic ? 3 : 2));
  // 4 f#^2, rounded as ((4 f#) f#), the order the definition is evaluated in
  const double four_f2 = __dmul_rn(__dmul_rn(4.0, P.fnum), P.fnum);

  float tot_re = 0.f, tot_im = 0.f;
  for (int q0 = 0; q0 < P.Q; q0 += kQc) {
    double tau_tx[kQc];
    float acc_re[kQc], acc_im[kQc], wq[kQc];
#pragma unroll
    for (int j = 0; j < kQc; ++j) {
      acc_re[j] = 0.f; acc_im[j] = 0.f;
      const int q = min(q0 + j, P.Q - 1);
      tau_tx[j] = tx_tau(P, q, n, px, py, pz);
      wq[j] = tx_weight(P, q, n);                 // 0: the voxel does not list this transmit
    }
    for (int m = 0; m < P.M; ++m) {
      const float4 e = __ldg(&P.elem[m]);
      const double dx = px - (double)e.x, dy = py - (double)e.y, dz = pz - (double)e.z;
      const double dx2 = __dmul_rn(dx, dx), dy2 = __dmul_rn(dy, dy), dz2 = __dmul_rn(dz, dz);
      const double dd = __dadd_rn(__dadd_rn(dx2, dy2), dz2);
      float w_rx = 1.f;
      if (P.apod) {
        double a, rho2;
        if (P.has_dir) {
          const float4 d = __ldg(&P.edir[m]);
          a = __dadd_rn(__dadd_rn(__dmul_rn(dx, (double)d.x), __dmul_rn(dy, (double)d.y)),
                        __dmul_rn(dz, (double)d.z));
          rho2 = __dadd_rn(dd, -__dmul_rn(a, a));
        } else {
          a = dz;
          rho2 = __dadd_rn(dx2, dy2);
        }
        const double lhs = __dmul_rn(four_f2, rho2), rhs = __dmul_rn(a, a);
        if (!(a > 0.0 && lhs <= rhs)) continue;
        if (P.window != DAS_WINDOW_BOXCAR) w_rx = rx_window(P.window, P.taper, (float)(lhs / rhs));
      }
      const double tau_rx = sqrt(dd) * inv_c;
      const T* rowm = conv + (long long)m * P.Q * P.Kp;
#pragma unroll
      for (int j = 0; j < kQc; ++j) {
        if (q0 + j >= P.Q) break;
        if (wq[j] == 0.f) continue;
        const double tau = tau_tx[j] + tau_rx;
        const double t = (tau - P.t_start) * P.fs;
        const double kf = floor(t);
        if (!(kf >= lim_lo && kf <= lim_hi)) continue;
        const float wg = wq[j] * w_rx;
        const T* ent = rowm + (long long)(q0 + j) * P.Kp + (kPadLeft + (int)kf);
        float s_re, s_im = 0.f;
        if (cubic) {
          // cubic convolution (Keys, a = -1/2) on y[k-1..k+2], rebuilt from the entries k-1 and k+1:
          // y_k = mid_k - slope_k / 2, y_k+1 = mid_k + slope_k / 2
          const float al = (float)(t - kf), a2 = al * al, a3 = a2 * al;
          const float c0 = -0.5f * a3 + a2 - 0.5f * al, c1 = 1.5f * a3 - 2.5f * a2 + 1.f;
          const float c2 = -1.5f * a3 + 2.f * a2 + 0.5f * al, c3 = 0.5f * a3 - 0.5f * a2;
          const EntryF lo = Sample<T>::load(ent - 1), hi = Sample<T>::load(ent + 1);
          s_re = c0 * fmaf(-0.5f, lo.slope_re, lo.mid_re) + c1 * fmaf(0.5f, lo.slope_re, lo.mid_re) +
                 c2 * fmaf(-0.5f, hi.slope_re, hi.mid_re) + c3 * fmaf(0.5f, hi.slope_re, hi.mid_re);
          if (IQ)
            s_im = c0 * fmaf(-0.5f, lo.slope_im, lo.mid_im) + c1 * fmaf(0.5f, lo.slope_im, lo.mid_im) +
                   c2 * fmaf(-0.5f, hi.slope_im, hi.mid_im) + c3 * fmaf(0.5f, hi.slope_im, hi.mid_im);
        } else {
          const float ah = (float)(t - kf) - 0.5f;             // y[t] = mid_k + (alpha - 1/2) slope_k
          const EntryF en = Sample<T>::load(ent);
          s_re = fmaf(ah, en.slope_re, en.mid_re);
          if (IQ) s_im = fmaf(ah, en.slope_im, en.mid_im);
        }
        s_re *= wg;
        if (IQ) {
          s_im *= wg;
          double cyc = P.fc * tau;
          cyc -= rint(cyc);                        // phase in cycles, reduced to [-1/2, 1/2] in FP64
          float sn, cs;
          sincospif(2.0f * (float)cyc, &sn, &cs);
          acc_re[j] = fmaf(s_re, cs, fmaf(-s_im, sn, acc_re[j]));
          acc_im[j] = fmaf(s_re, sn, fmaf(s_im, cs, acc_im[j]));
        } else {
          acc_re[j] += s_re;
        }
      }
    }
#pragma unroll
    for (int j = 0; j < kQc; ++j) { tot_re += acc_re[j]; tot_im += acc_im[j]; }
  }
  if (IQ) reinterpret_cast<float2*>(out_v)[n] = make_float2(tot_re, tot_im);
  else    reinterpret_cast<float*>(out_v)[n] = tot_re;
}

// Work counter (accounting for the bench's roofline, not part of the hot path): the number of
// (m, n) pairs with non-zero receive weight and the number of (q, m, n) terms that enter the sum
// (non-zero weight and 0 <= k <= K-2), classified by exactly the FP64 expressions of the general
// kernel above.  One thread per voxel, warp-shuffle + one atomicAdd per warp.
__global__ void __launch_bounds__(kThreads)
count_kernel(const Params P, unsigned long long* __restrict__ counters) {
  const long long N = (long long)P.nx * P.ny * P.nz;
  const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long pairs = 0, terms = 0;
  if (n < N) {
    const int iz = (int)(n % P.nz);
    const int iy = (int)((n / P.nz) % P.ny);
    const int ix = (int)(n / ((long long)P.nz * P.ny));
    double px, py, pz;
    if (P.vox) { const float4 v = __ldg(&P.vox[n]); px = (double)v.x; py = (double)v.y; pz = (double)v.z; }
    else { px = (double)P.xs[ix]; py = (double)P.ys[iy]; pz = (double)P.zs[iz]; }
    const double inv_c = 1.0 / P.c;
    const bool cubic = P.interp == DAS_INTERP_CUBIC;
    const double lim_lo = cubic ? 1.0 : 0.0, lim_hi = (double)(P.K - (cubic ? 3 : 2));
    const double four_f2 = __dmul_rn(__dmul_rn(4.0, P.fnum), P.fnum);
    for (int m = 0; m < P.M; ++m) {
      const float4 e = __ldg(&P.elem[m]);
      const double dx = px - (double)e.x, dy = py - (double)e.y, dz = pz - (double)e.z;
      const double dx2 = __dmul_rn(dx, dx), dy2 = __dmul_rn(dy, dy), dz2 = __dmul_rn(dz, dz);
      const double dd = __dadd_rn(__dadd_rn(dx2, dy2), dz2);
      if (P.apod) {
        double a, rho2;
        if (P.has_dir) {
          const float4 d = __ldg(&P.edir[m]);
          a = __dadd_rn(__dadd_rn(__dmul_rn(dx, (double)d.x), __dmul_rn(dy, (double)d.y)),
                        __dmul_rn(dz, (double)d.z));
          rho2 = __dadd_rn(dd, -__dmul_rn(a, a));
        } else {
          a = dz;
          rho2 = __dadd_rn(dx2, dy2);
        }
        if (!(a > 0.0 && __dmul_rn(four_f2, rho2) <= __dmul_rn(a, a))) continue;
      }
      ++pairs;
      const double tau_rx = sqrt(dd) * inv_c;
      for (int q = 0; q < P.Q; ++q) {
        if (tx_weight(P, q, n) == 0.f) continue;                // not on the voxel's observation list
        const double kf = floor((tx_tau(P, q, n, px, py, pz) + tau_rx - P.t_start) * P.fs);
        if (kf >= lim_lo && kf <= lim_hi) ++terms;
      }
    }
  }
  for (int o = 16; o > 0; o >>= 1) {
    pairs += __shfl_down_sync(0xffffffffu, pairs, o);
    terms += __shfl_down_sync(0xffffffffu, terms, o);
  }
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(&counters[0], pairs);
    atomicAdd(&counters[1], terms);
  }
}

}  // namespace

cudaError_t launch_count(const Params& P, unsigned long long* d_counters, cudaStream_t s) {
  const long long N = (long long)P.nx * P.ny * P.nz;
  const unsigned blocks = (unsigned)((N + kThreads - 1) / kThreads);
  count_kernel<<<blocks, kThreads, 0, s>>>(P, d_counters);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_general(const Params& P, const void* d_conv, void* d_out, cudaStream_t s) {
  const long long N = (long long)P.nx * P.ny * P.nz;
  const unsigned blocks = (unsigned)((N + kThreads - 1) / kThreads);
  if (P.iq) {
    if (P.fp8)       general_kernel<true, Fp8x4><<<blocks, kThreads, 0, s>>>(P, (const Fp8x4*)d_conv, d_out);
    else if (P.fp16) general_kernel<true, uint2><<<blocks, kThreads, 0, s>>>(P, (const uint2*)d_conv, d_out);
    else             general_kernel<true, float4><<<blocks, kThreads, 0, s>>>(P, (const float4*)d_conv, d_out);
  } else {
    if (P.fp8)       general_kernel<false, Fp8x2><<<blocks, kThreads, 0, s>>>(P, (const Fp8x2*)d_conv, d_out);
    else if (P.fp16) general_kernel<false, unsigned><<<blocks, kThreads, 0, s>>>(P, (const unsigned*)d_conv, d_out);
    else             general_kernel<false, float2><<<blocks, kThreads, 0, s>>>(P, (const float2*)d_conv, d_out);
  }
  count_launch();
  return cudaGetLastError();
}

}  // namespace das
