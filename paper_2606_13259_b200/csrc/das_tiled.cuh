// Tiled delay-and-sum kernel for planar arrays (all receivers in one plane z = z_a, normals +z,
// every voxel in front of that plane) -- the fast path of das_execute.
//
// Decomposition:
//   t_qmn = T_q(n) + e_m(n)                               [samples]
//     T_q(n) = (tau_tx(q,n) + a_n/c - t_start) fs          a_n = z_n - z_a   per (q, n), FP64
//     e_m(n) = (|p_n - r_m| - a_n) fs/c
//            = rho^2 (fs/c) / (a_n + sqrt(rho^2 + a_n^2))                    per (m, n), FP32
//   phase    exp(j 2 pi fc tau) = Ptx_q(n) * Prx_m(n),
//     Ptx = exp(j 2 pi (fc t_start + (fc/fs) T_q)),  Prx = exp(j 2 pi (fc/fs) e_m)
//   x_n = sum_q Ptx_q(n) * [ sum_m w_mn Prx_m(n) y_qm[t_qmn] ]
// The part common to all receivers of a voxel (whose rounding error would add coherently) is
// FP64 and amortised over M; the per-receiver excess path e_m is small (<= ~0.12 a fs/c inside
// an f/1 cone), so FP32 keeps ~1e-6 samples on it.
//
// Work split inside a CTA (one CTA = one voxel tile at a time, persistent over a static,
// work-sorted tile list); three warp roles connected by two mbarrier rings:
//   * ONE producer warp walks the tile's active-receiver list (built by the plan).  For each
//     receiver m it issues, per transmit q, one TMA bulk copy (cp.async.bulk global -> shared,
//     completion counted on an mbarrier) of the W table entries [k0, k0 + W),
//     k0 = K0tile_q + E0_m, of row (m, q) of the converted channel data (storage precision,
//     (mid, slope) pairs, zeros outside the valid sample range: das_internal.cuh) into the RAW
//     ring.
//   * CONVERTER warps turn one raw stage into one stage of the TABLE ring: FP32 line
//     coefficients in window-local coordinates, entry i = (c_i, slope_i) with
//     c_i = mid_i - i * slope_i, so that the interpolated sample at local position ts
//     (already shifted by -1/2) is  y = c_i + ts * slope_i : ONE fused multiply-add per
//     component with the position itself as the multiplier (no fraction to extract), FP32
//     whatever the storage precision ("converted to FP32 before interpolation").
//     This costs 4 conversions per staged entry instead of 2 per accumulated term.
//   * consumer threads own one voxel each (a warp = 8 x 4 lateral voxels at one depth, so all
//     lanes read nearly the same shared-memory words: broadcast), keep QC complex accumulators
//     and QC reduced transmit delays in registers, and run the (m outer, q inner) loop:
//       ts = Tf_q + e'     u = ts + MAGIC (its low mantissa bits are the rounded entry index)
//       (c, slope) = table[bits(u)]     s = c + ts * slope     acc_q += Prx * s
// Helper warps give most of their registers to the consumers (setmaxnreg).
#pragma once

#include "das_internal.cuh"

namespace das {

constexpr int kRawStages = 6;                   // ring of TMA-staged windows (storage precision)
constexpr int kTabStages = 6;                   // ring of FP32 line tables the consumers read
constexpr int kConvWarps = 3;
constexpr int kHelperWarps = 4;                 // one warpgroup: producer + converters (+ idle)
constexpr int kLaneX = 8, kLaneY = 4;          // a consumer warp covers 8 x 4 lateral voxels
constexpr int kWX = 1, kWY = 2, kWZ = 4;       // consumer warps per tile: tile = 8 x 8 x 4 voxels
constexpr int kConsumerWarps = kWX * kWY * kWZ;
constexpr int kConsumerThreads = kConsumerWarps * 32;
constexpr int kTiledThreads = (kConsumerWarps + kHelperWarps) * 32;
constexpr int kRegsConsumer = 104, kRegsHelper = 32;   // 256 * 104 + 128 * 32 <= 384 * 80
constexpr float kMagic = 12582912.0f;           // 1.5 * 2^23: adding it rounds to an integer
constexpr unsigned kMagicBits = 0x4B400000u;
constexpr float kBand = 4e-6f;                  // relative guard band of the FP32 aperture test
static_assert(kConsumerWarps % 4 == 0 && kHelperWarps == 4 && kConvWarps + 1 <= kHelperWarps, "warpgroup roles");
// The converter warps take the stages in turn.  Both rings must be a multiple of their number deep, so that a slot is
// always served by the SAME warp: an mbarrier parity wait cannot tell "round r + 1 complete" from "round r - 1
// complete", and the bulk copies of different stages complete in any order.  With 3 converters and 4 slots a warp
// could reach a slot whose previous round (another warp's) was still in flight, fall through the wait, convert a
// stale window and deadlock the rings (about one launch in fifty of the RF fp32 headline; fixed in round 2).
static_assert(kRawStages % kConvWarps == 0 && kTabStages % kConvWarps == 0, "a slot belongs to one converter warp");

enum Mode { kIQ32 = 0, kIQ16 = 1, kRF32 = 2, kRF16 = 3, kIQ8 = 4, kRF8 = 5 };
template <int MODE> struct ModeTraits;   // eb: bytes of a stored (mid, slope) entry; tb: of a table entry
template <> struct ModeTraits<kIQ32> { static constexpr bool iq = true;  static constexpr int eb = 16, tb = 16; };
template <> struct ModeTraits<kIQ16> { static constexpr bool iq = true;  static constexpr int eb = 8,  tb = 16; };
template <> struct ModeTraits<kRF32> { static constexpr bool iq = false; static constexpr int eb = 8,  tb = 8; };
template <> struct ModeTraits<kRF16> { static constexpr bool iq = false; static constexpr int eb = 4,  tb = 8; };
template <> struct ModeTraits<kIQ8>  { static constexpr bool iq = true;  static constexpr int eb = 4,  tb = 16; };
template <> struct ModeTraits<kRF8>  { static constexpr bool iq = false; static constexpr int eb = 2,  tb = 8; };
// bytes of a stored (mid, slope) entry; st = storage code (0 fp32, 1 fp16, 2 fp8)
__host__ __device__ inline int entry_bytes(int iq, int st) { return (iq ? 2 : 1) * 2 * (st == 0 ? 4 : (st == 1 ? 2 : 1)); }

struct TileDesc {       // one voxel tile
  int ix0, iy0, iz0;    // origin (voxel indices)
  int list_off;         // offset into the receiver list
  int list_cnt;         // number of (potentially) active receivers
};

struct TiledDev {
  int n_tiles;
  int n_chunks;               // ceil(Q / QC)
  const TileDesc* tiles;      // [n_tiles], sorted by decreasing work
  const int* k0tile;          // [n_tiles][Q]   window origin per transmit (multiple of 16/eb)
  const unsigned* list;       // receiver lists: m | (E0 << 16), E0 a multiple of 16/eb
  double z_array;             // z_a
  double kappa;               // fs / c
  double ratio;               // fc / fs
  double phase0;              // frac(fc * t_start), cycles
  float four_f2;              // 4 f#^2
  float kappa_f, ratio_f;     // float copies (no F2F conversions in the receiver loop)
  unsigned addr_bias;         // -(bits(MAGIC) << log2(table entry bytes)) mod 2^32: a kernel PARAMETER so
                              // that ptxas cannot split (bits(u) << s) + base into LEA + IADD
};

// ---- PTX helpers ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) {
  return static_cast<unsigned>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
// TMA bulk copy global -> this CTA's shared memory, completion (bytes) counted on an mbarrier
__device__ __forceinline__ void tma_bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
template <int OFF> __device__ __forceinline__ float4 lds128(unsigned addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4+%5];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr), "n"(OFF));
  return v;
}
template <int OFF> __device__ __forceinline__ float2 lds64f(unsigned addr) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0,%1}, [%2+%3];" : "=f"(v.x), "=f"(v.y) : "r"(addr), "n"(OFF));
  return v;
}
__device__ __forceinline__ uint2 lds64u(unsigned addr) {
  uint2 v;
  asm volatile("ld.shared.v2.b32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ unsigned short lds16u(unsigned addr) {
  unsigned short v;
  asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ unsigned lds32u(unsigned addr) {
  unsigned v;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts128(unsigned addr, float4 v) {
  asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void sts64(unsigned addr, float2 v) {
  asm volatile("st.shared.v2.f32 [%0], {%1,%2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
__device__ __forceinline__ float pin(float v) { return __shfl_sync(0xffffffffu, v, threadIdx.x & 31); }
__device__ __forceinline__ float rsqrt_approx(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rcp_approx(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sin_approx(float x) { float r; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float cos_approx(float x) { float r; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

template <int QC, int W, int MODE>
struct alignas(128) TiledSmem {
  unsigned char tab[kTabStages][QC * W * ModeTraits<MODE>::tb];
  unsigned char raw[kRawStages][QC * W * ModeTraits<MODE>::eb];
  float cyc[ModeTraits<MODE>::iq ? QC : 1][kConsumerThreads];   // transmit phase (cycles) per (q, voxel)
  float4 meta_raw[kRawStages];          // (ex, ey, E0, -) of the staged receiver
  float4 meta_tab[kTabStages];          // (ex, ey, E0, MAGIC + first entry of the stage)
  float4 dir_raw[kRawStages];           // its normal (plans with elem_dir only)
  float4 dir_tab[kTabStages];
  unsigned long long raw_full[kRawStages], raw_empty[kRawStages];
  unsigned long long tab_full[kTabStages], tab_empty[kTabStages];
};

// upper bound of sizeof(TiledSmem<QC, W, MODE>) for the plan's occupancy estimate
__host__ __device__ inline size_t tiled_smem_bytes(int QC, int W, int iq, int st) {
  const size_t tb = iq ? 16 : 8, eb = (size_t)entry_bytes(iq, st);
  return (size_t)QC * W * (kTabStages * tb + kRawStages * eb) + (size_t)(iq ? QC : 1) * kConsumerThreads * 4 + 768;
}

// exact (definition-order, FP64) aperture test for pairs inside the FP32 guard band
static __device__ __noinline__ bool aperture_exact(float x, float y, float ex, float ey, const float* zs, int iz, double z_array, double fnum) {
  const double a = (double)__ldg(&zs[iz]) - z_array;
  const double dx = (double)x - (double)ex, dy = (double)y - (double)ey;
  const double rho2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
  const double four_f2 = __dmul_rn(__dmul_rn(4.0, fnum), fnum);
  return __dmul_rn(four_f2, rho2) <= __dmul_rn(a, a);
}

// the same for a receiver with normal (nx, ny, nz): a = d.n, rho^2 = d.d - a^2, in the expression order of the
// general kernel and of the definition
static __device__ __noinline__ bool aperture_exact_dir(float x, float y, float ex, float ey, const float* zs, int iz, double z_array,
                                                       double fnum, float nx, float ny, float nz) {
  const double dz = (double)__ldg(&zs[iz]) - z_array;
  const double dx = (double)x - (double)ex, dy = (double)y - (double)ey;
  const double dd = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
  const double a = __dadd_rn(__dadd_rn(__dmul_rn(dx, (double)nx), __dmul_rn(dy, (double)ny)), __dmul_rn(dz, (double)nz));
  const double rho2 = __dadd_rn(dd, -__dmul_rn(a, a));
  const double four_f2 = __dmul_rn(__dmul_rn(4.0, fnum), fnum);
  return a > 0.0 && __dmul_rn(four_f2, rho2) <= __dmul_rn(a, a);
}
// FP32 aperture test for a tilted normal with the exact test inside a guard band; u2 = 4 f#^2 rho^2 / a^2.
// dx, dy: lateral offsets, az: depth above the array plane, rho2 = dx^2 + dy^2, a2 = az^2.
__device__ __forceinline__ bool aperture_dir(float x, float y, float ex, float ey, float dx, float dy, float az, float rho2, float a2,
                                             float4 dir, float four_f2, bool in_grid, const float* zs, int iz, double z_array,
                                             double fnum, float& u2) {
  const float an = fmaf(dx, dir.x, fmaf(dy, dir.y, az * dir.z));
  const float dd = rho2 + a2, rhs = an * an;
  const float lhs = four_f2 * (dd - rhs);
  u2 = lhs * rcp_approx(fmaxf(rhs, 1e-30f));
  bool act = in_grid && an > 0.f && lhs <= rhs;
  // the cancellation in dd - an^2 and the sign test of an: both errors are a few ulp of dd
  if (in_grid && (fabsf(lhs - rhs) <= 16.f * kBand * (four_f2 + 1.f) * dd || fabsf(an) <= 1e-5f * sqrtf(dd)))
    act = aperture_exact_dir(x, y, ex, ey, zs, iz, z_array, fnum, dir.x, dir.y, dir.z);
  return act;
}

__device__ __forceinline__ double tx_delay(const TxDev& tx, double x, double y, double z, double c) {
  if (tx.type == DAS_TX_PLANE) return (x * tx.vx + y * tx.vy + z * tx.vz) / c + tx.t0;
  const double bx = x - tx.vx, by = y - tx.vy, bz = z - tx.vz;
  return sqrt(bx * bx + by * by + bz * bz) / c + tx.t0;
}

// Per-(receiver, voxel) geometry carried from one receiver-loop iteration to the next.
struct Geo {
  float u2;         // 4 f#^2 rho^2 / a^2: squared normalised radius inside the f-number cone (receive window)
  float rho2;       // lateral distance^2
  float ep;         // excess path e - E0 [samples]
  float mg;         // MAGIC + first table entry of the stage
  float e0;         // E0 of the staged receiver
  float pr, pi;     // receive phase factor (IQ); (1, 0) for RF
  bool act;
};

// One accumulated term: gather the line of one transmit row at entry address a, interpolate at
// ts, rotate by Prx and add.  IQ: three packed FP32x2 instructions (FFMA2, new on sm_100: one
// issue slot for two lane-FMAs; the scalar operands ts, s.re, s.im are broadcast by the
// instruction itself):   s = c + ts * slope ;  acc += s.re * (pr, pi) ;  acc += s.im * (-pi, pr).
template <int MODE, int OFF>
__device__ __forceinline__ void term(unsigned a, float ts, float2 p1, float2 p2, float2& acc) {
  if constexpr (ModeTraits<MODE>::iq) {
    const float4 v = lds128<OFF>(a);                 // (c.re, c.im, slope.re, slope.im)
    const float2 sv = __ffma2_rn(make_float2(ts, ts), make_float2(v.z, v.w), make_float2(v.x, v.y));
    acc = __ffma2_rn(make_float2(sv.x, sv.x), p1, acc);
    acc = __ffma2_rn(make_float2(sv.y, sv.y), p2, acc);
  } else {
    const float2 v = lds64f<OFF>(a);                 // (c, slope)
    acc.x = fmaf(p1.x, fmaf(ts, v.y, v.x), acc.x);   // p1.x: the receive weight
  }
}

// Part 1: wait for the stage, read its meta entry, classify the aperture (exactly inside the
// guard band).  a2e / band carry "voxel outside the grid" and "no apodization" (see the caller).
template <bool GEN>
__device__ __forceinline__ void geo_test(Geo& g, unsigned tab_full0, unsigned meta0, unsigned slot, unsigned phase,
                                         float x, float y, int iz, float a, float a2, float a2e, float band,
                                         const TiledDev& tp, const Params& P) {
  mbar_wait(tab_full0 + 8 * slot, phase);
  const float4 meta = lds128<0>(meta0 + 16 * slot);      // (ex, ey, E0, MAGIC + stage offset)
  const float dx = x - meta.x, dy = y - meta.y;
  g.rho2 = fmaf(dx, dx, dy * dy);
  g.e0 = meta.z;
  g.mg = meta.w;
  if (GEN && P.has_dir && P.apod) {
    // tilted normal: the delays are those of the planar array, only the cone turns with the normal
    const float4 dir = lds128<0>(meta0 + 16 * (kTabStages + kRawStages + slot));     // dir_tab[slot]
    g.act = aperture_dir(x, y, meta.x, meta.y, dx, dy, a, g.rho2, a2, dir, tp.four_f2, a2e >= 0.f, P.zs, iz, tp.z_array, P.fnum, g.u2);
    return;
  }
  const float lhs = tp.four_f2 * g.rho2;
  if (GEN) g.u2 = lhs * rcp_approx(a2);
  g.act = lhs <= a2e;
  if (fabsf(lhs - a2e) <= band) g.act = aperture_exact(x, y, meta.x, meta.y, P.zs, iz, tp.z_array, P.fnum);
}
// Part 2 (active lanes): excess path and receive phase.
template <bool IQ, bool GEN>
__device__ __forceinline__ void geo_finish(Geo& g, float a, float a2, const TiledDev& tp, const Params& P) {
  const float s2 = g.rho2 + a2;
  const float d = s2 * rsqrt_approx(s2);
  const float e = (g.rho2 * tp.kappa_f) * rcp_approx(a + d);
  g.ep = e - g.e0;
  // receive window (include/das.h): the boxcar leaves the weight at 1
  const float wrx = (GEN && P.window != DAS_WINDOW_BOXCAR && P.apod) ? rx_window(P.window, P.taper, g.u2) : 1.f;
  if (IQ) {
    float cyc = tp.ratio_f * e;
    cyc -= rintf(cyc);
    const float ang = 6.283185307179586f * cyc;
    g.pr = wrx * cos_approx(ang);
    g.pi = wrx * sin_approx(ang);
  } else {
    g.pr = wrx;
    g.pi = 0.f;
  }
}

// GEN: the plan uses a part of the general interface (tilted normals, a smooth receive window, transmit delay / weight
// tables).  The common case (planar normals, boxcar, analytic transmits) is compiled without it: it costs registers
// in the receiver loop (the 16-transmit instance spilled with it).
template <int QC, int W, int MODE, bool GEN>
__global__ void __launch_bounds__(kTiledThreads, 2)
tiled_kernel(const TiledDev tp, const Params P, const unsigned char* __restrict__ conv, void* __restrict__ out_v) {
  constexpr bool IQ = ModeTraits<MODE>::iq;
  constexpr int EB = ModeTraits<MODE>::eb, TB = ModeTraits<MODE>::tb;
  constexpr int TSH = (TB == 16) ? 4 : 3;
  constexpr int NE = QC * W;                         // entries per stage
  constexpr int QP = (QC + 1) / 2;                   // transmit pairs per chunk
  extern __shared__ __align__(128) unsigned char smem_raw[];
  TiledSmem<QC, W, MODE>& sm = *reinterpret_cast<TiledSmem<QC, W, MODE>*>(smem_raw);

  const int tid = threadIdx.x;
  const int warp = tid >> 5, lane = tid & 31;
  const unsigned raw_full0 = smem_u32(&sm.raw_full[0]), raw_empty0 = smem_u32(&sm.raw_empty[0]);
  const unsigned tab_full0 = smem_u32(&sm.tab_full[0]), tab_empty0 = smem_u32(&sm.tab_empty[0]);
  if (tid == 0) {
    for (int s = 0; s < kRawStages; ++s) { mbar_init(raw_full0 + 8 * s, 1); mbar_init(raw_empty0 + 8 * s, 1); }
    for (int s = 0; s < kTabStages; ++s) { mbar_init(tab_full0 + 8 * s, 1); mbar_init(tab_empty0 + 8 * s, kConsumerWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  unsigned seq = 0;          // receiver stages produced / converted / consumed so far by this CTA

  if (warp >= kConsumerWarps) {
    reg_dec<kRegsHelper>();
    const int hw = warp - kConsumerWarps;
    if (hw == 0) {
      // =============================== PRODUCER (TMA) =======================================
      const unsigned raw0 = smem_u32(&sm.raw[0][0]);
      for (int tile_i = blockIdx.x; tile_i < tp.n_tiles; tile_i += gridDim.x) {
        const TileDesc td = tp.tiles[tile_i];
        for (int ch = 0; ch < tp.n_chunks; ++ch) {
          const int q = ch * QC + lane;
          const bool qok = lane < QC && q < P.Q;
          const int k0 = qok ? __ldg(&tp.k0tile[(long long)tile_i * P.Q + q]) : 0;
          const int nq = min(QC, P.Q - ch * QC);
          for (int li = 0; li < td.list_cnt; ++li, ++seq) {
            const unsigned slot = seq % kRawStages;
            const unsigned ent = __ldg(&tp.list[td.list_off + li]);
            const int m = (int)(ent & 0xFFFFu);
            const int e0 = (int)(ent >> 16);
            const float4 el = __ldg(&P.elem[m]);
            mbar_wait(raw_empty0 + 8 * slot, ((seq / kRawStages) & 1u) ^ 1u);
            if (lane == 0) {
              if (GEN && P.has_dir) sm.dir_raw[slot] = __ldg(&P.edir[m]);
              sm.meta_raw[slot] = make_float4(el.x, el.y, (float)e0, 0.f);
              mbar_arrive_expect_tx(raw_full0 + 8 * slot, (unsigned)(nq * W * EB));
            }
            __syncwarp();
            if (qok) {
              int i0 = kPadLeft + k0 + e0;                  // first table entry of the window
              i0 = max(0, min(i0, P.Kp - W));               // clamped windows lie entirely in a zero pad
              const unsigned char* src = conv + (((long long)m * P.Q + q) * P.Kp + i0) * EB;
              tma_bulk_g2s(raw0 + slot * (NE * EB) + lane * (W * EB), src, W * EB, raw_full0 + 8 * slot);
            }
          }
        }
      }
    } else if (hw <= kConvWarps) {
      // =============================== CONVERTERS ===========================================
      const unsigned cw = (unsigned)(hw - 1);
      const unsigned raw0 = smem_u32(&sm.raw[0][0]), tab0 = smem_u32(&sm.tab[0][0]);
      for (int tile_i = blockIdx.x; tile_i < tp.n_tiles; tile_i += gridDim.x) {
        const unsigned end = seq + (unsigned)(tp.tiles[tile_i].list_cnt * tp.n_chunks);
        for (unsigned s = seq + (cw + kConvWarps - seq % kConvWarps) % kConvWarps; s < end; s += kConvWarps) {
          const unsigned rs = s % kRawStages, ts = s % kTabStages;
          // (stage s always meets the same converter in its slot: kRawStages is a multiple of kConvWarps, see there)
          mbar_wait(raw_full0 + 8 * rs, (s / kRawStages) & 1u);
          mbar_wait(tab_empty0 + 8 * ts, ((s / kTabStages) & 1u) ^ 1u);
          if (lane == 0) {
            float4 mt = sm.meta_raw[rs];
            mt.w = kMagic + (float)(ts * NE);
            sm.meta_tab[ts] = mt;
            if (GEN && P.has_dir) sm.dir_tab[ts] = sm.dir_raw[rs];
          }
          const unsigned src = raw0 + rs * (NE * EB) + lane * EB, dst = tab0 + ts * (NE * TB) + lane * TB;
#pragma unroll
          for (int j = 0; j < (NE + 31) / 32; ++j) {
            const int e = lane + 32 * j;
            if (NE % 32 == 0 || e < NE) {
              const float kl = (float)(e % W);               // window-local entry index
              if constexpr (MODE == kIQ16) {
                const uint2 r = lds64u(src + j * 32 * EB);
                const float2 mid = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
                const float2 sl = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
                sts128(dst + j * 32 * TB, make_float4(fmaf(-kl, sl.x, mid.x), fmaf(-kl, sl.y, mid.y), sl.x, sl.y));
              } else if constexpr (MODE == kIQ32) {
                const float4 r = lds128<0>(src + j * 32 * EB);
                sts128(dst + j * 32 * TB, make_float4(fmaf(-kl, r.z, r.x), fmaf(-kl, r.w, r.y), r.z, r.w));
              } else if constexpr (MODE == kIQ8) {
                const unsigned r = lds32u(src + j * 32 * EB);
                const float2 mid = fp8x2_to_float2((unsigned short)(r & 0xffffu)), sl = fp8x2_to_float2((unsigned short)(r >> 16));
                sts128(dst + j * 32 * TB, make_float4(fmaf(-kl, sl.x, mid.x), fmaf(-kl, sl.y, mid.y), sl.x, sl.y));
              } else if constexpr (MODE == kRF8) {
                const float2 ms = fp8x2_to_float2(lds16u(src + j * 32 * EB));
                sts64(dst + j * 32 * TB, make_float2(fmaf(-kl, ms.y, ms.x), ms.y));
              } else if constexpr (MODE == kRF16) {
                const unsigned r = lds32u(src + j * 32 * EB);
                const float2 ms = __half22float2(*reinterpret_cast<const __half2*>(&r));
                sts64(dst + j * 32 * TB, make_float2(fmaf(-kl, ms.y, ms.x), ms.y));
              } else {
                const float2 r = lds64f<0>(src + j * 32 * EB);
                sts64(dst + j * 32 * TB, make_float2(fmaf(-kl, r.y, r.x), r.y));
              }
            }
          }
          __syncwarp();
          if (lane == 0) { mbar_arrive(tab_full0 + 8 * ts); mbar_arrive(raw_empty0 + 8 * rs); }
        }
        seq = end;
      }
    }
    return;
  }

  // ================================= CONSUMERS ==============================================
  reg_inc<kRegsConsumer>();
  const int wz = warp / (kWX * kWY), wy = (warp / kWX) % kWY, wx = warp % kWX;
  const int lx = lane % kLaneX, ly = lane / kLaneX;
  // table address of an entry: (bits(u) << TSH) + base_adj, where bits(u) still holds the float
  // exponent pattern of MAGIC; addr_bias (a kernel parameter) removes it mod 2^32
  const unsigned base_adj = smem_u32(&sm.tab[0][0]) + tp.addr_bias;
  const unsigned meta0 = smem_u32(&sm.meta_tab[0]);
  unsigned slot = 0, phase = 0;          // table-ring position of this warp (same in all consumer warps)

  for (int tile_i = blockIdx.x; tile_i < tp.n_tiles; tile_i += gridDim.x) {
    const TileDesc td = tp.tiles[tile_i];
    const int ix = td.ix0 + wx * kLaneX + lx;
    const int iy = td.iy0 + wy * kLaneY + ly;
    const int iz = td.iz0 + wz;
    const bool in_grid = ix < P.nx && iy < P.ny && iz < P.nz;
    const int izc = min(iz, P.nz - 1);
    const float x = P.xs[min(ix, P.nx - 1)], y = P.ys[min(iy, P.ny - 1)], z = P.zs[izc];
    const double a_d = (double)z - tp.z_array;
    const long long n_flat = ((long long)min(ix, P.nx - 1) * P.ny + min(iy, P.ny - 1)) * P.nz + izc;   // voxel index (tables)
    // pin(): values the receiver loop reads every iteration are routed through a shuffle so that
    // ptxas keeps them in registers instead of rematerialising them (FP64 ops, select chains)
    const float a = pin((float)a_d);
    // aperture test  4 f#^2 rho^2 <= a^2  with everything that switches it off folded into the
    // two thresholds: voxel outside the grid -> never active; no apodization -> always active
    const float a2 = a * a;
    const float a2e = pin(!in_grid ? -1.f : (P.apod ? a2 : __int_as_float(0x7f800000)));
    const float band = pin((in_grid && P.apod) ? kBand * a2 : -1.f);
    float out_re = 0.f, out_im = 0.f;

    for (int ch = 0; ch < tp.n_chunks; ++ch) {
      const int q0 = ch * QC;
      // ---- per-(q, n) part in FP64: reduced transmit delay and transmit phase -------------
      float2 Tf[QP];
      float2 acc[2 * QP];
#pragma unroll
      for (int j = 0; j < 2 * QP; ++j) {
        const int q = min(q0 + j, P.Q - 1);
        const double T = ((GEN ? tx_tau(P, q, n_flat, x, y, z) : tx_delay(P.tx[q], x, y, z, P.c)) + a_d / P.c - P.t_start) * P.fs;
        const int k0 = __ldg(&tp.k0tile[(long long)tile_i * P.Q + q]);
        const float tf = (float)(T - (double)k0 - 0.5);
        if (j & 1) Tf[j >> 1].y = tf; else Tf[j >> 1].x = tf;
        if (IQ && j < QC) {
          double cyc = tp.phase0 + tp.ratio * T;
          cyc -= rint(cyc);
          sm.cyc[IQ ? j : 0][tid] = (float)cyc;          // read back by this thread only
        }
        acc[j] = make_float2(0.f, 0.f);
      }

      // ---- receiver loop ---------------------------------------------------------------
      for (int li = 0; li < td.list_cnt; ++li) {
        Geo g;
        geo_test<GEN>(g, tab_full0, meta0, slot, phase, x, y, izc, a, a2, a2e, band, tp, P);
        if (g.act) {
          geo_finish<IQ, GEN>(g, a, a2, tp, P);
          const float2 ep2 = make_float2(g.ep, g.ep), mg2 = make_float2(g.mg, g.mg);
          const float2 p1 = make_float2(g.pr, g.pi), p2 = make_float2(-g.pi, g.pr);
          constexpr int kRow = W * TB;
#pragma unroll
          for (int jp = 0; jp < QP; ++jp) {
            const float2 ts = __fadd2_rn(Tf[jp], ep2);
            const float2 u = __fadd2_rn(ts, mg2);
            const unsigned a0 = (__float_as_uint(u.x) << TSH) + base_adj;
            const unsigned a1 = (__float_as_uint(u.y) << TSH) + base_adj;
            // immediates: row offsets of transmit 2 jp and 2 jp + 1 inside a stage
            switch (jp) {
#define DAS_CASE(JP) case JP: \
              term<MODE, (2 * JP) * kRow>(a0, ts.x, p1, p2, acc[2 * jp]); \
              term<MODE, ((2 * JP + 1) % (QC > 1 ? QC : 1)) * kRow>(a1, ts.y, p1, p2, acc[2 * jp + 1]); break;
              DAS_CASE(0) DAS_CASE(1) DAS_CASE(2) DAS_CASE(3) DAS_CASE(4) DAS_CASE(5) DAS_CASE(6) DAS_CASE(7)
#undef DAS_CASE
              default: break;
            }
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(tab_empty0 + 8 * slot);
        slot = (slot + 1) % kTabStages;
        phase ^= (slot == 0);
      }

      // ---- fold this chunk: x += sum_q Ptx_q * acc_q ---------------------------------------
#pragma unroll
      for (int j = 0; j < 2 * QP; ++j) {
        if (j < QC && q0 + j < P.Q) {
          const float wq = GEN ? tx_weight(P, q0 + j, n_flat) : 1.f;        // transmit weight (1 without a table)
          if (GEN && wq == 0.f) continue;      // reading W5: weight 0 = not listed; what its samples gave (inf, NaN) is dropped
          if (IQ) {
            const float ang = 6.283185307179586f * sm.cyc[IQ ? j : 0][tid];
            const float cs = wq * cos_approx(ang), sn = wq * sin_approx(ang);
            out_re = fmaf(acc[j].x, cs, fmaf(-acc[j].y, sn, out_re));
            out_im = fmaf(acc[j].x, sn, fmaf(acc[j].y, cs, out_im));
          } else {
            out_re = fmaf(wq, acc[j].x, out_re);
          }
        }
      }
    }
    if (in_grid) {
      const long long n = ((long long)ix * P.ny + iy) * P.nz + iz;
      if (IQ) reinterpret_cast<float2*>(out_v)[n] = make_float2(out_re, out_im);
      else    reinterpret_cast<float*>(out_v)[n] = out_re;
    }
  }
}

// ---- per-mode launcher, instantiated in das_tiled_inst_*.cu ----------------------------------
template <int QC, int W, int MODE, bool GEN>
cudaError_t launch_tiled_gen(const TiledDev& tp, const Params& P, const void* conv, void* out, int grid, cudaStream_t s) {
  auto k = tiled_kernel<QC, W, MODE, GEN>;
  const size_t smem = sizeof(TiledSmem<QC, W, MODE>);
  // per launch: the attribute belongs to the (device, context) the plan lives on, and setting it is cheap
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k<<<grid, kTiledThreads, smem, s>>>(tp, P, static_cast<const unsigned char*>(conv), out);
  return cudaGetLastError();
}
template <int QC, int W, int MODE>
cudaError_t launch_tiled_inst(const TiledDev& tp, const Params& P, const void* conv, void* out, int grid, cudaStream_t s) {
  const bool gen = P.has_dir || P.window != DAS_WINDOW_BOXCAR || P.tau_tab != nullptr || P.wtx_tab != nullptr;
  return gen ? launch_tiled_gen<QC, W, MODE, true>(tp, P, conv, out, grid, s) : launch_tiled_gen<QC, W, MODE, false>(tp, P, conv, out, grid, s);
}

template <int QC, int MODE>
cudaError_t launch_tiled_w(int W, const TiledDev& tp, const Params& P, const void* conv, void* out, int grid, cudaStream_t s) {
  switch (W) {
    case 16: return launch_tiled_inst<QC, 16, MODE>(tp, P, conv, out, grid, s);
    case 20: return launch_tiled_inst<QC, 20, MODE>(tp, P, conv, out, grid, s);
    case 24: return launch_tiled_inst<QC, 24, MODE>(tp, P, conv, out, grid, s);
    case 32: return launch_tiled_inst<QC, 32, MODE>(tp, P, conv, out, grid, s);
    case 48: return launch_tiled_inst<QC, 48, MODE>(tp, P, conv, out, grid, s);
    case 64: return launch_tiled_inst<QC, 64, MODE>(tp, P, conv, out, grid, s);
    default: return cudaErrorInvalidValue;
  }
}

template <int MODE>
cudaError_t launch_tiled_mode(int QC, int W, const TiledDev& tp, const Params& P, const void* conv, void* out, int grid, cudaStream_t s) {
  switch (QC) {
    case 1: return launch_tiled_w<1, MODE>(W, tp, P, conv, out, grid, s);
    case 2: return launch_tiled_w<2, MODE>(W, tp, P, conv, out, grid, s);
    case 4: return launch_tiled_w<4, MODE>(W, tp, P, conv, out, grid, s);
    case 8: return launch_tiled_w<8, MODE>(W, tp, P, conv, out, grid, s);
    case 16: return launch_tiled_w<16, MODE>(W, tp, P, conv, out, grid, s);
    default: return cudaErrorInvalidValue;
  }
}

// defined one per TU
cudaError_t launch_tiled_iq32(int QC, int W, const TiledDev&, const Params&, const void*, void*, int grid, cudaStream_t);
cudaError_t launch_tiled_iq16(int QC, int W, const TiledDev&, const Params&, const void*, void*, int grid, cudaStream_t);
cudaError_t launch_tiled_rf32(int QC, int W, const TiledDev&, const Params&, const void*, void*, int grid, cudaStream_t);
cudaError_t launch_tiled_rf16(int QC, int W, const TiledDev&, const Params&, const void*, void*, int grid, cudaStream_t);
cudaError_t launch_tiled_iq8(int QC, int W, const TiledDev&, const Params&, const void*, void*, int grid, cudaStream_t);
cudaError_t launch_tiled_rf8(int QC, int W, const TiledDev&, const Params&, const void*, void*, int grid, cudaStream_t);

constexpr int kWindows[] = {16, 20, 24, 32, 48, 64};

}  // namespace das
