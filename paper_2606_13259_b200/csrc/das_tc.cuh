// Frame-batch delay-and-sum on the 5th-generation tensor cores (tcgen05 / TMEM) -- the
// "tensor core" variant of the paper (section 3.4, Alg. 3 :218-249) on the
// batch-inner data layout (section 3.2), re-designed for sm_100a.
//
// For a batch of B frames that share geometry, Eq. 2 is, per frame b,
//     x_bn = sum_q sum_m  [ w_mn P_qmn (1-a) ] y_bqm[k] + [ w_mn P_qmn a ] y_bqm[k+1]
// with k = floor(t_qmn), a = t_qmn - k and P = exp(j 2 pi fc tau_qmn).  The bracketed
// interpolation-and-rotation weights do not depend on b.  For a group of 128 neighbouring
// voxels (16 x 8 lateral, one depth) the sample indices of one (q, m) pair cluster inside a few
// "k-blocks" of 4 consecutive samples, so the sum is a dense contraction
//
//     D[n, (b,c')] += sum_{(u,c)} A[n, (u,c)] * Y[(u,c), (b,c')]        n: 128 voxels (MMA M)
//                                                                       (u,c): 8 samples x re/im (K = 16)
//                                                                       (b,c'): frames x re/im (N = 2 Bc)
//     A[n,(u,0)] = Re W_n(u),  A[n,(u,1)] = -Im W_n(u),   W_n(u) = weight voxel n gives sample u
//     Y[(u,0),(b,0)] = Re y,  Y[(u,1),(b,0)] = Im y   |   Y[(u,0),(b,1)] = Im y,  Y[(u,1),(b,1)] = -Re y
//
// (the second column of each frame holds -j y, so that one real MMA yields Re and Im of the
// complex product).  A is GENERATED per (q, m, voxel) on the CUDA cores (FP32 arithmetic, FP64
// for the part common to all receivers exactly as in das_tiled.cuh), rounded to FP16 and
// written straight into tensor memory; Y is the converted channel data (das_convert, batch
// layout) staged in shared memory by TMA bulk copies; D accumulates in FP32 in tensor memory
// over all transmits and receivers of a voxel tile.  The weights are amortised over the Bc
// frames of a chunk: the per-frame cost on the CUDA cores drops by Bc.
//
// Roles inside a CTA (one CTA per SM, persistent over a work-sorted tile list):
//   warps 0..11  generators, 4 warps per voxel group (depth) of the tile; thread = voxel = MMA row
//                = TMEM lane.  Per receiver: aperture test, excess path, receive phase.  Per
//                (q, m): fractional index, weights, the 8 packed FP16 pairs of an A row ->
//                tcgen05.st.  After the last receiver: tcgen05.ld of D -> global, D zeroed again.
//   warp 12      TMA producer: one bulk copy per (q, m) of the k-blocks the tile needs.
//   warps 13..15 MMA issuers, one per voxel group: tcgen05.mma.kind::f16, A from TMEM, B from
//                shared memory (K-major, no swizzle: a k-block of N columns x 16 B is one slab),
//                D of the group in TMEM.  The issue loop is a serial latency chain (wait, MMA,
//                commit): every lane runs it, only the tcgen05 instructions sit under elect.sync.
//   (The issue arbiter favours high warp ids: the short, latency-critical service warps sit above
//   the generators; the other order measured 5 % slower.)
#pragma once

#include "das_tiled.cuh"

namespace das {

constexpr int kTcGX = 16, kTcGY = 8;        // a voxel group: 16 x 8 lateral voxels at one depth
constexpr int kTcRows = kTcGX * kTcGY;      // = 128 = MMA M
constexpr int kTcG = 3;                     // voxel groups (consecutive depths) per tile
constexpr int kTcBlk = 4;                   // samples per k-block (8 FP16 = 16 B per column)
constexpr int kTcPassBlocks = 2;            // k-blocks per pass = one MMA of K = 16
constexpr int kTcMaxABufs = 8;              // A ring per voxel group (TMEM), one MMA each; depth a power of two
constexpr int kTcMaxStages = 16;            // upper bound of the shared-memory ring of staged sample windows
constexpr int kTcMinStages = 2;
constexpr int kTcPadBlocks = 16;            // zero k-blocks before and after every (m, q) row
constexpr int kTcMaxStageBlocks = 16;       // largest window (k-blocks) one stage can hold
constexpr int kTcGenWarps = 4 * kTcG;
constexpr int kTcSvcWarps = 1 + kTcG;        // TMA producer + one MMA issuer per voxel group
constexpr int kTcThreads = (kTcSvcWarps + kTcGenWarps) * 32;
constexpr int kTcTmemCols = 512;
constexpr int kTcACols = 8;                 // TMEM columns of one A buffer (K = 16 FP16 per row)
constexpr float kTcMargin = 0.02f;          // samples: slack of the plan's transmit-delay bounds (tbase)

__host__ __device__ inline int tc_kblocks(int K) { return 2 * kTcPadBlocks + (K + kTcBlk - 1) / kTcBlk; }

struct TcTile {
  int ix0, iy0, iz0;
  int list_off, list_cnt;
  int edge;                    // 1 if a staged window touches sample 0 or K-1: the A6 rule needs the explicit test
};

struct TcDev {
  int n_tiles, n_chunks;       // work items = n_tiles * n_chunks
  int Bc;                      // frames per chunk; MMA N = 2 Bc
  int KBp;                     // k-blocks per (m, q) row of the converted data, pads included
  int stage_blocks;            // capacity of one window slot in k-blocks
  int qs;                      // window slots (consecutive transmits of one receiver) per stage: one barrier round per qs items
  int n_stages;                // depth of the stage ring (kTcMinStages..kTcMaxStages)
  int a_bufs, a_shift;         // depth of the A ring per voxel group (2^a_shift <= kTcMaxABufs, what TMEM holds)
  const TcTile* tiles;         // [n_tiles], sorted by decreasing work
  const int* tbase;            // [n_tiles][Q]: sample offset of the reduced delays, multiple of 4
  const uint2* list;           // receiver lists of the tiles: x = m, y = bit g set if group g has a window
  const unsigned short* codes; // [entry][G][16]: window of item (q, m) for group g, written by the plan's
                               //   window kernel from the delays of the group's ACTIVE voxels:
                               //   bits 0-1 = n_pass (MMAs of K = 16 = 8 samples; 0 = no active voxel),
                               //   bits 2-15 = first sample of the window in units of 2 samples, relative
                               //   to tbase_q
  double z_array, kappa, ratio, phase0;
  float four_f2, kappa_f, ratio_f;
};

constexpr float kTcDelta = 1.0f / 128;      // samples: the window kernel widens every delay by this much, so that
                                            // rounding differences between it and the generator cannot matter
__host__ __device__ inline int code_passes(unsigned c) { return (int)(c & 3u); }
__host__ __device__ inline int code_start2(unsigned c) { return (int)(c >> 2); }   // units of 2 samples

// Window of item (q, m) the producer stages: the union over the voxel groups, as (first k-block relative
// to tbase_q / 4, number of k-blocks).  `codes_q` points at the code of group 0 for this q.
__device__ __forceinline__ void tc_union_window(const unsigned short* codes_q, int& wlo, int& wn) {
  int lo = 0x7fffffff, hi = -0x7fffffff;
#pragma unroll
  for (int g = 0; g < kTcG; ++g) {
    const unsigned c = __ldg(&codes_q[g * 16]);
    if (code_passes(c)) {
      lo = min(lo, code_start2(c) >> 1);
      hi = max(hi, (code_start2(c) >> 1) + kTcPassBlocks * code_passes(c));
    }
  }
  wlo = hi > lo ? lo : 0;
  wn = hi > lo ? hi - lo : 0;
}

// ---- geometry shared by the generator warps and the plan's window kernel ---------------------
struct TcVoxel {
  float x, y, z, a, a2, a2e, band;
  double a_d;
  int ix, iy, iz, izc;
  bool in_grid;
};
// voxel of MMA row `row` (0..127: 16 x 8 lateral) in depth group g of tile td
__device__ __forceinline__ TcVoxel tc_voxel(const TcDev& tp, const Params& P, const TcTile& td, int row, int g) {
  TcVoxel v;
  v.ix = td.ix0 + row % kTcGX; v.iy = td.iy0 + row / kTcGX; v.iz = td.iz0 + g;
  v.in_grid = v.ix < P.nx && v.iy < P.ny && v.iz < P.nz;
  v.izc = min(v.iz, P.nz - 1);
  v.x = P.xs[min(v.ix, P.nx - 1)]; v.y = P.ys[min(v.iy, P.ny - 1)]; v.z = P.zs[v.izc];
  v.a_d = (double)v.z - tp.z_array;
  v.a = (float)v.a_d;
  v.a2 = v.a * v.a;
  v.a2e = !v.in_grid ? -1.f : (P.apod ? v.a2 : __int_as_float(0x7f800000));
  v.band = (v.in_grid && P.apod) ? kBand * v.a2 : -1.f;
  return v;
}
// the part of the sample coordinate common to all receivers: T_q(n) = (tau_tx + a / c - t_start) fs, FP64
__device__ __forceinline__ double tc_T(const Params& P, const TcVoxel& v, int q) {
  return (tx_delay(P.tx[q], v.x, v.y, v.z, P.c) + v.a_d / P.c - P.t_start) * P.fs;
}
// receive excess path e_m(n) in samples (FP32) and the exactly classified aperture weight
__device__ __forceinline__ float tc_excess(const TcDev& tp, const Params& P, const TcVoxel& v, float4 el, bool& act) {
  const float dx = v.x - el.x, dy = v.y - el.y;
  const float rho2 = fmaf(dx, dx, dy * dy);
  const float lhs = tp.four_f2 * rho2;
  act = lhs <= v.a2e;
  if (fabsf(lhs - v.a2e) <= v.band) act = aperture_exact(v.x, v.y, el.x, el.y, P.zs, v.izc, tp.z_array, P.fnum);
  const float s2 = rho2 + v.a2;
  const float d = s2 * rsqrt_approx(s2);
  return (rho2 * tp.kappa_f) * rcp_approx(v.a + d);
}

// mbarrier wait that parks the thread in hardware (suspend-time hint, ns) instead of spinning through
// issue slots the generator warps need; it resumes as soon as the phase completes
__device__ __forceinline__ void mbar_wait_park(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(bar), "r"(parity), "r"(20000u) : "memory");
}

// ---- tcgen05 / TMEM PTX ----------------------------------------------------------------------
__device__ __forceinline__ void tmem_alloc(unsigned smem_dst, unsigned cols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(unsigned taddr, unsigned cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
// one lane of the (converged) warp
__device__ __forceinline__ bool tc_elect() {
  unsigned pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(unsigned bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem descriptor];  M = 128, K = 16, FP16 inputs, FP32 accumulate
__device__ __forceinline__ void tc_mma_ts(unsigned d_tmem, unsigned a_tmem, unsigned long long b_desc, unsigned idesc, unsigned accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tmem_st8(unsigned taddr, const unsigned (&v)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
}
__device__ __forceinline__ void tmem_st8_zero(unsigned taddr) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(taddr), "r"(0u) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld16(unsigned taddr, float (&v)[16]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]),
                 "=f"(v[8]), "=f"(v[9]), "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]), "=f"(v[14]), "=f"(v[15])
               : "r"(taddr) : "memory");
}
// shared-memory matrix descriptor, K-major, no swizzle: 8-row core matrices of 16-byte rows;
// SBO = byte step between 8-column groups (N direction), LBO = byte step between the two
// 16-byte K chunks of a K = 16 MMA (here: one slab = one k-block)
__device__ __forceinline__ unsigned long long tc_smem_desc(unsigned addr, unsigned lbo_bytes, unsigned sbo_bytes) {
  return (unsigned long long)((addr >> 4) & 0x3FFFu) | ((unsigned long long)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
         ((unsigned long long)((sbo_bytes >> 4) & 0x3FFFu) << 32) | (1ull << 46);
}
// instruction descriptor: D = F32, A = B = F16, both K-major, dense, M = 128, N = n
__host__ __device__ inline unsigned tc_idesc(int n) {
  return (1u << 4) | ((unsigned)(n >> 3) << 17) | ((unsigned)(kTcRows >> 4) << 24);
}
__device__ __forceinline__ unsigned pack_half2(float lo, float hi) {
  unsigned r;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

struct alignas(128) TcSmemHeader {
  unsigned long long b_full[kTcMaxStages], b_empty[kTcMaxStages];
  unsigned long long a_full[kTcG * kTcMaxABufs], a_empty[kTcG * kTcMaxABufs];
  unsigned long long d_full, d_empty;
  unsigned long long sink;           // arrivals nobody waits for (no A tile in flight)
  unsigned tmem_base;
};

__host__ __device__ inline size_t tc_smem_bytes(int Bc, int stage_blocks, int qs, int n_stages) {
  return sizeof(TcSmemHeader) + 128 + (size_t)n_stages * qs * stage_blocks * (2 * Bc) * 16;
}

struct TcPlan;
TcPlan* tc_plan_create(const Params& P, const das_plan_desc_t& desc, int n_frames, int device,
                       char* why, size_t why_len, cudaError_t* cuda_err);
void tc_plan_destroy(TcPlan* tp);
size_t tc_converted_bytes(const TcPlan* tp, const Params& P);
int tc_frames_per_chunk(const TcPlan* tp);
cudaError_t launch_tc_windows(const TcDev& tp, const Params& P, uint2* list, unsigned short* codes, int* tile_work,
                              int* tile_edge, int* stats, cudaStream_t s);
cudaError_t launch_tc(const TcPlan* tp, const Params& P, const void* d_conv, void* d_out, cudaStream_t s);
cudaError_t launch_convert_batch(const TcPlan* tp, const Params& P, const void* d_raw, void* d_conv,
                                 float scale, cudaStream_t s);

}  // namespace das
