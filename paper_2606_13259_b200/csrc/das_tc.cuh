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
// layout) staged in shared memory by TMA tensor copies; D accumulates in FP32 in tensor memory
// over all transmits and receivers of a voxel tile.  The weights are amortised over the Bc
// frames of a chunk: the per-frame cost on the CUDA cores drops by Bc.
//
// Roles inside a CTA (one CTA per SM, persistent over a work-sorted tile list):
//   warps 0..11  generators, 4 warps per voxel group (depth) of the tile; thread = voxel = MMA row
//                = TMEM lane.  Per receiver: aperture test, excess path, receive phase.  Per
//                (q, m): fractional index, weights, the 8 packed FP16 pairs of an A row ->
//                tcgen05.st.  After the last receiver: tcgen05.ld of D -> global, D zeroed again.
//                The A tiles of a group live in a ring of 4 ITEM SLOTS in tensor memory plus one
//                OVERFLOW slot: item q of a receiver always uses slot q mod 4 (first MMA pass of its
//                window), the 2nd / 3rd pass of the 30 % of items that need one goes through the
//                overflow slot.  Slot, barrier address and (for 16 transmits) barrier phase of every
//                item are therefore compile-time constants in the unrolled transmit loop: one
//                mbarrier round per item with no ring arithmetic.
//   warp 12      TMA producer: one bulk copy per (q, m) of the k-blocks the tile needs.
//   warps 13..15 MMA issuers, one per voxel group: tcgen05.mma.kind::f16, A from TMEM, B from
//                shared memory, D of the group in TMEM.  B is MN-MAJOR without swizzle: a K row is one
//                (sample, y | -j y) vector over the N = 2 Bc frame columns, stored as N / 8 column
//                groups of 16 bytes; per column group the K rows are contiguous, so an MMA window
//                (8 samples = 16 K rows = two 8-row core matrices) may start at ANY sample of the
//                staged box: the descriptor's start address moves in steps of one row pair.  The issue loop is a serial latency chain (wait, MMA,
//                commit): every lane runs it, only the tcgen05 instructions sit under elect.sync.
//   (The issue arbiter favours high warp ids: the short, latency-critical service warps sit above
//   the generators; the other order measured 5 % slower.)
#pragma once

#include "das_tiled.cuh"

namespace das {

constexpr int kTcGX = 16, kTcGY = 8;        // a voxel group: 16 x 8 lateral voxels at one depth
constexpr int kTcRows = kTcGX * kTcGY;      // = 128 = MMA M
constexpr int kTcG = 3;                     // voxel groups (consecutive depths) per tile
constexpr int kTcBlk = 4;                   // samples per core matrix of the B operand (8 K rows: y and -j y of 4 samples)
constexpr int kTcPassBlocks = 2;            // core matrices per pass = one MMA of K = 16 = 8 samples
constexpr int kTcPass = kTcBlk * kTcPassBlocks;   // samples per MMA pass
// One staged box (a TMA tensor copy) holds the union of the windows of a tile's voxel groups for one (q, m).
// Two box sizes: the small one takes the common case (every group one MMA pass, 87 % of the items at the
// headline), the big one the rest; the stage slot has the big one's size.
constexpr int kTcBoxSmall = 12, kTcBoxBig = 20;   // samples
constexpr int kTcCodeBig = 0x8000;                // window code: the item uses the big box
constexpr int kTcSlots = 4;                 // item slots of a group's A ring (TMEM): item q uses slot q mod 4
constexpr int kTcOvf = kTcSlots;            // the overflow slot: 2nd / 3rd MMA pass of an item
constexpr int kTcABufs = kTcSlots + 1;      // A tiles per voxel group in tensor memory
constexpr int kTcMaxStages = 16;            // upper bound of the shared-memory ring of staged sample windows
constexpr int kTcMinStages = 2;
constexpr int kTcMaxQs = 16;                // upper bound of the window slots (transmits) per stage
constexpr int kTcGenWarps = 4 * kTcG;
constexpr int kTcSvcWarps = 4;               // TMA producer + one MMA issuer per voxel group (whole warpgroups: setmaxnreg)
constexpr int kTcThreads = (kTcSvcWarps + kTcGenWarps) * 32;
static_assert(1 + kTcG <= kTcSvcWarps && kTcSvcWarps % 4 == 0 && kTcGenWarps % 4 == 0, "warpgroup roles");
constexpr int kTcTmemCols = 512;
constexpr int kTcACols = 8;                 // TMEM columns of one A buffer (K = 16 FP16 per row)
constexpr float kTcMargin = 0.02f;          // samples: slack of the plan's transmit-delay bounds (tbase)
// Placement table (shared memory): row r (r = slot of sample k inside the MMA pass, kTcPlaceLo <= r <= kTcPlaceHi) holds
// the FP16x2 factors {1,1} / {0,0} that put W0 into slot r and W1 into slot r + 1 of the 8-slot A row: word j of a row
// is 1 iff r == j - 1.  A generator thread loads the 9 words of its row and forms slot i as W0 * word[i + 1] + W1 * word[i]
// (HMUL2 + HFMA2: the placement runs on the FMA pipe instead of 9 compares + 16 selects on the half-rate ALU pipe).
constexpr int kTcPlaceLo = -9, kTcPlaceHi = 16, kTcPlaceWords = 12;
constexpr int kTcPlaceRows = kTcPlaceHi - kTcPlaceLo + 1;


struct TcTile {
  int ix0, iy0, iz0;
  int list_off, list_cnt;
  int edge;                    // 1 if a staged window touches sample 0 or K-1: the A6 rule needs the explicit test
};

struct TcDev {
  int n_tiles, n_chunks;       // work items = n_tiles * n_chunks
  int Bc;                      // frames per chunk; MMA N = 2 Bc
  int groups;                  // depths per tile that carry voxels: kTcG, or 1 when the depths of the grid lie so
                               // far apart in delay that the windows of kTcG of them do not fit one staged box
  int qs;                      // window slots (consecutive transmits of one receiver) per stage: one barrier round per qs items
  int n_stages;                // depth of the stage ring (kTcMinStages..kTcMaxStages)
  const TcTile* tiles;         // [n_tiles], sorted by decreasing work
  const int* tbase;            // [n_tiles][Q]: sample offset of the reduced delays
  const uint2* list;           // receiver lists of the tiles: x = m, y = bit g set if group g has a window
  const unsigned short* codes; // [entry][G][16]: window of item (q, m) for group g, written by the plan's
                               //   window kernel from the delays of the group's ACTIVE voxels:
                               //   bits 0-1 = n_pass (MMAs of K = 16 = 8 samples; 0 = no active voxel),
                               //   bits 2-14 = first sample of the window relative to tbase_q, bit 15 = the
                               //   item (entry, q) uses the big box.  The windows of the groups of one
                               //   (entry, q) lie inside one box that starts at the smallest of their first samples.
  double z_array, kappa, ratio, phase0;
  float four_f2, kappa_f, ratio_f;
  unsigned long long* prof;    // cycle accounting per (CTA, warp), only in -DDAS_TC_PROF builds (else nullptr)
  unsigned long long* progress;// [grid] quad pacing of the TMA producers (das_tc.cu), nullptr = off
  unsigned long long epoch;    // launch counter << 40: progress words of earlier launches compare as far behind
  int pace;                    // receivers a producer may run ahead of the slowest CTA of its quad
  int pace_mask;               // a receiver is paced when (list index & pace_mask) == 0
};

constexpr float kTcDelta = 1.0f / 128;      // samples: the window kernel widens every delay by this much, so that
                                            // rounding differences between it and the generator cannot matter
__host__ __device__ inline int code_passes(unsigned c) { return (int)(c & 3u); }
__host__ __device__ inline int code_start(unsigned c) { return (int)((c >> 2) & 0x1fffu); }     // samples, relative to tbase_q

// ---- geometry shared by the generator warps and the plan's window kernel ---------------------
struct TcVoxel {
  float x, y, z, a, a2, a2e, band;
  double a_d;
  long long n;                 // flat voxel index (clamped into the grid): row of the transmit tables
  int ix, iy, iz, izc;
  bool in_grid;
};
// voxel of MMA row `row` (0..127: 16 x 8 lateral) in depth group g of tile td
__device__ __forceinline__ TcVoxel tc_voxel(const TcDev& tp, const Params& P, const TcTile& td, int row, int g) {
  TcVoxel v;
  v.ix = td.ix0 + row % kTcGX; v.iy = td.iy0 + row / kTcGX; v.iz = td.iz0 + g;
  v.in_grid = v.ix < P.nx && v.iy < P.ny && v.iz < P.nz && g < tp.groups;
  v.izc = min(v.iz, P.nz - 1);
  v.x = P.xs[min(v.ix, P.nx - 1)]; v.y = P.ys[min(v.iy, P.ny - 1)]; v.z = P.zs[v.izc];
  v.n = ((long long)min(v.ix, P.nx - 1) * P.ny + min(v.iy, P.ny - 1)) * P.nz + v.izc;
  v.a_d = (double)v.z - tp.z_array;
  v.a = (float)v.a_d;
  v.a2 = v.a * v.a;
  v.a2e = !v.in_grid ? -1.f : (P.apod ? v.a2 : __int_as_float(0x7f800000));
  v.band = (v.in_grid && P.apod) ? kBand * v.a2 : -1.f;
  return v;
}
// the part of the sample coordinate common to all receivers: T_q(n) = (tau_tx + a / c - t_start) fs, FP64
__device__ __forceinline__ double tc_T(const Params& P, const TcVoxel& v, int q) {
  return (tx_tau(P, q, v.n, v.x, v.y, v.z) + v.a_d / P.c - P.t_start) * P.fs;
}
// receive excess path e_m(n) in samples (FP32) and the exactly classified aperture weight
__device__ __forceinline__ float tc_excess(const TcDev& tp, const Params& P, const TcVoxel& v, float4 el, float4 dir, bool& act, float& wrx) {
  const float dx = v.x - el.x, dy = v.y - el.y;
  const float rho2 = fmaf(dx, dx, dy * dy);
  float u2;
  if (P.has_dir && P.apod) {
    // tilted normal (coplanar positions): the delays are the planar array's, only the cone turns
    act = aperture_dir(v.x, v.y, el.x, el.y, dx, dy, v.a, rho2, v.a2, dir, tp.four_f2, v.in_grid, P.zs, v.izc, tp.z_array, P.fnum, u2);
  } else {
    const float lhs = tp.four_f2 * rho2;
    u2 = lhs * rcp_approx(v.a2);
    act = lhs <= v.a2e;
    if (fabsf(lhs - v.a2e) <= v.band) act = aperture_exact(v.x, v.y, el.x, el.y, P.zs, v.izc, tp.z_array, P.fnum);
  }
  wrx = (P.window != DAS_WINDOW_BOXCAR && P.apod) ? rx_window(P.window, P.taper, u2) : 1.f;   // receive window
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
// The same MMA followed by a tcgen05.commit to `bar`, both under ONE elected lane and in one block (the
// elect / vote / uniform-register traffic of two separate elected statements doubled the issue chain).
__device__ __forceinline__ void tc_mma_commit(unsigned d_tmem, unsigned a_tmem, unsigned desc_lo, unsigned desc_hi, unsigned idesc, unsigned bar) {
  asm volatile(
      "{\n\t.reg .pred p, q;\n\t.reg .b64 dsc;\n\t"
      "mov.b64 dsc, {%2, %3};\n\t"
      "setp.ne.b32 q, %4, 0;\n\t"
      "elect.sync _|p, 0xffffffff;\n\t"
      "@p tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], dsc, %4, q;\n\t"
      "@p tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "r"(desc_lo), "r"(desc_hi), "r"(idesc), "r"(bar) : "memory");
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
// Shared-memory matrix descriptor of the B operand, MN-major, no swizzle ("interleave"): the canonical
// layout is ((8 columns), n column groups) x ((8 K rows), k row groups) with 16-byte units, the 8 K rows of
// a core matrix contiguous;  SBO = byte step between column groups, LBO = byte step between the two
// 8-row groups of a K = 16 MMA.  Bit 46: descriptor version of sm_100.
__device__ __forceinline__ unsigned long long tc_smem_desc(unsigned addr, unsigned lbo_bytes, unsigned sbo_bytes) {
  return (unsigned long long)((addr >> 4) & 0x3FFFu) | ((unsigned long long)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
         ((unsigned long long)((sbo_bytes >> 4) & 0x3FFFu) << 32) | (1ull << 46);
}
// instruction descriptor: D = F32, A = B = F16, A K-major (tensor memory), B MN-major (bit 16), dense, M = 128, N = n
__host__ __device__ inline unsigned tc_idesc(int n) {
  return (1u << 4) | (1u << 16) | ((unsigned)(n >> 3) << 17) | ((unsigned)(kTcRows >> 4) << 24);
}
// TMA tensor copy (3-D tile) global -> this CTA's shared memory, completion (bytes) counted on an mbarrier;
// elements outside the tensor read as zero
__device__ __forceinline__ void tma_tensor3_g2s(unsigned dst, const void* tmap, int c0, int c1, int c2, unsigned bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
               ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}
__device__ __forceinline__ unsigned pack_half2(float lo, float hi) {
  unsigned r;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

struct alignas(128) TcSmemHeader {
  unsigned long long b_full[kTcMaxStages], b_empty[kTcMaxStages];
  unsigned long long a_full[kTcG * kTcABufs], a_empty[kTcG * kTcABufs];
  unsigned long long d_full, d_empty;
  unsigned long long sink;           // arrivals nobody waits for (no A tile in flight)
  unsigned info[kTcMaxStages * kTcMaxQs * kTcG];   // per stage and window slot: what each group's issuer does with the item
  alignas(16) unsigned place[kTcPlaceRows][kTcPlaceWords];   // placement table (see kTcPlaceLo)
  unsigned tmem_base;
};

// bytes of one staged box: N / 8 column groups x 2 K rows per sample x 16 bytes
__host__ __device__ inline unsigned tc_box_bytes(int Bc, int samples) { return (unsigned)(2 * Bc / 8) * (unsigned)(2 * samples) * 16u; }
__host__ __device__ inline size_t tc_smem_bytes(int Bc, int qs, int n_stages) {
  return sizeof(TcSmemHeader) + 1024 + (size_t)n_stages * qs * tc_box_bytes(Bc, kTcBoxBig);
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
