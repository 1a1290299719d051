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
//   warps 0..11  three generator warpgroups, one per voxel group (depth) of the tile; thread =
//                voxel = MMA row = TMEM lane.  Per receiver: aperture test, excess path, receive
//                phase.  Per (q, m): fractional index, weights, the 8 packed FP16 pairs of an
//                A row -> tcgen05.st.  After the last receiver: tcgen05.ld of D -> global.
//   warp 12      TMA producer: one bulk copy per (q, m) of the k-blocks the tile needs.
//   warps 13..15 MMA issuers, one per voxel group (one thread each): tcgen05.mma.kind::f16,
//                A from TMEM, B from shared memory (K-major, no swizzle: a k-block of
//                N columns x 16 B is one slab), D of the group in TMEM.
#pragma once

#include "das_tiled.cuh"

namespace das {

constexpr int kTcGX = 16, kTcGY = 8;        // a voxel group: 16 x 8 lateral voxels at one depth
constexpr int kTcRows = kTcGX * kTcGY;      // = 128 = MMA M
constexpr int kTcG = 3;                     // voxel groups (consecutive depths) per tile
constexpr int kTcBlk = 4;                   // samples per k-block (8 FP16 = 16 B per column)
constexpr int kTcPassBlocks = 2;            // k-blocks per pass = one MMA of K = 16
constexpr int kTcABufs = 4;                 // A ring per voxel group (TMEM), one MMA each; power of two
constexpr int kTcStages = 4;                // shared-memory ring of staged sample windows
constexpr int kTcPadBlocks = 16;            // zero k-blocks before and after every (m, q) row
constexpr int kTcMaxStageBlocks = 16;       // largest window (k-blocks) one stage can hold
constexpr int kTcGenWarps = 4 * kTcG;
constexpr int kTcThreads = (kTcGenWarps + 1 + kTcG) * 32;   // + TMA producer + one MMA issuer per group
constexpr int kTcTmemCols = 512;
constexpr int kTcACols = 8;                 // TMEM columns of one A buffer (K = 16 FP16 per row)
constexpr float kTcMargin = 0.02f;          // samples: slack of the plan's delay bounds

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
  int stage_blocks;            // capacity of one stage in k-blocks
  const TcTile* tiles;         // [n_tiles], sorted by decreasing work
  const int2* trange;          // [n_tiles][G][Q]: floor(16 (Tmin - margin)), ceil(16 (Tmax + margin))
  const int* tbase;            // [n_tiles][Q]: sample offset of the reduced delays, multiple of 4
  const uint4* list;           // per tile: x = m, y/z/w = group 0/1/2: elo16 | ehi16 << 16
                               //   (bounds of 16 e over the group's active voxels); 0xFFFFFFFF = none active
  double z_array, kappa, ratio, phase0;
  float four_f2, kappa_f, ratio_f;
};

// k-block range of group g for item (q, m); identical integer arithmetic on host and device and
// in every warp role.  Returns the number of k-blocks (even, 0 if the group has no active voxel).
__host__ __device__ inline int tc_block_range(int2 tr, unsigned er, int& blk_lo) {
  if (er == 0xFFFFFFFFu) { blk_lo = 0; return 0; }
  const int elo = (int)(er & 0xFFFFu), ehi = (int)(er >> 16);
  const int s_lo = (tr.x + elo) >> 4;               // <= floor(t) of every active voxel
  const int s_hi = ((tr.y + ehi) >> 4) + 1;         // >= floor(t) + 1
  blk_lo = s_lo >> 2;
  const int nb = (s_hi >> 2) - blk_lo + 1;
  return (nb + 1) & ~1;
}

// ---- tcgen05 / TMEM PTX ----------------------------------------------------------------------
__device__ __forceinline__ void tmem_alloc(unsigned smem_dst, unsigned cols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(unsigned taddr, unsigned cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
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
  unsigned long long b_full[kTcStages], b_empty[kTcStages];
  unsigned long long a_full[kTcG][kTcABufs], a_empty[kTcG][kTcABufs];
  unsigned long long d_full, d_empty;
  int wlo[kTcStages];                // first k-block of the staged window (producer -> MMA issuer)
  unsigned tmem_base;
};

__host__ __device__ inline size_t tc_smem_bytes(int Bc, int stage_blocks) {
  return sizeof(TcSmemHeader) + 128 + (size_t)kTcStages * stage_blocks * (2 * Bc) * 16;
}

struct TcPlan;
TcPlan* tc_plan_create(const Params& P, const das_plan_desc_t& desc, int n_frames, int device,
                       char* why, size_t why_len, cudaError_t* cuda_err);
void tc_plan_destroy(TcPlan* tp);
size_t tc_converted_bytes(const TcPlan* tp, const Params& P);
int tc_frames_per_chunk(const TcPlan* tp);
cudaError_t launch_tc(const TcPlan* tp, const Params& P, const void* d_conv, void* d_out, cudaStream_t s);
cudaError_t launch_convert_batch(const TcPlan* tp, const Params& P, const void* d_raw, void* d_conv,
                                 float scale, cudaStream_t s);

}  // namespace das
