// Frame-batch tensor-core delay-and-sum kernel (tcgen05 / TMEM); design notes in das_tc.cuh.
#include "das_tc.cuh"

namespace das {

namespace {

// (k-block count, first k-block) of one (q, m) item for one voxel group, packed so that one
// shuffle hands it from the lane that computed it (lane = q) to the whole warp
__device__ __forceinline__ int pack_range(int nb, int lo) { return (lo << 8) | nb; }
__device__ __forceinline__ int range_nb(int pk) { return pk & 0xff; }
__device__ __forceinline__ int range_lo(int pk) { return pk >> 8; }

// Work items: (chunk, tile), tile fastest; every warp role walks the same sequence.
__global__ void __launch_bounds__(kTcThreads, 1)
tc_kernel(const TcDev tp, const Params P, const unsigned char* __restrict__ convb, float2* __restrict__ out) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  TcSmemHeader& sm = *reinterpret_cast<TcSmemHeader*>(smem_raw);
  const unsigned stage0 = (smem_u32(smem_raw) + (unsigned)sizeof(TcSmemHeader) + 127u) & ~127u;
  const int N = 2 * tp.Bc;                                   // MMA N
  const unsigned slab = (unsigned)N * 16u;                   // bytes of one k-block: N columns x 8 FP16
  const unsigned stage_bytes = (unsigned)tp.stage_blocks * slab;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_work = tp.n_tiles * tp.n_chunks;
  const long long n_vox = (long long)P.nx * P.ny * P.nz;
  const long long chunk_bytes = (long long)P.M * P.Q * tp.KBp * slab;
  const int ql = min(lane & 15, P.Q - 1);                    // the transmit this lane computes ranges for

  const unsigned b_full0 = smem_u32(&sm.b_full[0]), b_empty0 = smem_u32(&sm.b_empty[0]);
  const unsigned a_full0 = smem_u32(&sm.a_full[0][0]), a_empty0 = smem_u32(&sm.a_empty[0][0]);
  const unsigned d_full = smem_u32(&sm.d_full), d_empty = smem_u32(&sm.d_empty);

  if (tid == 0) {
    for (int s = 0; s < kTcStages; ++s) { mbar_init(b_full0 + 8 * s, 1); mbar_init(b_empty0 + 8 * s, kTcG); }
    for (int i = 0; i < kTcABufs * kTcG; ++i) { mbar_init(a_full0 + 8 * i, 4); mbar_init(a_empty0 + 8 * i, 1); }
    mbar_init(d_full, kTcG);
    mbar_init(d_empty, kTcGenWarps);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == kTcGenWarps) tmem_alloc(smem_u32(&sm.tmem_base), kTcTmemCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const unsigned tmem = sm.tmem_base;
  // TMEM columns: D of group g at g * N; A buffer (g, buf) at kTcG * N + (kTcABufs g + buf) * kTcACols
  const unsigned a_col0 = (unsigned)(kTcG * N);

  if (warp == kTcGenWarps) {
    // ===================================== TMA PRODUCER =======================================
    // lane q works out the window of item (q, m); lane 0 issues the copies in item order
    unsigned it = 0;
    for (int work = blockIdx.x; work < n_work; work += gridDim.x) {
      const int tile_i = work % tp.n_tiles, chunk = work / tp.n_tiles;
      const TcTile td = tp.tiles[tile_i];
      const unsigned char* base = convb + (long long)chunk * chunk_bytes;
      int2 tr[kTcG];
#pragma unroll
      for (int g = 0; g < kTcG; ++g) tr[g] = __ldg(&tp.trange[((long long)tile_i * kTcG + g) * P.Q + ql]);
      uint4 ent = td.list_cnt ? __ldg(&tp.list[td.list_off]) : make_uint4(0, 0, 0, 0);
      for (int li = 0; li < td.list_cnt; ++li) {
        const uint4 cur = ent;
        if (li + 1 < td.list_cnt) ent = __ldg(&tp.list[td.list_off + li + 1]);
        const unsigned er[kTcG] = {cur.y, cur.z, cur.w};
        int wlo = 0x7fffffff, whi = -0x7fffffff;
#pragma unroll
        for (int g = 0; g < kTcG; ++g) {
          int lo;
          const int nb = tc_block_range(tr[g], er[g], lo);
          if (nb) { wlo = min(wlo, lo); whi = max(whi, lo + nb); }
        }
        if (whi <= wlo) { wlo = 0; whi = 0; }
        const long long row0 = (long long)cur.x * P.Q * tp.KBp + kTcPadBlocks;
        for (int q = 0; q < P.Q; ++q, ++it) {
          const int wlo_q = __shfl_sync(0xffffffffu, wlo, q), whi_q = __shfl_sync(0xffffffffu, whi, q);
          if (lane == 0) {
            const unsigned s = it % kTcStages;
            mbar_wait(b_empty0 + 8 * s, ((it / kTcStages) & 1u) ^ 1u);
            sm.wlo[s] = wlo_q;
            const unsigned bytes = (unsigned)(whi_q - wlo_q) * slab;
            if (bytes) {
              mbar_arrive_expect_tx(b_full0 + 8 * s, bytes);
              tma_bulk_g2s(stage0 + s * stage_bytes, base + (row0 + (long long)q * tp.KBp + wlo_q) * (long long)slab, bytes, b_full0 + 8 * s);
            } else {
              mbar_arrive(b_full0 + 8 * s);
            }
          }
          __syncwarp();
        }
      }
    }
  } else if (warp > kTcGenWarps) {
    // ===================================== MMA ISSUERS ========================================
    // one warp per voxel group; lane q works out the k-block range of item (q, m), lane 0 issues
    const int g = warp - kTcGenWarps - 1;
    const unsigned idesc = tc_idesc(N);
    const unsigned d_tmem = tmem + (unsigned)(g * N);
    const unsigned a_tmem0 = tmem + a_col0 + (unsigned)(kTcABufs * g) * kTcACols;
    unsigned it = 0, a_it = 0, n_done = 0;
    for (int work = blockIdx.x; work < n_work; work += gridDim.x, ++n_done) {
      const int tile_i = work % tp.n_tiles;
      const TcTile td = tp.tiles[tile_i];
      const int2 tr = __ldg(&tp.trange[((long long)tile_i * kTcG + g) * P.Q + ql]);
      if (lane == 0) {
        mbar_wait(d_empty, (n_done & 1u) ^ 1u);            // epilogue of the previous tile has drained D
        tc_fence_after();
      }
      __syncwarp();
      unsigned acc = 0;
      uint4 ent = td.list_cnt ? __ldg(&tp.list[td.list_off]) : make_uint4(0, 0, 0, 0);
      for (int li = 0; li < td.list_cnt; ++li) {
        const uint4 cur = ent;
        if (li + 1 < td.list_cnt) ent = __ldg(&tp.list[td.list_off + li + 1]);
        int lo;
        const int nb = tc_block_range(tr, g == 0 ? cur.y : (g == 1 ? cur.z : cur.w), lo);
        const int pk = pack_range(nb, lo);
        for (int q = 0; q < P.Q; ++q, ++it) {
          const int pk_q = __shfl_sync(0xffffffffu, pk, q);
          if (lane == 0) {
            const unsigned s = it % kTcStages;
            const int nb_q = range_nb(pk_q), lo_q = range_lo(pk_q);
            mbar_wait(b_full0 + 8 * s, (it / kTcStages) & 1u);
            const unsigned b0 = stage0 + s * stage_bytes + (unsigned)(lo_q - sm.wlo[s]) * slab;
            for (int p0 = 0; p0 < nb_q; p0 += kTcPassBlocks, ++a_it) {
              const unsigned buf = a_it % kTcABufs;
              mbar_wait(a_full0 + 8 * (kTcABufs * g + buf), (a_it / kTcABufs) & 1u);
              tc_fence_after();
              tc_mma_ts(d_tmem, a_tmem0 + buf * kTcACols, tc_smem_desc(b0 + (unsigned)p0 * slab, slab, 128), idesc, acc);
              acc = 1;
              tc_commit(a_empty0 + 8 * (kTcABufs * g + buf));    // A buffer free once this MMA has read it
            }
            tc_commit(b_empty0 + 8 * s);                         // this group is done with the stage
          }
          __syncwarp();
        }
      }
      if (lane == 0) tc_commit(d_full);                          // this group's MMAs of the tile are complete
      __syncwarp();
    }
  } else {
    // ===================================== GENERATORS =========================================
    const int g = warp >> 2;                                  // voxel group = depth inside the tile
    const int row = (warp & 3) * 32 + lane;                   // MMA row = TMEM lane
    const int lx = row % kTcGX, ly = row / kTcGX;
    const unsigned lane_base = ((unsigned)((warp & 3) * 32)) << 16;
    const unsigned d_addr = tmem + lane_base + (unsigned)(g * N);
    const unsigned a_addr0 = tmem + lane_base + a_col0 + (unsigned)(kTcABufs * g) * kTcACols;
    const unsigned af0 = a_full0 + 8u * (unsigned)(kTcABufs * g), ae0 = a_empty0 + 8u * (unsigned)(kTcABufs * g);
    const bool lane0 = lane == 0;
    unsigned a_it = 0, n_done = 0;
    unsigned pend = 0;                                        // a_full barrier of the A tile whose store is in flight

    for (int work = blockIdx.x; work < n_work; work += gridDim.x, ++n_done) {
      const int tile_i = work % tp.n_tiles, chunk = work / tp.n_tiles;
      const TcTile td = tp.tiles[tile_i];
      const int ix = td.ix0 + lx, iy = td.iy0 + ly, iz = td.iz0 + g;
      const bool in_grid = ix < P.nx && iy < P.ny && iz < P.nz;
      const int izc = min(iz, P.nz - 1);
      const float x = P.xs[min(ix, P.nx - 1)], y = P.ys[min(iy, P.ny - 1)], z = P.zs[izc];
      const double a_d = (double)z - tp.z_array;
      const float a = (float)a_d;
      const float a2 = a * a;
      const float a2e = !in_grid ? -1.f : (P.apod ? a2 : __int_as_float(0x7f800000));
      const float band = (in_grid && P.apod) ? kBand * a2 : -1.f;
      const int2 tr = __ldg(&tp.trange[((long long)tile_i * kTcG + g) * P.Q + ql]);   // this lane's transmit
      const int tb_l = __ldg(&tp.tbase[(long long)tile_i * P.Q + ql]);

      // per-(q, n) part in FP64: reduced transmit delay and transmit phase factor
      float Tf[16], pc[16], ps[16];
#pragma unroll
      for (int q = 0; q < 16; ++q) {
        const int qq = min(q, P.Q - 1);
        const double T = (tx_delay(P.tx[qq], x, y, z, P.c) + a_d / P.c - P.t_start) * P.fs;
        Tf[q] = (float)(T - (double)__ldg(&tp.tbase[(long long)tile_i * P.Q + qq]));
        double cyc = tp.phase0 + tp.ratio * T;
        cyc -= rint(cyc);
        const float ang = 6.283185307179586f * (float)cyc;
        pc[q] = cos_approx(ang);
        ps[q] = sin_approx(ang);
      }
      bool produced = false;

      uint4 ent = td.list_cnt ? __ldg(&tp.list[td.list_off]) : make_uint4(0, 0, 0, 0);
      for (int li = 0; li < td.list_cnt; ++li) {
        const uint4 cur = ent;
        if (li + 1 < td.list_cnt) ent = __ldg(&tp.list[td.list_off + li + 1]);
        const unsigned er = g == 0 ? cur.y : (g == 1 ? cur.z : cur.w);
        if (er == 0xFFFFFFFFu) continue;                      // no voxel of this group sees receiver m
        // k-block range of item (q = lane, m): number of blocks and slot offset  r = ki + roff
        int lo;
        const int nb_l = tc_block_range(tr, er, lo);
        const int pk = pack_range(nb_l, tb_l - 4 * lo);
        const float4 el = __ldg(&P.elem[cur.x]);
        // per-(m, n): aperture, excess path, receive phase (as in das_tiled.cuh)
        const float dx = x - el.x, dy = y - el.y;
        const float rho2 = fmaf(dx, dx, dy * dy);
        const float lhs = tp.four_f2 * rho2;
        bool act = lhs <= a2e;
        if (fabsf(lhs - a2e) <= band) act = aperture_exact(x, y, el.x, el.y, P.zs, izc, tp.z_array, P.fnum);
        const float s2 = rho2 + a2;
        const float d = s2 * rsqrt_approx(s2);
        const float e = (rho2 * tp.kappa_f) * rcp_approx(a + d);
        float cyc = tp.ratio_f * e;
        cyc -= rintf(cyc);
        const float ang = 6.283185307179586f * cyc;
        const float pr = act ? cos_approx(ang) : 0.f, pi = act ? sin_approx(ang) : 0.f;
        produced = true;

#pragma unroll
        for (int q = 0; q < 16; ++q) {
          if (q < P.Q) {
            const int pk_q = __shfl_sync(0xffffffffu, pk, q);
            const int n_pass = range_nb(pk_q) >> 1;
            // fractional index: ki = floor(t) (round-to-nearest of t - 1/2), al = t - ki
            const float t = Tf[q] + e;
            const float u = (t - 0.5f) + kMagic;
            const float al = t - (u - kMagic);
            // slot of sample k inside the item's k-blocks:  r = ki + (tbase_q - 4 lo)
            int r = (int)__float_as_uint(u) + (range_lo(pk_q) - (int)kMagicBits);
            // weights: P = Ptx_q Prx_m;  W1 = al P (sample k + 1),  W0 = P - W1 (sample k)
            const float wre = fmaf(pc[q], pr, -ps[q] * pi), wim = fmaf(pc[q], pi, ps[q] * pr);
            const float w1re = al * wre, w1im = al * wim;
            unsigned w0 = pack_half2(wre - w1re, w1im - wim);                    // (Re W0, -Im W0)
            unsigned w1 = pack_half2(w1re, -w1im);
            if (td.edge) {
              // reading A6: the term is dropped unless 0 <= k <= K-2 (a pad sample may not lend its
              // neighbour a weight); only tiles whose windows touch the ends of the record get here
              const int tb_q = __shfl_sync(0xffffffffu, tb_l, q);
              const int ki = (int)(__float_as_uint(u) - kMagicBits);
              if ((unsigned)(ki + tb_q) > (unsigned)(P.K - 2)) { w0 = 0u; w1 = 0u; }
            }
#pragma unroll 1
            for (int p = 0; p < n_pass; ++p, r -= kTcBlk * kTcPassBlocks) {
              // the A row of this MMA: slot r holds W0, slot r + 1 holds W1, every other slot 0
              unsigned v[8];
#pragma unroll
              for (int i = 0; i < 8; ++i) v[i] = 0u;
#pragma unroll
              for (int i = -1; i < 8; ++i) {
                const bool hit = r == i;
                if (i >= 0) v[i] = hit ? w0 : v[i];
                if (i < 7) v[i + 1] = hit ? w1 : v[i + 1];
              }
              const unsigned buf = a_it & (kTcABufs - 1);
              // complete the previous A tile (its store has had the placement above to land)
              if (pend) {
                tmem_wait_st();
                tc_fence_before();
                if (lane0) mbar_arrive(pend);
              }
              mbar_wait(ae0 + 8u * buf, ((a_it / kTcABufs) & 1u) ^ 1u);
              tc_fence_after();
              tmem_st8(a_addr0 + buf * kTcACols, v);
              pend = af0 + 8u * buf;
              ++a_it;
            }
          }
        }
      }
      if (pend) {
        tmem_wait_st();
        tc_fence_before();
        if (lane0) mbar_arrive(pend);
        pend = 0;
      }

      // ---- epilogue: D (FP32, TMEM) -> out[frame][voxel] -------------------------------------
      mbar_wait(d_full, n_done & 1u);
      tc_fence_after();
      const long long vox = ((long long)ix * P.ny + iy) * P.nz + iz;
      float2* dst = out + (long long)chunk * tp.Bc * n_vox + vox;
      for (int c0 = 0; c0 < N; c0 += 16) {
        float v[16];
        tmem_ld16(d_addr + (unsigned)c0, v);
        tmem_wait_ld();
        if (in_grid) {
#pragma unroll
          for (int i = 0; i < 8; ++i)
            dst[(long long)(c0 / 2 + i) * n_vox] = produced ? make_float2(v[2 * i], v[2 * i + 1]) : make_float2(0.f, 0.f);
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(d_empty);
    }
  }

  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (warp == kTcGenWarps) tmem_dealloc(tmem, kTcTmemCols);
}

}  // namespace

cudaError_t launch_tc_kernel(const TcDev& tp, const Params& P, const void* d_conv, void* d_out, int grid, size_t smem, cudaStream_t s) {
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  tc_kernel<<<grid, kTcThreads, smem, s>>>(tp, P, static_cast<const unsigned char*>(d_conv), static_cast<float2*>(d_out));
  return cudaGetLastError();
}

}  // namespace das
