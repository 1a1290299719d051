// Frame-batch tensor-core delay-and-sum kernel (tcgen05 / TMEM); design notes in das_tc.cuh.
#include <climits>
#include <cstdlib>

#include "das_tc.cuh"

namespace das {

namespace {

// Ring state of one generator warp: the A tiles of its voxel group in tensor memory.
struct TcGenRing {
  unsigned a_it;        // passes written so far (slot = a_it mod depth, phase = a_it / depth)
  unsigned pend;        // a_full barrier of the A tile whose store is in flight (a sink while there is none)
  unsigned nab, nab_sh; // ring depth and its log2
  unsigned ae0, af0;    // first a_empty / a_full barrier of the group
  unsigned a_addr0;     // TMEM address of slot 0 for this warp's lane quarter
  bool lane0;
};

// One (q, m) item of a generator thread: the two packed weights, the slot of sample k, the passes.
struct TcItem { unsigned w0, w1; int r, n_pass; };

// The 16 items (q, m) of one receiver for one voxel row.  cw[] holds the 16 window codes of the group
// (two per word, loaded with one address for the whole warp: no shuffle in the chain).  The index and
// weight arithmetic runs on transmit PAIRS as packed FP32x2 instructions (FADD2 / FMUL2 / FFMA2, sm_100),
// and the pair after the current one is worked out before the stores of the current one, so that it
// fills the latency of the store / barrier sequence.  EDGE: the tile's windows touch the ends of the
// record (reading A6).  Tf2 / pc2 / ps2: (q = 2 j, q = 2 j + 1).
template <bool EDGE>
__device__ __forceinline__ void tc_gen_receiver(const float2 (&Tf2)[8], const float2 (&pc2)[8], const float2 (&ps2)[8],
                                                const float ex, const float pr, const float pi, const uint4 cw0,
                                                const uint4 cw1, const int tb_l, const int Q, const int K, TcGenRing& rg) {
  const unsigned cw[8] = {cw0.x, cw0.y, cw0.z, cw0.w, cw1.x, cw1.y, cw1.z, cw1.w};
  const float2 ex2 = make_float2(ex, ex), pr2 = make_float2(pr, pr), npr2 = make_float2(-pr, -pr);
  const float2 npi2 = make_float2(-pi, -pi);
  const float2 mh2 = make_float2(-0.5f, -0.5f), mg2 = make_float2(kMagic, kMagic), nmg2 = make_float2(-kMagic, -kMagic);
  auto item_pair = [&](const int jp, TcItem& i0, TcItem& i1) {
    const unsigned c0 = cw[jp] & 0xffffu, c1 = cw[jp] >> 16;
    i0.n_pass = code_passes(c0);
    i1.n_pass = code_passes(c1);
    // fractional index: ki = floor(t) (round-to-nearest of t - 1/2), al = t - ki
    const float2 t = __fadd2_rn(Tf2[jp], ex2);
    const float2 u = __fadd2_rn(__fadd2_rn(t, mh2), mg2);
    const float2 al = __ffma2_rn(__fadd2_rn(u, nmg2), make_float2(-1.f, -1.f), t);
    // slot of sample k inside the item's window:  r = ki - window start
    i0.r = (int)__float_as_uint(u.x) - (int)(kMagicBits + 2u * (unsigned)code_start2(c0));
    i1.r = (int)__float_as_uint(u.y) - (int)(kMagicBits + 2u * (unsigned)code_start2(c1));
    // weights: P = Ptx_q Prx_m;  W1 = al P (sample k + 1),  W0 = P - W1 (sample k); the imaginary parts
    // are carried negated (the A row holds (Re W, -Im W))
    const float2 wre = __ffma2_rn(pc2[jp], pr2, __fmul2_rn(ps2[jp], npi2));          //  Re P
    const float2 nwim = __ffma2_rn(pc2[jp], npi2, __fmul2_rn(ps2[jp], npr2));        // -Im P
    const float2 w1re = __fmul2_rn(al, wre), nw1im = __fmul2_rn(al, nwim);
    const float2 w0re = __ffma2_rn(w1re, make_float2(-1.f, -1.f), wre);
    const float2 nw0im = __ffma2_rn(nw1im, make_float2(-1.f, -1.f), nwim);
    i0.w0 = pack_half2(w0re.x, nw0im.x); i0.w1 = pack_half2(w1re.x, nw1im.x);
    i1.w0 = pack_half2(w0re.y, nw0im.y); i1.w1 = pack_half2(w1re.y, nw1im.y);
    if (EDGE) {
      // the term is dropped unless 0 <= k <= K-2 (a pad sample may not lend its neighbour a weight)
      const int tb0 = __shfl_sync(0xffffffffu, tb_l, min(2 * jp, Q - 1)), tb1 = __shfl_sync(0xffffffffu, tb_l, min(2 * jp + 1, Q - 1));
      const int k0 = (int)(__float_as_uint(u.x) - kMagicBits), k1 = (int)(__float_as_uint(u.y) - kMagicBits);
      if ((unsigned)(k0 + tb0) > (unsigned)(K - 2)) { i0.w0 = 0u; i0.w1 = 0u; }
      if ((unsigned)(k1 + tb1) > (unsigned)(K - 2)) { i1.w0 = 0u; i1.w1 = 0u; }
    }
  };
  auto passes = [&](const TcItem& cur) {
    int r = cur.r;
#pragma unroll 1
    for (int p = 0; p < cur.n_pass; ++p, r -= kTcBlk * kTcPassBlocks) {
      // the A row of this MMA: slot r holds W0, slot r + 1 holds W1, every other slot 0
      unsigned v[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) v[i] = 0u;
#pragma unroll
      for (int i = -1; i < 8; ++i) {
        const bool hit = r == i;
        if (i >= 0) v[i] = hit ? cur.w0 : v[i];
        if (i < 7) v[i + 1] = hit ? cur.w1 : v[i + 1];
      }
      const unsigned buf = rg.a_it & (rg.nab - 1u);
      // complete the previous A tile (its store has had the placement above to land)
      tmem_wait_st();
      tc_fence_before();
      if (rg.lane0) mbar_arrive(rg.pend);
      mbar_wait_park(rg.ae0 + 8u * buf, ((rg.a_it >> rg.nab_sh) & 1u) ^ 1u);
      tc_fence_after();
      tmem_st8(rg.a_addr0 + buf * kTcACols, v);
      rg.pend = rg.af0 + 8u * buf;
      ++rg.a_it;
    }
  };
  TcItem c0, c1;
  item_pair(0, c0, c1);
#pragma unroll
  for (int jp = 0; jp < 8; ++jp) {                               // items in transmit order, q = 2 jp, 2 jp + 1
    TcItem n0 = c0, n1 = c1;
    if (jp + 1 < 8) item_pair(jp + 1, n0, n1);
    passes(c0);
    passes(c1);
    c0 = n0; c1 = n1;
  }
}

// Work items: (chunk, tile), tile fastest; every warp role walks the same sequence.
__global__ void __launch_bounds__(kTcThreads, 1)
tc_kernel(const TcDev tp, const Params P, const unsigned char* __restrict__ convb, float2* __restrict__ out) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  TcSmemHeader& sm = *reinterpret_cast<TcSmemHeader*>(smem_raw);
  const unsigned stage0 = (smem_u32(smem_raw) + (unsigned)sizeof(TcSmemHeader) + 127u) & ~127u;
  const int N = 2 * tp.Bc;                                   // MMA N
  const unsigned slab = (unsigned)N * 16u;                   // bytes of one k-block: N columns x 8 FP16
  const unsigned stage_bytes = (unsigned)tp.stage_blocks * slab;   // one window slot; a stage has qs of them
  const unsigned qs = (unsigned)tp.qs;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_work = tp.n_tiles * tp.n_chunks;
  const long long n_vox = (long long)P.nx * P.ny * P.nz;
  const long long chunk_bytes = (long long)P.M * P.Q * tp.KBp * slab;
  const int ql = min(lane & 15, P.Q - 1);                    // the transmit this lane reads windows for

  const unsigned b_full0 = smem_u32(&sm.b_full[0]), b_empty0 = smem_u32(&sm.b_empty[0]);
  const unsigned a_full0 = smem_u32(&sm.a_full[0]), a_empty0 = smem_u32(&sm.a_empty[0]);
  const unsigned d_full = smem_u32(&sm.d_full), d_empty = smem_u32(&sm.d_empty);

  if (tid == 0) {
    for (int s = 0; s < kTcMaxStages; ++s) { mbar_init(b_full0 + 8 * s, 1); mbar_init(b_empty0 + 8 * s, kTcG); }
    for (int i = 0; i < kTcMaxABufs * kTcG; ++i) { mbar_init(a_full0 + 8 * i, 4); mbar_init(a_empty0 + 8 * i, 1); }
    mbar_init(d_full, kTcG);
    mbar_init(d_empty, kTcGenWarps);
    mbar_init(smem_u32(&sm.sink), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == kTcGenWarps) tmem_alloc(smem_u32(&sm.tmem_base), kTcTmemCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const unsigned tmem = sm.tmem_base;
  // TMEM columns: D of group g at g * N; A buffer (g, buf) at kTcG * N + (a_bufs g + buf) * kTcACols
  const unsigned a_col0 = (unsigned)(kTcG * N);
  const unsigned nab = (unsigned)tp.a_bufs, nab_sh = (unsigned)tp.a_shift;   // A ring depth (power of two)
  // The accumulators start from zero and the epilogue leaves them zero again, so every MMA accumulates
  // and no MMA has to be the first of its tile.
  if (warp < kTcGenWarps) {
    const unsigned d0 = tmem + (((unsigned)((warp & 3) * 32)) << 16) + (unsigned)((warp >> 2) * N);
    for (int c0 = 0; c0 < N; c0 += 8) tmem_st8_zero(d0 + (unsigned)c0);
    tmem_wait_st();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  if (warp == kTcGenWarps) {
    // ===================================== TMA PRODUCER =======================================
    // A stage holds the windows of `qs` consecutive transmits of one receiver (one barrier round
    // per qs items).  Lane q works out the window of item (q, m), the union over the voxel groups,
    // and issues its own bulk copy; lane 0 waits for the stage and posts the byte count.
    unsigned s = 0, ph = 0;                                  // stage and its phase parity
    const bool has_q = lane < P.Q;
    for (int work = blockIdx.x; work < n_work; work += gridDim.x) {
      const int tile_i = work % tp.n_tiles, chunk = work / tp.n_tiles;
      const TcTile td = tp.tiles[tile_i];
      const unsigned char* base = convb + (long long)chunk * chunk_bytes;
      const int tb4 = __ldg(&tp.tbase[(long long)tile_i * P.Q + ql]) >> 2;       // k-block of tbase_q
      // window of item (q = lane, m) of a list entry: byte offset inside the chunk and length; fetched
      // one entry ahead (the loads are a dependent chain through L2)
      auto entry_window = [&](const long long e, unsigned& any, unsigned& bytes) {
        const uint2 hd = __ldg(&tp.list[e]);
        any = hd.y;
        int wlo, wn;
        tc_union_window(tp.codes + e * kTcG * 16 + ql, wlo, wn);
        bytes = has_q ? (unsigned)wn * slab : 0u;
        return ((long long)hd.x * P.Q * tp.KBp + kTcPadBlocks + (long long)ql * tp.KBp + tb4 + wlo) * (long long)slab;
      };
      unsigned any_n = 0, bytes_n = 0;
      long long src_n = 0;
      if (td.list_cnt) src_n = entry_window(td.list_off, any_n, bytes_n);
      for (int li = 0; li < td.list_cnt; ++li) {
        const unsigned any = any_n, bytes_l = bytes_n;
        const long long src_l = src_n;
        if (li + 1 < td.list_cnt) src_n = entry_window((long long)td.list_off + li + 1, any_n, bytes_n);
        if (!any) continue;
        for (int q0 = 0; q0 < P.Q; q0 += (int)qs) {
          const bool mine = lane >= q0 && lane < q0 + (int)qs;
          const unsigned total = __reduce_add_sync(0xffffffffu, mine ? bytes_l : 0u);
          if (lane == 0) {
            mbar_wait_park(b_empty0 + 8 * s, ph ^ 1u);
            if (total) mbar_arrive_expect_tx(b_full0 + 8 * s, total);
            else mbar_arrive(b_full0 + 8 * s);
          }
          __syncwarp();
          if (mine && bytes_l)
            tma_bulk_g2s(stage0 + (s * qs + (unsigned)(lane - q0)) * stage_bytes, base + src_l, bytes_l, b_full0 + 8 * s);
          if (++s == (unsigned)tp.n_stages) { s = 0; ph ^= 1u; }
          __syncwarp();
        }
      }
    }
  } else if (warp > kTcGenWarps) {
    // ===================================== MMA ISSUERS ========================================
    // One warp per voxel group.  The issue loop is a serial chain (wait -> MMA -> commit) whose
    // latency bounds the MMA rate of a group, so it is kept as short as it can be: lane q prepares
    // item (q, m) (passes, offset of the group's window inside the staged one), every lane runs the
    // same scalar loop (no divergence, one shuffle per item), only the tcgen05 instructions sit
    // under an elected lane, and the stage barriers are visited once per qs items.
    const int g = warp - kTcGenWarps - 1;
    const unsigned idesc = tc_idesc(N);
    const unsigned d_tmem = tmem + (unsigned)(g * N);
    const unsigned a_tmem0 = tmem + a_col0 + (nab * (unsigned)g) * kTcACols;
    const unsigned af0 = a_full0 + 8u * (nab * (unsigned)g), ae0 = a_empty0 + 8u * (nab * (unsigned)g);
    // descriptor of a B tile at shared address 0: LBO = one slab (the two K chunks), SBO = 128 B
    const unsigned long long desc0 = tc_smem_desc(0u, slab, 128);
    unsigned s = 0, ph = 0, a_it = 0, n_done = 0;
    for (int work = blockIdx.x; work < n_work; work += gridDim.x, ++n_done) {
      const int tile_i = work % tp.n_tiles;
      const TcTile td = tp.tiles[tile_i];
      mbar_wait_park(d_empty, (n_done & 1u) ^ 1u);             // epilogue of the previous tile has drained D
      tc_fence_after();
      // item (q = lane, m) of a list entry: passes | 16-byte units from the start of the staged window to
      // this group's window << 2; fetched one entry ahead (the loads are a dependent chain through L2)
      auto entry_info = [&](const long long e, unsigned& any) {
        any = __ldg(&tp.list[e]).y;
        int wlo, wn;
        tc_union_window(tp.codes + e * kTcG * 16 + ql, wlo, wn);
        const unsigned c = __ldg(&tp.codes[(e * kTcG + g) * 16 + ql]);
        return (unsigned)code_passes(c) | ((code_passes(c) ? (unsigned)((code_start2(c) >> 1) - wlo) * (slab >> 4) : 0u) << 2);
      };
      unsigned any_n = 0, info_n = 0;
      if (td.list_cnt) info_n = entry_info(td.list_off, any_n);
      for (int li = 0; li < td.list_cnt; ++li) {
        const unsigned any = any_n, info_l = info_n;
        if (li + 1 < td.list_cnt) info_n = entry_info((long long)td.list_off + li + 1, any_n);
        if (!any) continue;
        for (int q0 = 0; q0 < P.Q; q0 += (int)qs) {
          mbar_wait_park(b_full0 + 8 * s, ph);                 // also keeps an idle group in step with the ring
          const int q1 = min(q0 + (int)qs, P.Q);
          for (int q = q0; q < q1; ++q) {
            const unsigned info = __shfl_sync(0xffffffffu, info_l, q);
            const int np = (int)(info & 3u);
            unsigned long long desc = desc0 + (unsigned long long)(((stage0 + (s * qs + (unsigned)(q - q0)) * stage_bytes) >> 4) + (info >> 2));
            for (int p = 0; p < np; ++p, ++a_it, desc += (unsigned long long)((kTcPassBlocks * slab) >> 4)) {
              const unsigned buf = a_it & (nab - 1u);
              mbar_wait_park(af0 + 8u * buf, (a_it >> nab_sh) & 1u);
              tc_fence_after();
              if (tc_elect()) {
                tc_mma_ts(d_tmem, a_tmem0 + buf * kTcACols, desc, idesc, 1u);
                tc_commit(ae0 + 8u * buf);                     // A buffer free once this MMA has read it
              }
            }
          }
          if (tc_elect()) tc_commit(b_empty0 + 8 * s);         // this group is done with the stage
          if (++s == (unsigned)tp.n_stages) { s = 0; ph ^= 1u; }
        }
      }
      if (tc_elect()) tc_commit(d_full);                       // this group's MMAs of the tile are complete
    }
  } else {
    // ===================================== GENERATORS =========================================
    const int g = warp >> 2;                                  // voxel group = depth inside the tile
    const int row = (warp & 3) * 32 + lane;                   // MMA row = TMEM lane (quarter warp % 4)
    const unsigned lane_base = ((unsigned)((warp & 3) * 32)) << 16;
    const unsigned d_addr = tmem + lane_base + (unsigned)(g * N);
    const unsigned a_addr0 = tmem + lane_base + a_col0 + (nab * (unsigned)g) * kTcACols;
    TcGenRing rg;
    rg.a_it = 0;
    rg.pend = smem_u32(&sm.sink);
    rg.nab = nab; rg.nab_sh = nab_sh;
    rg.ae0 = a_empty0 + 8u * (nab * (unsigned)g); rg.af0 = a_full0 + 8u * (nab * (unsigned)g);
    rg.a_addr0 = a_addr0;
    rg.lane0 = lane == 0;
    unsigned n_done = 0;

    for (int work = blockIdx.x; work < n_work; work += gridDim.x, ++n_done) {
      const int tile_i = work % tp.n_tiles, chunk = work / tp.n_tiles;
      const TcTile td = tp.tiles[tile_i];
      const TcVoxel vx = tc_voxel(tp, P, td, row, g);
      const int tb_l = __ldg(&tp.tbase[(long long)tile_i * P.Q + ql]);

      // per-(q, n) part in FP64: reduced transmit delay and transmit phase factor
      float2 Tf[8], pc[8], ps[8];                               // (q = 2 j, q = 2 j + 1)
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const int qq = min(j, P.Q - 1);
        const double T = tc_T(P, vx, qq);
        const float tf = (float)(T - (double)__ldg(&tp.tbase[(long long)tile_i * P.Q + qq]));
        double cyc = tp.phase0 + tp.ratio * T;
        cyc -= rint(cyc);
        const float ang = 6.283185307179586f * (float)cyc;
        if (j & 1) { Tf[j >> 1].y = tf; pc[j >> 1].y = cos_approx(ang); ps[j >> 1].y = sin_approx(ang); }
        else       { Tf[j >> 1].x = tf; pc[j >> 1].x = cos_approx(ang); ps[j >> 1].x = sin_approx(ang); }
      }

      // the list entry one iteration ahead: header, the group's 16 window codes, receiver position
      uint2 hd_n = make_uint2(0u, 0u);
      uint4 cw0_n = make_uint4(0u, 0u, 0u, 0u), cw1_n = cw0_n;
      float4 el_n = make_float4(0.f, 0.f, 0.f, 0.f);
      if (td.list_cnt) {
        const uint4* cp = reinterpret_cast<const uint4*>(tp.codes + ((long long)td.list_off * kTcG + g) * 16);
        hd_n = __ldg(&tp.list[td.list_off]);
        cw0_n = __ldg(cp); cw1_n = __ldg(cp + 1);
        el_n = __ldg(&P.elem[hd_n.x]);
      }
      for (int li = 0; li < td.list_cnt; ++li) {
        const uint2 hd = hd_n;
        const uint4 cw0 = cw0_n, cw1 = cw1_n;
        const float4 el = el_n;
        if (li + 1 < td.list_cnt) {
          const long long e = td.list_off + li + 1;
          const uint4* cp = reinterpret_cast<const uint4*>(tp.codes + (e * kTcG + g) * 16);
          hd_n = __ldg(&tp.list[e]);
          cw0_n = __ldg(cp); cw1_n = __ldg(cp + 1);
          el_n = __ldg(&P.elem[hd_n.x]);
        }
        if (!((hd.y >> g) & 1u)) continue;                    // no voxel of this group sees receiver m
        // per-(m, n): aperture, excess path, receive phase (as in das_tiled.cuh)
        bool act;
        const float ex = tc_excess(tp, P, vx, el, act);
        float cyc = tp.ratio_f * ex;
        cyc -= rintf(cyc);
        const float ang = 6.283185307179586f * cyc;
        const float pr = act ? cos_approx(ang) : 0.f, pi = act ? sin_approx(ang) : 0.f;
        if (td.edge) tc_gen_receiver<true>(Tf, pc, ps, ex, pr, pi, cw0, cw1, tb_l, P.Q, P.K, rg);
        else tc_gen_receiver<false>(Tf, pc, ps, ex, pr, pi, cw0, cw1, tb_l, P.Q, P.K, rg);
      }
      tmem_wait_st();
      tc_fence_before();
      if (rg.lane0) mbar_arrive(rg.pend);
      rg.pend = smem_u32(&sm.sink);

      // ---- epilogue: D (FP32, TMEM) -> out[frame][voxel] -------------------------------------
      mbar_wait_park(d_full, n_done & 1u);
      tc_fence_after();
      const long long vox = ((long long)vx.ix * P.ny + vx.iy) * P.nz + vx.iz;
      float2* dst = out + (long long)chunk * tp.Bc * n_vox + vox;
      for (int c0 = 0; c0 < N; c0 += 16) {
        float v[16];
        tmem_ld16(d_addr + (unsigned)c0, v);
        tmem_wait_ld();
        if (vx.in_grid) {
#pragma unroll
          for (int i = 0; i < 8; ++i)
            dst[(long long)(c0 / 2 + i) * n_vox] = make_float2(v[2 * i], v[2 * i + 1]);
        }
        tmem_st8_zero(d_addr + (unsigned)c0);                  // leave the accumulator zero for the next tile
        tmem_st8_zero(d_addr + (unsigned)c0 + 8u);
      }
      tmem_wait_st();
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

// ---- plan-time window kernel -------------------------------------------------------------------
// One CTA per tile, thread = (voxel group, MMA row).  For every listed receiver m and transmit q
// it takes the minimum and maximum of floor(t_qmn) over the ACTIVE voxels of each group, with the
// same FP32 arithmetic as the generator warps (tc_voxel / tc_T / tc_excess) widened by kTcDelta,
// and writes the window code the three warp roles of tc_kernel read (TcDev::codes).
//   stats[0] = largest staged window (k-blocks), stats[1] = error bits
//   (1: window needs more than 3 passes, 2: window leaves the zero pads, 4: negative start)
__global__ void __launch_bounds__(kTcG * kTcRows)
tc_window_kernel(const TcDev tp, const Params P, uint2* __restrict__ list, unsigned short* __restrict__ codes,
                 int* __restrict__ tile_work, int* __restrict__ tile_edge, int* __restrict__ stats) {
  __shared__ int kmn[kTcG][16], kmx[kTcG][16];
  const int tile_i = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
  const int g = tid / kTcRows, row = tid % kTcRows;
  const TcTile td = tp.tiles[tile_i];
  const TcVoxel vx = tc_voxel(tp, P, td, row, g);
  const int Kb = (P.K + kTcBlk - 1) / kTcBlk;
  float Tf[16];
#pragma unroll
  for (int q = 0; q < 16; ++q) {
    const int qq = min(q, P.Q - 1);
    Tf[q] = (float)(tc_T(P, vx, qq) - (double)__ldg(&tp.tbase[(long long)tile_i * P.Q + qq]));
  }
  const int tb4 = tid < 16 ? (__ldg(&tp.tbase[(long long)tile_i * P.Q + min(tid, P.Q - 1)]) >> 2) : 0;
  int work = 0, edge = 0, stage = 0, err = 0;

  for (int li = 0; li < td.list_cnt; ++li) {
    const long long e = td.list_off + li;
    if (tid < kTcG * 16) { kmn[tid / 16][tid % 16] = INT_MAX; kmx[tid / 16][tid % 16] = INT_MIN; }
    __syncthreads();
    const float4 el = __ldg(&P.elem[list[e].x]);
    bool act;
    const float ex = tc_excess(tp, P, vx, el, act);
#pragma unroll
    for (int q = 0; q < 16; ++q) {
      if (q < P.Q) {
        const float t = Tf[q] + ex;
        int lo = act ? (int)floorf(t - kTcDelta) : INT_MAX, hi = act ? (int)floorf(t + kTcDelta) : INT_MIN;
        lo = __reduce_min_sync(0xffffffffu, lo);
        hi = __reduce_max_sync(0xffffffffu, hi);
        if (lane == 0 && lo != INT_MAX) { atomicMin(&kmn[g][q], lo); atomicMax(&kmx[g][q], hi); }
      }
    }
    __syncthreads();
    if (tid < 16) {
      const int q = tid;
      int wlo = INT_MAX, whi = INT_MIN;
      unsigned flags = 0;
      for (int gg = 0; gg < kTcG; ++gg) {
        unsigned code = 0;
        if (q < P.Q && kmn[gg][q] != INT_MAX) {
          const int smin = kmn[gg][q], smax = kmx[gg][q];
          if (smin < 0) err |= 4;
          const int b0 = max(smin, 0) >> 2;
          const int nb = ((smax + 1) >> 2) - b0 + 1;
          const int np = (nb + kTcPassBlocks - 1) / kTcPassBlocks;
          if (np > 3 || b0 * 2 > 0x3fff) err |= 1;
          code = (unsigned)min(np, 3) | ((unsigned)(b0 * 2) << 2);
          wlo = min(wlo, tb4 + b0);
          whi = max(whi, tb4 + b0 + kTcPassBlocks * np);
          flags |= 1u << gg;
          work += np;
        }
        codes[(e * kTcG + gg) * 16 + q] = (unsigned short)code;
      }
      if (whi > wlo) {
        stage = max(stage, whi - wlo);
        if (wlo < -kTcPadBlocks || whi > Kb + kTcPadBlocks) err |= 2;
        if (kTcBlk * wlo <= 0 || kTcBlk * whi >= P.K - 1) edge = 1;
      }
      flags = __reduce_or_sync(0x0000ffffu, flags);
      if (tid == 0) list[e].y = flags;
    }
    __syncthreads();                                          // kmn / kmx are re-initialised at the loop top
  }
  if (tid < 16) {
    work = __reduce_add_sync(0x0000ffffu, work);
    edge = __reduce_or_sync(0x0000ffffu, edge);
    stage = __reduce_max_sync(0x0000ffffu, stage);
    err = __reduce_or_sync(0x0000ffffu, err);
    if (tid == 0) {
      tile_work[tile_i] = work;
      tile_edge[tile_i] = edge;
      atomicMax(&stats[0], stage);
      if (err) atomicOr(&stats[1], err);
    }
  }
}

}  // namespace

cudaError_t launch_tc_windows(const TcDev& tp, const Params& P, uint2* list, unsigned short* codes, int* tile_work,
                              int* tile_edge, int* stats, cudaStream_t s) {
  tc_window_kernel<<<tp.n_tiles, kTcG * kTcRows, 0, s>>>(tp, P, list, codes, tile_work, tile_edge, stats);
  return cudaGetLastError();
}

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
