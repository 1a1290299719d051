// Frame-batch tensor-core delay-and-sum kernel (tcgen05 / TMEM); design notes in das_tc.cuh.
#include <climits>
#include <cstdlib>

#include <cuda.h>

#include "das_tc.cuh"

namespace das {

namespace {

// Cycle accounting of the barrier waits per warp role (compile with -DDAS_TC_PROF, run with DAS_TC_PROF=1):
// prof[cta][warp][k]: k = 0 total cycles of the role loop, 1..6 cycles spent in the waits listed at the use sites.
#ifdef DAS_TC_PROF
#define TC_PROF_DECL unsigned long long pf_[8] = {0, 0, 0, 0, 0, 0, 0, 0}; const long long pf_t0_ = clock64();
#define TC_PROF_WAIT(k, stmt) { const long long c0_ = clock64(); stmt; pf_[k] += (unsigned long long)(clock64() - c0_); }
#define TC_PROF_END if (tp.prof && lane == 0) { pf_[0] = (unsigned long long)(clock64() - pf_t0_); for (int k_ = 0; k_ < 8; ++k_) tp.prof[((long long)blockIdx.x * 32 + warp) * 8 + k_] = pf_[k_]; }
#else
#define TC_PROF_DECL
#define TC_PROF_WAIT(k, stmt) { stmt; }
#define TC_PROF_END
#endif

// State of one generator warp: the A slots of its voxel group in tensor memory (das_tc.cuh).
struct TcGenState {
  unsigned a_addr0;     // TMEM address of slot 0 for this warp's lane quarter
  unsigned tbl0;        // shared-memory address of row r = 0 of the placement table
  unsigned af0, ae0;    // a_full / a_empty barrier of slot 0 of the group (shared-memory addresses)
  unsigned pend;        // a_full barrier of the item tile whose store is in flight (the sink while there is none)
  unsigned pend2;       // the same for the overflow tile
  unsigned sink;
  unsigned par;         // bit s: phase parity of the next use of slot s (bit kTcOvf: the overflow slot)
  unsigned it;          // item tiles stored so far (slot = it mod 4 when the transmit count is not 16)
#ifdef DAS_TC_PROF
  unsigned long long pf1, pf2, pf3;
#endif
  bool free_next;       // the next item's slot was seen free by the probe issued one item ahead
};

// One (q, m) item of a generator thread: the two packed weights, the shared-memory address of the placement-table row of
// slot r (sample k sits in slot r of the item's window), the passes.
struct TcItem { unsigned w0, w1, ra; int n_pass; };

// The A row of one MMA pass: slot r holds W0, slot r + 1 holds W1, every other slot 0.  `ra` addresses row r of the
// placement table (das_tc.cuh): 9 words, word j = {1,1} iff r == j - 1, so slot i = W0 * word[i + 1] + W1 * word[i].
// The loads are plain (non-volatile) asm: the table never changes, so they may be scheduled across the barrier operations.
__device__ __forceinline__ void tc_place(const unsigned ra, const unsigned w0, const unsigned w1, unsigned (&v)[8]) {
  unsigned t[9];
  asm("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(t[0]), "=r"(t[1]), "=r"(t[2]), "=r"(t[3]) : "r"(ra));
  asm("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4+16];" : "=r"(t[4]), "=r"(t[5]), "=r"(t[6]), "=r"(t[7]) : "r"(ra));
  asm("ld.shared.u32 %0, [%1+32];" : "=r"(t[8]) : "r"(ra));
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    unsigned m;
    asm("mul.rn.f16x2 %0, %1, %2;" : "=r"(m) : "r"(w1), "r"(t[i]));
    asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(v[i]) : "r"(w0), "r"(t[i + 1]), "r"(m));
  }
}

// One NON-BLOCKING probe of an mbarrier phase (test_wait: a scoreboarded read, unlike try_wait, which
// suspends the warp for 60-150 cycles even when the phase has long completed).  The result is consumed
// an item later, so the probe's latency overlaps the placement arithmetic.
__device__ __forceinline__ bool mbar_test(unsigned bar, unsigned parity) {
  unsigned ok;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ unsigned lds_volatile(unsigned addr) {
  unsigned v;
  asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
// Two mbarrier arrivals by ONE elected lane of the (converged) warp: the a_full barriers of the item tile and of the
// overflow tile whose stores have just been seen complete (the sink barrier when there is none).
__device__ __forceinline__ void mbar_arrive2_elect(unsigned bar0, unsigned bar1) {
  asm volatile("{\n\t.reg .pred p;\n\t.reg .b64 st;\n\telect.sync _|p, 0xffffffff;\n\t"
               "@p mbarrier.arrive.shared::cta.b64 st, [%0];\n\t@p mbarrier.arrive.shared::cta.b64 st, [%1];\n\t}"
               ::"r"(bar0), "r"(bar1) : "memory");
}

// Hand item I of the current receiver to the MMA issuer.  With 16 transmits per receiver (Q16) the slot
// S = I mod 4 and the barrier phases are compile-time constants.  Order of events:
//   placement of this item | completion of the PREVIOUS item's stores (they have had the placement to land) and
//   their publication | slot S free? (probed one item ahead) | store | probe of the next item's slot.
// The second pass of a wide window (13 % of the items at the headline) goes through the overflow slot on a path of
// its own, so that a one-pass item pays nothing for it.
template <bool ZERO, bool Q16, int I>
__device__ __forceinline__ void tc_gen_item(const TcItem& cur, TcGenState& st) {
  const unsigned S = Q16 ? (unsigned)(I & (kTcSlots - 1)) : (st.it & (unsigned)(kTcSlots - 1));
  const unsigned pe = Q16 ? (unsigned)(((I / kTcSlots) & 1) ^ 1) : (((st.par >> S) & 1u) ^ 1u);
  unsigned v[8];
  if (!ZERO) tc_place(cur.ra, cur.w0, cur.w1, v);
#ifdef DAS_TC_PROF
  { const long long c0_ = clock64(); tmem_wait_st(); st.pf3 += (unsigned long long)(clock64() - c0_); }
#else
  tmem_wait_st();
#endif
  tc_fence_before();
  mbar_arrive2_elect(st.pend, st.pend2);
  st.pend2 = st.sink;
#ifdef DAS_TC_PROF
  if (!st.free_next) { const long long c0_ = clock64(); mbar_wait_park(st.ae0 + 8u * S, pe); st.pf1 += (unsigned long long)(clock64() - c0_); }
#else
  if (!st.free_next) mbar_wait_park(st.ae0 + 8u * S, pe);
#endif
  tc_fence_after();
  if (ZERO) tmem_st8_zero(st.a_addr0 + S * kTcACols); else tmem_st8(st.a_addr0 + S * kTcACols, v);
  st.pend = st.af0 + 8u * S;
  if (!Q16) { st.par ^= 1u << S; ++st.it; }
  {
    // probe the slot of the next item (of this receiver or of the next one)
    const unsigned Sn = Q16 ? (unsigned)((I + 1) & (kTcSlots - 1)) : (st.it & (unsigned)(kTcSlots - 1));
    const unsigned pn = Q16 ? (unsigned)(((((I + 1) & 15) / kTcSlots) & 1) ^ 1) : (((st.par >> Sn) & 1u) ^ 1u);
    st.free_next = mbar_test(st.ae0 + 8u * Sn, pn);
  }
  if (cur.n_pass > 1) {
    if (!ZERO) tc_place(cur.ra - (unsigned)(kTcPass * kTcPlaceWords * 4), cur.w0, cur.w1, v);
    const unsigned po = ((st.par >> kTcOvf) & 1u) ^ 1u;
#ifdef DAS_TC_PROF
    if (!mbar_test(st.ae0 + 8u * kTcOvf, po)) { const long long c0_ = clock64(); mbar_wait_park(st.ae0 + 8u * kTcOvf, po); st.pf2 += (unsigned long long)(clock64() - c0_); }
#else
    if (!mbar_test(st.ae0 + 8u * kTcOvf, po)) mbar_wait_park(st.ae0 + 8u * kTcOvf, po);
#endif
    st.par ^= 1u << kTcOvf;
    tc_fence_after();
    if (ZERO) tmem_st8_zero(st.a_addr0 + kTcOvf * kTcACols); else tmem_st8(st.a_addr0 + kTcOvf * kTcACols, v);
    st.pend2 = st.af0 + 8u * kTcOvf;
  }
}

// The 16 items (q, m) of one receiver for one voxel row.  cw[] holds the 16 window codes of the group
// (two per word, loaded with one address for the whole warp: no shuffle in the chain).  The index and
// weight arithmetic runs on transmit PAIRS as packed FP32x2 instructions (FADD2 / FMUL2 / FFMA2, sm_100),
// and the pair after the current one is worked out before the stores of the current one, so that it
// fills the latency of the store / barrier sequence.  EDGE: the tile's windows touch the ends of the
// record (reading A6).  ZERO: no voxel of this warp sees the receiver (all rows are zero: only the
// slot protocol runs).  Q16: 16 transmits, every slot is used 4 times per receiver, so the barrier
// phases are compile-time constants.  Tf2 / pc2 / ps2: (q = 2 j, q = 2 j + 1).
template <bool EDGE, bool ZERO, bool Q16>
__device__ __forceinline__ void tc_gen_receiver(const float2 (&Tf2)[8], const float2 (&pc2)[8], const float2 (&ps2)[8],
                                                const float ex, const float pr, const float pi, const unsigned am, const uint4 cw0,
                                                const uint4 cw1, const int tb_l, const int Q, const int K, TcGenState& st) {
  const unsigned cw[8] = {cw0.x, cw0.y, cw0.z, cw0.w, cw1.x, cw1.y, cw1.z, cw1.w};
  const float2 ex2 = make_float2(ex, ex), pr2 = make_float2(pr, pr), npr2 = make_float2(-pr, -pr);
  const float2 npi2 = make_float2(-pi, -pi);
  const float2 mh2 = make_float2(-0.5f, -0.5f), mg2 = make_float2(kMagic, kMagic), nmg2 = make_float2(-kMagic, -kMagic);
  auto item_pair = [&](const int jp, TcItem& i0, TcItem& i1) {
    const unsigned c0 = cw[jp] & 0xffffu, c1 = cw[jp] >> 16;
    i0.n_pass = code_passes(c0);
    i1.n_pass = code_passes(c1);
    if (ZERO) return;
    // fractional index: ki = floor(t) (round-to-nearest of t - 1/2), al = t - ki
    const float2 t = __fadd2_rn(Tf2[jp], ex2);
    const float2 u = __fadd2_rn(__fadd2_rn(t, mh2), mg2);
    const float2 al = __ffma2_rn(__fadd2_rn(u, nmg2), make_float2(-1.f, -1.f), t);
    // slot of sample k inside the item's window:  r = ki - window start
    // (a thread outside the aperture has zero weights and an arbitrary index: `am` = 0 sends it to row 0)
    i0.ra = st.tbl0 + (unsigned)(kTcPlaceWords * 4) * ((__float_as_uint(u.x) - (kMagicBits + (unsigned)code_start(c0))) & am);
    i1.ra = st.tbl0 + (unsigned)(kTcPlaceWords * 4) * ((__float_as_uint(u.y) - (kMagicBits + (unsigned)code_start(c1))) & am);
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
  TcItem c0, c1;
  c0.w0 = c0.w1 = c1.w0 = c1.w1 = 0u; c0.ra = c1.ra = st.tbl0;
  item_pair(0, c0, c1);
#define DAS_TC_PAIR(JP)                                                        \
  {                                                                            \
    TcItem n0 = c0, n1 = c1;                                                   \
    if (JP + 1 < 8) item_pair(JP + 1, n0, n1);                                 \
    if (Q16 || c0.n_pass) tc_gen_item<ZERO, Q16, 2 * JP>(c0, st);              \
    if (Q16 || c1.n_pass) tc_gen_item<ZERO, Q16, 2 * JP + 1>(c1, st);          \
    c0 = n0; c1 = n1;                                                          \
  }
  DAS_TC_PAIR(0) DAS_TC_PAIR(1) DAS_TC_PAIR(2) DAS_TC_PAIR(3)
  DAS_TC_PAIR(4) DAS_TC_PAIR(5) DAS_TC_PAIR(6) DAS_TC_PAIR(7)
#undef DAS_TC_PAIR
}

// Work items: (chunk, tile), tile fastest; every warp role walks the same sequence.
__global__ void __launch_bounds__(kTcThreads, 1)
tc_kernel(const TcDev tp, const Params P, const __grid_constant__ CUtensorMap tmap_small,
          const __grid_constant__ CUtensorMap tmap_big, float2* __restrict__ out) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  TcSmemHeader& sm = *reinterpret_cast<TcSmemHeader*>(smem_raw);
  const unsigned stage0 = (smem_u32(smem_raw) + (unsigned)sizeof(TcSmemHeader) + 1023u) & ~1023u;
  const int N = 2 * tp.Bc;                                   // MMA N
  const unsigned stage_bytes = tc_box_bytes(tp.Bc, kTcBoxBig);    // one window slot holds one box; a stage has qs of them
  const unsigned small_bytes = tc_box_bytes(tp.Bc, kTcBoxSmall);
  const unsigned qs = (unsigned)tp.qs;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_work = tp.n_tiles * tp.n_chunks;
  const long long n_vox = (long long)P.nx * P.ny * P.nz;
  const int ql = min(lane & 15, P.Q - 1);                    // the transmit this lane reads windows for
  // 16 transmits and no weight table: every receiver of a group has all 16 items, so the A-slot phases are
  // compile-time constants (Q16 path).  With a weight table single items may be missing (nobody lists them): the
  // general path, which tracks the slots at run time, takes those plans.
  const bool q16 = P.Q == 16 && P.wtx_tab == nullptr;

  // barrier addresses: taken once through an opaque move so that ptxas keeps them in registers instead of
  // rebuilding the shared-window base (S2UR + ULEA) at every use
  unsigned b_full0, b_empty0, a_full0, a_empty0, d_full, d_empty, sinkb;
  asm volatile("mov.u32 %0, %1;" : "=r"(b_full0) : "r"(smem_u32(&sm.b_full[0])));
  asm volatile("mov.u32 %0, %1;" : "=r"(b_empty0) : "r"(smem_u32(&sm.b_empty[0])));
  asm volatile("mov.u32 %0, %1;" : "=r"(a_full0) : "r"(smem_u32(&sm.a_full[0])));
  asm volatile("mov.u32 %0, %1;" : "=r"(a_empty0) : "r"(smem_u32(&sm.a_empty[0])));
  asm volatile("mov.u32 %0, %1;" : "=r"(d_full) : "r"(smem_u32(&sm.d_full)));
  asm volatile("mov.u32 %0, %1;" : "=r"(d_empty) : "r"(smem_u32(&sm.d_empty)));
  asm volatile("mov.u32 %0, %1;" : "=r"(sinkb) : "r"(smem_u32(&sm.sink)));

  if (tid == 0) {
    for (int s = 0; s < kTcMaxStages; ++s) { mbar_init(b_full0 + 8 * s, 1); mbar_init(b_empty0 + 8 * s, kTcG); }
    for (int i = 0; i < kTcABufs * kTcG; ++i) { mbar_init(a_full0 + 8 * i, 4); mbar_init(a_empty0 + 8 * i, 1); }
    mbar_init(d_full, kTcG);
    mbar_init(d_empty, kTcGenWarps);
    mbar_init(sinkb, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == kTcGenWarps) tmem_alloc(smem_u32(&sm.tmem_base), kTcTmemCols);
  for (int i = tid; i < kTcPlaceRows * kTcPlaceWords; i += kTcThreads)
    sm.place[i / kTcPlaceWords][i % kTcPlaceWords] = (i / kTcPlaceWords + kTcPlaceLo == i % kTcPlaceWords - 1) ? 0x3C003C00u : 0u;
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const unsigned tmem = sm.tmem_base;
  // TMEM columns: D of group g at g * N; A slot (g, s) at kTcG * N + (kTcABufs g + s) * kTcACols
  const unsigned a_col0 = (unsigned)(kTcG * N);
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

  // 512 threads x 128 registers: every role keeps its full share (no setmaxnreg; the service warps spill at 40)
  if (warp == kTcGenWarps) {
    // ===================================== TMA PRODUCER =======================================
    // A stage holds the windows of `qs` consecutive transmits of one receiver (one barrier round
    // per qs items).  Lane q works out the window of item (q, m), the union over the voxel groups,
    // and issues its own bulk copy; lane 0 waits for the stage and posts the byte count.  Lane q also
    // tells the MMA issuers what to do with item (q, m): one word per voxel group in the stage's info
    // block (passes | offset of the group's window inside the staged one), published by the stage's
    // full barrier.  Bit 31 of a stage's first info word marks the last stage of a tile.
    unsigned s = 0, ph = 0;                                  // stage and its phase parity
    const bool has_q = lane < P.Q;
    // quad pacing (below): what lanes 1..3 may still spend waiting for their partner CTA.  A wait that runs its
    // budget out quarters it, so a partner that is not there (not co-resident: an SM limit, a kernel of another
    // stream on its SM; or simply far behind) costs this CTA about 5 300 polls per LAUNCH (a few ms), not 4 000
    // per paced receiver, and after six expiries the lane stops looking at that partner.
    int pace_budget = 4000;
    TC_PROF_DECL
    for (int work = blockIdx.x; work < n_work; work += gridDim.x) {
      const int tile_i = work % tp.n_tiles, chunk = work / tp.n_tiles;
      const TcTile td = tp.tiles[tile_i];
      const int tb_q = __ldg(&tp.tbase[(long long)tile_i * P.Q + ql]);
      // item (q = lane, m) of a list entry: first K row of its box (the union of the groups' windows), the
      // tensor coordinate of its (m, q) record, and the issuers' info words; fetched one entry ahead (the
      // loads are a dependent chain through L2)
      struct Ent { unsigned any, bytes, inf[kTcG], m; int c0, c2; bool big; };
      auto entry_window = [&](const long long e) {
        Ent r;
        const uint2 hd = __ldg(&tp.list[e]);
        r.any = hd.y;
        r.m = hd.x;
        int lo = 0x7fffffff;
        unsigned c[kTcG];
        bool used = false;
        r.big = false;
#pragma unroll
        for (int g = 0; g < kTcG; ++g) {
          c[g] = __ldg(&tp.codes[(e * kTcG + g) * 16 + ql]);
          if (code_passes(c[g])) { lo = min(lo, code_start(c[g])); used = true; r.big = r.big || (c[g] & kTcCodeBig); }
        }
        if (!used) lo = 0;
        // info word: K-row offset of the group's window inside the box (16-byte units; the stage slot's address is
        // added when the word is published) | passes << 14 | big box << 16
#pragma unroll
        for (int g = 0; g < kTcG; ++g)
          r.inf[g] = has_q ? (((unsigned)code_passes(c[g]) << 14) | (code_passes(c[g]) ? (unsigned)(2 * (code_start(c[g]) - lo)) : 0u) |
                              (r.big ? 0x10000u : 0u)) : 0u;
        r.bytes = (has_q && used) ? (r.big ? stage_bytes : small_bytes) : 0u;
        r.c0 = 8 * (tb_q + lo);                               // 32-bit elements: 4 per K row, 2 K rows per sample
        r.c2 = (chunk * P.M + (int)hd.x) * P.Q + ql;
        return r;
      };
      // index of the last list entry any group uses (its last stage ends the tile for the issuers)
      int last_li = -1;
      for (int li0 = 0; li0 < td.list_cnt; li0 += 32) {
        const int li = li0 + lane;
        const bool used = li < td.list_cnt && __ldg(&tp.list[td.list_off + li]).y != 0u;
        const unsigned m = __ballot_sync(0xffffffffu, used);
        if (m) last_li = li0 + 31 - __clz(m);
      }
      Ent nx;
      nx.any = 0; nx.bytes = 0; nx.c0 = 0; nx.c2 = 0; nx.big = false; nx.m = 0;
      if (td.list_cnt) nx = entry_window(td.list_off);
      bool sent = false;
      for (int li = 0; li < td.list_cnt || !sent; ++li) {
        Ent cur;
        if (li < td.list_cnt) {
          cur = nx;
          if (li + 1 < td.list_cnt) nx = entry_window((long long)td.list_off + li + 1);
          if (!cur.any) continue;
        } else {
          // a tile without any receiver: one empty stage, so that the issuers see the end of the tile
          cur.any = 0; cur.bytes = 0; cur.c0 = 0; cur.c2 = 0; cur.big = false; cur.m = 0xffffu;
#pragma unroll
          for (int g = 0; g < kTcG; ++g) cur.inf[g] = 0u;
        }
        sent = true;
        // ---- quad pacing (L2 reuse) --------------------------------------------------------------------------
        // CTAs 4 j .. 4 j + 3 work on a 2 x 2 block of laterally adjacent tiles (the plan orders the tiles so), whose
        // receiver lists and sample windows overlap almost entirely.  Each producer publishes (launch, round, receiver)
        // before it fetches a receiver's windows and holds back while a partner is more than `pace` receivers behind:
        // the four then read the same records within microseconds of each other and three of the four reads hit L2.
        // Advisory only: the wait is bounded per receiver and per launch (pace_budget), nothing else depends on it.
        // The partners' words are loaded here and looked at only after the wait for the stage below, so that the
        // round trip to L2 hides under it; one receiver in four is paced.
        const bool paced = tp.progress != nullptr && (li & tp.pace_mask) == 0;
        unsigned long long me = 0ull, seen = ~0ull;
        const unsigned long long* pp = tp.progress + (blockIdx.x ^ (unsigned)(lane & 3));
        if (paced) {
          me = tp.epoch | ((unsigned long long)(unsigned)(work / (int)gridDim.x) << 16) | (unsigned long long)min(cur.m, 0xffffu);
          if (lane == 0) asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(tp.progress + blockIdx.x), "l"(me) : "memory");
          if (lane >= 1 && lane <= 3 && pace_budget > 0) asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(seen) : "l"(pp) : "memory");
        }
        for (int q0 = 0; q0 < P.Q; q0 += (int)qs) {
          const bool mine = lane >= q0 && lane < q0 + (int)qs;
          const unsigned total = __reduce_add_sync(0xffffffffu, mine ? cur.bytes : 0u);
          const bool last_stage = li >= last_li && q0 + (int)qs >= P.Q;
          TC_PROF_WAIT(1, if (lane == 0) mbar_wait_park(b_empty0 + 8 * s, ph ^ 1u); __syncwarp())
          __syncwarp();
          if (paced && q0 == 0) {
            if (lane >= 1 && lane <= 3) {
              int spin = 0;
              for (; seen + (unsigned long long)tp.pace < me && spin < pace_budget; ++spin) {
                __nanosleep(64);
                asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(seen) : "l"(pp) : "memory");
              }
              if (spin > 0 && spin >= pace_budget) pace_budget >>= 2;          // expired: this partner gets less from now on
            }
            __syncwarp();
          }
          if (mine) {
            const unsigned slot_u16 = (stage0 + (s * qs + (unsigned)(lane - q0)) * stage_bytes) >> 4;   // the item's window slot
#pragma unroll
            for (int g = 0; g < kTcG; ++g)
              sm.info[(s * kTcMaxQs + (unsigned)(lane - q0)) * kTcG + g] = (cur.inf[g] + slot_u16) | ((last_stage && lane == q0) ? 0x80000000u : 0u);
          }
          __syncwarp();
          if (lane == 0) {
            if (total) mbar_arrive_expect_tx(b_full0 + 8 * s, total);
            else mbar_arrive(b_full0 + 8 * s);
          }
          __syncwarp();
          if (mine && cur.bytes)
            tma_tensor3_g2s(stage0 + (s * qs + (unsigned)(lane - q0)) * stage_bytes, cur.big ? &tmap_big : &tmap_small, cur.c0, 0, cur.c2, b_full0 + 8 * s);
          if (++s == (unsigned)tp.n_stages) { s = 0; ph ^= 1u; }
          __syncwarp();
        }
      }
      // this tile's list is through: the partners need not wait for this CTA before its next tile
      if (tp.progress && lane == 0) {
        const unsigned long long me = tp.epoch | ((unsigned long long)(unsigned)(work / (int)gridDim.x) << 16) | 0xffffull;
        asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(tp.progress + blockIdx.x), "l"(me) : "memory");
      }
    }
    TC_PROF_END
  } else if (warp > kTcGenWarps + kTcG) {
    // no role
  } else if (warp > kTcGenWarps) {
    // ===================================== MMA ISSUERS ========================================
    // One warp per voxel group.  The issue loop is a serial chain (probe -> MMA -> commit) whose
    // latency bounds the MMA rate of a group (measured: it, not the generators' instruction count,
    // set the pace), so it is kept short and small: the producer publishes the ready-made start
    // address of every window, EVERY lane runs the same loop (a loop under `lane == 0` makes ptxas
    // wrap each tcgen05 instruction in an elect / broadcast loop), the MMA and its commit sit under
    // elect.sync inside one asm block, and the stage barriers are visited once per qs items.  Item q
    // takes its A tile from slot q mod 4, a second pass from the overflow slot (das_tc.cuh).
    const int g = warp - kTcGenWarps - 1;
    {
      const unsigned idesc = tc_idesc(N);
      const unsigned d_tmem = tmem + (unsigned)(g * N);
      const unsigned a_tmem0 = tmem + a_col0 + (unsigned)(kTcABufs * g) * kTcACols;
      const unsigned af0 = a_full0 + 8u * (unsigned)(kTcABufs * g), ae0 = a_empty0 + 8u * (unsigned)(kTcABufs * g);
      // descriptor of a B tile: LBO = 8 K rows (the next core matrix along K), SBO = one column group of the box (its K
      // rows: small or big box); the 14-bit start address (16-byte units = K rows) comes ready-made from the producer
      const unsigned long long desc_s = tc_smem_desc(0u, 8 * 16, 2 * kTcBoxSmall * 16), desc_b = tc_smem_desc(0u, 8 * 16, 2 * kTcBoxBig * 16);
      const unsigned desc_lo0 = (unsigned)desc_s, desc_hi_s = (unsigned)(desc_s >> 32), desc_hi_b = (unsigned)(desc_b >> 32);
      const unsigned info0 = smem_u32(&sm.info[0]) + 4u * (unsigned)g;
      // Item tiles use their 4 slots round robin: aoff = 8 * slot is the byte offset of the slot's barriers and its
      // column offset in tensor memory; apar / opar = phase parity of the next use of the item slots / the overflow slot
      unsigned s = 0, ph = 0, n_done = 0, aoff = 0, apar = 0, opar = 0;
      TC_PROF_DECL
      for (int work = blockIdx.x; work < n_work; work += gridDim.x, ++n_done) {
        TC_PROF_WAIT(1, mbar_wait_park(d_empty, (n_done & 1u) ^ 1u))           // epilogue of the previous tile has drained D
        tc_fence_after();
        bool last = false;
        while (!last) {
          TC_PROF_WAIT(2, if (!mbar_test(b_full0 + 8 * s, ph)) mbar_wait_park(b_full0 + 8 * s, ph))
          unsigned ia = info0 + s * (kTcMaxQs * kTcG * 4u);
          unsigned info = lds_volatile(ia);
          last = (info >> 31) != 0u;
          for (unsigned i = 0; i < qs; ++i) {
            ia += kTcG * 4u;
            const unsigned info_next = (i + 1 < qs) ? lds_volatile(ia) : 0u;   // one item ahead (slots beyond Q hold 0)
            const unsigned np = (info >> 14) & 3u;
            if (np) {
              const unsigned dlo = desc_lo0 | (info & 0x3fffu);
              const unsigned dhi = (info & 0x10000u) ? desc_hi_b : desc_hi_s;
              TC_PROF_WAIT(3, if (!mbar_test(af0 + aoff, apar)) mbar_wait_park(af0 + aoff, apar))
              tc_fence_after();
              tc_mma_commit(d_tmem, a_tmem0 + aoff, dlo, dhi, idesc, ae0 + aoff);   // the commit completes when the MMA has read its A slot
              if (np > 1) {
                TC_PROF_WAIT(4, if (!mbar_test(af0 + 8u * kTcOvf, opar)) mbar_wait_park(af0 + 8u * kTcOvf, opar))
                opar ^= 1u;
                tc_fence_after();
                tc_mma_commit(d_tmem, a_tmem0 + kTcOvf * kTcACols, dlo + 2u * kTcPass, dhi, idesc, ae0 + 8u * kTcOvf);
              }
              aoff = (aoff + 8u) & (8u * kTcSlots - 1u);
              apar ^= (aoff == 0u) ? 1u : 0u;
            }
            info = info_next;
          }
          if (tc_elect()) tc_commit(b_empty0 + 8 * s);         // this group is done with the stage
          __syncwarp();
          if (++s == (unsigned)tp.n_stages) { s = 0; ph ^= 1u; }
        }
        if (tc_elect()) tc_commit(d_full);                     // this group's MMAs of the tile are complete
        __syncwarp();
      }
      TC_PROF_END
    }
  } else {
    // ===================================== GENERATORS =========================================
    const int g = warp >> 2;                                  // voxel group = depth inside the tile
    const int row = (warp & 3) * 32 + lane;                   // MMA row = TMEM lane (quarter warp % 4)
    const unsigned lane_base = ((unsigned)((warp & 3) * 32)) << 16;
    const unsigned d_addr = tmem + lane_base + (unsigned)(g * N);
    TcGenState st;
    asm volatile("mov.u32 %0, %1;" : "=r"(st.a_addr0) : "r"(tmem + lane_base + a_col0 + (unsigned)(kTcABufs * g) * kTcACols));
    asm volatile("mov.u32 %0, %1;" : "=r"(st.ae0) : "r"(a_empty0 + 8u * (unsigned)(kTcABufs * g)));
    asm volatile("mov.u32 %0, %1;" : "=r"(st.af0) : "r"(a_full0 + 8u * (unsigned)(kTcABufs * g)));
    asm volatile("mov.u32 %0, %1;" : "=r"(st.tbl0) : "r"(smem_u32(&sm.place[-kTcPlaceLo][0])));
    st.sink = sinkb;
    st.pend = sinkb;
    st.pend2 = sinkb;
    st.it = 0u;
    st.par = 0u;
    st.free_next = false;
    unsigned n_done = 0;
    TC_PROF_DECL
#ifdef DAS_TC_PROF
    st.pf1 = st.pf2 = st.pf3 = 0;
#endif

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
        const float wq = tx_weight(P, qq, vx.n);                  // transmit weight (1 without a table), carried by Ptx
        if (j & 1) { Tf[j >> 1].y = tf; pc[j >> 1].y = wq * cos_approx(ang); ps[j >> 1].y = wq * sin_approx(ang); }
        else       { Tf[j >> 1].x = tf; pc[j >> 1].x = wq * cos_approx(ang); ps[j >> 1].x = wq * sin_approx(ang); }
      }

      // the list entry one iteration ahead: header, the group's 16 window codes, receiver position
      uint2 hd_n = make_uint2(0u, 0u);
      uint4 cw0_n = make_uint4(0u, 0u, 0u, 0u), cw1_n = cw0_n;
      float4 el_n = make_float4(0.f, 0.f, 0.f, 0.f), dir_n = make_float4(0.f, 0.f, 1.f, 0.f);
      if (td.list_cnt) {
        const uint4* cp = reinterpret_cast<const uint4*>(tp.codes + ((long long)td.list_off * kTcG + g) * 16);
        hd_n = __ldg(&tp.list[td.list_off]);
        cw0_n = __ldg(cp); cw1_n = __ldg(cp + 1);
        el_n = __ldg(&P.elem[hd_n.x]);
        if (P.has_dir) dir_n = __ldg(&P.edir[hd_n.x]);
      }
      for (int li = 0; li < td.list_cnt; ++li) {
        const uint2 hd = hd_n;
        const uint4 cw0 = cw0_n, cw1 = cw1_n;
        const float4 el = el_n, dir = dir_n;
        if (li + 1 < td.list_cnt) {
          const long long e = td.list_off + li + 1;
          const uint4* cp = reinterpret_cast<const uint4*>(tp.codes + (e * kTcG + g) * 16);
          hd_n = __ldg(&tp.list[e]);
          cw0_n = __ldg(cp); cw1_n = __ldg(cp + 1);
          el_n = __ldg(&P.elem[hd_n.x]);
          if (P.has_dir) dir_n = __ldg(&P.edir[hd_n.x]);
        }
        if (!((hd.y >> g) & 1u)) continue;                    // no voxel of this group sees receiver m
        // per-(m, n): aperture, excess path, receive phase (as in das_tiled.cuh)
        bool act;
        float wrx;
        const float ex = tc_excess(tp, P, vx, el, dir, act, wrx);
        if (!__any_sync(0xffffffffu, act)) {
          // no voxel of this WARP sees the receiver: 32 zero rows per item, no arithmetic
          if (q16) tc_gen_receiver<false, true, true>(Tf, pc, ps, 0.f, 0.f, 0.f, 0u, cw0, cw1, tb_l, P.Q, P.K, st);
          else tc_gen_receiver<false, true, false>(Tf, pc, ps, 0.f, 0.f, 0.f, 0u, cw0, cw1, tb_l, P.Q, P.K, st);
          continue;
        }
        float cyc = tp.ratio_f * ex;
        cyc -= rintf(cyc);
        const float ang = 6.283185307179586f * cyc;
        const float pr = act ? wrx * cos_approx(ang) : 0.f, pi = act ? wrx * sin_approx(ang) : 0.f;
        if (q16) {
          if (td.edge) tc_gen_receiver<true, false, true>(Tf, pc, ps, ex, pr, pi, act ? 0xffffffffu : 0u, cw0, cw1, tb_l, P.Q, P.K, st);
          else tc_gen_receiver<false, false, true>(Tf, pc, ps, ex, pr, pi, act ? 0xffffffffu : 0u, cw0, cw1, tb_l, P.Q, P.K, st);
        } else {
          if (td.edge) tc_gen_receiver<true, false, false>(Tf, pc, ps, ex, pr, pi, act ? 0xffffffffu : 0u, cw0, cw1, tb_l, P.Q, P.K, st);
          else tc_gen_receiver<false, false, false>(Tf, pc, ps, ex, pr, pi, act ? 0xffffffffu : 0u, cw0, cw1, tb_l, P.Q, P.K, st);
        }
      }
      tmem_wait_st();
      tc_fence_before();
      mbar_arrive2_elect(st.pend, st.pend2);
      st.pend = sinkb;
      st.pend2 = sinkb;

      // ---- epilogue: D (FP32, TMEM) -> out[frame][voxel] -------------------------------------
      TC_PROF_WAIT(3, mbar_wait_park(d_full, n_done & 1u))
      tc_fence_after();
#ifdef DAS_TC_PROF
      const long long ep0_ = clock64();
#endif
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
#ifdef DAS_TC_PROF
      pf_[4] += (unsigned long long)(clock64() - ep0_);
#endif
    }
#ifdef DAS_TC_PROF
    pf_[1] = st.pf1; pf_[2] = st.pf2; pf_[5] = st.pf3;
#endif
    TC_PROF_END
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
// and writes the window code the warp roles of tc_kernel read (TcDev::codes): a group needs the
// samples [smin, smax + 1], i.e. ceil((smax + 2 - smin) / 8) MMA passes from sample smin on.  The
// windows of the groups of one (entry, q) must lie in one box (kTcBoxSmall samples if every group needs one
// pass and the item needs no more than that, else kTcBoxBig) starting at the smallest smin: a window that
// would stick out of the box is moved down (it then starts before its smin, which costs nothing).
//   stats[0] = largest number of samples one (entry, q) needs, stats[1] = error bits
//   (1: a group needs more than 2 passes, 2: the groups of an item do not fit one box, 4: negative start)
__global__ void __launch_bounds__(kTcG * kTcRows)
tc_window_kernel(const TcDev tp, const Params P, uint2* __restrict__ list, unsigned short* __restrict__ codes,
                 int* __restrict__ tile_work, int* __restrict__ tile_edge, int* __restrict__ stats) {
  __shared__ int kmn[kTcG][16], kmx[kTcG][16];
  __shared__ unsigned lst[kTcG];                              // per group: transmits some active voxel lists, this receiver
  const int tile_i = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
  const int g = tid / kTcRows, row = tid % kTcRows;
  const TcTile td = tp.tiles[tile_i];
  const TcVoxel vx = tc_voxel(tp, P, td, row, g);
  float Tf[16];
#pragma unroll
  for (int q = 0; q < 16; ++q) {
    const int qq = min(q, P.Q - 1);
    Tf[q] = (float)(tc_T(P, vx, qq) - (double)__ldg(&tp.tbase[(long long)tile_i * P.Q + qq]));
  }
  const int tb = tid < 16 ? __ldg(&tp.tbase[(long long)tile_i * P.Q + min(tid, P.Q - 1)]) : 0;
  int work = 0, edge = 0, span = 0, err = 0;
  // transmits this voxel sums over: all of them, or those with a non-zero weight when the plan has a weight table
  // (observation lists are stored as zeros of that table; reading W5).  An item (q, m, group) that NO voxel of the
  // group lists gets no window at all: no box, no A tile, no MMA ("skip these negligible contributions").
  unsigned listed = 0xffffu;
  if (P.wtx_tab) {
    listed = 0u;
    for (int q = 0; q < P.Q; ++q) listed |= (tx_weight(P, q, vx.n) != 0.f ? 1u : 0u) << q;
  }

  for (int li = 0; li < td.list_cnt; ++li) {
    const long long e = td.list_off + li;
    if (tid < kTcG * 16) { kmn[tid / 16][tid % 16] = INT_MAX; kmx[tid / 16][tid % 16] = INT_MIN; }
    if (tid < kTcG) lst[tid] = 0u;
    __syncthreads();
    const float4 el = __ldg(&P.elem[list[e].x]);
    const float4 dir = P.has_dir ? __ldg(&P.edir[list[e].x]) : make_float4(0.f, 0.f, 1.f, 0.f);
    bool act;
    float wrx_unused;
    const float ex = tc_excess(tp, P, vx, el, dir, act, wrx_unused);
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
    {
      // the windows above span ALL voxels inside the aperture (a voxel that does not list q still indexes the
      // placement table with its own sample position); only "does anybody list q" decides whether the item exists
      const unsigned any_l = __reduce_or_sync(0xffffffffu, act ? listed : 0u);
      if (lane == 0 && any_l) atomicOr(&lst[g], any_l);
    }
    __syncthreads();
    if (tid < 16) {
      const int q = tid;
      unsigned flags = 0;
      int u0 = INT_MAX, uend = INT_MIN;                          // samples the item needs: [u0, uend)
      if (q < P.Q)
        for (int gg = 0; gg < kTcG; ++gg) {
          if (!((lst[gg] >> q) & 1u)) kmn[gg][q] = INT_MAX;      // nobody in the group lists q (only this thread touches column q now)
          if (kmn[gg][q] != INT_MAX) { u0 = min(u0, kmn[gg][q]); uend = max(uend, kmx[gg][q] + 2); }
        }
      bool big = false;
      if (u0 != INT_MAX) {
        big = uend - u0 > kTcBoxSmall;
        for (int gg = 0; gg < kTcG; ++gg)
          if (kmn[gg][q] != INT_MAX && kmx[gg][q] + 2 - kmn[gg][q] > kTcPass) big = true;   // a two-pass window needs 16 samples
        if (u0 < 0 || u0 > 0x1fff - kTcBoxBig) err |= 4;
        if (uend - u0 > kTcBoxBig) err |= 2;
        span = max(span, uend - u0);
        if (tb + u0 <= 0 || tb + u0 + kTcBoxBig >= P.K - 1) edge = 1;
      }
      const int box = big ? kTcBoxBig : kTcBoxSmall;
      for (int gg = 0; gg < kTcG; ++gg) {
        unsigned code = 0;
        if (q < P.Q && kmn[gg][q] != INT_MAX) {
          const int smin = kmn[gg][q], smax = kmx[gg][q];
          const int np = (smax + 2 - smin + kTcPass - 1) / kTcPass;
          if (np > 2) err |= 1;
          const int npc = min(np, 2);
          const int start = max(min(smin, u0 + box - kTcPass * npc), 0);
          code = (unsigned)npc | ((unsigned)min(start, 0x1fff) << 2) | (big ? (unsigned)kTcCodeBig : 0u);
          flags |= 1u << gg;
          work += npc;
        }
        codes[(e * kTcG + gg) * 16 + q] = (unsigned short)code;
      }
      flags = __reduce_or_sync(0x0000ffffu, flags);
      if (tid == 0) list[e].y = flags;
    }
    __syncthreads();                                          // kmn / kmx are re-initialised at the loop top
  }
  if (tid < 16) {
    work = __reduce_add_sync(0x0000ffffu, work);
    edge = __reduce_or_sync(0x0000ffffu, edge);
    span = __reduce_max_sync(0x0000ffffu, span);
    err = __reduce_or_sync(0x0000ffffu, err);
    if (tid == 0) {
      tile_work[tile_i] = work;
      tile_edge[tile_i] = edge;
      atomicMax(&stats[0], span);
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

cudaError_t launch_tc_kernel(const TcDev& tp, const Params& P, const void* tmaps, void* d_out, int grid, size_t smem, cudaStream_t s) {
  // per launch: the attribute belongs to the (device, context) the plan lives on, and it is cheap
  cudaError_t e = cudaFuncSetAttribute(tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024 + 2048);
  if (e != cudaSuccess) return e;
  const CUtensorMap* maps = static_cast<const CUtensorMap*>(tmaps);                  // [0] small box, [1] big box
  tc_kernel<<<grid, kTcThreads, smem, s>>>(tp, P, maps[0], maps[1], static_cast<float2*>(d_out));
  return cudaGetLastError();
}

}  // namespace das
