// Host side of the frame-batch tensor-core kernel (das_tc.cuh): applicability, voxel tiles,
// per-tile receiver lists with per-group delay bounds, stage sizing, batch-inner convert kernel.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <numeric>
#include <vector>

#include "das_tc.cuh"

namespace das {

cudaError_t launch_tc_kernel(const TcDev& tp, const Params& P, const void* d_conv, void* d_out, int grid, size_t smem, cudaStream_t s);

struct TcPlan {
  TcDev dev{};
  int grid = 1;
  size_t smem = 0;
  int n_frames = 0;
  std::vector<void*> allocs;
};

void tc_plan_destroy(TcPlan* tp) {
  if (!tp) return;
  for (void* d : tp->allocs) cudaFree(d);
  delete tp;
}

size_t tc_converted_bytes(const TcPlan* tp, const Params& P) {
  return (size_t)tp->dev.n_chunks * P.M * P.Q * tp->dev.KBp * (size_t)(2 * tp->dev.Bc) * 16;
}
int tc_frames_per_chunk(const TcPlan* tp) { return tp->dev.Bc; }

namespace {
template <typename T>
cudaError_t up(TcPlan* tp, const std::vector<T>& h, const T** d_out) {
  void* d = nullptr;
  cudaError_t e = cudaMalloc(&d, std::max<size_t>(h.size(), 1) * sizeof(T));
  if (e != cudaSuccess) return e;
  tp->allocs.push_back(d);
  if (!h.empty()) e = cudaMemcpy(d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
  *d_out = static_cast<const T*>(d);
  return e;
}
}  // namespace

TcPlan* tc_plan_create(const Params& P, const das_plan_desc_t& d, int n_frames, int device, char* why,
                       size_t why_len, cudaError_t* cuda_err) {
  *cuda_err = cudaSuccess;
  auto refuse = [&](const char* msg) -> TcPlan* { snprintf(why, why_len, "%s", msg); return nullptr; };
  // ---- applicability ------------------------------------------------------------------------
  if (!P.iq || !P.fp16) return refuse("the tensor-core path needs IQ data in fp16 storage");
  if (d.n_tx > 16) return refuse("more than 16 transmits");
  if (n_frames < 8 || n_frames % 8) return refuse("frame count is not a multiple of 8");
  int Bc = n_frames;
  if (n_frames > 64) { if (n_frames % 64) return refuse("frame count above 64 is not a multiple of 64"); Bc = 64; }
  const double z_a = d.elem_pos[2];
  for (int m = 0; m < d.n_elem; ++m)
    if ((double)d.elem_pos[3 * m + 2] != z_a) return refuse("receivers are not in one plane z = const");
  if (d.elem_dir)
    for (int m = 0; m < d.n_elem; ++m)
      if (d.elem_dir[3 * m] != 0.f || d.elem_dir[3 * m + 1] != 0.f || d.elem_dir[3 * m + 2] != 1.f)
        return refuse("receiver normals are not all (0,0,1)");
  for (int i = 0; i < d.nz; ++i)
    if (!((double)d.zs[i] > z_a)) return refuse("a voxel plane is not in front of the array (z <= z_array)");

  const double c = d.c, fs = d.fs, fc = d.fc, t_start = d.t_start, fnum = d.f_number;
  const bool apod = fnum > 0.0;
  const double kappa = fs / c;
  const int Q = d.n_tx, M = d.n_elem;
  const int ntx = (d.nx + kTcGX - 1) / kTcGX, nty = (d.ny + kTcGY - 1) / kTcGY, ntz = (d.nz + kTcG - 1) / kTcG;
  const long long n_tiles_ll = (long long)ntx * nty * ntz;
  if (n_tiles_ll > (1 << 22)) return refuse("too many tiles");
  const int n_tiles = (int)n_tiles_ll;

  // ---- host part: tiles, sample base per (tile, q), conservative receiver lists ------------------
  std::vector<TcTile> tiles(n_tiles);
  std::vector<int> tbase((size_t)n_tiles * Q);
  std::vector<uint2> list;
  list.reserve((size_t)n_tiles * std::min(M, 512));
  const double cone = apod ? 1.0 / (2.0 * fnum) : 0.0;

  int t = 0;
  for (int tz = 0; tz < ntz; ++tz)
    for (int ty = 0; ty < nty; ++ty)
      for (int txi = 0; txi < ntx; ++txi, ++t) {
        TcTile& td = tiles[t];
        td.ix0 = txi * kTcGX; td.iy0 = ty * kTcGY; td.iz0 = tz * kTcG;
        td.edge = 0;
        const int ix1 = std::min(td.ix0 + kTcGX, d.nx), iy1 = std::min(td.iy0 + kTcGY, d.ny);
        const int iz1 = std::min(td.iz0 + kTcG, d.nz);
        double xlo = 1e300, xhi = -1e300, ylo = 1e300, yhi = -1e300;
        for (int i = td.ix0; i < ix1; ++i) { xlo = std::min(xlo, (double)d.xs[i]); xhi = std::max(xhi, (double)d.xs[i]); }
        for (int i = td.iy0; i < iy1; ++i) { ylo = std::min(ylo, (double)d.ys[i]); yhi = std::max(yhi, (double)d.ys[i]); }
        // sample base: a multiple of 4 below T_q of every voxel of the tile (the kernels clamp the rows
        // and columns beyond the grid edge to the last voxel, which is inside these ranges)
        for (int q = 0; q < Q; ++q) {
          const das_transmit_t& tx = d.tx[q];
          double lo = 1e300;
          for (int k = td.iz0; k < iz1; ++k) {
            const double z = d.zs[k], a = z - z_a;
            for (int i = td.ix0; i < ix1; ++i)
              for (int j = td.iy0; j < iy1; ++j) {
                const double x = d.xs[i], y = d.ys[j];
                double tau;
                if (tx.type == DAS_TX_PLANE) tau = (x * tx.v[0] + y * tx.v[1] + z * tx.v[2]) / c + tx.t0;
                else tau = std::sqrt((x - tx.v[0]) * (x - tx.v[0]) + (y - tx.v[1]) * (y - tx.v[1]) + (z - tx.v[2]) * (z - tx.v[2])) / c + tx.t0;
                lo = std::min(lo, (tau + a / c - t_start) * fs);
              }
          }
          if (!(std::fabs(lo) < 1e8)) return refuse("sample coordinate out of range");
          tbase[(size_t)t * Q + q] = (int)std::floor((lo - kTcMargin) / 4.0) * 4;
        }
        // receivers whose aperture cone can reach a voxel of the tile (bounding-box test; the window
        // kernel below classifies every voxel exactly and drops the receivers no group sees)
        td.list_off = (int)list.size();
        const double a_max = (double)d.zs[iz1 - 1] - z_a, a_min = (double)d.zs[td.iz0] - z_a;
        const double a_far = std::max(a_max, a_min);
        for (int m = 0; m < M; ++m) {
          const double ex = d.elem_pos[3 * m], ey = d.elem_pos[3 * m + 1];
          const double nx_ = std::max(std::max(xlo - ex, ex - xhi), 0.0), ny_ = std::max(std::max(ylo - ey, ey - yhi), 0.0);
          const double rho_min = std::sqrt(nx_ * nx_ + ny_ * ny_);
          if (apod && rho_min > cone * a_far * (1.0 + 1e-5)) continue;
          list.push_back(make_uint2((unsigned)m, 0u));
        }
        td.list_cnt = (int)list.size() - td.list_off;
      }
  if (list.size() > (size_t)0x7fffffff / (kTcG * 16)) return refuse("receiver lists too long");

  TcPlan* tp = new TcPlan();
  tp->n_frames = n_frames;
  cudaDeviceProp prop;
  cudaError_t e = cudaGetDeviceProperties(&prop, device);
  if (e != cudaSuccess) { *cuda_err = e; delete tp; return nullptr; }
  TcDev& dv = tp->dev;
  dv.n_tiles = n_tiles;
  dv.Bc = Bc;
  dv.n_chunks = n_frames / Bc;
  dv.KBp = tc_kblocks(P.K);
  dv.z_array = z_a; dv.kappa = kappa; dv.ratio = fc / fs;
  dv.phase0 = fc * t_start - std::floor(fc * t_start);
  dv.four_f2 = (float)(4.0 * fnum * fnum);
  dv.kappa_f = (float)kappa; dv.ratio_f = (float)(fc / fs);

  // ---- device part: exact windows per (receiver, transmit, voxel group) ---------------------------
  auto fail = [&](cudaError_t ce) -> TcPlan* { *cuda_err = ce; tc_plan_destroy(tp); return nullptr; };
  const TcTile* d_tiles0 = nullptr;
  const int* d_tbase0 = nullptr;
  void *d_codes = nullptr, *d_work = nullptr, *d_edge = nullptr, *d_stats = nullptr;
  if ((e = up(tp, tiles, &d_tiles0)) != cudaSuccess || (e = up(tp, tbase, &d_tbase0)) != cudaSuccess ||
      (e = up(tp, list, &dv.list)) != cudaSuccess) return fail(e);
  const size_t n_codes = std::max<size_t>(list.size(), 1) * kTcG * 16;
  if ((e = cudaMalloc(&d_codes, n_codes * sizeof(unsigned short))) != cudaSuccess) return fail(e);
  tp->allocs.push_back(d_codes);
  if ((e = cudaMalloc(&d_work, sizeof(int) * n_tiles)) != cudaSuccess) return fail(e);
  tp->allocs.push_back(d_work);
  if ((e = cudaMalloc(&d_edge, sizeof(int) * n_tiles)) != cudaSuccess) return fail(e);
  tp->allocs.push_back(d_edge);
  if ((e = cudaMalloc(&d_stats, sizeof(int) * 2)) != cudaSuccess) return fail(e);
  tp->allocs.push_back(d_stats);
  if ((e = cudaMemset(d_stats, 0, sizeof(int) * 2)) != cudaSuccess) return fail(e);
  dv.tiles = d_tiles0;
  dv.tbase = d_tbase0;
  dv.codes = static_cast<const unsigned short*>(d_codes);
  if ((e = launch_tc_windows(dv, P, const_cast<uint2*>(dv.list), static_cast<unsigned short*>(d_codes), static_cast<int*>(d_work),
                             static_cast<int*>(d_edge), static_cast<int*>(d_stats), nullptr)) != cudaSuccess) return fail(e);
  std::vector<int> work(n_tiles), edge(n_tiles);
  int stats[2] = {0, 0};
  if ((e = cudaMemcpy(work.data(), d_work, sizeof(int) * n_tiles, cudaMemcpyDeviceToHost)) != cudaSuccess ||
      (e = cudaMemcpy(edge.data(), d_edge, sizeof(int) * n_tiles, cudaMemcpyDeviceToHost)) != cudaSuccess ||
      (e = cudaMemcpy(stats, d_stats, sizeof(stats), cudaMemcpyDeviceToHost)) != cudaSuccess) return fail(e);
  auto refuse_free = [&](const char* msg) -> TcPlan* { tc_plan_destroy(tp); return refuse(msg); };
  if (getenv("DAS_TC_VERBOSE")) {
    long long tw = 0; for (int w_ : work) tw += w_;
    fprintf(stderr, "[das tc plan] tiles %d, list entries %zu, MMA passes %lld, largest window %d k-blocks\n", n_tiles, list.size(), tw, stats[0]);
  }
  if (stats[1] & 1) return refuse_free("a sample window of a voxel group needs more than 3 MMA passes (grid too coarse)");
  if (stats[1] & 2) return refuse_free("a sample window leaves the zero-padded record");
  if (stats[1] & 4) return refuse_free("internal: negative window start");
  const int stage_blocks = std::max(stats[0], kTcPassBlocks);
  if (stage_blocks > kTcMaxStageBlocks) {
    snprintf(why, why_len, "sample window per tile (%d k-blocks) exceeds the stage capacity (%d)", stage_blocks, kTcMaxStageBlocks);
    tc_plan_destroy(tp);
    return nullptr;
  }

  // Tile order: depth slab by depth slab (heaviest slab first), all lateral tiles of a slab side by
  // side.  The CTAs of a wave then walk the same receivers of the same depth at about the same
  // time, so the sample windows one CTA pulls from HBM are found in L2 by its lateral neighbours
  // (they overlap almost entirely); the cheap shallow slabs come last and level the tail.
  std::vector<double> slab_work(ntz, 0.0);
  for (int i = 0; i < n_tiles; ++i) slab_work[i / (ntx * nty)] += work[i];
  std::vector<int> order(n_tiles);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
    const int sa = a / (ntx * nty), sb = b / (ntx * nty);
    if (sa != sb) return slab_work[sa] > slab_work[sb];
    return work[a] > work[b];
  });
  std::vector<TcTile> tiles_s(n_tiles);
  std::vector<int> tbase_s(tbase.size());
  for (int i = 0; i < n_tiles; ++i) {
    tiles_s[i] = tiles[order[i]];
    tiles_s[i].edge = edge[order[i]];
    std::memcpy(&tbase_s[(size_t)i * Q], &tbase[(size_t)order[i] * Q], sizeof(int) * Q);
  }
  if ((e = up(tp, tiles_s, &dv.tiles)) != cudaSuccess || (e = up(tp, tbase_s, &dv.tbase)) != cudaSuccess) return fail(e);

  dv.stage_blocks = stage_blocks;
  // A ring: as deep as tensor memory allows next to the accumulators (512 columns: kTcG * 2 Bc of D)
  dv.a_shift = 3;
  if (const char* ev = getenv("DAS_TC_ABUFS")) dv.a_shift = std::min(3, std::max(0, atoi(ev)));   // tuning sweeps only
  while (dv.a_shift > 0 && kTcG * 2 * Bc + kTcG * (1 << dv.a_shift) * kTcACols > kTcTmemCols) --dv.a_shift;
  dv.a_bufs = 1 << dv.a_shift;
  // Stage ring: `qs` window slots per stage (the fewer barrier rounds the better: the producer and
  // the MMA issuers are serial latency chains) and as many stages as cover the L2 latency of a
  // window.  Measured at the headline: (qs, stages) = (8, 2) 94 ms, (4, 4) 96 ms, (1, 6) 111 ms.
  dv.qs = 8;
  dv.n_stages = 2;
  while (dv.qs > 1 && tc_smem_bytes(Bc, stage_blocks, dv.qs, 2) > 200 * 1024) dv.qs /= 2;
  if (const char* ev = getenv("DAS_TC_QS")) dv.qs = std::min(16, std::max(1, atoi(ev)));                               // tuning sweeps only
  if (const char* ev = getenv("DAS_TC_STAGES")) dv.n_stages = std::min(kTcMaxStages, std::max(kTcMinStages, atoi(ev)));   // tuning sweeps only
  else while (dv.n_stages < 4 && dv.qs * dv.n_stages < 8 && tc_smem_bytes(Bc, stage_blocks, dv.qs, dv.n_stages + 1) <= 200 * 1024) ++dv.n_stages;
  while (dv.n_stages > kTcMinStages && tc_smem_bytes(Bc, stage_blocks, dv.qs, dv.n_stages) > 200 * 1024) --dv.n_stages;
  tp->smem = tc_smem_bytes(Bc, stage_blocks, dv.qs, dv.n_stages);
  if (tp->smem > 200 * 1024) return refuse_free("stage ring does not fit in shared memory");
  tp->grid = std::max(1, std::min(n_tiles * dv.n_chunks, prop.multiProcessorCount));
  return tp;
}

cudaError_t launch_tc(const TcPlan* tp, const Params& P, const void* d_conv, void* d_out, cudaStream_t s) {
  count_launch();
  return launch_tc_kernel(tp->dev, P, d_conv, d_out, tp->grid, tp->smem, s);
}

// ---- batch-inner layout transform + cast (PAPER.md:149 permute to batch-inner, :194-200 FP16) ----
//   in : raw   [B][Q][M][K] complex64, samples contiguous in k (the paper's input layout)
//   out: convb [chunk][M][Q][KBp][N = 2 Bc][8] FP16; k-block kb holds samples 4 (kb - kTcPadBlocks) + u,
//        u = 0..3; column 2 b: (re, im) of frame b per sample; column 2 b + 1: (im, -re) = -j y;
//        zero outside 0 <= k < K.
// One CTA per (m, q, chunk): reads Bc rows of K samples (coalesced along k), transposes through
// shared memory in pieces of 64 samples, writes 16-byte column entries (coalesced along columns).
namespace {
constexpr int kCbSamples = 64;      // samples per piece = 16 k-blocks

__global__ void __launch_bounds__(256)
convert_batch_kernel(const float2* __restrict__ raw, uint4* __restrict__ convb, int M, int Q, int K, int KBp,
                     int Bc, int n_frames, float scale) {
  extern __shared__ __align__(16) unsigned char cb_smem[];
  unsigned* tile = reinterpret_cast<unsigned*>(cb_smem);          // [Bc][kCbSamples + 1] half2 (re, im)
  const int q = blockIdx.x % Q, m = (blockIdx.x / Q) % M, chunk = blockIdx.x / (Q * M);
  const int N = 2 * Bc;
  uint4* row = convb + (((long long)chunk * M + m) * Q + q) * (long long)KBp * N;
  const uint4 zero4 = make_uint4(0u, 0u, 0u, 0u);
  const int Kb = (K + kTcBlk - 1) / kTcBlk;
  // zero pads
  for (int i = threadIdx.x; i < kTcPadBlocks * N; i += blockDim.x) {
    row[i] = zero4;
    row[(long long)(kTcPadBlocks + Kb) * N + i] = zero4;
  }
  for (int k0 = 0; k0 < K; k0 += kCbSamples) {
    __syncthreads();
    for (int i = threadIdx.x; i < Bc * kCbSamples; i += blockDim.x) {
      const int b = i / kCbSamples, kk = i % kCbSamples, k = k0 + kk;
      unsigned v = 0u;
      if (k < K) {
        const float2 s = raw[(((long long)(chunk * Bc + b) * Q + q) * M + m) * K + k];
        const __half2 h = __floats2half2_rn(s.x * scale, s.y * scale);
        v = *reinterpret_cast<const unsigned*>(&h);
      }
      tile[b * (kCbSamples + 1) + kk] = v;
    }
    __syncthreads();
    const int nblk = min(kCbSamples / kTcBlk, Kb - k0 / kTcBlk);
    for (int i = threadIdx.x; i < nblk * N; i += blockDim.x) {
      const int col = i % N, kb = i / N, b = col >> 1;
      unsigned w[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const unsigned v = tile[b * (kCbSamples + 1) + kb * kTcBlk + u];        // (re, im)
        // odd column: (im, -re): swap halves, flip the sign of the new high half
        w[u] = (col & 1) ? (((v >> 16) | (v << 16)) ^ 0x80000000u) : v;
      }
      row[(long long)(kTcPadBlocks + k0 / kTcBlk + kb) * N + col] = make_uint4(w[0], w[1], w[2], w[3]);
    }
  }
}
}  // namespace

cudaError_t launch_convert_batch(const TcPlan* tp, const Params& P, const void* d_raw, void* d_conv,
                                 float scale, cudaStream_t s) {
  const TcDev& dv = tp->dev;
  const size_t smem = (size_t)dv.Bc * (kCbSamples + 1) * 4;
  const long long blocks = (long long)dv.n_chunks * P.M * P.Q;
  convert_batch_kernel<<<(unsigned)blocks, 256, smem, s>>>(static_cast<const float2*>(d_raw), static_cast<uint4*>(d_conv),
                                                             P.M, P.Q, P.K, dv.KBp, dv.Bc, tp->n_frames, scale);
  count_launch();
  return cudaGetLastError();
}

}  // namespace das
