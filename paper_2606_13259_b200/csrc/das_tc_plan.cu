// Host side of the frame-batch tensor-core kernel (das_tc.cuh): applicability, voxel tiles,
// per-tile receiver lists with per-group delay bounds, stage sizing, batch-inner convert kernel.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <numeric>
#include <vector>

#include <cuda.h>

#include "das_tc.cuh"

namespace das {

cudaError_t launch_tc_kernel(const TcDev& tp, const Params& P, const void* tmap, void* d_out, int grid, size_t smem, cudaStream_t s);

struct TcPlan {
  mutable std::atomic<unsigned long long> launches{0};   // epoch of the quad pacing words
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

// [chunk][m][q][N / 8 column groups][2 K rows][8 columns] FP16
size_t tc_converted_bytes(const TcPlan* tp, const Params& P) {
  return (size_t)tp->dev.n_chunks * P.M * P.Q * (size_t)(2 * tp->dev.Bc / 8) * (2 * (size_t)P.K) * 16;
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

static TcPlan* tc_plan_create_groups(const Params& P, const das_plan_desc_t& d, int n_frames, int device, char* why,
                                     size_t why_len, cudaError_t* cuda_err, int groups, bool* retry_narrow);

TcPlan* tc_plan_create(const Params& P, const das_plan_desc_t& d, int n_frames, int device, char* why,
                       size_t why_len, cudaError_t* cuda_err) {
  // kTcG consecutive depths per tile share the staged samples; if the depths of the grid are so far apart in
  // delay that their windows do not fit one box, one depth per tile still works (the other groups stay empty)
  bool retry = false;
  TcPlan* tp = tc_plan_create_groups(P, d, n_frames, device, why, why_len, cuda_err, kTcG, &retry);
  if (!tp && retry && *cuda_err == cudaSuccess) tp = tc_plan_create_groups(P, d, n_frames, device, why, why_len, cuda_err, 1, &retry);
  return tp;
}

static TcPlan* tc_plan_create_groups(const Params& P, const das_plan_desc_t& d, int n_frames, int device, char* why,
                                     size_t why_len, cudaError_t* cuda_err, int groups, bool* retry_narrow) {
  *cuda_err = cudaSuccess;
  *retry_narrow = false;
  auto refuse = [&](const char* msg) -> TcPlan* { snprintf(why, why_len, "%s", msg); return nullptr; };
  // ---- applicability ------------------------------------------------------------------------
  if (!P.iq || !P.fp16) return refuse("the tensor-core path needs IQ data in fp16 storage");
  if (d.interp != DAS_INTERP_LINEAR || d.vox_pos) return refuse("voxel lists / cubic interpolation run in the general kernel");
  if (d.n_tx > 16) return refuse("more than 16 transmits");
  if (d.n_samples < 2 * kTcBoxBig) return refuse("fewer samples per trace than two staged boxes");
  if (n_frames < 8 || n_frames % 8) return refuse("frame count is not a multiple of 8");
  int Bc = n_frames;
  if (n_frames > 64) { if (n_frames % 64) return refuse("frame count above 64 is not a multiple of 64"); Bc = 64; }
  const double z_a = d.elem_pos[2];
  for (int m = 0; m < d.n_elem; ++m)
    if ((double)d.elem_pos[3 * m + 2] != z_a) return refuse("receivers are not in one plane z = const");
  // tilted normals (elem_dir) are fine as long as the positions are coplanar: only the cone turns with the normal
  for (int i = 0; i < d.nz; ++i)
    if (!((double)d.zs[i] > z_a)) return refuse("a voxel plane is not in front of the array (z <= z_array)");

  const double c = d.c, fs = d.fs, fc = d.fc, t_start = d.t_start, fnum = d.f_number;
  const bool apod = fnum > 0.0;
  const double kappa = fs / c;
  const int Q = d.n_tx, M = d.n_elem;
  const int ntx = (d.nx + kTcGX - 1) / kTcGX, nty = (d.ny + kTcGY - 1) / kTcGY, ntz = (d.nz + groups - 1) / groups;
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
        td.ix0 = txi * kTcGX; td.iy0 = ty * kTcGY; td.iz0 = tz * groups;
        td.edge = 0;
        const int ix1 = std::min(td.ix0 + kTcGX, d.nx), iy1 = std::min(td.iy0 + kTcGY, d.ny);
        const int iz1 = std::min(td.iz0 + groups, d.nz);
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
                if (d.tau_tx) tau = d.tau_tx[(size_t)q * d.nx * d.ny * d.nz + ((size_t)i * d.ny + j) * d.nz + k];
                else if (tx.type == DAS_TX_PLANE) tau = (x * tx.v[0] + y * tx.v[1] + z * tx.v[2]) / c + tx.t0;
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
        double a_far = 0.0;                                   // deepest plane of the tile (the axis need not be monotonic)
        for (int k = td.iz0; k < iz1; ++k) a_far = std::max(a_far, (double)d.zs[k] - z_a);
        for (int m = 0; m < M; ++m) {
          const double ex = d.elem_pos[3 * m], ey = d.elem_pos[3 * m + 1];
          const double nx_ = std::max(std::max(xlo - ex, ex - xhi), 0.0), ny_ = std::max(std::max(ylo - ey, ey - yhi), 0.0);
          const double rho_min = std::sqrt(nx_ * nx_ + ny_ * ny_);
          if (apod && d.elem_dir) {
            // tilted cone: bounding-sphere test of the angle between (p - e) and the normal (das_tiled_plan.cu)
            double zlo = 1e300, zhi = -1e300;
            for (int k = td.iz0; k < iz1; ++k) { zlo = std::min(zlo, (double)d.zs[k]); zhi = std::max(zhi, (double)d.zs[k]); }
            const double cx = 0.5 * (xlo + xhi) - ex, cy = 0.5 * (ylo + yhi) - ey, cz = 0.5 * (zlo + zhi) - z_a;
            const double R = 0.5 * std::sqrt((xhi - xlo) * (xhi - xlo) + (yhi - ylo) * (yhi - ylo) + (zhi - zlo) * (zhi - zlo));
            const double dc = std::sqrt(cx * cx + cy * cy + cz * cz);
            if (dc > R) {
              const double ang = std::acos(std::max(-1.0, std::min(1.0, (cx * d.elem_dir[3 * m] + cy * d.elem_dir[3 * m + 1] + cz * d.elem_dir[3 * m + 2]) / dc)));
              if (ang - std::asin(R / dc) > std::atan(cone) * (1.0 + 1e-5) + 1e-7) continue;
            }
          } else if (apod && rho_min > cone * a_far * (1.0 + 1e-5)) continue;
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
  dv.groups = groups;
  dv.n_chunks = n_frames / Bc;
  dv.z_array = z_a; dv.kappa = kappa; dv.ratio = fc / fs;
  dv.phase0 = fc * t_start - std::floor(fc * t_start);
  dv.prof = nullptr;
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
#ifdef DAS_TUNING
  if (getenv("DAS_TC_VERBOSE")) {
    long long tw = 0; for (int w_ : work) tw += w_;
    fprintf(stderr, "[das tc plan] tiles %d, list entries %zu, MMA passes %lld, widest item %d samples, error bits %d\n", n_tiles, list.size(), tw, stats[0], stats[1]);
  }
#endif
  if (stats[1] & 1) return refuse_free("a sample window of a voxel group needs more than 2 MMA passes (grid too coarse)");
  if (stats[1] & 2) {
    *retry_narrow = groups > 1 && !(stats[1] & 1);
    return refuse_free("the sample windows of a tile's voxel groups do not fit one staged box (grid too coarse)");
  }
  if (stats[1] & 4) return refuse_free("internal: window start out of range");

  // Tile order: depth slab by depth slab (heaviest slab first), inside a slab 2 x 2 blocks of laterally adjacent
  // tiles ("quads", heaviest first), the four tiles of a quad side by side in the list.  The grid is a multiple of
  // four CTAs and CTA c takes the list entries c, c + grid, ..., so CTAs 4 j .. 4 j + 3 always hold one quad: their
  // receiver lists and sample windows overlap almost entirely, and the kernel's producers pace each other (das_tc.cu,
  // "quad pacing") so that the windows one CTA pulls from HBM are found in L2 by the other three.  A quad at the
  // rim of an odd tile grid is filled up with empty tiles.
  std::vector<double> slab_work(ntz, 0.0);
  for (int i = 0; i < n_tiles; ++i) slab_work[i / (ntx * nty)] += work[i];
  const int nqx = (ntx + 1) / 2, nqy = (nty + 1) / 2;
  struct Quad { int tz; int t[4]; double w; };
  std::vector<Quad> quads;
  quads.reserve((size_t)ntz * nqx * nqy);
  for (int tz = 0; tz < ntz; ++tz)
    for (int qy = 0; qy < nqy; ++qy)
      for (int qx = 0; qx < nqx; ++qx) {
        Quad qd{tz, {-1, -1, -1, -1}, 0.0};
        for (int mth = 0; mth < 4; ++mth) {
          const int txi = 2 * qx + (mth & 1), ty = 2 * qy + (mth >> 1);
          if (txi < ntx && ty < nty) { qd.t[mth] = (tz * nty + ty) * ntx + txi; qd.w += work[qd.t[mth]]; }
        }
        quads.push_back(qd);
      }
  std::stable_sort(quads.begin(), quads.end(), [&](const Quad& a, const Quad& b) {
    if (a.tz != b.tz) return slab_work[a.tz] > slab_work[b.tz];
    return a.w > b.w;
  });
  const int n_tiles_q = 4 * (int)quads.size();
  std::vector<TcTile> tiles_s(n_tiles_q);
  std::vector<int> tbase_s((size_t)n_tiles_q * Q, 0);
  for (size_t u = 0; u < quads.size(); ++u)
    for (int mth = 0; mth < 4; ++mth) {
      const size_t i = 4 * u + mth;
      const int t0 = quads[u].t[mth];
      if (t0 >= 0) {
        tiles_s[i] = tiles[t0];
        tiles_s[i].edge = edge[t0];
        std::memcpy(&tbase_s[i * Q], &tbase[(size_t)t0 * Q], sizeof(int) * Q);
      } else {
        tiles_s[i] = TcTile{d.nx, d.ny, d.nz, 0, 0, 0};        // no voxel, no receiver
      }
    }
  dv.n_tiles = n_tiles_q;
  if ((e = up(tp, tiles_s, &dv.tiles)) != cudaSuccess || (e = up(tp, tbase_s, &dv.tbase)) != cudaSuccess) return fail(e);

  static_assert(kTcG * 2 * 64 + kTcG * kTcABufs * kTcACols <= kTcTmemCols, "accumulators + A slots exceed tensor memory");
  // Stage ring: `qs` boxes (consecutive transmits of one receiver) per stage, one barrier round per qs items
  // (the producer and the MMA issuers are serial latency chains), and as many stages as shared memory holds
  // (boxes in flight = what covers the L2 / HBM latency of the TMA copies).
  dv.qs = std::min(8, Q);
#ifdef DAS_TUNING
  if (const char* ev = getenv("DAS_TC_QS")) dv.qs = std::min(kTcMaxQs, std::max(1, atoi(ev)));
#endif
  while (dv.qs > 1 && tc_smem_bytes(Bc, dv.qs, kTcMinStages) > 200 * 1024) dv.qs /= 2;
  dv.n_stages = kTcMinStages;
  while (dv.n_stages < 6 && tc_smem_bytes(Bc, dv.qs, dv.n_stages + 1) <= 200 * 1024) ++dv.n_stages;
#ifdef DAS_TUNING
  if (const char* ev = getenv("DAS_TC_STAGES")) dv.n_stages = std::min(kTcMaxStages, std::max(kTcMinStages, atoi(ev)));
#endif
  while (dv.n_stages > kTcMinStages && tc_smem_bytes(Bc, dv.qs, dv.n_stages) > 200 * 1024) --dv.n_stages;
  tp->smem = tc_smem_bytes(Bc, dv.qs, dv.n_stages);
  if (tp->smem > 200 * 1024) return refuse_free("stage ring does not fit in shared memory");
  tp->grid = std::max(4, std::min(dv.n_tiles * dv.n_chunks, prop.multiProcessorCount) / 4 * 4);
  // quad pacing: one progress word per CTA; the lead in receivers is 16 unless the descriptor's debug field says
  // otherwise (-1 = no pacing)
  dv.pace = d.debug_tc_pace > 0 ? d.debug_tc_pace : (d.debug_tc_pace < 0 ? 0 : 16);
  dv.pace_mask = 3;
#ifdef DAS_TUNING
  if (const char* ev = getenv("DAS_TC_PACE")) dv.pace = atoi(ev);
  if (const char* ev = getenv("DAS_TC_PACE_MASK")) dv.pace_mask = atoi(ev);
#endif
  dv.progress = nullptr;
  dv.epoch = 0;
  if (dv.pace > 0) {
    void* dp = nullptr;
    if ((e = cudaMalloc(&dp, sizeof(unsigned long long) * tp->grid)) != cudaSuccess) return fail(e);
    tp->allocs.push_back(dp);
    if ((e = cudaMemset(dp, 0, sizeof(unsigned long long) * tp->grid)) != cudaSuccess) return fail(e);
    dv.progress = static_cast<unsigned long long*>(dp);
  }
  return tp;
}

// The TMA descriptor of the converted data (caller-owned buffer, so it is encoded per launch: a host-side
// table fill, no driver call into the device).  3-D tensor of FP16:
//   dim 0: one column group's record, 2 K rows (16 bytes each) per sample, contiguous
//   dim 1: the N / 8 column groups of a record      dim 2: the records (chunk, m, q)
// box = (2 box_samples K rows, N / 8, 1): lands in shared memory as [column group][K row][8 columns], the
// MN-major no-swizzle operand layout of tcgen05.mma with SBO = (K rows of the box) * 16 bytes.  Out-of-range K rows (before
// sample 0, beyond sample K - 1) are filled with zeros by the TMA unit: no padding in memory.
namespace {
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
cudaError_t tc_encode_map(const TcPlan* tp, const Params& P, const void* d_conv, int box_samples, CUtensorMap* map) {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q);
    if (e != cudaSuccess) return e;
    if (!p || q != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
    fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  const cuuint64_t J = (cuuint64_t)(2 * tp->dev.Bc / 8);
  // elements are 32-bit words (the box's inner extent is limited to 256 ELEMENTS): 4 per K row
  const cuuint64_t dims[3] = {8ull * (cuuint64_t)P.K, J, (cuuint64_t)tp->dev.n_chunks * P.M * P.Q};
  const cuuint64_t strides[2] = {dims[0] * 4ull, dims[0] * 4ull * J};
  const cuuint32_t box[3] = {8u * (cuuint32_t)box_samples, (cuuint32_t)J, 1u};
  const cuuint32_t estr[3] = {1u, 1u, 1u};
  const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_UINT32, 3, const_cast<void*>(d_conv), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}
}  // namespace

cudaError_t launch_tc(const TcPlan* tp, const Params& P, const void* d_conv, void* d_out, cudaStream_t s) {
  count_launch();
  alignas(64) CUtensorMap map[2];
  cudaError_t me = tc_encode_map(tp, P, d_conv, kTcBoxSmall, &map[0]);
  if (me == cudaSuccess) me = tc_encode_map(tp, P, d_conv, kTcBoxBig, &map[1]);
  if (me != cudaSuccess) return me;
#ifdef DAS_TC_PROF
  // development aid: cycle accounting per warp role, printed after a synchronising launch
  if (getenv("DAS_TC_PROF")) {
    TcDev dv = tp->dev;
    const size_t n = (size_t)tp->grid * 32 * 8;
    cudaMalloc(&dv.prof, n * sizeof(unsigned long long));
    cudaMemset(dv.prof, 0, n * sizeof(unsigned long long));
    cudaError_t e = launch_tc_kernel(dv, P, map, d_out, tp->grid, tp->smem, s);
    cudaStreamSynchronize(s);
    std::vector<unsigned long long> h(n);
    cudaMemcpy(h.data(), dv.prof, n * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
    cudaFree(dv.prof);
    double acc[20][8] = {};
    for (int c = 0; c < tp->grid; ++c) for (int w = 0; w < 20; ++w) for (int k = 0; k < 8; ++k) acc[w][k] += (double)h[((size_t)c * 32 + w) * 8 + k] / tp->grid;
    for (int w = 0; w < 20; ++w)
      fprintf(stderr, "[tc prof] warp %2d total %.3e  w1 %.3e w2 %.3e w3 %.3e w4 %.3e w5 %.3e w6 %.3e\n", w, acc[w][0], acc[w][1], acc[w][2], acc[w][3], acc[w][4], acc[w][5], acc[w][6]);
    return e;
  }
#endif
  TcDev dv = tp->dev;
  dv.epoch = (tp->launches.fetch_add(1) + 1) << 40;       // concurrent launches of one plan only blur the pacing (it is advisory)
  return launch_tc_kernel(dv, P, map, d_out, tp->grid, tp->smem, s);
}

// ---- batch-inner layout transform + cast (PAPER.md:149 permute to batch-inner, :194-200 FP16) ----
//   in : raw   [B][Q][M][K] complex64, samples contiguous in k (the paper's input layout)
//   out: convb [chunk][M][Q][J = 2 Bc / 8][2 K][8] FP16.  Record (chunk, m, q), column group j (the frames
//        4 j .. 4 j + 3 of the chunk), K row 2 k holds y_k of those frames as (re, im) pairs, K row 2 k + 1
//        holds -j y_k = (im, -re): one real MMA then yields Re and Im of the complex product (das_tc.cuh).
//        No padding: the TMA copies of tc_kernel fill the rows outside 0 <= k < K with zeros.
// One CTA per (m, q, chunk): reads Bc rows of K samples (coalesced along k), transposes through
// shared memory in pieces of 64 samples, writes 32-byte row pairs (coalesced along k within a column group).
namespace {
constexpr int kCbSamples = 64;      // samples per piece

__global__ void __launch_bounds__(256)
convert_batch_kernel(const float2* __restrict__ raw, uint4* __restrict__ convb, int M, int Q, int K,
                     int Bc, int n_frames, float scale) {
  extern __shared__ __align__(16) unsigned char cb_smem[];
  unsigned* tile = reinterpret_cast<unsigned*>(cb_smem);          // [Bc][kCbSamples + 1] half2 (re, im)
  const int q = blockIdx.x % Q, m = (blockIdx.x / Q) % M, chunk = blockIdx.x / (Q * M);
  const int J = 2 * Bc / 8;
  uint4* rec = convb + (((long long)chunk * M + m) * Q + q) * (long long)J * (2LL * K);
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
    const int nk = min(kCbSamples, K - k0);
    for (int i = threadIdx.x; i < J * nk; i += blockDim.x) {
      const int j = i / nk, kk = i % nk;
      unsigned y[4], z[4];
#pragma unroll
      for (int f = 0; f < 4; ++f) {
        const unsigned v = tile[(4 * j + f) * (kCbSamples + 1) + kk];             // (re, im)
        y[f] = v;
        z[f] = ((v >> 16) | (v << 16)) ^ 0x80000000u;                              // (im, -re): swap halves, flip the new high half
      }
      uint4* dst = rec + ((long long)j * (2LL * K) + 2LL * (k0 + kk));
      dst[0] = make_uint4(y[0], y[1], y[2], y[3]);
      dst[1] = make_uint4(z[0], z[1], z[2], z[3]);
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
                                                             P.M, P.Q, P.K, dv.Bc, tp->n_frames, scale);
  count_launch();
  return cudaGetLastError();
}

}  // namespace das
