// Host side of the tiled kernel: applicability test, tile list, per-tile receiver lists,
// window origins, window size selection, work-sorted static schedule.  See das_tiled.cuh.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <numeric>
#include <vector>

#include "das_tiled.cuh"

namespace das {

struct TiledPlan {
  TiledDev dev{};
  int QC = 16, W = 16, grid = 1;
  std::vector<void*> allocs;
};

void tiled_plan_destroy(TiledPlan* tp) {
  if (!tp) return;
  for (void* d : tp->allocs) cudaFree(d);
  delete tp;
}

namespace {
template <typename T>
cudaError_t up(TiledPlan* tp, const std::vector<T>& h, const T** d_out) {
  void* d = nullptr;
  cudaError_t e = cudaMalloc(&d, std::max<size_t>(h.size(), 1) * sizeof(T));
  if (e != cudaSuccess) return e;
  tp->allocs.push_back(d);
  if (!h.empty()) e = cudaMemcpy(d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
  *d_out = static_cast<const T*>(d);
  return e;
}
// receive excess path |d| - a for lateral offset rho and depth a > 0 (metres)
inline double excess(double rho, double a) { return rho * rho / (a + std::sqrt(rho * rho + a * a)); }
inline int floor_to_multiple(int v, int a) { int r = v % a; if (r < 0) r += a; return v - r; }
}  // namespace

TiledPlan* tiled_plan_create(const Params& P, const das_plan_desc_t& d, int device, char* why,
                             size_t why_len, cudaError_t* cuda_err) {
  *cuda_err = cudaSuccess;
  auto refuse = [&](const char* msg) -> TiledPlan* { snprintf(why, why_len, "%s", msg); return nullptr; };
  // ---- applicability ------------------------------------------------------------------------
  if (d.n_elem > 65535) return refuse("more than 65535 receivers");
  if (d.interp != DAS_INTERP_LINEAR || d.vox_pos) return refuse("voxel lists / cubic interpolation run in the general kernel");
  const double z_a = d.elem_pos[2];
  for (int m = 0; m < d.n_elem; ++m)
    if ((double)d.elem_pos[3 * m + 2] != z_a) return refuse("receivers are not in one plane z = const");
  // tilted normals (elem_dir) are fine as long as the POSITIONS are coplanar: the delays are those of the
  // planar array, only the f-number cone turns with the normal
  for (int i = 0; i < d.nz; ++i)
    if (!((double)d.zs[i] > z_a)) return refuse("a voxel plane is not in front of the array (z <= z_array)");

  const double c = d.c, fs = d.fs, fc = d.fc, t_start = d.t_start, fnum = d.f_number;
  const bool apod = fnum > 0.0;
  const double kappa = fs / c;
  const int Q = d.n_tx, M = d.n_elem;
  const int st = storage_code(P.fp16, P.fp8);
  const int align = 16 / entry_bytes(P.iq, st);         // window origins in units the TMA copy accepts
  const int TXv = kWX * kLaneX, TYv = kWY * kLaneY, TZv = kWZ;
  const int ntx = (d.nx + TXv - 1) / TXv, nty = (d.ny + TYv - 1) / TYv, ntz = (d.nz + TZv - 1) / TZv;
  const long long n_tiles_ll = (long long)ntx * nty * ntz;
  if (n_tiles_ll > (1 << 24)) return refuse("too many tiles");
  const int n_tiles = (int)n_tiles_ll;

  int QC = 16;
  if (Q <= 1) QC = 1; else if (Q <= 2) QC = 2; else if (Q <= 4) QC = 4; else if (Q <= 8) QC = 8;

  std::vector<TileDesc> tiles(n_tiles);
  std::vector<int> k0tile((size_t)n_tiles * Q);
  std::vector<unsigned> list;
  std::vector<double> work(n_tiles, 0.0);
  list.reserve((size_t)n_tiles * std::min(M, 256));
  double w_needed = 0.0;

  int t = 0;
  for (int tz = 0; tz < ntz; ++tz)
    for (int ty = 0; ty < nty; ++ty)
      for (int txi = 0; txi < ntx; ++txi, ++t) {
        TileDesc& td = tiles[t];
        td.ix0 = txi * TXv; td.iy0 = ty * TYv; td.iz0 = tz * TZv;
        const int ix1 = std::min(td.ix0 + TXv, d.nx), iy1 = std::min(td.iy0 + TYv, d.ny), iz1 = std::min(td.iz0 + TZv, d.nz);
        double xlo = 1e300, xhi = -1e300, ylo = 1e300, yhi = -1e300, zlo = 1e300, zhi = -1e300;
        for (int i = td.ix0; i < ix1; ++i) { xlo = std::min(xlo, (double)d.xs[i]); xhi = std::max(xhi, (double)d.xs[i]); }
        for (int i = td.iy0; i < iy1; ++i) { ylo = std::min(ylo, (double)d.ys[i]); yhi = std::max(yhi, (double)d.ys[i]); }
        for (int i = td.iz0; i < iz1; ++i) { zlo = std::min(zlo, (double)d.zs[i]); zhi = std::max(zhi, (double)d.zs[i]); }
        const double a_lo = zlo - z_a, a_hi = zhi - z_a;
        // transmit part: bounds of T_q = (tau_tx + a/c - t_start) fs over the tile box
        double span_t_max = 0.0;
        for (int q = 0; q < Q; ++q) {
          const das_transmit_t& tx = d.tx[q];
          const double v[3] = {tx.v[0], tx.v[1], tx.v[2]};
          const double bl[3] = {xlo, ylo, zlo}, bh[3] = {xhi, yhi, zhi};
          double lo = 0.0, hi = 0.0;
          if (tx.type == DAS_TX_PLANE) {
            for (int k = 0; k < 3; ++k) { lo += std::min(v[k] * bl[k], v[k] * bh[k]); hi += std::max(v[k] * bl[k], v[k] * bh[k]); }
          } else {
            double dmin2 = 0.0, dmax2 = 0.0;
            for (int k = 0; k < 3; ++k) {
              const double near = std::max(std::max(bl[k] - v[k], v[k] - bh[k]), 0.0);
              const double far = std::max(std::fabs(bl[k] - v[k]), std::fabs(bh[k] - v[k]));
              dmin2 += near * near; dmax2 += far * far;
            }
            lo = std::sqrt(dmin2); hi = std::sqrt(dmax2);
          }
          double t_lo = (lo / c + tx.t0 + a_lo / c - t_start) * fs;
          double t_hi = (hi / c + tx.t0 + a_hi / c - t_start) * fs;
          if (d.tau_tx) {
            // transmit delays from the table: exact bounds of T_q over the voxels of the tile
            t_lo = 1e300; t_hi = -1e300;
            for (int i = td.ix0; i < ix1; ++i)
              for (int j = td.iy0; j < iy1; ++j)
                for (int k = td.iz0; k < iz1; ++k) {
                  const double tau = d.tau_tx[(size_t)q * d.nx * d.ny * d.nz + ((size_t)i * d.ny + j) * d.nz + k];
                  const double T = (tau + ((double)d.zs[k] - z_a) / c - t_start) * fs;
                  t_lo = std::min(t_lo, T); t_hi = std::max(t_hi, T);
                }
          }
          if (!(std::fabs(t_lo) < 1e9 && std::fabs(t_hi) < 1e9)) return refuse("sample coordinate out of int range");
          // Tf = T - k0 - 1/2 >= 1/2: the rounded entry index can never be negative
          const int k0 = floor_to_multiple((int)std::floor(t_lo) - 1, align);
          k0tile[(size_t)t * Q + q] = k0;
          span_t_max = std::max(span_t_max, t_hi - (double)k0);
        }
        // receiver part: active list, E0 and the span of e over the (active part of the) tile
        td.list_off = (int)list.size();
        const double cone = apod ? 1.0 / (2.0 * fnum) : 0.0;
        double span_e_max = 0.0;
        for (int m = 0; m < M; ++m) {
          const double ex = d.elem_pos[3 * m], ey = d.elem_pos[3 * m + 1];
          const double nx_ = std::max(std::max(xlo - ex, ex - xhi), 0.0), ny_ = std::max(std::max(ylo - ey, ey - yhi), 0.0);
          const double fx = std::max(std::fabs(xlo - ex), std::fabs(xhi - ex)), fy = std::max(std::fabs(ylo - ey), std::fabs(yhi - ey));
          const double rho_min = std::sqrt(nx_ * nx_ + ny_ * ny_), rho_max = std::sqrt(fx * fx + fy * fy);
          double e_hi = excess(rho_max, a_lo);
          if (apod && d.elem_dir) {
            // tilted cone: a voxel is active iff the angle between (p - e) and the normal is <= atan(1 / (2 f#)).
            // Over the tile that angle is at least angle(centre) - (angular radius of the tile's bounding sphere).
            const double nv[3] = {d.elem_dir[3 * m], d.elem_dir[3 * m + 1], d.elem_dir[3 * m + 2]};
            const double cx = 0.5 * (xlo + xhi) - ex, cy = 0.5 * (ylo + yhi) - ey, cz = 0.5 * (zlo + zhi) - z_a;
            const double R = 0.5 * std::sqrt((xhi - xlo) * (xhi - xlo) + (yhi - ylo) * (yhi - ylo) + (zhi - zlo) * (zhi - zlo));
            const double dc = std::sqrt(cx * cx + cy * cy + cz * cz);
            const double theta_c = std::atan(cone);
            if (dc > R) {
              const double ang = std::acos(std::max(-1.0, std::min(1.0, (cx * nv[0] + cy * nv[1] + cz * nv[2]) / dc)));
              if (ang - std::asin(R / dc) > theta_c * (1.0 + 1e-5) + 1e-7) continue;   // no voxel of the tile sees m
            }
            // lateral reach of the tilted cone at the deepest plane of the tile bounds the excess path
            const double tilt = std::acos(std::max(-1.0, std::min(1.0, nv[2])));
            const double reach = theta_c + tilt;
            if (reach < 1.5) e_hi = std::min(e_hi, excess(std::tan(reach) * a_hi * (1.0 + 1e-5), a_hi));
          } else if (apod) {
            if (rho_min > cone * a_hi * (1.0 + 1e-5)) continue;             // no voxel of the tile sees m
            e_hi = std::min(e_hi, excess(cone * a_hi * (1.0 + 1e-5), a_hi));
          }
          const double e_lo = excess(rho_min, a_hi);
          const int e0 = floor_to_multiple(std::max((int)std::floor(e_lo * kappa), 0), align);
          if (e0 > 65535) return refuse("receive delay offset exceeds 16 bits");
          span_e_max = std::max(span_e_max, e_hi * kappa - (double)e0);
          list.push_back((unsigned)m | ((unsigned)e0 << 16));
          work[t] += 1.0;
        }
        td.list_cnt = (int)list.size() - td.list_off;
        if (td.list_cnt) w_needed = std::max(w_needed, span_t_max + span_e_max);
      }

  // entry index = round(Tf + e') with Tf + e' in [1/2, span_t + span_e - 1/2]: it must stay <= W - 1
  int W = 0;
  for (int cand : kWindows)                                // a staged row (W entries) must be a whole number of 16-byte units
    if (w_needed + 0.02 <= (double)cand && (cand * entry_bytes(P.iq, st)) % 16 == 0) { W = cand; break; }
  if (!W) { snprintf(why, why_len, "sample window per tile (%.1f samples) exceeds the largest staged window (%d)", w_needed, kWindows[sizeof(kWindows) / sizeof(int) - 1]); return nullptr; }

  // order tiles by decreasing work (static round-robin schedule over persistent CTAs)
  std::vector<int> order(n_tiles);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return work[a] > work[b]; });
  std::vector<TileDesc> tiles_sorted(n_tiles);
  std::vector<int> k0_sorted((size_t)n_tiles * Q);
  for (int i = 0; i < n_tiles; ++i) {
    tiles_sorted[i] = tiles[order[i]];
    std::memcpy(&k0_sorted[(size_t)i * Q], &k0tile[(size_t)order[i] * Q], sizeof(int) * Q);
  }

  TiledPlan* tp = new TiledPlan();
  tp->QC = QC; tp->W = W;
  cudaDeviceProp prop;
  cudaError_t e = cudaGetDeviceProperties(&prop, device);
  if (e != cudaSuccess) { *cuda_err = e; delete tp; return nullptr; }
  const size_t smem = tiled_smem_bytes(QC, W, P.iq, st);
  const int ctas_per_sm = (smem + 1024) * 2 <= (size_t)prop.sharedMemPerMultiprocessor ? 2 : 1;
  tp->grid = std::max(1, std::min(n_tiles, prop.multiProcessorCount * ctas_per_sm));
  if (d.debug_tiled_grid > 0) tp->grid = std::max(1, std::min(n_tiles, d.debug_tiled_grid));      // das.h: debugging aid
#ifdef DAS_TUNING
  if (getenv("DAS_TC_VERBOSE")) fprintf(stderr, "[das tiled plan] tiles %d, QC %d, W %d, smem %zu, grid %d\n", n_tiles, QC, W, smem, tp->grid);
#endif
  TiledDev& dv = tp->dev;
  dv.n_tiles = n_tiles;
  dv.n_chunks = (Q + QC - 1) / QC;
  dv.z_array = z_a; dv.kappa = kappa; dv.ratio = fc / fs;
  dv.phase0 = fc * t_start - std::floor(fc * t_start);
  dv.four_f2 = (float)(4.0 * fnum * fnum);
  dv.kappa_f = (float)kappa; dv.ratio_f = (float)(fc / fs);
  dv.addr_bias = 0u - (kMagicBits << (P.iq ? 4 : 3));
  if ((e = up(tp, tiles_sorted, &dv.tiles)) != cudaSuccess || (e = up(tp, k0_sorted, &dv.k0tile)) != cudaSuccess ||
      (e = up(tp, list, &dv.list)) != cudaSuccess) {
    *cuda_err = e; tiled_plan_destroy(tp); return nullptr;
  }
  return tp;
}

cudaError_t launch_tiled(const TiledPlan* tp, const Params& P, const void* d_conv, void* d_out,
                         cudaStream_t s, int* n_launches) {
  *n_launches = 1;
  count_launch();
  if (P.fp8) return P.iq ? launch_tiled_iq8(tp->QC, tp->W, tp->dev, P, d_conv, d_out, tp->grid, s)
                         : launch_tiled_rf8(tp->QC, tp->W, tp->dev, P, d_conv, d_out, tp->grid, s);
  if (P.iq) return P.fp16 ? launch_tiled_iq16(tp->QC, tp->W, tp->dev, P, d_conv, d_out, tp->grid, s)
                          : launch_tiled_iq32(tp->QC, tp->W, tp->dev, P, d_conv, d_out, tp->grid, s);
  return P.fp16 ? launch_tiled_rf16(tp->QC, tp->W, tp->dev, P, d_conv, d_out, tp->grid, s)
                : launch_tiled_rf32(tp->QC, tp->W, tp->dev, P, d_conv, d_out, tp->grid, s);
}

}  // namespace das
