// C ABI of libdas_b200.so (include/das.h): plan creation / validation, dispatch, errors.
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <initializer_list>
#include <new>
#include <vector>

#include "das_internal.cuh"
#include "das_tc.cuh"

namespace das {

static std::atomic<unsigned long long> g_launches{0};
void count_launch(unsigned long long n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

static thread_local char g_err[512] = "";

static void set_err(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

static das_status_t cuda_fail(cudaError_t e, const char* what) {
  set_err("%s: %s (%s)", what, cudaGetErrorString(e), cudaGetErrorName(e));
  return DAS_ERR_CUDA;
}

// Restores the caller's current device on scope exit.
struct DeviceGuard {
  int prev = -1;
  bool ok = false;
  cudaError_t err = cudaSuccess;
  explicit DeviceGuard(int dev) {
    err = cudaGetDevice(&prev);
    if (err != cudaSuccess) return;
    if (prev != dev) {
      err = cudaSetDevice(dev);
      if (err != cudaSuccess) return;
    }
    ok = true;
  }
  ~DeviceGuard() { if (ok && prev >= 0) cudaSetDevice(prev); }
};

}  // namespace das

using namespace das;

struct das_plan {
  Params P{};
  int device = 0;
  int algo = DAS_ALGO_GENERAL;
  size_t raw_bytes = 0, conv_bytes = 0, out_bytes = 0;
  std::vector<void*> dev_allocs;          // geometry tables
  TiledPlan* tiled = nullptr;
  TcPlan* tc = nullptr;
  int frames = 1;                         // B
  size_t raw1 = 0, conv1 = 0, out1 = 0;   // per-frame sizes (frame-by-frame path)
  // staging for das_beamform_host[_begin / _wait] (lazy): two raw / output slots, one converted buffer
  struct HostSlot {
    void* d_raw = nullptr;
    void* d_out = nullptr;
    cudaEvent_t ev_h2d = nullptr, ev_exec = nullptr, ev_d2h = nullptr;
    bool used = false;           // ev_exec / ev_d2h have been recorded at least once
  } slot[2];
  void* st_conv = nullptr;
  cudaStream_t s_in = nullptr, s_out = nullptr;
  unsigned long long begun = 0, waited = 0;
};

static void free_plan(das_plan* p) {
  if (!p) return;
  DeviceGuard g(p->device);
  if (p->tiled) tiled_plan_destroy(p->tiled);
  if (p->tc) tc_plan_destroy(p->tc);
  for (void* d : p->dev_allocs) cudaFree(d);
  for (auto& sl : p->slot) {
    if (sl.d_raw) cudaFree(sl.d_raw);
    if (sl.d_out) cudaFree(sl.d_out);
    if (sl.ev_h2d) cudaEventDestroy(sl.ev_h2d);
    if (sl.ev_exec) cudaEventDestroy(sl.ev_exec);
    if (sl.ev_d2h) cudaEventDestroy(sl.ev_d2h);
  }
  if (p->st_conv) cudaFree(p->st_conv);
  if (p->s_in) cudaStreamDestroy(p->s_in);
  if (p->s_out) cudaStreamDestroy(p->s_out);
  delete p;
}

template <typename T>
static cudaError_t upload(das_plan* p, const std::vector<T>& h, const T** d_out) {
  void* d = nullptr;
  cudaError_t e = cudaMalloc(&d, h.size() * sizeof(T));
  if (e != cudaSuccess) return e;
  p->dev_allocs.push_back(d);
  e = cudaMemcpy(d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
  *d_out = static_cast<const T*>(d);
  return e;
}

static bool finite_all(const float* p, long long n) {
  for (long long i = 0; i < n; ++i) if (!std::isfinite(p[i])) return false;
  return true;
}

extern "C" {
#pragma GCC visibility push(default)

const char* das_status_string(das_status_t s) {
  switch (s) {
    case DAS_OK: return "DAS_OK";
    case DAS_ERR_INVALID_ARG: return "DAS_ERR_INVALID_ARG";
    case DAS_ERR_UNSUPPORTED: return "DAS_ERR_UNSUPPORTED";
    case DAS_ERR_ALLOC: return "DAS_ERR_ALLOC";
    case DAS_ERR_CUDA: return "DAS_ERR_CUDA";
    case DAS_ERR_SIZE: return "DAS_ERR_SIZE";
  }
  return "DAS_ERR_UNKNOWN";
}

const char* das_last_error(void) { return g_err; }

unsigned long long das_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

das_status_t das_plan_create(const das_plan_desc_t* d, das_plan_t** out_plan) {
  g_err[0] = 0;
  if (!out_plan) { set_err("out_plan is NULL"); return DAS_ERR_INVALID_ARG; }
  *out_plan = nullptr;
  if (!d) { set_err("desc is NULL"); return DAS_ERR_INVALID_ARG; }
  if (!d->elem_pos || !d->tx || (!d->vox_pos && (!d->xs || !d->ys || !d->zs))) {
    set_err("elem_pos, tx, xs, ys, zs must be non-NULL"); return DAS_ERR_INVALID_ARG;
  }
  if (d->n_elem < 1 || d->n_tx < 1 || d->nx < 1 || d->ny < 1 || d->nz < 1) {
    set_err("n_elem, n_tx, nx, ny, nz must be >= 1"); return DAS_ERR_INVALID_ARG;
  }
  if (d->n_samples < 2) { set_err("n_samples must be >= 2 (linear interpolation needs k and k+1)"); return DAS_ERR_INVALID_ARG; }
  if (!(std::isfinite(d->c) && d->c > 0.f)) { set_err("c must be finite and > 0"); return DAS_ERR_INVALID_ARG; }
  if (!(std::isfinite(d->fs) && d->fs > 0.f)) { set_err("fs must be finite and > 0"); return DAS_ERR_INVALID_ARG; }
  if (!(std::isfinite(d->fc) && d->fc >= 0.f)) { set_err("fc must be finite and >= 0"); return DAS_ERR_INVALID_ARG; }
  if (!std::isfinite(d->t_start)) { set_err("t_start must be finite"); return DAS_ERR_INVALID_ARG; }
  if (!std::isfinite(d->f_number)) { set_err("f_number must be finite"); return DAS_ERR_INVALID_ARG; }
  if (d->data_kind != DAS_DATA_IQ && d->data_kind != DAS_DATA_RF) { set_err("unknown data_kind %d", d->data_kind); return DAS_ERR_UNSUPPORTED; }
  if (d->storage != DAS_STORE_FP32 && d->storage != DAS_STORE_FP16 && d->storage != DAS_STORE_FP8) { set_err("unknown storage %d", d->storage); return DAS_ERR_UNSUPPORTED; }
  if (d->algo != DAS_ALGO_AUTO && d->algo != DAS_ALGO_GENERAL && d->algo != DAS_ALGO_TILED && d->algo != DAS_ALGO_TC) { set_err("unknown algo %d", d->algo); return DAS_ERR_UNSUPPORTED; }
  if (d->n_frames < 0 || d->n_frames > 4096) { set_err("n_frames = %d is outside [0, 4096]", d->n_frames); return DAS_ERR_INVALID_ARG; }
  if (d->algo == DAS_ALGO_TC) {
    const int B = d->n_frames;
    if (B < 8 || B % 8 || (B > 64 && B % 64) || d->data_kind != DAS_DATA_IQ || d->storage != DAS_STORE_FP16 || d->n_tx > 16) {
      set_err("DAS_ALGO_TC needs n_frames a multiple of 8 (of 64 above 64), IQ data, fp16 storage and <= 16 transmits");
      return DAS_ERR_UNSUPPORTED;
    }
  }
  if (d->data_kind == DAS_DATA_RF && d->fc != 0.f) { set_err("fc must be 0 for RF data (no phase rotation)"); return DAS_ERR_INVALID_ARG; }
  if (d->window != DAS_WINDOW_BOXCAR && d->window != DAS_WINDOW_HANN && d->window != DAS_WINDOW_TUKEY) { set_err("unknown window %d", d->window); return DAS_ERR_UNSUPPORTED; }
  if (d->window == DAS_WINDOW_TUKEY && !(d->window_param > 0.f && d->window_param <= 1.f)) { set_err("the Tukey taper must lie in (0, 1]"); return DAS_ERR_INVALID_ARG; }
  if (d->interp != DAS_INTERP_LINEAR && d->interp != DAS_INTERP_CUBIC) { set_err("unknown interp %d", d->interp); return DAS_ERR_UNSUPPORTED; }
  if (d->interp == DAS_INTERP_CUBIC && d->n_samples < 4) { set_err("cubic interpolation needs n_samples >= 4"); return DAS_ERR_INVALID_ARG; }
  if (d->vox_pos && (d->ny != 1 || d->nz != 1)) { set_err("with a voxel list set nx = N, ny = nz = 1"); return DAS_ERR_INVALID_ARG; }
  if ((d->obs_off != nullptr) != (d->obs_q != nullptr)) { set_err("obs_off and obs_q go together"); return DAS_ERR_INVALID_ARG; }
  const bool general_only = d->vox_pos != nullptr || d->interp == DAS_INTERP_CUBIC;
  if (general_only && (d->algo == DAS_ALGO_TILED || d->algo == DAS_ALGO_TC)) {
    set_err("voxel lists and cubic interpolation run in the general kernel only"); return DAS_ERR_UNSUPPORTED;
  }
  if (!finite_all(d->elem_pos, 3LL * d->n_elem) || (!d->vox_pos && (!finite_all(d->xs, d->nx) ||
      !finite_all(d->ys, d->ny) || !finite_all(d->zs, d->nz))) ||
      (d->elem_dir && !finite_all(d->elem_dir, 3LL * d->n_elem)) || (d->vox_pos && !finite_all(d->vox_pos, 3LL * d->nx))) {
    set_err("non-finite geometry value"); return DAS_ERR_INVALID_ARG;
  }
  {
    const long long NQ = (long long)d->nx * d->ny * d->nz * d->n_tx;
    if ((d->tau_tx && !finite_all(d->tau_tx, NQ)) || (d->w_tx && !finite_all(d->w_tx, NQ))) {
      set_err("non-finite value in a transmit table"); return DAS_ERR_INVALID_ARG;
    }
  }
  for (int q = 0; q < d->n_tx; ++q) {
    const das_transmit_t& t = d->tx[q];
    if (t.type != DAS_TX_PLANE && t.type != DAS_TX_DIVERGING) { set_err("tx[%d]: unknown type %d", q, t.type); return DAS_ERR_UNSUPPORTED; }
    if (!finite_all(t.v, 3) || !std::isfinite(t.t0)) { set_err("tx[%d]: non-finite value", q); return DAS_ERR_INVALID_ARG; }
    if (t.type == DAS_TX_PLANE) {
      const double n2 = (double)t.v[0] * t.v[0] + (double)t.v[1] * t.v[1] + (double)t.v[2] * t.v[2];
      if (std::fabs(std::sqrt(n2) - 1.0) > 1e-4) { set_err("tx[%d]: plane-wave direction is not a unit vector", q); return DAS_ERR_INVALID_ARG; }
    }
  }
  if (d->elem_dir) {
    for (int m = 0; m < d->n_elem; ++m) {
      const float* v = d->elem_dir + 3 * m;
      const double n2 = (double)v[0] * v[0] + (double)v[1] * v[1] + (double)v[2] * v[2];
      if (std::fabs(std::sqrt(n2) - 1.0) > 1e-4) { set_err("elem_dir[%d] is not a unit vector", m); return DAS_ERR_INVALID_ARG; }
    }
  }
  const long long N = (long long)d->nx * d->ny * d->nz;
  const int Kp = padded_samples(d->n_samples);
  const long long rows = (long long)d->n_elem * d->n_tx;
  if (N > (1LL << 40) || rows * Kp > (1LL << 40)) { set_err("problem too large"); return DAS_ERR_SIZE; }

  das_plan* p = new (std::nothrow) das_plan();
  if (!p) { set_err("out of host memory"); return DAS_ERR_ALLOC; }
  p->device = d->device;
  Params& P = p->P;
  P.M = d->n_elem; P.Q = d->n_tx; P.K = d->n_samples; P.Kp = Kp;
  P.nx = d->nx; P.ny = d->ny; P.nz = d->nz;
  P.iq = d->data_kind == DAS_DATA_IQ;
  P.fp16 = d->storage == DAS_STORE_FP16;
  P.fp8 = d->storage == DAS_STORE_FP8;
  P.apod = d->f_number > 0.f;
  P.has_dir = d->elem_dir != nullptr;
  P.c = d->c; P.fc = d->fc; P.fs = d->fs; P.t_start = d->t_start; P.fnum = d->f_number;
  const size_t in_elem = P.iq ? 8 : 4;
  const size_t st_elem = (P.iq ? 2 : 1) * 2 * (P.fp8 ? 1 : (P.fp16 ? 2 : 4));   // (mid, slope) entry
  p->frames = d->n_frames > 1 ? d->n_frames : 1;
  p->raw1 = (size_t)rows * P.K * in_elem;
  p->conv1 = (size_t)rows * Kp * st_elem;
  p->out1 = (size_t)N * in_elem;
  p->raw_bytes = p->raw1 * p->frames;
  p->conv_bytes = p->conv1 * p->frames;
  p->out_bytes = p->out1 * p->frames;

  DeviceGuard g(d->device);
  if (!g.ok) { das_status_t s = cuda_fail(g.err, "selecting the CUDA device"); delete p; return s; }

  std::vector<float> hx, hy, hz;
  std::vector<float4> hv;
  if (d->vox_pos) {
    hx.assign(d->nx, 0.f); hy.assign(1, 0.f); hz.assign(1, 0.f);
    hv.resize(d->nx);
    for (int i = 0; i < d->nx; ++i) hv[i] = make_float4(d->vox_pos[3 * i], d->vox_pos[3 * i + 1], d->vox_pos[3 * i + 2], 0.f);
  } else {
    hx.assign(d->xs, d->xs + d->nx); hy.assign(d->ys, d->ys + d->ny); hz.assign(d->zs, d->zs + d->nz);
  }
  // transmit tables; the observation lists are folded into the weights as exact zeros, which
  // the kernels skip: a voxel then sums over its listed transmits only
  std::vector<float> hw;
  if (d->obs_off) {
    if (d->obs_off[0] != 0) { set_err("obs_off[0] must be 0"); delete p; return DAS_ERR_INVALID_ARG; }
    hw.assign((size_t)N * d->n_tx, 0.f);
    for (long long n = 0; n < N; ++n) {
      if (d->obs_off[n + 1] < d->obs_off[n]) { set_err("obs_off is not non-decreasing"); delete p; return DAS_ERR_INVALID_ARG; }
      for (long long i = d->obs_off[n]; i < d->obs_off[n + 1]; ++i) {
        const int q = d->obs_q[i];
        if (q < 0 || q >= d->n_tx) { set_err("obs_q[%lld] = %d is not a transmit index", i, q); delete p; return DAS_ERR_INVALID_ARG; }
        float& w = hw[(size_t)q * N + n];
        if (w != 0.f) { set_err("voxel %lld lists transmit %d twice", n, q); delete p; return DAS_ERR_INVALID_ARG; }
        w = 1.f;
      }
    }
    if (d->w_tx) for (size_t i = 0; i < hw.size(); ++i) hw[i] = hw[i] != 0.f ? d->w_tx[i] : 0.f;
  } else if (d->w_tx) {
    hw.assign(d->w_tx, d->w_tx + (size_t)N * d->n_tx);
  }
  std::vector<float> htau;
  if (d->tau_tx) htau.assign(d->tau_tx, d->tau_tx + (size_t)N * d->n_tx);
  P.window = d->window; P.interp = d->interp; P.taper = d->window == DAS_WINDOW_TUKEY ? d->window_param : 1.f;
  std::vector<float4> he(d->n_elem), hd;
  for (int m = 0; m < d->n_elem; ++m) he[m] = make_float4(d->elem_pos[3 * m], d->elem_pos[3 * m + 1], d->elem_pos[3 * m + 2], 0.f);
  if (d->elem_dir) {
    hd.resize(d->n_elem);
    for (int m = 0; m < d->n_elem; ++m) hd[m] = make_float4(d->elem_dir[3 * m], d->elem_dir[3 * m + 1], d->elem_dir[3 * m + 2], 0.f);
  }
  std::vector<TxDev> ht(d->n_tx);
  for (int q = 0; q < d->n_tx; ++q) {
    ht[q].type = d->tx[q].type; ht[q].pad = 0;
    ht[q].vx = d->tx[q].v[0]; ht[q].vy = d->tx[q].v[1]; ht[q].vz = d->tx[q].v[2];
    ht[q].t0 = d->tx[q].t0;
  }
  cudaError_t e;
  if ((e = upload(p, hx, &P.xs)) != cudaSuccess || (e = upload(p, hy, &P.ys)) != cudaSuccess ||
      (e = upload(p, hz, &P.zs)) != cudaSuccess || (e = upload(p, he, &P.elem)) != cudaSuccess ||
      (e = upload(p, ht, &P.tx)) != cudaSuccess ||
      (d->elem_dir && (e = upload(p, hd, &P.edir)) != cudaSuccess) ||
      (!hv.empty() && (e = upload(p, hv, &P.vox)) != cudaSuccess) ||
      (!hw.empty() && (e = upload(p, hw, &P.wtx_tab)) != cudaSuccess) ||
      (!htau.empty() && (e = upload(p, htau, &P.tau_tab)) != cudaSuccess)) {
    das_status_t s = (e == cudaErrorMemoryAllocation) ? DAS_ERR_ALLOC : DAS_ERR_CUDA;
    cuda_fail(e, "uploading plan tables");
    free_plan(p);
    return s;
  }

  p->algo = DAS_ALGO_GENERAL;
  if (!general_only && (d->algo == DAS_ALGO_TC || (d->algo == DAS_ALGO_AUTO && p->frames > 1))) {
    char why[256] = "";
    cudaError_t ce = cudaSuccess;
    p->tc = tc_plan_create(P, *d, p->frames, d->device, why, sizeof(why), &ce);
    if (p->tc) {
      p->algo = DAS_ALGO_TC;
      p->conv_bytes = tc_converted_bytes(p->tc, P);
    } else if (ce != cudaSuccess) {
      das_status_t s = cuda_fail(ce, "building the tensor-core plan");
      free_plan(p);
      return s;
    } else if (d->algo == DAS_ALGO_TC) {
      set_err("tensor-core kernel not applicable: %s", why);
      free_plan(p);
      return DAS_ERR_UNSUPPORTED;
    }
  }
  if (p->algo != DAS_ALGO_TC && d->algo != DAS_ALGO_GENERAL && !general_only) {
    char why[256] = "";
    cudaError_t ce = cudaSuccess;
    p->tiled = tiled_plan_create(P, *d, d->device, why, sizeof(why), &ce);
    if (p->tiled) {
      p->algo = DAS_ALGO_TILED;
    } else if (ce != cudaSuccess) {
      das_status_t s = cuda_fail(ce, "building the tiled plan");
      free_plan(p);
      return s;
    } else if (d->algo == DAS_ALGO_TILED) {
      set_err("tiled kernel not applicable: %s", why);
      free_plan(p);
      return DAS_ERR_UNSUPPORTED;
    }
  }
  *out_plan = p;
  return DAS_OK;
}

das_status_t das_plan_destroy(das_plan_t* plan) {
  free_plan(plan);
  return DAS_OK;
}

size_t das_raw_bytes(const das_plan_t* p) { return p ? p->raw_bytes : 0; }
size_t das_converted_bytes(const das_plan_t* p) { return p ? p->conv_bytes : 0; }
size_t das_output_bytes(const das_plan_t* p) { return p ? p->out_bytes : 0; }
int das_plan_algo(const das_plan_t* p) { return p ? p->algo : -1; }
int das_plan_frames(const das_plan_t* p) { return p ? p->frames : 0; }

das_status_t das_convert(const das_plan_t* p, const void* d_raw, void* d_conv, float scale, void* stream) {
  if (!p || !d_raw || !d_conv) { set_err("das_convert: NULL argument"); return DAS_ERR_INVALID_ARG; }
  if (!std::isfinite(scale)) { set_err("das_convert: scale must be finite"); return DAS_ERR_INVALID_ARG; }
  if (reinterpret_cast<uintptr_t>(d_conv) % 16 || reinterpret_cast<uintptr_t>(d_raw) % 8) {
    set_err("das_convert: d_conv must be 16-byte and d_raw 8-byte aligned"); return DAS_ERR_INVALID_ARG;
  }
  DeviceGuard g(p->device);
  if (!g.ok) return cuda_fail(g.err, "selecting the CUDA device");
  cudaError_t e = cudaSuccess;
  if (p->algo == DAS_ALGO_TC) {
    e = launch_convert_batch(p->tc, p->P, d_raw, d_conv, scale, static_cast<cudaStream_t>(stream));
  } else {
    for (int b = 0; b < p->frames && e == cudaSuccess; ++b)
      e = launch_convert(p->P, static_cast<const char*>(d_raw) + b * p->raw1, static_cast<char*>(d_conv) + b * p->conv1,
                         scale, static_cast<cudaStream_t>(stream));
  }
  if (e != cudaSuccess) return cuda_fail(e, "das_convert launch");
  return DAS_OK;
}

das_status_t das_execute(const das_plan_t* p, const void* d_conv, void* d_out, void* stream) {
  if (!p || !d_conv || !d_out) { set_err("das_execute: NULL argument"); return DAS_ERR_INVALID_ARG; }
  if (reinterpret_cast<uintptr_t>(d_conv) % 16 || reinterpret_cast<uintptr_t>(d_out) % 8) {
    set_err("das_execute: d_conv must be 16-byte and d_out 8-byte aligned"); return DAS_ERR_INVALID_ARG;
  }
  DeviceGuard g(p->device);
  if (!g.ok) return cuda_fail(g.err, "selecting the CUDA device");
  cudaError_t e = cudaSuccess;
  if (p->algo == DAS_ALGO_TC) {
    e = launch_tc(p->tc, p->P, d_conv, d_out, static_cast<cudaStream_t>(stream));
  } else {
    for (int b = 0; b < p->frames && e == cudaSuccess; ++b) {
      const char* cv = static_cast<const char*>(d_conv) + b * p->conv1;
      char* o = static_cast<char*>(d_out) + b * p->out1;
      if (p->algo == DAS_ALGO_TILED) {
        int nl = 0;
        e = launch_tiled(p->tiled, p->P, cv, o, static_cast<cudaStream_t>(stream), &nl);
      } else {
        e = launch_general(p->P, cv, o, static_cast<cudaStream_t>(stream));
      }
    }
  }
  if (e != cudaSuccess) return cuda_fail(e, "das_execute launch");
  return DAS_OK;
}

static das_status_t host_staging(das_plan* p) {
  if (p->st_conv) return DAS_OK;
  cudaError_t e = cudaSuccess;
  auto fail = [&](const char* what) {
    cuda_fail(e, what);
    for (auto& sl : p->slot) {
      if (sl.d_raw) { cudaFree(sl.d_raw); sl.d_raw = nullptr; }
      if (sl.d_out) { cudaFree(sl.d_out); sl.d_out = nullptr; }
    }
    if (p->st_conv) { cudaFree(p->st_conv); p->st_conv = nullptr; }
    return e == cudaErrorMemoryAllocation ? DAS_ERR_ALLOC : DAS_ERR_CUDA;
  };
  for (auto& sl : p->slot) {
    if ((e = cudaMalloc(&sl.d_raw, p->raw_bytes)) != cudaSuccess || (e = cudaMalloc(&sl.d_out, p->out_bytes)) != cudaSuccess)
      return fail("allocating staging buffers");
    for (cudaEvent_t* ev : {&sl.ev_h2d, &sl.ev_exec, &sl.ev_d2h})
      if (!*ev && (e = cudaEventCreateWithFlags(ev, cudaEventDisableTiming)) != cudaSuccess) { *ev = nullptr; return fail("creating events"); }
  }
  // each stream under its own check: after a partial failure the next call must not take a missing s_out for
  // "both exist" and copy out on the legacy default stream
  if (!p->s_in && (e = cudaStreamCreateWithFlags(&p->s_in, cudaStreamNonBlocking)) != cudaSuccess) { p->s_in = nullptr; return fail("creating copy streams"); }
  if (!p->s_out && (e = cudaStreamCreateWithFlags(&p->s_out, cudaStreamNonBlocking)) != cudaSuccess) { p->s_out = nullptr; return fail("creating copy streams"); }
  if ((e = cudaMalloc(&p->st_conv, p->conv_bytes)) != cudaSuccess) return fail("allocating staging buffers");
  return DAS_OK;
}

das_status_t das_beamform_host_begin(das_plan_t* p, const void* h_raw, void* h_out, void* stream) {
  if (!p || !h_raw || !h_out) { set_err("das_beamform_host: NULL argument"); return DAS_ERR_INVALID_ARG; }
  if (p->begun - p->waited >= 2) { set_err("das_beamform_host_begin: two calls are outstanding already"); return DAS_ERR_INVALID_ARG; }
  DeviceGuard g(p->device);
  if (!g.ok) return cuda_fail(g.err, "selecting the CUDA device");
  das_status_t st = host_staging(p);
  if (st != DAS_OK) return st;
  das_plan::HostSlot& sl = p->slot[p->begun & 1];
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  cudaError_t e;
  // A failure after the first enqueue leaves copies / kernels of this call in flight on a slot that is not
  // recorded as begun: drain the three streams before reporting it, so that the next begin finds the slot idle.
  struct Drain {
    das_plan* p; cudaStream_t s; bool armed = true;
    ~Drain() { if (armed) { cudaStreamSynchronize(p->s_in); cudaStreamSynchronize(s); cudaStreamSynchronize(p->s_out); } }
  } drain{p, s};
  // slot reuse: the previous user's kernels have read d_raw (ev_exec), its copy-out has read d_out (ev_d2h)
  if (sl.used && (e = cudaStreamWaitEvent(p->s_in, sl.ev_exec, 0)) != cudaSuccess) return cuda_fail(e, "stream wait");
  if ((e = cudaMemcpyAsync(sl.d_raw, h_raw, p->raw_bytes, cudaMemcpyHostToDevice, p->s_in)) != cudaSuccess)
    return cuda_fail(e, "host-to-device copy");
  if ((e = cudaEventRecord(sl.ev_h2d, p->s_in)) != cudaSuccess || (e = cudaStreamWaitEvent(s, sl.ev_h2d, 0)) != cudaSuccess ||
      (sl.used && (e = cudaStreamWaitEvent(s, sl.ev_d2h, 0)) != cudaSuccess))
    return cuda_fail(e, "event chain");
  if ((st = das_convert(p, sl.d_raw, p->st_conv, 1.0f, stream)) != DAS_OK) return st;
  if ((st = das_execute(p, p->st_conv, sl.d_out, stream)) != DAS_OK) return st;
  if ((e = cudaEventRecord(sl.ev_exec, s)) != cudaSuccess || (e = cudaStreamWaitEvent(p->s_out, sl.ev_exec, 0)) != cudaSuccess)
    return cuda_fail(e, "event chain");
  if ((e = cudaMemcpyAsync(h_out, sl.d_out, p->out_bytes, cudaMemcpyDeviceToHost, p->s_out)) != cudaSuccess)
    return cuda_fail(e, "device-to-host copy");
  if ((e = cudaEventRecord(sl.ev_d2h, p->s_out)) != cudaSuccess) return cuda_fail(e, "event record");
  sl.used = true;
  ++p->begun;
  drain.armed = false;
  return DAS_OK;
}

das_status_t das_beamform_host_wait(das_plan_t* p) {
  if (!p) { set_err("das_beamform_host_wait: NULL plan"); return DAS_ERR_INVALID_ARG; }
  if (p->begun == p->waited) { set_err("das_beamform_host_wait: nothing outstanding"); return DAS_ERR_INVALID_ARG; }
  DeviceGuard g(p->device);
  if (!g.ok) return cuda_fail(g.err, "selecting the CUDA device");
  cudaError_t e = cudaEventSynchronize(p->slot[p->waited & 1].ev_d2h);
  ++p->waited;
  if (e != cudaSuccess) return cuda_fail(e, "waiting for the device-to-host copy");
  return DAS_OK;
}

das_status_t das_beamform_host(das_plan_t* p, const void* h_raw, void* h_out, void* stream) {
  if (p && p->begun != p->waited) { set_err("das_beamform_host: pipelined calls are outstanding; wait for them first"); return DAS_ERR_INVALID_ARG; }
  das_status_t st = das_beamform_host_begin(p, h_raw, h_out, stream);
  if (st != DAS_OK) return st;
  return das_beamform_host_wait(p);
}

das_status_t das_plan_count_work(const das_plan_t* p, unsigned long long* n_pairs, unsigned long long* n_terms) {
  if (!p || !n_pairs || !n_terms) { set_err("das_plan_count_work: NULL argument"); return DAS_ERR_INVALID_ARG; }
  DeviceGuard g(p->device);
  if (!g.ok) return cuda_fail(g.err, "selecting the CUDA device");
  unsigned long long* d = nullptr;
  cudaError_t e = cudaMalloc(&d, 2 * sizeof(unsigned long long));
  if (e != cudaSuccess) { cuda_fail(e, "allocating counters"); return DAS_ERR_ALLOC; }
  unsigned long long h[2] = {0, 0};
  if ((e = cudaMemset(d, 0, sizeof(h))) == cudaSuccess && (e = launch_count(p->P, d, nullptr)) == cudaSuccess)
    e = cudaMemcpy(h, d, sizeof(h), cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return cuda_fail(e, "das_plan_count_work");
  *n_pairs = h[0];
  *n_terms = h[1];
  return DAS_OK;
}

#pragma GCC visibility pop
}  // extern "C"

// What das_static.cu (das_beamform_static) needs from the opaque plan and the error channel.
namespace das {
int plan_device(const das_plan* p) { return p->device; }
void set_error_text(const char* msg) { set_err("%s", msg); }
}  // namespace das
