// das_beamform_static (include/das.h): raw channel data in, volume out, and no device allocation anywhere on
// the way -- neither by the caller nor by the library.
//
// Who this is for.  das_convert + das_execute already allocate nothing, but they make the CALLER bring the
// converted buffer (das_converted_bytes()), i.e. the caller has to be able to allocate device memory.  Some
// callers cannot:
//   - an acquisition / display loop with a latency budget: cudaMalloc and cudaFree take a driver lock and may
//     synchronise the whole device, so one allocation in the loop is a dropped frame;
//   - a plug-in inside a host application whose own pool already owns all of the device memory (a deep-learning
//     framework's caching allocator, a scanner vendor's runtime): cudaMalloc from the plug-in simply fails;
//   - code that runs after set-up under a "no allocation from here on" rule (safety-reviewed real-time software).
// For them the intermediate buffer between the two kernels lives in the file-scope array below, which is part of
// the library image: it is placed in device memory when the CUDA module is loaded on a GPU and stays there until
// the process exits.  That costs DAS_STATIC_SCRATCH_BYTES (16 MiB) on every GPU that loads libdas_b200.so, used
// or not, which is why the limit is modest: it takes the converted data of BASELINE.json configs 1 and 2
// (0.4 MB and 13 MB at fp32 storage), not the 151 MB of the headline configuration.
//
// The kernels are the ones das_convert and das_execute launch, unchanged: they get the array's address where
// they would get the caller's d_conv.
#include <cstdio>
#include <mutex>

#include "das_internal.cuh"

namespace {

// The scratch: the converted (device-layout) channel data of the call in flight.  256-byte aligned (the TMA
// bulk copies of tiled_kernel and the tensor map of tc_kernel need 16).  Shared by every call in the process
// that runs on this GPU; it keeps the previous call's bytes, which is harmless because das_convert overwrites
// all das_converted_bytes() bytes before das_execute reads any of them -- nothing has to start at zero.
static __device__ __align__(256) unsigned char g_static_conv[DAS_STATIC_SCRATCH_BYTES];

// In host code `g_static_conv` is only a handle for the runtime's symbol table, NOT a device address: a kernel
// handed &g_static_conv[0] from the host would fault (or scribble over host memory on a system where the GPU
// can reach it).  The device address is asked for once per device, with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_dev_addr[kMaxDevices] = {};

cudaError_t static_conv_address(int device, void** out) {
  if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_dev_addr[device]) {
    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e != cudaSuccess) return e;
    if (prev != device && (e = cudaSetDevice(device)) != cudaSuccess) return e;
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_conv);      // loads this module on the device if it is not yet
    if (prev != device) cudaSetDevice(prev);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_dev_addr[device] = p;
  }
  *out = g_dev_addr[device];
  return cudaSuccess;
}

}  // namespace

extern "C" {
#pragma GCC visibility push(default)

das_status_t das_beamform_static(const das_plan_t* plan, const void* d_raw, void* d_out, float scale, void* stream) {
  if (!plan || !d_raw || !d_out) {
    das::set_error_text("das_beamform_static: NULL argument");
    return DAS_ERR_INVALID_ARG;
  }
  const size_t need = das_converted_bytes(plan);
  if (need > (size_t)DAS_STATIC_SCRATCH_BYTES) {
    char msg[256];
    snprintf(msg, sizeof(msg),
             "das_beamform_static: this plan's converted data takes %zu bytes, the built-in scratch holds %zu "
             "(DAS_STATIC_SCRATCH_BYTES); use das_convert + das_execute with a buffer of your own",
             need, (size_t)DAS_STATIC_SCRATCH_BYTES);
    das::set_error_text(msg);
    return DAS_ERR_SIZE;
  }
  void* conv = nullptr;
  const cudaError_t e = static_conv_address(das::plan_device(plan), &conv);
  if (e != cudaSuccess) {
    char msg[256];
    snprintf(msg, sizeof(msg), "das_beamform_static: looking up the built-in scratch on device %d: %s (%s)",
             das::plan_device(plan), cudaGetErrorString(e), cudaGetErrorName(e));
    das::set_error_text(msg);
    return DAS_ERR_CUDA;
  }
  const das_status_t st = das_convert(plan, d_raw, conv, scale, stream);
  if (st != DAS_OK) return st;
  return das_execute(plan, conv, d_out, stream);
}

#pragma GCC visibility pop
}  // extern "C"
