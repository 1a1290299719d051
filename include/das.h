/*
 * das.h -- C ABI of the B200-native volumetric delay-and-sum (DAS) beamformer.
 *
 * The library computes, for every voxel p_n of a rectilinear grid,
 *
 *     x_n = sum_q sum_m  w_rx(m,n) * y_qm[ t_qmn ] * R(tau_qmn)                       (Eq. 2)
 *
 *     tau_qmn = tau_tx(q,n) + |p_n - r_m| / c                    (Eq. 1)
 *     tau_tx  = (p_n . u_q)/c + t0_q          plane wave          (fn. 2; sign
 *             = |p_n - v_q|/c + t0_q          diverging wave       and t0 per DESIGN.md A1/A2)
 *     t_qmn   = (tau_qmn - t_start) * fs,  y[t] = (1-a) y[k] + a y[k+1], k = floor(t), a = t-k
 *               (linear interpolation); the term is dropped unless 0 <= k <= K-2
 *     w_rx    = 1 if f_number <= 0, else 1 iff a > 0 and 4 f#^2 rho^2 <= a^2 with
 *               a = (p_n - r_m).n_m, rho^2 = |p_n - r_m|^2 - a^2   (f-number boxcar on a cone
 *               about the element normal; "origin and a direction")
 *     R(tau)  = exp(+j 2 pi fc tau) for IQ data (BASELINE.json north_star), 1 for RF data
 *
 * All delays are computed in-kernel; nothing of size N*M*Q is ever stored.
 * Accumulation is FP32 whatever the storage precision.
 *
 * Conventions
 *   - Plain C, no exceptions cross this boundary; every call returns a das_status_t
 *     (or a size / string).  das_last_error() gives a thread-local detail string.
 *   - "host" / "device" on a pointer says where the memory lives.  Device pointers must
 *     belong to the plan's CUDA device.  The library never takes ownership of caller memory.
 *   - das_convert / das_execute only enqueue work on the given CUDA stream (a cudaStream_t
 *     passed as void*; NULL = the legacy default stream).  They never synchronise and never
 *     allocate.  A plan's geometry and launch shapes never change after creation: concurrent das_execute
 *     calls on different streams with different buffers are allowed (a DAS_ALGO_TC plan also owns pacing words
 *     that its launches write; see das_execute).
 */
#ifndef DAS_B200_H_
#define DAS_B200_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct das_plan das_plan_t;      /* opaque, owned by the library */

typedef enum {
  DAS_OK = 0,
  DAS_ERR_INVALID_ARG = 1,   /* null pointer, size < 1, non-finite or non-positive c / fs, ... */
  DAS_ERR_UNSUPPORTED = 2,   /* unknown enum value or a combination this build does not implement */
  DAS_ERR_ALLOC = 3,         /* host or device allocation failed */
  DAS_ERR_CUDA = 4,          /* a CUDA runtime call or kernel launch failed (see das_last_error) */
  DAS_ERR_SIZE = 5           /* problem exceeds an internal limit (index overflow) */
} das_status_t;

typedef enum { DAS_TX_PLANE = 0, DAS_TX_DIVERGING = 1 } das_tx_type_t;
typedef enum { DAS_DATA_IQ = 0, DAS_DATA_RF = 1 } das_data_kind_t;
typedef enum {
  DAS_STORE_FP32 = 0,
  DAS_STORE_FP16 = 1,    /* the paper's mixed-precision storage */
  DAS_STORE_FP8 = 2      /* e4m3, round to nearest even, saturating ("FP8 storage"): general and tiled
                            kernels (n_frames > 1 runs frame by frame; DAS_ALGO_TC refuses it).  What is stored is
                            the interval table (mid, slope) = ((y_k + y_k+1)/2, y_k+1 - y_k) of the scaled data, so
                            the caller's `scale` must bring BOTH into the e4m3 range: |y_k| <= 448 and
                            |y_k+1 - y_k| <= 448 (two neighbours of opposite sign near full scale break the
                            second); a larger slope is clipped to +-448 without an error and that interval is then
                            interpolated wrongly.  Resolution 2^-9 near zero; DESIGN.md gives the image quality */
} das_storage_t;
/* Receive window on the f-number cone ("receive weight ... origin and a direction"; DESIGN.md
 * reading W1).  With u = 2 f# rho / a in [0, 1] the normalised radius inside the cone:
 *   BOXCAR w_rx = 1 | HANN w_rx = (1 + cos(pi u)) / 2 | TUKEY(b) w_rx = 1 for u <= 1 - b,
 *   (1 + cos(pi (u - 1 + b) / b)) / 2 beyond; 0 outside the cone; every window is 1 when f_number <= 0. */
typedef enum { DAS_WINDOW_BOXCAR = 0, DAS_WINDOW_HANN = 1, DAS_WINDOW_TUKEY = 2 } das_window_t;
/* Temporal interpolation: LINEAR is the paper's; CUBIC is the 4-tap cubic convolution
 * (Keys, a = -1/2) on y[k-1..k+2], the term dropped unless 1 <= k <= K-3 (reading W2). */
typedef enum { DAS_INTERP_LINEAR = 0, DAS_INTERP_CUBIC = 1 } das_interp_t;
typedef enum {
  DAS_ALGO_AUTO = 0,     /* tiled kernel when the geometry allows it, else the general kernel */
  DAS_ALGO_GENERAL = 1,  /* one thread per voxel, any element positions / normals (Alg. 1 shape) */
  DAS_ALGO_TILED = 2,    /* voxel-tiled, shared-memory staged kernel; needs a planar array with
                            all normals (0,0,1); DAS_ERR_UNSUPPORTED otherwise */
  DAS_ALGO_TC = 3        /* frame batch on the tensor cores (tcgen05, section 3.4 on
                            the batch-inner layout of section 3.2): n_frames a multiple of 8 (of 64 above
                            64), IQ data, fp16 storage, <= 16 transmits, planar array with normals
                            (0,0,1); DAS_ERR_UNSUPPORTED otherwise.  AUTO picks it when it applies. */
} das_algo_t;

/* One transmit event (one "observation" q of the paper). */
typedef struct {
  int   type;      /* das_tx_type_t */
  float v[3];      /* PLANE: unit propagation direction u_q.  DIVERGING: virtual source v_q [m] */
  float t0;        /* seconds added to tau_tx (time-zero convention, reading A2) */
} das_transmit_t;

/* Everything that defines a reconstruction except the channel data.  All pointers are HOST
 * pointers; the plan copies what it needs, the caller may free them after das_plan_create. */
typedef struct {
  const float* elem_pos;  int n_elem;   /* [M][3] receiver positions r_m, metres */
  const float* elem_dir;                /* [M][3] unit normals n_m, or NULL = (0,0,1) for all */
  const das_transmit_t* tx; int n_tx;   /* [Q] */
  const float* xs; int nx;              /* axis vectors of the rectilinear voxel grid, metres; */
  const float* ys; int ny;              /*   voxel (ix,iy,iz) sits at (xs[ix], ys[iy], zs[iz])  */
  const float* zs; int nz;
  float c;            /* speed of sound c0 [m/s], > 0 */
  float fc;           /* demodulation frequency [Hz] for the IQ phase rotation, >= 0; must be 0 for RF */
  float fs;           /* sampling rate of the channel data [Hz], > 0 */
  float t_start;      /* time of sample k = 0 [s] */
  float f_number;     /* receive f-number of the boxcar apodization; <= 0 disables apodization */
  int   n_samples;    /* K >= 2, samples per (transmit, element) */
  int   data_kind;    /* das_data_kind_t: IQ = complex64 in, complex64 out; RF = float32 in/out */
  int   storage;      /* das_storage_t: precision of the converted (device-layout) channel data */
  int   algo;         /* das_algo_t */
  int   device;       /* CUDA device ordinal */
  int   n_frames;     /* B, frames per call that share this geometry; 0 or 1 = one frame.
                         With B > 1 das_convert / das_execute / das_beamform_host take B frames:
                         raw [B][Q][M][K], output [B][nx][ny][nz]; every frame is the sum Eq. 2 defines
                         for it (DAS_ALGO_TC: weights rounded to FP16, else frame by frame). */
  /* ---- the paper's general interface (Alg. 1 "Require"); zero / NULL = off.  All HOST
   *      pointers, copied at plan creation.  N = nx*ny*nz, voxel order = output order. ---- */
  const float* tau_tx;      /* [Q][N] transmit delays tau_tx_qn in seconds; when given they
                               replace the delay models of tx[] (type / v / t0 are then ignored) */
  const float* w_tx;        /* [Q][N] transmit weights w_tx_qn (magnitude of the transmit field).  A weight of
                               exactly 0 means the same as voxel n not listing transmit q (below): the samples of that
                               (q, n) are not summed, whatever they hold, and das_plan_count_work does not count them */
  const long long* obs_off; /* [N+1] CSR offsets of the per-voxel observation lists: voxel n sums */
  const int* obs_q;         /* [obs_off[N]] only over the transmits listed for it, each at most once */
  const float* vox_pos;     /* [N][3] an arbitrary voxel list ("{p_n}") instead of the grid axes:
                               set nx = N, ny = nz = 1; xs / ys / zs are ignored.  General kernel only. */
  int   window;             /* das_window_t */
  float window_param;       /* TUKEY: taper fraction b in (0, 1] */
  int   interp;             /* das_interp_t; CUBIC: general kernel only, one frame per call */
  /* ---- debugging aids; 0 = the library's choice.  They change launch shapes, never results (tests use them to
   *      force a ragged grid of CTAs and to compare paced with unpaced launches).  The library reads no
   *      environment variable unless it is built with -DDAS_TUNING (kernel-tuning sweeps). ---- */
  int   debug_tiled_grid;   /* CTAs of the one-frame tiled kernel (default: one or two per SM, at most one per tile) */
  int   debug_tc_pace;      /* DAS_ALGO_TC quad pacing (das_execute): lead in receivers, default 16; -1 = no pacing */
} das_plan_desc_t;

/* The problem statement of PAPER.md:29-50 (Eq. 1: delays; Eq. 2: the weighted sum; linear interpolation) and
 * PAPER.md:99-133 (Alg. 1 "Require": geometry, transmit set, voxel positions) as a plan.  Validates *desc,
 * uploads geometry and small derived tables to desc->device, chooses kernel and launch shapes (with
 * n_frames = B >= 8 and IQ data in fp16 storage: per-tile sample windows from a plan-time kernel, about
 * 1.5 s at the headline size).  On success *out_plan is a new plan (free with das_plan_destroy). */
das_status_t das_plan_create(const das_plan_desc_t* desc, das_plan_t** out_plan);
das_status_t das_plan_destroy(das_plan_t* plan);            /* NULL is allowed */

size_t das_raw_bytes(const das_plan_t* plan);        /* B*Q*M*K * (8 for IQ, 4 for RF)            */
size_t das_converted_bytes(const das_plan_t* plan);  /* size of the buffer das_convert writes      */
size_t das_output_bytes(const das_plan_t* plan);     /* B*nx*ny*nz * (8 for IQ, 4 for RF)          */
int    das_plan_algo(const das_plan_t* plan);        /* the das_algo_t actually selected           */
int    das_plan_frames(const das_plan_t* plan);      /* B (>= 1)                                   */

/* Layout transform + cast (the paper's permute-and-convert pre-pass).
 *   d_raw   device, [B][Q][M][K] complex64 (re,im interleaved) for IQ or float32 for RF,
 *           samples contiguous in k (the paper's input layout)
 *   d_conv  device, das_converted_bytes() bytes, 16-byte aligned; written entirely
 *   scale   every sample is multiplied by it before the cast (1.0f = none); lets the caller
 *           keep fp16 storage inside its normal range
 * fp16 storage rounds to nearest even; overflow gives +-inf (reading A11).  The one-frame kernels read a
 * sample only for the terms that use it, so an infinite sample spoils only the voxels whose sum contains it (as
 * in the definition).  DAS_ALGO_TC multiplies whole sample windows by weight rows that are zero where a voxel does
 * not use a sample, and 0 * inf = NaN: there the scaled data must stay finite in FP16 (|scale * y| < 65504). */
das_status_t das_convert(const das_plan_t* plan, const void* d_raw, void* d_conv, float scale,
                         void* stream);

/* Beamform one volume per frame (B volumes): Eq. 2 with the delays of Eq. 1
 * and linear interpolation evaluated in-kernel for every voxel, rows a2-a6 of SURVEY.md section 8.
 *   d_conv  device, produced by das_convert with this plan, or with a plan of the same algo (das_plan_algo),
 *           n_frames, n_tx, n_elem, n_samples, data_kind and storage: the converted layout depends on all of
 *           them (DAS_ALGO_TC: batch-inner [chunk][M][Q][column group][2K][8] FP16; else [M][Q][Kp] intervals);
 *           a buffer converted for another layout is not detected
 *   d_out   device, das_output_bytes() bytes, [B][nx][ny][nz] with z fastest (C order), complex64
 *           (IQ) or float32 (RF); overwritten, not accumulated into; 8-byte aligned
 * Calls on one plan may overlap (different streams, different buffers).  For DAS_ALGO_TC the CTAs of a launch pace
 * each other through progress words owned by the plan (L2 reuse between neighbouring tiles): overlapping launches
 * of ONE such plan stay correct (the pacing is advisory and its waits are bounded) but lose the pacing's benefit;
 * use one plan per stream.  A launch whose CTAs are not all resident at once (an SM limit, MIG, a kernel of another
 * stream holding SMs) also stays correct: a CTA waits for an absent partner for a few ms per launch at most (the
 * wait budget shrinks each time it runs out), on top of the serialisation the missing SMs cause anyway. */
das_status_t das_execute(const das_plan_t* plan, const void* d_conv, void* d_out, void* stream);

/* End-to-end convenience for HOST buffers: copies h_raw to the device, runs das_convert
 * (scale 1) and das_execute, copies the volume back to h_out and synchronises the stream
 * before returning.  Uses device staging buffers owned by the plan (allocated on first use and
 * freed by das_plan_destroy), therefore NOT safe to call concurrently on one plan.  For full
 * copy bandwidth h_raw / h_out should be page-locked. */
das_status_t das_beamform_host(das_plan_t* plan, const void* h_raw, void* h_out, void* stream);

/* The same as a two-deep pipeline for streaming callers (BASELINE.json configs[4]: frames arrive from the
 * host one batch after another).  das_beamform_host_begin enqueues the host-to-device copy of h_raw on a
 * copy stream of the plan, das_convert + das_execute on `stream`, and the device-to-host copy into h_out on
 * a second copy stream, chained by events, and returns without waiting; das_beamform_host_wait blocks until
 * the OLDEST outstanding call has delivered its h_out.  At most two calls may be outstanding (the plan owns
 * two raw / output staging buffers and one converted buffer); a third begin returns DAS_ERR_INVALID_ARG.
 * With two calls in flight the copies of one batch run under the kernels of the other, so the sustained rate
 * is that of the slower of the two (PCIe for the headline batch: 8.6 GB in, 1.1 GB out per 64 frames).
 * h_raw must stay valid until the matching wait returns; both buffers should be page-locked.  Always pass the
 * same `stream` for one plan.  das_beamform_host == begin + wait. */
das_status_t das_beamform_host_begin(das_plan_t* plan, const void* h_raw, void* h_out, void* stream);
das_status_t das_beamform_host_wait(das_plan_t* plan);

/* The same raw -> volume path for callers that cannot allocate device memory, and for which the library must
 * not allocate either: a real-time acquisition / display loop (cudaMalloc and cudaFree take a driver lock and may
 * synchronise the device: a dropped frame), a plug-in inside an application whose own memory pool already owns
 * the whole GPU (cudaMalloc just fails there), software under a "no allocation after set-up" rule.
 * das_convert + das_execute need a converted buffer from the caller; das_beamform_host allocates staging buffers
 * on first use.  This call needs neither: the converted data goes through a scratch array that is part of the
 * library image (a file-scope __device__ array of DAS_STATIC_SCRATCH_BYTES, resident on every GPU that loads the
 * library, from module load until the process exits).  It calls no cudaMalloc / cudaFree and no allocating
 * library routine, synchronises nothing, and enqueues exactly the kernels of das_convert(scale) + das_execute on
 * `stream`, so the result is bit-identical to theirs.
 *   d_raw, d_out   device, as for das_convert / das_execute (inputs and outputs stay the caller's)
 *   limit          das_converted_bytes(plan) <= DAS_STATIC_SCRATCH_BYTES, else DAS_ERR_SIZE and nothing is
 *                  enqueued (16 MiB takes BASELINE.json configs 1 and 2; the headline needs 151 MB: use
 *                  das_convert + das_execute with your own buffer there)
 *   first call     the first call on each device looks the array's device address up (cudaGetSymbolAddress,
 *                  which loads the CUDA module on that device if it is not loaded yet).  Make that call during
 *                  set-up, before any stream capture and before the no-allocation phase begins.
 *   sharing        there is ONE array per GPU for the whole process: two das_beamform_static calls that can
 *                  overlap on the GPU (different streams, or different plans on different streams) race on it
 *                  and give garbage.  Keep all calls of one GPU on one stream, or order them with events.  The
 *                  array keeps the last call's bytes between calls; nothing in it has to be cleared, because
 *                  das_convert rewrites every byte das_execute reads. */
#define DAS_STATIC_SCRATCH_BYTES (16u << 20)
das_status_t das_beamform_static(const das_plan_t* plan, const void* d_raw, void* d_out, float scale,
                                 void* stream);

/* Work accounting (used by the bench's roofline; not part of the hot path).  Runs a counting
 * kernel on the plan's device and SYNCHRONISES.  On success
 *   *n_pairs = number of (m, n) receiver/voxel pairs with non-zero receive weight w_rx
 *   *n_terms = number of (q, m, n) terms that enter Eq. 2: non-zero weight and 0 <= k <= K-2
 * both classified exactly as das_execute classifies them.  Host pointers. */
das_status_t das_plan_count_work(const das_plan_t* plan, unsigned long long* n_pairs,
                                 unsigned long long* n_terms);

const char* das_status_string(das_status_t s);
const char* das_last_error(void);        /* thread-local, never NULL */

/* Number of kernels the library has launched in this process (all plans, all threads).
 * The bench reports it as gpu_launches. */
unsigned long long das_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* DAS_B200_H_ */
