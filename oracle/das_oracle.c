/*
 * das_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU delay-and-sum.  It is the oracle the CUDA
 * path is checked against.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant with paper_2606_13259_b200/.
 *
 * DAS is an exact finite sum, so this file is the *definition* written out
 * (SURVEY.md 8(c.1)), in the loop order of the paper's Algorithm 1:
 *
 *   Eq. 1   tau_qmn = tau_tx_qn + tau_rx_mn,  tau_rx_mn = |p_n - r_m| / c0
 *   fn. 2      plane wave / diverging wave transmit delay, with the sign and the
 *                            per-transmit time-zero offset t0 of DESIGN.md readings A1, A2:
 *                              PLANE      tau_tx = (p . u)/c + t0
 *                              DIVERGING  tau_tx = |p - v|/c + t0
 *   weights    w = w_tx * w_rx with w_tx == 1 (reading: north_star has none) and
 *                            w_rx the f-number boxcar on a cone about the element normal
 *                            (reading A3): active iff a > 0 and 4 f#^2 rho^2 <= a^2,
 *                            a = d . n_m, rho^2 = d.d - a^2, d = p - e_m;  f# <= 0: w_rx = 1
 *   Eq. 2   x_n = sum_q sum_m w_qmn * y_qm[tau_qmn]
 *   interpolation  linear between y[k], y[k+1], k = floor(t),
 *                            t = (tau - t_start) * fs, 0-based (reading A5); the term is
 *                            dropped unless 0 <= k <= K-2 (reading A6)
 *   phase rotation           IQ data: each term is multiplied by exp(+j 2 pi fc tau), tau the
 *                            absolute time of flight (BASELINE.json north_star; readings A7, A8)
 *   no normalisation (A9).
 *
 * Extensions of the paper's general interface (das_oracle_ex), each OFF
 * unless its option is set, in which case the lines above change as stated:
 *   tau_tx table (Alg. 1 "Require")   tau_tx_qn read from a table [Q][N] (seconds) instead of fn. 2
 *   w_tx table   (PAPER.md:43 "transmit weight ... magnitude of the transmit wavefield", :101)
 *                            w = w_tx_qn * w_rx_mn with w_tx_qn from a table [Q][N]
 *   observation lists ("sparse per-voxel lists of observations")   voxel n sums only over the
 *                            transmits q listed for it (CSR: obs_off[N+1], obs_q[])
 *   voxel list   (Alg. 1 "voxel positions {p_n}")   p_n read from a list [N][3] instead of a grid
 *   receive window (PAPER.md:43 receive weight from origin and direction; reading W1)   with
 *                            u = 2 f# rho / a in [0, 1] the normalised radius inside the f-number cone:
 *                              BOXCAR  w_rx = 1                                  (the default above)
 *                              HANN    w_rx = (1 + cos(pi u)) / 2
 *                              TUKEY   w_rx = 1 for u <= 1 - b, (1 + cos(pi (u - 1 + b) / b)) / 2 beyond (taper b)
 *                            all 0 outside the cone (u > 1 or a <= 0); with f# <= 0 every window is 1
 *   interpolation ("Alternative interpolation schemes follow the same principles"; reading W2)
 *                            CUBIC: 4-tap cubic convolution (Keys, a = -1/2) on y[k-1..k+2], exact for
 *                            quadratics; the term is dropped unless 1 <= k <= K-3
 *
 * Every float input is promoted to double as is; nothing is re-derived.
 * Compile WITHOUT -ffast-math and with -ffp-contract=off (oracle/build.py does).
 *
 * Pins: tests/test_oracle_pins.py (closed forms from Pythagorean-triple geometries stored in
 * tests/golden/, impulse response, dense-matrix brute force, linearity, time-shift invariance,
 * transmit additivity, mirror symmetry, RF = Re(IQ at fc = 0), aperture count in exact rational
 * arithmetic, point-scatterer peak and peak value bound); tests/test_oracle_ext_pins.py for the
 * extensions (tables that restate fn. 2 reproduce the formula path bit for bit, unit weights and full
 * lists reproduce the plain result bit for bit, hand-derived weighted / windowed / cubic golden
 * cases in tests/golden/ext_cases.json, window closed forms, quadratic reproduction of the cubic
 * kernel, dense-matrix brute force with every option on).  Parity unpinned: none of the sum
 * itself; the out-of-range rule (A6) and the a <= 0 rule (A10) are this build's own readings,
 * pinned only against their statement in DESIGN.md.
 */
#include <math.h>
#include <stddef.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_TX_PLANE 0
#define ORACLE_TX_DIVERGING 1
#define ORACLE_DATA_IQ 0
#define ORACLE_DATA_RF 1

static const double ORACLE_TWO_PI = 6.283185307179586476925286766559;

int das_oracle_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/*
 * Arguments (all host pointers, caller-owned):
 *   elem_pos [M][3], elem_dir [M][3] or NULL (= (0,0,1), reading A4)
 *   tx_type [Q], tx_v [Q][3] (unit direction or virtual source), tx_t0 [Q]
 *   xs[nx], ys[ny], zs[nz]: axes of the rectilinear grid; voxel (ix,iy,iz) = (xs[ix],ys[iy],zs[iz])
 *   y: [Q][M][K] interleaved (re,im) float pairs for IQ, plain floats for RF
 *   vox_idx/n_vox: flat indices (ix*ny + iy)*nz + iz to evaluate, or NULL/0 for the full grid
 *   out: per evaluated voxel 2 doubles (re,im) for IQ, 1 double for RF
 *   out_count   (optional) number of (q,m) terms that entered the sum
 *   out_l1      (optional) sum over entered terms of (1-a)|y_k|_1 + a|y_k+1|_1
 *               (|.|_1 = |re|+|im|); times 2^-11 this bounds the effect of fp16 storage rounding
 *   out_slack   (optional) sum of |term| over (q,m) whose aperture margin
 *               |4 f#^2 rho^2 - a^2| <= slack_rel * a^2 (near-ties of the boxcar edge)
 * Returns 0, or -1 on a bad argument.
 */
#define ORACLE_WIN_BOXCAR 0
#define ORACLE_WIN_HANN 1
#define ORACLE_WIN_TUKEY 2
#define ORACLE_INTERP_LINEAR 0
#define ORACLE_INTERP_CUBIC 1

/* Options of das_oracle_ex; a zeroed struct (or NULL) is the plain definition above. */
typedef struct {
  const float* tau_tx_tab;   /* [Q][N] transmit delays in seconds, N = nx*ny*nz, or NULL (fn. 2 formulas) */
  const float* w_tx_tab;     /* [Q][N] transmit weights, or NULL (== 1) */
  const long long* obs_off;  /* [N+1] CSR offsets of the per-voxel observation lists, or NULL (all q) */
  const int* obs_q;          /* [obs_off[N]] transmit indices */
  const float* vox_pos;      /* [N][3] voxel positions, or NULL (grid axes); with it nx = N, ny = nz = 1 */
  int window;                /* ORACLE_WIN_* */
  float window_param;        /* TUKEY: taper fraction b in (0, 1] */
  int interp;                /* ORACLE_INTERP_* */
} das_oracle_opts;

int das_oracle_ex(const float* elem_pos, const float* elem_dir, int M,
                  const int* tx_type, const float* tx_v, const float* tx_t0, int Q,
                  const float* xs, int nx, const float* ys, int ny, const float* zs, int nz,
                  float c_f, float fc_f, float fs_f, float t_start_f, float f_number_f,
                  int K, int data_kind, const float* y,
                  const long long* vox_idx, long long n_vox,
                  double* out, long long* out_count, double* out_l1,
                  double* out_slack, double slack_rel, const das_oracle_opts* opts) {
  static const das_oracle_opts none = {0, 0, 0, 0, 0, 0, 0.f, 0};
  const das_oracle_opts* o = opts ? opts : &none;
  if (!elem_pos || !tx_type || !tx_v || !tx_t0 || !y || !out) return -1;
  if (!o->vox_pos && (!xs || !ys || !zs)) return -1;
  if (M < 1 || Q < 1 || nx < 1 || ny < 1 || nz < 1 || K < 2) return -1;
  if (data_kind != ORACLE_DATA_IQ && data_kind != ORACLE_DATA_RF) return -1;
  if (o->window < 0 || o->window > ORACLE_WIN_TUKEY || o->interp < 0 || o->interp > ORACLE_INTERP_CUBIC) return -1;
  if (o->window == ORACLE_WIN_TUKEY && !(o->window_param > 0.f && o->window_param <= 1.f)) return -1;
  if (o->obs_off && !o->obs_q) return -1;
  const double taper = (double)o->window_param;
  const double c = (double)c_f, fc = (double)fc_f, fs = (double)fs_f;
  const double t_start = (double)t_start_f, fnum = (double)f_number_f;
  const int iq = (data_kind == ORACLE_DATA_IQ);
  const long long n_total = (long long)nx * ny * nz;
  const long long n_eval = vox_idx ? n_vox : n_total;
  int bad = 0;

#pragma omp parallel for schedule(dynamic, 8) reduction(|:bad)
  for (long long i = 0; i < n_eval; ++i) {
    const long long n = vox_idx ? vox_idx[i] : i;
    if (n < 0 || n >= n_total) { bad = 1; continue; }
    const int iz = (int)(n % nz);
    const int iy = (int)((n / nz) % ny);
    const int ix = (int)(n / ((long long)nz * ny));
    double px, py, pz;
    if (o->vox_pos) { px = (double)o->vox_pos[3 * n]; py = (double)o->vox_pos[3 * n + 1]; pz = (double)o->vox_pos[3 * n + 2]; }
    else { px = (double)xs[ix]; py = (double)ys[iy]; pz = (double)zs[iz]; }
    double acc_re = 0.0, acc_im = 0.0, l1 = 0.0, slack = 0.0;
    long long count = 0;
    const long long n_obs = o->obs_off ? o->obs_off[n + 1] - o->obs_off[n] : (long long)Q;

    for (long long iq_ = 0; iq_ < n_obs; ++iq_) {
      const int q = o->obs_off ? o->obs_q[o->obs_off[n] + iq_] : (int)iq_;
      if (q < 0 || q >= Q) { bad = 1; continue; }
      const double vx = (double)tx_v[3 * q], vy = (double)tx_v[3 * q + 1], vz = (double)tx_v[3 * q + 2];
      const double w_tx = o->w_tx_tab ? (double)o->w_tx_tab[(size_t)q * (size_t)n_total + (size_t)n] : 1.0;
      /* reading W5 ("skip these negligible contributions"): a transmit weight of
         exactly 0 is the same as not listing the transmit -- its samples are never read and its terms not counted */
      if (w_tx == 0.0) continue;
      double tau_tx;
      if (o->tau_tx_tab) {
        tau_tx = (double)o->tau_tx_tab[(size_t)q * (size_t)n_total + (size_t)n];
      } else if (tx_type[q] == ORACLE_TX_PLANE) {
        tau_tx = (px * vx + py * vy + pz * vz) / c + (double)tx_t0[q];
      } else {
        const double ax = px - vx, ay = py - vy, az = pz - vz;
        tau_tx = sqrt(ax * ax + ay * ay + az * az) / c + (double)tx_t0[q];
      }
      for (int m = 0; m < M; ++m) {
        const double dx = px - (double)elem_pos[3 * m];
        const double dy = py - (double)elem_pos[3 * m + 1];
        const double dz = pz - (double)elem_pos[3 * m + 2];
        double nxm = 0.0, nym = 0.0, nzm = 1.0;
        if (elem_dir) { nxm = (double)elem_dir[3 * m]; nym = (double)elem_dir[3 * m + 1]; nzm = (double)elem_dir[3 * m + 2]; }
        const double dd = dx * dx + dy * dy + dz * dz;
        const double a = dx * nxm + dy * nym + dz * nzm;
        /* rho^2 = d.d - a^2.  For the default normal (0,0,1) this is dx^2 + dy^2; written that
           way there so that the edge test sees no cancellation. */
        const double rho2 = elem_dir ? (dd - a * a) : (dx * dx + dy * dy);
        int w = 1;
        double margin = 1.0;
        double w_rx = 1.0;
        if (fnum > 0.0) {
          const double lhs = 4.0 * fnum * fnum * rho2;
          const double rhs = a * a;
          w = (a > 0.0 && lhs <= rhs) ? 1 : 0;
          margin = (rhs > 0.0) ? fabs(lhs - rhs) / rhs : 1.0;
          if (w && o->window != ORACLE_WIN_BOXCAR) {
            const double u = 2.0 * fnum * sqrt(rho2 > 0.0 ? rho2 : 0.0) / a;       /* in [0, 1] */
            if (o->window == ORACLE_WIN_HANN) w_rx = 0.5 * (1.0 + cos(0.5 * ORACLE_TWO_PI * u));
            else if (u > 1.0 - taper) w_rx = 0.5 * (1.0 + cos(0.5 * ORACLE_TWO_PI * (u - 1.0 + taper) / taper));
          }
        }
        const double wgt = w_tx * w_rx;
        const double tau = tau_tx + sqrt(dd) / c;
        const double t = (tau - t_start) * fs;
        const double kf = floor(t);
        const double alpha = t - kf;
        const size_t row = ((size_t)q * M + m) * (size_t)K;
        double s_re, s_im = 0.0, mag1;
        if (o->interp == ORACLE_INTERP_CUBIC) {
          /* cubic convolution (Keys 1981, a = -1/2) on y[k-1], y[k], y[k+1], y[k+2] */
          if (!(kf >= 1.0 && kf <= (double)(K - 3))) continue;
          const long long k = (long long)kf;
          const double a2 = alpha * alpha, a3 = a2 * alpha;
          const double cw[4] = {-0.5 * a3 + a2 - 0.5 * alpha, 1.5 * a3 - 2.5 * a2 + 1.0,
                                -1.5 * a3 + 2.0 * a2 + 0.5 * alpha, 0.5 * a3 - 0.5 * a2};
          s_re = 0.0; mag1 = 0.0;
          for (int j = 0; j < 4; ++j) {
            if (iq) {
              const float* p0 = y + 2 * (row + (size_t)(k - 1 + j));
              s_re += cw[j] * (double)p0[0]; s_im += cw[j] * (double)p0[1];
              mag1 += fabs(cw[j]) * (fabs((double)p0[0]) + fabs((double)p0[1]));
            } else {
              const double yj = y[row + (size_t)(k - 1 + j)];
              s_re += cw[j] * yj; mag1 += fabs(cw[j]) * fabs(yj);
            }
          }
        } else {
        if (!(kf >= 0.0 && kf <= (double)(K - 2))) continue;
        const long long k = (long long)kf;
        if (iq) {
          const float* p0 = y + 2 * (row + (size_t)k);
          const double y0r = p0[0], y0i = p0[1], y1r = p0[2], y1i = p0[3];
          s_re = (1.0 - alpha) * y0r + alpha * y1r;
          s_im = (1.0 - alpha) * y0i + alpha * y1i;
          mag1 = (1.0 - alpha) * (fabs(y0r) + fabs(y0i)) + alpha * (fabs(y1r) + fabs(y1i));
        } else {
          const double y0 = y[row + (size_t)k], y1 = y[row + (size_t)k + 1];
          s_re = (1.0 - alpha) * y0 + alpha * y1;
          mag1 = (1.0 - alpha) * fabs(y0) + alpha * fabs(y1);
        }
        }
        if (out_slack && fnum > 0.0 && a > 0.0 && margin <= slack_rel)
          slack += sqrt(s_re * s_re + s_im * s_im);
        if (!w) continue;
        if (iq) {
          const double ph = ORACLE_TWO_PI * fc * tau;
          const double cr = cos(ph), ci = sin(ph);
          acc_re += wgt * (s_re * cr - s_im * ci);
          acc_im += wgt * (s_re * ci + s_im * cr);
        } else {
          acc_re += wgt * s_re;
        }
        l1 += fabs(wgt) * mag1;
        ++count;
      }
    }
    if (iq) { out[2 * i] = acc_re; out[2 * i + 1] = acc_im; }
    else    { out[i] = acc_re; }
    if (out_count) out_count[i] = count;
    if (out_l1) out_l1[i] = l1;
    if (out_slack) out_slack[i] = slack;
  }
  return bad ? -1 : 0;
}

/* The plain definition: das_oracle_ex with every option off. */
int das_oracle(const float* elem_pos, const float* elem_dir, int M,
               const int* tx_type, const float* tx_v, const float* tx_t0, int Q,
               const float* xs, int nx, const float* ys, int ny, const float* zs, int nz,
               float c_f, float fc_f, float fs_f, float t_start_f, float f_number_f,
               int K, int data_kind, const float* y,
               const long long* vox_idx, long long n_vox,
               double* out, long long* out_count, double* out_l1,
               double* out_slack, double slack_rel) {
  return das_oracle_ex(elem_pos, elem_dir, M, tx_type, tx_v, tx_t0, Q, xs, nx, ys, ny, zs, nz, c_f, fc_f, fs_f,
                       t_start_f, f_number_f, K, data_kind, y, vox_idx, n_vox, out, out_count, out_l1, out_slack,
                       slack_rel, (const das_oracle_opts*)0);
}
