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
 * Every float input is promoted to double as is; nothing is re-derived.
 * Compile WITHOUT -ffast-math and with -ffp-contract=off (oracle/build.py does).
 *
 * Pins: tests/test_oracle_pins.py (closed forms from Pythagorean-triple geometries stored in
 * tests/golden/, impulse response, dense-matrix brute force, linearity, time-shift invariance,
 * transmit additivity, mirror symmetry, RF = Re(IQ at fc = 0), aperture count in exact rational
 * arithmetic, point-scatterer peak and peak value bound).  Parity unpinned: none of the sum
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
int das_oracle(const float* elem_pos, const float* elem_dir, int M,
               const int* tx_type, const float* tx_v, const float* tx_t0, int Q,
               const float* xs, int nx, const float* ys, int ny, const float* zs, int nz,
               float c_f, float fc_f, float fs_f, float t_start_f, float f_number_f,
               int K, int data_kind, const float* y,
               const long long* vox_idx, long long n_vox,
               double* out, long long* out_count, double* out_l1,
               double* out_slack, double slack_rel) {
  if (!elem_pos || !tx_type || !tx_v || !tx_t0 || !xs || !ys || !zs || !y || !out) return -1;
  if (M < 1 || Q < 1 || nx < 1 || ny < 1 || nz < 1 || K < 2) return -1;
  if (data_kind != ORACLE_DATA_IQ && data_kind != ORACLE_DATA_RF) return -1;
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
    const double px = (double)xs[ix], py = (double)ys[iy], pz = (double)zs[iz];
    double acc_re = 0.0, acc_im = 0.0, l1 = 0.0, slack = 0.0;
    long long count = 0;

    for (int q = 0; q < Q; ++q) {
      const double vx = (double)tx_v[3 * q], vy = (double)tx_v[3 * q + 1], vz = (double)tx_v[3 * q + 2];
      double tau_tx;
      if (tx_type[q] == ORACLE_TX_PLANE) {
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
        if (fnum > 0.0) {
          const double lhs = 4.0 * fnum * fnum * rho2;
          const double rhs = a * a;
          w = (a > 0.0 && lhs <= rhs) ? 1 : 0;
          margin = (rhs > 0.0) ? fabs(lhs - rhs) / rhs : 1.0;
        }
        const double tau = tau_tx + sqrt(dd) / c;
        const double t = (tau - t_start) * fs;
        const double kf = floor(t);
        const double alpha = t - kf;
        if (!(kf >= 0.0 && kf <= (double)(K - 2))) continue;
        const long long k = (long long)kf;
        double s_re, s_im = 0.0, mag1;
        const size_t row = ((size_t)q * M + m) * (size_t)K;
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
        if (out_slack && fnum > 0.0 && a > 0.0 && margin <= slack_rel)
          slack += sqrt(s_re * s_re + s_im * s_im);
        if (!w) continue;
        if (iq) {
          const double ph = ORACLE_TWO_PI * fc * tau;
          const double cr = cos(ph), ci = sin(ph);
          acc_re += s_re * cr - s_im * ci;
          acc_im += s_re * ci + s_im * cr;
        } else {
          acc_re += s_re;
        }
        l1 += mag1;
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
