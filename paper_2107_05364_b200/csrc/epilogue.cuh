// epilogue.cuh — per-row fused epilogue of the demag kernels: local fields (A5), Landau-Lifshitz
// right-hand side (A6), Runge-Kutta stage combine and DP45 error estimate (A8/A9).
// One thread handles one (row i, state b) pair once the row's H_d is reduced.
#pragma once
#include "mt_internal.cuh"

__device__ __forceinline__ void atomic_max_nonneg(unsigned long long* p, double v) {
  // bit patterns of non-negative doubles order like unsigned integers; NaN (all-ones exponent with
  // mantissa) compares above every finite value, so a NaN handed to this function is never lost —
  // callers must not launder it through fmax() first (fmax drops NaN operands).  A NaN is stored as the
  // canonical positive quiet NaN so that the word also orders correctly as a SIGNED integer (the
  // max-reduction over ranks of a row-sharded problem may be done on int64, mt.h section 8(e)).
  atomicMax(p, v != v ? 0x7ff8000000000000ull : (unsigned long long)__double_as_longlong(v));
}

__device__ __forceinline__ void cross3(const double a[3], const double b[3], double o[3]) {
  o[0] = a[1] * b[2] - a[2] * b[1];
  o[1] = a[2] * b[0] - a[0] * b[2];
  o[2] = a[0] * b[1] - a[1] * b[0];
}

// Runge-Kutta stage combine: y_out = base + h * sum_j coef[j] k_j (k_j == k_out taken from kcur when
// given), optional renormalisation, optional staging of Ms*y_out for the next field evaluation.
__device__ __forceinline__ void stage_combine(const EpiArgs& e, int64_t i, int b, const double* kcur) {
  const int64_t n = e.n;
  const int64_t sb = (int64_t)b * 3 * n;
  const double h = e.h_dev ? *e.h_dev : e.h;
  double yo[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double s = 0.0;
    for (int j = 0; j < e.ncomb; ++j) {
      const double kj = (kcur && e.kptr[j] == e.k_out) ? kcur[a] : e.kptr[j][sb + a * n + i];
      s += e.coef[j] * kj;
    }
    yo[a] = e.base[sb + a * n + i] + h * s;
  }
  if (e.renorm) {
    // a zero-length m_i (a non-magnetic tile) stays zero instead of becoming 0/0 (Q10c)
    const double r = sqrt(yo[0] * yo[0] + yo[1] * yo[1] + yo[2] * yo[2]);
    if (r > 0.0) {
#pragma unroll
      for (int a = 0; a < 3; ++a) yo[a] /= r;
    }
  }
  const int64_t yld = e.y_ld ? e.y_ld : n;
  double* yout = e.y_out + (int64_t)b * 3 * yld + (i - e.y_row0);
#pragma unroll
  for (int a = 0; a < 3; ++a) yout[a * yld] = yo[a];
  if (e.M_out) {
    const double ms = e.Ms[i];
    const int64_t sm = (int64_t)b * 3 * e.npad;
    if (e.M_dtype == MT_F32) {
      float* M = (float*)e.M_out + sm;
#pragma unroll
      for (int a = 0; a < 3; ++a) M[a * e.npad + i] = (float)(ms * yo[a]);
    } else {
      double* M = (double*)e.M_out + sm;
#pragma unroll
      for (int a = 0; a < 3; ++a) M[a * e.npad + i] = ms * yo[a];
    }
  }
}

// hd = H_d,i for state b (already carrying the minus sign of H = -N.M); i = row of the launch.
__device__ __forceinline__ void row_epilogue(const EpiArgs& e, int64_t i, int b, const double hd[3]) {
  if (e.mode == 0) {
    double* o = e.Hd + (int64_t)b * 3 * e.n_rows;
    o[i] = hd[0];
    o[e.n_rows + i] = hd[1];
    o[2 * e.n_rows + i] = hd[2];
    return;
  }
  if (e.active_dev && !*e.active_dev) return;  // device-resident controller: this attempt does not integrate
  i += e.row0;  // per-tile arrays and state vectors are full-size: global tile index from here on
  const int64_t n = e.n;
  const int64_t sb = (int64_t)b * 3 * n;
  const double* y = e.y + sb;
  const double mi[3] = {y[i], y[n + i], y[2 * n + i]};
  double H[3] = {hd[0], hd[1], hd[2]};
  double ed[4] = {0.0, 0.0, 0.0, 0.0};  // m.H_d, m.H_exch, m.H_anis, m.H_a (only used for e.e_dens)
  // exchange: Eq. 12, 3-point stencil, Neumann ghost = self
  if (e.nbr) {
    const double cex = e.c_ex ? e.c_ex[i] : e.c_ex_s;
    double hx[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int dir = 0; dir < 3; ++dir) {
      const int32_t jm = e.nbr[6 * i + 2 * dir], jp = e.nbr[6 * i + 2 * dir + 1];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        const double mm = jm >= 0 ? y[a * n + jm] : mi[a];
        const double mp = jp >= 0 ? y[a * n + jp] : mi[a];
        hx[a] += (mp - 2.0 * mi[a] + mm) * e.inv_d2[dir];
      }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) H[a] += cex * hx[a];
    ed[1] = cex * (mi[0] * hx[0] + mi[1] * hx[1] + mi[2] * hx[2]);
  }
  // uniaxial anisotropy: Eq. 16; applied field: Eq. 7
  {
    const double can = e.c_an ? e.c_an[i] : e.c_an_s;
    double ax[3], ha[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      ax[a] = e.easy ? e.easy[3 * i + a] : e.easy_c[a];
      ha[a] = e.H_a ? e.H_a[3 * i + a] : e.H_a_c[a];
    }
    const double me = mi[0] * ax[0] + mi[1] * ax[1] + mi[2] * ax[2];
#pragma unroll
    for (int a = 0; a < 3; ++a) H[a] += can * me * ax[a] + ha[a];
    ed[2] = can * me * me;
    ed[3] = mi[0] * ha[0] + mi[1] * ha[1] + mi[2] * ha[2];
  }
  // F4: energy densities of the four terms (Eq. 8, 11, 15, 6: PAPER.md:74, 89, 110, 66), each through
  // its field: -(1/2) Ms V m.H for the terms quadratic in m, -Ms V m.H_a for the Zeeman term
  if (e.e_dens) {
    ed[0] = mi[0] * hd[0] + mi[1] * hd[1] + mi[2] * hd[2];
    const double w = e.Ms[i] * (e.vol ? e.vol[i] : 1.0);
    double* eo = e.e_dens + (int64_t)b * 4 * n;
    eo[i] = -0.5 * w * ed[0];
    eo[n + i] = -0.5 * w * ed[1];
    eo[2 * n + i] = -0.5 * w * ed[2];
    eo[3 * n + i] = -w * ed[3];
  }
  // Landau-Lifshitz: Eq. 1
  double mxH[3], mxmxH[3], k[3];
  cross3(mi, H, mxH);
  cross3(mi, mxH, mxmxH);
#pragma unroll
  for (int a = 0; a < 3; ++a) k[a] = -e.gamma * mxH[a] - e.alpha * mxmxH[a];
  if (e.k_out) {
    double* ko = e.k_out + sb;
#pragma unroll
    for (int a = 0; a < 3; ++a) ko[a * n + i] = k[a];
  }
  if (e.heff_out) {
    double* ho = e.heff_out + sb;
#pragma unroll
    for (int a = 0; a < 3; ++a) ho[a * n + i] = H[a];
  }
  if (e.torque_bits)
    atomic_max_nonneg(e.torque_bits, sqrt(mxH[0] * mxH[0] + mxH[1] * mxH[1] + mxH[2] * mxH[2]));
  // DP45 error estimate (uses k just stored when eptr[j] == k_out)
  if (e.nerr > 0) {
    double err = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      double s = 0.0;
      for (int j = 0; j < e.nerr; ++j) {
        const double kj = (e.eptr[j] == e.k_out) ? k[a] : e.eptr[j][sb + a * n + i];
        s += e.ecoef[j] * kj;
      }
      s *= e.h_dev ? *e.h_dev : e.h;
      const double sc = e.atol + e.rtol * fmax(fabs(e.ebase[sb + a * n + i]), fabs(mi[a]));
      const double q = fabs(s) / sc;
      err = (q > err || q != q) ? q : err;  // a NaN must reach the controller (Q11b)
    }
    atomic_max_nonneg(e.err_bits, err);
  }
  if (e.do_comb) stage_combine(e, i, b, k);
}
