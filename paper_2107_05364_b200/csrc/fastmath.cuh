// fastmath.cuh — fp64 helpers of the assembly kernels (A1/A2) for the argument ranges the closed
// forms produce.  ncu (profiles/r04_b8_ncu_full.md): the shipped kernel issued 1,289 instructions per
// tile pair of which 478 were FP64 arithmetic; most of the rest was the scaffolding of the library
// log / atan2 / division (exponent extraction, special cases, slow-path checks).  All but the nearest
// pairs have SMALL arguments — the angle of a diagonal component and the logarithm of an off-diagonal
// one are O((edge/r)^3) — where a division by a positive, well-scaled number and a short odd series
// are all that is needed:
//   atan(t)  = t - t^3/3 + t^5/5 - ...          |t| <= 1/8: 8 terms after t, truncation 3e-18 relative
//   atanh(s) = s + s^3/3 + s^5/5 + ...          |s| <= 1/8: same
// (Taylor coefficients are exact rationals; at |x| <= 1/8 the series needs no minimax fit.)
// Everything outside the small range goes to the library function, so accuracy near the source is what
// it was.  Inputs of quot_pos must be finite with a positive NORMAL denominator well inside the exponent
// range (the callers normalise lengths to the source's size).
#pragma once

// 1/c for positive normal c: 64-bit MUFU seed (20 mantissa bits) + one cubic Newton step: the
// approximation error becomes e^3 ~ 2^-60, what is left is the rounding of the last fma
__device__ __forceinline__ double rcp_pos(double c) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(c));
  const double e = fma(-c, r, 1.0);
  return fma(r, fma(e, e, e), r);
}
// s / c: product with the reciprocal, then one residual correction (<= 1 ulp)
__device__ __forceinline__ double quot_pos(double s, double c) {
  const double r = rcp_pos(c);
  const double t = s * r;
  return fma(fma(-c, t, s), r, t);
}
// sum_{k>=1} sign^k z^k / (2k+1), 8 terms, z = x^2 <= 1/64
template <bool kAlternating>
__device__ __forceinline__ double odd_series_tail(double z) {
  constexpr double sg = kAlternating ? -1.0 : 1.0;
  double p = 1.0 / 17.0;                // k = 8: sign^8 = +
  p = fma(p, z, sg / 15.0);
  p = fma(p, z, 1.0 / 13.0);
  p = fma(p, z, sg / 11.0);
  p = fma(p, z, 1.0 / 9.0);
  p = fma(p, z, sg / 7.0);
  p = fma(p, z, 1.0 / 5.0);
  p = fma(p, z, sg / 3.0);
  return p * z;
}
__device__ __forceinline__ double atan_small(double t) { return fma(t, odd_series_tail<true>(t * t), t); }
__device__ __forceinline__ double atanh_small(double s) { return fma(s, odd_series_tail<false>(s * s), s); }

// atan2(s, c), any arguments; the small-angle branch needs c > 0 (implied by its test unless both are 0)
__device__ __forceinline__ double atan2_fast(double s, double c) {
  if (fabs(s) <= 0.125 * c && c > 0.0) return atan_small(quot_pos(s, c));
  return atan2(s, c);
}
// ln(a / b) for a, b > 0: 2 atanh((a - b)/(a + b)) near 1 (the subtraction is exact there), log otherwise
__device__ __forceinline__ double log_ratio_fast(double a, double b) {
  const double d = a - b, s = a + b;
  if (fabs(d) <= 0.125 * s) return 2.0 * atanh_small(quot_pos(d, s));
  return log(a / b);
}

// sqrt(x) for positive normal x without the library's special-case branch (whose convergence barriers
// keep the compiler from interleaving the eight independent square roots of a pair): 64-bit MUFU seed
// of 1/sqrt(x) (20 bits), ONE coupled Goldschmidt step (g -> sqrt(x), h -> 1/(2 sqrt(x)): 40 bits) and one
// residual correction g += (x - g^2) h, which squares the error once more: <= 1 ulp (checked against long
// double on 2e6 arguments with seed errors up to 2^-20: worst 0.999 x 2^-53 relative).  x = 0 gives NaN
// (inf * 0): a target on a source corner is singular anyway.
__device__ __forceinline__ double sqrt_pos(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y, h = 0.5 * y;
  const double e = fma(-h, g, 0.5);
  g = fma(g, e, g);
  h = fma(h, e, h);
  return fma(fma(-g, g, x), h, g);
}

// 1/sqrt(x) to ~1e-12 relative for positive normal x: 64-bit MUFU seed (20 bits) + one Goldschmidt step
// (40 bits), branch-free.  For the far-field quadrature (F2), whose own truncation error is of that size
// and whose terms do not cancel; NOT for the closed forms.
__device__ __forceinline__ double rsqrt_pos_40(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double h = 0.5 * y;
  const double e = fma(-h, x * y, 0.5);
  return fma(y, e, y);
}

// Several small-argument evaluations at once: r[k] = atan(n[k]/d[k]) for k < NA, atanh(n[k]/d[k]) for
// NA <= k < NA + NH (atan's series is atanh's at -t^2, so all share the coefficients and run as
// independent chains the compiler can interleave).  Requires |n[k]| <= d[k]/8, d[k] > 0.
// A cuboid pair has NA = 3 angles + NH = 3 logs, a tetrahedron pair 4 solid angles + 6 edge logs.
template <int NA, int NH>
__device__ __forceinline__ void many_small(const double* n, const double* d, double* r) {
  constexpr int K = NA + NH;
  double t[K], u[K], p[K];
#pragma unroll
  for (int k = 0; k < K; ++k) t[k] = quot_pos(n[k], d[k]);
#pragma unroll
  for (int k = 0; k < K; ++k) {
    u[k] = t[k] * t[k];
    if (k < NA) u[k] = -u[k];
    p[k] = 1.0 / 17.0;
  }
  constexpr double c[7] = {1.0 / 15.0, 1.0 / 13.0, 1.0 / 11.0, 1.0 / 9.0, 1.0 / 7.0, 1.0 / 5.0, 1.0 / 3.0};
#pragma unroll
  for (int j = 0; j < 7; ++j)
#pragma unroll
    for (int k = 0; k < K; ++k) p[k] = fma(p[k], u[k], c[j]);
#pragma unroll
  for (int k = 0; k < K; ++k) r[k] = fma(t[k], p[k] * u[k], t[k]);
}
