// dp_control.cuh — the DP45 step controller (A9) as device functions on a DpState: used by the one-thread
// controller kernels of the graph-replayed attempt (demag.cu) and by the tensor-resident DP45 kernel
// (resident.cu), where thread 0 of every CTA runs them on the CTA's own copy of the state.
#pragma once
#include "mt_internal.cuh"

// ---- device-resident DP45 controller (A9): the host loop of mt_integrate, one thread ------------------
// Same rules as the host controller (Q11/Q11b): dp_begin is the top of the loop (stop tests,
// clipping to the next sample time / t_end, h_min), dp_decide its bottom (accept / reject, next dt).
__device__ __forceinline__ double dp_bits(unsigned long long b) { return __longlong_as_double((long long)b); }

__device__ __forceinline__ void dp_take_sample(DpState* s) {
  if (s->has_samples && s->n_samples < s->sample_cap) {
    s->sample_flag = 1;
    s->sample_row = s->n_samples++;
    s->sample_t = s->t;
  }
  s->next_sample++;
}

__device__ __forceinline__ void dp_begin(DpState* s) {
  s->active = 0;
  s->accept = 0;
  s->sample_flag = 0;
  if (s->status != MT_DP_RUN) return;
  if (!(s->t < s->t_end)) { s->status = MT_DP_T_END; return; }
  if (s->torque_tol > 0 && s->max_torque <= s->torque_tol) { s->status = MT_DP_TORQUE; return; }
  if (s->max_steps > 0 && s->accepted + s->rejected >= s->max_steps) { s->status = MT_DP_MAX_STEPS; return; }
  double t_target = s->t_end;
  int hit_sample = 0;
  if (s->sample_dt > 0) {
    const double ts = s->t0 + (double)s->next_sample * s->sample_dt;
    if (ts <= t_target) { t_target = ts; hit_sample = 1; }
  }
  double h = s->dt;
  int clipped = 0;
  if (s->t + h >= t_target) { h = t_target - s->t; clipped = 1; }
  const double h_min = 16.0 * 2.220446049250313e-16 * fmax(fabs(s->t), fabs(s->t_end));
  if (h <= h_min) {
    if (clipped) {  // land on the target without a step
      s->t = t_target;
      if (hit_sample) dp_take_sample(s);
      return;
    }
    s->status = MT_DP_UNDERFLOW;
    return;
  }
  s->h = h;
  s->t_target = t_target;
  s->clipped = clipped;
  s->hit_sample = hit_sample;
  s->err_bits = 0ull;
  s->tq_bits = 0ull;
  s->active = 1;
}

__device__ __forceinline__ void dp_decide(DpState* s) {
  if (!s->active) return;
  s->rhs_calls += 6;
  const double err = dp_bits(s->err_bits), tq7 = dp_bits(s->tq_bits);
  if (!(err == err) || err > 1.79e308) {  // NaN/inf state or slope: no step size can repair it (Q11b)
    s->rejected++;
    s->status = MT_DP_NONFINITE;
    return;
  }
  double fac = err > 0 ? 0.9 * pow(err, -0.2) : 5.0;
  fac = fmin(5.0, fmax(0.2, fac));
  const double h = s->h;
  if (err <= 1.0) {
    s->t = s->clipped ? s->t_target : s->t + h;
    s->accept = 1;
    s->max_torque = tq7;
    s->accepted++;
    s->dt_last = h;
    if (s->clipped && s->hit_sample) dp_take_sample(s);
    s->dt = s->clipped ? fmax(s->dt, h * fac) : h * fac;
  } else {
    s->rejected++;
    s->dt = h * fmin(1.0, fac);
  }
}

