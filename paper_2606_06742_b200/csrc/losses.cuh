// losses.cuh -- the loss table of the library on the device: psi = d loss / d f of the (smoothed) training
// losses (S5; readings G10, G20) and the nominal losses that score held-out rows (S9).
#pragma once

#include "common.cuh"

namespace tkm {

__device__ __forceinline__ double psi_dev(int loss, double y, double f, double smooth, double tau) {
  if (loss == TKM_LOSS_HINGE) {
    const double u = y * f;   // L'_delta(u): -1 | (u - 1 - delta)/(2 delta) | 0
    const double lp = (u <= 1.0 - smooth) ? -1.0 : ((u >= 1.0 + smooth) ? 0.0 : (u - 1.0 - smooth) / (2.0 * smooth));
    return y * lp;
  } else if (loss == TKM_LOSS_LOGISTIC) {
    const double u = y * f;   // -y / (1 + e^u), overflow-safe
    const double e = exp(-fabs(u));
    const double sg = (u >= 0.0) ? e / (1.0 + e) : 1.0 / (1.0 + e);
    return -y * sg;
  } else if (loss == TKM_LOSS_DWD) {
    const double u = y * f;   // V'(u) = -1 (u <= 1/2), -1/(4 u^2) (u > 1/2)   (reading G20)
    return y * ((u <= 0.5) ? -1.0 : -1.0 / (4.0 * u * u));
  } else {
    const double t = y - f;   // -H'_gamma(t)  (reading G10)
    const double hp = (t < -smooth) ? tau - 1.0 : ((t > smooth) ? tau : t / (2.0 * smooth) + tau - 0.5);
    return -hp;
  }
}

__device__ __forceinline__ double nominal_loss_dev(int loss, double y, double f, double tau) {
  if (loss == TKM_LOSS_HINGE) return fmax(1.0 - y * f, 0.0);
  if (loss == TKM_LOSS_LOGISTIC) {
    const double u = y * f;
    return fmax(-u, 0.0) + log1p(exp(-fabs(u)));
  }
  if (loss == TKM_LOSS_DWD) {
    const double u = y * f;
    return (u <= 0.5) ? 1.0 - u : 1.0 / (4.0 * u);
  }
  const double t = y - f;
  return t * (tau - (t < 0.0 ? 1.0 : 0.0));
}

}  // namespace tkm
