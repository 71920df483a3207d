// sd_policy.cu -- the scalar HOST logic of SURVEY.md 8(f) f2 behind include/er.h: block efficiency,
// roofline cost model (L111-L115, L455-L476), SD toggle pi_SD (L119 Eq. 3), adaptive draft length (L168 Alg. 1 lines
// 11-12), two-step calibration (L478-L484) and the shrinking-batch rollout driver.  No device code: the file is a .cu only
// because the library is built by one nvcc command line.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

#include "er.h"

namespace {

inline double tau_series(double alpha, int gamma) {
  if (alpha == 1.0) return (double)(gamma + 1);
  return (1.0 - std::pow(alpha, (double)(gamma + 1))) / (1.0 - alpha);
}

struct Times { double T_p, T_q, T_V; };

inline double compute_term(const er_roofline_model& m, double B, double S) {
  return B * (m.C_dense + S * m.C_attn) / m.F_eff;
}

inline Times times_of(const er_roofline_model& m, double B, double S, int gamma) {
  const double kv = m.rho_kappa * m.kappa * B * S;
  const double M_T = (m.W_T + kv) / m.BW_eff;
  const double M_D = (m.eta_D * m.W_D + kv) / m.BW_eff;
  const double C = compute_term(m, B, S);
  Times t;
  t.T_p = std::max(M_T, C) + m.c_T * B + m.c_comm;
  t.T_q = std::max(M_D, C) + m.c_D * B + m.c_comm;
  t.T_V = std::max(M_T, (double)(gamma + 1) * C) + m.c_V * B + m.c_comm;
  return t;
}

inline bool model_ok(const er_roofline_model* m) { return m->F_eff > 0.0 && m->BW_eff > 0.0; }

// min ||A x - b|| for an m x k system (k <= 3) by Householder QR on column-scaled A; a column that is all zero leaves its
// unknown at 0.  A is row-major and is destroyed.
void least_squares(std::vector<double>& A, std::vector<double>& b, int m, int k, double* x) {
  int map[3], kk = 0;
  double scale[3];
  for (int j = 0; j < k; ++j) {
    double mx = 0.0;
    for (int i = 0; i < m; ++i) mx = std::max(mx, std::fabs(A[(size_t)i * k + j]));
    x[j] = 0.0;
    if (mx > 0.0) { map[kk] = j; scale[kk] = mx; ++kk; }
  }
  if (kk == 0 || m < kk) return;
  std::vector<double> Q((size_t)m * kk);
  for (int i = 0; i < m; ++i)
    for (int j = 0; j < kk; ++j) Q[(size_t)i * kk + j] = A[(size_t)i * k + map[j]] / scale[j];
  for (int j = 0; j < kk; ++j) {            // Householder reflections, applied to the right-hand side as well
    double norm = 0.0;
    for (int i = j; i < m; ++i) norm += Q[(size_t)i * kk + j] * Q[(size_t)i * kk + j];
    norm = std::sqrt(norm);
    if (norm == 0.0) continue;
    const double alpha = Q[(size_t)j * kk + j] > 0.0 ? -norm : norm;
    std::vector<double> v(m - j);
    for (int i = j; i < m; ++i) v[i - j] = Q[(size_t)i * kk + j];
    v[0] -= alpha;
    double vv = 0.0;
    for (double e : v) vv += e * e;
    if (vv == 0.0) continue;
    for (int c = j; c < kk; ++c) {
      double dot = 0.0;
      for (int i = j; i < m; ++i) dot += v[i - j] * Q[(size_t)i * kk + c];
      const double f = 2.0 * dot / vv;
      for (int i = j; i < m; ++i) Q[(size_t)i * kk + c] -= f * v[i - j];
    }
    double dot = 0.0;
    for (int i = j; i < m; ++i) dot += v[i - j] * b[i];
    const double f = 2.0 * dot / vv;
    for (int i = j; i < m; ++i) b[i] -= f * v[i - j];
  }
  double y[3] = {0.0, 0.0, 0.0};
  for (int j = kk - 1; j >= 0; --j) {       // back substitution on R
    double s = b[j];
    for (int c = j + 1; c < kk; ++c) s -= Q[(size_t)j * kk + c] * y[c];
    const double d = Q[(size_t)j * kk + j];
    y[j] = d != 0.0 ? s / d : 0.0;
  }
  for (int j = 0; j < kk; ++j) x[map[j]] = y[j] / scale[j];
}

}  // namespace

extern "C" {

int er_tau_of_alpha(double alpha, int32_t gamma, double* tau_out) {
  if (!tau_out) return ER_ERR_NULL;
  if (gamma < 1) return ER_ERR_SHAPE;
  *tau_out = tau_series(alpha, gamma);
  return ER_OK;
}

int er_alpha_of_tau(double tau, int32_t gamma, double* alpha_out) {
  if (!alpha_out) return ER_ERR_NULL;
  if (gamma < 1) return ER_ERR_SHAPE;
  if (tau <= 1.0) { *alpha_out = 0.0; return ER_OK; }
  if (tau >= (double)(gamma + 1)) { *alpha_out = 1.0; return ER_OK; }
  double lo = 0.0, hi = 1.0;                // tau is strictly increasing in alpha on [0, 1]
  for (int it = 0; it < 200; ++it) {
    const double mid = 0.5 * (lo + hi);
    if (tau_series(mid, gamma) < tau) lo = mid; else hi = mid;
  }
  *alpha_out = 0.5 * (lo + hi);
  return ER_OK;
}

int er_roofline_times(const er_roofline_model* model, double B, double S, int32_t gamma, double* T_p, double* T_q,
                      double* T_V) {
  if (!model || !T_p || !T_q || !T_V) return ER_ERR_NULL;
  if (gamma < 1 || !model_ok(model)) return ER_ERR_SHAPE;
  const Times t = times_of(*model, B, S, gamma);
  *T_p = t.T_p; *T_q = t.T_q; *T_V = t.T_V;
  return ER_OK;
}

int er_sd_toggle(const er_roofline_model* model, double B, double S, double tau, int32_t gamma, double eps, int32_t* on,
                 double* speedup) {
  if (!model || !on) return ER_ERR_NULL;
  if (gamma < 1 || !model_ok(model)) return ER_ERR_SHAPE;
  const Times t = times_of(*model, B, S, gamma);
  const double s = tau * t.T_p / ((double)gamma * t.T_q + t.T_V);     // Eq. 1 with the modelled times
  *on = s >= 1.0 + eps ? 1 : 0;
  if (speedup) *speedup = s;
  return ER_OK;
}

int er_gamma_next(const int32_t* Gamma, int32_t n, int32_t gamma_t, const double* tau_hist, int32_t n_hist, int32_t P,
                  double alpha_up, double alpha_down, int32_t* gamma_out) {
  if (!Gamma || !gamma_out || (n_hist > 0 && !tau_hist)) return ER_ERR_NULL;
  if (n < 1 || n_hist < 0 || P < 1) return ER_ERR_SHAPE;
  int idx = -1;
  for (int i = 0; i < n; ++i) {
    if (i > 0 && Gamma[i] <= Gamma[i - 1]) return ER_ERR_SHAPE;
    if (Gamma[i] == gamma_t) idx = i;
  }
  if (idx < 0) return ER_ERR_SHAPE;
  *gamma_out = gamma_t;
  if (n_hist < P) return ER_OK;             // the condition cannot have held for P consecutive steps yet
  double lo = tau_hist[n_hist - P], hi = lo;
  for (int i = n_hist - P + 1; i < n_hist; ++i) { lo = std::min(lo, tau_hist[i]); hi = std::max(hi, tau_hist[i]); }
  if (lo >= 1.0 + (double)gamma_t * alpha_up && idx + 1 < n) *gamma_out = Gamma[idx + 1];
  else if (hi <= 1.0 + (double)gamma_t * alpha_down && idx > 0) *gamma_out = Gamma[idx - 1];
  return ER_OK;
}

int er_roofline_calibrate(er_roofline_model* model, const double* tB, const double* tS, const double* tT, int32_t n_target,
                          const double* dB, const double* dS, const double* dT, int32_t n_drafter, const double* vB,
                          const double* vS, const int32_t* vgamma, const double* vT, int32_t n_verify) {
  if (!model) return ER_ERR_NULL;
  if (n_target < 0 || n_drafter < 0 || n_verify < 0 || !model_ok(model)) return ER_ERR_SHAPE;
  if ((n_target > 0 && (!tB || !tS || !tT)) || (n_drafter > 0 && (!dB || !dS || !dT)) ||
      (n_verify > 0 && (!vB || !vS || !vgamma || !vT)))
    return ER_ERR_NULL;
  er_roofline_model& m = *model;
  const int kIters = 50;
  // step 1: T_p - c_comm = max{a W_T + b kappa B S, C} + c_T B with a = 1 / BW_eff, b = rho_kappa / BW_eff
  if (n_target > 0) {
    double a = 1.0 / m.BW_eff, b = m.rho_kappa / m.BW_eff, cT = m.c_T;
    std::vector<char> cls, prev;
    for (int it = 0; it < kIters; ++it) {
      cls.assign(n_target, 0);
      for (int i = 0; i < n_target; ++i)
        cls[i] = (a * m.W_T + b * m.kappa * tB[i] * tS[i] >= compute_term(m, tB[i], tS[i])) ? 1 : 0;
      if (cls == prev) break;
      prev = cls;
      std::vector<double> A((size_t)n_target * 3), rhs(n_target);
      for (int i = 0; i < n_target; ++i) {
        A[(size_t)i * 3 + 0] = cls[i] ? m.W_T : 0.0;
        A[(size_t)i * 3 + 1] = cls[i] ? m.kappa * tB[i] * tS[i] : 0.0;
        A[(size_t)i * 3 + 2] = tB[i];
        rhs[i] = tT[i] - m.c_comm - (cls[i] ? 0.0 : compute_term(m, tB[i], tS[i]));
      }
      double x[3];
      least_squares(A, rhs, n_target, 3, x);
      if (x[0] > 0.0) a = x[0];
      b = x[1];
      cT = x[2];
    }
    m.BW_eff = 1.0 / a;
    m.rho_kappa = b / a;
    m.c_T = cT;
  }
  // step 2a: eta_D, c_D from the drafter sweep (BW_eff, rho_kappa fixed)
  if (n_drafter > 0) {
    double eta = m.eta_D, cD = m.c_D;
    std::vector<char> cls, prev;
    for (int it = 0; it < kIters; ++it) {
      cls.assign(n_drafter, 0);
      for (int i = 0; i < n_drafter; ++i) {
        const double kv = m.rho_kappa * m.kappa * dB[i] * dS[i] / m.BW_eff;
        cls[i] = (eta * m.W_D / m.BW_eff + kv >= compute_term(m, dB[i], dS[i])) ? 1 : 0;
      }
      if (cls == prev) break;
      prev = cls;
      std::vector<double> A((size_t)n_drafter * 2), rhs(n_drafter);
      for (int i = 0; i < n_drafter; ++i) {
        const double kv = m.rho_kappa * m.kappa * dB[i] * dS[i] / m.BW_eff;
        A[(size_t)i * 2 + 0] = cls[i] ? m.W_D / m.BW_eff : 0.0;
        A[(size_t)i * 2 + 1] = dB[i];
        rhs[i] = dT[i] - m.c_comm - (cls[i] ? kv : compute_term(m, dB[i], dS[i]));
      }
      double x[3];
      least_squares(A, rhs, n_drafter, 2, x);
      if (x[0] > 0.0) eta = x[0];
      cD = x[1];
    }
    m.eta_D = eta;
    m.c_D = cD;
  }
  // step 2b: c_V from the verification sweep: T_V - c_comm - max{M_T, (gamma + 1) C} = c_V B
  if (n_verify > 0) {
    double num = 0.0, den = 0.0;
    for (int i = 0; i < n_verify; ++i) {
      const double kv = m.rho_kappa * m.kappa * vB[i] * vS[i];
      const double base = std::max((m.W_T + kv) / m.BW_eff, (double)(vgamma[i] + 1) * compute_term(m, vB[i], vS[i]));
      num += vB[i] * (vT[i] - m.c_comm - base);
      den += vB[i] * vB[i];
    }
    if (den > 0.0) m.c_V = num / den;
  }
  return ER_OK;
}

int er_rollout_simulate(const er_roofline_model* model, const double* lengths, int32_t n, double S0, int32_t gamma,
                        double tau, double eps, int32_t mode, double* seconds, int64_t* steps, int64_t* ar_steps) {
  if (!model || !seconds || !steps || !ar_steps || (n > 0 && !lengths)) return ER_ERR_NULL;
  if (n < 0 || gamma < 1 || mode < 0 || mode > 2 || !model_ok(model) || !(tau > 0.0)) return ER_ERR_SHAPE;
  std::vector<double> L(lengths, lengths + n);
  std::sort(L.begin(), L.end());
  double pos = 0.0, t = 0.0;
  int64_t st = 0, ar = 0;
  bool sd_on = mode == 1;
  const double Lmax = n > 0 ? L[n - 1] : 0.0;
  size_t done = 0;                           // sequences with length <= pos
  while (pos < Lmax) {
    while (done < L.size() && L[done] <= pos) ++done;
    const double B = (double)(L.size() - done), S = S0 + pos;
    const Times tm = times_of(*model, B, S, gamma);
    if (mode == 2 && !sd_on && tau * tm.T_p / ((double)gamma * tm.T_q + tm.T_V) >= 1.0 + eps) sd_on = true;
    if (sd_on) {
      t += (double)gamma * tm.T_q + tm.T_V;
      pos += tau;
    } else {
      t += tm.T_p;
      pos += 1.0;
      ++ar;
    }
    ++st;
  }
  *seconds = t; *steps = st; *ar_steps = ar;
  return ER_OK;
}

}  // extern "C"
