// oracle/eos.h — CPU ORACLE (test infrastructure only; see oracle.h): equation of state.
//
// kind 0: ideal gas, P = (Gamma-1) rho eps, T = P/rho (DESIGN.md §3 O1, reading R3).
// kind 1: piecewise-polytropic hybrid EOS ("supports ideal gases and piecewise polytropic
//   hybrid EOSs"; the paper prints no formula — DESIGN.md reading R29 fixes the usual one):
//     cold part, segment i (rho_b[i-1] <= rho < rho_b[i]):
//       P_c = K_i rho^Gamma_i,   eps_c = a_i + K_i rho^(Gamma_i - 1) / (Gamma_i - 1)
//       with K_i, a_i continuous at the breakpoints (a_0 = 0), so d eps_c / d rho = P_c / rho^2;
//     thermal part: P = P_c + (Gamma_th - 1) rho (eps - eps_c),  eps >= eps_c;
//     "temperature" T = (P - P_c)/rho, so that K = 0 is the ideal gas with Gamma = Gamma_th;
//     h = 1 + eps + P/rho,   c_s^2 = [Gamma_i P_c + Gamma_th (P - P_c)] / (rho h).
// Every function below evaluates the ideal gas with exactly the operations of DESIGN.md §3.
// Pins: tests/test_oracle_eos.py (T31).  Parity unpinned: which temperature the floors of P:139
// act on for the hybrid EOS (the paper is silent; R29 takes the thermal one).
#ifndef GRMHD_ORACLE_EOS_H
#define GRMHD_ORACLE_EOS_H
#include "oracle.h"
#include <cmath>

struct OrcEos {
  int kind;
  double gam, gm1, gm1r;           // ideal gas: Gamma, Gamma-1, Gamma/(Gamma-1)
  int nseg;
  double K[4], G[4], a[4], rb[3];  // hybrid: K_i, Gamma_i, eps offsets a_i, breakpoints
  double gth, gthm1;               // Gamma_th, Gamma_th - 1
};

inline OrcEos orc_make_eos(const orc_params* p) {
  OrcEos e{};
  e.kind = p->eos;
  e.gam = p->gamma_ad; e.gm1 = p->gamma_ad - 1.0; e.gm1r = p->gamma_ad / (p->gamma_ad - 1.0);
  if (e.kind == 1) {
    e.nseg = p->pp_nseg;
    e.gth = p->gamma_th; e.gthm1 = p->gamma_th - 1.0;
    for (int i = 0; i < e.nseg; ++i) e.G[i] = p->pp_gamma[i];
    for (int i = 0; i + 1 < e.nseg; ++i) e.rb[i] = p->pp_rho[i];
    e.K[0] = p->pp_K0; e.a[0] = 0.0;
    for (int i = 1; i < e.nseg; ++i) {
      const double r = e.rb[i - 1];
      e.K[i] = e.K[i - 1] * std::pow(r, e.G[i - 1] - e.G[i]);               // P_c continuous
      e.a[i] = e.a[i - 1] + e.K[i - 1] * std::pow(r, e.G[i - 1] - 1.0) / (e.G[i - 1] - 1.0)
               - e.K[i] * std::pow(r, e.G[i] - 1.0) / (e.G[i] - 1.0);       // eps_c continuous
    }
  }
  return e;
}

// cold part at rho (hybrid only): P_c, eps_c and the segment's Gamma_i
inline void eos_cold(const OrcEos& e, double rho, double& Pc, double& epsc, double& Gi) {
  int i = 0;
  while (i + 1 < e.nseg && rho >= e.rb[i]) ++i;
  Gi = e.G[i];
  Pc = e.K[i] * std::pow(rho, Gi);
  epsc = e.a[i] + Pc / ((Gi - 1.0) * rho);
}

// h - 1 and c_s^2 from (rho, P)
inline void eos_hm1_cs2(const OrcEos& e, double rho, double P, double& hm1, double& cs2) {
  if (e.kind == 0) {
    const double T = P / rho;
    hm1 = e.gm1r * T;
    const double h = 1.0 + hm1;
    cs2 = e.gam * T / h;                      // Gamma P / (rho h)
  } else {
    double Pc, epsc, Gi;
    eos_cold(e, rho, Pc, epsc, Gi);
    const double Pth = P - Pc;
    const double eps = epsc + Pth / (e.gthm1 * rho);
    hm1 = eps + P / rho;
    const double h = 1.0 + hm1;
    cs2 = (Gi * Pc + e.gth * Pth) / (rho * h);
  }
}
inline double eos_hm1(const OrcEos& e, double rho, double P) {
  double hm1, cs2;
  eos_hm1_cs2(e, rho, P, hm1, cs2);
  return hm1;
}

// P(rho, eps)
inline double eos_P(const OrcEos& e, double rho, double eps) {
  if (e.kind == 0) {
    const double T = e.gm1 * eps;
    return rho * T;
  }
  double Pc, epsc, Gi;
  eos_cold(e, rho, Pc, epsc, Gi);
  return Pc + e.gthm1 * rho * (eps - epsc);
}

// pressure and specific internal energy of matter of density rho at temperature T
inline double eos_P_at_T(const OrcEos& e, double rho, double T) {
  if (e.kind == 0) return rho * T;
  double Pc, epsc, Gi;
  eos_cold(e, rho, Pc, epsc, Gi);
  return Pc + rho * T;
}
inline double eos_eps_at_T(const OrcEos& e, double rho, double T) {
  if (e.kind == 0) return T / e.gm1;
  double Pc, epsc, Gi;
  eos_cold(e, rho, Pc, epsc, Gi);
  return epsc + T / e.gthm1;
}
// temperature floor: returns true and raises P if T(rho, P) < T_atm
inline bool eos_T_floor(const OrcEos& e, double rho, double T_atm, double& P) {
  if (e.kind == 0) {
    if (P < rho * T_atm) { P = rho * T_atm; return true; }
    return false;
  }
  double Pc, epsc, Gi;
  eos_cold(e, rho, Pc, epsc, Gi);
  if (P - Pc < rho * T_atm) { P = Pc + rho * T_atm; return true; }
  return false;
}

#endif
