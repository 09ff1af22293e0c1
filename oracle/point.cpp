// oracle/point.cpp — CPU ORACLE, point-level steps O0..O6 (test infrastructure only;
// see oracle.h).  Build with -O2 -ffp-contract=off: every operation below is a single
// IEEE fp64 +,-,*,/,sqrt,fmin,fmax or comparison, evaluated in the order written.
#include "oracle.h"
#include "eos.h"
#include <cmath>

namespace {

inline bool fin(double x) { return std::isfinite(x); }

// a_i = g_ij a^j, accumulated left to right (DESIGN.md §3 "canonical arithmetic").
inline void lower(const double g[6], const double a[3], double out[3]) {
  out[0] = g[0] * a[0] + g[1] * a[1] + g[2] * a[2];
  out[1] = g[1] * a[0] + g[3] * a[1] + g[4] * a[2];
  out[2] = g[2] * a[0] + g[4] * a[1] + g[5] * a[2];
}
inline double dot(const double a[3], const double b[3]) {
  return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}

}  // namespace

// ---------------------------------------------------------------- O0 -------
// P:103 only defines A~ = sqrt(gamma) A; determinant by cofactors of row 1,
// inverse = cofactor * (1/det).
extern "C" void orc_metric_inverse(const double g[6], double* det, double* sdet,
                                   double ginv[6]) {
  const double gxx = g[0], gxy = g[1], gxz = g[2], gyy = g[3], gyz = g[4], gzz = g[5];
  const double cxx = gyy * gzz - gyz * gyz;
  const double cxy = gxz * gyz - gxy * gzz;
  const double cxz = gxy * gyz - gxz * gyy;
  const double d = gxx * cxx + gxy * cxy + gxz * cxz;
  const double id = 1.0 / d;
  ginv[0] = cxx * id;
  ginv[1] = cxy * id;
  ginv[2] = cxz * id;
  ginv[3] = (gxx * gzz - gxz * gxz) * id;
  ginv[4] = (gxy * gxz - gxx * gyz) * id;
  ginv[5] = (gxx * gyy - gxy * gxy) * id;
  *det = d;
  *sdet = std::sqrt(d);
}

// ---------------------------------------------------------------- O1/O2 ----
// Eq. 6 with the ideal gas h = 1 + Gamma/(Gamma-1) T, T = P/rho
// ("temperature"; P = rho T pinned by P:283).  tau in the algebraically
// identical cancellation-free form (DESIGN.md §3 O2).
namespace {
void prim2cons_eos(const OrcEos& e, const double g[6], const double prim[5], const double B[3],
                   double cons[5]) {
  const double rho = prim[0], P = prim[4];
  const double u[3] = {prim[1], prim[2], prim[3]};
  double ul[3], Bl[3];
  lower(g, u, ul);
  const double usq = dot(ul, u);
  const double W = std::sqrt(1.0 + usq);
  const double iW = 1.0 / W;
  const double vl[3] = {ul[0] * iW, ul[1] * iW, ul[2] * iW};
  lower(g, B, Bl);
  const double B2 = dot(Bl, B);
  const double Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2];
  const double hm1 = eos_hm1(e, rho, P);
  const double h = 1.0 + hm1;
  const double D = rho * W;
  const double wtot = rho * h * W * W + B2;
  cons[0] = D;
  cons[1] = wtot * vl[0] - Bv * Bl[0];
  cons[2] = wtot * vl[1] - Bv * Bl[1];
  cons[3] = wtot * vl[2] - Bv * Bl[2];
  cons[4] = D * (hm1 * W + usq / (1.0 + W)) + B2 - P - 0.5 * (Bv * Bv + B2 * iW * iW);
}
}  // namespace

extern "C" void orc_prim2cons(double gamma_ad, const double g[6], const double prim[5],
                              const double B[3], double cons[5]) {
  orc_params ideal{};
  ideal.gamma_ad = gamma_ad;
  prim2cons_eos(orc_make_eos(&ideal), g, prim, B, cons);
}
extern "C" void orc_prim2cons_eos(const orc_params* p, const double g[6], const double prim[5],
                                  const double B[3], double cons[5]) {
  prim2cons_eos(orc_make_eos(p), g, prim, B, cons);
}
extern "C" void orc_eos_point(const orc_params* p, double rho, double eps, double out[5]) {
  const OrcEos e = orc_make_eos(p);
  out[0] = eos_P(e, rho, eps);
  eos_hm1_cs2(e, rho, out[0], out[1], out[2]);
  out[3] = 0.0; out[4] = 0.0;
  if (e.kind == 1) { double Gi; eos_cold(e, rho, out[3], out[4], Gi); }
}

// ---------------------------------------------------------------- O3 -------
// Master function of the bracketed 1-D solve for mu = 1/(W h) ("based on
// the algorithm presented in Kastaun et al. (2021)").  h0 = 1 for the ideal gas.
namespace {
struct C2PState { double q, r2, bs2, rb2, v0sq, gm1; const OrcEos* eos; double D; };
struct C2PAux { double x, rbar2, qbar, vsq, iW, What, eps; };

inline void c2p_aux(const C2PState& s, double mu, C2PAux& a) {
  a.x = 1.0 / (1.0 + mu * s.bs2);
  a.rbar2 = s.r2 * a.x * a.x + mu * a.x * (1.0 + a.x) * s.rb2;
  a.qbar = s.q - 0.5 * s.bs2 - 0.5 * mu * mu * a.x * a.x * (s.bs2 * s.r2 - s.rb2);
  a.vsq = std::fmin(mu * mu * a.rbar2, s.v0sq);
  a.iW = std::sqrt(1.0 - a.vsq);
  a.What = 1.0 / a.iW;
  a.eps = a.What * (a.qbar - mu * a.rbar2) + a.vsq * a.What * a.What / (1.0 + a.What);
}
inline double c2p_f(const C2PState& s, double mu) {
  C2PAux a;
  c2p_aux(s, mu, a);
  double eps, ahat;
  if (s.eos->kind == 0) {
    eps = std::fmax(a.eps, 0.0);
    ahat = s.gm1 * eps / (1.0 + eps);  // P/(rho(1+eps)) for P=(Gamma-1) rho eps
  } else {                             // general form: a^ = P(rho^, eps^) / (rho^ (1 + eps^))
    const double rhohat = s.D * a.iW;
    double Pc, epsc, Gi;
    eos_cold(*s.eos, rhohat, Pc, epsc, Gi);
    eps = std::fmax(a.eps, epsc);      // eps^ clamped into the EOS range (eps >= eps_c)
    const double Phat = Pc + s.eos->gthm1 * rhohat * (eps - epsc);
    ahat = Phat / (rhohat * (1.0 + eps));
  }
  const double nuA = (1.0 + ahat) * (1.0 + eps) * a.iW;
  const double nuB = (1.0 + ahat) * (1.0 + a.qbar - mu * a.rbar2);
  return mu - 1.0 / (std::fmax(nuA, nuB) + mu * a.rbar2);
}
// auxiliary function for the upper bracket when r >= h0
inline double c2p_fa(const C2PState& s, double mu) {
  const double x = 1.0 / (1.0 + mu * s.bs2);
  const double rbar2 = s.r2 * x * x + mu * x * (1.0 + x) * s.rb2;
  return mu * std::sqrt(1.0 + rbar2) - 1.0;
}

// Illinois-modified regula falsi on [a,b], fa < 0 <= fb known.  which: 0 = f, 1 = fa.
// Returns false on NaN or more than max_iter evaluations.
inline bool illinois(const C2PState& s, int which, double a, double b, double fa, double fb,
                     int max_iter, double tol, double* root, int* nev) {
  int side = 0;
  double cprev = b;
  for (int it = 0; it < max_iter; ++it) {
    const double c = (a * fb - b * fa) / (fb - fa);
    const double fc = which ? c2p_fa(s, c) : c2p_f(s, c);
    ++*nev;
    if (!(fc == fc)) return false;
    if (fc == 0.0) { *root = c; return true; }
    if (fc > 0.0) {
      b = c; fb = fc;
      if (side == -1) fa = 0.5 * fa;
      side = -1;
    } else {
      a = c; fa = fc;
      if (side == 1) fb = 0.5 * fb;
      side = 1;
    }
    if (std::fabs(c - cprev) <= tol * c) { *root = c; return true; }
    cprev = c;
  }
  return false;
}
}  // namespace

extern "C" double orc_c2p_master(double gamma_ad, double q, double r2, double bs2, double rb2,
                                 double mu) {
  orc_params ideal{};
  ideal.gamma_ad = gamma_ad;
  const OrcEos e = orc_make_eos(&ideal);
  C2PState s{q, r2, bs2, rb2, r2 / (1.0 + r2), gamma_ad - 1.0, &e, 1.0};
  return c2p_f(s, mu);
}
extern "C" double orc_c2p_master_eos(const orc_params* p, double D, double q, double r2, double bs2,
                                     double rb2, double mu) {
  const OrcEos e = orc_make_eos(p);
  C2PState s{q, r2, bs2, rb2, r2 / (1.0 + r2), e.gm1, &e, D};
  return c2p_f(s, mu);
}

extern "C" int orc_con2prim_cell(const orc_params* p, const double g[6], double Ut[5],
                                 const double Btcc[3], double Wout[5], int check_only,
                                 int* iters) {
  int status = 0, nev = 0;
  const OrcEos eos = orc_make_eos(p);
  const double gm1 = eos.gm1;
  const double P_atm = eos_P_at_T(eos, p->rho_atm, p->T_atm);
  double det, sdet, gi[6];
  orc_metric_inverse(g, &det, &sdet, gi);
  const double isd = 1.0 / sdet;
  double D = Ut[0] * isd, tau = Ut[4] * isd;
  double Sl[3] = {Ut[1] * isd, Ut[2] * isd, Ut[3] * isd};
  const double B[3] = {Btcc[0] * isd, Btcc[1] * isd, Btcc[2] * isd};
  double rho = p->rho_atm, ux = 0.0, uy = 0.0, uz = 0.0, P = P_atm;  // atmosphere
  bool solve = true;

  // step 2: non-finite input -> failure, atmosphere
  if (!(fin(D) && fin(Sl[0]) && fin(Sl[1]) && fin(Sl[2]) && fin(tau) &&
        fin(B[0]) && fin(B[1]) && fin(B[2]))) {
    status |= ORC_FAIL;
    solve = false;
  }
  double Bl[3];
  lower(g, B, Bl);
  const double B2 = dot(Bl, B);
  // step 3: conserved floors, order D floor -> magnetisation cap -> tau floor
  bool atmo = false;  // D floor: static fluid at T_atm, no solve
  if (solve && D < p->f_thr * p->rho_atm) {
    status |= ORC_DFLOOR;
    D = p->rho_atm;
    atmo = true;
  }
  if (solve && B2 > p->mag_max * D) { D = B2 / p->mag_max; status |= ORC_MAGCAP; }
  if (solve && atmo) {
    rho = D; P = eos_P_at_T(eos, D, p->T_atm);   // u = 0
    solve = false;
  }
  if (solve) {
    const double tau_atm = D * eos_eps_at_T(eos, D, p->T_atm) + 0.5 * B2;
    if (tau < tau_atm) { tau = tau_atm; status |= ORC_TAUFLOOR; }
    // step 4
    const double iD = 1.0 / D;
    C2PState s;
    s.q = tau * iD;
    const double rl[3] = {Sl[0] * iD, Sl[1] * iD, Sl[2] * iD};
    const double ru[3] = {gi[0] * rl[0] + gi[1] * rl[1] + gi[2] * rl[2],
                          gi[1] * rl[0] + gi[3] * rl[1] + gi[4] * rl[2],
                          gi[2] * rl[0] + gi[4] * rl[1] + gi[5] * rl[2]};
    s.r2 = dot(rl, ru);
    s.bs2 = B2 * iD;
    const double rB = dot(rl, B);
    s.rb2 = rB * rB * iD;
    s.v0sq = s.r2 / (1.0 + s.r2);
    s.gm1 = gm1;
    s.eos = &eos;
    s.D = D;
    // step 5: bracket
    bool ok = true;
    double mu_hi = 1.0;
    if (!(s.r2 < 1.0)) {
      ok = illinois(s, 1, 0.0, 1.0, -1.0, c2p_fa(s, 1.0), p->c2p_max_iter, p->c2p_tol, &mu_hi,
                    &nev);
      mu_hi = mu_hi * (1.0 + 1e-14);
      if (mu_hi > 1.0) mu_hi = 1.0;
    }
    double mu = 0.0;
    if (ok) {
      const double f_hi = c2p_f(s, mu_hi);
      const double f_lo = c2p_f(s, 0.0);
      nev += 2;
      if (!(f_hi >= 0.0) || !(f_lo < 0.0)) ok = false;
      else if (f_hi == 0.0) mu = mu_hi;
      else ok = illinois(s, 0, 0.0, mu_hi, f_lo, f_hi, p->c2p_max_iter, p->c2p_tol, &mu, &nev);
    }
    if (!ok) {
      status |= ORC_FAIL;
    } else {
      // step 6: primitives at the root
      C2PAux a;
      c2p_aux(s, mu, a);
      rho = D * a.iW;
      P = eos_P(eos, rho, a.eps);
      const double c = mu * rB * iD;
      const double mx = mu * a.x;
      ux = a.What * (mx * (ru[0] + c * B[0]));
      uy = a.What * (mx * (ru[1] + c * B[1]));
      uz = a.What * (mx * (ru[2] + c * B[2]));
      if (!(fin(rho) && fin(P) && fin(ux) && fin(uy) && fin(uz))) {
        status |= ORC_FAIL;
        rho = p->rho_atm; ux = uy = uz = 0.0; P = P_atm;
      }
    }
  }
  // step 7: primitive floors
  if (rho < p->f_thr * p->rho_atm) {
    rho = p->rho_atm; ux = uy = uz = 0.0; P = P_atm;
    status |= ORC_RHOFLOOR;
  } else if (eos_T_floor(eos, rho, p->T_atm, P)) {
    status |= ORC_TFLOOR;
  }
  Wout[0] = rho; Wout[1] = ux; Wout[2] = uy; Wout[3] = uz; Wout[4] = P;
  // step 8: "A similar policy holds for the conserved variables"
  if (status != 0 && !check_only) {
    double c5[5];
    prim2cons_eos(eos, g, Wout, B, c5);
    for (int v = 0; v < 5; ++v) Ut[v] = sdet * c5[v];
  }
  if (iters) *iters = nev;
  return status;
}

// ---------------------------------------------------------------- O4 -------
// donor cell, PPM4 (Colella & Woodward 1984), WENO-Z (Borges et al. 2008).
extern "C" void orc_reconstruct(int kind, const double q[5], double* qm, double* qp) {
  const double qmm = q[0], qm1 = q[1], q0 = q[2], qp1 = q[3], qpp = q[4];
  if (kind == 0) { *qm = q0; *qp = q0; return; }
  if (kind == 1) {
    const double c12 = 1.0 / 12.0;
    double ql = (7.0 * (qm1 + q0) - (qmm + qp1)) * c12;   // interface i-1/2
    double qr = (7.0 * (q0 + qp1) - (qm1 + qpp)) * c12;   // interface i+1/2
    ql = std::fmax(std::fmin(ql, std::fmax(qm1, q0)), std::fmin(qm1, q0));
    qr = std::fmax(std::fmin(qr, std::fmax(q0, qp1)), std::fmin(q0, qp1));
    if ((qr - q0) * (q0 - ql) <= 0.0) {
      ql = q0; qr = q0;
    } else {
      const double dq = qr - ql;
      const double eta = 6.0 * (q0 - 0.5 * (ql + qr));
      if (dq * eta > dq * dq) ql = 3.0 * q0 - 2.0 * qr;
      else if (dq * eta < -(dq * dq)) qr = 3.0 * q0 - 2.0 * ql;
    }
    *qm = ql; *qp = qr;
    return;
  }
  if (kind == 3) {
    // PLM with the monotonized-central slope limiter ("a van Leer monotonized slope
    // limiter"; reading R27): slope = minmod(2 dl, 2 dr, (dl + dr)/2)
    const double dl = q0 - qm1, dr = qp1 - q0;
    double sl = 0.0;
    if (dl * dr > 0.0) {
      const double dc = 0.5 * (dl + dr);
      sl = std::copysign(std::fmin(std::fmin(2.0 * std::fabs(dl), 2.0 * std::fabs(dr)), std::fabs(dc)), dc);
    }
    *qm = q0 - 0.5 * sl;
    *qp = q0 + 0.5 * sl;
    return;
  }
  if (kind == 4) {
    // PPMX: PPM with the extremum-preserving limiter of Colella & Sekora (2008), C = 1.25
    // ("a newer variant with an extrema-preserving limiter"; reading R28).
    const double C2 = 1.25, c12 = 1.0 / 12.0;
    // (1) fourth-order interface values, limited where they leave the range of the two cells
    double ql = (7.0 * (qm1 + q0) - (qmm + qp1)) * c12;
    double qr = (7.0 * (q0 + qp1) - (qm1 + qpp)) * c12;
    const double dL = qmm - 2.0 * qm1 + q0, dC = qm1 - 2.0 * q0 + qp1, dR = q0 - 2.0 * qp1 + qpp;
    if ((ql - qm1) * (q0 - ql) < 0.0) {
      const double d2 = 3.0 * (qm1 - 2.0 * ql + q0);
      double lim = 0.0;
      if (d2 * dL > 0.0 && d2 * dC > 0.0) lim = std::copysign(std::fmin(std::fmin(C2 * std::fabs(dL), C2 * std::fabs(dC)), std::fabs(d2)), d2);
      ql = 0.5 * (qm1 + q0) - lim * (1.0 / 6.0);
    }
    if ((qr - q0) * (qp1 - qr) < 0.0) {
      const double d2 = 3.0 * (q0 - 2.0 * qr + qp1);
      double lim = 0.0;
      if (d2 * dC > 0.0 && d2 * dR > 0.0) lim = std::copysign(std::fmin(std::fmin(C2 * std::fabs(dC), C2 * std::fabs(dR)), std::fabs(d2)), d2);
      qr = 0.5 * (q0 + qp1) - lim * (1.0 / 6.0);
    }
    // (2) the parabola: at a local extremum scale both deviations by the ratio of limited to
    // actual second derivative; elsewhere the usual no-overshoot rule
    const double dm = ql - q0, dp = qr - q0;
    if (dp * dm >= 0.0 || (qp1 - q0) * (q0 - qm1) <= 0.0) {
      const double d2 = 6.0 * (ql + qr) - 12.0 * q0;
      double lim = 0.0;
      if (d2 * dL > 0.0 && d2 * dC > 0.0 && d2 * dR > 0.0)
        lim = std::copysign(std::fmin(std::fmin(C2 * std::fabs(dL), C2 * std::fabs(dR)), std::fmin(C2 * std::fabs(dC), std::fabs(d2))), d2);
      const double ratio = d2 != 0.0 ? lim / d2 : 0.0;
      ql = q0 + dm * ratio;
      qr = q0 + dp * ratio;
    } else {
      if (std::fabs(dp) >= 2.0 * std::fabs(dm)) qr = q0 - 2.0 * dm;
      else if (std::fabs(dm) >= 2.0 * std::fabs(dp)) ql = q0 - 2.0 * dp;
    }
    *qm = ql; *qp = qr;
    return;
  }
  // WENO-Z, p = 2, eps = 1e-40
  const double c6 = 1.0 / 6.0, c1312 = 13.0 / 12.0, eps = 1e-40;
  const double a0 = qmm - 2.0 * qm1 + q0, a1 = qm1 - 2.0 * q0 + qp1, a2 = q0 - 2.0 * qp1 + qpp;
  const double e0 = qmm - 4.0 * qm1 + 3.0 * q0, e1 = qm1 - qp1, e2 = 3.0 * q0 - 4.0 * qp1 + qpp;
  const double b0 = c1312 * (a0 * a0) + 0.25 * (e0 * e0) + eps;
  const double b1 = c1312 * (a1 * a1) + 0.25 * (e1 * e1) + eps;
  const double b2 = c1312 * (a2 * a2) + 0.25 * (e2 * e2) + eps;
  const double tau5 = std::fabs(b0 - b2);
  // tau5/(beta_k+eps) for k=0,1,2 through one reciprocal of the product
  const double ib = 1.0 / (b0 * b1 * b2);
  const double r0 = tau5 * (b1 * b2) * ib, r1 = tau5 * (b0 * b2) * ib, r2 = tau5 * (b0 * b1) * ib;
  const double t0 = 1.0 + r0 * r0, t1 = 1.0 + r1 * r1, t2 = 1.0 + r2 * r2;
  // right face of cell i
  {
    const double p0 = (2.0 * qmm - 7.0 * qm1 + 11.0 * q0) * c6;
    const double p1 = (-qm1 + 5.0 * q0 + 2.0 * qp1) * c6;
    const double p2 = (2.0 * q0 + 5.0 * qp1 - qpp) * c6;
    const double w0 = 0.1 * t0, w1 = 0.6 * t1, w2 = 0.3 * t2;
    *qp = (w0 * p0 + w1 * p1 + w2 * p2) / (w0 + w1 + w2);
  }
  // left face: mirror image i+m <-> i-m
  {
    const double p0 = (2.0 * qpp - 7.0 * qp1 + 11.0 * q0) * c6;
    const double p1 = (-qp1 + 5.0 * q0 + 2.0 * qm1) * c6;
    const double p2 = (2.0 * q0 + 5.0 * qm1 - qmm) * c6;
    const double w0 = 0.1 * t2, w1 = 0.6 * t1, w2 = 0.3 * t0;
    *qm = (w0 * p0 + w1 * p1 + w2 * p2) / (w0 + w1 + w2);
  }
}

// ---------------------------------------------------------------- O5/O6 ----
namespace {
struct Side { double U[7], F[7], lm, lp; };

// One side of the Riemann problem at a face of direction d (Eq. 8).
// prim = {rho,u^x,u^y,u^z,P}; Bt1,Bt2 densitised transverse B; Bd undensitised normal B.
inline void side_state(const OrcEos& eos, int d, const double g[6], double gdd, double sdet,
                       double isd, double alp, double ialp, const double bet[3],
                       const double prim[5], double Bt1t, double Bt2t, double Bd, Side& s) {
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  const double rho = prim[0], P = prim[4];
  const double u[3] = {prim[1], prim[2], prim[3]};
  double B[3];
  B[d] = Bd; B[t1] = Bt1t * isd; B[t2] = Bt2t * isd;
  double ul[3], Bl[3];
  lower(g, u, ul);
  const double usq = dot(ul, u);
  const double W = std::sqrt(1.0 + usq);
  const double iW = 1.0 / W;
  const double v[3] = {u[0] * iW, u[1] * iW, u[2] * iW};
  const double vl[3] = {ul[0] * iW, ul[1] * iW, ul[2] * iW};
  lower(g, B, Bl);
  const double B2 = dot(Bl, B);
  const double Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2];
  const double b2 = B2 * iW * iW + Bv * Bv;                       // Eq. 7
  const double bl[3] = {Bl[0] * iW + Bv * ul[0], Bl[1] * iW + Bv * ul[1],
                        Bl[2] * iW + Bv * ul[2]};
  const double ab0 = W * Bv;                                       // alpha b^0 (Eq. 7a)
  double hm1, cs2;
  eos_hm1_cs2(eos, rho, P, hm1, cs2);
  const double h = 1.0 + hm1;
  const double Ptot = P + 0.5 * b2;
  const double D = rho * W;
  const double wtot = rho * h * W * W + B2;
  const double S[3] = {wtot * vl[0] - Bv * Bl[0], wtot * vl[1] - Bv * Bl[1],
                       wtot * vl[2] - Bv * Bl[2]};
  const double tau = D * (hm1 * W + usq / (1.0 + W)) + B2 - P - 0.5 * (Bv * Bv + B2 * iW * iW);
  const double vh[3] = {v[0] - bet[0] * ialp, v[1] - bet[1] * ialp, v[2] - bet[2] * ialp};
  const double BdW = B[d] * iW;
  const double aP = alp * Ptot;
  s.U[0] = sdet * D;
  s.U[1] = sdet * S[0]; s.U[2] = sdet * S[1]; s.U[3] = sdet * S[2];
  s.U[4] = sdet * tau;
  s.U[5] = Bt1t; s.U[6] = Bt2t;
  s.F[0] = sdet * (alp * D * vh[d]);
  for (int i = 0; i < 3; ++i) {
    double f = alp * S[i] * vh[d] - alp * bl[i] * BdW;
    if (i == d) f = f + aP;
    s.F[1 + i] = sdet * f;
  }
  s.F[4] = sdet * (alp * tau * vh[d] - alp * ab0 * BdW + aP * v[d]);
  s.F[5] = sdet * (alp * (B[t1] * vh[d] - B[d] * vh[t1]));
  s.F[6] = sdet * (alp * (B[t2] * vh[d] - B[d] * vh[t2]));
  // signal speeds: fast-magnetosonic bound (DESIGN.md §3 O6)
  const double vsq = v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2];
  const double rhoh = rho * h;
  const double va2 = b2 / (rhoh + b2);
  const double a2 = cs2 + va2 - cs2 * va2;
  const double om = 1.0 - vsq * a2;
  const double disc = a2 * (1.0 - vsq) * (gdd * om - v[d] * v[d] * (1.0 - a2));
  const double root = std::sqrt(std::fmax(0.0, disc));
  const double iom = 1.0 / om;
  const double vd1 = v[d] * (1.0 - a2);
  s.lm = alp * ((vd1 - root) * iom) - bet[d];
  s.lp = alp * ((vd1 + root) * iom) - bet[d];
}

// face-state floor of P:139 ("after reconstruction")
inline void face_floor(const orc_params* p, const OrcEos& eos, double prim[5]) {
  if (prim[0] < p->f_thr * p->rho_atm) {
    prim[0] = p->rho_atm; prim[1] = 0.0; prim[2] = 0.0; prim[3] = 0.0;
    prim[4] = eos_P_at_T(eos, p->rho_atm, p->T_atm);
  } else {
    eos_T_floor(eos, prim[0], p->T_atm, prim[4]);
  }
}
}  // namespace

extern "C" void orc_face_flux(const orc_params* p, int dir, int riemann, const double gL[10],
                              const double gR[10], const double WL[7], const double WR[7],
                              double Bfd, int apply_floor, double F[7], double lam[4]) {
  // O5: every metric function at the face is the arithmetic mean of the two cells
  double m[10];
  for (int c = 0; c < 10; ++c) m[c] = (gL[c] + gR[c]) * 0.5;
  const double alp = m[0];
  const double bet[3] = {m[1], m[2], m[3]};
  const double* g = m + 4;
  double det, sdet, gi[6];
  orc_metric_inverse(g, &det, &sdet, gi);
  const double gdd = dir == 0 ? gi[0] : (dir == 1 ? gi[3] : gi[5]);
  const double isd = 1.0 / sdet;
  const double ialp = 1.0 / alp;
  const double Bd = Bfd * isd;
  double pl[5] = {WL[0], WL[1], WL[2], WL[3], WL[4]};
  double pr[5] = {WR[0], WR[1], WR[2], WR[3], WR[4]};
  const OrcEos eos = orc_make_eos(p);
  if (apply_floor) { face_floor(p, eos, pl); face_floor(p, eos, pr); }
  Side L, R;
  side_state(eos, dir, g, gdd, sdet, isd, alp, ialp, bet, pl, WL[5], WL[6], Bd, L);
  side_state(eos, dir, g, gdd, sdet, isd, alp, ialp, bet, pr, WR[5], WR[6], Bd, R);
  if (lam) { lam[0] = L.lm; lam[1] = L.lp; lam[2] = R.lm; lam[3] = R.lp; }
  if (riemann == 1) {  // HLLE
    const double lL = std::fmin(0.0, std::fmin(L.lm, R.lm));
    const double lR = std::fmax(0.0, std::fmax(L.lp, R.lp));
    const double dl = lR - lL;
    if (dl == 0.0) {
      for (int c = 0; c < 7; ++c) F[c] = 0.5 * (L.F[c] + R.F[c]);
    } else {
      const double idl = 1.0 / dl;
      const double lRL = lR * lL;
      for (int c = 0; c < 7; ++c)
        F[c] = (lR * L.F[c] - lL * R.F[c] + lRL * (R.U[c] - L.U[c])) * idl;
    }
  } else {  // LLF
    const double lam_max = std::fmax(std::fmax(std::fabs(L.lm), std::fabs(L.lp)),
                                     std::fmax(std::fabs(R.lm), std::fabs(R.lp)));
    for (int c = 0; c < 7; ++c)
      F[c] = 0.5 * (L.F[c] + R.F[c]) - 0.5 * lam_max * (R.U[c] - L.U[c]);
  }
}
