// ak_flux.cuh — reconstruction (O4), face geometry (O5) and Riemann fluxes (O6).
// DESIGN.md §3; PAPER.md P:133 (donor cell / PPM4 / WENO-Z, LLF / HLLE), Eq. 7-8,
// face-state floor P:139.  Device code only.  Same canonical expression trees as oracle/point.cpp,
// restated in another file (see ak_dev.cuh); nothing is included from or linked with oracle/.
#pragma once
#include "ak_dev.cuh"

namespace ak {

// ------------------------------------------------------------------ O4: reconstruction
// Five cell values qmm..qpp centred on cell i  ->  qm at its left face, qp at its right face.
// PLAIN: the two weighted means of WENO-Z by a plain division instead of ddiv() — the same quotient bit for bit
// (ddiv only sidesteps the division's slow path for a ZERO dividend); for fields that are never zero (rho, P in
// the light kernel) it saves the ~10 instructions of ddiv's test and selects per quotient.
template <int KIND, bool PLAIN = false>
__device__ __forceinline__ void recon(double qmm, double qm1, double q0, double qp1, double qpp,
                                      double& qm, double& qp) {
  if (KIND == 0) {            // donor cell
    qm = q0; qp = q0;
  } else if (KIND == 1) {     // PPM4 (Colella & Woodward 1984): 4th-order interface values,
                              // clamped, then the parabola monotonicity rule
    const double c12 = 1.0 / 12.0;
    double ql = (7.0 * (qm1 + q0) - (qmm + qp1)) * c12;
    double qr = (7.0 * (q0 + qp1) - (qm1 + qpp)) * c12;
    ql = fmax(fmin(ql, fmax(qm1, q0)), fmin(qm1, q0));
    qr = fmax(fmin(qr, fmax(q0, qp1)), fmin(q0, qp1));
    if ((qr - q0) * (q0 - ql) <= 0.0) {
      ql = q0; qr = q0;
    } else {
      const double dq = qr - ql;
      const double eta = 6.0 * (q0 - 0.5 * (ql + qr));
      if (dq * eta > dq * dq) ql = 3.0 * q0 - 2.0 * qr;
      else if (dq * eta < -(dq * dq)) qr = 3.0 * q0 - 2.0 * ql;
    }
    qm = ql; qp = qr;
  } else if (KIND == 3) {     // PLM, monotonized-central limiter: slope = minmod(2 dl, 2 dr, (dl + dr)/2)
    const double dl = q0 - qm1, dr = qp1 - q0;
    double sl = 0.0;
    if (dl * dr > 0.0) {
      const double dc = 0.5 * (dl + dr);
      sl = copysign(fmin(fmin(2.0 * fabs(dl), 2.0 * fabs(dr)), fabs(dc)), dc);
    }
    qm = q0 - 0.5 * sl;
    qp = q0 + 0.5 * sl;
  } else if (KIND == 4) {
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
      if (d2 * dL > 0.0 && d2 * dC > 0.0) lim = copysign(fmin(fmin(C2 * fabs(dL), C2 * fabs(dC)), fabs(d2)), d2);
      ql = 0.5 * (qm1 + q0) - lim * (1.0 / 6.0);
    }
    if ((qr - q0) * (qp1 - qr) < 0.0) {
      const double d2 = 3.0 * (q0 - 2.0 * qr + qp1);
      double lim = 0.0;
      if (d2 * dC > 0.0 && d2 * dR > 0.0) lim = copysign(fmin(fmin(C2 * fabs(dC), C2 * fabs(dR)), fabs(d2)), d2);
      qr = 0.5 * (q0 + qp1) - lim * (1.0 / 6.0);
    }
    // (2) the parabola: at a local extremum scale both deviations by the ratio of limited to
    // actual second derivative; elsewhere the usual no-overshoot rule
    const double dm = ql - q0, dp = qr - q0;
    if (dp * dm >= 0.0 || (qp1 - q0) * (q0 - qm1) <= 0.0) {
      const double d2 = 6.0 * (ql + qr) - 12.0 * q0;
      double lim = 0.0;
      if (d2 * dL > 0.0 && d2 * dC > 0.0 && d2 * dR > 0.0)
        lim = copysign(fmin(fmin(C2 * fabs(dL), C2 * fabs(dR)), fmin(C2 * fabs(dC), fabs(d2))), d2);
      const double ratio = d2 != 0.0 ? lim / d2 : 0.0;
      ql = q0 + dm * ratio;
      qr = q0 + dp * ratio;
    } else {
      if (fabs(dp) >= 2.0 * fabs(dm)) qr = q0 - 2.0 * dm;
      else if (fabs(dm) >= 2.0 * fabs(dp)) ql = q0 - 2.0 * dp;
    }
    qm = ql; qp = qr;
  } else {                    // WENO-Z (Borges et al. 2008), p = 2, eps = 1e-40
    const double c6 = 1.0 / 6.0, c1312 = 13.0 / 12.0, eps = 1e-40;
    const double a0 = qmm - 2.0 * qm1 + q0, a1 = qm1 - 2.0 * q0 + qp1, a2 = q0 - 2.0 * qp1 + qpp;
    const double e0 = qmm - 4.0 * qm1 + 3.0 * q0, e1 = qm1 - qp1, e2 = 3.0 * q0 - 4.0 * qp1 + qpp;
    const double b0 = c1312 * (a0 * a0) + 0.25 * (e0 * e0) + eps;
    const double b1 = c1312 * (a1 * a1) + 0.25 * (e1 * e1) + eps;
    const double b2 = c1312 * (a2 * a2) + 0.25 * (e2 * e2) + eps;
    const double tau5 = fabs(b0 - b2);
    // the three ratios tau5/beta_k through one reciprocal of the product
    const double ib = 1.0 / (b0 * b1 * b2);
    const double r0 = tau5 * (b1 * b2) * ib, r1 = tau5 * (b0 * b2) * ib, r2 = tau5 * (b0 * b1) * ib;
    const double t0 = 1.0 + r0 * r0, t1 = 1.0 + r1 * r1, t2 = 1.0 + r2 * r2;
    {
      const double p0 = (2.0 * qmm - 7.0 * qm1 + 11.0 * q0) * c6;
      const double p1 = (-qm1 + 5.0 * q0 + 2.0 * qp1) * c6;
      const double p2 = (2.0 * q0 + 5.0 * qp1 - qpp) * c6;
      const double w0 = 0.1 * t0, w1 = 0.6 * t1, w2 = 0.3 * t2;
      qp = PLAIN ? (w0 * p0 + w1 * p1 + w2 * p2) / (w0 + w1 + w2) : ddiv(w0 * p0 + w1 * p1 + w2 * p2, w0 + w1 + w2);
    }
    {  // mirror image
      const double p0 = (2.0 * qpp - 7.0 * qp1 + 11.0 * q0) * c6;
      const double p1 = (-qp1 + 5.0 * q0 + 2.0 * qm1) * c6;
      const double p2 = (2.0 * q0 + 5.0 * qm1 - qmm) * c6;
      const double w0 = 0.1 * t2, w1 = 0.6 * t1, w2 = 0.3 * t0;
      qm = PLAIN ? (w0 * p0 + w1 * p1 + w2 * p2) / (w0 + w1 + w2) : ddiv(w0 * p0 + w1 * p1 + w2 * p2, w0 + w1 + w2);
    }
  }
}

// ------------------------------------------------------------------ O5: face geometry
struct FaceGeo {
  double alp, ialp, bet[3];
  Met3 g;
  double gdd, sdet, isd;
};

// mL, mR = {alp, betx, bety, betz, gxx, gxy, gxz, gyy, gyz, gzz} of the lower / upper cell
template <int DIR>
__device__ __forceinline__ void face_geometry(const double mL[10], const double mR[10], FaceGeo& G) {
  double m[10];
#pragma unroll
  for (int c = 0; c < 10; ++c) m[c] = (mL[c] + mR[c]) * 0.5;
  G.alp = m[0];
  G.bet[0] = m[1]; G.bet[1] = m[2]; G.bet[2] = m[3];
  G.g.xx = m[4]; G.g.xy = m[5]; G.g.xz = m[6]; G.g.yy = m[7]; G.g.yz = m[8]; G.g.zz = m[9];
  metric_det_gdd<DIR>(G.g, G.sdet, G.gdd);
  G.isd = 1.0 / G.sdet;
  G.ialp = 1.0 / G.alp;
}

// face-state floor ("after reconstruction"); s = rho,ux,uy,uz,P,...
template <int EOS = 0>
__device__ __forceinline__ void face_floor(const Par& P, double s[7]) {
  if (s[0] < P.thr) {
    s[0] = P.rho_atm; s[1] = 0.0; s[2] = 0.0; s[3] = 0.0;
    s[4] = P.P_atm;
  } else if (EOS == 0) {
    if (s[4] < s[0] * P.T_atm) s[4] = s[0] * P.T_atm;
  } else {
    eos_T_floor<EOS>(P, s[0], s[4]);
  }
}

// ------------------------------------------------------------------ O6: one side (Eq. 8)
// s = rho,u^x,u^y,u^z,P,B~t1,B~t2 (transverse B densitised); Bd = undensitised normal B.
// Out: densitised conserved U[7], densitised fluxes F[7], signal speeds lm, lp.
// NOB (exact shortcut, mask bit 2): every B component of this state is +0.0 exactly (the caller's tile test).
// Then, operation by operation (finite metric, alpha > 0, positive diagonal, rho, P > 0 after the face floor):
//   B_i = B^2 = +0; (Bv) = 0 vl_x + 0 vl_y + 0 vl_z = +-0 (kept: its sign is inherited below);
//   b^2 = +0 + (+-0)^2 = +0; b_i = +0 + (+-0) u_i = +0; alpha b^0 = W (+-0) = (Bv); Ptot = P + 0 = P;
//   wtot = rho h W^2 + 0; S_i = wtot v_i - (Bv)(+0) = wtot v_i - (Bv) (the product is (Bv) itself);
//   tau = X + 0 - P - 0.5 (+0 + +0) = X - P (X >= +0); B^d / W = +0; alpha b_i B^d / W = +0 and A - +0 = A;
//   alpha (alpha b^0) B^d / W = (Bv); v_A^2 = ddiv(+0, rho h) = +0; a^2 = c_s^2 + 0 - c_s^2 0 = c_s^2.
// What is dropped is ~90 fp64 instructions per side, among them the Alfven division.
template <int DIR, int EOS = 0, bool NOB = false>
__device__ __forceinline__ void side_state(const Par& P, const FaceGeo& G, const double s[7], double Bd,
                                           double U[7], double F[7], double& lm, double& lp) {
  constexpr int t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  const double rho = s[0], pr = s[4];
  const double u[3] = {s[1], s[2], s[3]};
  if (NOB) {
    double ul[3];
    lower(G.g, u, ul);
    const double usq = dot3(ul, u);
    const double W = sqrt(1.0 + usq);
    const double iW = 1.0 / W;
    const double v[3] = {u[0] * iW, u[1] * iW, u[2] * iW};
    const double vl[3] = {ul[0] * iW, ul[1] * iW, ul[2] * iW};
    const double Bv = 0.0 * vl[0] + 0.0 * vl[1] + 0.0 * vl[2];
    double hm1, cs2;
    eos_hm1_cs2<EOS>(P, rho, pr, hm1, cs2);
    const double h = 1.0 + hm1;
    const double D = rho * W;
    const double wtot = rho * h * W * W;
    const double S[3] = {wtot * vl[0] - Bv, wtot * vl[1] - Bv, wtot * vl[2] - Bv};
    const double tau = D * (hm1 * W + ddiv(usq, 1.0 + W)) - pr;
    const double vh[3] = {v[0] - G.bet[0] * G.ialp, v[1] - G.bet[1] * G.ialp, v[2] - G.bet[2] * G.ialp};
    const double aP = G.alp * pr;
    U[0] = G.sdet * D;
    U[1] = G.sdet * S[0]; U[2] = G.sdet * S[1]; U[3] = G.sdet * S[2];
    U[4] = G.sdet * tau;
    U[5] = s[5]; U[6] = s[6];
    F[0] = G.sdet * (G.alp * D * vh[DIR]);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      double f = G.alp * S[i] * vh[DIR];
      if (i == DIR) f = f + aP;
      F[1 + i] = G.sdet * f;
    }
    F[4] = G.sdet * (G.alp * tau * vh[DIR] - Bv + aP * v[DIR]);
    const double zd = 0.0 * vh[DIR];
    F[5] = G.sdet * (G.alp * (zd - 0.0 * vh[t1]));
    F[6] = G.sdet * (G.alp * (zd - 0.0 * vh[t2]));
    const double vsq = v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2];
    const double a2 = cs2;
    const double om = 1.0 - vsq * a2;
    const double disc = a2 * (1.0 - vsq) * (G.gdd * om - v[DIR] * v[DIR] * (1.0 - a2));
    const double root = sqrt(fmax(0.0, disc));
    const double iom = 1.0 / om;
    const double vd1 = v[DIR] * (1.0 - a2);
    lm = G.alp * ((vd1 - root) * iom) - G.bet[DIR];
    lp = G.alp * ((vd1 + root) * iom) - G.bet[DIR];
    return;
  }
  double B[3];
  B[DIR] = Bd; B[t1] = s[5] * G.isd; B[t2] = s[6] * G.isd;
  double ul[3], Bl[3];
  lower(G.g, u, ul);
  const double usq = dot3(ul, u);
  const double W = sqrt(1.0 + usq);
  const double iW = 1.0 / W;
  const double v[3] = {u[0] * iW, u[1] * iW, u[2] * iW};
  const double vl[3] = {ul[0] * iW, ul[1] * iW, ul[2] * iW};
  lower(G.g, B, Bl);
  const double B2 = dot3(Bl, B);
  const double Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2];
  const double b2 = B2 * iW * iW + Bv * Bv;                                   // Eq. 7
  const double bl[3] = {Bl[0] * iW + Bv * ul[0], Bl[1] * iW + Bv * ul[1], Bl[2] * iW + Bv * ul[2]};
  const double ab0 = W * Bv;                                                  // alpha b^0
  double hm1, cs2;
  eos_hm1_cs2<EOS>(P, rho, pr, hm1, cs2);
  const double h = 1.0 + hm1;
  const double Ptot = pr + 0.5 * b2;
  const double D = rho * W;
  const double wtot = rho * h * W * W + B2;
  const double S[3] = {wtot * vl[0] - Bv * Bl[0], wtot * vl[1] - Bv * Bl[1], wtot * vl[2] - Bv * Bl[2]};
  const double tau = D * (hm1 * W + ddiv(usq, 1.0 + W)) + B2 - pr - 0.5 * (Bv * Bv + B2 * iW * iW);
  const double vh[3] = {v[0] - G.bet[0] * G.ialp, v[1] - G.bet[1] * G.ialp, v[2] - G.bet[2] * G.ialp};
  const double BdW = B[DIR] * iW;
  const double aP = G.alp * Ptot;
  U[0] = G.sdet * D;
  U[1] = G.sdet * S[0]; U[2] = G.sdet * S[1]; U[3] = G.sdet * S[2];
  U[4] = G.sdet * tau;
  U[5] = s[5]; U[6] = s[6];
  F[0] = G.sdet * (G.alp * D * vh[DIR]);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double f = G.alp * S[i] * vh[DIR] - G.alp * bl[i] * BdW;
    if (i == DIR) f = f + aP;
    F[1 + i] = G.sdet * f;
  }
  F[4] = G.sdet * (G.alp * tau * vh[DIR] - G.alp * ab0 * BdW + aP * v[DIR]);
  F[5] = G.sdet * (G.alp * (B[t1] * vh[DIR] - B[DIR] * vh[t1]));
  F[6] = G.sdet * (G.alp * (B[t2] * vh[DIR] - B[DIR] * vh[t2]));
  // fast-magnetosonic bound on the characteristic speeds (DESIGN.md §3 O6, reading R18)
  const double vsq = v[0] * vl[0] + v[1] * vl[1] + v[2] * vl[2];
  const double rhoh = rho * h;
  const double va2 = ddiv(b2, rhoh + b2);
  const double a2 = cs2 + va2 - cs2 * va2;
  const double om = 1.0 - vsq * a2;
  const double disc = a2 * (1.0 - vsq) * (G.gdd * om - v[DIR] * v[DIR] * (1.0 - a2));
  const double root = sqrt(fmax(0.0, disc));
  const double iom = 1.0 / om;
  const double vd1 = v[DIR] * (1.0 - a2);
  lm = G.alp * ((vd1 - root) * iom) - G.bet[DIR];
  lp = G.alp * ((vd1 + root) * iom) - G.bet[DIR];
}

// Face flux from left/right states (floored here when FLOOR), the face-normal B~ and the
// two adjacent cells' metric.  RS: 0 LLF, 1 HLLE.
template <int DIR, bool FLOOR, int EOS = 0>
__device__ __forceinline__ void face_flux(const Par& P, int rs, const double mL[10], const double mR[10],
                                          double sL[7], double sR[7], double Bfd, double Fo[7]) {
  FaceGeo G;
  face_geometry<DIR>(mL, mR, G);
  const double Bd = Bfd * G.isd;
  if (FLOOR) { face_floor<EOS>(P, sL); face_floor<EOS>(P, sR); }
  double UL[7], FL[7], UR[7], FR[7], lmL, lpL, lmR, lpR;
  side_state<DIR, EOS>(P, G, sL, Bd, UL, FL, lmL, lpL);
  side_state<DIR, EOS>(P, G, sR, Bd, UR, FR, lmR, lpR);
  if (rs == 1) {   // HLLE
    const double lL = fmin(0.0, fmin(lmL, lmR));
    const double lR = fmax(0.0, fmax(lpL, lpR));
    const double dl = lR - lL;
    if (dl == 0.0) {
#pragma unroll
      for (int c = 0; c < 7; ++c) Fo[c] = 0.5 * (FL[c] + FR[c]);
    } else {
      const double idl = 1.0 / dl;
      const double lRL = lR * lL;
#pragma unroll
      for (int c = 0; c < 7; ++c) Fo[c] = (lR * FL[c] - lL * FR[c] + lRL * (UR[c] - UL[c])) * idl;
    }
  } else {         // LLF
    const double lam = fmax(fmax(fabs(lmL), fabs(lpL)), fmax(fabs(lmR), fabs(lpR)));
#pragma unroll
    for (int c = 0; c < 7; ++c) Fo[c] = 0.5 * (FL[c] + FR[c]) - 0.5 * lam * (UR[c] - UL[c]);
  }
}

// The same face flux with the long-lived intermediates parked in shared memory instead of spilled to
// local memory (which is written through to L2): the right state waits there (pkR, put there by the
// caller, unfloored) while the left side is evaluated, the left side's U and F (pk, [14][stride]) while
// the right side is.  Columns no other thread touches.  Same operations as face_flux<DIR, true>.
template <int DIR, int EOS = 0, bool NOB = false>
__device__ __forceinline__ void face_flux_parked(const Par& P, int rs, const FaceGeo& G, double sL[7],
                                                 double* parkR, int strideR, double Bfd, double Fo[7],
                                                 double* park, int stride) {
  volatile double* pk = park;
  volatile double* pkR = parkR;
  const double Bd = Bfd * G.isd;
  face_floor<EOS>(P, sL);
  double UR[7], FR[7], lmL, lpL, lmR, lpR;
  {
    double UL[7], FL[7];
    side_state<DIR, EOS, NOB>(P, G, sL, Bd, UL, FL, lmL, lpL);
#pragma unroll
    for (int c = 0; c < 7; ++c) { pk[c * stride] = UL[c]; pk[(7 + c) * stride] = FL[c]; }
  }
  {
    double sRq[7];
#pragma unroll
    for (int v = 0; v < 7; ++v) sRq[v] = pkR[v * strideR];
    face_floor<EOS>(P, sRq);
    side_state<DIR, EOS, NOB>(P, G, sRq, Bd, UR, FR, lmR, lpR);
  }
  if (rs == 1) {   // HLLE
    const double lL = fmin(0.0, fmin(lmL, lmR));
    const double lR = fmax(0.0, fmax(lpL, lpR));
    const double dl = lR - lL;
    if (dl == 0.0) {
#pragma unroll
      for (int c = 0; c < 7; ++c) Fo[c] = 0.5 * (pk[(7 + c) * stride] + FR[c]);
    } else {
      const double idl = 1.0 / dl;
      const double lRL = lR * lL;
#pragma unroll
      for (int c = 0; c < 7; ++c) {
        const double ULc = pk[c * stride], FLc = pk[(7 + c) * stride];
        Fo[c] = (lR * FLc - lL * FR[c] + lRL * (UR[c] - ULc)) * idl;
      }
    }
  } else {         // LLF
    const double lam = fmax(fmax(fabs(lmL), fabs(lpL)), fmax(fabs(lmR), fabs(lpR)));
#pragma unroll
    for (int c = 0; c < 7; ++c) {
      const double ULc = pk[c * stride], FLc = pk[(7 + c) * stride];
      Fo[c] = 0.5 * (FLc + FR[c]) - 0.5 * lam * (UR[c] - ULc);
    }
  }
}

// ------------------------------------------------------------------ O6 for a static unmagnetised face
// The face flux when BOTH states have u^i = +0.0 and every B component is +0.0 exactly (static atmosphere
// without field: most of a merger grid) — exact shortcut, mask bit 2 of ak_set_exact_shortcuts.  Derived from
// side_state() operation by operation, dropping only operations whose result is then known exactly, for a
// finite metric with gamma_xx, gamma_zz... > 0:
//   u_i = g_ij 0 = +0 (a sum that contains the +0 of a positive diagonal term is +0), usq = +0, W = sqrt(1) = 1,
//   1/W = 1, v^i = v_i = +0, B_i = B^2 = (Bv) = b^2 = b_i = alpha b^0 = +0, Ptot = P + 0 = P, D = rho 1 = rho,
//   wtot = rho h, S_i = +0 - +0 = +0, tau = rho (hm1 + ddiv(+0, 2)) + 0 - P - 0 = rho hm1 - P,
//   vhat^i = +0 - beta^i / alpha (the subtraction is kept: it fixes the sign of a zero shift),
//   v_A^2 = ddiv(+0, rho h) = +0, a^2 = c_s^2, 1 - v^2 a^2 = 1, disc = a^2 gamma^dd, vd1 = +0.
// Products with a zero whose SIGN the result inherits (0 * vhat) are kept, so signed zeros come out as in the
// full evaluation.  The HLLE / LLF combination is the one of face_flux(), unchanged.
template <int DIR, int EOS = 0>
__device__ __forceinline__ void static_side(const Par& P, const FaceGeo& G, const double vh[3], double rho, double pr,
                                            double U[7], double F[7], double& lm, double& lp) {
  constexpr int t1 = (DIR + 1) % 3;
  double hm1, cs2;
  eos_hm1_cs2<EOS>(P, rho, pr, hm1, cs2);
  const double h = 1.0 + hm1;
  const double tau = rho * hm1 - pr;
  const double aP = G.alp * pr;
  U[0] = G.sdet * rho;
  U[1] = G.sdet * 0.0; U[2] = U[1]; U[3] = U[1];
  U[4] = G.sdet * tau;
  U[5] = 0.0; U[6] = 0.0;
  F[0] = G.sdet * (G.alp * rho * vh[DIR]);
  const double zS = (G.alp * 0.0) * vh[DIR] - 0.0;            // alpha S_i vhat^d - alpha b_i B^d / W with S_i = b_i = +0
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    double f = zS;
    if (i == DIR) f = f + aP;
    F[1 + i] = G.sdet * f;
  }
  F[4] = G.sdet * (G.alp * tau * vh[DIR] - 0.0 + aP * 0.0);
  const double zd = 0.0 * vh[DIR];
  F[5] = G.sdet * (G.alp * (zd - 0.0 * vh[t1]));
  F[6] = G.sdet * (G.alp * (zd - 0.0 * vh[(DIR + 2) % 3]));
  const double rhoh = rho * h;
  (void)rhoh;                                                  // v_A^2 = +0 whatever rho h > 0 is
  const double a2 = cs2;
  const double disc = a2 * G.gdd;
  const double root = sqrt(fmax(0.0, disc));
  const double vd1 = 0.0 * (1.0 - a2);
  lm = G.alp * (vd1 - root) - G.bet[DIR];
  lp = G.alp * (vd1 + root) - G.bet[DIR];
}

// sL, sR: rho at [0], P at [4] (floored here); everything else is +0.0 by the caller's test.
template <int DIR, int EOS = 0>
__device__ __forceinline__ void face_flux_static(const Par& P, int rs, const FaceGeo& G, double sL[7], double sR[7],
                                                 double Fo[7]) {
  face_floor<EOS>(P, sL);
  face_floor<EOS>(P, sR);
  const double vh[3] = {0.0 - G.bet[0] * G.ialp, 0.0 - G.bet[1] * G.ialp, 0.0 - G.bet[2] * G.ialp};
  double UL[7], FL[7], UR[7], FR[7], lmL, lpL, lmR, lpR;
  static_side<DIR, EOS>(P, G, vh, sL[0], sL[4], UL, FL, lmL, lpL);
  static_side<DIR, EOS>(P, G, vh, sR[0], sR[4], UR, FR, lmR, lpR);
  if (rs == 1) {   // HLLE
    const double lL = fmin(0.0, fmin(lmL, lmR));
    const double lR = fmax(0.0, fmax(lpL, lpR));
    const double dl = lR - lL;
    if (dl == 0.0) {
#pragma unroll
      for (int c = 0; c < 7; ++c) Fo[c] = 0.5 * (FL[c] + FR[c]);
    } else {
      const double idl = 1.0 / dl;
      const double lRL = lR * lL;
#pragma unroll
      for (int c = 0; c < 7; ++c) Fo[c] = (lR * FL[c] - lL * FR[c] + lRL * (UR[c] - UL[c])) * idl;
    }
  } else {         // LLF
    const double lam = fmax(fmax(fabs(lmL), fabs(lpL)), fmax(fabs(lmR), fabs(lpR)));
#pragma unroll
    for (int c = 0; c < 7; ++c) Fo[c] = 0.5 * (FL[c] + FR[c]) - 0.5 * lam * (UR[c] - UL[c]);
  }
}

}  // namespace ak
