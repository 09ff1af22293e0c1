// ak_dev.cuh — device-side point operators of the GRMHD RHS stage (sm_100a, fp64).
//
// Written from DESIGN.md §3 (steps O0..O6, restating PAPER.md Eqs. 6-9; P:133;
// P:137-139).  No file, header or table is shared with oracle/, but the point operators
// here evaluate the SAME canonical expression trees as oracle/point.cpp, restated (that is what makes
// the masks bit-reproducible): GPU == oracle therefore certifies indexing, tiling, staging and
// compaction, and the physics rests on the oracle's pins.  The library is compiled with
// --fmad=false: every +,-,*,/ and sqrt below is one IEEE fp64 operation evaluated in the
// order written (C++ left-to-right association), which is what makes the status/flag masks
// reproducible bit for bit (DESIGN.md §3 "reference arithmetic").
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <math_constants.h>

namespace ak {

// Stores of data that no later kernel of the stage finds in L2 anyway (the batch is two hundred times the L2):
// st.global.cs (evict-first) keeps the lines that ARE re-read — halo rows of neighbouring tiles — resident longer.
// AK_STREAM_ST bits: 1 light sweep kernel, 2 general sweep kernels, 4 con2prim, 8 div+sources.  Measured on C4
// (same-box A/B, stage): 0: 12.25-12.32 ms, 1: 12.24, 3: 12.23, 12: 12.22, 15: 12.19.
#ifndef AK_STREAM_ST
#define AK_STREAM_ST 15
#endif
template <int BIT>
__device__ __forceinline__ void st_out(double* p, double v) {
  if (AK_STREAM_ST & BIT) __stcs(p, v); else *p = v;
}


// ------------------------------------------------------------------ parameters / fields
struct Par {
  int nmb, n, nt, px, is, ie;   // is = 4, ie = n + 3
  double Gam, gm1, gm1r;        // Gamma, Gamma-1, Gamma/(Gamma-1)
  double rho_atm, T_atm, P_atm, eps_atm, thr;   // thr = f_thr * rho_atm
  double mag_max;
  double dmp_M, dmp_iM;
  int max_iter;
  double tol;
  int recon, riemann, fofc, fofc_riemann;
  int shortcuts;                // exact data-dependent shortcuts (ak_set_exact_shortcuts): bit 0 reconstruction of
                                // all-zero fields, bit 1 root solve of static unmagnetised cells; same bits out
  // piecewise-polytropic hybrid EOS (ak_set_eos_hybrid; reading R29); eos = 0: ideal gas
  int eos, nseg;
  double ppK[4], ppG[4], ppa[4], pprb[3];   // K_i, Gamma_i, eps offsets a_i, breakpoints
  double gth, gthm1;                        // Gamma_th, Gamma_th - 1
};

// All field pointers one stage touches (passed by value as a kernel parameter).
struct Fields {
  double* U[5];
  const double* Bf[3];
  const double* adm[16];        // gxx gxy gxz gyy gyz gzz alp bx by bz Kxx..Kzz
  double* W[8];                 // rho ux uy uz P Bccx Bccy Bccz
  double* F[21];                // face fluxes [dir][7]
  double* Ecc[3];               // cell-centred EMFs (scratch)
  double* dU[5];
  double* E[3];
  unsigned char* flag;
  unsigned char* status;
  const double* dx;             // [nmb][3] device copy
  unsigned int* list;           // FOFC: compacted flagged cells
  unsigned int* count;          // [0..2] faces redone per direction, [3] length of list
  unsigned long long* stats;    // device counters (see ak_api.cu)
  const double* U0[5];          // FOFC estimate of a later RK stage: U* = fa U0 + fb (U - dt div F);
  double fa, fb;                // U0[0] == nullptr: U* = U - dt div F (R9)
  double* M[10];                // matter terms E, S_i, S_ij written by K6 on interior cells (M[0] == nullptr: none)
  unsigned int* zflags;         // [nmb] bit q set: primitive field W[q] (q = 1..3 u^i, 5..7 B~cc^i) of that block holds
                                // a value that is not +0.0 (written by k_con2prim, conservative); bits 8..10: a face
                                // value of B~f^x,y,z of that block is not +0.0; nullptr: unknown
  unsigned char* rowflag;       // [nmb][nt][nt] 1: row (m, k, j) holds a u^i or a face B~ that is not +0.0 (written by
                                // k_con2prim, cleared before it); nullptr: not wanted
  const unsigned int* tlist;    // sweeps over TILE lists (k_split_tiles): list 2 d + w of direction d (w = 0 static
  const unsigned int* tcount;   // tiles, 1 the others) starts at tlist + (2 d + w) tcap and holds tcount[2 d + w] tile
  unsigned int tcap;            // numbers (m e + o') tiles + td; nullptr: every tile, in order
};

enum { ST_DFLOOR = 1, ST_TAUFLOOR = 2, ST_MAGCAP = 4, ST_RHOFLOOR = 8, ST_TFLOOR = 16,
       ST_FAIL = 32, ST_DMP = 64 };

// ------------------------------------------------------------------ O0: 3-metric algebra
struct Met3 {
  double xx, xy, xz, yy, yz, zz;
};

// determinant by cofactors of the first row; inverse = cofactor * (1/det)
__device__ __forceinline__ void metric_inverse(const Met3& g, double& det, double& sdet, Met3& u) {
  const double cxx = g.yy * g.zz - g.yz * g.yz;
  const double cxy = g.xz * g.yz - g.xy * g.zz;
  const double cxz = g.xy * g.yz - g.xz * g.yy;
  det = g.xx * cxx + g.xy * cxy + g.xz * cxz;
  const double id = 1.0 / det;
  u.xx = cxx * id;
  u.xy = cxy * id;
  u.xz = cxz * id;
  u.yy = (g.xx * g.zz - g.xz * g.xz) * id;
  u.yz = (g.xy * g.xz - g.xx * g.yz) * id;
  u.zz = (g.xx * g.yy - g.xy * g.xy) * id;
  sdet = sqrt(det);
}
// determinant and its square root only: the same operations as in metric_inverse
__device__ __forceinline__ void metric_det(const Met3& g, double& det, double& sdet) {
  const double cxx = g.yy * g.zz - g.yz * g.yz;
  const double cxy = g.xz * g.yz - g.xy * g.zz;
  const double cxz = g.xy * g.yz - g.xz * g.yy;
  det = g.xx * cxx + g.xy * cxy + g.xz * cxz;
  sdet = sqrt(det);
}
// determinant and one diagonal element of the inverse only (face geometry, O5)
template <int DIR>
__device__ __forceinline__ void metric_det_gdd(const Met3& g, double& sdet, double& gdd) {
  const double cxx = g.yy * g.zz - g.yz * g.yz;
  const double cxy = g.xz * g.yz - g.xy * g.zz;
  const double cxz = g.xy * g.yz - g.xz * g.yy;
  const double det = g.xx * cxx + g.xy * cxy + g.xz * cxz;
  const double id = 1.0 / det;
  if (DIR == 0) gdd = cxx * id;
  else if (DIR == 1) gdd = (g.xx * g.zz - g.xz * g.xz) * id;
  else gdd = (g.xx * g.yy - g.xy * g.xy) * id;
  sdet = sqrt(det);
}

// a_i = g_ij a^j, accumulated left to right
__device__ __forceinline__ void lower(const Met3& g, const double a[3], double o[3]) {
  o[0] = g.xx * a[0] + g.xy * a[1] + g.xz * a[2];
  o[1] = g.xy * a[0] + g.yy * a[1] + g.yz * a[2];
  o[2] = g.xz * a[0] + g.yz * a[1] + g.zz * a[2];
}
__device__ __forceinline__ double dot3(const double a[3], const double b[3]) {
  return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}

// IEEE a / b.  The division sequence nvcc emits takes a ~75-instruction slow path whenever the
// dividend is zero (or subnormal); exact zeros are the common case here (static atmosphere:
// u^i = 0, B = 0), and one lane is enough to send the whole warp there (ncu: 25 % of all
// instructions of the flux sweep).  A zero dividend over a finite non-zero divisor is a signed
// zero, produced here without dividing; every other case is the plain division, bit for bit.
__device__ __forceinline__ double ddiv(double a, double b) {
  const bool z = (a == 0.0) && (fabs(b) > 0.0) && (fabs(b) < CUDART_INF);
  // the substitution goes through an opaque select: written in C++ the compiler proves the
  // quotient unused when z holds and divides the raw (zero) dividend again
  double an;
  asm("{\n.reg .pred p;\nsetp.ne.s32 p, %2, 0;\nselp.f64 %0, 0d3FF0000000000000, %1, p;\n}" : "=d"(an) : "d"(a), "r"((int)z));
  const double q = an / b;
  return z ? (b > 0.0 ? a : -a) : q;
}

// ------------------------------------------------------------------ O1: equation of state
// EOS = 0: ideal gas, P = (Gamma-1) rho eps, T = P/rho, h - 1 = Gamma/(Gamma-1) T, c_s^2 = Gamma T / h.
// EOS = 1: piecewise-polytropic hybrid (R29): cold curve P_c = K_i rho^Gamma_i,
//   eps_c = a_i + P_c / ((Gamma_i - 1) rho) in the segment that holds rho; thermal part
//   P - P_c = (Gamma_th - 1) rho (eps - eps_c); T = (P - P_c)/rho; h = 1 + eps + P/rho;
//   c_s^2 = (Gamma_i P_c + Gamma_th (P - P_c)) / (rho h).
__device__ __forceinline__ void eos_cold(const Par& P, double rho, double& Pc, double& epsc, double& Gi) {
  int i = 0;
  while (i + 1 < P.nseg && rho >= P.pprb[i]) ++i;
  Gi = P.ppG[i];
  Pc = P.ppK[i] * pow(rho, Gi);
  epsc = P.ppa[i] + Pc / ((Gi - 1.0) * rho);
}
template <int EOS>
__device__ __forceinline__ void eos_hm1_cs2(const Par& P, double rho, double pr, double& hm1, double& cs2) {
  if (EOS == 0) {
    const double T = pr / rho;
    hm1 = P.gm1r * T;
    const double h = 1.0 + hm1;
    cs2 = P.Gam * T / h;
  } else {
    double Pc, epsc, Gi;
    eos_cold(P, rho, Pc, epsc, Gi);
    const double Pth = pr - Pc;
    const double eps = epsc + Pth / (P.gthm1 * rho);
    hm1 = eps + pr / rho;
    const double h = 1.0 + hm1;
    cs2 = (Gi * Pc + P.gth * Pth) / (rho * h);
  }
}
template <int EOS>
__device__ __forceinline__ double eos_hm1(const Par& P, double rho, double pr) {
  if (EOS == 0) return P.gm1r * (pr / rho);
  double hm1, cs2;
  eos_hm1_cs2<EOS>(P, rho, pr, hm1, cs2);
  return hm1;
}
// pressure / specific internal energy of matter of density rho at temperature T
template <int EOS>
__device__ __forceinline__ double eos_P_at_T(const Par& P, double rho, double T) {
  if (EOS == 0) return rho * T;
  double Pc, epsc, Gi;
  eos_cold(P, rho, Pc, epsc, Gi);
  return Pc + rho * T;
}
template <int EOS>
__device__ __forceinline__ double eos_eps_at_T(const Par& P, double rho, double T) {
  if (EOS == 0) return P.eps_atm;            // T_atm / (Gamma - 1): the only temperature asked for
  double Pc, epsc, Gi;
  eos_cold(P, rho, Pc, epsc, Gi);
  return epsc + T / P.gthm1;
}
// P(rho, eps)
template <int EOS>
__device__ __forceinline__ double eos_P(const Par& P, double rho, double eps) {
  if (EOS == 0) {
    const double T = P.gm1 * eps;
    return rho * T;
  }
  double Pc, epsc, Gi;
  eos_cold(P, rho, Pc, epsc, Gi);
  return Pc + P.gthm1 * rho * (eps - epsc);
}
// temperature floor: raises pr and returns true if T(rho, pr) < T_atm
template <int EOS>
__device__ __forceinline__ bool eos_T_floor(const Par& P, double rho, double& pr) {
  if (EOS == 0) {
    if (pr < rho * P.T_atm) { pr = rho * P.T_atm; return true; }
    return false;
  }
  double Pc, epsc, Gi;
  eos_cold(P, rho, Pc, epsc, Gi);
  if (pr - Pc < rho * P.T_atm) { pr = Pc + rho * P.T_atm; return true; }
  return false;
}

// ------------------------------------------------------------------ O2: prim -> cons (Eq. 6)
// prim = rho, u^i = W v^i, P; B undensitised; cons = D, S_i, tau (undensitised).
// tau in the cancellation-free form of DESIGN.md §3 O2.
template <int EOS = 0>
__device__ __forceinline__ void prim2cons(const Par& P, const Met3& g, double rho, const double u[3],
                                          double pr, const double B[3], double c[5]) {
  double ul[3], Bl[3];
  lower(g, u, ul);
  const double usq = dot3(ul, u);
  const double W = sqrt(1.0 + usq);
  const double iW = 1.0 / W;
  const double vl[3] = {ul[0] * iW, ul[1] * iW, ul[2] * iW};
  lower(g, B, Bl);
  const double B2 = dot3(Bl, B);
  const double Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2];
  const double hm1 = eos_hm1<EOS>(P, rho, pr);
  const double h = 1.0 + hm1;
  const double D = rho * W;
  const double wtot = rho * h * W * W + B2;
  c[0] = D;
  c[1] = wtot * vl[0] - Bv * Bl[0];
  c[2] = wtot * vl[1] - Bv * Bl[1];
  c[3] = wtot * vl[2] - Bv * Bl[2];
  c[4] = D * (hm1 * W + ddiv(usq, 1.0 + W)) + B2 - pr - 0.5 * (Bv * Bv + B2 * iW * iW);
}

// ------------------------------------------------------------------ O3: con2prim
// Bracketed 1-D solve for mu = 1/(W h) (scheme of Kastaun et al. 2021), h0 = 1.
template <int EOS = 0>
struct C2P {
  double q, r2, bs2, rb2, v0sq, gm1;
  const Par* par; double D;    // EOS = 1 only: the EOS constants and the conserved density (rho^ = D / W^)
  // quantities at a trial mu
  double x, rbar2, qbar, vsq, iW, What, eps;
  // static unmagnetised cell (r2 = bs2 = rb2 = 0): x = W^ = 1, rbar2 = 0, eps = qbar = q for every mu, so
  // f(mu) = mu - inv with inv = 1/nu the same number at every evaluation: after one full evaluation
  // (which leaves inv and the trial state behind) the root finder runs on that one subtraction
  bool stat; double inv;
  // unmagnetised cell (exact shortcut, bit 1): bs2 and rb2 are +0.0, r2 is finite and q > 0.  Then for every trial
  // mu >= +0 (the root finder never leaves [0, mu_hi]): x = 1/(1 + mu 0) = 1; rbar2 = r2 1 1 + ((mu 1) 2)(+0) =
  // r2 + 0 (the addition is kept: it turns a -0 into the +0 of the full expression); bs2 r2 - rb2 = +-0, so qbar
  // = (q - 0) - (+-0) = q for q != 0.  One reciprocal and ~15 further operations per evaluation dropped.
  bool nob;
  __device__ __forceinline__ void aux(double mu) {
    if (nob) {
      x = 1.0;
      rbar2 = r2 + 0.0;
      qbar = q;
    } else {
      x = 1.0 / (1.0 + mu * bs2);
      rbar2 = r2 * x * x + mu * x * (1.0 + x) * rb2;
      qbar = q - 0.5 * bs2 - 0.5 * mu * mu * x * x * (bs2 * r2 - rb2);
    }
    vsq = fmin(mu * mu * rbar2, v0sq);
    iW = sqrt(1.0 - vsq);
    What = 1.0 / iW;
    eps = What * (qbar - mu * rbar2) + ddiv(vsq * What * What, 1.0 + What);
  }
  // master function f(mu)
  __device__ __forceinline__ double f(double mu) {
    if (stat) return mu - inv;
    aux(mu);
    double e, ahat;
    if (EOS == 0) {
      e = fmax(eps, 0.0);
      ahat = ddiv(gm1 * e, 1.0 + e);
    } else {                     // general form a^ = P(rho^, eps^) / (rho^ (1 + eps^)), eps^ >= eps_c(rho^)
      const double rhohat = D * iW;
      double Pc, epsc, Gi;
      eos_cold(*par, rhohat, Pc, epsc, Gi);
      e = fmax(eps, epsc);
      const double Phat = Pc + par->gthm1 * rhohat * (e - epsc);
      ahat = Phat / (rhohat * (1.0 + e));
    }
    const double nuA = (1.0 + ahat) * (1.0 + e) * iW;
    const double nuB = (1.0 + ahat) * (1.0 + qbar - mu * rbar2);
    inv = 1.0 / (fmax(nuA, nuB) + mu * rbar2);
    return mu - inv;
  }
  // f(0), ideal gas: the master function at mu = +0 without the operations whose results are then known
  // exactly -- x = 1/(1 + 0 bs2) = 1, W^ = 1/sqrt(1 - 0) = 1, (+-0)/2 = +-0 -- i.e. two reciprocals, a square
  // root and a division fewer; every other operation of aux()/f() is kept as written (products with 0.0
  // included, so that signed zeros come out as they do in the full evaluation): the same bits.  Needs finite
  // r2, bs2, rb2 and v^2 = fmin(0 rbar2, v0sq) == 0 (f0_ok); leaves the trial state (x .. eps) alone.
  __device__ __forceinline__ bool f0_ok() const {
    const double rb0 = r2 + 0.0 * rb2;
    return EOS == 0 && isfinite(r2) && isfinite(bs2) && isfinite(rb2) && fmin(0.0 * rb0, v0sq) == 0.0;
  }
  __device__ __forceinline__ double f0() const {
    const double rb0 = r2 + 0.0 * rb2;                              // rbar2
    const double qb0 = q - 0.5 * bs2 - 0.0 * (bs2 * r2 - rb2);      // qbar
    const double vs0 = fmin(0.0 * rb0, v0sq);                       // +-0
    const double ep0 = (qb0 - 0.0 * rb0) + vs0;                     // W^ (qbar - mu rbar2) + (v^2 W^2)/(1 + W^)
    const double e = fmax(ep0, 0.0);
    const double ahat = ddiv(gm1 * e, 1.0 + e);
    const double nuA = (1.0 + ahat) * (1.0 + e);
    const double nuB = (1.0 + ahat) * (1.0 + qb0 - 0.0 * rb0);
    return 0.0 - 1.0 / (fmax(nuA, nuB) + 0.0 * rb0);
  }
  // auxiliary function whose root bounds mu from above when r >= h0
  __device__ __forceinline__ double fa(double mu) const {
    const double xx = 1.0 / (1.0 + mu * bs2);
    const double rb = r2 * xx * xx + mu * xx * (1.0 + xx) * rb2;
    return mu * sqrt(1.0 + rb) - 1.0;
  }
};

// Illinois-modified regula falsi on [a,b] with fa_ < 0 <= fb_.  AUX selects fa over f.
// The iteration cap is uniform (a parameter), so a warp leaves the loop together at the
// latest after max_iter evaluations.
template <bool AUX, int EOS>
__device__ __forceinline__ bool illinois(C2P<EOS>& s, double a, double b, double fa_, double fb_,
                                         int max_iter, double tol, double& root) {
  int side = 0;
  double cprev = b;
  for (int it = 0; it < max_iter; ++it) {
    const double c = (a * fb_ - b * fa_) / (fb_ - fa_);
    const double fc = AUX ? s.fa(c) : s.f(c);
    if (!(fc == fc)) return false;
    if (fc == 0.0) { root = c; return true; }
    if (fc > 0.0) {
      b = c; fb_ = fc;
      if (side == -1) fa_ = 0.5 * fa_;
      side = -1;
    } else {
      a = c; fa_ = fc;
      if (side == 1) fb_ = 0.5 * fb_;
      side = 1;
    }
    if (fabs(c - cprev) <= tol * c) { root = c; return true; }
    cprev = c;
  }
  return false;
}

// Rare paths: the upper
// bracket when r >= h0 (ultra-relativistic momentum) and the write-back of floored cells (optionally out of line).
#ifndef AK_C2P_RARE_NOINLINE
#define AK_C2P_RARE_NOINLINE 0   // measured: out-of-line costs 17 % (call ABI, stack frame); kept inline
#endif
#if AK_C2P_RARE_NOINLINE
#define AK_RARE __noinline__
#else
#define AK_RARE __forceinline__
#endif
template <int EOS>
__device__ AK_RARE bool c2p_upper_bracket(C2P<EOS>& s, int max_iter, double tol, double& mu_hi) {
  return illinois<true, EOS>(s, 0.0, 1.0, -1.0, s.fa(1.0), max_iter, tol, mu_hi);
}
template <int EOS>
__device__ AK_RARE void c2p_write_back(const Par& P, const Met3& g, double sdet, double rho, double ux, double uy,
                                       double uz, double pr, const double B[3], double Ut[5]) {
  double c5[5];
  const double u[3] = {ux, uy, uz};
  prim2cons<EOS>(P, g, rho, u, pr, B, c5);
  for (int v = 0; v < 5; ++v) Ut[v] = sdet * c5[v];
}

// One cell.  Ut = densitised D,S_i,tau (rewritten from the final primitives when WRITE_BACK
// and the status is non-zero); Bt = densitised cell-centred B; W5 = rho,u^x,u^y,u^z,P.
template <bool WRITE_BACK, int EOS = 0>
__device__ __forceinline__ int c2p_cell(const Par& P, const Met3& g, double Ut[5], const double Bt[3],
                                        double W5[5]) {
  int status = 0;
  double det, sdet;
  metric_det(g, det, sdet);                   // the inverse metric is formed only where a cell needs it (below)
  const double isd = 1.0 / sdet;
  // Static unmagnetised cell (exact shortcut, bit 1; ideal gas): S~_i = +0.0 and B~ = +-0.0.  Then B_i, B^2, r_i,
  // r^i, r^2, (rB) are all zeros, and everything the solve leaves behind is known in closed form (see below).
  const bool zero_SB = EOS == 0 && (P.shortcuts & 2) != 0 &&
                       (__double_as_longlong(Ut[1]) | __double_as_longlong(Ut[2]) | __double_as_longlong(Ut[3])) == 0LL &&
                       Bt[0] == 0.0 && Bt[1] == 0.0 && Bt[2] == 0.0;
  double D = Ut[0] * isd, tau = Ut[4] * isd;
  const double Sl[3] = {Ut[1] * isd, Ut[2] * isd, Ut[3] * isd};
  const double B[3] = {Bt[0] * isd, Bt[1] * isd, Bt[2] * isd};
  double rho = P.rho_atm, ux = 0.0, uy = 0.0, uz = 0.0, pr = P.P_atm;   // P_atm = P(rho_atm, T_atm) of the EOS
  bool solve = true;
  if (!(isfinite(D) && isfinite(Sl[0]) && isfinite(Sl[1]) && isfinite(Sl[2]) && isfinite(tau) &&
        isfinite(B[0]) && isfinite(B[1]) && isfinite(B[2]))) {
    status |= ST_FAIL;
    solve = false;
  }
  double B2 = 0.0;                            // B = +-0: B_i B^i is a zero, and no use below sees its sign
  if (!zero_SB) {
    double Bl[3];
    lower(g, B, Bl);
    B2 = dot3(Bl, B);
  }
  // conserved floors: D floor -> magnetisation cap -> tau floor (reading R5)
  bool atmo = false;
  if (solve && D < P.thr) {
    status |= ST_DFLOOR;
    D = P.rho_atm;
    atmo = true;
  }
  if (solve && B2 > P.mag_max * D) {
    D = B2 / P.mag_max;
    status |= ST_MAGCAP;
  }
  if (solve && atmo) {
    rho = D;
    pr = eos_P_at_T<EOS>(P, D, P.T_atm);
    solve = false;
  }
  if (solve && zero_SB) {
    // tau floor: D eps_atm + 0.5 (+-0) = D eps_atm (non-zero).  Then q = tau/D > 0 and, for EVERY trial mu of the
    // master function: x = 1/(1 + mu 0) = 1, rbar^2 = +0, qbar = q, v^2 = 0, W^ = 1/sqrt(1) = 1, eps^ = 1 (q - mu 0)
    // + ddiv(0, 2) = q.  The state the root finder leaves behind does not depend on the root, so neither do rho =
    // D 1, P = rho (Gamma - 1) q, u^i = W^ mu x (r^i + c B^i) = (+)(+0 + +-0) = +0 (S~_i = +0 makes r_i, r^i = +0).
    // The bracket cannot fail: nu = (1 + a^)(1 + q) > 1, f(1) = 1 - 1/nu > 0 > f(0) = -1/nu; and the Illinois
    // iteration on the linear f(mu) = mu - 1/nu repeats its secant point to ~3 ulp at once (|dmu| <= tol mu).
    const double tau_atm = D * eos_eps_at_T<EOS>(P, D, P.T_atm);
    if (tau < tau_atm) { tau = tau_atm; status |= ST_TAUFLOOR; }
    const double iD = 1.0 / D;
    const double q = tau * iD;
    if (q > 0.0 && isfinite(q)) {
      rho = D;
      pr = eos_P<EOS>(P, rho, q);
      if (!(isfinite(rho) && isfinite(pr))) {
        status |= ST_FAIL;
        rho = P.rho_atm; pr = P.P_atm;
      }
      solve = false;                          // done: on to the primitive floors
    }
  }
  if (solve) {
    Met3 gu;
    {
      double det_, sdet_;
      metric_inverse(g, det_, sdet_, gu);
    }
    const double tau_atm = D * eos_eps_at_T<EOS>(P, D, P.T_atm) + 0.5 * B2;
    if (tau < tau_atm) { tau = tau_atm; status |= ST_TAUFLOOR; }
    const double iD = 1.0 / D;
    C2P<EOS> s;
    s.par = &P; s.D = D;
    s.q = tau * iD;
    const double rl[3] = {Sl[0] * iD, Sl[1] * iD, Sl[2] * iD};
    const double ru[3] = {gu.xx * rl[0] + gu.xy * rl[1] + gu.xz * rl[2],
                          gu.xy * rl[0] + gu.yy * rl[1] + gu.yz * rl[2],
                          gu.xz * rl[0] + gu.yz * rl[1] + gu.zz * rl[2]};
    s.r2 = dot3(rl, ru);
    s.bs2 = B2 * iD;
    const double rB = dot3(rl, B);
    s.rb2 = rB * rB * iD;
    s.v0sq = ddiv(s.r2, 1.0 + s.r2);
    s.gm1 = P.gm1;
    s.stat = false; s.inv = 0.0;
    s.nob = (P.shortcuts & 2) != 0 && (__double_as_longlong(s.bs2) | __double_as_longlong(s.rb2)) == 0LL &&
            isfinite(s.r2) && s.q > 0.0;
    bool ok = true;
    double mu_hi = 1.0;
    if (!(s.r2 < 1.0)) {
      ok = c2p_upper_bracket(s, P.max_iter, P.tol, mu_hi);
      mu_hi = mu_hi * (1.0 + 1e-14);
      if (mu_hi > 1.0) mu_hi = 1.0;
    }
    double mu = 0.0;
    // Static unmagnetised cell, ideal gas (exact shortcut, bit 1): with S = 0 and B = 0 exactly, r^2 = b^2 =
    // (rb)^2 = 0 and, for EVERY trial mu, x = 1/(1 + mu 0) = 1, rbar^2 = +0, qbar = q - 0 - 0 = q, v^2 = 0, W^ =
    // 1/sqrt(1) = 1, eps^ = 1 (q - mu 0) + ddiv(0, 2) = q: the state the root finder would leave behind does not
    // depend on the root, so neither do rho = D 1, P = rho (Gamma - 1) q and u^i = W^ mu x (+-0) = +-0 (mu > 0
    // enters through its sign only).  The bracket cannot fail: nu = (1 + a^)(1 + q) > 1 gives f(1) = 1 - 1/nu >
    // 0 > f(0) = -1/nu, and the Illinois iteration on the linear f(mu) = mu - 1/nu reaches |dmu| <= tol mu within
    // a few steps (the second secant point already repeats the first to ~3 ulp).  So: no master-function
    // evaluation, no iteration.
    const bool closed = EOS == 0 && (P.shortcuts & 2) && ok && s.r2 == 0.0 && s.bs2 == 0.0 && s.rb2 == 0.0 &&
                        s.q > 0.0 && isfinite(s.q);
    if (closed) {                             // zeros of other signs (S~_i = -0.0): the same closed form, r^i kept
      s.x = 1.0; s.rbar2 = 0.0; s.qbar = s.q; s.vsq = 0.0; s.iW = 1.0; s.What = 1.0; s.eps = s.q;
      mu = 1.0;
    } else if (ok) {
      const double f_hi = s.f(mu_hi);
      // S = 0 and B = 0 exactly (static atmosphere, the bulk of a merger grid): every later evaluation is
      // mu - inv with the inv this one left behind (q > 0 keeps eps = qbar away from a signed zero)
      s.stat = (P.shortcuts & 2) && s.r2 == 0.0 && s.bs2 == 0.0 && s.rb2 == 0.0 && s.q > 0.0;
      // f(0) by its shortcut where that is exact; it does not touch the trial state, which then still
      // belongs to mu_hi
      bool state_hi = true;
      double f_lo;
      if (s.stat) f_lo = 0.0 - s.inv;
      else if (s.f0_ok()) f_lo = s.f0();
      else { f_lo = s.f(0.0); state_hi = false; }
      if (!(f_hi >= 0.0) || !(f_lo < 0.0)) ok = false;
      else if (f_hi == 0.0) { mu = mu_hi; if (!state_hi) s.aux(mu); }
      else ok = illinois<false, EOS>(s, 0.0, mu_hi, f_lo, f_hi, P.max_iter, P.tol, mu);
    }
    if (!ok) {
      status |= ST_FAIL;
    } else {
      // the trial state (x, rbar2, qbar, W^, eps) is that of mu already: the root finder returns the last
      // point it evaluated, so aux(mu) would recompute the same values (one reciprocal pair, sqrt, division)
      rho = D * s.iW;
      pr = eos_P<EOS>(P, rho, s.eps);
      const double c = mu * rB * iD;
      const double mx = mu * s.x;
      ux = s.What * (mx * (ru[0] + c * B[0]));
      uy = s.What * (mx * (ru[1] + c * B[1]));
      uz = s.What * (mx * (ru[2] + c * B[2]));
      if (!(isfinite(rho) && isfinite(pr) && isfinite(ux) && isfinite(uy) && isfinite(uz))) {
        status |= ST_FAIL;
        rho = P.rho_atm; ux = uy = uz = 0.0; pr = P.P_atm;
      }
    }
  }
  // primitive floors
  if (rho < P.thr) {
    rho = P.rho_atm; ux = uy = uz = 0.0; pr = P.P_atm;
    status |= ST_RHOFLOOR;
  } else if (eos_T_floor<EOS>(P, rho, pr)) {
    status |= ST_TFLOOR;
  }
  W5[0] = rho; W5[1] = ux; W5[2] = uy; W5[3] = uz; W5[4] = pr;
  if (WRITE_BACK && status != 0) c2p_write_back<EOS>(P, g, sdet, rho, ux, uy, uz, pr, B, Ut);
  return status;
}

}  // namespace ak
