// oracle/stage.cpp — CPU ORACLE, block-level steps O3 (all cells), O4-O6 sweeps, O7 FOFC
// (+DMP), O8 constrained-transport corner EMFs, O9 flux divergence + geometric sources.
// Test infrastructure only (see oracle.h).  Straight loops, one MeshBlock at a time.
#include "oracle.h"
#include "eos.h"
#include <cmath>
#include <cstring>
#include <functional>
#include <thread>
#include <vector>

namespace {

struct Geo {
  int n, ng, nt, px, is, ie;
  long ncell;                         // nt^3
  long nxf, nyf, nzf;                 // per-block sizes of the three face layouts
  Geo(int n_, int ng_) : n(n_), ng(ng_) {
    nt = n + 2 * ng; px = nt + 4; is = ng; ie = ng + n - 1;
    ncell = (long)nt * nt * nt;
    nxf = (long)nt * nt * px; nyf = (long)nt * (nt + 1) * nt; nzf = (long)(nt + 1) * nt * nt;
  }
  long c(int m, int k, int j, int i) const { return (((long)m * nt + k) * nt + j) * nt + i; }
  // face of direction d whose d-index is the one among (k,j,i)
  long f(int d, int m, int k, int j, int i) const {
    if (d == 0) return (((long)m * nt + k) * nt + j) * px + i;
    if (d == 1) return (((long)m * nt + k) * (nt + 1) + j) * nt + i;
    return (((long)m * (nt + 1) + k) * nt + j) * nt + i;
  }
  long fsize(int d) const { return d == 0 ? nxf : (d == 1 ? nyf : nzf); }
  // edge EMF component c
  long e(int c, int m, int k, int j, int i) const {
    if (c == 0) return (((long)m * (nt + 1) + k) * (nt + 1) + j) * nt + i;
    if (c == 1) return (((long)m * (nt + 1) + k) * nt + j) * px + i;
    return (((long)m * nt + k) * (nt + 1) + j) * px + i;
  }
};

inline void ijk_from(int d, int id, int it1, int it2, int& k, int& j, int& i) {
  // d-index id, transverse indices it1 (direction d+1), it2 (direction d+2); 0=x(i),1=y(j),2=z(k)
  int v[3];
  v[d] = id; v[(d + 1) % 3] = it1; v[(d + 2) % 3] = it2;
  i = v[0]; j = v[1]; k = v[2];
}

struct Stage {
  const orc_params* p;
  Geo G;
  const double* dx;
  double* const* U;
  const double* const* Bf;
  const double* const* adm;
  double* const* W;
  double dt;
  double* const* dU;
  double* const* E;
  unsigned char* flag;
  unsigned char* status;
  double* const* flux_out;
  unsigned char* const* refl;
  // FOFC estimate of a later Runge-Kutta stage ("the next Runge-Kutta step is estimated"):
  // U* = fa * U0 + fb * (U - dt div F) when U0 is given (reading R9), else U - dt div F
  const double* const* U0 = nullptr;
  double fa = 0.0, fb = 1.0;
  Stage(const orc_params* p_) : p(p_), G(p_->n, p_->ng) {}

  void cell_metric10(long c, double m[10]) const {
    m[0] = adm[6][c]; m[1] = adm[7][c]; m[2] = adm[8][c]; m[3] = adm[9][c];
    for (int q = 0; q < 6; ++q) m[4 + q] = adm[q][c];
  }

  // ---------------- O3 over one block ----------------
  void con2prim_block(int m) const {
    const int nt = G.nt;
    for (int k = 0; k < nt; ++k)
      for (int j = 0; j < nt; ++j)
        for (int i = 0; i < nt; ++i) {
          const long c = G.c(m, k, j, i);
          double g[6], Ut[5], Bc[3], Wc[5];
          for (int q = 0; q < 6; ++q) g[q] = adm[q][c];
          for (int v = 0; v < 5; ++v) Ut[v] = U[v][c];
          Bc[0] = 0.5 * (Bf[0][G.f(0, m, k, j, i)] + Bf[0][G.f(0, m, k, j, i + 1)]);
          Bc[1] = 0.5 * (Bf[1][G.f(1, m, k, j, i)] + Bf[1][G.f(1, m, k, j + 1, i)]);
          Bc[2] = 0.5 * (Bf[2][G.f(2, m, k, j, i)] + Bf[2][G.f(2, m, k + 1, j, i)]);
          const int st = orc_con2prim_cell(p, g, Ut, Bc, Wc, 0, nullptr);
          for (int v = 0; v < 5; ++v) W[v][c] = Wc[v];
          for (int v = 0; v < 3; ++v) W[5 + v][c] = Bc[v];
          if (st != 0) for (int v = 0; v < 5; ++v) U[v][c] = Ut[v];
          if (status) status[c] = (unsigned char)st;
        }
  }

  // ---------------- O4-O6: one face ----------------
  void face(int d, int m, int k, int j, int i, int recon, int riemann, double F[7]) const {
    const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
    const int var[7] = {0, 1, 2, 3, 4, 5 + t1, 5 + t2};
    const long stride = d == 0 ? 1 : (d == 1 ? G.nt : (long)G.nt * G.nt);
    const long cu = G.c(m, k, j, i);  // upper cell of the face
    const long cl = cu - stride;      // lower cell
    double WL[7], WR[7], q[5], qm, qp;
    for (int v = 0; v < 7; ++v) {
      const double* w = W[var[v]];
      for (int s = 0; s < 5; ++s) q[s] = w[cl + (s - 2) * stride];
      orc_reconstruct(recon, q, &qm, &qp);
      WL[v] = qp;                      // right face of the lower cell
      for (int s = 0; s < 5; ++s) q[s] = w[cu + (s - 2) * stride];
      orc_reconstruct(recon, q, &qm, &qp);
      WR[v] = qm;                      // left face of the upper cell
    }
    double gL[10], gR[10];
    cell_metric10(cl, gL);
    cell_metric10(cu, gR);
    orc_face_flux(p, d, riemann, gL, gR, WL, WR, Bf[d][G.f(d, m, k, j, i)], 1, F, nullptr);
  }

  // ---------------- one block, whole stage ----------------
  void block(int m) const {
    const int nt = G.nt, is = G.is, ie = G.ie;
    if (W_needs_c2p) con2prim_block(m);
    // face fluxes F[d][7], each in the face layout of direction d (one block)
    std::vector<double> Fs[3][7];
    for (int d = 0; d < 3; ++d)
      for (int v = 0; v < 7; ++v) Fs[d][v].assign(G.fsize(d), 0.0);
    auto fl = [&](int d, int k, int j, int i) { return G.f(d, 0, k, j, i); };
    for (int d = 0; d < 3; ++d)
      for (int id = is - 1; id <= ie + 2; ++id)
        for (int a = is - 1; a <= ie + 1; ++a)
          for (int b = is - 1; b <= ie + 1; ++b) {
            int k, j, i;
            ijk_from(d, id, a, b, k, j, i);
            double F[7];
            face(d, m, k, j, i, p->recon, p->riemann, F);
            for (int v = 0; v < 7; ++v) Fs[d][v][fl(d, k, j, i)] = F[v];
          }
    // ---------------- O7: FOFC (+DMP), P:141-157 ----------------
    std::vector<unsigned char> flg(G.ncell, 0);
    const double idx[3] = {1.0 / dx[3 * m + 0], 1.0 / dx[3 * m + 1], 1.0 / dx[3 * m + 2]};
    if (p->fofc) {
      const double iM = p->dmp_M > 0.0 ? 1.0 / p->dmp_M : 0.0;
      for (int k = is - 1; k <= ie + 1; ++k)
        for (int j = is - 1; j <= ie + 1; ++j)
          for (int i = is - 1; i <= ie + 1; ++i) {
            const long c = G.c(m, k, j, i);
            double Us[5], g[6], Bc[3], Wc[5];
            for (int v = 0; v < 5; ++v) {
              const double div = (Fs[0][v][fl(0, k, j, i + 1)] - Fs[0][v][fl(0, k, j, i)]) * idx[0] +
                                 (Fs[1][v][fl(1, k, j + 1, i)] - Fs[1][v][fl(1, k, j, i)]) * idx[1] +
                                 (Fs[2][v][fl(2, k + 1, j, i)] - Fs[2][v][fl(2, k, j, i)]) * idx[2];
              if (U0) Us[v] = fa * U0[v][c] + fb * (U[v][c] - dt * div);
              else Us[v] = U[v][c] - dt * div;
            }
            for (int q = 0; q < 6; ++q) g[q] = adm[q][c];
            for (int v = 0; v < 3; ++v) Bc[v] = W[5 + v][c];
            int st = orc_con2prim_cell(p, g, Us, Bc, Wc, 1, nullptr);
            if (p->dmp_M > 0.0) {  // Eq. 12 on D~ and tau~ over the 27-cell neighbourhood
              double Dmin = U[0][c], Dmax = U[0][c], tmin = U[4][c], tmax = U[4][c];
              for (int kk = -1; kk <= 1; ++kk)
                for (int jj = -1; jj <= 1; ++jj)
                  for (int ii = -1; ii <= 1; ++ii) {
                    const long cn = G.c(m, k + kk, j + jj, i + ii);
                    Dmin = std::fmin(Dmin, U[0][cn]); Dmax = std::fmax(Dmax, U[0][cn]);
                    tmin = std::fmin(tmin, U[4][cn]); tmax = std::fmax(tmax, U[4][cn]);
                  }
              if (Us[0] < Dmin * iM || Us[0] > p->dmp_M * Dmax || Us[4] < tmin * iM ||
                  Us[4] > p->dmp_M * tmax)
                st |= ORC_DMP;
            }
            flg[G.c(0, k, j, i)] = (unsigned char)st;
          }
      // re-flux every computed face with a flagged neighbour (both cells of the face
      // are looked up; cells outside the test range carry flag 0)
      for (int d = 0; d < 3; ++d)
        for (int id = is - 1; id <= ie + 2; ++id)
          for (int a = is - 1; a <= ie + 1; ++a)
            for (int b = is - 1; b <= ie + 1; ++b) {
              int k, j, i;
              ijk_from(d, id, a, b, k, j, i);
              const long stride = d == 0 ? 1 : (d == 1 ? nt : (long)nt * nt);
              const long cu = G.c(0, k, j, i);
              if (!(flg[cu] || flg[cu - stride])) continue;
              double F[7];
              face(d, m, k, j, i, 0, p->fofc_riemann, F);
              for (int v = 0; v < 7; ++v) Fs[d][v][fl(d, k, j, i)] = F[v];
              if (refl && refl[d]) refl[d][G.f(d, m, k, j, i)] = 1;
            }
    }
    if (flag) std::memcpy(flag + G.c(m, 0, 0, 0), flg.data(), G.ncell);
    if (flux_out)
      for (int d = 0; d < 3; ++d)
        for (int v = 0; v < 7; ++v)
          if (flux_out[7 * d + v])
            std::memcpy(flux_out[7 * d + v] + (long)m * G.fsize(d), Fs[d][v].data(),
                        sizeof(double) * G.fsize(d));

    // ---------------- O8: CT corner EMFs (Gardiner & Stone 2005) ----------------
    // cell-centred EMF  E_c = -alpha (vhat^a B~^b - vhat^b B~^a), (a,b) cyclic after c
    std::vector<double> Ecc[3];
    for (int c3 = 0; c3 < 3; ++c3) Ecc[c3].assign(G.ncell, 0.0);
    for (int k = 0; k < nt; ++k)
      for (int j = 0; j < nt; ++j)
        for (int i = 0; i < nt; ++i) {
          const long c = G.c(m, k, j, i);
          double g[6];
          for (int q = 0; q < 6; ++q) g[q] = adm[q][c];
          const double u[3] = {W[1][c], W[2][c], W[3][c]};
          const double ul[3] = {g[0] * u[0] + g[1] * u[1] + g[2] * u[2],
                                g[1] * u[0] + g[3] * u[1] + g[4] * u[2],
                                g[2] * u[0] + g[4] * u[1] + g[5] * u[2]};
          const double usq = ul[0] * u[0] + ul[1] * u[1] + ul[2] * u[2];
          const double iW = 1.0 / std::sqrt(1.0 + usq);
          const double alp = adm[6][c], ialp = 1.0 / alp;
          const double vh[3] = {u[0] * iW - adm[7][c] * ialp, u[1] * iW - adm[8][c] * ialp,
                                u[2] * iW - adm[9][c] * ialp};
          const double Bt[3] = {W[5][c], W[6][c], W[7][c]};
          for (int c3 = 0; c3 < 3; ++c3) {
            const int a = (c3 + 1) % 3, b = (c3 + 2) % 3;
            Ecc[c3][G.c(0, k, j, i)] = -(alp * (vh[a] * Bt[b] - vh[b] * Bt[a]));
          }
        }
    auto wgt = [](double fD) { return fD > 0.0 ? 1.0 : (fD < 0.0 ? 0.0 : 0.5); };
    for (int c3 = 0; c3 < 3; ++c3) {
      const int a = (c3 + 1) % 3, b = (c3 + 2) % 3;
      // index helpers: (ia, ib, ic) -> (k,j,i)
      auto KJI = [&](int ia, int ib, int ic, int& k, int& j, int& i) {
        int v[3]; v[a] = ia; v[b] = ib; v[c3] = ic; i = v[0]; j = v[1]; k = v[2];
      };
      auto Eaf = [&](int ia, int ib, int ic) {   // E_c on a-faces: -F^a[slot t1]
        int k, j, i; KJI(ia, ib, ic, k, j, i); return -Fs[a][5][fl(a, k, j, i)];
      };
      auto Ebf = [&](int ia, int ib, int ic) {   // E_c on b-faces: +F^b[slot t2]
        int k, j, i; KJI(ia, ib, ic, k, j, i); return Fs[b][6][fl(b, k, j, i)];
      };
      auto FaD = [&](int ia, int ib, int ic) { int k, j, i; KJI(ia, ib, ic, k, j, i); return Fs[a][0][fl(a, k, j, i)]; };
      auto FbD = [&](int ia, int ib, int ic) { int k, j, i; KJI(ia, ib, ic, k, j, i); return Fs[b][0][fl(b, k, j, i)]; };
      auto Ec = [&](int ia, int ib, int ic) { int k, j, i; KJI(ia, ib, ic, k, j, i); return Ecc[c3][G.c(0, k, j, i)]; };
      for (int ic = is; ic <= ie; ++ic)
        for (int ib = is; ib <= ie + 1; ++ib)
          for (int ia = is; ia <= ie + 1; ++ia) {
            const double w = wgt(FaD(ia, ib, ic)), wp = wgt(FaD(ia, ib - 1, ic));
            const double w2 = wgt(FbD(ia, ib, ic)), w2p = wgt(FbD(ia - 1, ib, ic));
            const double dbm = w * (Ec(ia - 1, ib, ic) - Ebf(ia - 1, ib, ic)) +
                               (1.0 - w) * (Ec(ia, ib, ic) - Ebf(ia, ib, ic));
            const double dbp = wp * (Ebf(ia - 1, ib, ic) - Ec(ia - 1, ib - 1, ic)) +
                               (1.0 - wp) * (Ebf(ia, ib, ic) - Ec(ia, ib - 1, ic));
            const double dam = w2 * (Ec(ia, ib - 1, ic) - Eaf(ia, ib - 1, ic)) +
                               (1.0 - w2) * (Ec(ia, ib, ic) - Eaf(ia, ib, ic));
            const double dap = w2p * (Eaf(ia, ib - 1, ic) - Ec(ia - 1, ib - 1, ic)) +
                               (1.0 - w2p) * (Eaf(ia, ib, ic) - Ec(ia - 1, ib, ic));
            const double e = 0.25 * (Eaf(ia, ib, ic) + Eaf(ia, ib - 1, ic) + Ebf(ia, ib, ic) +
                                     Ebf(ia - 1, ib, ic)) +
                             0.25 * ((dbp - dbm) + (dap - dam));
            int k, j, i; KJI(ia, ib, ic, k, j, i);
            E[c3][G.e(c3, m, k, j, i)] = e;
          }
    }

    // ---------------- O9: flux divergence + geometric sources (Eq. 9) --------
    const double h2[3] = {0.5 / dx[3 * m + 0], 0.5 / dx[3 * m + 1], 0.5 / dx[3 * m + 2]};
    const long st3[3] = {1, nt, (long)nt * nt};
    for (int k = is; k <= ie; ++k)
      for (int j = is; j <= ie; ++j)
        for (int i = is; i <= ie; ++i) {
          const long c = G.c(m, k, j, i);
          double du[5];
          for (int v = 0; v < 5; ++v) {
            const double div = (Fs[0][v][fl(0, k, j, i + 1)] - Fs[0][v][fl(0, k, j, i)]) * idx[0] +
                               (Fs[1][v][fl(1, k, j + 1, i)] - Fs[1][v][fl(1, k, j, i)]) * idx[1] +
                               (Fs[2][v][fl(2, k + 1, j, i)] - Fs[2][v][fl(2, k, j, i)]) * idx[2];
            du[v] = -div;
          }
          double g[6], det, sdet, gi[6];
          for (int q = 0; q < 6; ++q) g[q] = adm[q][c];
          orc_metric_inverse(g, &det, &sdet, gi);
          const double isd = 1.0 / sdet;
          const double prim[5] = {W[0][c], W[1][c], W[2][c], W[3][c], W[4][c]};
          const double B[3] = {W[5][c] * isd, W[6][c] * isd, W[7][c] * isd};
          double cons[5];
          orc_prim2cons_eos(p, g, prim, B, cons);
          const double rho = prim[0], P = prim[4];
          const double u[3] = {prim[1], prim[2], prim[3]};
          const double ul[3] = {g[0] * u[0] + g[1] * u[1] + g[2] * u[2],
                                g[1] * u[0] + g[3] * u[1] + g[4] * u[2],
                                g[2] * u[0] + g[4] * u[1] + g[5] * u[2]};
          const double usq = ul[0] * u[0] + ul[1] * u[1] + ul[2] * u[2];
          const double Wl = std::sqrt(1.0 + usq), iW = 1.0 / Wl;
          const double Bl[3] = {g[0] * B[0] + g[1] * B[1] + g[2] * B[2],
                                g[1] * B[0] + g[3] * B[1] + g[4] * B[2],
                                g[2] * B[0] + g[4] * B[1] + g[5] * B[2]};
          const double B2 = Bl[0] * B[0] + Bl[1] * B[1] + Bl[2] * B[2];
          const double vl[3] = {ul[0] * iW, ul[1] * iW, ul[2] * iW};
          const double Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2];
          const double b2 = B2 * iW * iW + Bv * Bv;
          const double bl[3] = {Bl[0] * iW + Bv * ul[0], Bl[1] * iW + Bv * ul[1],
                                Bl[2] * iW + Bv * ul[2]};
          const double h = 1.0 + eos_hm1(orc_make_eos(p), rho, P);
          const double Ptot = P + 0.5 * b2;
          const double wt = rho * h + b2;
          // S_ij = (rho h + b^2) u_i u_j + Ptot g_ij - b_i b_j ; packed xx,xy,xz,yy,yz,zz
          const int I[6] = {0, 0, 0, 1, 1, 2}, J[6] = {0, 1, 2, 1, 2, 2};
          double Sdd[3][3], gim[3][3];
          for (int q = 0; q < 6; ++q) {
            const double s = wt * ul[I[q]] * ul[J[q]] + Ptot * g[q] - bl[I[q]] * bl[J[q]];
            Sdd[I[q]][J[q]] = s; Sdd[J[q]][I[q]] = s;
            gim[I[q]][J[q]] = gi[q]; gim[J[q]][I[q]] = gi[q];
          }
          double T[3][3], Suu[6];
          for (int a = 0; a < 3; ++a)
            for (int l = 0; l < 3; ++l)
              T[a][l] = gim[a][0] * Sdd[0][l] + gim[a][1] * Sdd[1][l] + gim[a][2] * Sdd[2][l];
          for (int q = 0; q < 6; ++q)
            Suu[q] = T[I[q]][0] * gim[0][J[q]] + T[I[q]][1] * gim[1][J[q]] + T[I[q]][2] * gim[2][J[q]];
          const double Sl[3] = {cons[1], cons[2], cons[3]};
          const double Su[3] = {gi[0] * Sl[0] + gi[1] * Sl[1] + gi[2] * Sl[2],
                                gi[1] * Sl[0] + gi[3] * Sl[1] + gi[4] * Sl[2],
                                gi[2] * Sl[0] + gi[4] * Sl[1] + gi[5] * Sl[2]};
          const double Een = cons[4] + cons[0];
          const double alp = adm[6][c];
          double dalp[3];
          for (int a = 0; a < 3; ++a) {
            const long s = st3[a];
            dalp[a] = (adm[6][c + s] - adm[6][c - s]) * h2[a];
            double dg[6], dbeta[3];
            for (int q = 0; q < 6; ++q) dg[q] = (adm[q][c + s] - adm[q][c - s]) * h2[a];
            for (int b = 0; b < 3; ++b) dbeta[b] = (adm[7 + b][c + s] - adm[7 + b][c - s]) * h2[a];
            const double Sdg = Suu[0] * dg[0] + 2.0 * (Suu[1] * dg[1]) + 2.0 * (Suu[2] * dg[2]) +
                               Suu[3] * dg[3] + 2.0 * (Suu[4] * dg[4]) + Suu[5] * dg[5];
            const double Sdb = Sl[0] * dbeta[0] + Sl[1] * dbeta[1] + Sl[2] * dbeta[2];
            du[1 + a] = du[1 + a] + sdet * (0.5 * alp * Sdg + Sdb - Een * dalp[a]);
          }
          const double KS = adm[10][c] * Suu[0] + 2.0 * (adm[11][c] * Suu[1]) +
                            2.0 * (adm[12][c] * Suu[2]) + adm[13][c] * Suu[3] +
                            2.0 * (adm[14][c] * Suu[4]) + adm[15][c] * Suu[5];
          const double Sda = Su[0] * dalp[0] + Su[1] * dalp[1] + Su[2] * dalp[2];
          du[4] = du[4] + sdet * (alp * KS - Sda);
          for (int v = 0; v < 5; ++v) dU[v][c] = du[v];
        }
  }
  bool W_needs_c2p = true;
};

void run_blocks(int nmb, int nthreads, const std::function<void(int)>& fn) {
  if (nthreads <= 1) { for (int m = 0; m < nmb; ++m) fn(m); return; }
  std::vector<std::thread> th;
  for (int t = 0; t < nthreads; ++t)
    th.emplace_back([=, &fn]() { for (int m = t; m < nmb; m += nthreads) fn(m); });
  for (auto& t : th) t.join();
}
}  // namespace

// Matter terms a spacetime solver needs from the fluid ("E = tau + D ... S_ij = T_ij";
// P:129 "the matter source terms ... for the Z4c equations"): E, S_i, S_ij (undensitised) at
// every stored cell from the cell-centred primitives.  out[10] = E, Sx, Sy, Sz, Sxx, Sxy, Sxz, Syy, Syz, Szz.
extern "C" void orc_matter_sources(const orc_params* p, const double* const W[8],
                                   const double* const g6[6], double* const out[10]) {
  const Geo G(p->n, p->ng);
  const long ncell = (long)p->nmb * G.ncell;
  for (long c = 0; c < ncell; ++c) {
    double g[6], det, sdet, gi[6];
    for (int q = 0; q < 6; ++q) g[q] = g6[q][c];
    orc_metric_inverse(g, &det, &sdet, gi);
    const double isd = 1.0 / sdet;
    const double prim[5] = {W[0][c], W[1][c], W[2][c], W[3][c], W[4][c]};
    const double B[3] = {W[5][c] * isd, W[6][c] * isd, W[7][c] * isd};
    double cons[5];
    orc_prim2cons_eos(p, g, prim, B, cons);
    const double rho = prim[0], P = prim[4];
    const double u[3] = {prim[1], prim[2], prim[3]};
    const double ul[3] = {g[0] * u[0] + g[1] * u[1] + g[2] * u[2], g[1] * u[0] + g[3] * u[1] + g[4] * u[2],
                          g[2] * u[0] + g[4] * u[1] + g[5] * u[2]};
    const double usq = ul[0] * u[0] + ul[1] * u[1] + ul[2] * u[2];
    const double iW = 1.0 / std::sqrt(1.0 + usq);
    const double Bl[3] = {g[0] * B[0] + g[1] * B[1] + g[2] * B[2], g[1] * B[0] + g[3] * B[1] + g[4] * B[2],
                          g[2] * B[0] + g[4] * B[1] + g[5] * B[2]};
    const double B2 = Bl[0] * B[0] + Bl[1] * B[1] + Bl[2] * B[2];
    const double vl[3] = {ul[0] * iW, ul[1] * iW, ul[2] * iW};
    const double Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2];
    const double b2 = B2 * iW * iW + Bv * Bv;
    const double bl[3] = {Bl[0] * iW + Bv * ul[0], Bl[1] * iW + Bv * ul[1], Bl[2] * iW + Bv * ul[2]};
    const double h = 1.0 + eos_hm1(orc_make_eos(p), rho, P);
    const double Ptot = P + 0.5 * b2;
    const double wt = rho * h + b2;
    out[0][c] = cons[4] + cons[0];
    out[1][c] = cons[1]; out[2][c] = cons[2]; out[3][c] = cons[3];
    const int I[6] = {0, 0, 0, 1, 1, 2}, J[6] = {0, 1, 2, 1, 2, 2};
    for (int q = 0; q < 6; ++q) out[4 + q][c] = wt * ul[I[q]] * ul[J[q]] + Ptot * g[q] - bl[I[q]] * bl[J[q]];
  }
}

extern "C" void orc_con2prim(const orc_params* p, double* const U[5], const double* const Bf[3],
                             const double* const g[6], double* const W[8],
                             unsigned char* status, int nthreads) {
  Stage S(p);
  S.U = U; S.Bf = Bf; S.adm = g; S.W = W; S.status = status;
  run_blocks(p->nmb, nthreads, [&](int m) { S.con2prim_block(m); });
}

extern "C" void orc_rhs_blend(const orc_params* p, const double* dx, double* const U[5],
                              const double* const Bf[3], const double* const adm[16],
                              double* const W[8], int w_is_valid, double dt_fofc,
                              const double* const U0[5], double fa, double fb,
                              double* const out_dU[5], double* const out_E[3], unsigned char* flag,
                              unsigned char* c2p_status, int nthreads) {
  Stage S(p);
  S.dx = dx; S.U = U; S.Bf = Bf; S.adm = adm; S.W = W; S.dt = dt_fofc; S.dU = out_dU;
  S.E = out_E; S.flag = flag; S.status = c2p_status; S.flux_out = nullptr;
  S.refl = nullptr; S.W_needs_c2p = !w_is_valid;
  S.U0 = U0; S.fa = fa; S.fb = fb;
  run_blocks(p->nmb, nthreads, [&](int m) { S.block(m); });
}

extern "C" void orc_rhs(const orc_params* p, const double* dx, double* const U[5],
                        const double* const Bf[3], const double* const adm[16],
                        double* const W[8], int w_is_valid, double dt_fofc,
                        double* const out_dU[5], double* const out_E[3], unsigned char* flag,
                        unsigned char* c2p_status, double* const flux_out[21],
                        unsigned char* const face_refluxed[3], int nthreads) {
  Stage S(p);
  S.dx = dx; S.U = U; S.Bf = Bf; S.adm = adm; S.W = W; S.dt = dt_fofc; S.dU = out_dU;
  S.E = out_E; S.flag = flag; S.status = c2p_status; S.flux_out = flux_out;
  S.refl = face_refluxed; S.W_needs_c2p = !w_is_valid;
  run_blocks(p->nmb, nthreads, [&](int m) { S.block(m); });
}
