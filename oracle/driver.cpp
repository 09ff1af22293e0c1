// oracle/driver.cpp — CPU ORACLE, stage driver (test infrastructure only; see oracle.h).
// Ghost fill of a self-contained MeshBlock (periodic / outflow), the Shu-Osher register update
// of SSP-RK2 / SSP-RK3 ("RK2 ... RK3"), the constrained-transport update of the
// face-centred B~ from the edge EMFs, and the loop that strings them together.
// DESIGN.md §11.  Straight loops; -ffp-contract=off; every operation in the order written.
#include "oracle.h"
#include <cstring>
#include <vector>

namespace {

struct Lay {
  int n, ng, nt, px, is, ie;
  Lay(int n_, int ng_) : n(n_), ng(ng_) { nt = n + 2 * ng; px = nt + 4; is = ng; ie = ng + n - 1; }
  long c(int m, int k, int j, int i) const { return (((long)m * nt + k) * nt + j) * nt + i; }
  long f(int d, int m, int k, int j, int i) const {
    if (d == 0) return (((long)m * nt + k) * nt + j) * px + i;
    if (d == 1) return (((long)m * nt + k) * (nt + 1) + j) * nt + i;
    return (((long)m * (nt + 1) + k) * nt + j) * nt + i;
  }
  long e(int c3, int m, int k, int j, int i) const {
    if (c3 == 0) return (((long)m * (nt + 1) + k) * (nt + 1) + j) * nt + i;
    if (c3 == 1) return (((long)m * (nt + 1) + k) * nt + j) * px + i;
    return (((long)m * nt + k) * (nt + 1) + j) * px + i;
  }
  // source index of a cell-like index q in [0, nt): itself when interior
  int src_cell(int q, int bc) const {
    if (q >= is && q <= ie) return q;
    if (bc == 0) { int r = (q - is) % n; if (r < 0) r += n; return is + r; }
    return q < is ? is : ie;
  }
  // source index of a face-normal index q in [0, nt]: faces is..ie+1 bound the interior;
  // periodic: face ie+1 is face is
  int src_face(int q, int bc) const {
    if (bc == 0) { int r = (q - is) % n; if (r < 0) r += n; return is + r; }
    if (q < is) return is;
    if (q > ie + 1) return ie + 1;
    return q;
  }
};

}  // namespace

extern "C" void orc_fill_ghosts(const orc_params* p, const int bc[3], double* const U[5],
                                double* const Bf[3]) {
  const Lay L(p->n, p->ng);
  const int nt = L.nt;
  for (int m = 0; m < p->nmb; ++m) {
    for (int k = 0; k < nt; ++k)
      for (int j = 0; j < nt; ++j)
        for (int i = 0; i < nt; ++i) {
          const int ks = L.src_cell(k, bc[2]), js = L.src_cell(j, bc[1]), is_ = L.src_cell(i, bc[0]);
          if (ks == k && js == j && is_ == i) continue;
          for (int v = 0; v < 5; ++v) U[v][L.c(m, k, j, i)] = U[v][L.c(m, ks, js, is_)];
        }
    // face fields: normal index over nt+1 faces, transverse like cells
    for (int d = 0; d < 3; ++d) {
      const int ni = nt + (d == 0), nj = nt + (d == 1), nk = nt + (d == 2);
      for (int k = 0; k < nk; ++k)
        for (int j = 0; j < nj; ++j)
          for (int i = 0; i < ni; ++i) {
            const int ks = d == 2 ? L.src_face(k, bc[2]) : L.src_cell(k, bc[2]);
            const int js = d == 1 ? L.src_face(j, bc[1]) : L.src_cell(j, bc[1]);
            const int is_ = d == 0 ? L.src_face(i, bc[0]) : L.src_cell(i, bc[0]);
            if (ks == k && js == j && is_ == i) continue;
            Bf[d][L.f(d, m, k, j, i)] = Bf[d][L.f(d, m, ks, js, is_)];
          }
    }
  }
}

// ---- same-level ghost exchange between MeshBlocks ("interblock
// communication") ---------------------------------------------------------------------------
// nbr[m][27]: block adjacent to m at offset (oz+1)*9 + (oy+1)*3 + (ox+1), ox,oy,oz in {-1,0,1}; -1 = none.
// Pass 1: a ghost element whose offset block exists is copied from that block's interior (index
// shifted by n per offset direction; the shared face ie+1 is taken from the upper neighbour's
// face is).  Pass 2: for the others, every offset direction whose face neighbour is missing is a
// physical side and gets bc[d] (periodic onto the block itself, or outflow); the source may be a
// ghost element filled in pass 1.
namespace {
inline int region_cell(const Lay& L, int q) { return q < L.is ? -1 : (q > L.ie ? 1 : 0); }
// faces along their normal: is..ie are owned; ie+1 is the upper neighbour's face is when there is
// such a neighbour (or the side is periodic onto the block itself), else it is owned too
inline int region_face(const Lay& L, int q, bool upper_is_image) {
  if (q < L.is) return -1;
  if (q > L.ie + 1) return 1;
  return (q == L.ie + 1 && upper_is_image) ? 1 : 0;
}
inline int phys_cell(const Lay& L, int q, int bc) { return L.src_cell(q, bc); }
inline int phys_face(const Lay& L, int q, int bc) { return L.src_face(q, bc); }
}  // namespace

extern "C" void orc_exchange_ghosts(const orc_params* p, const int* nbr, const int bc[3],
                                    double* const U[5], double* const Bf[3]) {
  const Lay L(p->n, p->ng);
  const int nt = L.nt, n = L.n;
  for (int pass = 0; pass < 2; ++pass)
    for (int m = 0; m < p->nmb; ++m) {
      const int* nb = nbr + 27 * m;
      // field 0: cells (5 variables); fields 1..3: faces of direction d = field - 1
      for (int fld = 0; fld < 4; ++fld) {
        const int d = fld - 1;
        const int ni = nt + (d == 0), nj = nt + (d == 1), nk = nt + (d == 2);
        for (int k = 0; k < nk; ++k)
          for (int j = 0; j < nj; ++j)
            for (int i = 0; i < ni; ++i) {
              const int ox = d == 0 ? region_face(L, i, nb[14] >= 0 || bc[0] == 0) : region_cell(L, i);
              const int oy = d == 1 ? region_face(L, j, nb[16] >= 0 || bc[1] == 0) : region_cell(L, j);
              const int oz = d == 2 ? region_face(L, k, nb[22] >= 0 || bc[2] == 0) : region_cell(L, k);
              if (ox == 0 && oy == 0 && oz == 0) continue;
              const int mb = nb[(oz + 1) * 9 + (oy + 1) * 3 + (ox + 1)];
              int ms, is_, js, ks;
              if (pass == 0) {
                if (mb < 0) continue;
                ms = mb; is_ = i - ox * n; js = j - oy * n; ks = k - oz * n;
              } else {
                if (mb >= 0) continue;
                ms = m; is_ = i; js = j; ks = k;
                if (ox != 0 && nb[13 + ox] < 0) is_ = d == 0 ? phys_face(L, i, bc[0]) : phys_cell(L, i, bc[0]);
                if (oy != 0 && nb[13 + 3 * oy] < 0) js = d == 1 ? phys_face(L, j, bc[1]) : phys_cell(L, j, bc[1]);
                if (oz != 0 && nb[13 + 9 * oz] < 0) ks = d == 2 ? phys_face(L, k, bc[2]) : phys_cell(L, k, bc[2]);
                if (is_ == i && js == j && ks == k) continue;
              }
              if (fld == 0) {
                for (int v = 0; v < 5; ++v) U[v][L.c(m, k, j, i)] = U[v][L.c(ms, ks, js, is_)];
              } else {
                Bf[d][L.f(d, m, k, j, i)] = Bf[d][L.f(d, ms, ks, js, is_)];
              }
            }
      }
    }
}

extern "C" void orc_stage_update(const orc_params* p, const double* dx, double a, double b, double dt,
                                 const double* const U0[5], const double* const B0[3],
                                 double* const U[5], double* const Bf[3],
                                 const double* const dU[5], const double* const E[3]) {
  const Lay L(p->n, p->ng);
  const int is = L.is, ie = L.ie;
  for (int m = 0; m < p->nmb; ++m) {
    const double idx = 1.0 / dx[3 * m + 0], idy = 1.0 / dx[3 * m + 1], idz = 1.0 / dx[3 * m + 2];
    for (int k = is; k <= ie; ++k)
      for (int j = is; j <= ie; ++j)
        for (int i = is; i <= ie; ++i) {
          const long c = L.c(m, k, j, i);
          for (int v = 0; v < 5; ++v) U[v][c] = a * U0[v][c] + b * (U[v][c] + dt * dU[v][c]);
        }
    // d_t B~^i = -eps^{ijk} d_j E_k on the faces of interior cells
    for (int k = is; k <= ie; ++k)
      for (int j = is; j <= ie; ++j)
        for (int i = is; i <= ie + 1; ++i) {
          const double dB = -((E[2][L.e(2, m, k, j + 1, i)] - E[2][L.e(2, m, k, j, i)]) * idy -
                              (E[1][L.e(1, m, k + 1, j, i)] - E[1][L.e(1, m, k, j, i)]) * idz);
          const long q = L.f(0, m, k, j, i);
          Bf[0][q] = a * B0[0][q] + b * (Bf[0][q] + dt * dB);
        }
    for (int k = is; k <= ie; ++k)
      for (int j = is; j <= ie + 1; ++j)
        for (int i = is; i <= ie; ++i) {
          const double dB = -((E[0][L.e(0, m, k + 1, j, i)] - E[0][L.e(0, m, k, j, i)]) * idz -
                              (E[2][L.e(2, m, k, j, i + 1)] - E[2][L.e(2, m, k, j, i)]) * idx);
          const long q = L.f(1, m, k, j, i);
          Bf[1][q] = a * B0[1][q] + b * (Bf[1][q] + dt * dB);
        }
    for (int k = is; k <= ie + 1; ++k)
      for (int j = is; j <= ie; ++j)
        for (int i = is; i <= ie; ++i) {
          const double dB = -((E[1][L.e(1, m, k, j, i + 1)] - E[1][L.e(1, m, k, j, i)]) * idx -
                              (E[0][L.e(0, m, k, j + 1, i)] - E[0][L.e(0, m, k, j, i)]) * idy);
          const long q = L.f(2, m, k, j, i);
          Bf[2][q] = a * B0[2][q] + b * (Bf[2][q] + dt * dB);
        }
  }
}

extern "C" void orc_advance_nbr(const orc_params* p, const double* dx, int integrator, int nsteps,
                                double dt, const int bc[3], const int* nbr, double* const U[5],
                                double* const Bf[3], const double* const adm[16], double* const W[8],
                                unsigned char* flag_or, int nthreads);
extern "C" int orc_advance_hooked(const orc_params* p, const double* dx, int integrator, int nsteps,
                                  double dt, const int bc[3], const int* nbr, double* const U[5],
                                  double* const Bf[3], const double* const adm[16], double* const W[8],
                                  unsigned char* flag_or, int nthreads, int (*refresh)(void*), void* user);

extern "C" void orc_advance(const orc_params* p, const double* dx, int integrator, int nsteps,
                            double dt, const int bc[3], double* const U[5], double* const Bf[3],
                            const double* const adm[16], double* const W[8],
                            unsigned char* flag_or, int nthreads) {
  orc_advance_nbr(p, dx, integrator, nsteps, dt, bc, nullptr, U, Bf, adm, W, flag_or, nthreads);
}

extern "C" void orc_advance_nbr(const orc_params* p, const double* dx, int integrator, int nsteps,
                                double dt, const int bc[3], const int* nbr, double* const U[5],
                                double* const Bf[3], const double* const adm[16], double* const W[8],
                                unsigned char* flag_or, int nthreads) {
  orc_advance_hooked(p, dx, integrator, nsteps, dt, bc, nbr, U, Bf, adm, W, flag_or, nthreads, nullptr, nullptr);
}

// The same loop with a caller hook run before every ghost fill (every stage, and the final fill): where a
// multi-rank driver refreshes the mirror blocks its neighbour table points at.  A non-zero return aborts.
extern "C" int orc_advance_hooked(const orc_params* p, const double* dx, int integrator, int nsteps,
                                  double dt, const int bc[3], const int* nbr, double* const U[5],
                                  double* const Bf[3], const double* const adm[16], double* const W[8],
                                  unsigned char* flag_or, int nthreads, int (*refresh)(void*), void* user) {
  const Lay L(p->n, p->ng);
  const long nt = L.nt, px = L.px, nb = p->nmb;
  const long ncell = nb * nt * nt * nt;
  const long nface[3] = {nb * nt * nt * px, nb * nt * (nt + 1) * nt, nb * (nt + 1) * nt * nt};
  const long nedge[3] = {nb * (nt + 1) * (nt + 1) * nt, nb * (nt + 1) * nt * px, nb * nt * (nt + 1) * px};
  std::vector<double> sU0[5], sB0[3], sdU[5], sE[3];
  std::vector<unsigned char> flag(ncell, 0);
  double* dU[5]; double* E[3]; const double* U0[5]; const double* B0[3];
  for (int v = 0; v < 5; ++v) { sU0[v].assign(ncell, 0.0); sdU[v].assign(ncell, 0.0); dU[v] = sdU[v].data(); U0[v] = sU0[v].data(); }
  for (int d = 0; d < 3; ++d) { sB0[d].assign(nface[d], 0.0); sE[d].assign(nedge[d], 0.0); E[d] = sE[d].data(); B0[d] = sB0[d].data(); }
  // Shu-Osher coefficients: U <- a U0 + b (U + dt L(U))
  const double A[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.5, 0.0}, {0.0, 0.75, 1.0 / 3.0}};
  const double B[3][3] = {{1.0, 0.0, 0.0}, {1.0, 0.5, 0.0}, {1.0, 0.25, 2.0 / 3.0}};
  const int ns = integrator;
  for (int step = 0; step < nsteps; ++step)
    for (int s = 0; s < ns; ++s) {
      const double a = A[ns - 1][s], b = B[ns - 1][s];
      if (refresh) { const int hr = refresh(user); if (hr != 0) return hr; }
      if (nbr) orc_exchange_ghosts(p, nbr, bc, U, Bf); else orc_fill_ghosts(p, bc, U, Bf);
      orc_rhs_blend(p, dx, U, Bf, adm, W, 0, dt, s == 0 ? nullptr : U0, a, b, dU, E, flag.data(),
                    nullptr, nthreads);
      if (flag_or) for (long c = 0; c < ncell; ++c) flag_or[c] |= flag[c];
      if (s == 0 && ns > 1) {
        for (int v = 0; v < 5; ++v) std::memcpy(sU0[v].data(), U[v], sizeof(double) * ncell);
        for (int d = 0; d < 3; ++d) std::memcpy(sB0[d].data(), Bf[d], sizeof(double) * nface[d]);
      }
      // for s == 0, a == 0: the register is not read (0 * x would turn inf/nan into nan)
      if (s == 0) {
        const double* Uc[5] = {U[0], U[1], U[2], U[3], U[4]};
        const double* Bc[3] = {Bf[0], Bf[1], Bf[2]};
        orc_stage_update(p, dx, 0.0, 1.0, dt, Uc, Bc, U, Bf, dU, E);
      } else {
        orc_stage_update(p, dx, a, b, dt, U0, B0, U, Bf, dU, E);
      }
    }
  if (refresh) { const int hr = refresh(user); if (hr != 0) return hr; }
  if (nbr) orc_exchange_ghosts(p, nbr, bc, U, Bf); else orc_fill_ghosts(p, bc, U, Bf);
  return 0;
}
