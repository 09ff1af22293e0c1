// ak_source.cuh — K6: flux divergence + geometric source terms (Eq. 9) on the
// interior cells.  DESIGN.md §3 O9: sources from the cell-centred primitives of the stage
// input (reading R22), second-order centred metric derivatives (reading R20).
#pragma once
#include "ak_kernels.cuh"

namespace ak {

#ifndef AK_SRC_MINB
#define AK_SRC_MINB 4
#endif
// k_div_src runs at 128 registers (16 warps per SM), and the compiler issues the loads of the metric, rho and P
// only after the flux differences: an exposed DRAM latency per group.  Register-free prefetches of those
// centre lines before the first load: div+sources 2.15 -> 1.94 ms on C4.  Measured and NOT done: the same for
// K_ij (+16: no gain), for the y/z neighbours of the metric that the centred differences read (before the first
// load: 2.08; after the centre loads, in flight during the stress-tensor arithmetic: 2.2-3.4 ms — they evict
// the lines the other warps are waiting for), and the metric lines of k_fofc_test (2.01 -> 2.07 ms).
// 0: off; 4 | 1: prefetch.global.L1; 4 | 2: prefetch.global.L2 (same time); +16: K_ij as well.
#ifndef AK_SRC_PREFETCH
#define AK_SRC_PREFETCH 5
#endif
__device__ __forceinline__ void src_prefetch(const void* p) {
#if (AK_SRC_PREFETCH & 3) == 1
  asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
#elif (AK_SRC_PREFETCH & 3) == 2
  asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
#endif
}
// Part (6) for ONE interior cell c of block m, given the flux differences div[v] (div_flux) of the five hydro
// variables: dU~/dt = -div + geometric sources (Eq. 9); also the matter epilogue.  Called by k_div_src (one
// thread per interior cell), by the fused FOFC-test kernel (k_fofc_test<EOS, STRIDE, true>, which has the
// same div in registers) and by k_src_fix (cells next to re-fluxed faces).
template <int EOS>
__device__ __forceinline__ void div_src_cell(const Par& P, const Fields& f, int m, long long c, const double div[5]) {
  const double dxm[3] = {f.dx[3 * m + 0], f.dx[3 * m + 1], f.dx[3 * m + 2]};
  const double h2[3] = {0.5 / dxm[0], 0.5 / dxm[1], 0.5 / dxm[2]};
  double du[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) du[v] = -div[v];

  Met3 g, gu;
  load_met3(f, c, g);
  double det, sdet;
  metric_inverse(g, det, sdet, gu);
  const double isd = 1.0 / sdet;
  const double rho = f.W[0][c], pr = f.W[4][c];
  const unsigned zf = (f.zflags && (P.shortcuts & 1)) ? f.zflags[m] : 0xffu;    // clear bit: the field is +0.0 in this block
  double u[3], Bt[3];
#pragma unroll
  for (int v = 0; v < 3; ++v) {
    u[v] = ((zf >> (1 + v)) & 1u) ? f.W[1 + v][c] : 0.0;
    Bt[v] = ((zf >> (5 + v)) & 1u) ? f.W[5 + v][c] : 0.0;
  }
  const double B[3] = {Bt[0] * isd, Bt[1] * isd, Bt[2] * isd};
  double cons[5];
  prim2cons<EOS>(P, g, rho, u, pr, B, cons);
  double ul[3], Bl[3];
  lower(g, u, ul);
  const double usq = dot3(ul, u);
  const double Wl = sqrt(1.0 + usq), iW = 1.0 / Wl;
  lower(g, B, Bl);
  const double B2 = dot3(Bl, B);
  const double vl[3] = {ul[0] * iW, ul[1] * iW, ul[2] * iW};
  const double Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2];
  const double b2 = B2 * iW * iW + Bv * Bv;
  const double bl[3] = {Bl[0] * iW + Bv * ul[0], Bl[1] * iW + Bv * ul[1], Bl[2] * iW + Bv * ul[2]};
  const double h = EOS == 0 ? 1.0 + P.Gam / (P.Gam - 1.0) * (pr / rho) : 1.0 + eos_hm1<EOS>(P, rho, pr);
  const double Ptot = pr + 0.5 * b2;
  const double wt = rho * h + b2;
  // S_ij = (rho h + b^2) u_i u_j + Ptot gamma_ij - b_i b_j
  const double gd[6] = {g.xx, g.xy, g.xz, g.yy, g.yz, g.zz};
  const double gi6[6] = {gu.xx, gu.xy, gu.xz, gu.yy, gu.yz, gu.zz};
  constexpr int I6[6] = {0, 0, 0, 1, 1, 2}, J6[6] = {0, 1, 2, 1, 2, 2};
  double Sdd[3][3], gim[3][3];
#pragma unroll
  for (int q = 0; q < 6; ++q) {
    const double s = wt * ul[I6[q]] * ul[J6[q]] + Ptot * gd[q] - bl[I6[q]] * bl[J6[q]];
    Sdd[I6[q]][J6[q]] = s; Sdd[J6[q]][I6[q]] = s;
    gim[I6[q]][J6[q]] = gi6[q]; gim[J6[q]][I6[q]] = gi6[q];
  }
  // fused epilogue (S:§8(f) rank 4): the matter terms a spacetime (Z4c) right-hand side needs
  // are E = tau + D, S_i and S_ij = T_ij of exactly this state -- written here, from the registers that hold
  // them, instead of by a second pass over W and the metric (k_matter; same expressions, same bits)
  if (f.M[0]) {
    f.M[0][c] = cons[4] + cons[0];
    f.M[1][c] = cons[1]; f.M[2][c] = cons[2]; f.M[3][c] = cons[3];
    f.M[4][c] = Sdd[0][0]; f.M[5][c] = Sdd[0][1]; f.M[6][c] = Sdd[0][2];
    f.M[7][c] = Sdd[1][1]; f.M[8][c] = Sdd[1][2]; f.M[9][c] = Sdd[2][2];
  }
  // S^{ij} = gamma^{ik} S_kl gamma^{lj}
  double T[3][3], Suu[6];
#pragma unroll
  for (int aa = 0; aa < 3; ++aa)
#pragma unroll
    for (int l = 0; l < 3; ++l)
      T[aa][l] = gim[aa][0] * Sdd[0][l] + gim[aa][1] * Sdd[1][l] + gim[aa][2] * Sdd[2][l];
#pragma unroll
  for (int q = 0; q < 6; ++q)
    Suu[q] = T[I6[q]][0] * gim[0][J6[q]] + T[I6[q]][1] * gim[1][J6[q]] + T[I6[q]][2] * gim[2][J6[q]];
  const double Sl[3] = {cons[1], cons[2], cons[3]};
  const double Su[3] = {gu.xx * Sl[0] + gu.xy * Sl[1] + gu.xz * Sl[2],
                        gu.xy * Sl[0] + gu.yy * Sl[1] + gu.yz * Sl[2],
                        gu.xz * Sl[0] + gu.yz * Sl[1] + gu.zz * Sl[2]};
  const double Een = cons[4] + cons[0];
  const double alp = __ldg(f.adm[6] + c);
  const long long st3[3] = {1, P.nt, (long long)P.nt * P.nt};
  double dalp[3];
#pragma unroll
  for (int aa = 0; aa < 3; ++aa) {
    const long long s = st3[aa];
    dalp[aa] = (__ldg(f.adm[6] + c + s) - __ldg(f.adm[6] + c - s)) * h2[aa];
    double dg[6], dbeta[3];
#pragma unroll
    for (int q = 0; q < 6; ++q) dg[q] = (__ldg(f.adm[q] + c + s) - __ldg(f.adm[q] + c - s)) * h2[aa];
#pragma unroll
    for (int bb = 0; bb < 3; ++bb)
      dbeta[bb] = (__ldg(f.adm[7 + bb] + c + s) - __ldg(f.adm[7 + bb] + c - s)) * h2[aa];
    const double Sdg = Suu[0] * dg[0] + 2.0 * (Suu[1] * dg[1]) + 2.0 * (Suu[2] * dg[2]) + Suu[3] * dg[3] +
                       2.0 * (Suu[4] * dg[4]) + Suu[5] * dg[5];
    const double Sdb = Sl[0] * dbeta[0] + Sl[1] * dbeta[1] + Sl[2] * dbeta[2];
    du[1 + aa] = du[1 + aa] + sdet * (0.5 * alp * Sdg + Sdb - Een * dalp[aa]);
  }
  const double KS = __ldg(f.adm[10] + c) * Suu[0] + 2.0 * (__ldg(f.adm[11] + c) * Suu[1]) +
                    2.0 * (__ldg(f.adm[12] + c) * Suu[2]) + __ldg(f.adm[13] + c) * Suu[3] +
                    2.0 * (__ldg(f.adm[14] + c) * Suu[4]) + __ldg(f.adm[15] + c) * Suu[5];
  const double Sda = Su[0] * dalp[0] + Su[1] * dalp[1] + Su[2] * dalp[2];
  du[4] = du[4] + sdet * (alp * KS - Sda);
#pragma unroll
  for (int v = 0; v < 5; ++v) st_out<8>(f.dU[v] + c, du[v]);
}

template <int EOS = 0, bool STRIDE = false>
__global__ void __launch_bounds__(128, AK_SRC_MINB) k_div_src(const __grid_constant__ Par P,
                                                 const __grid_constant__ Fields f) {
  const int n = P.n;
  const long long per = (long long)n * n * n;
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  do {
  if (idx >= per * P.nmb) return;
  const int m = (int)(idx / per);
  int r = (int)(idx - (long long)m * per);
  const int i = r % n + P.is; r /= n;
  const int j = r % n + P.is;
  const int k = r / n + P.is;
  const Ix ix{P.nt, P.px};
  const long long c = ix.cell(m, k, j, i);
#if AK_SRC_PREFETCH
  {
#if AK_SRC_PREFETCH & 16
#pragma unroll
    for (int q = 10; q < 16; ++q) src_prefetch(f.adm[q] + c);
#endif
#if AK_SRC_PREFETCH & 4
#pragma unroll
    for (int q = 0; q < 10; ++q) src_prefetch(f.adm[q] + c);
    src_prefetch(f.W[0] + c); src_prefetch(f.W[4] + c);
#endif
  }
#endif
  const double idx3[3] = {1.0 / f.dx[3 * m + 0], 1.0 / f.dx[3 * m + 1], 1.0 / f.dx[3 * m + 2]};
  double div[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) div[v] = div_flux(f, ix, v, m, k, j, i, idx3);
  div_src_cell<EOS>(P, f, m, c, div);
  idx += (long long)gridDim.x * blockDim.x;
  } while (STRIDE);
}

// Part (6) again for the interior cells that have a re-fluxed face: the flagged cells of the FOFC list and
// their six face neighbours (a face is redone iff one of its two cells is flagged).  The fused FOFC-test
// kernel wrote dU~/dt of every interior cell from the high-order fluxes; these cells are recomputed from the
// final ones with the same per-cell function, so every value equals what k_div_src after the re-flux would
// write.  A cell reached from two flagged neighbours is written twice with the same bits.
template <int EOS = 0>
__global__ void __launch_bounds__(128, AK_SRC_MINB) k_src_fix(const __grid_constant__ Par P,
                                                              const __grid_constant__ Fields f) {
  const unsigned cnt = f.count[3];
  const Ix ix{P.nt, P.px};
  const long long nt = P.nt;
  for (unsigned long long e = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; e < 7ull * cnt;
       e += (unsigned long long)gridDim.x * blockDim.x) {
    const unsigned which = (unsigned)(e / cnt);                 // 0: the cell itself, 1..6: -x +x -y +y -z +z
    long long c = (long long)f.list[e - (unsigned long long)which * cnt];
    const long long st = which == 0 ? 0 : (which <= 2 ? 1 : (which <= 4 ? nt : nt * nt));
    c += (which & 1u) ? -st : st;
    const int i = (int)(c % nt);
    const long long row = c / nt;
    const int j = (int)(row % nt);
    const long long mk = row / nt;
    const int k = (int)(mk % nt), m = (int)(mk / nt);
    if (i < P.is || i > P.ie || j < P.is || j > P.ie || k < P.is || k > P.ie) continue;     // interior cells only
    const double idx3[3] = {1.0 / f.dx[3 * m + 0], 1.0 / f.dx[3 * m + 1], 1.0 / f.dx[3 * m + 2]};
    double div[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) div[v] = div_flux(f, ix, v, m, k, j, i, idx3);
    div_src_cell<EOS>(P, f, m, c, div);
  }
}

// ---- matter terms for a spacetime solver: E = tau + D, S_i, S_ij = T_ij, undensitised,
// at every stored cell from the cell-centred primitives ----------------------------------------------
struct MatterOut { double* q[10]; };   // E, Sx, Sy, Sz, Sxx, Sxy, Sxz, Syy, Syz, Szz

template <int EOS = 0>
__global__ void __launch_bounds__(128) k_matter(const __grid_constant__ Par P, const __grid_constant__ Fields f,
                                                const __grid_constant__ MatterOut o) {
  const long long ncell = (long long)P.nmb * P.nt * P.nt * P.nt;
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  Met3 g, gu;
  load_met3(f, c, g);
  double det, sdet;
  metric_inverse(g, det, sdet, gu);
  const double isd = 1.0 / sdet;
  const double rho = f.W[0][c], pr = f.W[4][c];
  const double u[3] = {f.W[1][c], f.W[2][c], f.W[3][c]};
  const double B[3] = {f.W[5][c] * isd, f.W[6][c] * isd, f.W[7][c] * isd};
  double cons[5];
  prim2cons<EOS>(P, g, rho, u, pr, B, cons);
  double ul[3], Bl[3];
  lower(g, u, ul);
  const double usq = dot3(ul, u);
  const double iW = 1.0 / sqrt(1.0 + usq);
  lower(g, B, Bl);
  const double B2 = dot3(Bl, B);
  const double vl[3] = {ul[0] * iW, ul[1] * iW, ul[2] * iW};
  const double Bv = B[0] * vl[0] + B[1] * vl[1] + B[2] * vl[2];
  const double b2 = B2 * iW * iW + Bv * Bv;
  const double bl[3] = {Bl[0] * iW + Bv * ul[0], Bl[1] * iW + Bv * ul[1], Bl[2] * iW + Bv * ul[2]};
  const double h = EOS == 0 ? 1.0 + P.Gam / (P.Gam - 1.0) * (pr / rho) : 1.0 + eos_hm1<EOS>(P, rho, pr);
  const double Ptot = pr + 0.5 * b2;
  const double wt = rho * h + b2;
  o.q[0][c] = cons[4] + cons[0];
  o.q[1][c] = cons[1]; o.q[2][c] = cons[2]; o.q[3][c] = cons[3];
  const double gd[6] = {g.xx, g.xy, g.xz, g.yy, g.yz, g.zz};
  constexpr int I6[6] = {0, 0, 0, 1, 1, 2}, J6[6] = {0, 1, 2, 1, 2, 2};
#pragma unroll
  for (int q = 0; q < 6; ++q) o.q[4 + q][c] = wt * ul[I6[q]] * ul[J6[q]] + Ptot * gd[q] - bl[I6[q]] * bl[J6[q]];
}

}  // namespace ak
