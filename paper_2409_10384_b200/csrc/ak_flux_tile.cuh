// ak_flux_tile.cuh — K2, tiled: reconstruct once per cell, exchange the right-face states and the
// cell metric through shared memory, then one Riemann problem per face.
//
// A CUDA block covers NA cells along the sweep direction d times NB pencils (a pencil = a line of
// cells along d at fixed transverse indices).  Thread (a, b):
//   phase 1  reconstructs cell a of pencil b for the seven variables (both faces from one set of
//            smoothness indicators), keeps q^- in registers, writes q^+ and the cell's ten metric
//            values to shared memory;
//   phase 2  (a >= 1) solves the face between cells a-1 and a:  L = q^+ of thread (a-1, b) from
//            shared memory, R = its own q^-.
// DIR = x: NA = n+4 is the whole pencil (a fastest: threads run along x, coalesced), NB rows.
// DIR = y,z: NB = 32 pencils (b fastest: lanes run along x), NA = 8 cells -> 7 faces per tile, the
//            tiles along d overlap by one cell.
// Shared memory: 17 doubles per thread, index [field][thread]: conflict-free (stride-1 doubles).
#pragma once
#include "ak_kernels.cuh"

namespace ak {

#ifndef AK_TILE_MINB
#define AK_TILE_MINB 2
#endif
constexpr int TILE_MAX_THREADS = 320;
constexpr int TILE_SMEM_DOUBLES = 17;

template <int DIR, int RECON>
__global__ void __launch_bounds__(TILE_MAX_THREADS, AK_TILE_MINB)
k_flux_tile(const __grid_constant__ Par P, const __grid_constant__ Fields f, int NA, int NB) {
  extern __shared__ double sm[];
  const int BD = NA * NB;
  const int t = threadIdx.x;
  int a, b;
  if (DIR == 0) { a = t % NA; b = t / NA; } else { b = t % NB; a = t / NB; }
  const int off = DIR == 0 ? 1 : NB;                 // shared-memory distance to thread (a-1, b)
  const int e = P.n + 2;
  const long long np_all = (long long)P.nmb * e * e;
  const long long p = (long long)blockIdx.x * NB + b;
  const int cd = P.is - 2 + (NA - 1) * (int)blockIdx.y + a;   // index along d of this thread's cell
  const bool valid = p < np_all && cd <= P.ie + 2;
  constexpr int t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  double qm[7], mR[10];
  long long c = 0;
  int m = 0, i = 0, j = 0, k = 0;
  if (valid) {
    m = (int)(p / (e * e));
    const int r = (int)(p - (long long)m * e * e);
    const int u = r % e + P.is - 1, w = r / e + P.is - 1;
    if (DIR == 0) { i = cd; j = u; k = w; }
    else if (DIR == 1) { i = u; j = cd; k = w; }
    else { i = u; j = w; k = cd; }
    const Ix ix{P.nt, P.px};
    c = ix.cell(m, k, j, i);
    const long long s = DIR == 0 ? 1 : (DIR == 1 ? P.nt : (long long)P.nt * P.nt);
    load_met10(f, c, mR);
    const int var[7] = {0, 1, 2, 3, 4, 5 + t1, 5 + t2};
#pragma unroll
    for (int v = 0; v < 7; ++v) {
      const double* w5 = f.W[var[v]] + c;
      double qp;
      if (RECON == 0) {
        qm[v] = qp = w5[0];
      } else {
        recon<RECON>(w5[-2 * s], w5[-s], w5[0], w5[s], w5[2 * s], qm[v], qp);
      }
      sm[v * BD + t] = qp;
    }
#pragma unroll
    for (int q = 0; q < 10; ++q) sm[(7 + q) * BD + t] = mR[q];
  }
  __syncthreads();
  if (!valid || a == 0) return;
  double sL[7], mL[10], Fo[7];
#pragma unroll
  for (int v = 0; v < 7; ++v) sL[v] = sm[v * BD + t - off];
#pragma unroll
  for (int q = 0; q < 10; ++q) mL[q] = sm[(7 + q) * BD + t - off];
  const Ix ix{P.nt, P.px};
  const long long fi = ix.face(DIR, m, k, j, i);
  face_flux<DIR, true>(P, P.riemann, mL, mR, sL, qm, __ldg(f.Bf[DIR] + fi), Fo);
#pragma unroll
  for (int v = 0; v < 7; ++v) f.F[7 * DIR + v][fi] = Fo[v];
}

}  // namespace ak
