// ak_flux_pencil.cuh — K2 for the y and z sweeps, reconstruct-once on whole pencils (round 2).
//
// A block owns WI neighbouring pencils along the sweep direction: the cells c = 0 .. nt-1 of WI
// consecutive x-lanes at one fixed transverse index.  One tensor-map TMA box copy per field
// (cp.async.bulk.tensor.3d, SASS UTMALDG) brings the [nt][WI] tile of each of the 7 reconstructed
// fields and 10 metric fields into shared memory — 17 copies per block, issued by one thread, against
// the ~200 one-row bulk copies per tile of k_flux_tma.  The box is dense in shared memory ([c][lane]),
// so thread t = r * WI + lane reads its five stencil cells at sm[t + s * WI]: consecutive threads,
// consecutive addresses, no bank conflicts, and q^+ is handed to the thread of the next cell at
// sQ[t - WI] the same way.
//
// One thread per CELL c = 2 + r (r = 0 .. n+3): both face values of the cell from ONE set of smoothness
// indicators (WENO-Z: one reciprocal and the beta's shared by q^- and q^+), then the face on its lower
// side (faces 3 .. n+5; the thread row r = 0 has none: 1 idle row in n+4 instead of 1 in 8 for the
// tile-based variants of round 1).  Same operations per value as k_flux_tma / the oracle: same bits.
//
// Tensor maps (host: ak_api.cu, cuTensorMapEncodeTiled): every cell field is the rank-3 tensor
// (i: nt, j: nt, K = m * nt + k) of doubles; the y sweep uses the box (WI, nt, 1) at (i0, 0, m nt + k),
// the z sweep the box (WI, 1, nt) at (i0, j, m nt).  n even keeps every stride a multiple of 16 B.
#pragma once
#include <cuda.h>
#include "ak_flux_tma.cuh"

namespace ak {

#ifndef AK_PENCIL_MAXT
#define AK_PENCIL_MAXT 224    // threads: WI * (n + 4) rounded up to warps; 6 lanes x 36 cells for 32^3 blocks
#endif
#ifndef AK_PENCIL_MINB
#define AK_PENCIL_MINB 3
#endif

typedef TileMaps PencilMaps;   // the same 17 fields, boxes of WI lanes x nt cells

// tile_d: doubles per field tile in shared memory (nt * WI rounded up to a multiple of 16: 128-byte tiles)
template <int DIR, int RECON, int EOS = 0>
__global__ void __launch_bounds__(AK_PENCIL_MAXT, AK_PENCIL_MINB)
k_flux_pencil(const __grid_constant__ Par P, const __grid_constant__ Fields f,
              const __grid_constant__ PencilMaps maps, int WI, int tile_d, int i_first, int ntile_i) {
  static_assert(DIR == 1 || DIR == 2, "pencil kernel: y and z sweeps");
  extern __shared__ __align__(128) double sm[];
  __shared__ uint64_t mbar, mbarM;       // primitives / metric: the metric lands while the cells are reconstructed
  const int nt = P.nt, e = P.n + 2, t = threadIdx.x;
  double* sW = sm;                        // [7][tile_d]
  double* sM = sm + 7 * tile_d;           // [10][tile_d]
  double* sQ = sm + 17 * tile_d;          // [7][blockDim.x]  q^+ of every cell
  int bid = blockIdx.x;
  const int ti = bid % ntile_i; bid /= ntile_i;
  const int o = bid % e + P.is - 1;       // fixed transverse index: k (y sweep) or j (z sweep)
  const int m = bid / e;
  const int i0 = i_first + ti * WI;       // first x-lane of the tile
  __shared__ unsigned nzacc;
  if (t == 0) { mbar_init(&mbar, 1); mbar_init(&mbarM, 1); nzacc = 0; }
  __syncthreads();
  if (t == 0) {
    const int c1 = DIR == 1 ? 0 : o, c2 = DIR == 1 ? m * nt + o : m * nt;
    mbar_arrive_expect_tx(&mbar, (unsigned)(7 * nt * WI * sizeof(double)));
#pragma unroll
    for (int v = 0; v < 7; ++v) tma_load_3d(sW + v * tile_d, &maps.w[v], i0, c1, c2, &mbar);
    mbar_arrive_expect_tx(&mbarM, (unsigned)(10 * nt * WI * sizeof(double)));
#pragma unroll
    for (int q = 0; q < 10; ++q) tma_load_3d(sM + q * tile_d, &maps.m[q], i0, c1, c2, &mbarM);
  }
  // ---- this thread's cell: row r along the sweep, lane l along x
  const int r = t / WI, l = t - r * WI;
  const int cc = 2 + r;                   // cell index along the sweep; its lower face is face cc
  const int ii = i0 + l;
  const bool active = r < P.n + 4 && ii >= P.is - 1 && ii <= P.ie + 1;
  const bool has_face = active && r >= 1;
  const Ix ix{nt, P.px};
  long long fi = 0;
  double Bfd = 0.0;
  if (has_face) {
    fi = DIR == 1 ? ix.face(1, m, o, cc, ii) : ix.face(2, m, cc, o, ii);
    Bfd = __ldg(f.Bf[DIR] + fi);
  }
  mbar_wait(&mbar, 0);
  const unsigned nzm = ((RECON != 0 && (P.shortcuts & 1)) || (P.shortcuts & 4))
                           ? tile_nonzero_mask(sW, tile_d, nt * WI, &nzacc, (__double_as_longlong(Bfd) != 0LL) ? 0x80u : 0u)
                           : ALWAYS_NZ;
  const bool stat = tile_is_static(P, nzm);          // block-uniform
  const unsigned rzm = (P.shortcuts & 1) ? nzm : ALWAYS_NZ;   // which slots are reconstructed
  double qm[7];
  if (active) {
#pragma unroll
    for (int v = 0; v < 7; ++v) {
      const double* w = sW + v * tile_d + t;     // cell cc-2 of this lane; cells cc-2 .. cc+2 at stride WI
      double qp;
      if (!((rzm >> v) & 1u)) { qm[v] = qp = 0.0; }          // the field is +0.0 on the whole tile
      else if (RECON == 0) { qm[v] = qp = w[2 * WI]; }
      else recon<RECON>(w[0], w[WI], w[2 * WI], w[3 * WI], w[4 * WI], qm[v], qp);
      sQ[v * (int)blockDim.x + t] = qp;
    }
  }
  double mL[10], mR[10];
  mbar_wait(&mbarM, 0);
  if (has_face) {
#pragma unroll
    for (int q = 0; q < 10; ++q) {
      const double* g = sM + q * tile_d + WI + t;   // cell cc-1, then cell cc
      mL[q] = g[0];
      mR[q] = g[WI];
    }
  }
  __syncthreads();                        // every q^+ is written
  double sL[7], Fo[7];
  if (has_face) {
#pragma unroll
    for (int v = 0; v < 7; ++v) sL[v] = sQ[v * (int)blockDim.x + t - WI];
  }
  FaceGeo G;
  if (has_face) face_geometry<DIR>(mL, mR, G);
  if (stat) {                             // static unmagnetised tile: nothing to park, no barrier
    if (!has_face) return;
    face_flux_static<DIR, EOS>(P, P.riemann, G, sL, qm, Fo);
#pragma unroll
    for (int v = 0; v < 7; ++v) f.F[7 * DIR + v][fi] = Fo[v];
    return;
  }
  __syncthreads();                        // tile and q^+ are spent: the allocation becomes parking space
  if (!has_face) return;
  {
    volatile double* pR = sm + 14 * (int)blockDim.x + t;
#pragma unroll
    for (int v = 0; v < 7; ++v) pR[v * (int)blockDim.x] = qm[v];
  }
  face_flux_parked<DIR, EOS>(P, P.riemann, G, sL, sm + 14 * (int)blockDim.x + t, (int)blockDim.x, Bfd, Fo, sm + t,
                             (int)blockDim.x);
#pragma unroll
  for (int v = 0; v < 7; ++v) f.F[7 * DIR + v][fi] = Fo[v];
}

}  // namespace ak
