// ak_flux_static.cuh — K2 for tiles that are static and unmagnetised as a whole (round 2).
//
// k_con2prim records per ROW of cells whether any u^i or any face B~ of the row holds a value that is not +0.0
// (Fields::rowflag).  A tile none of whose rows does — static atmosphere without field: 72 % of C4's MeshBlocks
// and four tiles in five of the others — needs of the 17 staged fields only rho, P and the ten metric fields,
// and of the Riemann solve only static_side() (ak_flux.cuh: Eq. 8 with W = 1, v = 0, B = 0 substituted term by
// term, the same bits as the general code on such data).  This kernel does just that: 12 tensor-map box copies
// per tile, 33 KB of shared memory instead of 52 KB and no general side_state() in the register budget, so that
// 5 blocks are resident on an SM instead of 3 and the tile-load latency — the top stall of the default-mode
// sweeps (profiles/r2_final.md) — is covered.  k_split_tiles makes, per direction, the two lists of tiles
// (static / general) on the device; both sweep kernels are launched over the full grid and a block whose list
// entry does not exist returns at once.
//
// Same tiles as k_flux_tma: x: NA rows of n+3 faces; y, z: NA face rows of n+2 lanes.
#pragma once
#include "ak_flux_tma.cuh"

namespace ak {

#ifndef AK_STATIC_MINB
#define AK_STATIC_MINB 4
#endif
#ifndef AK_STATIC_PLAIN_DIV
#define AK_STATIC_PLAIN_DIV 1   // rho and P are never zero: WENO-Z's quotients by plain division (see recon<>)
#endif
#ifndef AK_STATIC_ONCE_MASK
#define AK_STATIC_ONCE_MASK 1   // bit d: the sweep of direction d reconstructs every cell once (below)
#endif

// Tile lists.  One thread per tile of one direction: the tile is static iff none of the rows of cells it stages
// has its row flag set (conservative: the flags cover all three u^i and all face fields, the tile test of the
// general kernel only what that direction uses; a static tile that lands in the general list is still
// recognised there).  shape[d] = {NA, tiles} of direction d (the launcher's tiling).
struct TileShapes { int NA[3], tiles[3]; };
__global__ void __launch_bounds__(256) k_split_tiles(const __grid_constant__ Par P, const unsigned char* __restrict__ rowflag,
                                                     const __grid_constant__ TileShapes sh, unsigned* __restrict__ tlist,
                                                     unsigned* __restrict__ tcount, unsigned tcap) {
  const int e = P.n + 2, nt = P.nt;
  const int d = blockIdx.y;
  const int tiles = sh.tiles[d], NA = sh.NA[d];
  const long long ntile = (long long)P.nmb * e * tiles;
  const long long tile = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  bool live = tile < ntile, any = false;
  if (live) {
    long long b = tile;
    const int td = (int)(b % tiles); b /= tiles;
    const int o = (int)(b % e) + P.is - 1;
    const int m = (int)(b / e);
    const int nfd = d == 0 ? e : P.n + 3;
    const int d0 = P.is - 1 + td * NA;
    const int na = min(NA, P.is - 1 + nfd - d0);
    // rows of cells the tile stages: x: (k = o, j in [d0, d0+na)); y: (k = o, j in [d0-3, d0+na+2));
    // z: (k in [d0-3, d0+na+2), j = o)
    const int r0 = d == 0 ? d0 : d0 - 3, nr = d == 0 ? na : na + 5;
    const unsigned char* rf = rowflag + (size_t)m * nt * nt;
    for (int r = r0; r < r0 + nr; ++r) any |= (d == 2 ? rf[r * nt + o] : rf[o * nt + r]) != 0;
  }
  // append: one atomic per thread block and list, so that 256 consecutive tiles (~1.5 MeshBlocks' worth of one
  // direction) stay consecutive in their list and run together -- neighbouring tiles share halo rows, L2 lines
  // and DRAM pages (appending warp by warp leaves the lists in the order warps happen to arrive: +0.03 ms per stage)
  __shared__ unsigned wcnt[2][8], wbase[2][8];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  unsigned bal[2];
#pragma unroll
  for (int w = 0; w < 2; ++w) {
    bal[w] = __ballot_sync(0xffffffffu, live && (any == (w == 1)));
    if (lane == 0) wcnt[w][wid] = (unsigned)__popc(bal[w]);
  }
  __syncthreads();
  if (threadIdx.x < 2) {
    const int w = threadIdx.x;
    unsigned tot = 0;
    for (int q = 0; q < 8; ++q) { wbase[w][q] = tot; tot += wcnt[w][q]; }
    const unsigned base = tot ? atomicAdd(tcount + 2 * d + w, tot) : 0u;
    for (int q = 0; q < 8; ++q) wbase[w][q] += base;
  }
  __syncthreads();
  if (live) {
    const int w = any ? 1 : 0;
    tlist[(size_t)(2 * d + w) * tcap + wbase[w][wid] + __popc(bal[w] & ((1u << lane) - 1u))] = (unsigned)tile;
  }
}

template <int DIR, int RECON, int EOS = 0>
__global__ void __launch_bounds__(TMA_THREADS, AK_STATIC_MINB)
k_flux_static(const __grid_constant__ Par P, const __grid_constant__ Fields f, int NA,
              const __grid_constant__ TileMaps maps) {
  extern __shared__ __align__(128) double sm[];
  __shared__ uint64_t mbar, mbarM;
  const int nt = P.nt, e = P.n + 2, t = threadIdx.x;
  const int maxW = DIR == 0 ? NA : NA + 5, maxM = DIR == 0 ? NA : NA + 1;
  const int slotW = tile_slot(maxW, nt), slotM = tile_slot(maxM, nt);
  double* sW = sm;                             // [2][slotW]   rho, P
  double* sM = sm + 2 * slotW;                 // [10][slotM]
  const int nfd = DIR == 0 ? e : P.n + 3;
  const int tiles = (nfd + NA - 1) / NA;
  if (blockIdx.x >= f.tcount[2 * DIR]) return; // fewer static tiles than the grid provides for (block-uniform)
  int bid = (int)f.tlist[(size_t)(2 * DIR) * f.tcap + blockIdx.x];
  const int td = bid % tiles; bid /= tiles;
  const int o = bid % e + P.is - 1;
  const int m = bid / e;
  const int d0 = P.is - 1 + td * NA;
  const int na = min(NA, P.is - 1 + nfd - d0);
  const Ix ix{nt, P.px};
  const unsigned rowb = (unsigned)(nt * sizeof(double));
  if (t == 0) { mbar_init(&mbar, 1); mbar_init(&mbarM, 1); }
  __syncthreads();
  if (t < 32) {                                // lanes 0..11 of warp 0: one field each
    if (t == 0) {
      mbar_arrive_expect_tx(&mbar, (unsigned)(2 * maxW) * rowb);
      mbar_arrive_expect_tx(&mbarM, (unsigned)(10 * maxM) * rowb);
    }
    __syncwarp();
    const int K = DIR == 2 ? m * nt + d0 : m * nt + o;
    if (t < 2) {
      const int cW1 = DIR == 0 ? d0 : (DIR == 1 ? d0 - 3 : o), cW2 = DIR == 2 ? K - 3 : K;
      tma_load_3d(sW + (size_t)t * slotW, &maps.w[t == 0 ? 0 : 4], 0, cW1, cW2, &mbar);
    } else if (t < 12) {
      const int cM1 = DIR == 0 ? d0 : (DIR == 1 ? d0 - 1 : o), cM2 = DIR == 2 ? K - 1 : K;
      tma_load_3d(sM + (size_t)(t - 2) * slotM, &maps.m[t - 2], 0, cM1, cM2, &mbarM);
    }
  }
  // One two-sided reconstruction per cell instead of two one-sided ones per face (they share the smoothness
  // indicators: ~160 against 2 x 110 fp64 instructions for WENO-Z): a thread reconstructs the cell on the UPPER
  // side of its face, keeps q^- as its right state and hands q^+ to the thread of the next face through xch.
  //   x   : one thread per cell i in [is-2, ie+2] of a row; the first cell of a row has no face of its own;
  //   y, z: one thread per face; the threads of tile row 0 also reconstruct the cell below the tile (one-sided).
  constexpr bool ONCE = (AK_STATIC_ONCE_MASK >> DIR) & 1;
  __shared__ double xch[ONCE ? 2 : 1][ONCE ? TMA_THREADS : 1];
  const int nfi = DIR == 0 ? (ONCE ? P.n + 4 : P.n + 3) : e;      // threads per tile row
  const int a = t / nfi, ii = t - a * nfi + (DIR == 0 && ONCE ? P.is - 2 : P.is - 1);
  const bool active = a < na;
  const bool has_face = active && (DIR != 0 || ii >= P.is - 1);
  long long fi = 0;
  if (has_face) {
    if (DIR == 0) fi = ix.face(0, m, o, d0 + a, ii);
    else if (DIR == 1) fi = ix.face(1, m, o, d0 + a, ii);
    else fi = ix.face(2, m, d0 + a, o, ii);
  }
  mbar_wait(&mbar, 0);
  double sL[7], sR[7];
#pragma unroll
  for (int v = 0; v < 7; ++v) { sL[v] = 0.0; sR[v] = 0.0; }
  if (active) {
#pragma unroll
    for (int v2 = 0; v2 < 2; ++v2) {
      const int v = v2 == 0 ? 0 : 4;
      // x: w[0] = cell ii-3 (w[3] is this thread's cell); y, z: w[0] = shared row a (the upper cell is row a+3)
      const double* w = DIR == 0 ? sW + (size_t)v2 * slotW + a * nt + ii - 3 : sW + (size_t)v2 * slotW + a * nt + ii;
      const int s = DIR == 0 ? 1 : nt;
      if (RECON == 0) {
        sL[v] = w[2 * s]; sR[v] = w[3 * s];
      } else if (!ONCE) {
        const double q0 = w[0], q1 = w[s], q2 = w[2 * s], q3 = w[3 * s], q4 = w[4 * s], q5 = w[5 * s];
        double qm, qp;
        recon<RECON, AK_STATIC_PLAIN_DIV != 0>(q0, q1, q2, q3, q4, qm, qp);
        sL[v] = qp;
        recon<RECON, AK_STATIC_PLAIN_DIV != 0>(q1, q2, q3, q4, q5, qm, qp);
        sR[v] = qm;
      } else {
        const double q1 = w[s], q2 = w[2 * s], q3 = w[3 * s], q4 = w[4 * s], q5 = w[5 * s];
        double qm, qp;
        recon<RECON, AK_STATIC_PLAIN_DIV != 0>(q1, q2, q3, q4, q5, qm, qp);
        sR[v] = qm;
        xch[v2][t] = qp;
        if (DIR != 0 && a == 0) {
          double qm0;
          recon<RECON, AK_STATIC_PLAIN_DIV != 0>(w[0], q1, q2, q3, q4, qm0, qp);
          sL[v] = qp;
        }
      }
    }
  }
  if (RECON != 0 && ONCE) {
    __syncthreads();
    if (has_face && (DIR == 0 || a >= 1)) {
      sL[0] = xch[0][t - (DIR == 0 ? 1 : nfi)];
      sL[4] = xch[1][t - (DIR == 0 ? 1 : nfi)];
    }
  }
  if (!has_face) return;                       // no barrier below
  mbar_wait(&mbarM, 0);
  double mL[10], mR[10], Fo[7];
#pragma unroll
  for (int q = 0; q < 10; ++q) {
    const double* g = DIR == 0 ? sM + (size_t)q * slotM + a * nt + ii - 1 : sM + (size_t)q * slotM + a * nt + ii;
    mL[q] = g[0];
    mR[q] = g[DIR == 0 ? 1 : nt];
  }
  FaceGeo G;
  face_geometry<DIR>(mL, mR, G);
  face_flux_static<DIR, EOS>(P, P.riemann, G, sL, sR, Fo);
#pragma unroll
  for (int v = 0; v < 7; ++v) st_out<1>(f.F[7 * DIR + v] + fi, Fo[v]);
}

}  // namespace ak
