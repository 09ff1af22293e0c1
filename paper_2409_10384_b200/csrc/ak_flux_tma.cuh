// ak_flux_tma.cuh — K2, TMA-staged: the rows of primitives and metric a tile of faces needs are
// copied global -> shared memory with 1-D bulk TMA copies (cp.async.bulk, SASS UBLKCP) that
// complete on an mbarrier; the threads then reconstruct and solve one face each out of shared
// memory.  No thread holds a register for data in flight, stencil re-reads hit shared memory,
// and the 2-3 blocks resident on an SM overlap one block's copies with the others' arithmetic.
//
// Tile (n even, so every row of nt doubles is a multiple of 16 B):
//   DIR = x : NA rows (consecutive j at fixed k, m); faces i in [is-1, ie+2] of those rows.
//             shared rows: NA per field (primitives and metric alike).
//   DIR = y : one k-plane, NA consecutive face rows jf; faces i in [is-1, ie+1].
//   DIR = z : one j-row,   NA consecutive face planes kf; faces i in [is-1, ie+1].
//             shared rows: NA+5 per primitive field (cells f-3 .. f+2), NA+1 per metric field.
// Shared layout: [field][row][nt] doubles; lanes run along i: conflict-free.
#pragma once
#include <cstdint>
#include <cuda.h>
#include "ak_kernels.cuh"

namespace ak {

#ifndef AK_FLUX_PARK
#define AK_FLUX_PARK 1   // k_flux_tma: intermediates of the Riemann solve parked in the (spent) tile
#endif
#ifndef AK_TMA_MINB
#define AK_TMA_MINB 3
#endif
constexpr int TMA_THREADS = 256;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(void* dst, const void* src, unsigned bytes, uint64_t* b) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "AK_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra AK_DONE;\n"
      "bra AK_WAIT;\n"
      "AK_DONE:\n"
      "}\n" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}

// Which of the five often-zero fields of a staged tile (slots 1, 2, 3 = u^i and 5, 6 = the transverse B~cc)
// hold anything but +0.0: bit s of the result.  A field that is +0.0 on the whole tile reconstructs to
// +0.0 on both sides of every face, for every scheme here, so its reconstruction can be
// skipped: static atmosphere (u = 0) and unmagnetised regions (B = 0) are most of a merger grid.  All
// threads of the block call this (one barrier); `acc` is a shared word that thread 0 zeroed before an
// earlier barrier.
// `extra`: bits the calling thread adds (bit 7: its face-normal B~ is not +0.0).
// `loaded`: slots that were staged at all (a slot the block's zero flags ruled out is not in shared memory and
// counts as zero).
__device__ __forceinline__ unsigned tile_nonzero_mask(const double* sW, int slot_stride, int count, unsigned* acc,
                                                      unsigned extra = 0u, unsigned loaded = 0x7fu) {
  unsigned nz = extra;
  if (loaded & 0x6eu) {
    for (int q = threadIdx.x; q < count; q += (int)blockDim.x) {
#pragma unroll
      for (int s = 1; s < 7; ++s)
        if (s != 4 && ((loaded >> s) & 1u)) nz |= (unsigned)(__double_as_longlong(sW[(size_t)s * slot_stride + q]) != 0LL) << s;
    }
  }
  nz = __reduce_or_sync(0xffffffffu, nz);
  if ((threadIdx.x & 31) == 0 && nz) atomicOr(acc, nz);
  __syncthreads();
  return *acc | 0x11u;                  // slots 0 (rho) and 4 (P) are never zero: always reconstructed
}
// Slots of a sweep of direction DIR that have to be staged, from the block's zero flags (Fields::zflags, written
// by k_con2prim): slot 0 rho, 1..3 u^i, 4 P, 5 / 6 the transverse B~cc.
template <int DIR>
__device__ __forceinline__ unsigned slots_to_load(const Par& P, const Fields& f, int m) {
  if (!f.zflags || !(P.shortcuts & 1)) return 0x7fu;
  constexpr int t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  const unsigned z = f.zflags[m];
  return 0x11u | (z & 0x0eu) | (((z >> (5 + t1)) & 1u) << 5) | (((z >> (5 + t2)) & 1u) << 6);
}
constexpr unsigned ALWAYS_NZ = 0xffu;   // every slot reconstructed, face not static (shortcuts off)
// u^i, both transverse B~cc and the face-normal B~ are +0.0 on the whole tile: the static face flux applies
__device__ __forceinline__ bool tile_is_static(const Par& P, unsigned nzm) { return (P.shortcuts & 4) && !(nzm & 0xeeu); }

// both transverse B~cc and the face-normal B~ are +0.0 on the whole tile: side_state<.., NOB = true> applies
__device__ __forceinline__ bool tile_has_no_B(const Par& P, unsigned nzm) {
#ifdef AK_NO_NOB
  return false;
#else
  return (P.shortcuts & 4) && !(nzm & 0xe0u);
#endif
}
// Tensor maps of the 17 fields a sweep stages (host: ak_api.cu, cuTensorMapEncodeTiled).  Every cell field is
// the rank-3 tensor (i: nt, j: nt, K = m nt + k) of doubles; the box is the whole tile of one field, so a
// block issues 17 tensor copies (cp.async.bulk.tensor.3d, SASS UTMALDG) instead of one 1-D bulk copy per
// (field, row) -- about 200 per tile, whose issue cost showed once the arithmetic shrank (profiles/r2_final.md).
struct TileMaps {
  CUtensorMap w[7];     // rho, u^x, u^y, u^z, P, B~cc^{t1}, B~cc^{t2} of this direction
  CUtensorMap m[10];    // alp, betx, bety, betz, gxx .. gzz
};
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
      : "memory");
}
// doubles per field slot of a tile: rows * nt rounded up to 16 (tensor copies want 128-byte destinations)
__host__ __device__ __forceinline__ int tile_slot(int rows, int nt) { return ((rows * nt + 15) / 16) * 16; }

// use_tm != 0: the tile comes as 17 tensor-map box copies (maps); else as one bulk copy per (field, row)
template <int DIR, int RECON, int EOS = 0>
__global__ void __launch_bounds__(TMA_THREADS, AK_TMA_MINB)
k_flux_tma(const __grid_constant__ Par P, const __grid_constant__ Fields f, int NA,
           const __grid_constant__ TileMaps maps, int use_tm) {
  extern __shared__ __align__(128) double sm[];
  __shared__ uint64_t mbar, mbarM;      // primitive slabs / metric slabs: the metric lands while the states are reconstructed
  const int nt = P.nt, e = P.n + 2, t = threadIdx.x;
  constexpr int t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  const int maxW = DIR == 0 ? NA : NA + 5, maxM = DIR == 0 ? NA : NA + 1;
  const int slotW = tile_slot(maxW, nt), slotM = tile_slot(maxM, nt);
  double* sW = sm;                             // [7][slotW]   (maxW rows of nt)
  double* sM = sm + 7 * slotW;                 // [10][slotM]  (maxM rows of nt)
  // ---- which tile
  const int nfd = DIR == 0 ? e : P.n + 3;      // extent that NA tiles: rows (x) or faces along d (y,z)
  const int tiles = (nfd + NA - 1) / NA;
  int bid = blockIdx.x;
  if (f.tlist) {                               // the general tiles of k_split_tiles (block-uniform exit)
    if (blockIdx.x >= f.tcount[2 * DIR + 1]) return;
    bid = (int)f.tlist[(size_t)(2 * DIR + 1) * f.tcap + blockIdx.x];
  }
  const int td = bid % tiles; bid /= tiles;
  const int o = bid % e + P.is - 1;            // the fixed transverse index (k for x,y; j for z)
  const int m = bid / e;
  const int d0 = P.is - 1 + td * NA;           // first row (x) / first face along d (y,z)
  const int na = min(NA, P.is - 1 + nfd - d0); // rows / faces actually present in this tile
  const int nW = DIR == 0 ? na : na + 5, nM = DIR == 0 ? na : na + 1;
  const Ix ix{nt, P.px};
  // first cell of shared row 0 of the primitive slab / of the metric slab, and the row stride
  long long baseW, baseM, rs;
  if (DIR == 0) { baseW = baseM = ix.cell(m, o, d0, 0); rs = nt; }
  else if (DIR == 1) { baseW = ix.cell(m, o, d0 - 3, 0); baseM = ix.cell(m, o, d0 - 1, 0); rs = nt; }
  else { baseW = ix.cell(m, d0 - 3, o, 0); baseM = ix.cell(m, d0 - 1, o, 0); rs = (long long)nt * nt; }
  const unsigned rowb = (unsigned)(nt * sizeof(double));
  __shared__ unsigned nzacc;
  if (t == 0) { mbar_init(&mbar, 1); mbar_init(&mbarM, 1); nzacc = 0; }
  const unsigned ld = slots_to_load<DIR>(P, f, m);                  // block-uniform: slots that are staged at all
  __syncthreads();
  if (use_tm) {
    // ---- one tensor copy per field: the box holds maxW (maxM) rows whether or not the tile is ragged
    if (t < 32) {                                                   // lanes 0..16 of warp 0: one field each
      if (t == 0) {
        mbar_arrive_expect_tx(&mbar, (unsigned)(__popc(ld) * maxW) * rowb);
        mbar_arrive_expect_tx(&mbarM, (unsigned)(10 * maxM) * rowb);
      }
      __syncwarp();
      const int K = DIR == 2 ? m * nt + d0 : m * nt + o;            // plane coordinate of tile row 0 ...
      if (t < 7) {
        if ((ld >> t) & 1u) {
        const int cW1 = DIR == 0 ? d0 : (DIR == 1 ? d0 - 3 : o), cW2 = DIR == 2 ? K - 3 : K;
        tma_load_3d(sW + (size_t)t * slotW, &maps.w[t], 0, cW1, cW2, &mbar);
        }
      } else if (t < 17) {
        const int cM1 = DIR == 0 ? d0 : (DIR == 1 ? d0 - 1 : o), cM2 = DIR == 2 ? K - 1 : K;
        tma_load_3d(sM + (size_t)(t - 7) * slotM, &maps.m[t - 7], 0, cM1, cM2, &mbarM);
      }
    }
  } else {
  if (t == 0) {
    mbar_arrive_expect_tx(&mbar, (unsigned)(__popc(ld) * nW) * rowb);
    mbar_arrive_expect_tx(&mbarM, (unsigned)(10 * nM) * rowb);
  }
  // ---- one bulk copy per (field, row)
  const int ncW = 7 * nW, nc = ncW + 10 * nM;
  for (int c = t; c < nc; c += (int)blockDim.x) {
    if (c < ncW) {
      const int v = c / nW, r = c - v * nW;
      const int fld = v < 5 ? v : (v == 5 ? 5 + t1 : 5 + t2);
      if ((ld >> v) & 1u) bulk_copy_g2s(sW + (size_t)v * slotW + r * nt, f.W[fld] + baseW + r * rs, rowb, &mbar);
    } else {
      const int cc = c - ncW;
      const int q = cc / nM, r = cc - q * nM;
      const int fld = q == 0 ? 6 : (q < 4 ? 6 + q : q - 4);   // alp, betx..betz, gxx..gzz
      bulk_copy_g2s(sM + (size_t)q * slotM + r * nt, f.adm[fld] + baseM + r * rs, rowb, &mbarM);
    }
  }
  }
  // ---- this thread's face
  const int nfi = DIR == 0 ? P.n + 3 : e;      // faces per shared row
  const int a = t / nfi, ii = t - a * nfi + P.is - 1;   // row within the tile, i index of the face
  const bool active = a < na;
  long long fi = 0;
  double Bfd = 0.0;
  if (active) {
    if (DIR == 0) fi = ix.face(0, m, o, d0 + a, ii);
    else if (DIR == 1) fi = ix.face(1, m, o, d0 + a, ii);
    else fi = ix.face(2, m, d0 + a, o, ii);
    Bfd = __ldg(f.Bf[DIR] + fi);
  }
  mbar_wait(&mbar, 0);
  const unsigned nzm = ((RECON != 0 && (P.shortcuts & 1)) || (P.shortcuts & 4) || ld != 0x7fu)
                           ? tile_nonzero_mask(sW, slotW, nW * nt, &nzacc, (__double_as_longlong(Bfd) != 0LL) ? 0x80u : 0u, ld)
                           : ALWAYS_NZ;
  const bool stat = tile_is_static(P, nzm);          // block-uniform
  const unsigned rzm = (P.shortcuts & 1) ? nzm : ALWAYS_NZ;   // which slots are reconstructed
#if !AK_FLUX_PARK
  if (!active) return;
#endif
  double sL[7], sR[7], mL[10], mR[10], Fo[7];
  if (active) {
#pragma unroll
    for (int v = 0; v < 7; ++v) {
      // six stencil cells f-3 .. f+2: along i in one row (x) or one per shared row (y, z)
      const double* w = DIR == 0 ? sW + (size_t)v * slotW + a * nt + ii - 3 : sW + (size_t)v * slotW + a * nt + ii;
      const int s = DIR == 0 ? 1 : nt;
      if (!((rzm >> v) & 1u)) {
        sL[v] = 0.0; sR[v] = 0.0;           // the field is +0.0 on the whole tile (or was not even staged)
      } else if (RECON == 0) {
        sL[v] = w[2 * s]; sR[v] = w[3 * s];
      } else {
        const double q0 = w[0], q1 = w[s], q2 = w[2 * s], q3 = w[3 * s], q4 = w[4 * s], q5 = w[5 * s];
        double qm, qp;
        recon<RECON>(q0, q1, q2, q3, q4, qm, qp);
        sL[v] = qp;
        recon<RECON>(q1, q2, q3, q4, q5, qm, qp);
        sR[v] = qm;
      }
    }
  }
  mbar_wait(&mbarM, 0);
  if (active) {
#pragma unroll
    for (int q = 0; q < 10; ++q) {
      const double* g = DIR == 0 ? sM + (size_t)q * slotM + a * nt + ii - 1 : sM + (size_t)q * slotM + a * nt + ii;
      mL[q] = g[0];
      mR[q] = g[DIR == 0 ? 1 : nt];
    }
  }
#if AK_FLUX_PARK
  // every thread has read its stencils: the tile is reused as the parking space of face_flux_parked
  // (21 doubles per thread; the launcher sizes the allocation for both uses)
  FaceGeo G;
  if (active) face_geometry<DIR>(mL, mR, G);
  if (stat) {                                        // static unmagnetised tile: nothing to park, no barrier
    if (!active) return;
    face_flux_static<DIR, EOS>(P, P.riemann, G, sL, sR, Fo);
#pragma unroll
    for (int v = 0; v < 7; ++v) st_out<2>(f.F[7 * DIR + v] + fi, Fo[v]);
    return;
  }
  __syncthreads();
  if (!active) return;
  {   // (parking the right state behind the tile while it is reconstructed measured 3 % slower: more shared memory)
    volatile double* pR = sm + 14 * (int)blockDim.x + t;
#pragma unroll
    for (int v = 0; v < 7; ++v) pR[v * (int)blockDim.x] = sR[v];
  }
  if (tile_has_no_B(P, nzm))                         // block-uniform: moving but unmagnetised matter
    face_flux_parked<DIR, EOS, true>(P, P.riemann, G, sL, sm + 14 * (int)blockDim.x + t, (int)blockDim.x, Bfd, Fo,
                                     sm + t, (int)blockDim.x);
  else
    face_flux_parked<DIR, EOS>(P, P.riemann, G, sL, sm + 14 * (int)blockDim.x + t, (int)blockDim.x, Bfd, Fo, sm + t,
                               (int)blockDim.x);
#else
  face_flux<DIR, true, EOS>(P, P.riemann, mL, mR, sL, sR, Bfd, Fo);
#endif
#pragma unroll
  for (int v = 0; v < 7; ++v) st_out<2>(f.F[7 * DIR + v] + fi, Fo[v]);
}

// ---- reconstruct-once variant -------------------------------------------------------------------
// One thread per CELL of the tile: it reconstructs its cell once (both faces from one set of
// smoothness indicators), hands q^+ to the thread of the next cell through shared memory, and
// solves the face on its lower side with its own q^-.  Per face this needs one two-sided instead
// of two one-sided reconstructions (1810 -> ~1400 fp64 instructions for WENO-Z).  Measured on C4:
// 10 % faster than k_flux_tma for the x sweep (whole pencils, 35 of 36 threads solve a face),
// 10 % slower for y/z (6 of 7 thread rows solve a face, one redundant row per tile): the launcher
// uses it for x only.
//   DIR = x : NA rows x (n+4) cells (i in [is-2, ie+2]); the first cell of a row has no face.
//   DIR = y,z: (NA+1) cell rows x (n+2) lanes for NA face rows; the first cell row has no face.
// Same shared slabs as k_flux_tma plus 7 doubles per thread for q^+.
#ifndef AK_FLUXC_PARK
#define AK_FLUXC_PARK 1   // Riemann intermediates parked in the spent tile after a second barrier
#endif
#ifndef AK_TMAC_MINB
#define AK_TMAC_MINB 3    // with parking 80 registers do (3 blocks/SM: 4.19 -> 4.11 ms on C4; 2 blocks at 128: 4.29)
#endif
template <int DIR, int RECON, int EOS = 0>
__global__ void __launch_bounds__(TMA_THREADS, AK_TMAC_MINB)
k_flux_tma_cell(const __grid_constant__ Par P, const __grid_constant__ Fields f, int NA,
                const __grid_constant__ TileMaps maps, int use_tm) {
  extern __shared__ __align__(128) double sm[];
  __shared__ uint64_t mbar, mbarM;      // primitive slabs / metric slabs: the metric lands while the states are reconstructed
  const int nt = P.nt, e = P.n + 2, t = threadIdx.x;
  constexpr int t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  const int maxW = DIR == 0 ? NA : NA + 5, maxM = DIR == 0 ? NA : NA + 1;
  const int slotW = tile_slot(maxW, nt), slotM = tile_slot(maxM, nt);
  double* sW = sm;                             // [7][slotW]   (maxW rows of nt)
  double* sM = sm + 7 * slotW;                 // [10][slotM]  (maxM rows of nt)
  double* sQ = sM + 10 * slotM;                // [7][TMA_THREADS]
  const int nfd = DIR == 0 ? e : P.n + 3;
  const int tiles = (nfd + NA - 1) / NA;
  int bid = blockIdx.x;
  if (f.tlist) {                               // the general tiles of k_split_tiles (block-uniform exit)
    if (blockIdx.x >= f.tcount[2 * DIR + 1]) return;
    bid = (int)f.tlist[(size_t)(2 * DIR + 1) * f.tcap + blockIdx.x];
  }
  const int td = bid % tiles; bid /= tiles;
  const int o = bid % e + P.is - 1;            // the fixed transverse index (k for x,y; j for z)
  const int m = bid / e;
  const int d0 = P.is - 1 + td * NA;
  const int na = min(NA, P.is - 1 + nfd - d0);
  const int nW = DIR == 0 ? na : na + 5, nM = DIR == 0 ? na : na + 1;
  const Ix ix{nt, P.px};
  long long baseW, baseM, rs;
  if (DIR == 0) { baseW = baseM = ix.cell(m, o, d0, 0); rs = nt; }
  else if (DIR == 1) { baseW = ix.cell(m, o, d0 - 3, 0); baseM = ix.cell(m, o, d0 - 1, 0); rs = nt; }
  else { baseW = ix.cell(m, d0 - 3, o, 0); baseM = ix.cell(m, d0 - 1, o, 0); rs = (long long)nt * nt; }
  const unsigned rowb = (unsigned)(nt * sizeof(double));
  __shared__ unsigned nzacc;
  if (t == 0) { mbar_init(&mbar, 1); mbar_init(&mbarM, 1); nzacc = 0; }
  const unsigned ld = slots_to_load<DIR>(P, f, m);                  // block-uniform: slots that are staged at all
  __syncthreads();
  if (use_tm) {
    if (t < 32) {                                                   // lanes 0..16 of warp 0: one field each
      if (t == 0) {
        mbar_arrive_expect_tx(&mbar, (unsigned)(__popc(ld) * maxW) * rowb);
        mbar_arrive_expect_tx(&mbarM, (unsigned)(10 * maxM) * rowb);
      }
      __syncwarp();
      const int K = DIR == 2 ? m * nt + d0 : m * nt + o;            // plane coordinate of tile row 0 ...
      if (t < 7) {
        if ((ld >> t) & 1u) {
        const int cW1 = DIR == 0 ? d0 : (DIR == 1 ? d0 - 3 : o), cW2 = DIR == 2 ? K - 3 : K;
        tma_load_3d(sW + (size_t)t * slotW, &maps.w[t], 0, cW1, cW2, &mbar);
        }
      } else if (t < 17) {
        const int cM1 = DIR == 0 ? d0 : (DIR == 1 ? d0 - 1 : o), cM2 = DIR == 2 ? K - 1 : K;
        tma_load_3d(sM + (size_t)(t - 7) * slotM, &maps.m[t - 7], 0, cM1, cM2, &mbarM);
      }
    }
  } else {
  if (t == 0) {
    mbar_arrive_expect_tx(&mbar, (unsigned)(__popc(ld) * nW) * rowb);
    mbar_arrive_expect_tx(&mbarM, (unsigned)(10 * nM) * rowb);
  }
  const int ncW = 7 * nW, nc = ncW + 10 * nM;
  for (int c = t; c < nc; c += (int)blockDim.x) {
    if (c < ncW) {
      const int v = c / nW, r = c - v * nW;
      const int fld = v < 5 ? v : (v == 5 ? 5 + t1 : 5 + t2);
      if ((ld >> v) & 1u) bulk_copy_g2s(sW + (size_t)v * slotW + r * nt, f.W[fld] + baseW + r * rs, rowb, &mbar);
    } else {
      const int cc = c - ncW;
      const int q = cc / nM, r = cc - q * nM;
      const int fld = q == 0 ? 6 : (q < 4 ? 6 + q : q - 4);
      bulk_copy_g2s(sM + (size_t)q * slotM + r * nt, f.adm[fld] + baseM + r * rs, rowb, &mbarM);
    }
  }
  }
  // ---- this thread's cell: row a of the tile, index ii along x
  const int nci = DIR == 0 ? P.n + 4 : e;              // cells per row of threads
  const int a = t / nci;
  const int ii = t - a * nci + (DIR == 0 ? P.is - 2 : P.is - 1);
  const int nrow = DIR == 0 ? na : na + 1;             // rows of cells in this tile
  const bool active = a < nrow;
  const bool has_face = active && (DIR == 0 ? ii >= P.is - 1 : a >= 1);
  long long fi = 0;
  double Bfd = 0.0;
  if (has_face) {
    if (DIR == 0) fi = ix.face(0, m, o, d0 + a, ii);
    else if (DIR == 1) fi = ix.face(1, m, o, d0 - 1 + a, ii);
    else fi = ix.face(2, m, d0 - 1 + a, o, ii);
    Bfd = __ldg(f.Bf[DIR] + fi);
  }
  mbar_wait(&mbar, 0);
  const unsigned nzm = ((RECON != 0 && (P.shortcuts & 1)) || (P.shortcuts & 4) || ld != 0x7fu)
                           ? tile_nonzero_mask(sW, slotW, nW * nt, &nzacc, (__double_as_longlong(Bfd) != 0LL) ? 0x80u : 0u, ld)
                           : ALWAYS_NZ;
  const bool stat = tile_is_static(P, nzm);          // block-uniform
  const unsigned rzm = (P.shortcuts & 1) ? nzm : ALWAYS_NZ;   // which slots are reconstructed
  double qm[7];
  if (active) {
#pragma unroll
    for (int v = 0; v < 7; ++v) {
      // stencil c-2 .. c+2: along i in the row (x); shared rows a .. a+4 (y, z: my cell is row a+2)
      const double* w = DIR == 0 ? sW + (size_t)v * slotW + a * nt + ii - 2 : sW + (size_t)v * slotW + a * nt + ii;
      const int s = DIR == 0 ? 1 : nt;
      double qp;
      if (!((rzm >> v) & 1u)) { qm[v] = qp = 0.0; }          // the field is +0.0 on the whole tile (or was not staged)
      else if (RECON == 0) { qm[v] = qp = w[2 * s]; }
      else recon<RECON>(w[0], w[s], w[2 * s], w[3 * s], w[4 * s], qm[v], qp);
      sQ[v * TMA_THREADS + t] = qp;
    }
  }
  __syncthreads();
#if !AK_FLUXC_PARK
  if (!has_face) return;
#endif
  const int back = DIR == 0 ? 1 : nci;                 // thread of the lower cell
  double sL[7], mL[10], mR[10], Fo[7];
  mbar_wait(&mbarM, 0);
  if (has_face) {
#pragma unroll
    for (int v = 0; v < 7; ++v) sL[v] = sQ[v * TMA_THREADS + t - back];
#pragma unroll
    for (int q = 0; q < 10; ++q) {
      const double* g = DIR == 0 ? sM + (size_t)q * slotM + a * nt + ii - 1 : sM + (size_t)q * slotM + (a - 1) * nt + ii;
      mL[q] = g[0];
      mR[q] = g[DIR == 0 ? 1 : nt];
    }
  }
#if AK_FLUXC_PARK
  // second barrier: states and metric are in registers, the whole allocation becomes parking space
  FaceGeo G;
  if (has_face) face_geometry<DIR>(mL, mR, G);
  if (stat) {                                        // static unmagnetised tile: nothing to park, no barrier
    if (!has_face) return;
    face_flux_static<DIR, EOS>(P, P.riemann, G, sL, qm, Fo);
#pragma unroll
    for (int v = 0; v < 7; ++v) st_out<2>(f.F[7 * DIR + v] + fi, Fo[v]);
    return;
  }
  __syncthreads();
  if (!has_face) return;
  {
    volatile double* pR = sm + 14 * (int)blockDim.x + t;
#pragma unroll
    for (int v = 0; v < 7; ++v) pR[v * (int)blockDim.x] = qm[v];
  }
  if (tile_has_no_B(P, nzm))                         // block-uniform: moving but unmagnetised matter
    face_flux_parked<DIR, EOS, true>(P, P.riemann, G, sL, sm + 14 * (int)blockDim.x + t, (int)blockDim.x, Bfd, Fo,
                                     sm + t, (int)blockDim.x);
  else
    face_flux_parked<DIR, EOS>(P, P.riemann, G, sL, sm + 14 * (int)blockDim.x + t, (int)blockDim.x, Bfd, Fo, sm + t,
                               (int)blockDim.x);
#else
  face_flux<DIR, true, EOS>(P, P.riemann, mL, mR, sL, qm, Bfd, Fo);
#endif
#pragma unroll
  for (int v = 0; v < 7; ++v) st_out<2>(f.F[7 * DIR + v] + fi, Fo[v]);
}

}  // namespace ak
