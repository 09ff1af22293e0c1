// ak_kernels.cuh — the kernels of one RHS stage.
//   K1  k_con2prim      part (1)  all stored cells
//   K2  k_flux<DIR>     parts (2)+(3)  one thread per face, direction DIR
//   K3  k_fofc_test     part (4a) estimate + check-only con2prim (+DMP) -> flag bytes and the
//                       warp-ballot-compacted list of flagged cells
//   K4  k_fofc_reflux   part (4b) first-order re-solve of the faces of the listed cells
//   K5a k_cell_emf      part (5a) cell-centred EMFs
//   K5  k_ct<C3>        part (5b) Gardiner-Stone corner EMFs
//   K6  k_div_src       part (6)  flux divergence + geometric sources (Eq. 9)
#pragma once
#include "ak_flux.cuh"

namespace ak {

// occupancy targets (blocks of 128 threads per SM) — tuned with ncu, see profiles/
#ifndef AK_C2P_MINB
#define AK_C2P_MINB 8
#endif
#ifndef AK_C2P_PARK
#define AK_C2P_PARK 1   // k_con2prim parks the metric and B in shared memory across the root solve
#endif
#ifndef AK_FLUX_MINB
#define AK_FLUX_MINB 5
#endif
#ifndef AK_FOFC_MINB
#define AK_FOFC_MINB 8
#endif

// stats slots (device counters)
enum { S_C2P_FAIL = 0, S_CONS_FLOOR, S_PRIM_FLOOR, S_FOFC_CELLS, S_DMP_CELLS, S_NSTAT };

__device__ __forceinline__ void warp_count(unsigned long long* ctr, bool pred) {
  const unsigned m = __ballot_sync(__activemask(), pred);
  if (m != 0 && (threadIdx.x & 31) == (__ffs(m) - 1)) atomicAdd(ctr, (unsigned long long)__popc(m));
}

// Register-free prefetch of a line a thread reads only after a long dependent computation: lapse and
// shift for the cell EMFs after the con2prim solve (profiles/r1_v10_final.md: the largest long-scoreboard
// stall of that kernel; measured 3.156 -> 3.117 ms on C4).  The same for the DMP neighbourhood of the
// FOFC test measured 3 % slower and is not done.
#ifndef AK_PREFETCH
#define AK_PREFETCH 1   // 0: off, 1: prefetch.global.L1, 2: prefetch.global.L2
#endif
__device__ __forceinline__ void prefetch(const void* p) {
#if AK_PREFETCH == 1
  asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
#elif AK_PREFETCH == 2
  asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
#endif
}

// ---- index helpers (layouts of include/ak.h) ------------------------------------------
struct Ix {
  int nt, px;
  __device__ __forceinline__ long long cell(int m, int k, int j, int i) const {
    return (((long long)m * nt + k) * nt + j) * nt + i;
  }
  __device__ __forceinline__ long long face(int d, int m, int k, int j, int i) const {
    if (d == 0) return (((long long)m * nt + k) * nt + j) * px + i;
    if (d == 1) return (((long long)m * nt + k) * (nt + 1) + j) * nt + i;
    return (((long long)m * (nt + 1) + k) * nt + j) * nt + i;
  }
  __device__ __forceinline__ long long edge(int c, int m, int k, int j, int i) const {
    if (c == 0) return (((long long)m * (nt + 1) + k) * (nt + 1) + j) * nt + i;
    if (c == 1) return (((long long)m * (nt + 1) + k) * nt + j) * px + i;
    return (((long long)m * nt + k) * (nt + 1) + j) * px + i;
  }
};

__device__ __forceinline__ void load_met3(const Fields& f, long long c, Met3& g) {
  g.xx = __ldg(f.adm[0] + c); g.xy = __ldg(f.adm[1] + c); g.xz = __ldg(f.adm[2] + c);
  g.yy = __ldg(f.adm[3] + c); g.yz = __ldg(f.adm[4] + c); g.zz = __ldg(f.adm[5] + c);
}
// {alp, betx, bety, betz, gxx..gzz}
__device__ __forceinline__ void load_met10(const Fields& f, long long c, double m[10]) {
  m[0] = __ldg(f.adm[6] + c); m[1] = __ldg(f.adm[7] + c); m[2] = __ldg(f.adm[8] + c);
  m[3] = __ldg(f.adm[9] + c);
#pragma unroll
  for (int q = 0; q < 6; ++q) m[4 + q] = __ldg(f.adm[q] + c);
}

// ---- K1 ------------------------------------------------------------------------------
// EMF: also write the cell-centred EMFs of the final primitives (the arithmetic of k_cell_emf), so
// that a stage that runs part (1) does not re-read W and the metric for them.
// STRIDE: grid-stride loop for a capped grid (overlapped schedule only; the plain one-cell-per-thread
// form is 0.05-0.12 ms faster on C4 and is what the serial schedule launches)
template <bool EMF, int EOS = 0, bool STRIDE = false>
__global__ void __launch_bounds__(128, AK_C2P_MINB) k_con2prim(const __grid_constant__ Par P,
                                                  const __grid_constant__ Fields f) {
  const int nt = P.nt;
  const long long ncell = (long long)P.nmb * nt * nt * nt;
#if AK_C2P_PARK
  __shared__ double park[9][128];
#endif
  // grid-stride: the launcher may cap the grid (a few blocks per SM) so that the kernel shares the SMs
  // with the flux sweeps of another chunk of blocks (ak_set_overlap)
  long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  do {
  if (c >= ncell) return;
  const int i = (int)(c % nt);
  const long long row = c / nt;               // (m*nt + k)*nt + j
  const int j = (int)(row % nt);
  const long long mk = row / nt;              // m*nt + k
  const int k = (int)(mk % nt);
  const int m = (int)(mk / nt);
  Met3 g;
  load_met3(f, c, g);
  double Ut[5], Bc[3], W5[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) Ut[v] = f.U[v][c];
  if (EMF) {
#pragma unroll
    for (int q = 6; q < 10; ++q) prefetch(f.adm[q] + c);   // lapse and shift, read after the solve
  }
  const long long fx = row * P.px + i;
  const long long fy = (mk * (nt + 1) + j) * nt + i;
  const long long fz = (((long long)m * (nt + 1) + k) * nt + j) * nt + i;
  // every face of the block is the lower or the upper face of one of its cells: the OR of the bit patterns
  // tells whether the block holds a face value that is not +0.0 (zflags bits 8..10)
  unsigned fnz = 0;
  {
    const double a0 = __ldg(f.Bf[0] + fx), a1 = __ldg(f.Bf[0] + fx + 1);
    const double b0 = __ldg(f.Bf[1] + fy), b1 = __ldg(f.Bf[1] + fy + nt);
    const double c0 = __ldg(f.Bf[2] + fz), c1 = __ldg(f.Bf[2] + fz + (long long)nt * nt);
    Bc[0] = 0.5 * (a0 + a1); Bc[1] = 0.5 * (b0 + b1); Bc[2] = 0.5 * (c0 + c1);
    fnz = ((unsigned)((__double_as_longlong(a0) | __double_as_longlong(a1)) != 0LL) << 8) |
          ((unsigned)((__double_as_longlong(b0) | __double_as_longlong(b1)) != 0LL) << 9) |
          ((unsigned)((__double_as_longlong(c0) | __double_as_longlong(c1)) != 0LL) << 10);
  }
#if AK_C2P_PARK
  // The metric and B are needed again only after the root solve.  Parked in shared memory they
  // leave the registers for the solve; left to the compiler they are spilled to local memory,
  // which is written through to L2 and partly on to DRAM (profiles/r1_v10_final.md): 3.12 -> 2.90 ms
  // on C4.  Parking r^i and B^i inside c2p_cell as well, or in k_fofc_test, measured no gain / 1 % loss.
  park[0][threadIdx.x] = g.xx; park[1][threadIdx.x] = g.xy; park[2][threadIdx.x] = g.xz;
  park[3][threadIdx.x] = g.yy; park[4][threadIdx.x] = g.yz; park[5][threadIdx.x] = g.zz;
#pragma unroll
  for (int v = 0; v < 3; ++v) park[6 + v][threadIdx.x] = Bc[v];
  const int st = c2p_cell<false, EOS>(P, g, Ut, Bc, W5);
  {
    volatile double* pk = &park[0][threadIdx.x];
    g.xx = pk[0]; g.xy = pk[128]; g.xz = pk[2 * 128]; g.yy = pk[3 * 128]; g.yz = pk[4 * 128]; g.zz = pk[5 * 128];
#pragma unroll
    for (int v = 0; v < 3; ++v) Bc[v] = pk[(6 + v) * 128];
  }
  if (st != 0) {   // "a similar policy holds for the conserved variables": rewrite them from the final primitives
    double det, sdet;
    Met3 gu;
    metric_inverse(g, det, sdet, gu);
    const double isd = 1.0 / sdet;
    const double B[3] = {Bc[0] * isd, Bc[1] * isd, Bc[2] * isd};
    c2p_write_back<EOS>(P, g, sdet, W5[0], W5[1], W5[2], W5[3], W5[4], B, Ut);
  }
#else
  const int st = c2p_cell<true, EOS>(P, g, Ut, Bc, W5);
#endif
#pragma unroll
  for (int v = 0; v < 5; ++v) st_out<4>(f.W[v] + c, W5[v]);
#pragma unroll
  for (int v = 0; v < 3; ++v) st_out<4>(f.W[5 + v] + c, Bc[v]);
  if (st != 0) {
#pragma unroll
    for (int v = 0; v < 5; ++v) f.U[v][c] = Ut[v];
  }
  if (f.status) f.status[c] = (unsigned char)st;
  if (f.zflags) {
    // which of this block's often-zero fields hold anything but +0.0: later kernels of the stage do not
    // load a field whose bit stays clear.  A set bit is only ever added: the flag may say
    // "non-zero" for a field that is zero (another thread's stale read), never the reverse.
    unsigned nz = fnz;
#pragma unroll
    for (int v = 1; v < 4; ++v) nz |= (unsigned)(__double_as_longlong(W5[v]) != 0LL) << v;
#pragma unroll
    for (int v = 0; v < 3; ++v) nz |= (unsigned)(__double_as_longlong(Bc[v]) != 0LL) << (5 + v);
    if (nz != 0 && (__ldcg(f.zflags + m) & nz) != nz) atomicOr(f.zflags + m, nz);
    // the same per ROW of cells (m, k, j), for the tile lists of k_split_tiles: a row whose byte stays 0 has
    // u^i = +0 and every face B~ of its cells = +0 (hence B~cc = +0).
    if (f.rowflag) {                           // (one store per row segment of the warp, not one per cell)
      const bool fl = (nz & 0x70eu) != 0;
      const unsigned act = __activemask();
      const unsigned bal = __ballot_sync(act, fl);
      if (bal != 0) {
        const int rw = (int)row;
        const unsigned same = __match_any_sync(act, rw);
        if (fl && (int)(threadIdx.x & 31) == __ffs(bal & same) - 1) f.rowflag[rw] = 1;
      }
    }
  }
  if (EMF) {
    const double u[3] = {W5[1], W5[2], W5[3]};
    double ul[3];
    lower(g, u, ul);
    const double usq = dot3(ul, u);
    const double iW = 1.0 / sqrt(1.0 + usq);
    const double alp = __ldg(f.adm[6] + c), ialp = 1.0 / alp;
    const double vh[3] = {u[0] * iW - __ldg(f.adm[7] + c) * ialp, u[1] * iW - __ldg(f.adm[8] + c) * ialp,
                          u[2] * iW - __ldg(f.adm[9] + c) * ialp};
    st_out<4>(f.Ecc[0] + c, -(alp * (vh[1] * Bc[2] - vh[2] * Bc[1])));
    st_out<4>(f.Ecc[1] + c, -(alp * (vh[2] * Bc[0] - vh[0] * Bc[2])));
    st_out<4>(f.Ecc[2] + c, -(alp * (vh[0] * Bc[1] - vh[1] * Bc[0])));
  }
  warp_count(f.stats + S_C2P_FAIL, (st & ST_FAIL) != 0);
  warp_count(f.stats + S_CONS_FLOOR, (st & (ST_DFLOOR | ST_TAUFLOOR | ST_MAGCAP)) != 0);
  warp_count(f.stats + S_PRIM_FLOOR, (st & (ST_RHOFLOOR | ST_TFLOOR)) != 0);
  c += (long long)gridDim.x * blockDim.x;
  } while (STRIDE);
}

// ---- computed-face range decoding ----------------------------------------------------
// Faces of direction DIR: DIR-index in [is-1, ie+2] (n+3), transverse in [is-1, ie+1] (n+2).
template <int DIR>
__device__ __forceinline__ bool decode_face(const Par& P, long long idx, int& m, int& k, int& j, int& i) {
  const int ei = P.n + (DIR == 0 ? 3 : 2), ej = P.n + (DIR == 1 ? 3 : 2), ek = P.n + (DIR == 2 ? 3 : 2);
  const long long per = (long long)ei * ej * ek;
  if (idx >= per * P.nmb) return false;
  m = (int)(idx / per);
  int r = (int)(idx - (long long)m * per);
  i = r % ei + P.is - 1; r /= ei;
  j = r % ej + P.is - 1;
  k = r / ej + P.is - 1;
  return true;
}

// ---- K2 (v1: one thread per face; both one-sided reconstructions done by the thread) ----
template <int DIR, int RECON, int EOS = 0>
__global__ void __launch_bounds__(128, AK_FLUX_MINB) k_flux(const __grid_constant__ Par P,
                                              const __grid_constant__ Fields f) {
  int m, k, j, i;
  if (!decode_face<DIR>(P, (long long)blockIdx.x * blockDim.x + threadIdx.x, m, k, j, i)) return;
  const Ix ix{P.nt, P.px};
  constexpr int t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  const long long stride = DIR == 0 ? 1 : (DIR == 1 ? P.nt : (long long)P.nt * P.nt);
  const long long cu = ix.cell(m, k, j, i), cl = cu - stride;
  const int var[7] = {0, 1, 2, 3, 4, 5 + t1, 5 + t2};
  double sL[7], sR[7];
#pragma unroll
  for (int v = 0; v < 7; ++v) {
    const double* w = f.W[var[v]] + cu;
    if (RECON == 0) {
      sL[v] = w[-stride]; sR[v] = w[0];
    } else {
      const double q0 = w[-3 * stride], q1 = w[-2 * stride], q2 = w[-stride], q3 = w[0],
                   q4 = w[stride], q5 = w[2 * stride];
      double qm, qp;
      recon<RECON>(q0, q1, q2, q3, q4, qm, qp);
      sL[v] = qp;                         // right face of the lower cell
      recon<RECON>(q1, q2, q3, q4, q5, qm, qp);
      sR[v] = qm;                         // left face of the upper cell
    }
  }
  double mL[10], mR[10], Fo[7];
  load_met10(f, cl, mL);
  load_met10(f, cu, mR);
  const long long fi = ix.face(DIR, m, k, j, i);
  face_flux<DIR, true, EOS>(P, P.riemann, mL, mR, sL, sR, __ldg(f.Bf[DIR] + fi), Fo);
#pragma unroll
  for (int v = 0; v < 7; ++v) f.F[7 * DIR + v][fi] = Fo[v];
}

// ---- test-cell range decoding: cells in [is-1, ie+1]^3 ----------------------------------
__device__ __forceinline__ bool decode_test(const Par& P, long long idx, int& m, int& k, int& j, int& i) {
  const int e = P.n + 2;
  const long long per = (long long)e * e * e;
  if (idx >= per * P.nmb) return false;
  m = (int)(idx / per);
  int r = (int)(idx - (long long)m * per);
  i = r % e + P.is - 1; r /= e;
  j = r % e + P.is - 1;
  k = r / e + P.is - 1;
  return true;
}

// flux difference of component v across cell (m,k,j,i), summed x then y then z
__device__ __forceinline__ double div_flux(const Fields& f, const Ix& ix, int v, int m, int k, int j, int i,
                                           const double idx[3]) {
  const long long fx = ix.face(0, m, k, j, i), fy = ix.face(1, m, k, j, i), fz = ix.face(2, m, k, j, i);
  const long long sy = ix.nt, sz = (long long)ix.nt * ix.nt;
  return (f.F[v][fx + 1] - f.F[v][fx]) * idx[0] + (f.F[7 + v][fy + sy] - f.F[7 + v][fy]) * idx[1] +
         (f.F[14 + v][fz + sz] - f.F[14 + v][fz]) * idx[2];
}

template <int EOS>
__device__ __forceinline__ void div_src_cell(const Par& P, const Fields& f, int m, long long c, const double div[5]);   // ak_source.cuh

#ifndef AK_FOFC_PREFETCH_U
#define AK_FOFC_PREFETCH_U 1   // the conserved state's lines ahead of the flux loads (the metric's: slower, ak_source.cuh)
#endif
#ifndef AK_FSRC_MINB
#define AK_FSRC_MINB 4    // blocks/SM of the FOFC test fused with part (6)
#endif
// ---- K3: FOFC estimate and test (DMP Eq. 12) -------------------------------
// SRC: also part (6) for the interior cells, from the flux differences this kernel forms anyway (the high-order
// fluxes; cells next to re-fluxed faces are redone by k_src_fix): the 15 flux fields are read once instead of
// twice, and the memory-bound sources of one warp overlap the dependent chains of another's con2prim check.
template <int EOS = 0, bool STRIDE = false, bool SRC = false>
__global__ void __launch_bounds__(128, SRC ? AK_FSRC_MINB : AK_FOFC_MINB) k_fofc_test(const __grid_constant__ Par P,
                                                   const __grid_constant__ Fields f, double dt) {
  long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  do {
  int m, k, j, i;
  if (!decode_test(P, tid, m, k, j, i)) return;
  const Ix ix{P.nt, P.px};
  const long long c = ix.cell(m, k, j, i);
#if AK_FOFC_PREFETCH_U
#pragma unroll
  for (int q = 0; q < 5; ++q) prefetch(f.U[q] + c);      // read after the 30 flux values (1.94 -> 1.92 ms on C4)
#endif
  const double idx[3] = {1.0 / f.dx[3 * m + 0], 1.0 / f.dx[3 * m + 1], 1.0 / f.dx[3 * m + 2]};
  double Us[5], Bc[3], W5[5];
  {
    double dv[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) dv[v] = div_flux(f, ix, v, m, k, j, i, idx);
    if (SRC && i >= P.is && i <= P.ie && j >= P.is && j <= P.ie && k >= P.is && k <= P.ie)
      div_src_cell<EOS>(P, f, m, c, dv);
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      if (f.U0[0]) Us[v] = f.fa * f.U0[v][c] + f.fb * (f.U[v][c] - dt * dv[v]);
      else Us[v] = f.U[v][c] - dt * dv[v];
    }
  }
  Met3 g;
  load_met3(f, c, g);
  const unsigned zf = (f.zflags && (P.shortcuts & 1)) ? f.zflags[m] : 0xffu;    // clear bit: the field is +0.0 in this block
#pragma unroll
  for (int v = 0; v < 3; ++v) Bc[v] = ((zf >> (5 + v)) & 1u) ? f.W[5 + v][c] : 0.0;
  const double Ds = Us[0], ts = Us[4];
  int st = c2p_cell<false, EOS>(P, g, Us, Bc, W5);
  // Eq. 12 asks whether D~*, tau~* lie in [min/M, M max] of the 27-cell neighbourhood.  The centre cell is one
  // of the 27, so min <= U_c <= max, and rounding is monotonic (x <= y => x iM <= y iM for iM > 0): a value
  // inside [U_c/M, M U_c] is inside [min/M, M max] whatever the neighbours hold -- no flag, and no need to
  // read them.  Only a cell whose estimate moved by more than the factor M against its own value (a NaN
  // fails every comparison and lands here too) scans the neighbourhood; a warp skips the scan when none of
  // its lanes needs it (on C4: 92 % of warps; FOFC test 2.38 -> x ms).  Same flags bit for bit.
  bool dmp_scan = false;
  if (P.dmp_M > 0.0) {
    const double Dc = f.U[0][c], tc = f.U[4][c];
    dmp_scan = !(Ds >= Dc * P.dmp_iM && Ds <= P.dmp_M * Dc && ts >= tc * P.dmp_iM && ts <= P.dmp_M * tc);
  }
  if (dmp_scan) {
    // fmin/fmax over the 27 cells (the centre is one of them) written as compare-and-select from
    // +-inf: the same values for every input (a NaN is skipped either way; only the sign of a zero
    // can differ, which no comparison below sees) at a third of the instructions of fmin/fmax.
    double Dmin = CUDART_INF, Dmax = -CUDART_INF, tmin = CUDART_INF, tmax = -CUDART_INF;
    const long long sy = P.nt, sz = (long long)P.nt * P.nt;
#ifndef AK_DMP_UNROLL
#define AK_DMP_UNROLL 1
#endif
    constexpr int dmp_unroll = AK_DMP_UNROLL;   // 1: the 27-cell loop stays rolled over k and j (smaller code)
#pragma unroll dmp_unroll
    for (int kk = -1; kk <= 1; ++kk)
#pragma unroll dmp_unroll
      for (int jj = -1; jj <= 1; ++jj)
#pragma unroll
        for (int ii = -1; ii <= 1; ++ii) {
          const long long cn = c + kk * sz + jj * sy + ii;
          const double d = f.U[0][cn], t = f.U[4][cn];
          Dmin = d < Dmin ? d : Dmin; Dmax = d > Dmax ? d : Dmax;
          tmin = t < tmin ? t : tmin; tmax = t > tmax ? t : tmax;
        }
    if (Ds < Dmin * P.dmp_iM || Ds > P.dmp_M * Dmax || ts < tmin * P.dmp_iM || ts > P.dmp_M * tmax)
      st |= ST_DMP;
  }
  f.flag[c] = (unsigned char)st;
  warp_count(f.stats + S_DMP_CELLS, (st & ST_DMP) != 0);
  // compact the flagged cells (warp ballot + one atomic per warp); count[3] = list length.
  // The order of entries depends on the atomics but no output does.
  const unsigned act = __activemask();
  const unsigned bal = __ballot_sync(act, st != 0);
  if (bal != 0) {
    const int lane = threadIdx.x & 31, leader = __ffs(bal) - 1;
    unsigned base = 0;
    if (lane == leader) base = atomicAdd(f.count + 3, (unsigned)__popc(bal));
    base = __shfl_sync(act, base, leader);
    if (st != 0) f.list[base + __popc(bal & ((1u << lane) - 1u))] = (unsigned)c;
  }
  tid += (long long)gridDim.x * blockDim.x;
  } while (STRIDE);
}

// ---- K4: first-order re-solve of the faces of the flagged cells ("recalculate the fluxes
// for all flagged cells but using a first-order scheme").  A face between cells A (lower) and B
// (upper) is redone exactly once: by B's entry if B is flagged, else by A's.  So entry c handles
// its lower DIR-face always and its upper DIR-face only when the upper neighbour is not flagged.
// Thread t < 2 * count: which = t / count (0 lower, 1 upper) keeps warps uniform.
template <int DIR, int EOS = 0>
__global__ void __launch_bounds__(128) k_fofc_reflux(const __grid_constant__ Par P,
                                                     const __grid_constant__ Fields f) {
  const unsigned cnt = f.count[3];
  const Ix ix{P.nt, P.px};
  constexpr int t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  const unsigned nt = (unsigned)P.nt;
  const unsigned stride = DIR == 0 ? 1u : (DIR == 1 ? nt : nt * nt);
  const int var[7] = {0, 1, 2, 3, 4, 5 + t1, 5 + t2};
  unsigned nface = 0;
  for (unsigned e = blockIdx.x * blockDim.x + threadIdx.x; e < 2u * cnt; e += gridDim.x * blockDim.x) {
    const unsigned which = e >= cnt ? 1u : 0u;
    const unsigned c = f.list[e - which * cnt];
    if (which && f.flag[c + stride] != 0) continue;       // the upper neighbour's entry does this face
    const unsigned cu = c + which * stride, cl = cu - stride;
    const int i = (int)(cu % nt);
    const unsigned row = cu / nt;
    const int j = (int)(row % nt);
    const unsigned mk = row / nt;
    const int k = (int)(mk % nt), m = (int)(mk / nt);
    double sL[7], sR[7], mL[10], mR[10], Fo[7];
#pragma unroll
    for (int v = 0; v < 7; ++v) { sL[v] = f.W[var[v]][cl]; sR[v] = f.W[var[v]][cu]; }
    load_met10(f, cl, mL);
    load_met10(f, cu, mR);
    const long long fi = ix.face(DIR, m, k, j, i);
    face_flux<DIR, true, EOS>(P, P.fofc_riemann, mL, mR, sL, sR, __ldg(f.Bf[DIR] + fi), Fo);
#pragma unroll
    for (int v = 0; v < 7; ++v) f.F[7 * DIR + v][fi] = Fo[v];
    ++nface;
  }
  // faces redone in this direction (reported by ak_get_stats)
  for (int o = 16; o > 0; o >>= 1) nface += __shfl_xor_sync(0xffffffffu, nface, o);
  if ((threadIdx.x & 31) == 0 && nface) atomicAdd(f.count + DIR, nface);
}

// ---- K5a: cell-centred EMFs  E_c = -alpha (vhat^a B~^b - vhat^b B~^a) on [is-1,ie+1]^3 --------
__global__ void __launch_bounds__(128) k_cell_emf(const __grid_constant__ Par P,
                                                  const __grid_constant__ Fields f) {
  int m, k, j, i;
  if (!decode_test(P, (long long)blockIdx.x * blockDim.x + threadIdx.x, m, k, j, i)) return;
  const Ix ix{P.nt, P.px};
  const long long c = ix.cell(m, k, j, i);
  Met3 g;
  load_met3(f, c, g);
  const double u[3] = {f.W[1][c], f.W[2][c], f.W[3][c]};
  double ul[3];
  lower(g, u, ul);
  const double usq = dot3(ul, u);
  const double iW = 1.0 / sqrt(1.0 + usq);
  const double alp = __ldg(f.adm[6] + c), ialp = 1.0 / alp;
  const double vh[3] = {u[0] * iW - __ldg(f.adm[7] + c) * ialp, u[1] * iW - __ldg(f.adm[8] + c) * ialp,
                        u[2] * iW - __ldg(f.adm[9] + c) * ialp};
  const double Bt[3] = {f.W[5][c], f.W[6][c], f.W[7][c]};
  f.Ecc[0][c] = -(alp * (vh[1] * Bt[2] - vh[2] * Bt[1]));
  f.Ecc[1][c] = -(alp * (vh[2] * Bt[0] - vh[0] * Bt[2]));
  f.Ecc[2][c] = -(alp * (vh[0] * Bt[1] - vh[1] * Bt[0]));
}

// ---- K5: corner EMFs, component C3 (Gardiner & Stone 2005; DESIGN.md §3 O8) ------------------
// a, b cyclic after C3.  Edge (ia, ib, ic): ia, ib in [is, ie+1], ic in [is, ie].
template <int C3>
__device__ __forceinline__ void ct_edge(const Par& P, const Fields& f, const Ix& ix, int m, const int p3[3]) {
  constexpr int a = (C3 + 1) % 3, b = (C3 + 2) % 3;
  // offsets of one step along a and b, in cells and in the a-face / b-face layouts
  const long long cst[3] = {1, P.nt, (long long)P.nt * P.nt};
  const long long c0 = ix.cell(m, p3[2], p3[1], p3[0]);
  const long long fa0 = ix.face(a, m, p3[2], p3[1], p3[0]);
  const long long fb0 = ix.face(b, m, p3[2], p3[1], p3[0]);
  // step of index b inside the a-face layout, and of index a inside the b-face layout
  int q3[3] = {p3[0], p3[1], p3[2]};
  q3[b] -= 1;
  const long long fa_b = ix.face(a, m, q3[2], q3[1], q3[0]) - fa0;   // (ia, ib-1)
  q3[b] += 1; q3[a] -= 1;
  const long long fb_a = ix.face(b, m, q3[2], q3[1], q3[0]) - fb0;   // (ia-1, ib)
  const double* FaB = f.F[7 * a + 5];   // a-face flux of B~^b  -> E_c = -F
  const double* FbB = f.F[7 * b + 6];   // b-face flux of B~^a  -> E_c = +F
  const double* FaD = f.F[7 * a];
  const double* FbD = f.F[7 * b];
  const double* Ec = f.Ecc[C3];
  const double Eaf_00 = -FaB[fa0], Eaf_0m = -FaB[fa0 + fa_b];      // (ia,ib), (ia,ib-1)
  const double Ebf_00 = FbB[fb0], Ebf_m0 = FbB[fb0 + fb_a];        // (ia,ib), (ia-1,ib)
  const double Ec_00 = Ec[c0], Ec_m0 = Ec[c0 - cst[a]], Ec_0m = Ec[c0 - cst[b]],
               Ec_mm = Ec[c0 - cst[a] - cst[b]];
  const double fD_a0 = FaD[fa0], fD_am = FaD[fa0 + fa_b], fD_b0 = FbD[fb0], fD_bm = FbD[fb0 + fb_a];
  const double w = fD_a0 > 0.0 ? 1.0 : (fD_a0 < 0.0 ? 0.0 : 0.5);
  const double wp = fD_am > 0.0 ? 1.0 : (fD_am < 0.0 ? 0.0 : 0.5);
  const double w2 = fD_b0 > 0.0 ? 1.0 : (fD_b0 < 0.0 ? 0.0 : 0.5);
  const double w2p = fD_bm > 0.0 ? 1.0 : (fD_bm < 0.0 ? 0.0 : 0.5);
  const double dbm = w * (Ec_m0 - Ebf_m0) + (1.0 - w) * (Ec_00 - Ebf_00);
  const double dbp = wp * (Ebf_m0 - Ec_mm) + (1.0 - wp) * (Ebf_00 - Ec_0m);
  const double dam = w2 * (Ec_0m - Eaf_0m) + (1.0 - w2) * (Ec_00 - Eaf_00);
  const double dap = w2p * (Eaf_0m - Ec_mm) + (1.0 - w2p) * (Eaf_00 - Ec_m0);
  const double e = 0.25 * (Eaf_00 + Eaf_0m + Ebf_00 + Ebf_m0) + 0.25 * ((dbp - dbm) + (dap - dam));
  f.E[C3][ix.edge(C3, m, p3[2], p3[1], p3[0])] = e;
}

template <int C3, bool STRIDE = false>
__global__ void __launch_bounds__(128) k_ct(const __grid_constant__ Par P,
                                            const __grid_constant__ Fields f) {
  const int n = P.n;
  const int ei = n + (C3 == 0 ? 0 : 1), ej = n + (C3 == 1 ? 0 : 1), ek = n + (C3 == 2 ? 0 : 1);
  const long long per = (long long)ei * ej * ek;
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  do {
  if (idx >= per * P.nmb) return;
  const int m = (int)(idx / per);
  int r = (int)(idx - (long long)m * per);
  int p3[3];
  p3[0] = r % ei + P.is; r /= ei;
  p3[1] = r % ej + P.is;
  p3[2] = r / ej + P.is;
  const Ix ix{P.nt, P.px};
  ct_edge<C3>(P, f, ix, m, p3);
  idx += (long long)gridDim.x * blockDim.x;
  } while (STRIDE);
}

// All three components in one launch: one thread per corner point (i, j, k) in [is, ie+1]^3, which owns the edges
// that start there (E_x if i <= ie, E_y if j <= ie, E_z if k <= ie).  Each mass-flux field is needed by two
// components and each face EMF field by one; in one kernel the second use hits L1/L2 instead of DRAM.
__global__ void __launch_bounds__(128) k_ct_all(const __grid_constant__ Par P, const __grid_constant__ Fields f) {
  const int n1 = P.n + 1;
  const long long per = (long long)n1 * n1 * n1;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= per * P.nmb) return;
  const int m = (int)(idx / per);
  int r = (int)(idx - (long long)m * per);
  int p3[3];
  p3[0] = r % n1 + P.is; r /= n1;
  p3[1] = r % n1 + P.is;
  p3[2] = r / n1 + P.is;
  const Ix ix{P.nt, P.px};
  if (p3[0] <= P.ie) ct_edge<0>(P, f, ix, m, p3);
  if (p3[1] <= P.ie) ct_edge<1>(P, f, ix, m, p3);
  if (p3[2] <= P.ie) ct_edge<2>(P, f, ix, m, p3);
}

}  // namespace ak
