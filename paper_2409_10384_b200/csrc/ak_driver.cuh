// ak_driver.cuh — stage driver kernels ("RK2 / RK3", constrained transport):
//   k_fill_cells / k_fill_faces<D>   ghost fill of self-contained MeshBlocks (periodic / outflow)
//   k_update_cells / k_update_faces<D>  Shu-Osher register update  U <- a U0 + b (U + dt dU),
//                                    B~f <- a B0 + b (B~f + dt (-curl E)) on faces of interior cells
//   k_or_bytes                       OR-accumulation of FOFC flag bytes over stages
#pragma once
#include "ak_kernels.cuh"

namespace ak {

struct DrvFields {
  double* U[5];
  double* Bf[3];
  const double* U0[5];
  const double* B0[3];
  const double* dU[5];
  const double* E[3];
  const double* dx;
};

// source index of a cell-like index q (itself when interior); bc 0 periodic, 1 outflow
__device__ __forceinline__ int src_cell(int q, int bc, int is, int ie, int n) {
  if (q >= is && q <= ie) return q;
  if (bc == 0) { int r = (q - is) % n; if (r < 0) r += n; return is + r; }
  return q < is ? is : ie;
}
// source index of a face-normal index q in [0, nt]; periodic: face ie+1 is face is
__device__ __forceinline__ int src_face(int q, int bc, int is, int ie, int n) {
  if (bc == 0) { int r = (q - is) % n; if (r < 0) r += n; return is + r; }
  if (q < is) return is;
  if (q > ie + 1) return ie + 1;
  return q;
}

__global__ void __launch_bounds__(256) k_fill_cells(const __grid_constant__ Par P, const __grid_constant__ DrvFields f,
                                                    int bcx, int bcy, int bcz) {
  const unsigned nt = (unsigned)P.nt;
  const unsigned ncell = (unsigned)P.nmb * nt * nt * nt;
  const unsigned c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  const int i = (int)(c % nt);
  unsigned r = c / nt;
  const int j = (int)(r % nt); r /= nt;
  const int k = (int)(r % nt);
  const int m = (int)(r / nt);
  const int is_ = src_cell(i, bcx, P.is, P.ie, P.n), js = src_cell(j, bcy, P.is, P.ie, P.n),
            ks = src_cell(k, bcz, P.is, P.ie, P.n);
  if (is_ == i && js == j && ks == k) return;
  const Ix ix{P.nt, P.px};
  const long long s = ix.cell(m, ks, js, is_);
#pragma unroll
  for (int v = 0; v < 5; ++v) f.U[v][c] = f.U[v][s];
}

template <int D>
__global__ void __launch_bounds__(256) k_fill_faces(const __grid_constant__ Par P, const __grid_constant__ DrvFields f,
                                                    int bcx, int bcy, int bcz) {
  const unsigned nt = (unsigned)P.nt;
  const unsigned ni = nt + (D == 0), nj = nt + (D == 1), nk = nt + (D == 2);
  const unsigned tot = (unsigned)P.nmb * nk * nj * ni;
  const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= tot) return;
  const int i = (int)(t % ni);
  unsigned r = t / ni;
  const int j = (int)(r % nj); r /= nj;
  const int k = (int)(r % nk);
  const int m = (int)(r / nk);
  const int is_ = D == 0 ? src_face(i, bcx, P.is, P.ie, P.n) : src_cell(i, bcx, P.is, P.ie, P.n);
  const int js = D == 1 ? src_face(j, bcy, P.is, P.ie, P.n) : src_cell(j, bcy, P.is, P.ie, P.n);
  const int ks = D == 2 ? src_face(k, bcz, P.is, P.ie, P.n) : src_cell(k, bcz, P.is, P.ie, P.n);
  if (is_ == i && js == j && ks == k) return;
  const Ix ix{P.nt, P.px};
  f.Bf[D][ix.face(D, m, k, j, i)] = f.Bf[D][ix.face(D, m, ks, js, is_)];
}

__global__ void __launch_bounds__(256) k_update_cells(const __grid_constant__ Par P, const __grid_constant__ DrvFields f,
                                                      double a, double b, double dt) {
  const unsigned n = (unsigned)P.n;
  const unsigned tot = (unsigned)P.nmb * n * n * n;
  const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= tot) return;
  const int i = (int)(t % n) + P.is;
  unsigned r = t / n;
  const int j = (int)(r % n) + P.is; r /= n;
  const int k = (int)(r % n) + P.is;
  const int m = (int)(r / n);
  const Ix ix{P.nt, P.px};
  const long long c = ix.cell(m, k, j, i);
#pragma unroll
  for (int v = 0; v < 5; ++v) f.U[v][c] = a * f.U0[v][c] + b * (f.U[v][c] + dt * f.dU[v][c]);
}

// D-faces of interior cells: normal index in [is, ie+1], transverse in [is, ie]
template <int D>
__global__ void __launch_bounds__(256) k_update_faces(const __grid_constant__ Par P, const __grid_constant__ DrvFields f,
                                                      double a, double b, double dt) {
  const unsigned n = (unsigned)P.n;
  const unsigned ni = n + (D == 0), nj = n + (D == 1), nk = n + (D == 2);
  const unsigned tot = (unsigned)P.nmb * nk * nj * ni;
  const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= tot) return;
  const int i = (int)(t % ni) + P.is;
  unsigned r = t / ni;
  const int j = (int)(r % nj) + P.is; r /= nj;
  const int k = (int)(r % nk) + P.is;
  const int m = (int)(r / nk);
  const Ix ix{P.nt, P.px};
  const double idx = 1.0 / f.dx[3 * m + 0], idy = 1.0 / f.dx[3 * m + 1], idz = 1.0 / f.dx[3 * m + 2];
  double dB;
  if (D == 0)
    dB = -((f.E[2][ix.edge(2, m, k, j + 1, i)] - f.E[2][ix.edge(2, m, k, j, i)]) * idy -
           (f.E[1][ix.edge(1, m, k + 1, j, i)] - f.E[1][ix.edge(1, m, k, j, i)]) * idz);
  else if (D == 1)
    dB = -((f.E[0][ix.edge(0, m, k + 1, j, i)] - f.E[0][ix.edge(0, m, k, j, i)]) * idz -
           (f.E[2][ix.edge(2, m, k, j, i + 1)] - f.E[2][ix.edge(2, m, k, j, i)]) * idx);
  else
    dB = -((f.E[1][ix.edge(1, m, k, j, i + 1)] - f.E[1][ix.edge(1, m, k, j, i)]) * idx -
           (f.E[0][ix.edge(0, m, k, j + 1, i)] - f.E[0][ix.edge(0, m, k, j, i)]) * idy);
  const long long q = ix.face(D, m, k, j, i);
  f.Bf[D][q] = a * f.B0[D][q] + b * (f.Bf[D][q] + dt * dB);
}

__global__ void __launch_bounds__(256) k_or_bytes(unsigned char* __restrict__ acc, const unsigned char* __restrict__ src,
                                                  long long nbytes) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < nbytes; q += stride) acc[q] |= src[q];
}

// ---- same-level ghost exchange between MeshBlocks -----------------------------------
// nbr[m][27]: block at offset (oz+1)*9+(oy+1)*3+(ox+1), -1 = none.  FLD 0: the five cell fields;
// FLD 1..3: the face field of direction FLD-1.  pass 0 copies from existing offset blocks, pass 1
// applies bc[d] on the sides that have no face neighbour (sources may be ghosts filled in pass 0).
__device__ __forceinline__ int region_cell(int q, int is, int ie) { return q < is ? -1 : (q > ie ? 1 : 0); }
__device__ __forceinline__ int region_face(int q, int is, int ie, bool upper_is_image) {
  if (q < is) return -1;
  if (q > ie + 1) return 1;
  return (q == ie + 1 && upper_is_image) ? 1 : 0;
}

template <int FLD>
__global__ void __launch_bounds__(256) k_exchange(const __grid_constant__ Par P, const __grid_constant__ DrvFields f,
                                                  const int* __restrict__ nbr, int pass, int bcx, int bcy, int bcz) {
  constexpr int D = FLD - 1;
  const unsigned nt = (unsigned)P.nt;
  const unsigned ni = nt + (D == 0), nj = nt + (D == 1), nk = nt + (D == 2);
  const unsigned tot = (unsigned)P.nmb * nk * nj * ni;
  const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= tot) return;
  const int i = (int)(t % ni);
  unsigned r = t / ni;
  const int j = (int)(r % nj); r /= nj;
  const int k = (int)(r % nk);
  const int m = (int)(r / nk);
  const int* nb = nbr + 27 * m;
  const int is = P.is, ie = P.ie, n = P.n;
  const int ox = D == 0 ? region_face(i, is, ie, nb[14] >= 0 || bcx == 0) : region_cell(i, is, ie);
  const int oy = D == 1 ? region_face(j, is, ie, nb[16] >= 0 || bcy == 0) : region_cell(j, is, ie);
  const int oz = D == 2 ? region_face(k, is, ie, nb[22] >= 0 || bcz == 0) : region_cell(k, is, ie);
  if (ox == 0 && oy == 0 && oz == 0) return;
  const int mb = nb[(oz + 1) * 9 + (oy + 1) * 3 + (ox + 1)];
  int ms, is_, js, ks;
  if (pass == 0) {
    if (mb < 0) return;
    ms = mb; is_ = i - ox * n; js = j - oy * n; ks = k - oz * n;
  } else {
    if (mb >= 0) return;
    ms = m; is_ = i; js = j; ks = k;
    if (ox != 0 && nb[13 + ox] < 0) is_ = D == 0 ? src_face(i, bcx, is, ie, n) : src_cell(i, bcx, is, ie, n);
    if (oy != 0 && nb[13 + 3 * oy] < 0) js = D == 1 ? src_face(j, bcy, is, ie, n) : src_cell(j, bcy, is, ie, n);
    if (oz != 0 && nb[13 + 9 * oz] < 0) ks = D == 2 ? src_face(k, bcz, is, ie, n) : src_cell(k, bcz, is, ie, n);
    if (is_ == i && js == j && ks == k) return;
  }
  const Ix ix{P.nt, P.px};
  if (FLD == 0) {
    const long long dst = ix.cell(m, k, j, i), src = ix.cell(ms, ks, js, is_);
#pragma unroll
    for (int v = 0; v < 5; ++v) f.U[v][dst] = f.U[v][src];
  } else {
    f.Bf[D < 0 ? 0 : D][ix.face(D < 0 ? 0 : D, m, k, j, i)] = f.Bf[D < 0 ? 0 : D][ix.face(D < 0 ? 0 : D, ms, ks, js, is_)];
  }
}

// ---------------------------------------------------------------- ghost slabs for the cross-GPU exchange
// A slab is the part of one block that a block at the other end of neighbour code c reads in pass 0 of
// k_exchange (c = (oz+1)*9+(oy+1)*3+(ox+1), the offset from the reader to this block).  Per axis with
// offset o: cell-like indices [n, n+ng) for o = -1, [ng, 2ng) for o = +1, [ng, ng+n) for o = 0; along a
// face field's normal [n, n+ng), [ng, 2ng+1), [ng, ng+n+1).  Order in the buffer: the five cell fields,
// then B~f^x, B~f^y, B~f^z, each k-major.  include/ak.h: ak_halo_slab_elems, ak_halo_pack, ak_halo_unpack.
__host__ __device__ __forceinline__ int slab_start(int o, int n, int ng) { return o < 0 ? n : ng; }
__host__ __device__ __forceinline__ int slab_extent(int o, int n, int ng, bool normal) {
  if (normal) return o < 0 ? ng : (o > 0 ? ng + 1 : n + 1);
  return o != 0 ? ng : n;
}
__host__ __device__ inline long long slab_elems(int code, int n, int ng) {
  const int o[3] = {code % 3 - 1, (code / 3) % 3 - 1, code / 9 - 1};
  long long c[3], f[3];
  for (int a = 0; a < 3; ++a) { c[a] = slab_extent(o[a], n, ng, false); f[a] = slab_extent(o[a], n, ng, true); }
  return 5 * c[0] * c[1] * c[2] + f[0] * c[1] * c[2] + c[0] * f[1] * c[2] + c[0] * c[1] * f[2];
}

// desc[3*q + {0,1,2}] = block, code, offset of the slab in buf (elements).  grid (chunks, ndesc).
template <bool UNPACK>
__global__ void __launch_bounds__(256) k_halo_slabs(const __grid_constant__ Par P, const __grid_constant__ DrvFields f,
                                                    const long long* __restrict__ desc, double* __restrict__ buf,
                                                    int nblocks) {
  const long long* dq = desc + 3LL * blockIdx.y;
  const int m = (int)dq[0], code = (int)dq[1];
  if (m < 0 || m >= nblocks || code < 0 || code > 26) return;
  double* b = buf + dq[2];
  const int o[3] = {code % 3 - 1, (code / 3) % 3 - 1, code / 9 - 1};
  const int n = P.n, ng = P.is;
  const int s0 = slab_start(o[0], n, ng), s1 = slab_start(o[1], n, ng), s2 = slab_start(o[2], n, ng);
  const Ix ix{P.nt, P.px};
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
#pragma unroll 1
  for (int fld = 0; fld < 8; ++fld) {
    const int D = fld - 5;                                   // normal of a face field, < 0 for cell fields
    const int ex = slab_extent(o[0], n, ng, D == 0), ey = slab_extent(o[1], n, ng, D == 1),
              ez = slab_extent(o[2], n, ng, D == 2);
    const int cnt = ex * ey * ez;
    double* fp = D < 0 ? f.U[fld] : f.Bf[D];
    for (int e = tid; e < cnt; e += nth) {
      const int i = e % ex, j = (e / ex) % ey, k = e / (ex * ey);
      const long long g = D < 0 ? ix.cell(m, k + s2, j + s1, i + s0) : ix.face(D, m, k + s2, j + s1, i + s0);
      if (UNPACK) fp[g] = b[e]; else b[e] = fp[g];
    }
    b += cnt;
  }
}

}  // namespace ak
