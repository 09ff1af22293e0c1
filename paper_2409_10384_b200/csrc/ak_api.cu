// ak_api.cu — the C-ABI of include/ak.h: context, validation, launch sequence of one stage.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a --fmad=false -lineinfo (see build.py).
#include "../../include/ak.h"
#include "ak_source.cuh"
#ifndef AK_FLUX_TMA
#define AK_FLUX_TMA 1   // 1: TMA-staged sweeps (ak_flux_tma.cuh) when n is even and a face row fits a block
#endif
#include "ak_flux_tma.cuh"
#include "ak_flux_pencil.cuh"
#include "ak_flux_static.cuh"
#include "ak_driver.cuh"

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

using namespace ak;

namespace {

enum { KC_C2P = 0, KC_FX, KC_FY, KC_FZ, KC_FOFC_TEST, KC_FOFC_FIX, KC_CT, KC_SRC, KC_N };
constexpr int MAXCH = 64;     // most chunks of an overlapped schedule (counter slots per context)
// overlapped schedule: blocks per SM the memory-bound classes may take beside the sweeps (0 = no cap)
#ifndef AK_OV_CAP_C2P_DEFAULT
#define AK_OV_CAP_C2P_DEFAULT 3
#define AK_OV_CAP_FOFC_DEFAULT 3
#define AK_OV_CAP_FIX_DEFAULT 2
#define AK_OV_CAP_CT_DEFAULT 4
#define AK_OV_CAP_SRC_DEFAULT 2
#define AK_OV_SMEM_PAD_DEFAULT 0
#endif
#ifndef AK_PENCIL_WI_DEFAULT
#define AK_PENCIL_WI_DEFAULT 0      // x-lanes per block of the y/z pencil sweeps (even; 0 = k_flux_tma tiles)
#endif

struct Sizes {
  long long cell, xf, yf, zf, ex, ey, ez;   // elements per batch
};

}  // namespace

struct ak_ctx {
  ak_params hp;
  Par P;
  Sizes sz;
  cudaStream_t stream;
  bool have_metric, have_flux;
  const double* adm[16];
  // scratch
  double* F[21];
  double* Ecc[3];
  unsigned char* flag_own;
  unsigned int* list;
  unsigned int* count;          // [4]
  unsigned long long* stats;    // [S_NSTAT]
  double* dx;
  // host staging for ak_rhs_host
  double* stg_U[5]; double* stg_Bf[3]; double* stg_W[8]; double* stg_dU[5]; double* stg_E[3];
  unsigned char* stg_flag; unsigned char* stg_status;
  bool have_stg;
  // overlapped schedule (ak_set_overlap): chunks of blocks on internal streams
  int ov_chunks;                // < 2: serial
  cudaStream_t ovs[3];          // con2prim, sweeps, FOFC/CT/sources (ovs[2] may equal ovs[0])
  cudaEvent_t* ov_ev; int ov_nev;
  int cap[8];                   // grid caps (blocks) per kernel class in the overlapped schedule, 0 = none
  int sweep_smem_pad;           // bytes: dynamic shared memory the sweeps ask for at least when overlapped
  unsigned int* zflags;         // [nmb] per-block zero-field flags written by k_con2prim (Fields::zflags)
  unsigned char* rowflag;       // [nmb nt nt] per-row flags written by k_con2prim (Fields::rowflag)
  unsigned int* tlist;          // [6 tcap] static / general tiles per direction (k_split_tiles), [6] their counts behind
  unsigned int tcap;            // nmb (n+2) max_d tiles_d
  int ct_fused;                 // 1: the three CT components in one launch (k_ct_all)
  int split_blocks;             // 1: static tiles take k_flux_static (serial schedule, part (1) in the same call)
  // CUDA-graph replay of the serial stage (ak_set_graph): a few instantiated graphs keyed on the arguments
  int graph_on;
  cudaStream_t gstream;         // capture stream (the caller's may be the legacy default stream, which cannot capture)
  struct GraphSlot { unsigned long long key; cudaGraphExec_t exec; unsigned long long age; } gslot[4];
  unsigned long long gclock;
  long long graph_replays;      // stages replayed from a graph since ak_set_graph (diagnostic)
  int fuse_src;                 // 1: part (6) runs inside the FOFC-test kernel (+ k_src_fix), 0: k_div_src after the re-flux
  int tile_tm;                  // tile kernels: stage tiles with tensor-map box copies (1) or row by row (0)
  int pencil_wi;                // y/z sweeps: x-lanes per block of k_flux_pencil (0: tile kernels k_flux_tma)
  // FOFC stage blend (ak_set_fofc_blend)
  const double* blendU0[5]; double blend_a, blend_b;
  // stage-driver registers (ak_advance), allocated on first use
  double* regU0[5]; double* regB0[3]; double* reg_dU[5]; double* regE[3]; unsigned char* reg_flag;
  bool have_reg;
  int* nbr;                     // device copy of the neighbour table (ak_set_neighbors), or NULL
  int nmb_total;                // blocks in the caller's arrays (own + mirrors), 0 = nmb
  // pipelined host entry (ak_rhs_host): two lanes, each a child context over `lane_chunk` blocks
  // with its own stream and device staging; chunks alternate between the lanes
  double* host_dx;              // [nmb][3] host copy
  ak_ctx* lane[2]; int lane_chunk;
  double* lane_buf[2][24];      // staging: U5 Bf3 W8 dU5 E3
  unsigned char* lane_mask[2][2];
  unsigned long long* lane_stats_h;   // pinned [nchunks][S_NSTAT + 4]
  bool stats_from_host; ak_stats host_acc;
  // timing
  bool timing;
  cudaEvent_t ev0, ev1;
  double ms[KC_N];
  long long launches[KC_N];
  struct Pending { int which; cudaEvent_t a, b; };
  Pending* pend; int npend, cappend;
};

namespace {

#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { \
  last_cuda_error = e_; return e_ == cudaErrorMemoryAllocation ? AK_ENOMEM : AK_ECUDA; } } while (0)

thread_local cudaError_t last_cuda_error = cudaSuccess;

inline bool finite_pos(double x) { return std::isfinite(x) && x > 0.0; }

int validate(const ak_params* p, const double* dx3) {
  if (!p || !dx3) return AK_EINVAL;
  if (p->nmb < 1 || p->n < 2 || p->ng != 4) return AK_EINVAL;
  if (!(std::isfinite(p->gamma_ad) && p->gamma_ad > 1.0)) return AK_EINVAL;
  if (!finite_pos(p->rho_atm) || !finite_pos(p->T_atm) || !finite_pos(p->f_thr)) return AK_EINVAL;
  if (!(p->mag_max > 0.0)) return AK_EINVAL;   // +inf allowed, NaN rejected
  if (p->recon < 0 || p->recon > 4 || p->riemann < 0 || p->riemann > 1) return AK_EINVAL;
  if (p->fofc < 0 || p->fofc > 1 || p->fofc_riemann < 0 || p->fofc_riemann > 1) return AK_EINVAL;
  if (std::isnan(p->dmp_M) || (p->dmp_M > 0.0 && p->dmp_M < 1.0)) return AK_EINVAL;
  if (p->c2p_max_iter < 1 || p->c2p_max_iter > 1000) return AK_EINVAL;
  if (!(p->c2p_tol > 0.0 && p->c2p_tol < 1.0)) return AK_EINVAL;
  if (p->device < 0) return AK_EINVAL;
  const long long nt = p->n + 8;
  // face-list entries are 32-bit cell indices
  if ((long long)p->nmb * (nt + 1) * (nt + 1) * (nt + 4) >= (1LL << 31)) return AK_EINVAL;
  for (long long q = 0; q < 3LL * p->nmb; ++q)
    if (!finite_pos(dx3[q])) return AK_EINVAL;
  return AK_OK;
}

// the equation-of-state part of Par (ak_set_eos_hybrid), for the child contexts of ak_rhs_host
inline void copy_eos(Par& d, const Par& s) {
  d.eos = s.eos; d.nseg = s.nseg; d.gth = s.gth; d.gthm1 = s.gthm1; d.P_atm = s.P_atm;
  for (int i = 0; i < 4; ++i) { d.ppK[i] = s.ppK[i]; d.ppG[i] = s.ppG[i]; d.ppa[i] = s.ppa[i]; }
  for (int i = 0; i < 3; ++i) d.pprb[i] = s.pprb[i];
}

inline unsigned nblk(long long n, int t) { return (unsigned)((n + t - 1) / t); }

// One launch target: a contiguous range of blocks (Par.nmb of them, every field pointer of Fields moved to
// the first) on a stream.  Serial schedule: the whole batch on the context's stream.  Overlapped schedule
// (ak_set_overlap): one chunk of blocks on one of the internal streams.
struct Lane {
  const Par& P;
  const Fields& f;
  cudaStream_t st;
  bool ov;          // part of an overlapped schedule: grid caps and the sweep shared-memory pad apply
};

struct Timer {
  ak_ctx* c; int which; cudaEvent_t a, b; bool on; cudaStream_t st;
  Timer(ak_ctx* c_, int w, cudaStream_t st_) : c(c_), which(w), on(c_->timing), st(st_) {
    if (on) {
      cudaEventCreate(&a); cudaEventCreate(&b);
      cudaEventRecord(a, st);
    }
  }
  ~Timer() {
    if (!on) return;
    cudaEventRecord(b, st);
    if (c->npend == c->cappend) {
      int nc = c->cappend ? 2 * c->cappend : 256;
      ak_ctx::Pending* np = (ak_ctx::Pending*)realloc(c->pend, sizeof(ak_ctx::Pending) * nc);
      if (!np) { cudaEventDestroy(a); cudaEventDestroy(b); return; }
      c->pend = np; c->cappend = nc;
    }
    c->pend[c->npend++] = {which, a, b};
  }
};

void fill_fields(ak_ctx* c, Fields& f) {
  memset(&f, 0, sizeof(f));
  for (int q = 0; q < 16; ++q) f.adm[q] = c->adm[q];
  for (int q = 0; q < 21; ++q) f.F[q] = c->F[q];
  for (int q = 0; q < 3; ++q) f.Ecc[q] = c->Ecc[q];
  f.list = c->list;
  f.count = c->count;
  f.stats = c->stats;
  f.dx = c->dx;
  f.flag = c->flag_own;
  for (int q = 0; q < 5; ++q) f.U0[q] = c->blendU0[q];
  f.fa = c->blend_a; f.fb = c->blend_b;
}

// Fields / Par of the sub-batch of blocks [m0, m0 + nb): every pointer moved to block m0 of its own layout;
// counters and the flagged-cell list are the slots of chunk `ci`.
void chunk_fields(const ak_ctx* c, const Fields& f, int m0, int nb, int ci, Fields& g, Par& Pc) {
  Pc = c->P;
  Pc.nmb = nb;
  g = f;
  const long long nt = c->P.nt, px = c->P.px, n = c->P.n;
  const long long cell = nt * nt * nt * m0;
  const long long fsz[3] = {nt * nt * px * m0, nt * (nt + 1) * nt * m0, (nt + 1) * nt * nt * m0};
  const long long esz[3] = {(nt + 1) * (nt + 1) * nt * m0, (nt + 1) * nt * px * m0, nt * (nt + 1) * px * m0};
  for (int q = 0; q < 5; ++q) { g.U[q] += cell; if (g.dU[q]) g.dU[q] += cell; if (g.U0[q]) g.U0[q] += cell; }
  for (int q = 0; q < 3; ++q) { g.Bf[q] += fsz[q]; g.Ecc[q] += cell; if (g.E[q]) g.E[q] += esz[q]; }
  for (int q = 0; q < 16; ++q) g.adm[q] += cell;
  for (int q = 0; q < 8; ++q) g.W[q] += cell;
  for (int q = 0; q < 21; ++q) g.F[q] += fsz[q / 7];
  g.flag += cell;
  if (g.zflags) g.zflags += m0;
  if (g.rowflag) g.rowflag += nt * nt * m0;
  if (g.status) g.status += cell;
  if (g.M[0]) for (int q = 0; q < 10; ++q) g.M[q] += cell;
  g.dx += 3LL * m0;
  g.list += (n + 2) * (n + 2) * (n + 2) * m0;
  g.count += 4 * ci;
  g.stats += (long long)S_NSTAT * ci;
}

// 16-byte alignment of every caller field pointer ("Base pointers 16-B aligned (checked ->
// AK_EINVAL)"): the TMA-staged sweeps copy rows of W and of the metric with cp.async.bulk / tensor maps,
// which fault on a global address that is not a multiple of 16.
inline bool al16(const void* p) { return p && (((uintptr_t)p) & 15u) == 0; }

bool set_cons(Fields& f, const ak_cons* U) {
  if (!U || !al16(U->D) || !al16(U->Sx) || !al16(U->Sy) || !al16(U->Sz) || !al16(U->tau)) return false;
  f.U[0] = U->D; f.U[1] = U->Sx; f.U[2] = U->Sy; f.U[3] = U->Sz; f.U[4] = U->tau;
  return true;
}
bool set_faceB(Fields& f, const ak_faceB* B) {
  if (!B || !al16(B->bx) || !al16(B->by) || !al16(B->bz)) return false;
  f.Bf[0] = B->bx; f.Bf[1] = B->by; f.Bf[2] = B->bz;
  return true;
}
bool set_prim(Fields& f, const ak_prim* W) {
  if (!W || !al16(W->rho) || !al16(W->ux) || !al16(W->uy) || !al16(W->uz) || !al16(W->p) || !al16(W->bccx) ||
      !al16(W->bccy) || !al16(W->bccz))
    return false;
  f.W[0] = W->rho; f.W[1] = W->ux; f.W[2] = W->uy; f.W[3] = W->uz; f.W[4] = W->p;
  f.W[5] = W->bccx; f.W[6] = W->bccy; f.W[7] = W->bccz;
  return true;
}

// grid of a grid-stride kernel: what covers the items, or the cap of its class when one is set
inline unsigned capped(long long items, int threads, int cap_blocks) {
  const long long need = (items + threads - 1) / threads;
  return (unsigned)((cap_blocks > 0 && need > cap_blocks) ? cap_blocks : need);
}

int launch_c2p(ak_ctx* c, const Lane& L, bool with_emf) {
  Timer t(c, KC_C2P, L.st);
  CK(cudaMemsetAsync(L.f.stats, 0, sizeof(unsigned long long) * 3, L.st));
  if (L.f.zflags) CK(cudaMemsetAsync(L.f.zflags, 0, sizeof(unsigned) * L.P.nmb, L.st));   // this pass sets the bits
  if (L.f.rowflag) CK(cudaMemsetAsync(L.f.rowflag, 0, (size_t)L.P.nmb * L.P.nt * L.P.nt, L.st));
  const long long ncell = (long long)L.P.nmb * L.P.nt * L.P.nt * L.P.nt;
  const unsigned g = capped(ncell, 128, L.ov ? c->cap[KC_C2P] : 0);
  const bool stride = (long long)g * 128 < ncell;       // a capped grid needs the grid-stride form
  if (stride) {
    if (L.P.eos) {
      if (with_emf) k_con2prim<true, 1, true><<<g, 128, 0, L.st>>>(L.P, L.f);
      else k_con2prim<false, 1, true><<<g, 128, 0, L.st>>>(L.P, L.f);
    } else if (with_emf) k_con2prim<true, 0, true><<<g, 128, 0, L.st>>>(L.P, L.f);
    else k_con2prim<false, 0, true><<<g, 128, 0, L.st>>>(L.P, L.f);
  } else if (L.P.eos) {
    if (with_emf) k_con2prim<true, 1><<<g, 128, 0, L.st>>>(L.P, L.f);
    else k_con2prim<false, 1><<<g, 128, 0, L.st>>>(L.P, L.f);
  } else if (with_emf) k_con2prim<true><<<g, 128, 0, L.st>>>(L.P, L.f);
  else k_con2prim<false><<<g, 128, 0, L.st>>>(L.P, L.f);
  c->launches[KC_C2P] += 1;
  CK(cudaGetLastError());
  return AK_OK;
}

// ---- y/z sweeps on whole pencils with tensor-map TMA (ak_flux_pencil.cuh) -------------------------------
typedef CUresult (*TmapEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                 const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                 CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
// the driver's encoder through the runtime (no link against libcuda); NULL if this driver has none
TmapEncodeFn tmap_encoder() {
  static TmapEncodeFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (TmapEncodeFn)p;
    cudaGetLastError();
  }
  return fn;
}

// Tensor maps of the 17 fields of a sweep of direction DIR: every cell field is the rank-3 tensor
// (i: nt, j: nt, K = m nt + k); boxW / boxM are the boxes of the primitive and of the metric fields.
template <int DIR>
bool field_maps(const Par& P, const Fields& f, const cuuint32_t boxW[3], const cuuint32_t boxM[3], TileMaps& M) {
  TmapEncodeFn enc = tmap_encoder();
  if (!enc) return false;
  constexpr int t1 = (DIR + 1) % 3, t2 = (DIR + 2) % 3;
  const cuuint64_t nt = (cuuint64_t)P.nt;
  const cuuint64_t dims[3] = {nt, nt, nt * (cuuint64_t)P.nmb};
  const cuuint64_t strides[2] = {nt * 8, nt * nt * 8};                  // bytes, dimensions 1 and 2
  const cuuint32_t estr[3] = {1, 1, 1};
  auto one = [&](CUtensorMap* m, const double* base, const cuuint32_t* box) {
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(base), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
  };
  const int var[7] = {0, 1, 2, 3, 4, 5 + t1, 5 + t2};
  for (int v = 0; v < 7; ++v) if (!one(&M.w[v], f.W[var[v]], boxW)) return false;
  for (int q = 0; q < 10; ++q) {
    const int fld = q == 0 ? 6 : (q < 4 ? 6 + q : q - 4);               // alp, betx..betz, gxx..gzz
    if (!one(&M.m[q], f.adm[fld], boxM)) return false;
  }
  return true;
}

#ifndef AK_FLUX_CELL_MASK
#define AK_FLUX_CELL_MASK 1   // bit d set: direction d uses the reconstruct-once variant k_flux_tma_cell
#endif

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel function (per device), not to a
// context: two live contexts of different n share one instantiation and need different amounts.  The
// attribute is therefore only ever RAISED, tracked per instantiation and device.
template <typename K>
int raise_smem_attr(K kern, int device, size_t smem, int (&have)[64]) {
  const int d = device & 63;
  if ((int)smem > have[d]) {
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    have[d] = (int)smem;
  }
  return AK_OK;
}

template <int DIR, int RECON, int EOS>
int launch_flux_tma_eos(ak_ctx* c, const Lane& L, int NA, unsigned grid, int bd, size_t smem, const TileMaps& M,
                        int use_tm) {
  auto kern = ((AK_FLUX_CELL_MASK >> DIR) & 1) ? k_flux_tma_cell<DIR, RECON, EOS> : k_flux_tma<DIR, RECON, EOS>;
  static int have[64] = {0};
  const int r = raise_smem_attr(kern, c->hp.device, smem, have);
  if (r != AK_OK) return r;
  kern<<<grid, bd, smem, L.st>>>(L.P, L.f, NA, M, use_tm);
  return AK_OK;
}

template <int DIR, int RECON>
int launch_flux_tma(ak_ctx* c, const Lane& L, int NA, unsigned grid, int bd, size_t smem, const TileMaps& M,
                    int use_tm) {
  return L.P.eos ? launch_flux_tma_eos<DIR, RECON, 1>(c, L, NA, grid, bd, smem, M, use_tm)
                 : launch_flux_tma_eos<DIR, RECON, 0>(c, L, NA, grid, bd, smem, M, use_tm);
}

template <int DIR>
bool pencil_maps(const Par& P, const Fields& f, int WI, PencilMaps& M) {
  const cuuint32_t nt = (cuuint32_t)P.nt;
  const cuuint32_t box[3] = {(cuuint32_t)WI, DIR == 1 ? nt : 1u, DIR == 1 ? 1u : nt};
  return field_maps<DIR>(P, f, box, box, M);
}

template <int DIR, int RECON, int EOS>
int launch_pencil_eos(ak_ctx* c, const Lane& L, const PencilMaps& M, int WI, int tile_d, int i_first, int ntile_i,
                      unsigned grid, int bd, size_t smem) {
  auto kern = k_flux_pencil<DIR, RECON, EOS>;
  static int have[64] = {0};
  const int r = raise_smem_attr(kern, c->hp.device, smem, have);
  if (r != AK_OK) return r;
  kern<<<grid, bd, smem, L.st>>>(L.P, L.f, M, WI, tile_d, i_first, ntile_i);
  return AK_OK;
}

// returns AK_OK when launched, 1 when the pencil kernel does not apply (caller falls back)
template <int DIR>
int launch_pencil(ak_ctx* c, const Lane& L) {
  const int n = L.P.n, nt = L.P.nt;
  if (c->pencil_wi < 2 || n % 2 != 0) return 1;
  // x-lanes [is-1, ie+1] = [3, n+4] in tiles of WI lanes starting at the even lane 2 (a box must start on
  // a 16-byte boundary: an odd first lane faults).  WI: even, at most the configured width, the block within
  // AK_PENCIL_MAXT threads, least lanes wasted, the wider the better.
  const int i_first = 2, lanes = n + 3;
  int WI = 0, waste = 1 << 30;
  for (int w = 4; w <= c->pencil_wi; w += 2) {
    if (((w * (n + 4) + 31) / 32) * 32 > AK_PENCIL_MAXT) break;
    const int ws = (lanes + w - 1) / w * w - lanes;
    if (ws <= waste) { waste = ws; WI = w; }
  }
  if (WI == 0) return 1;
  const int bd = ((WI * (n + 4) + 31) / 32) * 32;
  PencilMaps M;
  if (!pencil_maps<DIR>(L.P, L.f, WI, M)) return 1;
  const int ntile_i = (lanes + WI - 1) / WI;
  const int tile_d = ((nt * WI + 15) / 16) * 16;
  size_t dbl = (size_t)17 * tile_d + (size_t)7 * bd;
  if ((size_t)21 * bd > dbl) dbl = (size_t)21 * bd;
  const size_t smem = sizeof(double) * dbl;
  if (smem > 200 * 1024) return 1;
  const unsigned grid = (unsigned)((long long)L.P.nmb * (n + 2) * ntile_i);
  int r;
#define AK_PENCIL_CASE(RC)                                                                                       \
  r = L.P.eos ? launch_pencil_eos<DIR, RC, 1>(c, L, M, WI, tile_d, i_first, ntile_i, grid, bd, smem)            \
              : launch_pencil_eos<DIR, RC, 0>(c, L, M, WI, tile_d, i_first, ntile_i, grid, bd, smem)
  switch (L.P.recon) {
    case 0: AK_PENCIL_CASE(0); break;
    case 1: AK_PENCIL_CASE(1); break;
    case 3: AK_PENCIL_CASE(3); break;
    case 4: AK_PENCIL_CASE(4); break;
    default: AK_PENCIL_CASE(2); break;
  }
#undef AK_PENCIL_CASE
  if (r != AK_OK) return r;
  CK(cudaGetLastError());
  return AK_OK;
}

// do the tile kernels apply to this batch (else launch_flux falls back to k_flux and knows no block lists)
// the tiling of a sweep of direction d: NA rows (x) / face rows (y, z) per tile, `tiles` tiles along the tiled extent;
// for the general kernel (face or cell variant) and for k_flux_static
void sweep_tiling(int d, int n, bool for_static, int& NA, int& tiles) {
  const int e = n + 2;
  const int cellv = for_static ? 0 : ((AK_FLUX_CELL_MASK >> d) & 1);
  const int nfi = for_static ? (d == 0 ? ((AK_STATIC_ONCE_MASK & 1) ? n + 4 : n + 3) : e)
                             : (cellv ? (d == 0 ? n + 4 : e) : (d == 0 ? n + 3 : e));
  const int nfd = d == 0 ? e : n + 3;
  const int namax = TMA_THREADS / nfi - (cellv && d != 0 ? 1 : 0);
  if (namax < 1) { NA = 1; tiles = nfd; return; }     // a row does not fit a block: the tile kernels do not apply
  tiles = (nfd + namax - 1) / namax;
  NA = (nfd + tiles - 1) / tiles;
}

bool tile_kernels_apply(const ak_ctx* c, const Par& P) {
  const int n = P.n, e = n + 2;
  if (!AK_FLUX_TMA || n % 2 != 0 || c->pencil_wi > 0) return false;
  for (int d = 0; d < 3; ++d) {
    const int cellv = (AK_FLUX_CELL_MASK >> d) & 1;
    const int nfi = cellv ? (d == 0 ? n + 4 : e) : (d == 0 ? n + 3 : e);
    if (nfi * (cellv && d != 0 ? 2 : 1) > TMA_THREADS) return false;
    const int nfd = d == 0 ? e : n + 3;
    const int namax = TMA_THREADS / nfi - (cellv && d != 0 ? 1 : 0);
    const int tiles = (nfd + namax - 1) / namax, NA = (nfd + tiles - 1) / tiles;
    const int maxW = d == 0 ? NA : NA + 5, maxM = d == 0 ? NA : NA + 1;
    if (sizeof(double) * ((size_t)7 * tile_slot(maxW, P.nt) + (size_t)10 * tile_slot(maxM, P.nt) + (cellv ? 7 * TMA_THREADS : 0)) >
        200 * 1024)
      return false;
  }
  return true;
}

template <int DIR, int RECON>
int launch_flux_static_r(ak_ctx* c, const Lane& L, int NA, unsigned grid, int bd, size_t smem, const TileMaps& M) {
  static int have0[64] = {0}, have1[64] = {0};
  if (L.P.eos) {
    auto kern = k_flux_static<DIR, RECON, 1>;
    const int r = raise_smem_attr(kern, c->hp.device, smem, have1);
    if (r != AK_OK) return r;
    kern<<<grid, bd, smem, L.st>>>(L.P, L.f, NA, M);
  } else {
    auto kern = k_flux_static<DIR, RECON, 0>;
    const int r = raise_smem_attr(kern, c->hp.device, smem, have0);
    if (r != AK_OK) return r;
    kern<<<grid, bd, smem, L.st>>>(L.P, L.f, NA, M);
  }
  return AK_OK;
}

template <int DIR>
int launch_flux_static(ak_ctx* c, const Lane& L) {
  const int n = L.P.n, nt = L.P.nt, e = n + 2;
  const int nfi = DIR == 0 ? ((AK_STATIC_ONCE_MASK & 1) ? n + 4 : n + 3) : e;   // threads per tile row
  int NA, tiles;
  sweep_tiling(DIR, n, true, NA, tiles);
  const int maxW = DIR == 0 ? NA : NA + 5, maxM = DIR == 0 ? NA : NA + 1;
  const size_t smem = sizeof(double) * ((size_t)2 * tile_slot(maxW, nt) + (size_t)10 * tile_slot(maxM, nt));
  TileMaps M;
  const cuuint32_t unt = (cuuint32_t)nt;
  const cuuint32_t bW[3] = {unt, DIR == 2 ? 1u : (cuuint32_t)maxW, DIR == 2 ? (cuuint32_t)maxW : 1u};
  const cuuint32_t bM[3] = {unt, DIR == 2 ? 1u : (cuuint32_t)maxM, DIR == 2 ? (cuuint32_t)maxM : 1u};
  if (!field_maps<DIR>(L.P, L.f, bW, bM, M)) return AK_ECUDA;
  const unsigned grid = (unsigned)((long long)L.P.nmb * e * tiles);
  const int bd = ((NA * nfi + 31) / 32) * 32;
  int r;
  switch (L.P.recon) {
    case 0: r = launch_flux_static_r<DIR, 0>(c, L, NA, grid, bd, smem, M); break;
    case 1: r = launch_flux_static_r<DIR, 1>(c, L, NA, grid, bd, smem, M); break;
    case 3: r = launch_flux_static_r<DIR, 3>(c, L, NA, grid, bd, smem, M); break;
    case 4: r = launch_flux_static_r<DIR, 4>(c, L, NA, grid, bd, smem, M); break;
    default: r = launch_flux_static_r<DIR, 2>(c, L, NA, grid, bd, smem, M); break;
  }
  if (r != AK_OK) return r;
  CK(cudaGetLastError());
  return AK_OK;
}

template <int DIR>
int launch_flux(ak_ctx* c, const Lane& L) {
  Timer t(c, KC_FX + DIR, L.st);
  const int n = L.P.n, nt = L.P.nt, e = n + 2;
  if (DIR != 0 && c->pencil_wi > 0) {
    const int pr = launch_pencil<(DIR == 0 ? 1 : DIR)>(c, L);
    if (pr == AK_OK) { c->launches[KC_FX + DIR] += 1; return AK_OK; }
    if (pr != 1) return pr;
  }
  constexpr int AK_FLUX_CELL = (AK_FLUX_CELL_MASK >> DIR) & 1;
  // threads per row of a tile: faces (k_flux_tma) or cells (k_flux_tma_cell)
  const int nfi = AK_FLUX_CELL ? (DIR == 0 ? n + 4 : e) : (DIR == 0 ? n + 3 : e);
  // bulk copies need 16-byte-aligned rows: n even, and (for chunk offsets) every field base a multiple of 16
  if (AK_FLUX_TMA && n % 2 == 0 && nfi * (AK_FLUX_CELL && DIR != 0 ? 2 : 1) <= TMA_THREADS) {
    // tile height: as many rows as fit the block, balanced over the extent it tiles
    const int nfd = DIR == 0 ? e : n + 3;
    const int namax = TMA_THREADS / nfi - (AK_FLUX_CELL && DIR != 0 ? 1 : 0);
    const int tiles = (nfd + namax - 1) / namax;
    const int NA = (nfd + tiles - 1) / tiles;
    const int maxW = DIR == 0 ? NA : NA + 5, maxM = DIR == 0 ? NA : NA + 1;
    size_t smem = sizeof(double) * ((size_t)7 * tile_slot(maxW, nt) + (size_t)10 * tile_slot(maxM, nt) +
                                    (AK_FLUX_CELL ? 7 * TMA_THREADS : 0));
    // the tile as 17 tensor-map box copies (one per field) when the driver can encode them, else row by row
    TileMaps M;
    int use_tm = 0;
    if (c->tile_tm) {
      const cuuint32_t unt = (cuuint32_t)nt;
      const cuuint32_t bW[3] = {unt, DIR == 2 ? 1u : (cuuint32_t)maxW, DIR == 2 ? (cuuint32_t)maxW : 1u};
      const cuuint32_t bM[3] = {unt, DIR == 2 ? 1u : (cuuint32_t)maxM, DIR == 2 ? (cuuint32_t)maxM : 1u};
      use_tm = field_maps<DIR>(L.P, L.f, bW, bM, M) ? 1 : 0;
    }
    if (!use_tm) memset(&M, 0, sizeof(M));
    if (AK_FLUX_CELL ? AK_FLUXC_PARK : AK_FLUX_PARK) {   // the spent tile is reused as 21 doubles of parking space per thread
      const size_t park = sizeof(double) * 21 * (size_t)TMA_THREADS;
      if (park > smem) smem = park;
    }
    // overlapped schedule: a larger allocation keeps a third sweep block off the SM, so that the
    // capped memory-bound kernels of the other stream find registers and thread slots there
    if (L.ov && c->sweep_smem_pad > 0 && smem < (size_t)c->sweep_smem_pad) smem = (size_t)c->sweep_smem_pad;
    if (smem <= 200 * 1024) {
      const unsigned grid = (unsigned)((long long)L.P.nmb * e * tiles);
      // threads: one per face (or cell) of the tile, rounded up to whole warps
      const int rows = NA + ((AK_FLUX_CELL && DIR != 0) ? 1 : 0);
      const int bd = ((rows * nfi + 31) / 32) * 32;
      int r;
      switch (L.P.recon) {
        case 0: r = launch_flux_tma<DIR, 0>(c, L, NA, grid, bd, smem, M, use_tm); break;
        case 1: r = launch_flux_tma<DIR, 1>(c, L, NA, grid, bd, smem, M, use_tm); break;
        case 3: r = launch_flux_tma<DIR, 3>(c, L, NA, grid, bd, smem, M, use_tm); break;
        case 4: r = launch_flux_tma<DIR, 4>(c, L, NA, grid, bd, smem, M, use_tm); break;
        default: r = launch_flux_tma<DIR, 2>(c, L, NA, grid, bd, smem, M, use_tm); break;
      }
      if (r != AK_OK) return r;
      CK(cudaGetLastError());
      c->launches[KC_FX + DIR] += 1;
      if (L.f.tlist) {                         // the static tiles of k_split_tiles: the light kernel
        r = launch_flux_static<DIR>(c, L);
        if (r != AK_OK) return r;
        c->launches[KC_FX + DIR] += 1;
      }
      return AK_OK;
    }
  }
  if (L.f.tlist) return AK_ESTATE;             // (lists are only handed out when the tile kernels apply)
  const long long nf = (long long)(n + 3) * (n + 2) * (n + 2) * L.P.nmb;
  const unsigned g = nblk(nf, 128);
  if (L.P.eos) {
    switch (L.P.recon) {
      case 0: k_flux<DIR, 0, 1><<<g, 128, 0, L.st>>>(L.P, L.f); break;
      case 1: k_flux<DIR, 1, 1><<<g, 128, 0, L.st>>>(L.P, L.f); break;
      case 3: k_flux<DIR, 3, 1><<<g, 128, 0, L.st>>>(L.P, L.f); break;
      case 4: k_flux<DIR, 4, 1><<<g, 128, 0, L.st>>>(L.P, L.f); break;
      default: k_flux<DIR, 2, 1><<<g, 128, 0, L.st>>>(L.P, L.f); break;
    }
  } else {
    switch (L.P.recon) {
      case 0: k_flux<DIR, 0><<<g, 128, 0, L.st>>>(L.P, L.f); break;
      case 1: k_flux<DIR, 1><<<g, 128, 0, L.st>>>(L.P, L.f); break;
      case 3: k_flux<DIR, 3><<<g, 128, 0, L.st>>>(L.P, L.f); break;
      case 4: k_flux<DIR, 4><<<g, 128, 0, L.st>>>(L.P, L.f); break;
      default: k_flux<DIR, 2><<<g, 128, 0, L.st>>>(L.P, L.f); break;
    }
  }
  CK(cudaGetLastError());
  c->launches[KC_FX + DIR] += 1;
  return AK_OK;
}

int launch_fofc(ak_ctx* c, const Lane& L, double dt) {
  const long long n = L.P.n, nt = L.P.nt;
  const long long ntest = (n + 2) * (n + 2) * (n + 2) * L.P.nmb;
  const long long nf = (n + 3) * (n + 2) * (n + 2) * L.P.nmb;
  {
    Timer t(c, KC_FOFC_TEST, L.st);
    CK(cudaMemsetAsync(L.f.flag, 0, (size_t)(nt * nt * nt * L.P.nmb), L.st));
    CK(cudaMemsetAsync(L.f.count, 0, sizeof(unsigned) * 4, L.st));
    CK(cudaMemsetAsync(L.f.stats + S_FOFC_CELLS, 0, sizeof(unsigned long long) * 2, L.st));
    if (L.P.fofc) {
      const unsigned g = capped(ntest, 128, L.ov ? c->cap[KC_FOFC_TEST] : 0);
      if (c->fuse_src && L.f.dU[0]) {
        // part (6) fused into the test kernel (k_src_fix after the re-flux redoes the cells it touches)
        if ((long long)g * 128 < ntest) {
          if (L.P.eos) k_fofc_test<1, true, true><<<g, 128, 0, L.st>>>(L.P, L.f, dt);
          else k_fofc_test<0, true, true><<<g, 128, 0, L.st>>>(L.P, L.f, dt);
        } else if (L.P.eos) k_fofc_test<1, false, true><<<g, 128, 0, L.st>>>(L.P, L.f, dt);
        else k_fofc_test<0, false, true><<<g, 128, 0, L.st>>>(L.P, L.f, dt);
      } else if ((long long)g * 128 < ntest) {
        if (L.P.eos) k_fofc_test<1, true><<<g, 128, 0, L.st>>>(L.P, L.f, dt);
        else k_fofc_test<0, true><<<g, 128, 0, L.st>>>(L.P, L.f, dt);
      } else if (L.P.eos) k_fofc_test<1><<<g, 128, 0, L.st>>>(L.P, L.f, dt);
      else k_fofc_test<0><<<g, 128, 0, L.st>>>(L.P, L.f, dt);
      c->launches[KC_FOFC_TEST] += 1;
      CK(cudaGetLastError());
    }
  }
  if (L.P.fofc) {
    Timer t(c, KC_FOFC_FIX, L.st);
    unsigned g = (unsigned)(nf < 148LL * 8 * 128 ? nblk(nf, 128) : 148 * 8);
    if (L.ov && c->cap[KC_FOFC_FIX] > 0 && g > (unsigned)c->cap[KC_FOFC_FIX]) g = (unsigned)c->cap[KC_FOFC_FIX];
    if (L.P.eos) {
      k_fofc_reflux<0, 1><<<g, 128, 0, L.st>>>(L.P, L.f);
      k_fofc_reflux<1, 1><<<g, 128, 0, L.st>>>(L.P, L.f);
      k_fofc_reflux<2, 1><<<g, 128, 0, L.st>>>(L.P, L.f);
    } else {
      k_fofc_reflux<0><<<g, 128, 0, L.st>>>(L.P, L.f);
      k_fofc_reflux<1><<<g, 128, 0, L.st>>>(L.P, L.f);
      k_fofc_reflux<2><<<g, 128, 0, L.st>>>(L.P, L.f);
    }
    CK(cudaGetLastError());
    c->launches[KC_FOFC_FIX] += 3;
  }
  return AK_OK;
}

int launch_ct(ak_ctx* c, const Lane& L, bool have_cell_emf) {
  Timer t(c, KC_CT, L.st);
  const long long n = L.P.n;
  const long long ntest = (n + 2) * (n + 2) * (n + 2) * L.P.nmb;
  const long long ne = n * (n + 1) * (n + 1) * L.P.nmb;
  const unsigned g = capped(ne, 128, L.ov ? c->cap[KC_CT] : 0);
  if (!have_cell_emf) k_cell_emf<<<nblk(ntest, 128), 128, 0, L.st>>>(L.P, L.f);
  if ((long long)g * 128 < ne) {
    k_ct<0, true><<<g, 128, 0, L.st>>>(L.P, L.f);
    k_ct<1, true><<<g, 128, 0, L.st>>>(L.P, L.f);
    k_ct<2, true><<<g, 128, 0, L.st>>>(L.P, L.f);
  } else if (c->ct_fused) {
    k_ct_all<<<nblk((n + 1) * (n + 1) * (n + 1) * L.P.nmb, 128), 128, 0, L.st>>>(L.P, L.f);
    c->launches[KC_CT] -= 2;
  } else {
    k_ct<0><<<g, 128, 0, L.st>>>(L.P, L.f);
    k_ct<1><<<g, 128, 0, L.st>>>(L.P, L.f);
    k_ct<2><<<g, 128, 0, L.st>>>(L.P, L.f);
  }
  CK(cudaGetLastError());
  c->launches[KC_CT] += have_cell_emf ? 3 : 4;
  return AK_OK;
}

int launch_src(ak_ctx* c, const Lane& L) {
  Timer t(c, KC_SRC, L.st);
  const long long n = L.P.n;
  if (c->fuse_src && L.P.fofc) {
    // the fused FOFC-test kernel has written dU~/dt from the high-order fluxes: redo the cells with a re-fluxed face
    const long long ntest = (n + 2) * (n + 2) * (n + 2) * L.P.nmb;
    unsigned g = (unsigned)(ntest < 148LL * 8 * 128 ? nblk(ntest, 128) : 148 * 8);
    if (L.ov && c->cap[KC_SRC] > 0 && g > (unsigned)c->cap[KC_SRC]) g = (unsigned)c->cap[KC_SRC];
    if (L.P.eos) k_src_fix<1><<<g, 128, 0, L.st>>>(L.P, L.f);
    else k_src_fix<0><<<g, 128, 0, L.st>>>(L.P, L.f);
    CK(cudaGetLastError());
    c->launches[KC_SRC] += 1;
    return AK_OK;
  }
  const unsigned g = capped(n * n * n * L.P.nmb, 128, L.ov ? c->cap[KC_SRC] : 0);
  if ((long long)g * 128 < n * n * n * L.P.nmb) {
    if (L.P.eos) k_div_src<1, true><<<g, 128, 0, L.st>>>(L.P, L.f);
    else k_div_src<0, true><<<g, 128, 0, L.st>>>(L.P, L.f);
  } else if (L.P.eos) k_div_src<1><<<g, 128, 0, L.st>>>(L.P, L.f);
  else k_div_src<0><<<g, 128, 0, L.st>>>(L.P, L.f);
  CK(cudaGetLastError());
  c->launches[KC_SRC] += 1;
  return AK_OK;
}

int drain_timers(ak_ctx* c) {
  for (int q = 0; q < c->npend; ++q) {
    float ms = 0.f;
    cudaError_t e = cudaEventSynchronize(c->pend[q].b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, c->pend[q].a, c->pend[q].b);
    cudaEventDestroy(c->pend[q].a); cudaEventDestroy(c->pend[q].b);
    if (e != cudaSuccess) { c->npend = 0; last_cuda_error = e; return AK_ECUDA; }
    c->ms[c->pend[q].which] += ms;
  }
  c->npend = 0;
  return AK_OK;
}

}  // namespace

// ------------------------------------------------------------------ probes (roofline denominators)
namespace {
__global__ void __launch_bounds__(256) k_probe_copy(double2* __restrict__ dst, const double2* __restrict__ src,
                                                    long long n2) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n2; q += stride) dst[q] = src[q];
}
// 8 independent accumulator chains per thread; FMA = 1 instruction (2 flop), else MUL + ADD.
template <bool FMA>
__global__ void __launch_bounds__(256) k_probe_fp64(double* out, int iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) x[q] = 1.0 + 1e-3 * (threadIdx.x + q);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      if (FMA) x[q] = __fma_rn(x[q], a, b);
      else x[q] = __dadd_rn(__dmul_rn(x[q], a), b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int q = 0; q < 8; ++q) s += x[q];
  if (s == 123.456) out[0] = s;   // never true; keeps the chains alive
}
}  // namespace

// ------------------------------------------------------------------ C-ABI
extern "C" {

const char* ak_version(void) { return "ak 0.1 (sm_100a, fp64, --fmad=false)"; }

const char* ak_strerror(int code) {
  switch (code) {
    case AK_OK: return "ok";
    case AK_EINVAL: return "invalid argument";
    case AK_ENOMEM: return "out of device memory";
    case AK_ECUDA: return last_cuda_error != cudaSuccess ? cudaGetErrorString(last_cuda_error) : "CUDA error";
    case AK_ESTATE: return "call out of order (metric or fluxes missing)";
    case AK_EHOOK: return "the caller's refresh hook reported a failure";
    case AK_ETOOBIG: return "batch larger than the static scratch of ak_con2prim_static (AK_STATIC_MAX_CELLS stored cells)";
    default: return "unknown error code";
  }
}

int ak_create(const ak_params* p, const double* dx3, ak_ctx** out) {
  if (!out) return AK_EINVAL;
  *out = nullptr;
  const int v = validate(p, dx3);
  if (v != AK_OK) return v;
  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (p->device >= ndev) return AK_EINVAL;
  CK(cudaSetDevice(p->device));
  ak_ctx* c = new (std::nothrow) ak_ctx();
  if (!c) return AK_ENOMEM;
  memset(c, 0, sizeof(*c));
  c->hp = *p;
  c->stream = (cudaStream_t)p->stream;
  c->blend_a = 0.0; c->blend_b = 1.0;
  {
    // overlapped-schedule tuning (ak_set_overlap): grid caps in blocks per SM, per kernel class; defaults
    // from the measurements recorded in DESIGN.md §6.2, overridable for experiments
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, p->device);
    auto envi = [](const char* k, int dflt) { const char* v = getenv(k); return v ? atoi(v) : dflt; };
    c->cap[KC_C2P] = nsm * envi("AK_OV_CAP_C2P", AK_OV_CAP_C2P_DEFAULT);
    c->cap[KC_FOFC_TEST] = nsm * envi("AK_OV_CAP_FOFC", AK_OV_CAP_FOFC_DEFAULT);
    c->cap[KC_FOFC_FIX] = nsm * envi("AK_OV_CAP_FIX", AK_OV_CAP_FIX_DEFAULT);
    c->cap[KC_CT] = nsm * envi("AK_OV_CAP_CT", AK_OV_CAP_CT_DEFAULT);
    c->cap[KC_SRC] = nsm * envi("AK_OV_CAP_SRC", AK_OV_CAP_SRC_DEFAULT);
    c->sweep_smem_pad = envi("AK_OV_SMEM_PAD", AK_OV_SMEM_PAD_DEFAULT);
    c->pencil_wi = envi("AK_PENCIL_WI", AK_PENCIL_WI_DEFAULT);
    c->tile_tm = envi("AK_TILE_TENSORMAP", 1);
    // measured on C4 (DESIGN.md §6 item 21): fused 4.18 + fix 0.51 ms against 1.95 + 2.15 ms separately -> off
    c->fuse_src = envi("AK_FUSE_SRC", 0);
    // -1: automatic — only for batches of >= 2^23 stored cells: the split adds 4 launches, empty thread blocks and
    // 51 tensor-map encodes per stage, which cost the small configs 3-14 % (C0 0.144 -> 0.165 ms, C3 1.53 -> 1.58)
    // and gain C4 1 % (13.75 -> 13.59 ms)
    c->split_blocks = envi("AK_SPLIT_BLOCKS", -1);
    c->ct_fused = envi("AK_CT_FUSED", 1);
  }
  Par& P = c->P;
  P.nmb = p->nmb; P.n = p->n; P.nt = p->n + 8; P.px = P.nt + 4; P.is = 4; P.ie = p->n + 3;
  P.Gam = p->gamma_ad; P.gm1 = p->gamma_ad - 1.0; P.gm1r = p->gamma_ad / (p->gamma_ad - 1.0);
  P.rho_atm = p->rho_atm; P.T_atm = p->T_atm; P.P_atm = p->rho_atm * p->T_atm;
  P.eps_atm = p->T_atm / P.gm1; P.thr = p->f_thr * p->rho_atm;
  P.mag_max = p->mag_max;
  P.dmp_M = p->dmp_M; P.dmp_iM = p->dmp_M > 0.0 ? 1.0 / p->dmp_M : 0.0;
  P.max_iter = p->c2p_max_iter; P.tol = p->c2p_tol;
  P.recon = p->recon; P.riemann = p->riemann; P.fofc = p->fofc; P.fofc_riemann = p->fofc_riemann;
  P.shortcuts = 7;
  if (const char* v = getenv("AK_EXACT_SHORTCUTS")) P.shortcuts = atoi(v) & 7;
  const long long nt = P.nt, px = P.px, nb = P.nmb;
  c->sz.cell = nb * nt * nt * nt;
  c->sz.xf = nb * nt * nt * px; c->sz.yf = nb * nt * (nt + 1) * nt; c->sz.zf = nb * (nt + 1) * nt * nt;
  c->sz.ex = nb * (nt + 1) * (nt + 1) * nt; c->sz.ey = nb * (nt + 1) * nt * px; c->sz.ez = nb * nt * (nt + 1) * px;
  const long long fsz[3] = {c->sz.xf, c->sz.yf, c->sz.zf};
  const long long ntest = nb * (P.n + 2) * (P.n + 2) * (P.n + 2);
  cudaError_t e = cudaSuccess;
  for (int d = 0; d < 3 && e == cudaSuccess; ++d) {
    for (int q = 0; q < 7 && e == cudaSuccess; ++q) {
      e = cudaMalloc(&c->F[7 * d + q], sizeof(double) * fsz[d]);
      // faces outside the computed range are never written: define them once
      if (e == cudaSuccess) e = cudaMemsetAsync(c->F[7 * d + q], 0, sizeof(double) * fsz[d], c->stream);
    }
    if (e == cudaSuccess) e = cudaMalloc(&c->Ecc[d], sizeof(double) * c->sz.cell);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->Ecc[d], 0, sizeof(double) * c->sz.cell, c->stream);
  }
  if (e == cudaSuccess) e = cudaMalloc(&c->list, sizeof(unsigned) * ntest);
  if (e == cudaSuccess) e = cudaMalloc(&c->flag_own, (size_t)c->sz.cell);
  if (e == cudaSuccess) e = cudaMalloc(&c->count, sizeof(unsigned) * 4 * MAXCH);
  if (e == cudaSuccess) e = cudaMalloc(&c->stats, sizeof(unsigned long long) * S_NSTAT * MAXCH);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->count, 0, sizeof(unsigned) * 4 * MAXCH, c->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->stats, 0, sizeof(unsigned long long) * S_NSTAT * MAXCH, c->stream);
  {
    int tmax = 1;
    for (int d = 0; d < 3; ++d) {
      int NA, tiles;
      sweep_tiling(d, p->n, false, NA, tiles);
      if (tiles > tmax) tmax = tiles;
    }
    c->tcap = (unsigned)((size_t)nb * (p->n + 2) * tmax);
  }
  if (e == cudaSuccess) e = cudaMalloc(&c->tlist, sizeof(unsigned) * (6 * (size_t)c->tcap + 6));
  if (e == cudaSuccess) e = cudaMalloc(&c->rowflag, (size_t)nb * c->P.nt * c->P.nt);
  if (e == cudaSuccess) e = cudaMalloc(&c->zflags, sizeof(unsigned) * nb);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->zflags, 0xff, sizeof(unsigned) * nb, c->stream);
  if (e == cudaSuccess) e = cudaMalloc(&c->dx, sizeof(double) * 3 * nb);
  if (e == cudaSuccess) e = cudaMemcpyAsync(c->dx, dx3, sizeof(double) * 3 * nb, cudaMemcpyHostToDevice, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);   // dx3 is the caller's: copy must be done
  c->host_dx = (double*)malloc(sizeof(double) * 3 * nb);
  if (!c->host_dx && e == cudaSuccess) e = cudaErrorMemoryAllocation;
  if (c->host_dx) memcpy(c->host_dx, dx3, sizeof(double) * 3 * nb);
  if (e != cudaSuccess) {
    last_cuda_error = e;
    ak_destroy(c);
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? AK_ENOMEM : AK_ECUDA;
  }
  *out = c;
  if (const char* v = getenv("AK_OV_CHUNKS")) {
    const int r = ak_set_overlap(c, atoi(v));
    if (r != AK_OK) { ak_destroy(c); *out = nullptr; return r; }
  }
  return AK_OK;
}

int ak_destroy(ak_ctx* c) {
  if (!c) return AK_EINVAL;
  cudaSetDevice(c->hp.device);
  cudaStreamSynchronize(c->stream);
  for (int q = 0; q < c->npend; ++q) { cudaEventDestroy(c->pend[q].a); cudaEventDestroy(c->pend[q].b); }
  free(c->pend);
  for (int q = 0; q < 21; ++q) cudaFree(c->F[q]);
  for (int q = 0; q < 3; ++q) { cudaFree(c->Ecc[q]); cudaFree(c->stg_Bf[q]); cudaFree(c->stg_E[q]); }
  cudaFree(c->list);
  for (int q = 0; q < 5; ++q) { cudaFree(c->stg_U[q]); cudaFree(c->stg_dU[q]); }
  for (int q = 0; q < 8; ++q) cudaFree(c->stg_W[q]);
  cudaFree(c->stg_flag); cudaFree(c->stg_status);
  for (int q = 0; q < 5; ++q) { cudaFree(c->regU0[q]); cudaFree(c->reg_dU[q]); }
  for (int q = 0; q < 3; ++q) { cudaFree(c->regB0[q]); cudaFree(c->regE[q]); }
  cudaFree(c->reg_flag);
  cudaFree(c->nbr);
  free(c->host_dx);
  for (int l = 0; l < 2; ++l) {
    if (c->lane[l]) { cudaStream_t st = c->lane[l]->stream; ak_destroy(c->lane[l]); cudaStreamDestroy(st); }
    for (int q = 0; q < 24; ++q) cudaFree(c->lane_buf[l][q]);
    cudaFree(c->lane_mask[l][0]); cudaFree(c->lane_mask[l][1]);
  }
  if (c->lane_stats_h) cudaFreeHost(c->lane_stats_h);
  for (auto& g : c->gslot) if (g.exec) cudaGraphExecDestroy(g.exec);
  if (c->gstream) cudaStreamDestroy(c->gstream);
  if (c->ov_ev) {
    for (int q = 0; q < c->ov_nev; ++q) if (c->ov_ev[q]) cudaEventDestroy(c->ov_ev[q]);
    free(c->ov_ev);
    for (int q = 0; q < 3; ++q)
      if (c->ovs[q] && !(q == 2 && c->ovs[2] == c->ovs[0])) cudaStreamDestroy(c->ovs[q]);
  }
  cudaFree(c->flag_own); cudaFree(c->count); cudaFree(c->stats); cudaFree(c->dx); cudaFree(c->zflags); cudaFree(c->tlist); cudaFree(c->rowflag);
  delete c;
  return AK_OK;
}

int ak_set_metric(ak_ctx* c, const ak_adm* a) {
  if (!c || !a) return AK_EINVAL;
  const double* p[16] = {a->gxx, a->gxy, a->gxz, a->gyy, a->gyz, a->gzz, a->alp, a->betx, a->bety, a->betz,
                         a->Kxx, a->Kxy, a->Kxz, a->Kyy, a->Kyz, a->Kzz};
  for (int q = 0; q < 16; ++q)
    if (!al16(p[q])) return AK_EINVAL;
  for (int q = 0; q < 16; ++q) c->adm[q] = p[q];
  c->have_metric = true;
  return AK_OK;
}

int ak_set_eos_hybrid(ak_ctx* c, int nseg, double K0, const double* gammas, const double* rho_breaks,
                      double gamma_th) {
  if (!c) return AK_EINVAL;
  Par& P = c->P;
  if (nseg == 0) {              // back to the ideal gas of ak_params.gamma_ad
    P.eos = 0; P.nseg = 0;
    P.P_atm = P.rho_atm * P.T_atm;
    c->have_flux = false;
    for (int l = 0; l < 2; ++l) if (c->lane[l]) copy_eos(c->lane[l]->P, P);
    return AK_OK;
  }
  if (nseg < 1 || nseg > 4 || !gammas || (nseg > 1 && !rho_breaks)) return AK_EINVAL;
  if (!(std::isfinite(K0) && K0 >= 0.0) || !(std::isfinite(gamma_th) && gamma_th > 1.0)) return AK_EINVAL;
  for (int i = 0; i < nseg; ++i)
    if (!(std::isfinite(gammas[i]) && gammas[i] > 1.0)) return AK_EINVAL;
  for (int i = 0; i + 1 < nseg; ++i)
    if (!finite_pos(rho_breaks[i]) || (i > 0 && !(rho_breaks[i] > rho_breaks[i - 1]))) return AK_EINVAL;
  // K_i and the offsets a_i of eps_c follow from continuity of P_c and eps_c at the breakpoints
  P.eos = 1; P.nseg = nseg; P.gth = gamma_th; P.gthm1 = gamma_th - 1.0;
  for (int i = 0; i < 4; ++i) { P.ppK[i] = 0.0; P.ppG[i] = 2.0; P.ppa[i] = 0.0; }
  for (int i = 0; i < 3; ++i) P.pprb[i] = 0.0;
  for (int i = 0; i < nseg; ++i) P.ppG[i] = gammas[i];
  for (int i = 0; i + 1 < nseg; ++i) P.pprb[i] = rho_breaks[i];
  P.ppK[0] = K0;
  for (int i = 1; i < nseg; ++i) {
    const double rb = P.pprb[i - 1], Ga = P.ppG[i - 1], Gb = P.ppG[i];
    P.ppK[i] = P.ppK[i - 1] * std::pow(rb, Ga - Gb);
    P.ppa[i] = P.ppa[i - 1] + P.ppK[i - 1] * std::pow(rb, Ga - 1.0) / (Ga - 1.0) -
               P.ppK[i] * std::pow(rb, Gb - 1.0) / (Gb - 1.0);
  }
  // atmosphere pressure P(rho_atm, T_atm) = P_c(rho_atm) + rho_atm T_atm (host pow, as the device's
  // differs from it by rounding only in the last place)
  int s0 = 0;
  while (s0 + 1 < nseg && P.rho_atm >= P.pprb[s0]) ++s0;
  P.P_atm = P.ppK[s0] * std::pow(P.rho_atm, P.ppG[s0]) + P.rho_atm * P.T_atm;
  c->have_flux = false;
  for (int l = 0; l < 2; ++l) if (c->lane[l]) copy_eos(c->lane[l]->P, P);
  return AK_OK;
}

int ak_con2prim(ak_ctx* c, const ak_cons* U, const ak_faceB* Bf, const ak_prim* W, unsigned char* status) {
  if (!c) return AK_EINVAL;
  if (!c->have_metric) return AK_ESTATE;
  Fields f;
  fill_fields(c, f);
  if (!set_cons(f, U) || !set_faceB(f, Bf) || !set_prim(f, W)) return AK_EINVAL;
  f.status = status;
  CK(cudaSetDevice(c->hp.device));
  const Lane L = {c->P, f, c->stream, false};
  return launch_c2p(c, L, false);
}

}  // extern "C"

namespace {
// tile lists are made when part (1) runs in the same call, every exact shortcut is on, and both sweep kernels
// tile each direction alike (they do for every n with the default build)
bool split_wanted(ak_ctx* c, int w_is_valid) {
  const bool want = c->split_blocks > 0 || (c->split_blocks < 0 && c->sz.cell >= (1LL << 23));
  if (w_is_valid || !want || (c->P.shortcuts & 5) != 5 || !c->tile_tm || !tmap_encoder() || !tile_kernels_apply(c, c->P))
    return false;
  for (int d = 0; d < 3; ++d) {
    int NAg, tg, NAs, ts;
    sweep_tiling(d, c->P.n, false, NAg, tg);
    sweep_tiling(d, c->P.n, true, NAs, ts);
    if (NAg != NAs || tg != ts) return false;
  }
  return true;
}

// the serial schedule of one stage: the whole batch, kernel after kernel, on stream st
int rhs_serial(ak_ctx* c, const Fields& f, int w_is_valid, double dt_fofc, cudaStream_t st) {
  // counters of every chunk slot start from zero (a stage that skips part (1) reports no con2prim counts)
  CK(cudaMemsetAsync(c->stats, 0, sizeof(unsigned long long) * S_NSTAT * MAXCH, st));
  CK(cudaMemsetAsync(c->count, 0, sizeof(unsigned) * 4 * MAXCH, st));
  int r;
  const Lane L = {c->P, f, st, false};
  if (!w_is_valid && (r = launch_c2p(c, L, true)) != AK_OK) return r;
  // tiles that part (1) found static and unmagnetised as a whole go to the light sweep kernel
  Fields fs = f;
  if (f.rowflag) {                             // (ak_rhs hands the row flags out only when split_wanted())
    TileShapes sh;
    int tmax = 0;
    for (int d = 0; d < 3; ++d) {
      sweep_tiling(d, c->P.n, false, sh.NA[d], sh.tiles[d]);
      if (sh.tiles[d] > tmax) tmax = sh.tiles[d];
    }
    unsigned* cnt = c->tlist + 6 * (size_t)c->tcap;
    CK(cudaMemsetAsync(cnt, 0, sizeof(unsigned) * 6, st));
    const dim3 grid(nblk((long long)c->P.nmb * (c->P.n + 2) * tmax, 256), 3);
    k_split_tiles<<<grid, 256, 0, st>>>(c->P, f.rowflag, sh, c->tlist, cnt, c->tcap);
    CK(cudaGetLastError());
    c->launches[KC_C2P] += 1;                  // counted with part (1), whose flags it sorts
    fs.tlist = c->tlist; fs.tcount = cnt; fs.tcap = c->tcap;
  }
  const Lane LS = {c->P, fs, st, false};
  if ((r = launch_flux<0>(c, LS)) != AK_OK) return r;
  if ((r = launch_flux<1>(c, LS)) != AK_OK) return r;
  if ((r = launch_flux<2>(c, LS)) != AK_OK) return r;
  if ((r = launch_fofc(c, L, dt_fofc)) != AK_OK) return r;
  if ((r = launch_ct(c, L, !w_is_valid)) != AK_OK) return r;
  return launch_src(c, L);
}

// FNV-1a over everything the launch sequence depends on: the parameters, every pointer, the blend, the flags
unsigned long long rhs_key(const ak_ctx* c, const Fields& f, int w_is_valid, double dt_fofc) {
  unsigned long long h = 1469598103934665603ull;
  auto mix = [&](const void* p, size_t n) {
    const unsigned char* b = (const unsigned char*)p;
    for (size_t q = 0; q < n; ++q) { h ^= b[q]; h *= 1099511628211ull; }
  };
  mix(&c->P, sizeof(Par)); mix(&f, sizeof(Fields)); mix(&w_is_valid, sizeof(int)); mix(&dt_fofc, sizeof(double));
  mix(&c->tile_tm, sizeof(int)); mix(&c->pencil_wi, sizeof(int)); mix(&c->fuse_src, sizeof(int));
  return h | 1ull;               // 0 marks an empty slot
}

// Serial stage through the graph cache.  First sighting of an argument set: plain launches (this also raises
// the shared-memory attributes, which must not happen inside a capture).  Second: the same launch code runs
// under stream capture on the context's capture stream and is instantiated.  From then on: one cudaGraphLaunch
// on the caller's stream.
int rhs_graphed(ak_ctx* c, const Fields& f, int w_is_valid, double dt_fofc) {
  const unsigned long long key = rhs_key(c, f, w_is_valid, dt_fofc);
  ak_ctx::GraphSlot* s = nullptr;
  for (auto& g : c->gslot) if (g.key == key) s = &g;
  if (s && s->exec) {
    s->age = ++c->gclock;
    CK(cudaGraphLaunch(s->exec, c->stream));
    c->graph_replays += 1;
    return AK_OK;
  }
  if (!s) {                      // remember the key (evicting the least recently used slot), run it plainly
    s = &c->gslot[0];
    for (auto& g : c->gslot) if (g.age < s->age) s = &g;
    if (s->exec) { cudaGraphExecDestroy(s->exec); s->exec = nullptr; }
    s->key = key; s->age = ++c->gclock;
    return rhs_serial(c, f, w_is_valid, dt_fofc, c->stream);
  }
  s->age = ++c->gclock;
  cudaGraph_t graph = nullptr;
  CK(cudaStreamBeginCapture(c->gstream, cudaStreamCaptureModeThreadLocal));
  const int r = rhs_serial(c, f, w_is_valid, dt_fofc, c->gstream);
  const cudaError_t e = cudaStreamEndCapture(c->gstream, &graph);
  if (r != AK_OK || e != cudaSuccess || !graph) {
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    s->key = 0;                  // do not try this argument set again under capture
    if (r != AK_OK) return r;
    return rhs_serial(c, f, w_is_valid, dt_fofc, c->stream);
  }
  const cudaError_t ei = cudaGraphInstantiate(&s->exec, graph, 0);
  cudaGraphDestroy(graph);
  if (ei != cudaSuccess) { s->exec = nullptr; s->key = 0; cudaGetLastError(); return rhs_serial(c, f, w_is_valid, dt_fofc, c->stream); }
  CK(cudaGraphLaunch(s->exec, c->stream));
  c->graph_replays += 1;
  return AK_OK;
}
}  // namespace

extern "C" {

int ak_set_graph(ak_ctx* c, int on) {
  if (!c) return AK_EINVAL;
  CK(cudaSetDevice(c->hp.device));
  if (on && !c->gstream) CK(cudaStreamCreateWithFlags(&c->gstream, cudaStreamNonBlocking));
  if (!on) {
    CK(cudaStreamSynchronize(c->stream));
    for (auto& g : c->gslot) { if (g.exec) cudaGraphExecDestroy(g.exec); g.exec = nullptr; g.key = 0; g.age = 0; }
  }
  c->graph_on = on != 0;
  c->graph_replays = 0;
  return AK_OK;
}

long long ak_graph_replays(const ak_ctx* c) { return c ? c->graph_replays : -1; }

int ak_rhs(ak_ctx* c, const ak_cons* U, const ak_faceB* Bf, const ak_prim* W, int w_is_valid, double dt_fofc,
           const ak_rhs_out* out) {
  if (!c || !out) return AK_EINVAL;
  if (!c->have_metric) return AK_ESTATE;
  if (!std::isfinite(dt_fofc)) return AK_EINVAL;
  Fields f;
  fill_fields(c, f);
  if (!set_cons(f, U) || !set_faceB(f, Bf) || !set_prim(f, W)) return AK_EINVAL;
  if (!out->dD || !out->dSx || !out->dSy || !out->dSz || !out->dtau || !out->Ex || !out->Ey || !out->Ez)
    return AK_EINVAL;
  f.dU[0] = out->dD; f.dU[1] = out->dSx; f.dU[2] = out->dSy; f.dU[3] = out->dSz; f.dU[4] = out->dtau;
  f.E[0] = out->Ex; f.E[1] = out->Ey; f.E[2] = out->Ez;
  if (out->fofc_flag) f.flag = out->fofc_flag;
  f.status = out->c2p_status;
  // per-block zero-field flags: part (1) of this call writes them, the later parts read them; primitives the
  // caller supplies (w_is_valid) come without
  f.zflags = w_is_valid ? nullptr : c->zflags;
  f.rowflag = (c->ov_chunks <= 1 && split_wanted(c, w_is_valid)) ? c->rowflag : nullptr;
  if (out->matter) {
    const ak_matter* mo = out->matter;
    double* mp[10] = {mo->E, mo->Sx, mo->Sy, mo->Sz, mo->Sxx, mo->Sxy, mo->Sxz, mo->Syy, mo->Syz, mo->Szz};
    for (int q = 0; q < 10; ++q) { if (!al16(mp[q])) return AK_EINVAL; f.M[q] = mp[q]; }
  }
  CK(cudaSetDevice(c->hp.device));
  c->stats_from_host = false;
  int r;
  const int nch = c->ov_chunks < 2 ? 1 : (c->ov_chunks < c->P.nmb ? c->ov_chunks : c->P.nmb);
  if (nch < 2) {
    // serial schedule; replayed from a CUDA graph when ak_set_graph is on (not while ak_timing brackets classes)
    r = (c->graph_on && !c->timing) ? rhs_graphed(c, f, w_is_valid, dt_fofc)
                                    : rhs_serial(c, f, w_is_valid, dt_fofc, c->stream);
    if (r == AK_OK) c->have_flux = true;
    return r;
  }
  // counters of every chunk slot start from zero (a stage that skips part (1) reports no con2prim counts)
  CK(cudaMemsetAsync(c->stats, 0, sizeof(unsigned long long) * S_NSTAT * MAXCH, c->stream));
  CK(cudaMemsetAsync(c->count, 0, sizeof(unsigned) * 4 * MAXCH, c->stream));
  // overlapped schedule: MeshBlocks are independent, so the batch is cut into nch chunks.
  // Stream A runs part (1) of chunk i+1 and stream C parts (4)-(6) of chunk i-1 (memory- and latency-bound,
  // capped grids, high priority) while stream B runs the fp64-bound sweeps of chunk i.  Only events order
  // the streams; no kernel waits on another.  Same kernels, same arithmetic: outputs are bit-identical.
  cudaStream_t sA = c->ovs[0], sB = c->ovs[1], sC = c->ovs[2];
  cudaEvent_t* ev = c->ov_ev;                     // [0] fork, [1..3] joins, [4 + 2 i] c2p(i), [5 + 2 i] flux(i)
  CK(cudaEventRecord(ev[0], c->stream));
  CK(cudaStreamWaitEvent(sA, ev[0], 0));
  CK(cudaStreamWaitEvent(sB, ev[0], 0));
  if (sC != sA) CK(cudaStreamWaitEvent(sC, ev[0], 0));
  static thread_local Fields CF[MAXCH];
  static thread_local Par CP[MAXCH];
  const int base = c->P.nmb / nch, rem = c->P.nmb % nch;
  for (int ci = 0, m0 = 0; ci < nch; ++ci) {
    const int nb = base + (ci < rem ? 1 : 0);
    chunk_fields(c, f, m0, nb, ci, CF[ci], CP[ci]);
    m0 += nb;
  }
  auto c2p = [&](int ci) -> int {
    if (w_is_valid) return AK_OK;
    const Lane L = {CP[ci], CF[ci], sA, true};
    const int rr = launch_c2p(c, L, true);
    if (rr != AK_OK) return rr;
    CK(cudaEventRecord(ev[4 + 2 * ci], sA));
    return AK_OK;
  };
  if ((r = c2p(0)) != AK_OK) return r;
  for (int ci = 0; ci < nch; ++ci) {
    if (ci + 1 < nch && (r = c2p(ci + 1)) != AK_OK) return r;
    const Lane LB = {CP[ci], CF[ci], sB, true};
    if (!w_is_valid) CK(cudaStreamWaitEvent(sB, ev[4 + 2 * ci], 0));
    if ((r = launch_flux<0>(c, LB)) != AK_OK) return r;
    if ((r = launch_flux<1>(c, LB)) != AK_OK) return r;
    if ((r = launch_flux<2>(c, LB)) != AK_OK) return r;
    CK(cudaEventRecord(ev[5 + 2 * ci], sB));
    const Lane LC = {CP[ci], CF[ci], sC, true};
    CK(cudaStreamWaitEvent(sC, ev[5 + 2 * ci], 0));
    if ((r = launch_fofc(c, LC, dt_fofc)) != AK_OK) return r;
    if ((r = launch_ct(c, LC, !w_is_valid)) != AK_OK) return r;
    if ((r = launch_src(c, LC)) != AK_OK) return r;
  }
  c->have_flux = true;
  CK(cudaEventRecord(ev[1], sA)); CK(cudaStreamWaitEvent(c->stream, ev[1], 0));
  CK(cudaEventRecord(ev[2], sB)); CK(cudaStreamWaitEvent(c->stream, ev[2], 0));
  if (sC != sA) { CK(cudaEventRecord(ev[3], sC)); CK(cudaStreamWaitEvent(c->stream, ev[3], 0)); }
  return AK_OK;
}

int ak_set_exact_shortcuts(ak_ctx* c, int mask) {
  if (!c || mask < 0 || mask > 7) return AK_EINVAL;
  c->P.shortcuts = mask;
  for (int l = 0; l < 2; ++l) if (c->lane[l]) c->lane[l]->P.shortcuts = mask;
  return AK_OK;
}

int ak_set_overlap(ak_ctx* c, int nchunks) {
  if (!c || nchunks < 0 || nchunks > MAXCH) return AK_EINVAL;
  CK(cudaSetDevice(c->hp.device));
  if (nchunks >= 2 && !c->ov_ev) {
    int lo = 0, hi = 0;
    CK(cudaDeviceGetStreamPriorityRange(&lo, &hi));          // lo = least, hi = greatest priority (numerically lower)
    const char* e3 = getenv("AK_OV_STREAMS");
    const char* ep = getenv("AK_OV_PRIO");                    // e.g. "hlh": priority of streams A, B, C
    const char* pr = (ep && strlen(ep) == 3) ? ep : "hlh";
    for (int q = 0; q < 3; ++q) {
      if (q == 2 && e3 && atoi(e3) == 2) { c->ovs[2] = c->ovs[0]; break; }
      CK(cudaStreamCreateWithPriority(&c->ovs[q], cudaStreamNonBlocking, pr[q] == 'h' ? hi : lo));
    }
    c->ov_nev = 4 + 2 * MAXCH;
    c->ov_ev = (cudaEvent_t*)calloc(c->ov_nev, sizeof(cudaEvent_t));
    if (!c->ov_ev) return AK_ENOMEM;
    for (int q = 0; q < c->ov_nev; ++q) CK(cudaEventCreateWithFlags(&c->ov_ev[q], cudaEventDisableTiming));
  }
  c->ov_chunks = nchunks;
  return AK_OK;
}

int ak_emf(ak_ctx* c, const ak_prim* W, double* Ex, double* Ey, double* Ez) {
  if (!c || !Ex || !Ey || !Ez) return AK_EINVAL;
  if (!c->have_metric || !c->have_flux) return AK_ESTATE;
  Fields f;
  fill_fields(c, f);
  if (!set_prim(f, W)) return AK_EINVAL;
  f.E[0] = Ex; f.E[1] = Ey; f.E[2] = Ez;
  CK(cudaSetDevice(c->hp.device));
  const Lane L = {c->P, f, c->stream, false};
  return launch_ct(c, L, false);
}

int ak_matter_sources(ak_ctx* c, const ak_prim* W, const ak_matter* out) {
  if (!c || !out) return AK_EINVAL;
  if (!c->have_metric) return AK_ESTATE;
  Fields f;
  fill_fields(c, f);
  if (!set_prim(f, W)) return AK_EINVAL;
  MatterOut o = {{out->E, out->Sx, out->Sy, out->Sz, out->Sxx, out->Sxy, out->Sxz, out->Syy, out->Syz, out->Szz}};
  for (int q = 0; q < 10; ++q) if (!o.q[q]) return AK_EINVAL;
  CK(cudaSetDevice(c->hp.device));
  if (c->P.eos) k_matter<1><<<nblk(c->sz.cell, 128), 128, 0, c->stream>>>(c->P, f, o);
  else k_matter<0><<<nblk(c->sz.cell, 128), 128, 0, c->stream>>>(c->P, f, o);
  CK(cudaGetLastError());
  return AK_OK;
}

int ak_get_stats(ak_ctx* c, ak_stats* o) {
  if (!c || !o) return AK_EINVAL;
  if (c->stats_from_host) { *o = c->host_acc; return AK_OK; }
  static thread_local unsigned long long h[S_NSTAT * MAXCH];
  static thread_local unsigned cnt[4 * MAXCH];
  CK(cudaSetDevice(c->hp.device));
  CK(cudaMemcpyAsync(h, c->stats, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaMemcpyAsync(cnt, c->count, sizeof(cnt), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  memset(o, 0, sizeof(*o));
  for (int ci = 0; ci < MAXCH; ++ci) {      // one slot per chunk of the overlapped schedule (slot 0 otherwise)
    const unsigned long long* hc = h + S_NSTAT * ci;
    o->n_c2p_fail += (long long)hc[S_C2P_FAIL];
    o->n_cons_floor += (long long)hc[S_CONS_FLOOR];
    o->n_prim_floor += (long long)hc[S_PRIM_FLOOR];
    o->n_dmp_cells += (long long)hc[S_DMP_CELLS];
    o->n_fofc_cells += (long long)cnt[4 * ci + 3];
    for (int d = 0; d < 3; ++d) o->n_fofc_faces[d] += cnt[4 * ci + d];
  }
  return AK_OK;
}

int ak_get_flux(ak_ctx* c, int dir, int comp, double* dst) {
  if (!c || !dst || dir < 0 || dir > 2 || comp < 0 || comp > 6) return AK_EINVAL;
  if (!c->have_flux) return AK_ESTATE;
  const long long fsz[3] = {c->sz.xf, c->sz.yf, c->sz.zf};
  CK(cudaSetDevice(c->hp.device));
  CK(cudaMemcpyAsync(dst, c->F[7 * dir + comp], sizeof(double) * fsz[dir], cudaMemcpyDeviceToDevice, c->stream));
  return AK_OK;
}

int ak_timing(ak_ctx* c, int enable) {
  if (!c) return AK_EINVAL;
  const int r = drain_timers(c);
  c->timing = enable != 0;
  for (int q = 0; q < KC_N; ++q) { c->ms[q] = 0.0; c->launches[q] = 0; }
  return r;
}

int ak_kernel_ms(ak_ctx* c, double ms_out[8], long long launches_out[8]) {
  if (!c || !ms_out || !launches_out) return AK_EINVAL;
  CK(cudaSetDevice(c->hp.device));
  const int r = drain_timers(c);
  for (int q = 0; q < KC_N; ++q) { ms_out[q] = c->ms[q]; launches_out[q] = c->launches[q]; }
  return r;
}

// Pipelined host path: the batch is cut into chunks of blocks that alternate between two lanes
// (child contexts with their own streams), so that the H2D copy of one chunk, the kernels of
// another and the D2H copy of a third overlap (PCIe is full duplex).
// Sparse write-back of U~ for the host path: con2prim rewrites only the cells whose status is non-zero, so when
// the caller's U~ arrays are pinned host memory the device can address, those cells alone are written there
// (zero-copy stores) instead of copying every field back whole.
__global__ void __launch_bounds__(256) k_writeback_floored(const unsigned char* __restrict__ status, long long ncell,
                                                           const double* u0, const double* u1, const double* u2,
                                                           const double* u3, const double* u4, double* h0, double* h1,
                                                           double* h2, double* h3, double* h4) {
  for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += (long long)gridDim.x * blockDim.x) {
    if (status[c] != 0) { h0[c] = u0[c]; h1[c] = u1[c]; h2[c] = u2[c]; h3[c] = u3[c]; h4[c] = u4[c]; }
  }
}
// device-side address of a host buffer the GPU can write (pinned / registered memory), or nullptr
static double* mapped_host(double* h) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, h) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  if (at.type != cudaMemoryTypeHost || !at.devicePointer) return nullptr;
  return (double*)at.devicePointer;
}

static int rhs_host_pipelined(ak_ctx* c, int chunk, double* const hU[5], const double* const hB[3], double* const hW[8],
                              double dt_fofc, double* const hdU[5], double* const hE[3], unsigned char* hflag,
                              unsigned char* hstatus) {
  const long long nt = c->P.nt, px = c->P.px;
  const long long per[7] = {nt * nt * nt, nt * nt * px, nt * (nt + 1) * nt, (nt + 1) * nt * nt,
                            (nt + 1) * (nt + 1) * nt, (nt + 1) * nt * px, nt * (nt + 1) * px};   // cell xf yf zf ex ey ez
  const int nchunks = c->P.nmb / chunk;
  c->have_flux = false;                       // the fluxes of this stage stay in the lanes: ak_emf / ak_get_flux -> AK_ESTATE
  if (c->lane_chunk != chunk) {
    if (c->lane_chunk != 0) return AK_ESTATE;
    for (int l = 0; l < 2; ++l) {               // left over from an attempt that failed half way
      if (c->lane[l]) { cudaStream_t st0 = c->lane[l]->stream; ak_destroy(c->lane[l]); cudaStreamDestroy(st0); c->lane[l] = nullptr; }
      for (int q = 0; q < 24; ++q) { cudaFree(c->lane_buf[l][q]); c->lane_buf[l][q] = nullptr; }
      for (int q = 0; q < 2; ++q) { cudaFree(c->lane_mask[l][q]); c->lane_mask[l][q] = nullptr; }
    }
    if (c->lane_stats_h) { cudaFreeHost(c->lane_stats_h); c->lane_stats_h = nullptr; }
    for (int l = 0; l < 2; ++l) {
      ak_params hp = c->hp;
      hp.nmb = chunk;
      cudaStream_t st;
      CK(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
      hp.stream = (void*)st;
      const int r = ak_create(&hp, c->host_dx, &c->lane[l]);
      if (r != AK_OK) { cudaStreamDestroy(st); return r; }
      copy_eos(c->lane[l]->P, c->P);
      c->lane[l]->P.shortcuts = c->P.shortcuts;
      // staging kinds: 0..4 U (cell), 5..7 Bf (xf yf zf), 8..15 W (cell), 16..20 dU (cell), 21..23 E (ex ey ez)
      for (int q = 0; q < 24; ++q) {
        const int kind = q < 5 ? 0 : (q < 8 ? 1 + (q - 5) : (q < 21 ? 0 : 4 + (q - 21)));
        const size_t bytes = sizeof(double) * per[kind] * chunk;
        CK(cudaMalloc(&c->lane_buf[l][q], bytes));
        CK(cudaMemsetAsync(c->lane_buf[l][q], 0, bytes, st));
      }
      CK(cudaMalloc(&c->lane_mask[l][0], (size_t)per[0] * chunk));
      CK(cudaMalloc(&c->lane_mask[l][1], (size_t)per[0] * chunk));
    }
    CK(cudaMallocHost(&c->lane_stats_h, sizeof(unsigned long long) * (S_NSTAT + 4) * nchunks));
    c->lane_chunk = chunk;
  }
  CK(cudaStreamSynchronize(c->stream));            // the metric and anything queued by the caller
  double* mU[5];
  bool sparse_u = true;                            // every U~ array pinned: floored cells are written back singly
  for (int q = 0; q < 5; ++q) { mU[q] = mapped_host(hU[q]); sparse_u = sparse_u && mU[q] != nullptr; }
  for (int ch = 0; ch < nchunks; ++ch) {
    const int l = ch & 1;
    ak_ctx* k = c->lane[l];
    cudaStream_t st = k->stream;
    const long long m0 = (long long)ch * chunk;
    double** b = c->lane_buf[l];
    CK(cudaMemcpyAsync(k->dx, c->host_dx + 3 * m0, sizeof(double) * 3 * chunk, cudaMemcpyHostToDevice, st));
    for (int q = 0; q < 5; ++q)
      CK(cudaMemcpyAsync(b[q], hU[q] + m0 * per[0], sizeof(double) * per[0] * chunk, cudaMemcpyHostToDevice, st));
    for (int q = 0; q < 3; ++q)
      CK(cudaMemcpyAsync(b[5 + q], hB[q] + m0 * per[1 + q], sizeof(double) * per[1 + q] * chunk, cudaMemcpyHostToDevice, st));
    for (int q = 0; q < 16; ++q) k->adm[q] = c->adm[q] + m0 * per[0];
    k->have_metric = true;
    const ak_cons dU_ = {b[0], b[1], b[2], b[3], b[4]};
    const ak_faceB dB_ = {b[5], b[6], b[7]};
    const ak_prim dW_ = {b[8], b[9], b[10], b[11], b[12], b[13], b[14], b[15]};
    const ak_rhs_out dO = {b[16], b[17], b[18], b[19], b[20], b[21], b[22], b[23], c->lane_mask[l][0], c->lane_mask[l][1], nullptr};
    const int r = ak_rhs(k, &dU_, &dB_, &dW_, 0, dt_fofc, &dO);
    if (r != AK_OK) return r;
    if (sparse_u) {
      const long long o0 = m0 * per[0];
      k_writeback_floored<<<148 * 4, 256, 0, st>>>(c->lane_mask[l][1], per[0] * chunk, b[0], b[1], b[2], b[3], b[4],
                                                   mU[0] + o0, mU[1] + o0, mU[2] + o0, mU[3] + o0, mU[4] + o0);
      CK(cudaGetLastError());
    }
    for (int q = 0; q < 5; ++q) {
      if (!sparse_u)
        CK(cudaMemcpyAsync(hU[q] + m0 * per[0], b[q], sizeof(double) * per[0] * chunk, cudaMemcpyDeviceToHost, st));
      CK(cudaMemcpyAsync(hdU[q] + m0 * per[0], b[16 + q], sizeof(double) * per[0] * chunk, cudaMemcpyDeviceToHost, st));
    }
    for (int q = 0; q < 8 && hW[0]; ++q)
      CK(cudaMemcpyAsync(hW[q] + m0 * per[0], b[8 + q], sizeof(double) * per[0] * chunk, cudaMemcpyDeviceToHost, st));
    for (int q = 0; q < 3; ++q)
      CK(cudaMemcpyAsync(hE[q] + m0 * per[4 + q], b[21 + q], sizeof(double) * per[4 + q] * chunk, cudaMemcpyDeviceToHost, st));
    if (hflag) CK(cudaMemcpyAsync(hflag + m0 * per[0], c->lane_mask[l][0], (size_t)per[0] * chunk, cudaMemcpyDeviceToHost, st));
    if (hstatus) CK(cudaMemcpyAsync(hstatus + m0 * per[0], c->lane_mask[l][1], (size_t)per[0] * chunk, cudaMemcpyDeviceToHost, st));
    unsigned long long* hs = c->lane_stats_h + (size_t)(S_NSTAT + 4) * ch;
    CK(cudaMemcpyAsync(hs, k->stats, sizeof(unsigned long long) * S_NSTAT, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(hs + S_NSTAT, k->count, sizeof(unsigned) * 4, cudaMemcpyDeviceToHost, st));
  }
  CK(cudaStreamSynchronize(c->lane[0]->stream));
  CK(cudaStreamSynchronize(c->lane[1]->stream));
  ak_stats acc;
  memset(&acc, 0, sizeof(acc));
  for (int ch = 0; ch < nchunks; ++ch) {
    const unsigned long long* hs = c->lane_stats_h + (size_t)(S_NSTAT + 4) * ch;
    const unsigned* cnt = (const unsigned*)(hs + S_NSTAT);
    acc.n_c2p_fail += (long long)hs[S_C2P_FAIL]; acc.n_cons_floor += (long long)hs[S_CONS_FLOOR];
    acc.n_prim_floor += (long long)hs[S_PRIM_FLOOR]; acc.n_dmp_cells += (long long)hs[S_DMP_CELLS];
    acc.n_fofc_cells += cnt[3];
    for (int d = 0; d < 3; ++d) acc.n_fofc_faces[d] += cnt[d];
  }
  c->host_acc = acc;
  c->stats_from_host = true;
  return AK_OK;
}

int ak_rhs_host(ak_ctx* c, const ak_cons* U, const ak_faceB* Bf, const ak_prim* W, double dt_fofc,
                const ak_rhs_out* out) {
  if (!c || !U || !Bf || !out || out->matter) return AK_EINVAL;
  if (!c->have_metric) return AK_ESTATE;
  CK(cudaSetDevice(c->hp.device));
  const size_t cb = sizeof(double) * c->sz.cell;
  const size_t fb[3] = {sizeof(double) * c->sz.xf, sizeof(double) * c->sz.yf, sizeof(double) * c->sz.zf};
  const size_t eb[3] = {sizeof(double) * c->sz.ex, sizeof(double) * c->sz.ey, sizeof(double) * c->sz.ez};
  double* hU[5] = {U->D, U->Sx, U->Sy, U->Sz, U->tau};
  const double* hB[3] = {Bf->bx, Bf->by, Bf->bz};
  // W == NULL (or all eight members NULL): the primitives stay on the device and are not copied back
  double* hW[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  if (W) { hW[0] = W->rho; hW[1] = W->ux; hW[2] = W->uy; hW[3] = W->uz; hW[4] = W->p; hW[5] = W->bccx; hW[6] = W->bccy; hW[7] = W->bccz; }
  int nW = 0;
  for (int q = 0; q < 8; ++q) nW += hW[q] != nullptr;
  if (nW != 0 && nW != 8) return AK_EINVAL;
  double* hdU[5] = {out->dD, out->dSx, out->dSy, out->dSz, out->dtau};
  double* hE[3] = {out->Ex, out->Ey, out->Ez};
  for (int q = 0; q < 5; ++q) if (!hU[q] || !hdU[q]) return AK_EINVAL;
  for (int q = 0; q < 3; ++q) if (!hB[q] || !hE[q]) return AK_EINVAL;
  {
    // chunk = the largest divisor of nmb not above max(8, nmb / 8); small batches go in one piece
    int chunk = 0;
    const int cap = c->P.nmb / 8 > 8 ? c->P.nmb / 8 : 8;
    if (c->P.nmb >= 16 && !c->blendU0[0])
      for (int q = cap; q >= 4; --q) if (c->P.nmb % q == 0) { chunk = q; break; }
    // lanes exist: keep their chunk size; a FOFC blend set since then goes the unpipelined way (the lanes
    // do not carry the register U0)
    if (c->lane_chunk) chunk = c->blendU0[0] ? 0 : c->lane_chunk;
    if (chunk) return rhs_host_pipelined(c, chunk, hU, hB, hW, dt_fofc, hdU, hE, out->fofc_flag, out->c2p_status);
  }
  if (!c->have_stg) {
    for (int q = 0; q < 5; ++q) { CK(cudaMalloc(&c->stg_U[q], cb)); CK(cudaMalloc(&c->stg_dU[q], cb)); }
    for (int q = 0; q < 8; ++q) CK(cudaMalloc(&c->stg_W[q], cb));
    for (int q = 0; q < 3; ++q) { CK(cudaMalloc(&c->stg_Bf[q], fb[q])); CK(cudaMalloc(&c->stg_E[q], eb[q])); }
    CK(cudaMalloc(&c->stg_flag, (size_t)c->sz.cell));
    CK(cudaMalloc(&c->stg_status, (size_t)c->sz.cell));
    for (int q = 0; q < 5; ++q) CK(cudaMemsetAsync(c->stg_dU[q], 0, cb, c->stream));
    for (int q = 0; q < 3; ++q) CK(cudaMemsetAsync(c->stg_E[q], 0, eb[q], c->stream));
    c->have_stg = true;
  }
  for (int q = 0; q < 5; ++q) CK(cudaMemcpyAsync(c->stg_U[q], hU[q], cb, cudaMemcpyHostToDevice, c->stream));
  for (int q = 0; q < 3; ++q) CK(cudaMemcpyAsync(c->stg_Bf[q], hB[q], fb[q], cudaMemcpyHostToDevice, c->stream));
  ak_cons dU_ = {c->stg_U[0], c->stg_U[1], c->stg_U[2], c->stg_U[3], c->stg_U[4]};
  ak_faceB dB_ = {c->stg_Bf[0], c->stg_Bf[1], c->stg_Bf[2]};
  ak_prim dW_ = {c->stg_W[0], c->stg_W[1], c->stg_W[2], c->stg_W[3], c->stg_W[4], c->stg_W[5], c->stg_W[6], c->stg_W[7]};
  ak_rhs_out dO = {c->stg_dU[0], c->stg_dU[1], c->stg_dU[2], c->stg_dU[3], c->stg_dU[4],
                   c->stg_E[0], c->stg_E[1], c->stg_E[2], c->stg_flag, c->stg_status, nullptr};
  const int r = ak_rhs(c, &dU_, &dB_, &dW_, 0, dt_fofc, &dO);
  if (r != AK_OK) return r;
  for (int q = 0; q < 5; ++q) {
    CK(cudaMemcpyAsync(hU[q], c->stg_U[q], cb, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaMemcpyAsync(hdU[q], c->stg_dU[q], cb, cudaMemcpyDeviceToHost, c->stream));
  }
  for (int q = 0; q < 8 && hW[0]; ++q) CK(cudaMemcpyAsync(hW[q], c->stg_W[q], cb, cudaMemcpyDeviceToHost, c->stream));
  for (int q = 0; q < 3; ++q) CK(cudaMemcpyAsync(hE[q], c->stg_E[q], eb[q], cudaMemcpyDeviceToHost, c->stream));
  if (out->fofc_flag) CK(cudaMemcpyAsync(out->fofc_flag, c->stg_flag, (size_t)c->sz.cell, cudaMemcpyDeviceToHost, c->stream));
  if (out->c2p_status) CK(cudaMemcpyAsync(out->c2p_status, c->stg_status, (size_t)c->sz.cell, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return AK_OK;
}

int ak_set_fofc_blend(ak_ctx* c, const ak_cons* U0, double a, double b) {
  if (!c) return AK_EINVAL;
  if (!U0) {
    for (int q = 0; q < 5; ++q) c->blendU0[q] = nullptr;
    c->blend_a = 0.0; c->blend_b = 1.0;
    return AK_OK;
  }
  if (!U0->D || !U0->Sx || !U0->Sy || !U0->Sz || !U0->tau || !std::isfinite(a) || !std::isfinite(b)) return AK_EINVAL;
  c->blendU0[0] = U0->D; c->blendU0[1] = U0->Sx; c->blendU0[2] = U0->Sy; c->blendU0[3] = U0->Sz; c->blendU0[4] = U0->tau;
  c->blend_a = a; c->blend_b = b;
  return AK_OK;
}

static bool bc_ok(const int bc[3]) {
  if (!bc) return false;
  for (int d = 0; d < 3; ++d) if (bc[d] != AK_BC_PERIODIC && bc[d] != AK_BC_OUTFLOW) return false;
  return true;
}

int ak_fill_ghosts(ak_ctx* c, const int bc[3], const ak_cons* U, const ak_faceB_rw* Bf) {
  if (!c || !bc_ok(bc) || !U || !Bf || !U->D || !U->Sx || !U->Sy || !U->Sz || !U->tau || !Bf->bx || !Bf->by || !Bf->bz)
    return AK_EINVAL;
  CK(cudaSetDevice(c->hp.device));
  DrvFields f;
  memset(&f, 0, sizeof(f));
  f.U[0] = U->D; f.U[1] = U->Sx; f.U[2] = U->Sy; f.U[3] = U->Sz; f.U[4] = U->tau;
  f.Bf[0] = Bf->bx; f.Bf[1] = Bf->by; f.Bf[2] = Bf->bz;
  const long long nt = c->P.nt, nb = c->P.nmb;
  if (c->nbr) {
    const unsigned gf = nblk(nb * nt * nt * (nt + 1), 256);
    for (int pass = 0; pass < 2; ++pass) {
      k_exchange<0><<<nblk(c->sz.cell, 256), 256, 0, c->stream>>>(c->P, f, c->nbr, pass, bc[0], bc[1], bc[2]);
      k_exchange<1><<<gf, 256, 0, c->stream>>>(c->P, f, c->nbr, pass, bc[0], bc[1], bc[2]);
      k_exchange<2><<<gf, 256, 0, c->stream>>>(c->P, f, c->nbr, pass, bc[0], bc[1], bc[2]);
      k_exchange<3><<<gf, 256, 0, c->stream>>>(c->P, f, c->nbr, pass, bc[0], bc[1], bc[2]);
    }
    CK(cudaGetLastError());
    return AK_OK;
  }
  k_fill_cells<<<nblk(c->sz.cell, 256), 256, 0, c->stream>>>(c->P, f, bc[0], bc[1], bc[2]);
  k_fill_faces<0><<<nblk(nb * nt * nt * (nt + 1), 256), 256, 0, c->stream>>>(c->P, f, bc[0], bc[1], bc[2]);
  k_fill_faces<1><<<nblk(nb * nt * nt * (nt + 1), 256), 256, 0, c->stream>>>(c->P, f, bc[0], bc[1], bc[2]);
  k_fill_faces<2><<<nblk(nb * nt * nt * (nt + 1), 256), 256, 0, c->stream>>>(c->P, f, bc[0], bc[1], bc[2]);
  CK(cudaGetLastError());
  return AK_OK;
}

long long ak_halo_slab_elems(const ak_ctx* c, int code) {
  if (!c || code < 0 || code > 26 || code == 13) return -1;
  return slab_elems(code, c->P.n, c->P.is);
}

static int halo_slabs(ak_ctx* c, bool unpack, int ndesc, const long long* desc, const ak_cons* U,
                      const ak_faceB_rw* Bf, double* buf) {
  if (!c || ndesc < 0 || !U || !Bf || !U->D || !U->Sx || !U->Sy || !U->Sz || !U->tau || !Bf->bx || !Bf->by || !Bf->bz)
    return AK_EINVAL;
  if (ndesc == 0) return AK_OK;
  if (!desc || !buf || (((uintptr_t)buf) & 15u) || (((uintptr_t)desc) & 7u)) return AK_EINVAL;
  CK(cudaSetDevice(c->hp.device));
  DrvFields f;
  memset(&f, 0, sizeof(f));
  f.U[0] = U->D; f.U[1] = U->Sx; f.U[2] = U->Sy; f.U[3] = U->Sz; f.U[4] = U->tau;
  f.Bf[0] = Bf->bx; f.Bf[1] = Bf->by; f.Bf[2] = Bf->bz;
  const int nblocks = c->nmb_total > c->P.nmb ? c->nmb_total : c->P.nmb;
  // a face slab of a 32^3 block has 5*4*32*32 cells: 8 chunks of 256 threads make ~10 passes per field
  const long long big = 5LL * c->P.is * c->P.n * c->P.n;
  unsigned chunks = (unsigned)((big + 256 * 10 - 1) / (256 * 10));
  if (chunks < 1) chunks = 1;
  for (int q0 = 0; q0 < ndesc; q0 += 65535) {
    const int nd = ndesc - q0 < 65535 ? ndesc - q0 : 65535;
    const dim3 grid(chunks, (unsigned)nd);
    if (unpack) k_halo_slabs<true><<<grid, 256, 0, c->stream>>>(c->P, f, desc + 3LL * q0, buf, nblocks);
    else k_halo_slabs<false><<<grid, 256, 0, c->stream>>>(c->P, f, desc + 3LL * q0, buf, nblocks);
  }
  CK(cudaGetLastError());
  return AK_OK;
}

int ak_halo_pack(ak_ctx* c, int ndesc, const long long* desc, const ak_cons* U, const ak_faceB_rw* Bf, double* buf) {
  return halo_slabs(c, false, ndesc, desc, U, Bf, buf);
}

int ak_halo_unpack(ak_ctx* c, int ndesc, const long long* desc, const double* buf, const ak_cons* U,
                   const ak_faceB_rw* Bf) {
  return halo_slabs(c, true, ndesc, desc, U, Bf, const_cast<double*>(buf));
}

int ak_set_neighbors(ak_ctx* c, const int* nbr, int nmb_total) {
  if (!c) return AK_EINVAL;
  CK(cudaSetDevice(c->hp.device));
  if (!nbr) {
    CK(cudaStreamSynchronize(c->stream));
    cudaFree(c->nbr); c->nbr = nullptr; c->nmb_total = 0;
    return AK_OK;
  }
  const long long cnt = 27LL * c->P.nmb;
  if (c->P.n < 6) return AK_EINVAL;             // a ghost layer must come from owned elements only
  for (long long q = 0; q < cnt; ++q)
    if (nbr[q] < -1 || nbr[q] >= (nmb_total > c->P.nmb ? nmb_total : c->P.nmb)) return AK_EINVAL;
  if (!c->nbr) CK(cudaMalloc(&c->nbr, sizeof(int) * cnt));
  CK(cudaMemcpyAsync(c->nbr, nbr, sizeof(int) * cnt, cudaMemcpyHostToDevice, c->stream));
  CK(cudaStreamSynchronize(c->stream));        // nbr is the caller's
  c->nmb_total = nmb_total;
  return AK_OK;
}

int ak_stage_update(ak_ctx* c, double a, double b, double dt, const ak_cons* U0, const ak_faceB* B0,
                    const ak_cons* U, const ak_faceB_rw* Bf, const ak_rhs_out* rhs) {
  if (!c || !U0 || !B0 || !U || !Bf || !rhs) return AK_EINVAL;
  if (!std::isfinite(a) || !std::isfinite(b) || !std::isfinite(dt)) return AK_EINVAL;
  DrvFields f;
  memset(&f, 0, sizeof(f));
  f.U[0] = U->D; f.U[1] = U->Sx; f.U[2] = U->Sy; f.U[3] = U->Sz; f.U[4] = U->tau;
  f.U0[0] = U0->D; f.U0[1] = U0->Sx; f.U0[2] = U0->Sy; f.U0[3] = U0->Sz; f.U0[4] = U0->tau;
  f.Bf[0] = Bf->bx; f.Bf[1] = Bf->by; f.Bf[2] = Bf->bz;
  f.B0[0] = B0->bx; f.B0[1] = B0->by; f.B0[2] = B0->bz;
  f.dU[0] = rhs->dD; f.dU[1] = rhs->dSx; f.dU[2] = rhs->dSy; f.dU[3] = rhs->dSz; f.dU[4] = rhs->dtau;
  f.E[0] = rhs->Ex; f.E[1] = rhs->Ey; f.E[2] = rhs->Ez;
  for (int q = 0; q < 5; ++q) if (!f.U[q] || !f.U0[q] || !f.dU[q]) return AK_EINVAL;
  for (int q = 0; q < 3; ++q) if (!f.Bf[q] || !f.B0[q] || !f.E[q]) return AK_EINVAL;
  f.dx = c->dx;
  CK(cudaSetDevice(c->hp.device));
  const long long n = c->P.n, nb = c->P.nmb;
  k_update_cells<<<nblk(nb * n * n * n, 256), 256, 0, c->stream>>>(c->P, f, a, b, dt);
  k_update_faces<0><<<nblk(nb * n * n * (n + 1), 256), 256, 0, c->stream>>>(c->P, f, a, b, dt);
  k_update_faces<1><<<nblk(nb * n * n * (n + 1), 256), 256, 0, c->stream>>>(c->P, f, a, b, dt);
  k_update_faces<2><<<nblk(nb * n * n * (n + 1), 256), 256, 0, c->stream>>>(c->P, f, a, b, dt);
  CK(cudaGetLastError());
  return AK_OK;
}

int ak_advance(ak_ctx* c, int integrator, int nsteps, double dt, const int bc[3], const ak_cons* U,
               const ak_faceB_rw* Bf, const ak_prim* W, unsigned char* flag_or) {
  return ak_advance_hooked(c, integrator, nsteps, dt, bc, U, Bf, W, flag_or, nullptr, nullptr);
}

int ak_advance_hooked(ak_ctx* c, int integrator, int nsteps, double dt, const int bc[3], const ak_cons* U,
                      const ak_faceB_rw* Bf, const ak_prim* W, unsigned char* flag_or, ak_refresh_fn refresh,
                      void* user) {
  if (!c || integrator < 1 || integrator > 3 || nsteps < 0 || !std::isfinite(dt) || !bc_ok(bc) || !U || !Bf || !W)
    return AK_EINVAL;
  if (!c->have_metric) return AK_ESTATE;
  CK(cudaSetDevice(c->hp.device));
  const size_t cb = sizeof(double) * c->sz.cell;
  const size_t fb[3] = {sizeof(double) * c->sz.xf, sizeof(double) * c->sz.yf, sizeof(double) * c->sz.zf};
  const size_t eb[3] = {sizeof(double) * c->sz.ex, sizeof(double) * c->sz.ey, sizeof(double) * c->sz.ez};
  if (!c->have_reg) {
    for (int q = 0; q < 5; ++q) { CK(cudaMalloc(&c->regU0[q], cb)); CK(cudaMalloc(&c->reg_dU[q], cb)); CK(cudaMemsetAsync(c->reg_dU[q], 0, cb, c->stream)); }
    for (int q = 0; q < 3; ++q) { CK(cudaMalloc(&c->regB0[q], fb[q])); CK(cudaMalloc(&c->regE[q], eb[q])); CK(cudaMemsetAsync(c->regE[q], 0, eb[q], c->stream)); }
    CK(cudaMalloc(&c->reg_flag, (size_t)c->sz.cell));
    c->have_reg = true;
  }
  // Shu-Osher form: U <- a U0 + b (U + dt L(U))
  static const double A[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.5, 0.0}, {0.0, 0.75, 1.0 / 3.0}};
  static const double B[3][3] = {{1.0, 0.0, 0.0}, {1.0, 0.5, 0.0}, {1.0, 0.25, 2.0 / 3.0}};
  double* Up[5] = {U->D, U->Sx, U->Sy, U->Sz, U->tau};
  double* Bp[3] = {Bf->bx, Bf->by, Bf->bz};
  const ak_cons R0 = {c->regU0[0], c->regU0[1], c->regU0[2], c->regU0[3], c->regU0[4]};
  const ak_faceB RB0 = {c->regB0[0], c->regB0[1], c->regB0[2]};
  const ak_faceB Bc = {Bf->bx, Bf->by, Bf->bz};
  const ak_rhs_out out = {c->reg_dU[0], c->reg_dU[1], c->reg_dU[2], c->reg_dU[3], c->reg_dU[4],
                          c->regE[0], c->regE[1], c->regE[2], c->reg_flag, nullptr, nullptr};
  // the caller's blend setting is restored afterwards
  const double* sv[5]; for (int q = 0; q < 5; ++q) sv[q] = c->blendU0[q];
  const double sa = c->blend_a, sb = c->blend_b;
  int r = AK_OK;
  for (int step = 0; step < nsteps && r == AK_OK; ++step)
    for (int s = 0; s < integrator && r == AK_OK; ++s) {
      const double a = A[integrator - 1][s], b = B[integrator - 1][s];
      if (refresh && refresh(user) != 0) { r = AK_EHOOK; break; }
      if ((r = ak_fill_ghosts(c, bc, U, Bf)) != AK_OK) break;
      if (s == 0) r = ak_set_fofc_blend(c, nullptr, 0.0, 1.0); else r = ak_set_fofc_blend(c, &R0, a, b);
      if (r != AK_OK) break;
      if ((r = ak_rhs(c, U, &Bc, W, 0, dt, &out)) != AK_OK) break;
      if (flag_or) k_or_bytes<<<148 * 8, 256, 0, c->stream>>>(flag_or, c->reg_flag, c->sz.cell);
      if (s == 0 && integrator > 1) {
        // step-start register: the state after the first stage's con2prim (floored)
        cudaError_t ce = cudaSuccess;
        for (int q = 0; q < 5 && ce == cudaSuccess; ++q)
          ce = cudaMemcpyAsync(c->regU0[q], Up[q], cb, cudaMemcpyDeviceToDevice, c->stream);
        for (int q = 0; q < 3 && ce == cudaSuccess; ++q)
          ce = cudaMemcpyAsync(c->regB0[q], Bp[q], fb[q], cudaMemcpyDeviceToDevice, c->stream);
        if (ce != cudaSuccess) { last_cuda_error = ce; r = AK_ECUDA; break; }   // the blend is restored below
      }
      if (s == 0) r = ak_stage_update(c, 0.0, 1.0, dt, U, &Bc, U, Bf, &out);    // register = the state itself
      else r = ak_stage_update(c, a, b, dt, &R0, &RB0, U, Bf, &out);
    }
  for (int q = 0; q < 5; ++q) c->blendU0[q] = sv[q];
  c->blend_a = sa; c->blend_b = sb;
  if (r != AK_OK) return r;
  if (refresh && refresh(user) != 0) return AK_EHOOK;
  return ak_fill_ghosts(c, bc, U, Bf);
}

int ak_probe_copy(ak_ctx* c, double* dst, const double* src, long long n, int reps, double* gbs) {
  if (!c || !dst || !src || n < 2 || reps < 1 || !gbs) return AK_EINVAL;
  if (((uintptr_t)dst | (uintptr_t)src) & 15u) return AK_EINVAL;
  CK(cudaSetDevice(c->hp.device));
  cudaEvent_t a, b;
  CK(cudaEventCreate(&a)); CK(cudaEventCreate(&b));
  const long long n2 = n / 2;
  double best = 0.0;
  for (int r = 0; r < reps + 1; ++r) {
    CK(cudaEventRecord(a, c->stream));
    k_probe_copy<<<148 * 16, 256, 0, c->stream>>>((double2*)dst, (const double2*)src, n2);
    CK(cudaEventRecord(b, c->stream));
    CK(cudaEventSynchronize(b));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, a, b));
    const double g = 2.0 * 16.0 * (double)n2 / (ms * 1e-3) * 1e-9;
    if (r > 0 && g > best) best = g;
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  CK(cudaGetLastError());
  *gbs = best;
  return AK_OK;
}

int ak_probe_fp64(ak_ctx* c, int use_fma, int reps, double* gops) {
  if (!c || reps < 1 || !gops) return AK_EINVAL;
  CK(cudaSetDevice(c->hp.device));
  cudaEvent_t a, b;
  CK(cudaEventCreate(&a)); CK(cudaEventCreate(&b));
  const int iters = 4096, grid = 148 * 8, block = 256;
  double best = 0.0;
  for (int r = 0; r < reps + 1; ++r) {
    CK(cudaEventRecord(a, c->stream));
    if (use_fma) k_probe_fp64<true><<<grid, block, 0, c->stream>>>((double*)c->stats, iters, 1.0000001, 1e-9);
    else k_probe_fp64<false><<<grid, block, 0, c->stream>>>((double*)c->stats, iters, 1.0000001, 1e-9);
    CK(cudaEventRecord(b, c->stream));
    CK(cudaEventSynchronize(b));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, a, b));
    // thread-level fp64 instructions: 8 chains x iters x (1 FMA | MUL+ADD)
    const double ops = (double)grid * block * 8.0 * iters * (use_fma ? 1.0 : 2.0);
    const double g = ops / (ms * 1e-3) * 1e-9;
    if (r > 0 && g > best) best = g;
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  CK(cudaGetLastError());
  *gops = best;
  return AK_OK;
}

// ------------------------------------------------------------------ allocation-free entry point
// ak_con2prim_static (include/ak.h): part (1) without a context.  k_con2prim needs scratch besides its inputs
// and outputs -- the device counters, and a place for the status bytes when the caller passes none -- which
// ak_create cudaMallocs.  Here that scratch is a file-scope device array of a fixed, modest size, so the call
// allocates nothing (callers under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc).
// Every GPU that loads the library holds the array until exit.
}  // extern "C" (closed for the file-scope definitions; reopened below)

namespace {
struct StaticScratch {
  unsigned long long stats[S_NSTAT];                 // device counters: must start at zero, cleared per call
  unsigned char status[AK_STATIC_MAX_CELLS];         // status bytes when the caller passes none: fully overwritten
};
static __device__ __align__(256) StaticScratch g_static_scratch;
// In host code `g_static_scratch` is a host-side stand-in, NOT a device address: the address a kernel may use
// comes from cudaGetSymbolAddress, once per device, with that device current.
StaticScratch* g_static_ptr[64] = {nullptr};
}  // namespace

extern "C" {

int ak_con2prim_static(const ak_params* p, const ak_cons* U, const ak_faceB* Bf, const ak_adm* adm,
                       const ak_prim* W, unsigned char* status, ak_stats* host_counts) {
  if (!p || !U || !Bf || !adm || !W) return AK_EINVAL;
  if (p->nmb < 1 || p->n < 2 || p->ng != 4) return AK_EINVAL;
  if (!(std::isfinite(p->gamma_ad) && p->gamma_ad > 1.0)) return AK_EINVAL;
  if (!finite_pos(p->rho_atm) || !finite_pos(p->T_atm) || !finite_pos(p->f_thr)) return AK_EINVAL;
  if (!(p->mag_max > 0.0)) return AK_EINVAL;
  if (p->c2p_max_iter < 1 || p->c2p_max_iter > 1000 || !(p->c2p_tol > 0.0 && p->c2p_tol < 1.0)) return AK_EINVAL;
  if (p->device < 0 || p->device >= 64) return AK_EINVAL;
  const long long nt = p->n + 8;
  const long long ncell = (long long)p->nmb * nt * nt * nt;
  if (ncell > (long long)AK_STATIC_MAX_CELLS) return AK_ETOOBIG;      // the status scratch holds no more
  Fields f;
  memset(&f, 0, sizeof(f));
  if (!set_cons(f, U) || !set_faceB(f, Bf) || !set_prim(f, W)) return AK_EINVAL;       // NULL or not 16-byte aligned
  const double* g6[6] = {adm->gxx, adm->gxy, adm->gxz, adm->gyy, adm->gyz, adm->gzz};   // part (1) reads gamma_ij only
  for (int q = 0; q < 6; ++q) { if (!al16(g6[q])) return AK_EINVAL; f.adm[q] = g6[q]; }
  CK(cudaSetDevice(p->device));
  StaticScratch*& sp = g_static_ptr[p->device];
  if (!sp) {                                   // set-up, once per device, with that device current
    void* a = nullptr;
    CK(cudaGetSymbolAddress(&a, g_static_scratch));
    sp = (StaticScratch*)a;
  }
  Par P;
  memset(&P, 0, sizeof(P));
  P.nmb = p->nmb; P.n = p->n; P.nt = (int)nt; P.px = P.nt + 4; P.is = 4; P.ie = p->n + 3;
  P.Gam = p->gamma_ad; P.gm1 = p->gamma_ad - 1.0; P.gm1r = p->gamma_ad / (p->gamma_ad - 1.0);
  P.rho_atm = p->rho_atm; P.T_atm = p->T_atm; P.P_atm = p->rho_atm * p->T_atm;
  P.eps_atm = p->T_atm / P.gm1; P.thr = p->f_thr * p->rho_atm;
  P.mag_max = p->mag_max;
  P.max_iter = p->c2p_max_iter; P.tol = p->c2p_tol;
  P.shortcuts = 3;
  f.stats = sp->stats;
  f.status = status ? status : sp->status;
  cudaStream_t st = (cudaStream_t)p->stream;
  CK(cudaMemsetAsync(sp->stats, 0, sizeof(unsigned long long) * S_NSTAT, st));   // the array keeps the last call's counts
  k_con2prim<false, 0><<<nblk(ncell, 128), 128, 0, st>>>(P, f);
  CK(cudaGetLastError());
  if (host_counts) {                           // the only part that synchronises
    unsigned long long h[S_NSTAT];
    CK(cudaMemcpyAsync(h, sp->stats, sizeof(h), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    memset(host_counts, 0, sizeof(*host_counts));
    host_counts->n_c2p_fail = (long long)h[S_C2P_FAIL];
    host_counts->n_cons_floor = (long long)h[S_CONS_FLOOR];
    host_counts->n_prim_floor = (long long)h[S_PRIM_FLOOR];
  }
  return AK_OK;
}

}  // extern "C"
