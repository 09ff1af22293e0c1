/* include/ak.h — C-ABI boundary of the B200-native GRMHD right-hand-side stage.
 *
 * What the library computes: one finite-volume RHS stage of the 3+1 Valencia GRMHD system
 * of arXiv:2409.10384 on a frozen ADM snapshot, over a batch of independent MeshBlocks.
 * Citations "P:n" are line numbers of PAPER.md; "D:§" are sections of DESIGN.md.
 *
 *   part (1) conservative -> primitive recovery, ideal gas, floors/atmosphere
 *   part (2) donor-cell / PPM4 / WENO-Z reconstruction of (rho, W v^i, P, B~)
 *   part (3) LLF / HLLE fluxes of Eq. 8 with a face-averaged metric
 *   part (4) first-order flux correction, optional relaxed maximum principle   P:141-157 (Eq. 12)
 *   part (5) upwind constrained-transport edge EMFs
 *   part (6) flux divergence + geometric sources of Eq. 9
 *
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.  All
 * arithmetic is IEEE fp64 (the library is built with --fmad=false so that masks are
 * bit-reproducible against the reference arithmetic stated in D:§3).
 *
 * ---- Layout (D:§2).  A MeshBlock has n^3 interior cells and ng = 4 ghost layers per side;
 * nt = n + 8 stored cells per direction; i (x) is the fastest index, then j, k, then block m.
 * px = nt + 4 is the padded pitch of every array that has nt+1 points along x (row stride a
 * multiple of 32 B).  Face i of direction x lies between cells i-1 and i; likewise j, k.
 *   cell field    [nmb][nt][nt][nt]
 *   x-face field  [nmb][nt][nt][px]        (nt+1 used)
 *   y-face field  [nmb][nt][nt+1][nt]
 *   z-face field  [nmb][nt+1][nt][nt]
 *   E_x (x-edges) [nmb][nt+1][nt+1][nt]
 *   E_y (y-edges) [nmb][nt+1][nt][px]
 *   E_z (z-edges) [nmb][nt][nt+1][px]
 * A tilde means "densitised", i.e. multiplied by sqrt(det gamma_ij).
 *
 * ---- Ownership.  Every field pointer is a DEVICE pointer owned by the caller (fp64, the base
 * of every field 16-byte aligned — checked, AK_EINVAL otherwise: rows are staged with TMA bulk
 * copies, which need it; or bytes for masks) unless a function says "host".  The context borrows
 * pointers for the duration of one call (metric: until replaced or ak_destroy) and owns
 * only its scratch (face fluxes, cell-centred EMFs, FOFC face lists, counters).
 *
 * ---- Asynchrony.  ak_con2prim / ak_rhs / ak_emf enqueue on the context's stream and
 * return; they never synchronise.  ak_get_stats and the *_host entry points synchronise.
 * With an overlapped schedule (ak_set_overlap) ak_rhs forks onto context-owned streams and
 * joins back: work enqueued on the context's stream before the call is complete before any
 * kernel of the stage starts, and work enqueued after it starts after the whole stage.
 *
 * ---- Errors.  Return codes report API misuse and CUDA failures only.  Unphysical cells
 * are data ("it is flagged"): they are reported through status / flag bytes and the
 * counters of ak_stats.
 */
#ifndef AK_H
#define AK_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ak_ctx ak_ctx; /* opaque */

enum { AK_OK = 0, AK_EINVAL = -1, AK_ENOMEM = -2, AK_ECUDA = -3, AK_ESTATE = -4, AK_EHOOK = -5, AK_ETOOBIG = -6 };
enum { AK_RECON_DC = 0, AK_RECON_PPM4 = 1, AK_RECON_WENOZ = 2, AK_RECON_PLM = 3, AK_RECON_PPMX = 4 };
enum { AK_RS_LLF = 0, AK_RS_HLLE = 1 };
enum { AK_BC_PERIODIC = 0, AK_BC_OUTFLOW = 1 };                  /* stage driver, D:§11 */
enum { AK_RK1 = 1, AK_RK2 = 2, AK_RK3 = 3 };                     /* SSP Runge-Kutta */

/* status / flag bits (D:§2.4).  status = what con2prim did to a cell; fofc_flag = the status
 * of the FOFC estimate of that cell, plus AK_ST_DMP (Eq. 12). */
enum {
  AK_ST_DFLOOR = 1,    /* D < f_thr rho_atm: cell reset to static atmosphere        */
  AK_ST_TAUFLOOR = 2,  /* tau raised to tau_atm(D,B)                                */
  AK_ST_MAGCAP = 4,    /* D raised to B^2 / M_max                                   */
  AK_ST_RHOFLOOR = 8,  /* recovered rho < f_thr rho_atm: reset to atmosphere        */
  AK_ST_TFLOOR = 16,   /* recovered T < T_atm: T reset, P recomputed                */
  AK_ST_FAIL = 32,     /* non-finite input, no bracket or no convergence: atmosphere */
  AK_ST_DMP = 64       /* discrete maximum principle violated (flag byte only)       */
};

typedef struct {
  int nmb, n, ng;            /* MeshBlocks, interior cells per edge (even, >= 4), ghosts (== 4) */
  double gamma_ad;           /* ideal-gas Gamma > 1; P = (Gamma-1) rho eps, T = P/rho (D:R3)     */
  double rho_atm, T_atm;     /* atmosphere density and temperature                      */
  double f_thr;              /* threshold factor on rho_atm                             */
  double mag_max;            /* M_max: cap on B^2/D; +inf disables                      */
  int recon;                 /* AK_RECON_* of the high-order pass                               */
  int riemann;               /* AK_RS_*    of the high-order pass                               */
  int fofc;                  /* 0/1: first-order flux correction                        */
  int fofc_riemann;          /* AK_RS_* used when a face is redone at first order       */
  double dmp_M;              /* <= 0: no maximum principle; else M >= 1 of Eq. 12       */
  int c2p_max_iter;          /* cap on master-function evaluations per root find (e.g. 40)      */
  double c2p_tol;            /* relative step tolerance on mu (e.g. 1e-15)                      */
  int device;                /* CUDA device ordinal                                             */
  void* stream;              /* cudaStream_t (0 = legacy default stream)                        */
} ak_params;

typedef struct { double *D, *Sx, *Sy, *Sz, *tau; } ak_cons;              /* cell fields, U~   */
typedef struct { const double *bx, *by, *bz; } ak_faceB;                 /* face fields, B~f  */
typedef struct { double *bx, *by, *bz; } ak_faceB_rw;                    /* ... written       */
typedef struct { double *rho, *ux, *uy, *uz, *p, *bccx, *bccy, *bccz; } ak_prim;
                                   /* cell fields: rho, u^i = W v^i, P, cell-centred B~^i     */
typedef struct {
  const double *gxx, *gxy, *gxz, *gyy, *gyz, *gzz, *alp, *betx, *bety, *betz,
               *Kxx, *Kxy, *Kxz, *Kyy, *Kyz, *Kzz;
} ak_adm;                          /* cell fields: gamma_ij, alpha, beta^i, K_ij (Eq. 5)      */
/* Matter terms a spacetime (Z4c) right-hand side needs from the fluid ("E = tau + D ...
 * S_ij = T_ij"): E, S_i, S_ij, undensitised.  Ten caller-owned device cell fields. */
typedef struct { double *E, *Sx, *Sy, *Sz, *Sxx, *Sxy, *Sxz, *Syy, *Syz, *Szz; } ak_matter;

typedef struct {
  double *dD, *dSx, *dSy, *dSz, *dtau; /* cell fields; interior cells written, rest untouched */
  double *Ex, *Ey, *Ez;                /* edge fields; edges of interior cells written        */
  unsigned char* fofc_flag;            /* [nmb][nt^3] bytes, fully written (0 outside the     */
                                       /* tested range); may be NULL                          */
  unsigned char* c2p_status;           /* [nmb][nt^3] bytes, written when part (1) runs;      */
                                       /* may be NULL                                         */
  const ak_matter* matter;             /* may be NULL.  Else part (6) also writes the matter  */
                                       /* terms of the stage's primitives on the INTERIOR     */
                                       /* cells (the rest untouched): a fused epilogue of the */
                                       /* divergence+source kernel, which holds E, S_i, S_ij  */
                                       /* in registers (S:§8(f) rank 4).  Same bits as        */
                                       /* ak_matter_sources.  Must be NULL for ak_rhs_host.   */
} ak_rhs_out;

typedef struct {
  long long n_c2p_fail;      /* cells whose con2prim status has AK_ST_FAIL (last part (1))      */
  long long n_cons_floor;    /* ... any of DFLOOR | TAUFLOOR | MAGCAP                           */
  long long n_prim_floor;    /* ... any of RHOFLOOR | TFLOOR                                    */
  long long n_fofc_cells;    /* cells flagged by the last FOFC test                             */
  long long n_dmp_cells;     /* ... of which carry AK_ST_DMP                                    */
  long long n_fofc_faces[3]; /* faces redone at first order, per direction                      */
} ak_stats;

/* Create a context for a batch shape and a parameter set.  dx3 is a HOST array [nmb][3] of
 * cell widths (dx,dy,dz) per block; it is copied.  Validates everything before touching
 * CUDA (AK_EINVAL), then allocates scratch (AK_ENOMEM / AK_ECUDA). */
int ak_create(const ak_params* p, const double* dx3, ak_ctx** out);

/* Borrow the frozen ADM snapshot (16 cell fields).  Must precede the compute calls. */
int ak_set_metric(ak_ctx*, const ak_adm* adm);

/* Part (1) over all nt^3 stored cells of every block (floors are applied "after ...
 * the conserved-to-primitive inversion"; ghosts are needed by parts (2)-(4)).
 * U is in-out: cells with a non-zero status are rewritten from the final primitives
 * ("a similar policy holds for the conserved variables").  status may be NULL. */
int ak_con2prim(ak_ctx*, const ak_cons* U, const ak_faceB* Bf, const ak_prim* W,
                unsigned char* status);

/* Parts (1)-(6).  If w_is_valid != 0 part (1) is skipped and W is read as given.
 * dt_fofc is the time step of the FOFC estimate U* = U - dt_fofc div F (D:R9). */
int ak_rhs(ak_ctx*, const ak_cons* U, const ak_faceB* Bf, const ak_prim* W, int w_is_valid,
           double dt_fofc, const ak_rhs_out* out);

/* Schedule of ak_rhs (and of the stages of ak_advance).  nchunks < 2 (the state after ak_create
 * unless the environment variable AK_OV_CHUNKS is set): the kernels of parts (1)-(6) run one after
 * another over the whole batch on the context's stream.  nchunks >= 2 (at most 64): MeshBlocks are
 * independent (S:§8(e)), so the batch is cut into nchunks contiguous groups of blocks and the stage is
 * pipelined over them on three context-owned streams: part (1) of group i+1 and parts (4)-(6) of group
 * i-1 — bound by memory latency and bandwidth — run with capped grids and high priority beside the
 * fp64-bound sweeps (2)+(3) of group i, so that both the fp64 pipe and HBM stay busy (D:§6.2).  Same
 * kernels, same arithmetic, the same bits out; only events order the streams (no kernel waits on
 * another).  nchunks is clamped to nmb. */
int ak_set_overlap(ak_ctx*, int nchunks);

/* CUDA-graph replay of the stage ("launches captured once in a CUDA graph per ctx"; D:§6.4).  With on != 0,
 * ak_rhs in the serial schedule runs an argument set (every pointer, the parameters, w_is_valid, dt_fofc, the
 * FOFC blend, the shortcut mask) plainly the first time it sees it, captures the same launch sequence into a
 * CUDA graph the second time (on a context-owned stream: the caller's may be the legacy default stream, which
 * cannot capture) and from then on replays it with one cudaGraphLaunch on the context's stream.  Up to four
 * argument sets are kept (the stages of an SSP-RK3 step differ in their blend), least recently used evicted.
 * Same kernels, same bits.  It pays where a stage is launch-bound (a few small MeshBlocks: D:§6.4 has the
 * numbers), not on large batches.  Bypassed while ak_timing is enabled and under ak_set_overlap.  on == 0
 * synchronises the context's stream and destroys the graphs.  ak_graph_replays: stages replayed from a graph
 * since the last ak_set_graph (diagnostic; < 0 for a NULL context). */
int ak_set_graph(ak_ctx*, int on);
long long ak_graph_replays(const ak_ctx*);

/* Exact data-dependent shortcuts (D:§6.3).  mask bit 0: a field of (u^x, u^y, u^z, B~cc^t1, B~cc^t2) that is
 * +0.0 on the whole tile a sweep block stages is not reconstructed (every scheme of P:133 returns +0.0 on
 * both sides of every face for it); bit 1: a cell with S~ = 0 and B~ = 0 exactly runs its con2prim root
 * find on f(mu) = mu - const, which is what the master function then is, and a cell with B = 0 evaluates
 * the master function with x = 1, rbar^2 = r^2, qbar = q; bit 2: a sweep block whose tile
 * holds u^i = +0.0 and every B~ component +0.0 evaluates the face flux of Eq. 8 with W = 1, v = 0, B = 0
 * substituted (no index lowering, no Lorentz factor, no Alfven speed: what side_state computes then, term
 * by term), and one whose tile holds moving matter but every B~ component +0.0 with B = 0 substituted.
 * With all three on, batches of >= 2^23 stored cells also sort their sweep tiles on the device into a static
 * and a general list and run the static ones through a lighter kernel (D:§6 item 29; AK_SPLIT_BLOCKS=0/1
 * at ak_create forces that off / on).  All of it leaves every output bit unchanged (the parity tests run with them on and off); what
 * they change is the time on inputs with exact zeros — static atmosphere, unmagnetised regions: most of a
 * merger grid.  Default 7 (all; also settable by the environment variable AK_EXACT_SHORTCUTS at
 * ak_create); 0 times the full arithmetic. */
int ak_set_exact_shortcuts(ak_ctx*, int mask);

/* Part (5) alone, from the (post-FOFC) fluxes the last ak_rhs left in the context
 * (AK_ESTATE if there are none) and the primitives W. */
int ak_emf(ak_ctx*, const ak_prim* W, double* Ex, double* Ey, double* Ez);

/* The matter terms (ak_matter above) at EVERY stored cell, ghosts included, from the primitives W and
 * the metric set with ak_set_metric: the stand-alone pass; ak_rhs_out.matter gives the interior cells
 * for free inside a stage. */
int ak_matter_sources(ak_ctx*, const ak_prim* W, const ak_matter* out);

/* Copy the device counters to the host.  Synchronises the stream. */
int ak_get_stats(ak_ctx*, ak_stats* host_out);

/* Read back one post-FOFC face-flux field kept in scratch (dir 0..2, comp 0..6 =
 * D,Sx,Sy,Sz,tau,B~t1,B~t2 with t1,t2 cyclic after dir) into a caller DEVICE buffer in the
 * face layout of dir.  For tests and diagnostics.  AK_ESTATE before the first ak_rhs. */
int ak_get_flux(ak_ctx*, int dir, int comp, double* dst);

/* End-to-end convenience: the same stage with HOST buffers.  All pointers inside U, Bf,
 * W, out are host pointers (pinned memory recommended); the metric must already be set with
 * ak_set_metric (device pointers: the snapshot is frozen across stages).  Copies U and Bf
 * to context-owned device staging, runs parts (1)-(6), copies back U (floored cells), W,
 * dU, E and the two masks, and synchronises.  Staging is allocated on first use.
 * U is written back only where part (1) changed it: when all five U arrays are pinned (cudaHostAlloc /
 * cudaHostRegister) host memory, the pipelined path stores just the cells with a non-zero status straight into
 * them instead of copying the fields back whole (the values are the same either way); pageable arrays are copied.
 * W == NULL (or all eight members NULL): the primitives are an intermediate of the stage and are not
 * copied back (3.1 of the 8.5 GB a C4 stage would otherwise return).  Batches of >= 16 blocks are
 * pipelined in chunks over two internal streams so that H2D, kernels and D2H overlap; the fluxes of such
 * a stage stay in the pipeline's contexts (ak_emf / ak_get_flux afterwards: AK_ESTATE). */
int ak_rhs_host(ak_ctx*, const ak_cons* U, const ak_faceB* Bf, const ak_prim* W,
                double dt_fofc, const ak_rhs_out* out);

/* ---- stage driver (D:§11; "RK2 ... RK3", method of lines; P:141 FOFC per stage) -------
 * Every MeshBlock is treated as its own domain: ghosts are filled from the block itself.
 *
 * FOFC estimate of a later Runge-Kutta stage ("the next Runge-Kutta step is estimated"):
 * subsequent ak_rhs calls test U* = a U0 + b (U - dt_fofc div F).  U0 (device, borrowed until
 * replaced) = the step-start register; U0 == NULL restores U* = U - dt_fofc div F. */
int ak_set_fofc_blend(ak_ctx*, const ak_cons* U0, double a, double b);

/* Equation of state (S:§8(f) rank 3; "supports ideal gases and piecewise polytropic hybrid
 * EOSs"; the paper prints no formula, D:§10 reading R29 fixes it).  After this call every part of
 * the stage (con2prim, floors, fluxes, FOFC test, sources, ak_matter_sources) uses
 *   cold curve, segment i (rho_breaks[i-1] <= rho < rho_breaks[i]):
 *     P_c = K_i rho^Gamma_i,  eps_c = a_i + K_i rho^(Gamma_i-1)/(Gamma_i-1),
 *     K_0 = K0, a_0 = 0, K_i and a_i continuous at the breakpoints;
 *   P = P_c + (gamma_th-1) rho (eps - eps_c);  T = (P - P_c)/rho (so T_atm floors the thermal part
 *   and K0 = 0 is the ideal gas with Gamma = gamma_th);  h = 1 + eps + P/rho;
 *   c_s^2 = (Gamma_i P_c + gamma_th (P - P_c))/(rho h);  atmosphere P = P_c(rho_atm) + rho_atm T_atm.
 * nseg in 1..4; gammas = HOST [nseg], each > 1; rho_breaks = HOST [nseg-1], positive and increasing
 * (ignored for nseg = 1); K0 >= 0; gamma_th > 1: else AK_EINVAL, nothing changed.  The arrays are
 * copied.  ak_params.gamma_ad is then unused.  nseg = 0 returns to the ideal gas of ak_params.
 * rho^Gamma is the device pow(): results agree with a libm evaluation to rounding, not bit for bit.
 * The hybrid stage runs the same TMA-staged flux sweeps as the ideal gas (kernels templated on the EOS). */
int ak_set_eos_hybrid(ak_ctx*, int nseg, double K0, const double* gammas, const double* rho_breaks,
                      double gamma_th);

/* Same-level neighbour table for ak_fill_ghosts / ak_advance (D:§12; "interblock
 * communication"): nbr = HOST int [nmb][27], entry (oz+1)*9+(oy+1)*3+(ox+1) = index of the block
 * adjacent at offset (ox,oy,oz) in {-1,0,1}^3, -1 = none (entry 13, the block itself, is ignored).
 * It is copied.  With a table set, ghosts whose offset block exists are copied from that block's
 * interior (the shared face ie+1 from the upper neighbour's face is); sides without a face
 * neighbour are physical and get bc[d].  Needs n >= 6.  nbr == NULL removes the table.
 * nmb_total >= nmb (0 = nmb): the U~ and B~f arrays later passed to ak_fill_ghosts / ak_advance hold
 * nmb_total blocks, of which only the first nmb are this context's; the others are read-only
 * mirrors of blocks owned elsewhere (another GPU's shard, refreshed by the caller before each
 * ghost fill — paper_2409_10384_b200/halo.py) and table entries may point at them. */
int ak_set_neighbors(ak_ctx*, const int* nbr, int nmb_total);

/* ---- ghost slabs for the exchange across GPUs (D:§12) ------------------------------
 * A slab is the part of one block that a block which has it as neighbour `code` (the table index
 * above: the offset from the reader to this block) reads in ak_fill_ghosts.  Per axis with offset o,
 * cell-like indices [n, n+ng) for o = -1, [ng, 2ng) for o = +1, [ng, ng+n) for o = 0; along the normal
 * of a face field [n, n+ng), [ng, 2ng+1), [ng, ng+n+1) (the faces it owns, plus face ie+1 where the
 * reader may take it).  In the buffer a slab holds D~, S~x, S~y, S~z, tau~, then B~f^x, B~f^y, B~f^z,
 * each box k-major.  ak_halo_slab_elems: doubles in one slab (host arithmetic; < 0 for a bad code).
 * ak_halo_pack gathers ndesc slabs into buf, ak_halo_unpack scatters them back (into mirror blocks):
 * desc = DEVICE int64 [ndesc][3] = {block, code, offset of the slab in buf in doubles}; block is an
 * index into the arrays passed (0 <= block < the nmb_total of ak_set_neighbors, else nmb); a
 * descriptor out of range is skipped.  buf = DEVICE doubles, caller-owned, 16-byte aligned.
 * Asynchronous on the context's stream; only these slabs' elements are touched. */
long long ak_halo_slab_elems(const ak_ctx*, int code);
int ak_halo_pack(ak_ctx*, int ndesc, const long long* desc, const ak_cons* U, const ak_faceB_rw* Bf,
                 double* buf);
int ak_halo_unpack(ak_ctx*, int ndesc, const long long* desc, const double* buf, const ak_cons* U,
                   const ak_faceB_rw* Bf);

/* Fill the ghost cells of U~ and the ghost faces of B~f in place.  bc[d] = AK_BC_* per direction:
 * periodic (face ie+1 is made a copy of face is) or outflow (zero-gradient copies). */
int ak_fill_ghosts(ak_ctx*, const int bc[3], const ak_cons* U, const ak_faceB_rw* Bf);

/* One Shu-Osher register update with the outputs of ak_rhs:
 *   U~ <- a U0 + b (U~ + dt dU~/dt) on interior cells,
 *   B~f <- a B0 + b (B~f + dt (-curl E)) on the faces of interior cells (constrained transport).
 * U0/B0 may alias U/Bf (first stage: a = 0, b = 1). */
int ak_stage_update(ak_ctx*, double a, double b, double dt, const ak_cons* U0, const ak_faceB* B0,
                    const ak_cons* U, const ak_faceB_rw* Bf, const ak_rhs_out* rhs);

/* nsteps steps of SSP-RK<integrator> with a fixed dt, all on the device: per stage
 * ak_fill_ghosts -> ak_rhs (with the stage's FOFC blend) -> ak_stage_update; ghosts filled at the
 * end.  Registers (U0, B0, dU, E, flags) are context-owned, allocated on first use.  W receives
 * the last stage's primitives.  flag_or (device bytes [nmb][nt^3], may be NULL) accumulates the OR
 * of the FOFC flags of every stage (caller zeroes it). */
int ak_advance(ak_ctx*, int integrator, int nsteps, double dt, const int bc[3], const ak_cons* U,
               const ak_faceB_rw* Bf, const ak_prim* W, unsigned char* flag_or);

/* ak_advance with a caller hook: refresh(user) is called on the HOST before every ghost fill (each
 * stage, and the fill at the end) — the point where a multi-GPU driver refreshes the mirror blocks of
 * ak_set_neighbors (pack, NCCL send/recv, unpack, all enqueued on the context's stream by the hook;
 * D:§12).  The stage sequence and the Shu-Osher weights stay inside the library.  A non-zero
 * return aborts with AK_EHOOK (the FOFC blend is restored).  refresh == NULL: ak_advance. */
typedef int (*ak_refresh_fn)(void* user);
int ak_advance_hooked(ak_ctx*, int integrator, int nsteps, double dt, const int bc[3], const ak_cons* U,
                      const ak_faceB_rw* Bf, const ak_prim* W, unsigned char* flag_or,
                      ak_refresh_fn refresh, void* user);

/* Device-timing hooks for the benchmark: bracket kernel class `which` (0 con2prim, 1-3 flux
 * sweeps x/y/z, 4 FOFC test, 5 FOFC list+reflux, 6 cell EMF+CT, 7 divergence+sources) with
 * CUDA events on the stream the class is launched on in subsequent calls; ak_kernel_ms synchronises
 * and returns the accumulated milliseconds and launch count since ak_timing was enabled.
 * Serial schedule: the classes partition the stage, their times add up to it.  Overlapped schedule:
 * a class's time is the span from its first block starting to its last block finishing while kernels
 * of the other streams share the SMs — spans overlap, their sum exceeds the stage time, and a span is
 * NOT the kernel's stand-alone duration (use the serial schedule for per-kernel rooflines). */
int ak_timing(ak_ctx*, int enable);
int ak_kernel_ms(ak_ctx*, double ms_out[8], long long launches_out[8]);

/* Peak probes used as same-run roofline denominators (D:§7): a fp64 copy kernel over
 * nbytes (read+write counted) and an independent-DADD/DMUL/DFMA stream.  Results in GB/s and
 * Gop/s (warp-wide fp64 instructions x 32 lanes / s).  Synchronise. */
int ak_probe_copy(ak_ctx*, double* dst, const double* src, long long n_doubles, int reps,
                  double* gbs_out);
int ak_probe_fp64(ak_ctx*, int use_fma, int reps, double* gops_out);

/* ---- allocation-free entry point -------------------------------------------------------------------
 * Part (1) (ideal gas) WITHOUT a context, for callers that cannot call cudaMalloc
 * (code under CUDA-graph capture, tight serving loops, harnesses that forbid it): ak_create allocates its
 * scratch with cudaMalloc; this call, and everything it calls, allocates nothing — no cudaMalloc, cudaFree
 * or allocating library routine.  The scratch the kernel needs (the device counters, and the status bytes
 * when `status` is NULL) lives in a file-scope device array inside the library, sized for at most
 * AK_STATIC_MAX_CELLS stored cells (nmb * (n+8)^3; 2 MiB + 64 B, held by every GPU that loads the library
 * until exit).  A larger batch is refused with AK_ETOOBIG before anything is launched.
 *   p        nmb, n, ng, gamma_ad, rho_atm, T_atm, f_thr, mag_max, c2p_max_iter, c2p_tol, device (< 64),
 *            stream are read; the rest is ignored.
 *   U        in-out, Bf in, W out: DEVICE fields as for ak_con2prim (16-byte aligned, else AK_EINVAL).
 *   adm      only gxx..gzz are read (DEVICE cell fields).
 *   status   DEVICE bytes [nmb][nt^3], or NULL.
 *   host_counts  NULL: the call only enqueues on p->stream and returns.  Else n_c2p_fail, n_cons_floor,
 *            n_prim_floor of this call are written there (the other members 0) and the call synchronises
 *            p->stream.
 * Same kernel and arithmetic as ak_con2prim: the same bits in W, U and status.
 * ALL calls share the one scratch array, which keeps the last call's contents (the counters are cleared at
 * the start of each call, on its stream).  Calls that overlap on the GPU — different streams, or another
 * thread — race on it: serialise them (one stream, or events).  Calls on different devices do not share. */
#define AK_STATIC_MAX_CELLS 2097152
int ak_con2prim_static(const ak_params* p, const ak_cons* U, const ak_faceB* Bf, const ak_adm* adm,
                       const ak_prim* W, unsigned char* status, ak_stats* host_counts);

int ak_destroy(ak_ctx*);
const char* ak_strerror(int code);
const char* ak_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AK_H */
