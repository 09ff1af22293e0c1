/* oracle/oracle.h — CPU ORACLE (TEST INFRASTRUCTURE ONLY).
 *
 * Plain, slow, fp64 restatement of the Valencia GRMHD right-hand-side stage of
 * arXiv:2409.10384 (PAPER.md, cited as P:line).  It exists to check the CUDA
 * library; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` leg may build, load or call it.  No file, header, table or helper is
 * shared with paper_2409_10384_b200/csrc (the product); the product's point operators restate
 * the same canonical expression trees, so agreement of the two to the last bit
 * certifies the product's plumbing, while the physics is certified by the pins below.
 *
 * Steps follow DESIGN.md §3 (O0..O9) which restates, in the paper's notation,
 *   Eq. 6 prim->cons, Eq. 7 b^mu, Eq. 8 fluxes,
 *   Eq. 9 sources, P:133 reconstruction/Riemann/CT choices,
 *   P:137-139 atmosphere, P:141-157 FOFC(+DMP, Eq. 12), P:161 con2prim.
 * No blocking, fusion or reordering: loops over blocks, cells, faces, edges.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): see DESIGN.md §5.  Round 2 added
 * tests/test_oracle_pins_r2.py: WENO-Z weights against the literal formula in exact
 * rationals, the CT upwind sense and weight locations, the face-state floor, and
 * lambda+- with B != 0 against the numerical flux Jacobian - each seen to fail on
 * one-line mutations of this code.  Policy choices the paper leaves open (floor
 * order R5, M_max R6, "requires a floor" R8, DMP variables R13, root-finder path R2)
 * are "parity unpinned" beyond oracle==GPU and are listed there.
 *
 * Data layout (the library boundary's, restated): a MeshBlock has n^3 interior
 * cells, ng=4 ghosts, nt=n+8 stored cells per direction; i fastest.
 *   cell field   [nmb][nt][nt][nt]
 *   x-face field [nmb][nt][nt][px]      px = nt+4 (nt+1 used)
 *   y-face field [nmb][nt][nt+1][nt]
 *   z-face field [nmb][nt+1][nt][nt]
 *   E_x          [nmb][nt+1][nt+1][nt]
 *   E_y          [nmb][nt+1][nt][px]
 *   E_z          [nmb][nt][nt+1][px]
 * Face i of direction x lies between cells i-1 and i.
 */
#ifndef GRMHD_ORACLE_H
#define GRMHD_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int nmb, n, ng;
  double gamma_ad;               /* ideal-gas Gamma                          */
  double rho_atm, T_atm, f_thr;
  double mag_max;                /* M_max of P:139 (+inf disables)           */
  int recon;                     /* 0 donor cell, 1 PPM4, 2 WENO-Z, 3 PLM, 4 PPMX */
  int riemann;                   /* 0 LLF, 1 HLLE                    */
  int fofc, fofc_riemann;
  double dmp_M;                  /* Eq. 12; <=0 off                          */
  int c2p_max_iter;
  double c2p_tol;
  /* equation of state (oracle/eos.h): 0 ideal gas with gamma_ad; 1 piecewise-polytropic hybrid
   * (reading R29) with pp_nseg (1..4) segments of exponent pp_gamma[i], the
   * first with constant pp_K0, breakpoints pp_rho[0] < pp_rho[1] < ..., thermal gamma_th. */
  int eos, pp_nseg;
  double pp_K0, pp_gamma[4], pp_rho[3], gamma_th;
} orc_params;

/* status / flag bits */
enum { ORC_DFLOOR = 1, ORC_TAUFLOOR = 2, ORC_MAGCAP = 4, ORC_RHOFLOOR = 8,
       ORC_TFLOOR = 16, ORC_FAIL = 32, ORC_DMP = 64 };

/* ---- point-level steps (unit-test surface) ------------------------------ */

/* O0: det, sqrt(det), inverse of the 3-metric g = {xx,xy,xz,yy,yz,zz}. */
void orc_metric_inverse(const double g[6], double* det, double* sdet, double ginv[6]);

/* O2 (Eq. 6): prim = {rho,ux,uy,uz,P} with u^i = W v^i, B = undensitised B^i;
 * cons = {D,Sx,Sy,Sz,tau}, undensitised. */
void orc_prim2cons(double gamma_ad, const double g[6], const double prim[5],
                   const double B[3], double cons[5]);

/* Same with the equation of state of p (ideal gas or hybrid). */
void orc_prim2cons_eos(const orc_params* p, const double g[6], const double prim[5],
                       const double B[3], double cons[5]);

/* O1 for the EOS of p: out = {P(rho,eps), h-1 and c_s^2 at (rho, P(rho,eps)), P_c, eps_c}
 * (P_c = eps_c = 0 for the ideal gas). */
void orc_eos_point(const orc_params* p, double rho, double eps, double out[5]);

/* O3: Ut = densitised {D,S_i,tau} (rewritten if floored and !check_only),
 * Btcc = densitised cell-centred B, W out = {rho,ux,uy,uz,P}.
 * Returns the status byte; *iters = master-function evaluations used. */
int orc_con2prim_cell(const orc_params* p, const double g[6], double Ut[5],
                      const double Btcc[3], double W[5], int check_only, int* iters);

/* O3 master function f(mu) exposed for the zero-at-true-root pin.
 * in: q, r2, bs2 (= B^2/D), rb2 (= (r_i B^i)^2 / D). */
double orc_c2p_master(double gamma_ad, double q, double r2, double bs2, double rb2, double mu);
/* the same for the EOS of p; D = undensitised conserved density (rho^ = D / W^). */
double orc_c2p_master_eos(const orc_params* p, double D, double q, double r2, double bs2,
                          double rb2, double mu);

/* O4: q[5] = cells i-2..i+2; qm = value at the left face of cell i, qp at the right. */
void orc_reconstruct(int kind, const double q[5], double* qm, double* qp);

/* O5+O6: one face of direction dir (0,1,2).  gL/gR = cell-centred
 * {alpha,betax,betay,betaz,gxx,gxy,gxz,gyy,gyz,gzz} of the lower/upper cell.
 * WL/WR = {rho,ux,uy,uz,P,Bt1,Bt2} (B densitised, t1,t2 cyclic after dir),
 * Bfd = densitised face-normal B.  apply_floor: face-state floor of P:139.
 * F[7] = {D,Sx,Sy,Sz,tau,Bt1,Bt2} fluxes.  lam (may be NULL) = {lm_L,lp_L,lm_R,lp_R}. */
void orc_face_flux(const orc_params* p, int dir, int riemann, const double gL[10],
                   const double gR[10], const double WL[7], const double WR[7],
                   double Bfd, int apply_floor, double F[7], double lam[4]);

/* ---- block-level steps --------------------------------------------------- */

/* O3 over all stored cells. U[5], Bf[3], g[6] field pointers; W[8] out
 * (rho,ux,uy,uz,P,Bccx,Bccy,Bccz); status may be NULL. */
void orc_con2prim(const orc_params* p, double* const U[5], const double* const Bf[3],
                  const double* const g[6], double* const W[8], unsigned char* status,
                  int nthreads);

/* Whole stage O3..O9.  adm[16] = gxx,gxy,gxz,gyy,gyz,gzz,alp,betx,bety,betz,
 * Kxx,Kxy,Kxz,Kyy,Kyz,Kzz.  dx[nmb][3].  out_dU[5] (interior cells written),
 * out_E[3] (edges of interior cells written), flag (test cells written; may be NULL),
 * flux_out[21] may be NULL; else x,y,z face-flux fields (7 each, face layouts above)
 * receive the post-FOFC fluxes on the computed range.  face_refluxed[3] may be
 * NULL; else byte per face (face layouts) = 1 where FOFC redid the face. */
void orc_rhs(const orc_params* p, const double* dx, double* const U[5],
             const double* const Bf[3], const double* const adm[16], double* const W[8],
             int w_is_valid, double dt_fofc, double* const out_dU[5],
             double* const out_E[3], unsigned char* flag, unsigned char* c2p_status,
             double* const flux_out[21], unsigned char* const face_refluxed[3],
             int nthreads);

/* Matter terms for a spacetime solver: out[10] = E = tau + D, S_i, S_ij = T_ij,
 * undensitised, at every stored cell, from the primitives W and gamma_ij. */
void orc_matter_sources(const orc_params* p, const double* const W[8], const double* const g6[6],
                        double* const out[10]);

/* Same stage with the FOFC estimate of a later Runge-Kutta stage (R9):
 * U* = fa * U0 + fb * (U - dt_fofc div F) when U0 != NULL. */
void orc_rhs_blend(const orc_params* p, const double* dx, double* const U[5],
                   const double* const Bf[3], const double* const adm[16], double* const W[8],
                   int w_is_valid, double dt_fofc, const double* const U0[5], double fa, double fb,
                   double* const out_dU[5], double* const out_E[3], unsigned char* flag,
                   unsigned char* c2p_status, int nthreads);

/* ---- stage driver ("RK2 / RK3", method of lines) --------------------
 * Each MeshBlock is its own domain: ghosts are filled from the block itself.
 * bc[d]: 0 periodic, 1 outflow (zero-gradient copy), per direction. */
void orc_fill_ghosts(const orc_params* p, const int bc[3], double* const U[5], double* const Bf[3]);

/* One stage register update on the interior cells and on the faces of interior cells:
 *   U  <- a U0 + b (U + dt dU),   B~f <- a B0 + b (B~f + dt (-curl E))      (dx[nmb][3]) */
void orc_stage_update(const orc_params* p, const double* dx, double a, double b, double dt,
                      const double* const U0[5], const double* const B0[3], double* const U[5],
                      double* const Bf[3], const double* const dU[5], const double* const E[3]);

/* nsteps steps of SSP-RK1/2/3 (integrator = 1,2,3) with a fixed dt: per stage fill ghosts,
 * orc_rhs_blend, orc_stage_update.  The step-start register is taken after the first stage's
 * con2prim (floored state).  W (8) is scratch/out.  flag_or (may be NULL): OR of all FOFC flags. */
void orc_advance(const orc_params* p, const double* dx, int integrator, int nsteps, double dt,
                 const int bc[3], double* const U[5], double* const Bf[3],
                 const double* const adm[16], double* const W[8], unsigned char* flag_or,
                 int nthreads);

/* Same-level ghost exchange between MeshBlocks.  nbr[nmb][27]: block at offset
 * (oz+1)*9+(oy+1)*3+(ox+1), -1 = none; sides without a face neighbour get bc[d]. */
void orc_exchange_ghosts(const orc_params* p, const int* nbr, const int bc[3], double* const U[5],
                         double* const Bf[3]);
/* ... with a caller hook run on the host before every ghost fill (multi-rank drivers refresh their
 * mirror blocks there); returns the hook's first non-zero value, else 0. */
int orc_advance_hooked(const orc_params* p, const double* dx, int integrator, int nsteps, double dt,
                       const int bc[3], const int* nbr, double* const U[5], double* const Bf[3],
                       const double* const adm[16], double* const W[8], unsigned char* flag_or,
                       int nthreads, int (*refresh)(void*), void* user);
void orc_advance_nbr(const orc_params* p, const double* dx, int integrator, int nsteps, double dt,
                     const int bc[3], const int* nbr, double* const U[5], double* const Bf[3],
                     const double* const adm[16], double* const W[8], unsigned char* flag_or,
                     int nthreads);

#ifdef __cplusplus
}
#endif
#endif
