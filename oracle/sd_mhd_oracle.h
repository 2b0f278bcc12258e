/* sd_mhd_oracle.h -- C interface of the CPU ORACLE (TEST INFRASTRUCTURE, not product code).
 *
 * A plain, slow, literal implementation of the spectral-difference MHD+GLM residual and the
 * SSPRK(5,3) step of arxiv 2502.17805 (CHORUS-MHD), written from /root/reference/PAPER.md.
 * It shares NO code with the CUDA library (include/chorus.h, paper_2502_17805_b200/csrc).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.  All pointers are HOST pointers; all arrays are fp64 on the interface.
 *
 * prec = 0: arithmetic in double.  prec = 1: arithmetic in long double (the "truth" run used
 * to measure the fp64 round-off floor, pin P16); I/O is still double.
 *
 * Layouts (n = order = solution points per direction):
 *   state / residual   [9][E][n^3]          i (xi) fastest; variables rho, rho*u,v,w, E, Bx,By,Bz, psi (Eq. 2)
 *   gradient           [27][E][n^3]         row 3*v+p = d Q_v / d x_p
 *   family-d arrays    n^2 (n+1) per element, natural (k,j,i) order with the d axis extended to n+1 entries
 *   face arrays        [n^2], index b*n+a with (a,b) = the two remaining axes in increasing order
 */
#ifndef SD_MHD_ORACLE_H
#define SD_MHD_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_ctx oracle_ctx;

typedef struct {
  int64_t n_elem;
  int32_t n_geom;            /* geometry nodes per direction (>=2), tensor grid, xi fastest          */
  const double* geom_nodes;  /* [n_geom] abscissae in [0,1], first = 0, last = 1                     */
  const double* xyz;         /* [n_elem][3][n_geom^3]                                                */
  const int32_t* nbr_elem;   /* [n_elem][6] neighbour element, -1 inner wall, -2 outer wall          */
  const uint8_t* nbr_face;   /* [n_elem][6] neighbour's local face 0..5 = xi0,xi1,eta0,eta1,zeta0,zeta1 */
  const uint8_t* nbr_orient; /* [n_elem][6] bit0 swap (a,b), bit1 reverse a, bit2 reverse b          */
} oracle_mesh;

typedef struct {
  double gamma, R_gas, Cp;
  double GM, Omega;
  double nu, kappa, eta;
  double kr_scale, kr_c[3], kr_wscale;
  double c_h, a_psi;
  double q_bottom, T_top;
  int32_t bc_mag_inner, bc_mag_outer;   /* 0 perfectly conducting, 1 perfectly radial */
  uint32_t flags;                       /* bit0 diffusion, 1 gravity, 2 coriolis, 3 powell, 4 glm damping,
                                           5 fixed-T outer wall, 6 fixed-flux inner wall, 7 centrifugal */
} oracle_physics;

/* ---- whole-mesh solver ---- */
oracle_ctx* oracle_init(const oracle_mesh* mesh, int order, const oracle_physics* phys, int prec);
void oracle_free(oracle_ctx*);
int  oracle_set_physics(oracle_ctx*, const oracle_physics* phys);
int  oracle_set_state(oracle_ctx*, const double* q);
int  oracle_get_state(oracle_ctx*, double* q);
/* r = dQ/dt (Eq. 16); a (may be NULL) = magnitude residual: the same sums with the terms of every flux
   (interior, the two central halves and the two dissipation halves of the Rusanov flux, viscous, wall) and of the
   sources replaced by their moduli -- the forward-error scale of reading G24 */
int  oracle_residual(oracle_ctx*, double* r, double* a);
int  oracle_step(oracle_ctx*, double dt, int nstages);   /* 5: SSPRK(5,3); 3: SSPRK(3,3); 1: Euler */
int  oracle_max_wavespeed(oracle_ctx*, double* out);
int  oracle_get_gradient(oracle_ctx*, double* g);        /* BR1 gradient of the current state */
/* out[3] = V, KE, E_B of the current state (Eq. 34-35) by the solution-point quadrature */
int  oracle_diagnostics(oracle_ctx*, double* out);
/* w [n]: interpolatory quadrature weights on the solution points of [0,1], w_i = int h_i (Eq. 19) */
int  oracle_quadrature_weights(int order, double* w);
/* any pointer may be NULL. detJ [E][n^3]; S [E][3 fam][3 comp][n^2(n+1)]; xsol [3][E][n^3];
   jinv [E][3 d][3 p][n^3] = (grad xi_d)_p */
int  oracle_get_geometry(oracle_ctx*, double* detJ, double* S, double* xsol, double* jinv);

/* ---- 1-D building blocks (pins P1, P2, P13) ---- */
int  oracle_nodes(int order, double* xs /*[n]*/, double* xf /*[n+1]*/);
/* Isf [(n+1)][n], Dfs [n][(n+1)], Efs [n][(n+1)], Dff [(n+1)][(n+1)]  (row-major); any may be NULL */
int  oracle_operators(int order, double* Isf, double* Dfs, double* Efs, double* Dff);
/* alpha [5][5], beta [5][5] of the Shu-Osher form: u(i) = sum_k alpha[i-1][k] u(k) + dt beta[i-1][k] F(u(k)) */
int  oracle_rk_tableau(int nstages, double* alpha, double* beta);

/* ---- pointwise physics (pins P5, P6, P7, P15) ---- */
void oracle_flux_inviscid(const oracle_physics*, const double* Q, const double* S, double* F);
void oracle_flux_viscous(const oracle_physics*, const double* Q, const double* G /*[27]*/, const double* S,
                         double kr, double* F);
void oracle_flux_rusanov(const oracle_physics*, const double* Qin, const double* Qout, const double* nhat, double* F);
double oracle_fast_speed(const oracle_physics*, const double* Q, const double* nhat);
double oracle_wavespeed(const oracle_physics*, const double* Q);
/* wall = -1 inner / -2 outer */
void oracle_wall_state(const oracle_physics*, int wall, const double* Q, const double* nhat, double* Qb);
void oracle_flux_wall_inviscid(const oracle_physics*, const double* Qb, const double* nhat, double* F);
/* wall viscous flux along nhat from (Q_b, grad Q_in) with the wall conditions applied to the wall gradients:
   rw = distance of the wall point from the origin (<= 0: plane wall) */
void oracle_flux_wall_viscous(const oracle_physics*, int wall, const double* Qb, const double* G, const double* nhat,
                              double rw, double kr, double* F);
/* the conditioned Jacobian of B at a wall point: dB, dBc [3][3] row-major d_j B_i; bc 0 perfectly conducting, 1 perfectly
   radial; Bb the wall state's field; er the wall's radial unit vector; rw as above */
void oracle_wall_condition_gradB(int bc, const double* dB, const double* Bb, const double* er, double rw, double* dBc);
void oracle_source(const oracle_physics*, const double* Q, const double* G, const double* x, double* M, double* Mabs);

#ifdef __cplusplus
}
#endif
#endif
