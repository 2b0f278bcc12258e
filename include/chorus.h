/* chorus.h -- C ABI of the B200-native CHORUS-MHD hot path (libchorus_b200.so).
 *
 * The hot path is the per-stage spectral-difference (SD) residual of the compressible MHD equations with
 * GLM divergence cleaning on curved hexahedra, plus the explicit SSPRK(5,3) update, as defined in
 * arxiv 2502.17805 (citations: PAPER.md:<line>, section / equation).  Every step runs in hand-written CUDA
 * kernels for sm_100a; there is no CPU fallback: every entry point fails with CHORUS_ECUDA when no device
 * is usable.  No torch types cross this boundary: plain pointers (HOST or DEVICE as stated) and sizes.
 *
 * Conventions
 *   n = order = solution points per direction; n^3 solution points (Chebyshev-Gauss, Eq. 18),
 *   n+1 flux points per direction (Legendre roots of P_{n-1} plus 0 and 1), three staggered
 *   flux families of n^2 (n+1) points.
 *   Variables (Eq. 2): rho, rho*u, rho*v, rho*w, E, Bx, By, Bz, psi -- 9 fp64 per point.
 *   state / residual layout  [9][n_elem][n^3]            i (xi) fastest, then j (eta), then k (zeta)
 *   gradient layout          [27][n_elem][n^3]           row 3*v+p = d Q_v / d x_p
 *   family-d layout          n^2 (n+1) per element: natural (k,j,i) order with axis d extended to n+1
 *   Faces 0..5 = xi0, xi1, eta0, eta1, zeta0, zeta1; a face point is (a,b) = the two remaining axes in
 *   increasing order.  Orientation code (bit0 swap a<->b, bit1 reverse a, bit2 reverse b, applied in that
 *   order) maps an own face point (a,b) to the coinciding neighbour face point (a',b').
 *
 * Ownership: the caller owns every buffer it passes.  chorus_init copies the mesh; the library owns all
 * device arrays until chorus_free.  One opaque context per mesh; contexts are not thread-safe.  The only
 * process-wide state is the table of 1-D operators in __constant__ memory, indexed by the order: chorus_init writes
 * the entry of its order with values that depend on the order alone, so contexts of any orders coexist.  All work is enqueued on the cudaStream_t given to chorus_init; calls that take or return
 * HOST data synchronise that stream, calls with on_device = 1 are asynchronous on it.
 *
 * Errors: every function returns 0 (CHORUS_OK) or a negative code; chorus_last_error gives a message.
 */
#ifndef CHORUS_H
#define CHORUS_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define CHORUS_OK 0
#define CHORUS_EINVAL (-1) /* bad argument / order / nstages / mesh                     */
#define CHORUS_ENOMEM (-2) /* device or host allocation failed                          */
#define CHORUS_ECUDA (-3)  /* CUDA runtime error (message kept for chorus_last_error)   */
#define CHORUS_ESTATE (-4) /* no state set, or a non-finite wave speed                  */

typedef struct chorus_ctx chorus_ctx; /* opaque, owned by the library */

/* Generic unstructured hexahedral mesh (PAPER.md:70-80 for the cubed-sphere shell; any conforming hex mesh).
 * All pointers are HOST pointers; the arrays are copied by chorus_init. */
typedef struct {
  int64_t n_elem;
  int32_t n_geom;            /* geometry nodes per direction (>= 2); tensor grid, xi fastest             */
  const double* geom_nodes;  /* [n_geom] abscissae in [0,1], first 0, last 1 (where the map was sampled) */
  const double* xyz;         /* [n_elem][3][n_geom^3] physical coordinates of the geometry nodes (Eq. 13) */
  const int32_t* nbr_elem;   /* [n_elem][6] neighbour element, or -1 = inner wall, -2 = outer wall        */
  const uint8_t* nbr_face;   /* [n_elem][6] neighbour's local face 0..5                                   */
  const uint8_t* nbr_orient; /* [n_elem][6] orientation code (see above)                                  */
} chorus_mesh;

/* Physical parameters (Eq. 3-10; walls PAPER.md:190-198; Table 1). */
typedef struct {
  double gamma, R_gas, Cp;   /* Eq. 3, 4, 10                                                              */
  double GM, Omega;          /* g = -GM r_hat / r^2; Omega along z (Eq. 5)                                */
  double nu, kappa, eta;     /* kinematic viscosity (mu = rho nu), thermal and magnetic diffusivity       */
  double kr_scale, kr_c[3];  /* kappa_r = kr_scale (c0 + c1 w + c2 w^2), w = r * kr_wscale */
  double kr_wscale;
  double c_h, a_psi;         /* GLM wave speed and damping rate (Eq. 5, 6)                                */
  double q_bottom, T_top;    /* thermal walls (Eq. 32), used only when the flags say so     */
  int32_t bc_mag_inner, bc_mag_outer; /* 0 perfectly conducting, 1 perfectly radial        */
  uint32_t flags;            /* bit0 diffusion (Eq. 7), bit1 gravity, bit2 Coriolis, bit3 Powell div B sources,
                                bit4 GLM damping, bit5 fixed-T outer wall, bit6 fixed-flux inner wall,
                                bit7 centrifugal (off by default: not in Eq. 5)                           */
} chorus_physics;

/* Build a context: copies the mesh to the device and runs the geometry precompute (free-stream preserving
 * curl-form metrics of the degree-n interpolant of the element map: S^d = |J| grad xi_d at the flux points,
 * |J|, grad xi_d and x at the solution points; Eq. 13-17).
 * order: 2..9.  cuda_stream: a cudaStream_t (NULL = default stream).  *out is NULL on failure. */
int chorus_init(chorus_ctx** out, const chorus_mesh* mesh, int order, const chorus_physics* phys, void* cuda_stream);
void chorus_free(chorus_ctx* ctx);
/* Replace the physical parameters (e.g. C_h once the initial wave speed is known).  The kappa_r profile (kr_scale, kr_c,
 * kr_wscale) is tabulated at the flux points by chorus_init and is fixed for the life of the context: a call that
 * changes any of them returns CHORUS_EINVAL and leaves the context unchanged. */
int chorus_set_physics(chorus_ctx* ctx, const chorus_physics* phys);

/* q: [9][n_elem][n^3] fp64, HOST (on_device = 0) or DEVICE (on_device = 1) pointer. */
int chorus_set_state(chorus_ctx* ctx, const double* q, int on_device);
int chorus_get_state(chorus_ctx* ctx, double* q, int on_device);

/* r = dQ/dt of the current state = -(1/|J|) div_xi F~ + M  (Eq. 16 with Eq. 5-10, 17; procedure PAPER.md:123,
 * face treatment PAPER.md:149: BR1 common solution, averaged viscous flux, Rusanov inviscid flux).
 * Same layout as the state.  The state is not changed. */
int chorus_residual(chorus_ctx* ctx, double* r, int on_device);

/* One time step of size dt.  nstages = 5: SSPRK(5,3) of Ruuth; 3: SSPRK(3,3); 1: forward Euler
 * (test aids).  Each stage is a residual evaluation fused with its Runge-Kutta combination. */
int chorus_step(chorus_ctx* ctx, double dt, int nstages);

/* The same step, one kernel at a time (orders 4..7): chorus_step_begin fixes dt and the scheme and makes sure the face traces
 * of the current state exist; then, for istage = 0 .. nstages-1, chorus_stage_main launches the element kernel of the stage and
 * chorus_stage_face finishes it (the viscous face kernel with diffusion; without diffusion it only completes the bookkeeping).
 * After the last chorus_stage_face the new state is current.  chorus_step(dt, nstages) is exactly this sequence.  Calls out of
 * sequence return CHORUS_ESTATE.  A partition (below) exchanges its halo between these calls. */
int chorus_step_begin(chorus_ctx* ctx, double dt, int nstages);
int chorus_stage_main(chorus_ctx* ctx, int istage);
int chorus_stage_face(chorus_ctx* ctx, int istage);

/* ---- element partitions for multi-GPU runs ----
 * A rank's local mesh lists the elements it OWNS first, then GHOST copies of the off-rank face neighbours of owned elements
 * (connectivity of owned elements refers to local indices; that of ghosts is ignored).  chorus_set_owned(n_owned) makes the
 * context advance elements [0, n_owned) only.  Two kinds of face data of ghosts come from their owners, every stage:
 *   field 0  face traces of the state being evaluated, 9 n^2 doubles per face   -- before chorus_stage_main
 *   field 1  own-side viscous face fluxes, 7 n^2 doubles per face (diffusion)    -- between chorus_stage_main and _face
 * chorus_halo_setup takes the faces to send (owned element, face) and to receive (ghost element, face), HOST arrays that are
 * copied; chorus_halo_pack gathers the send faces of a field into buf [n_send][w n^2] and chorus_halo_unpack scatters
 * buf [n_recv][w n^2] into the ghosts (DEVICE buffers, asynchronous on the context's stream; w = 9 or 7).  How the buffers
 * travel (NCCL all-to-all over NVLink, peer copies) is the caller's business: paper_2502_17805_b200/partition.py.
 * chorus_max_wavespeed and chorus_diagnostics_sums of a partition cover its owned elements; state arrays keep the local
 * layout [9][n_elem][n^3] (ghost slots are ignored on input and meaningless on output). */
int chorus_set_owned(chorus_ctx* ctx, int64_t n_owned);
int chorus_halo_setup(chorus_ctx* ctx, int64_t n_send, const int32_t* send_elem, const uint8_t* send_face, int64_t n_recv,
                      const int32_t* recv_elem, const uint8_t* recv_face);
int chorus_halo_pack(chorus_ctx* ctx, int field, double* buf);
int chorus_halo_unpack(chorus_ctx* ctx, int field, const double* buf);
/* out (HOST, 3 doubles) = int dV, int 1/2 rho U.U dV, int 1/2 B.B dV over the owned elements (the undivided sums of
 * chorus_diagnostics, to be added over the partitions). */
int chorus_diagnostics_sums(chorus_ctx* ctx, double* out);

/* *out (HOST) = max over solution points of |U| + sqrt((gamma p + |B|^2)/rho): the fast magnetosonic speed
 * maximised over direction, for the CFL condition.  Synchronises.  CHORUS_ESTATE if it is not finite. */
int chorus_max_wavespeed(chorus_ctx* ctx, double* out);

/* Volume-averaged diagnostics of the current state: out (HOST, 3 doubles) =
 *   V    = int dV,   KE = (1/V) int 1/2 rho U.U dV  (Eq. 34),   E_B = (1/V) int 1/2 B.B dV  (Eq. 35),
 * with the interpolatory quadrature of the solution points, int f dV = sum_e sum_ijk w_i w_j w_k |J| f (w = Fejer's first rule
 * on the Chebyshev-Gauss points of Eq. 18).  A deterministic two-kernel tree reduction; synchronises.  CHORUS_ESTATE without a state. */
int chorus_diagnostics(chorus_ctx* ctx, double* out);

const char* chorus_last_error(const chorus_ctx* ctx);

/* ---- accessors used by the parity tests and by input generation (not on the hot path) ---- */
/* Any pointer may be NULL.  detJ [n_elem][n^3]; S [n_elem][3 fam][3 comp][n^2(n+1)]; xsol [3][n_elem][n^3];
 * jinv [n_elem][3 d][3 p][n^3] = (grad xi_d)_p.  HOST or DEVICE pointers per on_device. */
int chorus_get_geometry(chorus_ctx* ctx, double* detJ, double* S, double* xsol, double* jinv, int on_device);
/* g [27][n_elem][n^3]: BR1 gradient of the current state at the solution points. */
int chorus_get_gradient(chorus_ctx* ctx, double* g, int on_device);
/* 1-D node sets and operators the library uses (HOST pointers, any may be NULL):
 * xs [n], xf [n+1], Isf [(n+1)][n], Dfs [n][(n+1)]. */
int chorus_get_operators(int order, double* xs, double* xf, double* Isf, double* Dfs);
/* Number of kernel launches this context has enqueued since chorus_init (for bench.py's gpu_launches). */
int64_t chorus_launch_count(const chorus_ctx* ctx);
/* Measurement: with profiling enabled every hot-path launch is bracketed by CUDA events on the context's stream.
 * chorus_profile_read synchronises, returns the accumulated device time (ms) and launch count per kernel class
 * -- index 0 face-trace kernel, 1 viscous face kernel (scalar path: gradient kernel), 2 element kernel (stage_main_kernel;
 * scalar path: residual_kernel) -- and resets them. */
int chorus_profile(chorus_ctx* ctx, int enable);
int chorus_profile_read(chorus_ctx* ctx, double* ms /*[3]*/, int64_t* launches /*[3]*/);

/* Measurement: sustained FP64 issue rate of the current device, the denominator of the "alu" roofline.
 * mode 0: independent DFMA chains on every warp; 1: DMMA.8x8x4 (mma.sync m8n8k4 f64) chains on every warp; 2: half the
 * warps of every SM sub-partition run DFMA and half DMMA at the same time (tells whether the two share one pipe).
 * Runs for at least `seconds` on the default stream, synchronises, *tflops (HOST) = 2 x FMA / time / 1e12 in total;
 * dfma_tflops / dmma_tflops (HOST, may be NULL) = the share of each instruction kind (equal halves in mode 2). */
int chorus_fp64_peak(int mode, double seconds, double* tflops, double* dfma_tflops, double* dmma_tflops);

/* ---- host jobs, pipelined ------------------------------------------------------------------------------------------
 * One job = chorus_set_state(q_in HOST) + chorus_step(dt, nstages) + chorus_get_state(q_out HOST) [+ the CFL wave speed of the
 * result into *ws_out (HOST), if ws_out is not NULL], enqueued WITHOUT synchronising: the host-to-device copy runs on a copy
 * stream of the library, the kernels on the context's stream, the device-to-host copies on a second copy stream, through two
 * staging slots each way (4 x the state's size of device memory, allocated on the first call).  Jobs issued back to back overlap:
 * the H2D of job k + 1 and the D2H of job k - 1 run beside the kernels of job k, so the step rate is max(copy, compute) instead
 * of their sum.  Jobs are independent (each starts from its own q_in) and complete in order.
 *   q_in, q_out, ws_out: HOST; [9][n_elem][n^3], the same, one double.  They are owned by the caller, must stay valid and
 *   untouched until chorus_sync returns, and should be PINNED (cudaHostAlloc / cudaHostRegister): pageable memory works but the
 *   copies then block the calling thread and nothing overlaps.  Results are bit-identical to the three separate calls.
 * chorus_sync waits for everything the context has enqueued, the copy streams included.  Unpartitioned contexts only; errors as
 * chorus_step.  After chorus_sync the context's state is the last job's result. */
int chorus_step_host(chorus_ctx* ctx, const double* q_in, double* q_out, double dt, int nstages, double* ws_out);
int chorus_sync(chorus_ctx* ctx);

/* ---- allocation-free entry point --------------------------------------------------------------------------------
 * The diagnostics of chorus_diagnostics (Eq. 34-35; same quadrature) for callers that cannot call
 * cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid allocation.  It needs no context and
 * calls no cudaMalloc, cudaFree or other allocating routine: the partial sums of its reduction live in a device array of
 * fixed size inside the library (96 KB, held by every GPU that loads the library until the process exits).
 *   order    2..9;  n_elem >= 1;  n_elem * order^3 <= CHORUS_STATIC_DIAG_MAX_POINTS, else CHORUS_EINVAL (nothing is launched)
 *   q        DEVICE, [9][n_elem][order^3] conserved variables in the interface layout (as chorus_get_state gives them)
 *   detJ     DEVICE, [n_elem][order^3]    |J| at the solution points (as chorus_get_geometry gives it)
 *   out      DEVICE, 3 doubles: V = int dV, KE (Eq. 34), E_B (Eq. 35)
 *   stream   a cudaStream_t (NULL = default stream); two kernels are enqueued on it, nothing synchronises
 * All pointers stay owned by the caller.  Uses the CURRENT device; its first call on a device looks up the array's address
 * (cudaGetSymbolAddress), so make one call per device outside graph capture.  Every call on a device shares the one scratch
 * array, which keeps the last call's contents (each call overwrites every entry it reads: nothing has to be cleared): calls
 * that OVERLAP on the GPU -- different streams, or concurrent graph launches -- race and must be serialised by the caller.
 * The summation tree is fixed by the size alone (8192 points per block), so results are bit-identical from call to call; they
 * differ from chorus_diagnostics at round-off (another tree).  On failure chorus_static_last_error() has the message
 * (per calling thread; valid until that thread's next call). */
#define CHORUS_STATIC_DIAG_MAX_POINTS 33554432 /* 2^25 solution points: 4096 blocks x 8192 points, 96 KB of partial sums */
int chorus_diagnostics_static(int order, int64_t n_elem, const double* q, const double* detJ, double* out, void* cuda_stream);
const char* chorus_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
