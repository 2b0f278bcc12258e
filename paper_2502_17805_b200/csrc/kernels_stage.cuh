// kernels_stage.cuh -- the production pipeline of one residual evaluation / Runge-Kutta stage (orders 4..8).
//
//   stage_main_kernel  per element: A2 face gather + BR1 common solution, A3 gradient (computed ONCE per stage),
//                      A6 Rusanov / wall inviscid face fluxes, A1 + A4 + A5 + A7 as register-resident FP64 tensor-core
//                      chains, A8 sources, A9 Runge-Kutta combination.  With diffusion it also emits the element's
//                      own viscous flux at its face points (Vf) and leaves out the common VISCOUS face flux, which
//                      needs the neighbours' Vf of the same stage; everything else of the residual is final.
//   stage_face_kernel  (diffusion only) per element: adds the divergence of the common viscous face flux
//                      1/2 (own + neighbour) ("a similar procedure is used for the viscous flux"),
//                      finishes the state / residual, and emits the face traces of the new state (A1 restricted to the
//                      faces) for the next stage.  A light, purely HBM-bound pass.
//   Without diffusion the main kernel is the whole stage and emits the next traces itself.
//
// Mapping of the main kernel (same mathematics as kernels_residual.cuh; Eq. 19-24): one warp owns 8 lines
// of one direction.  With mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4)
//   Q^, grad Q^ [line][col] = A[line][l] * B[l][col]     A = solution values of the line (shared memory),
//                                                        B = h_l(X_f,m(col))  (Eq. 19 at the flux points)
// land in the C fragment: thread (r = lane/4, c = lane%4) holds columns 2c, 2c+1 of line r, i.e. every interpolated
// quantity of two flux points -- what the pointwise fluxes (Eq. 6-10) need, with no shared-memory round trip.  The
// 27 gradient components are never held together: each variable's gradient is folded into a 14-number running state
// of the viscous flux (VStream) as soon as its three DMMA results arrive.  The fluxes F~ stay in registers and, the C
// layout of m8n8k4 being the A layout of two k-steps once the contraction index is permuted, feed the derivative
//   dF~/dxi [line][l] = F~[line][col] * B'[col][l]        B' = l'_{m(col)}(X_s,l)  (Eq. 20, 22-24)
// directly.  Columns: interior flux points, then the two face points, then padding.
#pragma once
#include "kernels_residual.cuh"

namespace chorus {

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// orders served by this pipeline
__host__ __device__ constexpr bool kMmaOrder(int n) { return n >= 4 && n <= 8; }
// orders that run one CTA per SM with two chain warpgroups (their tiles leave no room for a second CTA)
__host__ __device__ constexpr bool kWideOrder(int n) { return n >= 6 && n <= 8; }
// n = 8: the n + 1 = 9 flux points of a line do not fit the 8 columns of a DMMA tile.  The tile holds the 7 interior flux points
// and the face point m = n; the face point m = 0 enters the flux derivative as a third k-step whose A operand is the common face
// flux in shared memory, and the own-side viscous flux of the three m = 0 faces (Vf) is made by the helper warps.  S^d is read
// from global memory (L2) instead of a shared-memory tile: 212 KB of tiles in all.
__host__ __device__ constexpr bool kFaceOutOrder(int n) { return n == 8; }
// orders whose chains read S^d at the flux points from global memory (L2; prefetched an element ahead) instead of a shared-memory tile
__host__ __device__ constexpr bool kSglobalOrder(int n) { return n == 8; }
// orders whose shared-memory S^d tile holds the INTERIOR flux points only (Geo::Sint; the face points go through nfc): with two
// gradient buffers the full tile no longer fits twice
__host__ __device__ constexpr bool kSintOrder(int n) { return n == 6; }
// ... and, of these, the ones with room for a SECOND set of input tiles (state, own and neighbour traces, S^d): the next
// element's inputs stream in while the current element's chains run, so the chain warps never wait for them
__host__ __device__ constexpr bool kPrefetchOrder(int n) { return n == 6; }

template <int N>
struct Mma {
  static_assert(kMmaOrder(N), "DMMA chain kernel: orders 4..8");
  using I = Ix<N>;
  // Lines of a direction are handed to warps in groups of 8 (the M dimension of the DMMA).  n^2 = 8 FG + LO: the FG full
  // groups of a direction are "directional tasks" (compile-time direction); the LO left-over lines of the three directions
  // are chosen so that no two of them meet in a solution point and are packed together into "tail tasks" whose rows carry
  // their own direction at run time.  At most 4 warps per CTA: warp w runs on SM sub-partition w % 4, so a fifth warp
  // would double the load of one FP64 pipe (measured: 5 warps of DMMA take twice as long as 4).
  static constexpr int FG = I::n2 / 8, LO = I::n2 % 8;
  // n = 7 leaves room for only one CTA per SM (173 KB of tiles): it gets two chain warpgroups, two chain warps per sub-partition
  static constexpr int kChainWG = kWideOrder(N) ? 2 : 1;
  static constexpr int kWarps = FG < 4 * kChainWG ? FG : 4 * kChainWG;
  static constexpr int kTPD = (FG + kWarps - 1) / kWarps;     // directional tasks per warp and direction
  static constexpr int kTail = (3 * LO + 7) / 8;               // tail tasks per element
  static_assert(kTail <= kWarps, "tail tasks: one round");
  // Orders whose tiles leave room for one divergence accumulator PER DIRECTION (n <= 5 beside a second CTA; n = 7 alone on its
  // SM, 222 KB): no two tasks ever touch the same word, so all 3 FG + kTail tasks of an element are dealt to the chain warps
  // with no barrier in between (n = 4: 6 tasks on 4 warps, n = 5: 10, n = 7: 19 on 8 warps) instead of FG tasks per
  // barrier-separated direction round (at n = 7 that left two of the eight chain warps without work in every round).
  static constexpr bool kFree = N <= 7;                      // n = 8: one accumulator, barrier-separated direction rounds of 8 tasks
  static constexpr int kFreeWarps = 4 * kChainWG;             // kFree: chain warps that take tasks
  static constexpr int kTasks = 3 * FG + kTail;              // kFree: tasks per element ...
  static constexpr int kTPW = (kTasks + kFreeWarps - 1) / kFreeWarps;   // ... and per chain warp
  // left-over lines (a,b): d = 0: b = 0, a < LO;  d = 1: b = 1, a < LO;  d = 2: a, b >= LO, the first LO of them
  __host__ __device__ static constexpr bool is_lo(int d, int ab) {
    const int a = ab % N, b = ab / N;
    return d == 0 ? (b == 0 && a < LO) : d == 1 ? (b == 1 && a < LO) : (a >= LO && b >= LO && (b - LO) * (N - LO) + (a - LO) < LO);
  }
  // slot 0 .. 8 FG - 1: the lines that are not left over, in increasing order; slot 8 FG + i: the i-th left-over line.
  // n = 6: the full groups are ordered so that the four lines of a half-warp (rows r = 0..3, r = 4..7) start in shared-memory
  // banks that the 4 k-offsets of an A-operand load tile without overlap (a 64-bit load serves 16 lanes per wavefront over 16
  // double-wide banks): direction 0 (line pitch 6, k-offsets 0..3): bases 6 ab = {0,4,8,12} or {2,6,10,14} mod 16, i.e. four
  // even or four odd ab; direction 1 (bases 36 b + a, k-offsets {0,6,12,18}): bases {k, k+1, k+8, k+9} mod 16, i.e. lines (a,b),
  // (a+1,b), (a,b+2), (a+1,b+2); direction 2 (bases ab, k-offsets {0,4,8,12}) is conflict-free as it stands.
  __host__ __device__ static constexpr int line_of(int d, int slot) {
    if (N == 6 && slot < 8 * FG) {
      if (d == 0) {
        const int g = slot / 8, r = slot % 8;
        return 4 + 8 * g + (r < 4 ? 2 * r : 2 * (r - 4) + 1);
      }
      if (d == 1) {
        constexpr int t[32] = {0, 1, 12, 13, 2, 3, 14, 15, 4, 5, 16, 17, 10, 11, 22, 23, 18, 19, 30, 31, 20, 21, 32, 33, 24, 25, 34, 35, 26, 27, 28, 29};
        return t[slot];
      }
    }
    int cnt = 0, lo = 0;
    for (int ab = 0; ab < I::n2; ++ab) {
      if (is_lo(d, ab)) {
        if (slot == 8 * FG + lo) return ab;
        ++lo;
      } else {
        if (slot == cnt) return ab;
        ++cnt;
      }
    }
    return 0;
  }
  // column j of the 8-wide tile -> flux point index m, or -1 (padding).
  // interior points first; the two face points share the SECOND column of their thread pairs so that one divergent
  // pass serves both (cols 2c+1 of the last two thread columns that hold anything).
  __device__ __forceinline__ static int col_m(int j) {
    // 4 bits per column, value m + 1 (0 = padding).  N = 4: {1,2,3,0,-,4,-,-}; 5: {1,2,3,4,-,0,-,5}; 6: {1,2,3,4,5,0,-,6};
    // 7: {1,2,3,4,5,0,6,7}; 8: {1,2,3,4,5,6,7,8} (the face point m = 0 is not in the tile: kFaceOutOrder)
    constexpr uint32_t tbl = N == 4 ? 0x00501432u : N == 5 ? 0x60105432u : N == 6 ? 0x70165432u : N == 7 ? 0x87165432u : 0x98765432u;
    return (int)((tbl >> (4 * j)) & 15u) - 1;
  }
};

// What one stage reads and writes besides the geometry (all element-major unless stated).
struct StageIO {
  const double* Qe;      // state being evaluated                                   [E][9][n3]
  const double* Qf;      // its face traces                                         [E][6][9][n2]
  double* Vf;            // own-side viscous face fluxes (diffusion)                [E][6][7][n2]
  double* Part;          // diffusion: the main kernel's output (everything but the common viscous face flux), finished by
                         // the face kernel.  Step mode: the new-state buffer itself; residual mode: a scratch buffer.
  double* Rout;          // residual in the INTERFACE layout [9][E][n3], or nullptr (step mode)
  double* Qout;          // new state (step mode), or nullptr:  Qout = cq*Qe + c0*A0 + c1*A1 + bdt * R
  double* QfOut;         // face traces of Qout (step mode)
  const double* A0;      // stage registers other than Qe itself (SSPRK(5,3) needs at most two); nullptr contributes nothing
  const double* A1;
  double cq, c0, c1, bdt;
  unsigned* sm_arrivals; // [number of SMs] arrival counters (never reset: only the parity is used)
};

struct Geo {
  const double* Sfl;     // [E][3 fam][3 comp][nf]
  const double* Sint;    // [E][3 fam][3 comp][n2 (n-1)]  interior flux points only (kSintOrder), or nullptr
  const double* detJ;    // [E][n3]
  const double* jinv;    // [E][3 d][3 p][n3]
  const double* xsol;    // [E][3][n3]
  const double* krfl;    // [E][3 fam][nf] or nullptr
  const double* nfc;     // [E][6][4][n2]  outward unit normal (3) and sigma |S| at the face points
  const int32_t* nbr_elem;
  const uint8_t* nbr_face;
  const uint8_t* nbr_orient;
};

// Face traces of the element-resident state sQ [9][n3] -> Qf_e [6][9][n2]  (A1 restricted to the faces; Eq. 19, 21)
template <int N>
__device__ __forceinline__ void emit_traces(const double* sQ, double* __restrict__ Qf_e, int tid, int nthreads) {
  using I = Ix<N>;
  const OpsC& op = c_ops[N];
  for (int t = tid; t < 3 * 9 * I::n2; t += nthreads) {
    const int ab = t % I::n2, v = (t / I::n2) % 9, d = t / (9 * I::n2);
    const double* q = sQ + v * I::n3 + I::sbase(d, ab);
    const int st = I::stride(d);
    double lo = 0.0, hi = 0.0;
#pragma unroll
    for (int l = 0; l < N; ++l) {
      const double x = q[l * st];
      lo += op.Isf[l] * x;
      hi += op.Isf[N * N + l] * x;
    }
    Qf_e[((2 * d) * 9 + v) * I::n2 + ab] = lo;
    Qf_e[((2 * d + 1) * 9 + v) * I::n2 + ab] = hi;
  }
}

// Running state of the viscous flux of one flux point while the gradients of the nine conserved variables stream by
// (Eq. 7-10 contracted with an area vector S; chain rule of DESIGN.md O9).  14 numbers instead of 27.
struct VStream {
  double gr0, gr1, gr2;    // grad rho
  double mS0, mS1, mS2;    // S . grad m_i
  double W0, W1, W2;       // W_i = sum_j S_j d_i m_j
  double divm;             // sum_i d_i m_i
  double acc;              // S.grad E - sum_i B_i S.grad B_i - psi S.grad psi
  double J0, J1, J2;       // curl B
};

// fold the gradient (g0,g1,g2) of conserved variable V
template <int V>
__device__ __forceinline__ void vs_fold(VStream& s, const PrimD& p, double Sx, double Sy, double Sz, double g0, double g1, double g2) {
  const double gS = Sx * g0 + Sy * g1 + Sz * g2;
  if (V == 0) { s.gr0 = g0; s.gr1 = g1; s.gr2 = g2; }
  if (V == 1) { s.mS0 = gS; s.W0 = Sx * g0; s.W1 = Sx * g1; s.W2 = Sx * g2; s.divm = g0; }
  if (V == 2) { s.mS1 = gS; s.W0 += Sy * g0; s.W1 += Sy * g1; s.W2 += Sy * g2; s.divm += g1; }
  if (V == 3) { s.mS2 = gS; s.W0 += Sz * g0; s.W1 += Sz * g1; s.W2 += Sz * g2; s.divm += g2; }
  if (V == 4) s.acc = gS;
  if (V == 5) { s.acc -= p.Bx * gS; s.J1 = g2; s.J2 = -g1; }
  if (V == 6) { s.acc -= p.By * gS; s.J0 = -g2; s.J2 += g0; }
  if (V == 7) { s.acc -= p.Bz * gS; s.J0 += g1; s.J1 -= g0; }
  if (V == 8) s.acc -= p.psi * gS;
}

// tauS = tau.S, qS = q.S from the running state
__device__ __forceinline__ void vs_finish(const PhysD& ph, const VStream& s, const PrimD& p, double Sx, double Sy, double Sz, double kr,
                                          double& t0, double& t1, double& t2, double& qS) {
  const double ir = p.ir;
  const double grS = Sx * s.gr0 + Sy * s.gr1 + Sz * s.gr2;
  const double uS = p.u * Sx + p.v * Sy + p.w * Sz;
  const double divu = (s.divm - (p.u * s.gr0 + p.v * s.gr1 + p.w * s.gr2)) * ir;
  const double lam = -(2.0 / 3.0) * (p.rho * ph.nu) * divu;                        // Stokes; mu = rho nu (G11)
  const double mi = ph.nu;                                                         // mu / rho
  t0 = mi * ((s.mS0 - p.u * grS) + (s.W0 - uS * s.gr0)) + lam * Sx;                // Eq. 8 contracted with S
  t1 = mi * ((s.mS1 - p.v * grS) + (s.W1 - uS * s.gr1)) + lam * Sy;
  t2 = mi * ((s.mS2 - p.w * grS) + (s.W2 - uS * s.gr2)) + lam * Sz;
  const double u2 = p.u * p.u + p.v * p.v + p.w * p.w;
  const double dpS = ph.gm1 * (s.acc - (p.u * s.mS0 + p.v * s.mS1 + p.w * s.mS2) + 0.5 * u2 * grS);
  const double pr = p.p * ir;                                                      // p / rho = R T
  const double Tt = pr * ph.iR;
  const double dTS = (dpS - pr * grS) * ir * ph.iR;
  const double dSS = ph.Cp * (dpS * ph.igamma * (1.0 / p.p) - grS * ir);           // gradient of Eq. 10
  qS = -ph.kappa * p.rho * Tt * dSS - kr * p.rho * ph.Cp * dTS;                    // Eq. 9
}

// interior / interior-face viscous flux rows 1..7 along S
__device__ __forceinline__ void vs_flux(const PhysD& ph, const VStream& s, const PrimD& p, double Sx, double Sy, double Sz, double kr,
                                        double* Fv) {
  double t0, t1, t2, qS;
  vs_finish(ph, s, p, Sx, Sy, Sz, kr, t0, t1, t2, qS);
  const double BxJ0 = p.By * s.J2 - p.Bz * s.J1, BxJ1 = p.Bz * s.J0 - p.Bx * s.J2, BxJ2 = p.Bx * s.J1 - p.By * s.J0;
  Fv[0] = t0; Fv[1] = t1; Fv[2] = t2;
  Fv[3] = (p.u * t0 + p.v * t1 + p.w * t2) - qS + ph.eta * (BxJ0 * Sx + BxJ1 * Sy + BxJ2 * Sz);
  Fv[4] = -ph.eta * (Sy * s.J2 - Sz * s.J1);                                       // eta S_j (d_j B_i - d_i B_j) = -eta (S x J)_i
  Fv[5] = -ph.eta * (Sz * s.J0 - Sx * s.J2);
  Fv[6] = -ph.eta * (Sx * s.J1 - Sy * s.J0);
}

// wall viscous flux along the outward unit normal n from (Q_b, grad Q_in): PAPER.md:190-198, O12
__device__ __forceinline__ void vs_flux_wall(const PhysD& ph, int wall, const VStream& s, const PrimD& pb, double nx, double ny, double nz,
                                             double kr, double* Fv) {
  double t0, t1, t2, qn;
  vs_finish(ph, s, pb, nx, ny, nz, kr, t0, t1, t2, qn);
  const int bc = (wall == -1) ? ph.bc_inner : ph.bc_outer;
  const double tn = t0 * nx + t1 * ny + t2 * nz;                                   // stress-free: normal traction only
  Fv[0] = tn * nx; Fv[1] = tn * ny; Fv[2] = tn * nz;
  if (wall == -1 && (ph.flags & kFlagFixedFluxInner)) qn = -ph.q_bottom;            // Eq. 32
  double res = 0.0;
  Fv[4] = Fv[5] = Fv[6] = 0.0;
  if (bc != 0) {
    const double BxJ0 = pb.By * s.J2 - pb.Bz * s.J1, BxJ1 = pb.Bz * s.J0 - pb.Bx * s.J2, BxJ2 = pb.Bx * s.J1 - pb.By * s.J0;
    res = ph.eta * (BxJ0 * nx + BxJ1 * ny + BxJ2 * nz);
    Fv[4] = -ph.eta * (ny * s.J2 - nz * s.J1);
    Fv[5] = -ph.eta * (nz * s.J0 - nx * s.J2);
    Fv[6] = -ph.eta * (nx * s.J1 - ny * s.J0);
  }
  Fv[3] = -qn + res;
}

// first k-step of a product: D = A*B (accumulator starts at zero, no register zeroing)
__device__ __forceinline__ void dmma884z(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%4,%4};\n"
               : "=d"(d0), "=d"(d1) : "d"(a), "d"(b), "d"(0.0));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }
// ---- TMA (bulk asynchronous copy, SASS UBLKCP) with mbarrier completion
__device__ __forceinline__ void mbar_init(uint64_t* mb, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(mb)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* mb, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(mb)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* mb, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"((unsigned)__cvta_generic_to_shared(mb)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load(void* smem, const void* gmem, unsigned bytes, uint64_t* mb) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                   (unsigned)__cvta_generic_to_shared(smem)),
               "l"(gmem), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(mb))
               : "memory");
}
// Orders the generic-proxy accesses of a destination buffer (made by other threads and ordered before this point by a barrier)
// before the async-proxy writes of the bulk copy that overwrites it: issued by every thread that issues a bulk copy.
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p)); }
// all threads of the CTA: prefetch `bytes` starting at p into L2, one request per 128-byte line
__device__ __forceinline__ void prefetch_block_l2(const void* p, size_t bytes, int tid, int nthreads) {
  const char* b = (const char*)p;
  for (size_t o = (size_t)tid * 128; o < bytes; o += (size_t)nthreads * 128) prefetch_l2(b + o);
}

// named barriers of the element kernel (id 0 is left to __syncthreads)
enum : int { kBarChain = 1, kBarHelp = 2, kBarIn = 3, kBarGrad = 4, kBarFaces = 5, kBarRes = 6, kBarNext = 7, kBarWave = 8 };
__device__ __forceinline__ void bar_sync(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int nthreads) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }
template <int R>
__device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(R)); }
template <int R>
__device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(R)); }

// thread layout of the element kernel: chain warpgroup(s) first (DMMA), then one helper warpgroup (memory, faces, sources, RK)
template <int N> struct MainCfg {
  static constexpr int kChainWG = kWideOrder(N) ? 2 : 1;
  // one CTA per SM: two helper warpgroups as well.  The helpers' phases (wall states, Rusanov pass, sources, final combination,
  // loads) are latency-bound and partly in series with the chains: twice the threads, half the time (n = 7 measured with one
  // helper warpgroup at 96 registers and 200-register chains: 4.17 ms on sweep_n7; with two at 88 and 168-register chains: 3.40)
  static constexpr int kHelpWG = kWideOrder(N) ? 2 : 1;
  static constexpr int kThreads = 128 * (kChainWG + kHelpWG);
  static constexpr int kMinBlocks = kChainWG == 2 ? 1 : 2;
};
// 128 * (chain + helper) = the CTA's 256 * 128 registers: two CTAs per SM.  With diffusion the chain warps carry the streamed
// viscous flux state and need 160; without it they are light and the helpers (sources, RK, next-state traces) get the room.
template <bool DIFF, int CWG = 1, int HWG = 1> struct RegSplit {
  // one chain warpgroup: launch at 128 registers (two CTAs per SM);
  // two chain and two helper warpgroups (512 threads, one CTA per SM): launch at 128, 2 x 168 + 2 x 88 = 4 x 128
  static_assert(CWG == HWG, "one chain + one helper warpgroup, or two + two");
  static constexpr int kLaunch = 128;
  static constexpr int kChain = CWG == 2 ? 168 : DIFF ? 160 : 144;     // measured at n = 6: 152 / 160 / 168 / 176 / 184
  static constexpr int kHelp = CWG == 2 ? 88 : 256 - kChain;           // chain registers: 0.696 / 0.699 / 0.671 / 0.699 / 0.721 ms
};

// per-thread constants of the DMMA mapping
template <int N>
struct LaneK {
  double bI0, bI1;     // interpolation operand, k-steps 0 and 1
  double bD0, bD1;     // derivative operand
  double bD2;          // kFaceOutOrder: derivative operand of the third k-step (k = 0: face point m = 0; k >= 1: zero)
  double bG[3];        // BR1 gradient operand
  int m0, m1;          // flux point of the two columns this thread holds (-1 = padding)
  int r, c;
};

// A3 along direction D: d Q_v / d xi_D at the solution points of 8 lines, variables GV0 .. GV0+NGV-1, into sG[(vv*3+D)]
// D = 3: the direction is the run-time value dd (tail tasks); lv = false: the row is padding (nothing is stored)
// COMMON: sQn already holds the common end values (BR1 average or wall state), made by the helpers' face pass an element ahead
template <int N, int NGV, int GV0, int D, bool COMMON = false>
__device__ __forceinline__ void grad_dir(const LaneK<N>& L, const ElemNbr& nb, const double* sQ, const double* sQo, const double* sQn,
                                         double* sG, int ln, bool lv, int dd = 0) {
  using I = Ix<N>;
  const int d = D < 3 ? D : dd;
  const int st = D == 0 ? 1 : D == 1 ? N : D == 2 ? I::n2 : I::stride(dd);
  constexpr int KG = (N + 2 + 3) / 4;
  const int sb = I::sbase(d, ln);
  const int c = L.c;
  // operand of k-step s >= 1 in the unified form  a = wX * X[v * sX] + wY * Y[v * sY]
  const double* X[3];
  const double* Y[3];
  int sX[3], sY[3];
  double wX[3], wY[3];
#pragma unroll
  for (int s = 1; s < KG; ++s) {
    const int k = 4 * s + c;
    if (k < N) {
      X[s] = Y[s] = sQ + sb + k * st; sX[s] = sY[s] = I::n3; wX[s] = 1.0; wY[s] = 0.0;
    } else if (k <= N + 1) {
      const int f = 2 * d + (k - N);
      const bool wall = COMMON || nb.ne[f] < 0;
      X[s] = (COMMON ? sQn : sQo) + f * 9 * I::n2 + ln; Y[s] = sQn + f * 9 * I::n2 + ln; sX[s] = sY[s] = I::n2;
      wX[s] = wall ? 0.0 : 0.5; wY[s] = wall ? 1.0 : 0.5;            // BR1 average, or the wall state
    } else {
      X[s] = Y[s] = sQ + sb; sX[s] = sY[s] = I::n3; wX[s] = 0.0; wY[s] = 0.0;   // padding: the B operand is zero
    }
  }
  const double* A0 = sQ + sb + c * st;          // k-step 0: k = c < N
  const bool ok0 = lv && 2 * c < N, ok1 = lv && 2 * c + 1 < N;
  double* out = sG + d * I::n3 + sb + (2 * c) * st;
  constexpr int VB = NGV % 3 == 0 ? 3 : 1;      // variables in flight (hides the DMMA latency; 9 at a time measured slower)
#pragma unroll
  for (int v0 = 0; v0 < NGV; v0 += VB) {
    double d0[VB], d1[VB];
#pragma unroll
    for (int j = 0; j < VB; ++j) dmma884z(d0[j], d1[j], A0[(GV0 + v0 + j) * I::n3], L.bG[0]);
#pragma unroll
    for (int s = 1; s < KG; ++s)
#pragma unroll
      for (int j = 0; j < VB; ++j) {
        const int v = GV0 + v0 + j;
        const double a = wX[s] * X[s][v * sX[s]] + wY[s] * Y[s][v * sY[s]];
        dmma884(d0[j], d1[j], a, L.bG[s]);
      }
#pragma unroll
    for (int j = 0; j < VB; ++j) {
      if (ok0) out[(v0 + j) * 3 * I::n3] = d0[j];
      if (ok1) out[(v0 + j) * 3 * I::n3 + st] = d1[j];
    }
  }
}

// A1 + A4 + A5 + A7 along direction D for 8 lines: the register-resident chain
// D = 3: run-time direction dd (tail tasks).  Direction-0 tasks store into sR, all others accumulate.
// WAITF: this is the element's first chain task of the warp: the common face fluxes (written by the helper warps beside the
// chain rule and the first interpolations) are awaited here, just before they are needed, and the left-over direction-0
// points of sR are zeroed.
// STORE: 1 store the divergence contribution, 0 accumulate it, -1 (default): store for direction 0, accumulate otherwise.
// SYNCB: 1: this is the warp's first task of a round that accumulates: the chain-warp barrier that separates the rounds is taken
// here, just before the update, instead of before the task (the warps drift apart by less than the barrier used to cost);
// 2: the same with the barrier between the two waves of the kPre pipeline (the warps without a second task only arrive).
template <int N, bool DIFF, int D, bool WAITF = false, int STORE = -1, int SYNCB = 0>
__device__ __forceinline__ void chain_dir(const LaneK<N>& L, const PhysD& ph, const ElemNbr& nb, const StageIO& io, const Geo& geo,
                                          int64_t e, const double* sQ, const double* sG, const double* sFace, const double* sS, double* sR,
                                          int ln, bool lv, int dd = 0, int ctid = 0) {
  using I = Ix<N>;
  const int d = D < 3 ? D : dd;
  const int st = D == 0 ? 1 : D == 1 ? N : D == 2 ? I::n2 : I::stride(dd);
  const int sb = I::sbase(d, ln);
  const int c = L.c, m0 = L.m0, m1 = L.m1;
  const int l1 = 4 + c < N ? 4 + c : N - 1;     // second k-step: l = 4 + c, clamped where the B operand is zero anyway
  const double* A0 = sQ + sb + c * st;
  const double* A1 = sQ + sb + l1 * st;
  const bool int0 = m0 > 0 && m0 < N, int1 = m1 > 0 && m1 < N;
  const int fb = I::fbase(d, ln);
  double S0x = 0.0, S0y = 0.0, S0z = 0.0, S1x = 0.0, S1y = 0.0, S1z = 0.0, kr0 = 0.0, kr1 = 0.0;
  if constexpr (kSglobalOrder(N)) {   // S^d comes from global memory (L2): issued first, needed after the first interpolations
    if (int0) {
      const double* s = sS + (d * 3) * I::nf + fb + m0 * st;
      S0x = s[0]; S0y = s[I::nf]; S0z = s[2 * I::nf];
    }
    if (int1) {
      const double* s = sS + (d * 3) * I::nf + fb + m1 * st;
      S1x = s[0]; S1y = s[I::nf]; S1z = s[2 * I::nf];
    }
  }
  // A1: Q at the two flux points of this thread
  double q0[9], q1[9];
#pragma unroll
  for (int v = 0; v < 9; ++v) dmma884z(q0[v], q1[v], A0[v * I::n3], L.bI0);
  if (N > 4) {
#pragma unroll
    for (int v = 0; v < 9; ++v) dmma884(q0[v], q1[v], A1[v * I::n3], L.bI1);
  }
  // per-slot setup: area vector and the state the fluxes are evaluated on
  const bool face0 = m0 == 0 || m0 == N, face1 = m1 == 0 || m1 == N;     // m = -1: padding
  int fc0 = 0, fc1 = 0;
  constexpr int kNFS = kSintOrder(N) ? I::n2 * (N - 1) : I::nf;        // points per component of the S^d tile
  // interior-only tile: the natural family layout with n - 1 points per line, first point m = 1
  const int fbs = !kSintOrder(N) ? fb : d == 0 ? ln * (N - 1) - 1 : d == 1 ? (ln / N) * (N - 1) * N + ln % N - N : ln - I::n2;
  if (!kSglobalOrder(N) && int0) {
    const double* s = sS + (d * 3) * kNFS + fbs + m0 * st;
    S0x = s[0]; S0y = s[kNFS]; S0z = s[2 * kNFS];
  }
  if (!kSglobalOrder(N) && int1) {
    const double* s = sS + (d * 3) * kNFS + fbs + m1 * st;
    S1x = s[0]; S1y = s[kNFS]; S1z = s[2 * kNFS];
  }
  if (DIFF) {   // face columns: the own-side viscous flux along the outward unit normal, on Q_in (interior) or Q_b (wall)
    if (face0) {
      fc0 = 2 * d + (m0 == N ? 1 : 0);
      const double* nf_ = geo.nfc + ((e * 6 + fc0) * 4) * I::n2 + ln;
      S0x = nf_[0]; S0y = nf_[I::n2]; S0z = nf_[2 * I::n2];
      if (nb.ne[fc0] < 0) {
        double qb[9];
        wall_state(ph, nb.ne[fc0], q0, S0x, S0y, S0z, qb);
#pragma unroll
        for (int v = 0; v < 9; ++v) q0[v] = qb[v];
      }
    }
    if (face1) {
      fc1 = 2 * d + (m1 == N ? 1 : 0);
      const double* nf_ = geo.nfc + ((e * 6 + fc1) * 4) * I::n2 + ln;
      S1x = nf_[0]; S1y = nf_[I::n2]; S1z = nf_[2 * I::n2];
      if (nb.ne[fc1] < 0) {
        double qb[9];
        wall_state(ph, nb.ne[fc1], q1, S1x, S1y, S1z, qb);
#pragma unroll
        for (int v = 0; v < 9; ++v) q1[v] = qb[v];
      }
    }
    if (geo.krfl) {
      if (m0 >= 0) kr0 = geo.krfl[(e * 3 + d) * I::nf + fb + m0 * st];
      if (m1 >= 0) kr1 = geo.krfl[(e * 3 + d) * I::nf + fb + m1 * st];
    }
  }
  PrimD p0, p1;
  if (DIFF || int0) p0 = primitives(ph, q0);
  if (DIFF || int1) p1 = primitives(ph, q1);
  double Fv0[7], Fv1[7];
  if (DIFF) {
    // A4 + Eq. 7-10: stream the gradients of the nine variables through the tensor core, three components at a time
    VStream s0, s1;
    const double* G0 = sG + sb + c * st;
    const double* G1 = sG + sb + l1 * st;
#define CHORUS_STREAM_VAR(V)                                             \
  {                                                                      \
    double ga0, ga1, gb0, gb1, gc0, gc1;                                   \
    dmma884z(ga0, ga1, G0[(3 * (V)) * I::n3], L.bI0);                    \
    dmma884z(gb0, gb1, G0[(3 * (V) + 1) * I::n3], L.bI0);                \
    dmma884z(gc0, gc1, G0[(3 * (V) + 2) * I::n3], L.bI0);                \
    if (N > 4) {                                                         \
      dmma884(ga0, ga1, G1[(3 * (V)) * I::n3], L.bI1);                   \
      dmma884(gb0, gb1, G1[(3 * (V) + 1) * I::n3], L.bI1);               \
      dmma884(gc0, gc1, G1[(3 * (V) + 2) * I::n3], L.bI1);               \
    }                                                                    \
    vs_fold<V>(s0, p0, S0x, S0y, S0z, ga0, gb0, gc0);                    \
    vs_fold<V>(s1, p1, S1x, S1y, S1z, ga1, gb1, gc1);                    \
  }
    CHORUS_STREAM_VAR(0) CHORUS_STREAM_VAR(1) CHORUS_STREAM_VAR(2) CHORUS_STREAM_VAR(3) CHORUS_STREAM_VAR(4)
    CHORUS_STREAM_VAR(5) CHORUS_STREAM_VAR(6) CHORUS_STREAM_VAR(7) CHORUS_STREAM_VAR(8)
#undef CHORUS_STREAM_VAR
    if (face0 && nb.ne[fc0] < 0) vs_flux_wall(ph, nb.ne[fc0], s0, p0, S0x, S0y, S0z, kr0, Fv0);
    else vs_flux(ph, s0, p0, S0x, S0y, S0z, kr0, Fv0);
    if (face1 && nb.ne[fc1] < 0) vs_flux_wall(ph, nb.ne[fc1], s1, p1, S1x, S1y, S1z, kr1, Fv1);
    else vs_flux(ph, s1, p1, S1x, S1y, S1z, kr1, Fv1);
    if (lv && face0) {
      double* o = io.Vf + ((e * 6 + fc0) * 7) * I::n2 + ln;
#pragma unroll
      for (int k = 0; k < 7; ++k) o[k * I::n2] = Fv0[k];
    }
    if (lv && face1) {
      double* o = io.Vf + ((e * 6 + fc1) * 7) * I::n2 + ln;
#pragma unroll
      for (int k = 0; k < 7; ++k) o[k * I::n2] = Fv1[k];
    }
  }
  if (WAITF) {
    bar_sync(kBarFaces, MainCfg<N>::kThreads);     // common face fluxes are in sFace; own traces are dead: their region becomes sR
    // Direction 0 stores into sR, the others accumulate; the points of the left-over direction-0 lines, which no direction-0
    // task touches, start from zero (they are first accumulated into after the next chain-warp barrier).
    using MM = Mma<N>;
    if constexpr (MM::LO > 0 && !MM::kFree) {
      for (int t = ctid; t < 9 * MM::LO * N; t += 32 * MM::kWarps) {
        const int l = t % N, i = (t / N) % MM::LO, v = t / (N * MM::LO);
        sR[v * I::n3 + I::sbase(0, MM::line_of(0, 8 * MM::FG + i)) + l] = 0.0;
      }
    }
  }
  // A5: F~ at the interior flux points; face columns take the common flux of the face pass; results overwrite q0 / q1
  if (int0) {
    double F[9];
    flux_inviscid<false>(ph, p0, S0x, S0y, S0z, F);
    q0[0] = F[0]; q0[8] = F[8];
#pragma unroll
    for (int k = 0; k < 7; ++k) q0[1 + k] = DIFF ? F[1 + k] - Fv0[k] : F[1 + k];
  } else if (m0 >= 0) {
    const double* f = sFace + ((2 * d + (m0 == N ? 1 : 0)) * 9) * I::n2 + ln;
#pragma unroll
    for (int v = 0; v < 9; ++v) q0[v] = f[v * I::n2];
  } else {
#pragma unroll
    for (int v = 0; v < 9; ++v) q0[v] = 0.0;
  }
  if (int1) {
    double F[9];
    flux_inviscid<false>(ph, p1, S1x, S1y, S1z, F);
    q1[0] = F[0]; q1[8] = F[8];
#pragma unroll
    for (int k = 0; k < 7; ++k) q1[1 + k] = DIFF ? F[1 + k] - Fv1[k] : F[1 + k];
  } else if (m1 >= 0) {
    const double* f = sFace + ((2 * d + (m1 == N ? 1 : 0)) * 9) * I::n2 + ln;
#pragma unroll
    for (int v = 0; v < 9; ++v) q1[v] = f[v * I::n2];
  } else {
#pragma unroll
    for (int v = 0; v < 9; ++v) q1[v] = 0.0;
  }
  // A7: derivative of the flux polynomial at the solution points of the line: C fragments reused as A fragments
  const bool ok0 = lv && 2 * c < N, ok1 = lv && 2 * c + 1 < N;
  double* out = sR + sb + (2 * c) * st;
  double r0[9], r1[9];
#pragma unroll
  for (int v = 0; v < 9; ++v) dmma884z(r0[v], r1[v], q0[v], L.bD0);
#pragma unroll
  for (int v = 0; v < 9; ++v) dmma884(r0[v], r1[v], q1[v], L.bD1);
  if constexpr (kFaceOutOrder(N)) {   // third k-step: the common flux of the line's face point m = 0 (k = 0; the B operand of k >= 1 is zero)
    const double* f = sFace + ((2 * d) * 9) * I::n2 + ln;
#pragma unroll
    for (int v = 0; v < 9; ++v) dmma884(r0[v], r1[v], f[v * I::n2], L.bD2);
  }
  if (SYNCB == 1) bar_sync(kBarChain, 128 * Mma<N>::kChainWG);     // every update of the previous round is in sR
  if (SYNCB == 2) bar_sync(kBarWave, 128 * Mma<N>::kChainWG);      // kPre: every store of the first wave is in the accumulators
#pragma unroll
  for (int v = 0; v < 9; ++v) {
    constexpr bool kStore = STORE == 1 || (STORE == -1 && D == 0);
    if (ok0) out[v * I::n3] = kStore ? r0[v] : out[v * I::n3] + r0[v];
    if (ok1) out[v * I::n3 + st] = kStore ? r1[v] : out[v * I::n3 + st] + r1[v];
  }
}

// the next element of this CTA: pull what it will read towards L2 (issued by the helper warps while the chains run)
template <int N, int GRADV>
__device__ __forceinline__ void prefetch_next(const StageIO& io, const Geo& geo, int64_t en, int ne, int nf, int tid, int nthreads) {
  using I = Ix<N>;
  prefetch_block_l2(io.Qe + en * 9 * I::n3, sizeof(double) * 9 * I::n3, tid, nthreads);
  prefetch_block_l2(io.Qf + en * 54 * I::n2, sizeof(double) * 54 * I::n2, tid, nthreads);
  if (kSintOrder(N)) prefetch_block_l2(geo.Sint + en * 9 * I::n2 * (N - 1), sizeof(double) * 9 * I::n2 * (N - 1), tid, nthreads);
  else prefetch_block_l2(geo.Sfl + en * 9 * I::nf, sizeof(double) * 9 * I::nf, tid, nthreads);
  prefetch_block_l2(geo.nfc + en * 24 * I::n2, sizeof(double) * 24 * I::n2, tid, nthreads);
  prefetch_block_l2(geo.detJ + en * I::n3, sizeof(double) * I::n3, tid, nthreads);
  prefetch_block_l2(geo.xsol + en * 3 * I::n3, sizeof(double) * 3 * I::n3, tid, nthreads);
  if (GRADV != 0) prefetch_block_l2(geo.jinv + en * 9 * I::n3, sizeof(double) * 9 * I::n3, tid, nthreads);
  if (io.A0) prefetch_block_l2(io.A0 + en * 9 * I::n3, sizeof(double) * 9 * I::n3, tid, nthreads);
  if (io.A1) prefetch_block_l2(io.A1 + en * 9 * I::n3, sizeof(double) * 9 * I::n3, tid, nthreads);
  // threads 0..5 hold the neighbour (ne, nf) of face tid: one neighbour face block each, 9 n^2 doubles
  if (tid < 6 && ne >= 0) {
    const char* b = (const char*)(io.Qf + ((int64_t)ne * 6 + nf) * 9 * I::n2);
    for (size_t o = 0; o < sizeof(double) * 9 * I::n2; o += 128) prefetch_l2(b + o);
  }
}

// GRADV: 0 no gradient needed, 1 gradient of B only (Powell sources without diffusion), 2 all nine variables.
//
// A CTA works on ONE element at a time with two kinds of warps:
//   chain warps: the DMMA work -- gradient tasks, chain rule, the A1/A4/A5/A7 chains;
//   helper warps: everything that waits on memory or is pointwise -- bulk copies of the element's inputs, wall states, the
//     Rusanov face pass, the sources and Runge-Kutta registers (K, w), and the final combination out = w * (div_xi F~) + K.
// Four configurations (MainCfg, RegSplit):
//   n = 4, 5   two CTAs per SM, 4 chain warps (160 registers) + 4 helper warps (96); tasks dealt freely (kFree);
//              barriers per element: IN (inputs ready) -> GRAD (gradient DMMAs done, face fluxes in registers) -> FACES
//              (face fluxes in shared memory) -> RES (divergence accumulated); the helpers' face pass runs beside the gradient;
//   n = 7      one CTA per SM (222 KB of tiles), 8 chain warps (168) + 8 helper warps (88), tasks dealt freely;
//   n = 8      one CTA per SM (212 KB), 8 + 8 warps, three barrier-separated direction rounds of 8 tasks on one accumulator;
//              its tiles hold 7 interior flux points and the face point m = n (kFaceOutOrder), S^d comes from L2;
//   n = 6      one CTA per SM, 8 chain warps (168) + 8 helper warps (88), TWO sets of input tiles and TWO gradient buffers
//              (kPre, 223 KB in all; the S^d tile holds the interior flux points only, Geo::Sint, and the neighbour-trace /
//              common-solution tile exists once): while the chain warps work on element e the helpers bring in element
//              e + 1 -- bulk copies, wall states, common solution and common fluxes (face_pass) -- and the two chain warps
//              that have no task in the element's second wave compute the gradient of e + 1, so that between two elements
//              only the chain rule is left; the finish of element e is deferred until e + 1 is under way.  Barriers per
//              element: FACES (accumulators free: helpers arrive, chains wait inside their first task) -> WAVE (first-wave
//              stores done; chains only) -> NEXT (inputs of e + 1 handed over: helpers arrive, the gradient warps wait) ->
//              RES (chains done with e: they only arrive) -> GRAD (gradient of e + 1 complete: chains only arrive).
template <int N, bool DIFF, int GRADV>
__global__ void __launch_bounds__(MainCfg<N>::kThreads, MainCfg<N>::kMinBlocks)
stage_main_kernel(int64_t E, PhysD ph, StageIO io, Geo geo) {
  using I = Ix<N>;
  using M = Mma<N>;
  static_assert(!DIFF || GRADV == 2, "diffusion needs the gradient of all variables");
  constexpr int NGV = GRADV == 2 ? 9 : GRADV == 1 ? 3 : 0;
  constexpr int GV0 = GRADV == 1 ? 5 : 0;
  extern __shared__ __align__(16) double sm[];
  constexpr int kOwn = 54 * I::n2 > 9 * I::n3 ? 54 * I::n2 : 9 * I::n3;
  constexpr auto ev = [](int x) { return (x + 1) & ~1; };   // keep every array 16-byte aligned
  // one set of INPUT tiles: sQ [9][n3] | sQo [6][9][n2] own traces, reused as sR [9][n3] after the face pass | sQn [6][9][n2]
  // neighbour traces / wall states, overwritten by the face fluxes | sS [3 fam][3 comp][nf] S^d at the flux points
  constexpr bool kSglobal = kSglobalOrder(N);   // S^d read from global memory by the chains (no shared-memory tile)
  constexpr bool kPre = kPrefetchOrder(N);   // two input sets, used alternately (element i of this CTA: set i & 1)
  static_assert(!kPre || kSintOrder(N), "the kPre layout stages the interior-only S^d tile");
  constexpr int kST = kSglobal ? 0 : kSintOrder(N) ? 9 * I::n2 * (N - 1) : 9 * I::nf;    // doubles of the S^d tile
  // kPre: the neighbour traces / common solution tile sQn is NOT part of the set: it lives from the loads of an element to the
  // end of that element's gradient tasks, which run an element ahead -- one copy is enough
  constexpr int kIn = ev(9 * I::n3) + ev(kOwn) + (kPre ? 0 : ev(54 * I::n2)) + kST;
  double* sQn1 = sm + 2 * kIn;               // kPre: the single sQn
  double* sG = sm + (kPre ? 2 * kIn + ev(54 * I::n2) : kIn);    // [3*NGV][n3]; kPre: two of them (the next gradient is made ahead)
  constexpr int kGS = ev(3 * NGV * I::n3);
  double* sR12 = sG + (kPre ? 2 : 1) * kGS;  // kFree: the accumulators of directions 1 and 2, [2][9][n3] (direction 0: sR);
  constexpr int kRS = ev(9 * I::n3);         // kPre: the two accumulators of the two task waves (see the chain loop)
  // kPre without diffusion, step mode: the new state of the finished element, from which its face traces are made -- by the
  // chain warps, in the time they would otherwise wait for the next gradient (without diffusion the helpers are the longer side)
  double* sNew = sR12 + 2 * kRS;
  constexpr bool kChainTraces = kPre && !DIFF;
  __shared__ ElemNbr nbs[2];
  __shared__ int s_second;
  __shared__ int s_task[kPre ? M::kTasks * 8 : 1];   // kPre: (task, row) -> line | direction << 16 | row carries a line << 20
  __shared__ __align__(8) uint64_t mbar;   // completion of the bulk (TMA) copies of one element
  if (threadIdx.x == 0) {
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    s_second = (int)(atomicAdd(io.sm_arrivals + smid, 1u) & 1u);
    mbar_init(&mbar, 2);     // two producer arrivals per element: part A and part B of its loads
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  if constexpr (kPre) {
    for (int t = threadIdx.x; t < M::kTasks * 8; t += blockDim.x) {
      const int i = t >> 3, r = t & 7;
      int d, ln, ok = 1;
      if (i < 3 * M::FG) {
        d = i / M::FG;
        ln = M::line_of(d, (i % M::FG) * 8 + r);
      } else {
        const int q = (i - 3 * M::FG) * 8 + r;               // index among the 3 LO left-over lines
        ok = q < 3 * M::LO;
        d = ok ? q / (M::LO > 0 ? M::LO : 1) : 0;
        ln = M::line_of(d, 8 * M::FG + (ok ? q % (M::LO > 0 ? M::LO : 1) : 0));
      }
      s_task[t] = ln | (d << 16) | (ok << 20);
    }
  }
  __syncthreads();
  constexpr int kMainThreads = MainCfg<N>::kThreads, kCT = 128 * M::kChainWG;      // all threads / chain threads
  using RS = RegSplit<DIFF, M::kChainWG, MainCfg<N>::kHelpWG>;
  const bool is_chain = M::kChainWG == 1 ? (threadIdx.x >> 7) == 0 : threadIdx.x < kCT;
  const int tid = M::kChainWG == 1 ? (int)(threadIdx.x & 127) : is_chain ? (int)threadIdx.x : (int)threadIdx.x - kCT;
  // The contiguous per-element blocks (state, own traces, S^d) go by TMA bulk copy when they are 16-byte aligned (n even);
  // the neighbour traces are gathered through the orientation map with 8-byte cp.async either way.
  constexpr bool kBulk = (9 * I::n3) % 2 == 0 && (54 * I::n2) % 2 == 0;
  constexpr int H = 128 * MainCfg<N>::kHelpWG;   // helper threads

  if (is_chain) {
    // =============================================== chain warps ===============================================
    constexpr int CH = kCT;              // chain threads
    if (RS::kChain > RS::kLaunch) setmaxnreg_inc<RS::kChain>();
    else if (RS::kChain < RS::kLaunch) setmaxnreg_dec<RS::kChain>();
    const OpsC& op = c_ops[N];
    const int lane = tid & 31, warp = tid >> 5;
    const bool active = warp < M::kWarps;
    // ---- per-lane operator fragments (B operands), fixed for the whole kernel
    LaneK<N> L;
    L.r = lane >> 2; L.c = lane & 3;
    {
      const int r = L.r, c = L.c;
      // interpolation: B[k = l][n = col r] = h_l(X_f,m(r));  k-step s covers l = 4s + c
      const int mB = M::col_m(r);
      L.bI0 = 0.0; L.bI1 = 0.0;
      if (mB >= 0) {
        L.bI0 = op.Isf[mB * N + c];
        if (4 + c < N) L.bI1 = op.Isf[mB * N + 4 + c];
      }
      // derivative: B[k = col][n = l_out r] = l'_{m(col)}(X_s,l_out);  k-step s covers col = 2c + s  (the C -> A reuse)
      L.m0 = M::col_m(2 * c); L.m1 = M::col_m(2 * c + 1);
      L.bD0 = 0.0; L.bD1 = 0.0;
      if (r < N) {
        if (L.m0 >= 0) L.bD0 = op.Dfs[r * (N + 1) + L.m0];
        if (L.m1 >= 0) L.bD1 = op.Dfs[r * (N + 1) + L.m1];
      }
      L.bD2 = (r < N && c == 0) ? op.Dfs[r * (N + 1)] : 0.0;
      // BR1 gradient: x = (q_0..q_{N-1}, common value at m = 0, at m = N), K = N + 2 -> up to 3 k-steps of 4
      // B[k][n = l_out r]: k < N: Dss[l_out][k]; k = N: Dfs[l_out][0]; k = N+1: Dfs[l_out][N]
#pragma unroll
      for (int s = 0; s < 3; ++s) {
        const int k = 4 * s + c;
        L.bG[s] = 0.0;
        if (r < N) {
          if (k < N) L.bG[s] = op.Dss[r * N + k];
          else if (k == N) L.bG[s] = op.Dfs[r * (N + 1)];
          else if (k == N + 1) L.bG[s] = op.Dfs[r * (N + 1) + N];
        }
      }
    }
    // lines of this thread's row: directional tasks g = warp, warp + kWarps, ... of each direction, and one row of a tail task
    int lnd[3][M::kTPD];
#pragma unroll
    for (int d = 0; d < 3; ++d)
#pragma unroll
      for (int k = 0; k < M::kTPD; ++k) {
        const int g = warp + k * M::kWarps;
        lnd[d][k] = M::line_of(d, (g < M::FG ? g : 0) * 8 + L.r);
      }
    // kFree: task i = warp + kFreeWarps t of this warp: direction, line of this thread's row, validity of the row
    int fd[M::kTPW], fl[M::kTPW];
    bool fv[M::kTPW], fr[M::kTPW];        // task exists / row carries a line
#pragma unroll
    for (int t = 0; t < M::kTPW; ++t) {
      const int i = warp + M::kFreeWarps * t;
      fv[t] = M::kFree && i < M::kTasks;
      fr[t] = fv[t];
      fd[t] = 0; fl[t] = 0;
      if (fv[t]) {
        if (i < 3 * M::FG) {
          fd[t] = i / M::FG;
          fl[t] = M::line_of(fd[t], (i % M::FG) * 8 + L.r);
        } else {
          const int q = (i - 3 * M::FG) * 8 + L.r;            // index among the 3 LO left-over lines
          fr[t] = q < 3 * M::LO;
          fd[t] = fr[t] ? q / (M::LO > 0 ? M::LO : 1) : 0;
          fl[t] = M::line_of(fd[t], 8 * M::FG + (fr[t] ? q % (M::LO > 0 ? M::LO : 1) : 0));
        }
      }
    }
    // tail tasks rotate over the warps (hence over the SM sub-partitions) from element to element, and every second CTA
    // arriving on an SM starts half a turn ahead
    int tail_rot = s_second ? M::kWarps / 2 : 0;
    constexpr int P2 = (I::n3 + CH - 1) / CH;     // solution points per chain thread in the chain rule
    unsigned ld_phase = 0;
    int it = 0;
    if constexpr (kPre) {
      // ---- The pipeline of the order with two sets of input tiles and two gradient buffers.  An element's 14 tasks run in two
      //      waves on the 8 chain warps: wave 1 = the 2 FG full-group tasks of directions 0 and 1 (one per warp; each STORES
      //      into the accumulator of its direction, acc0 / acc1), wave 2 = the FG tasks of direction 2 (warps 0..FG-1, which ADD
      //      into acc0) and the tail tasks (which ADD into acc1; left-over lines never meet in a point).  The warps without a
      //      second task (kGW0..7) compute the NEXT element's gradient tasks meanwhile, into the other gradient buffer, so that
      //      the gradient phase leaves the critical path: between two elements only the chain rule is left.
      static_assert(M::kTPW == 2 && 2 * M::FG == M::kFreeWarps && M::kChainWG == 2, "wave structure of the kPre pipeline");
      constexpr int kGW0 = M::kTasks - M::kFreeWarps;          // first warp without a second-wave task
      constexpr int kGW = M::kFreeWarps - kGW0;                // warps that make the next gradient
      double* acc0 = sR12;
      double* acc1 = sR12 + kRS;
      auto wait_inputs = [&]() {                               // bulk copies: completion is observed by every consumer thread itself
        if (kBulk) mbar_wait(&mbar, ld_phase);
        ld_phase ^= 1u;
      };
      double jv[P2][9];
      auto load_jv = [&](int64_t el) {     // chain-rule metrics of this thread's solution points (L2-resident: prefetched ahead)
        if (GRADV != 0) {
#pragma unroll
          for (int q = 0; q < P2; ++q) {
            const int sc = tid + q * CH < I::n3 ? tid + q * CH : 0;
#pragma unroll
            for (int k = 0; k < 9; ++k) jv[q][k] = geo.jinv[el * 9 * I::n3 + k * I::n3 + sc];
          }
        }
      };
      auto chain_rule = [&](double* G) {
        if constexpr (GRADV != 0) {
#pragma unroll
          for (int q = 0; q < P2; ++q) {
            const int sp = tid + q * CH;
            if (sp < I::n3) {
#pragma unroll
              for (int vv = 0; vv < NGV; ++vv) {
                const double g0 = G[(vv * 3 + 0) * I::n3 + sp], g1 = G[(vv * 3 + 1) * I::n3 + sp], g2 = G[(vv * 3 + 2) * I::n3 + sp];
#pragma unroll
                for (int pp = 0; pp < 3; ++pp) G[(vv * 3 + pp) * I::n3 + sp] = jv[q][pp] * g0 + jv[q][3 + pp] * g1 + jv[q][6 + pp] * g2;
              }
            }
          }
        }
      };
      // first element: its gradient is made by all chain warps
      if ((int64_t)blockIdx.x < E) {
        load_jv(blockIdx.x);
        wait_inputs();
        bar_sync(kBarIn, kMainThreads);          // inputs, common solution and common fluxes of the first element are in shared memory
        if constexpr (GRADV != 0) {
          const double* q0 = sm;
#pragma unroll
          for (int t = 0; t < M::kTPW; ++t)
            if (fv[t]) grad_dir<N, NGV, GV0, 3, true>(L, nbs[0], q0, q0 + ev(9 * I::n3), sQn1, sG, fl[t], fr[t], fd[t]);
        }
        bar_sync(kBarChain, CH);
        chain_rule(sG);
        bar_sync(kBarChain, CH);
        bar_arrive(kBarGrad, kMainThreads);      // the gradient is complete: the helpers' sources (div B) wait for it
      }
      for (int64_t e = blockIdx.x; e < E; e += gridDim.x, ++it) {
        const int cur = it & 1;
        const bool more = e + gridDim.x < E;
        double* sQ = sm + cur * kIn;
        double* sQo = sQ + ev(9 * I::n3);        // the common face fluxes
        const double* sS = sQo + ev(kOwn);       // S^d at the interior flux points
        const double* sGc = sG + cur * kGS;
        // wave 1: stores; the FACES barrier (accumulators free) is taken inside, just before the common fluxes are needed
        chain_dir<N, DIFF, 3, true, 1>(L, ph, nbs[cur], io, geo, e, sQ, sGc, sQo, sS, fd[0] == 0 ? acc0 : acc1, fl[0], fr[0], fd[0], tid);
        // the points of the left-over lines of directions 0 and 1, which no first-wave task stores, start from zero
        if constexpr (M::LO > 0) {
          for (int t = tid; t < 2 * 9 * M::LO * N; t += CH) {
            const int l = t % N, i = (t / N) % M::LO, v = (t / (N * M::LO)) % 9, d = t / (9 * N * M::LO);
            const int ln = s_task[(3 * M::FG) * 8 + d * M::LO + i] & 0xffff;      // tail rows: direction-major, LO lines each
            (d == 0 ? acc0 : acc1)[v * I::n3 + I::sbase(d, ln) + l * I::stride(d)] = 0.0;
          }
        }
        if (warp < kGW0) {
          // wave 2: accumulates; the barrier between the waves is taken inside, just before the update
          chain_dir<N, DIFF, 3, false, 0, 2>(L, ph, nbs[cur], io, geo, e, sQ, sGc, sQo, sS, warp < M::FG ? acc0 : acc1, fl[1], fr[1], fd[1]);
          // The bulk copies of the next element are observed BEFORE this warp reports that it is done with element e: after
          // that report the helpers may start the copies of the element after the next, and a wait for "the phase of this
          // parity" would then match the wrong phase.
          if (kChainTraces && io.Qout != nullptr && it > 0)     // traces of the element before, whose new state the helpers left in sNew
            emit_traces<N>(sNew, io.QfOut + (e - gridDim.x) * 54 * I::n2, tid, 32 * kGW0);
          if (more) wait_inputs();
          bar_arrive(kBarRes, kMainThreads);     // this warp is done with element e (and with sNew)
          if (!more) break;
          load_jv(e + gridDim.x);
        } else {
          bar_arrive(kBarWave, CH);
          if (more) {
            wait_inputs();
            bar_sync(kBarNext, H + 32 * kGW);    // inputs, common solution and common fluxes of the next element are in shared memory
          }
          if (!more) {
            bar_arrive(kBarRes, kMainThreads);
            break;
          }
          if constexpr (GRADV != 0) {
            const double* qn = sm + (cur ^ 1) * kIn;
            double* sGn = sG + (cur ^ 1) * kGS;
            for (int i = warp - kGW0; i < M::kTasks; i += kGW) {
              const int td = s_task[i * 8 + L.r];
              grad_dir<N, NGV, GV0, 3, true>(L, nbs[cur ^ 1], qn, qn + ev(9 * I::n3), sQn1, sGn, td & 0xffff,
                                              (td >> 20) != 0, (td >> 16) & 3);
            }
          }
          // done with element e AND with the common solution of the next one in the single sQn tile: after this report the
          // helpers may start the copies of the element after the next into it
          bar_arrive(kBarRes, kMainThreads);
          load_jv(e + gridDim.x);
        }
        bar_sync(kBarChain, CH);                 // the next element's gradient tasks are done, and every chain warp with element e
        chain_rule(sG + (cur ^ 1) * kGS);
        bar_sync(kBarChain, CH);
        bar_arrive(kBarGrad, kMainThreads);
      }
      if (kChainTraces && io.Qout != nullptr && (int64_t)blockIdx.x < E) {   // the last element's traces, once the helpers have finished it
        const int64_t e_last = (int64_t)blockIdx.x + (int64_t)it * gridDim.x;
        bar_sync(kBarIn, kMainThreads);
        emit_traces<N>(sNew, io.QfOut + e_last * 54 * I::n2, tid, CH);
      }
    } else
    for (int64_t e = blockIdx.x; e < E; e += gridDim.x, ++it) {
      const int cur = 0;
      double* sQ = sm + cur * kIn;
      double* sQo = sQ + ev(9 * I::n3);
      double* sQn = sQo + ev(kOwn);
      const double* sS = kSglobal ? geo.Sfl + e * 9 * I::nf : sQn + ev(54 * I::n2);
      double* sR = sQo;
      double* sFace = sQn;       // where the common face fluxes are
      const ElemNbr& nb = nbs[cur];
      int tw = M::kWarps, tl_d = 0, tl_ln = 0;
      bool tl_ok = false;
      if (M::kTail > 0 && active) {
        tw = (warp + tail_rot) % M::kWarps;          // this warp's tail-task index for this element (>= kTail: none)
        const int q = tw * 8 + L.r;                  // index among the 3 LO left-over lines
        tl_ok = tw < M::kTail && q < 3 * M::LO;
        tl_d = tl_ok ? q / (M::LO > 0 ? M::LO : 1) : 0;
        tl_ln = M::line_of(tl_d, 8 * M::FG + (tl_ok ? q % (M::LO > 0 ? M::LO : 1) : 0));
        tail_rot = (tail_rot + 1) % M::kWarps;
      }
      double jv[P2][9];
      auto load_jv = [&]() {     // chain-rule metrics of this thread's solution points (L2-resident: prefetched an element ahead)
        if (GRADV != 0) {
#pragma unroll
          for (int q = 0; q < P2; ++q) {
            const int s = tid + q * CH;
            const int sc = s < I::n3 ? s : 0;
#pragma unroll
            for (int k = 0; k < 9; ++k) jv[q][k] = geo.jinv[e * 9 * I::n3 + k * I::n3 + sc];
          }
        }
      };
      load_jv();                 // issued now, consumed after the gradient DMMAs
      if (kBulk) mbar_wait(&mbar, ld_phase);   // bulk copies: completion is observed by every consumer thread itself
      ld_phase ^= 1u;
      bar_sync(kBarIn, kMainThreads);          // inputs and wall states are in shared memory
      // ---- A3: BR1 gradient.  d/dxi_d by DMMA, then the chain rule per point.
      if constexpr (GRADV != 0 && M::kFree) {
#pragma unroll
        for (int t = 0; t < M::kTPW; ++t)
          if (fv[t]) grad_dir<N, NGV, GV0, 3, kPre>(L, nb, sQ, sQo, sQn, sG, fl[t], fr[t], fd[t]);
      } else if constexpr (GRADV != 0) {
        if (active) {
#pragma unroll
          for (int k = 0; k < M::kTPD; ++k)
            if (warp + k * M::kWarps < M::FG) {
              grad_dir<N, NGV, GV0, 0>(L, nb, sQ, sQo, sQn, sG, lnd[0][k], true);
              grad_dir<N, NGV, GV0, 1>(L, nb, sQ, sQo, sQn, sG, lnd[1][k], true);
              grad_dir<N, NGV, GV0, 2>(L, nb, sQ, sQo, sQn, sG, lnd[2][k], true);
            }
          if (M::kTail > 0 && tw < M::kTail) grad_dir<N, NGV, GV0, 3>(L, nb, sQ, sQo, sQn, sG, tl_ln, tl_ok, tl_d);
        }
      }
      // gradient DMMAs done: the helpers, who hold the first face fluxes in registers, may overwrite the neighbour traces.  The
      // chain warps only signal it (the chain rule and the first interpolations need nothing from the Rusanov pass) and
      // synchronise among themselves: the chain rule mixes the three directions' derivatives of every warp.
      if (!kPre) bar_arrive(kBarGrad, kMainThreads);
      bar_sync(kBarChain, CH);
      if constexpr (GRADV != 0) {
#pragma unroll
        for (int q = 0; q < P2; ++q) {
          const int s = tid + q * CH;
          if (s < I::n3) {
#pragma unroll
            for (int vv = 0; vv < NGV; ++vv) {
              const double g0 = sG[(vv * 3 + 0) * I::n3 + s], g1 = sG[(vv * 3 + 1) * I::n3 + s], g2 = sG[(vv * 3 + 2) * I::n3 + s];
#pragma unroll
              for (int p = 0; p < 3; ++p) sG[(vv * 3 + p) * I::n3 + s] = jv[q][p] * g0 + jv[q][3 + p] * g1 + jv[q][6 + p] * g2;
            }
          }
        }
      }
      bar_sync(kBarChain, CH);                  // the gradient is complete in shared memory
      if (kPre) bar_arrive(kBarGrad, kMainThreads);   // ... which the helpers' sources (div B) wait for
      if constexpr (M::kFree) {
        // ---- A1, A4, A5, A7: every task stores into the accumulator of its own direction; no barrier between tasks
#pragma unroll
        for (int t = 0; t < M::kTPW; ++t) {
          if (!fv[t]) continue;
          double* acc = fd[t] == 0 ? sR : sR12 + (fd[t] - 1) * kRS;
          if (t == 0) chain_dir<N, DIFF, 3, true, 1>(L, ph, nb, io, geo, e, sQ, sG, sFace, sS, acc, fl[t], fr[t], fd[t], tid);
          else chain_dir<N, DIFF, 3, false, 1>(L, ph, nb, io, geo, e, sQ, sG, sFace, sS, acc, fl[t], fr[t], fd[t]);
        }
      } else {
      // ---- A1, A4, A5, A7: one DMMA chain per warp and direction, directions separated by chain-warp barriers
        if (active) {
          chain_dir<N, DIFF, 0, true>(L, ph, nb, io, geo, e, sQ, sG, sQn, sS, sR, lnd[0][0], true, 0, tid);
#pragma unroll
          for (int k = 1; k < M::kTPD; ++k)
            if (warp + k * M::kWarps < M::FG) chain_dir<N, DIFF, 0>(L, ph, nb, io, geo, e, sQ, sG, sQn, sS, sR, lnd[0][k], true);
        } else {
          bar_sync(kBarFaces, kMainThreads);
        }
        {   // rounds 1, 2 and the tail round: the round barrier sits inside the warp's first task of the round
          bool first = true;
          if (active) {
#pragma unroll
            for (int k = 0; k < M::kTPD; ++k)
              if (warp + k * M::kWarps < M::FG) {
                if (k == 0) chain_dir<N, DIFF, 1, false, -1, 1>(L, ph, nb, io, geo, e, sQ, sG, sQn, sS, sR, lnd[1][k], true);
                else chain_dir<N, DIFF, 1>(L, ph, nb, io, geo, e, sQ, sG, sQn, sS, sR, lnd[1][k], true);
                first = false;
              }
          }
          if (first) bar_sync(kBarChain, CH);
          first = true;
          if (active) {
#pragma unroll
            for (int k = 0; k < M::kTPD; ++k)
              if (warp + k * M::kWarps < M::FG) {
                if (k == 0) chain_dir<N, DIFF, 2, false, -1, 1>(L, ph, nb, io, geo, e, sQ, sG, sQn, sS, sR, lnd[2][k], true);
                else chain_dir<N, DIFF, 2>(L, ph, nb, io, geo, e, sQ, sG, sQn, sS, sR, lnd[2][k], true);
                first = false;
              }
          }
          if (first) bar_sync(kBarChain, CH);
          if (M::kTail > 0) {   // left-over lines of the three directions: no two of them share a solution point
            if (active && tw < M::kTail) chain_dir<N, DIFF, 3, false, -1, 1>(L, ph, nb, io, geo, e, sQ, sG, sQn, sS, sR, tl_ln, tl_ok, tl_d);
            else bar_sync(kBarChain, CH);
          }
        }
      }
      bar_sync(kBarRes, kMainThreads);         // divergence accumulated: the helpers finish the element
    }
  } else {
    // =============================================== helper warps ==============================================
    if (RS::kHelp < RS::kLaunch) setmaxnreg_dec<RS::kHelp>();
    else if (RS::kHelp > RS::kLaunch) setmaxnreg_inc<RS::kHelp>();
    constexpr int P2 = (I::n3 + H - 1) / H;              // solution points per helper thread
    // connectivity of the element this CTA handles next, fetched one element ahead by helper threads 0..5
    int pn_e = 0, pn_f = 0, pn_o = 0;
    auto fetch_nbr = [&](int64_t el) {
      if (tid < 6 && el < E) {
        pn_e = geo.nbr_elem[el * 6 + tid];
        pn_f = geo.nbr_face[el * 6 + tid];
        pn_o = geo.nbr_orient[el * 6 + tid];
      }
    };
    // asynchronous load of one element's inputs: state, own traces, S^d, neighbour traces through the orientation map (A2)
    // part A: state, S^d and neighbour traces (their shared memory is dead as soon as the chains are done);
    // part B: own traces (their region doubles as the divergence accumulator sR, read by the final combination)
    auto issue_loads_a = [&](int64_t el, int set) {
      double* sQ = sm + set * kIn;
      double* sQn = kPre ? sQn1 : sQ + ev(9 * I::n3) + ev(kOwn);
      double* sS = kPre ? sQ + ev(9 * I::n3) + ev(kOwn) : sQn + ev(54 * I::n2);
      ElemNbr& nb = nbs[set];
      if (tid < 6) { nb.ne[tid] = pn_e; nb.nf[tid] = pn_f; nb.no[tid] = pn_o; }
      const double* q = io.Qe + el * 9 * I::n3;
      const double* g = kSintOrder(N) ? geo.Sint + el * kST : geo.Sfl + el * 9 * I::nf;
      if (kBulk) {
        if (tid < 32) {
          // neighbour faces that meet this element with the identity orientation (all faces inside a panel, most seam faces)
          // are contiguous 9 n^2 blocks in the same indexing: one bulk copy each, issued by the thread that holds the face
          const bool whole = tid < 6 && pn_e >= 0 && pn_o == 0;
          const unsigned cnt = __popc(__ballot_sync(0xffffffffu, whole));
          if (tid == 0) {
            fence_proxy_async();
            mbar_expect_tx(&mbar, (unsigned)(sizeof(double) * (9 * I::n3 + kST + cnt * 9 * I::n2)));
            tma_load(sQ, q, sizeof(double) * 9 * I::n3, &mbar);
          }
          if (whole) {
            if (tid != 0) fence_proxy_async();
            tma_load(sQn + tid * 9 * I::n2, io.Qf + ((int64_t)pn_e * 6 + pn_f) * 9 * I::n2, sizeof(double) * 9 * I::n2, &mbar);
          }
        } else if (tid == 32 && !kSglobal) {
          fence_proxy_async();
          tma_load(sS, g, sizeof(double) * kST, &mbar);
        }
      } else {
        for (int k = tid; k < 9 * I::n3; k += H) cp_async8(sQ + k, q + k);
        if (!kSglobal)
          for (int k = tid; k < kST / 2; k += H) cp_async16(sS + 2 * k, g + 2 * k);
      }
      bar_sync(kBarHelp, H);   // nb visible
      for (int k = tid; k < 6 * I::n2; k += H) {
        const int f = k / I::n2, ab = k % I::n2;
        const int ne = nb.ne[f];
        if (ne >= 0 && !(kBulk && nb.no[f] == 0)) {     // the other orientations: gathered point by point
          const double* src = io.Qf + (((int64_t)ne * 6 + nb.nf[f]) * 9) * I::n2 + I::orient(nb.no[f], ab);
#pragma unroll
          for (int v = 0; v < 9; ++v) cp_async8(sQn + (f * 9 + v) * I::n2 + ab, src + v * I::n2);
        }
      }
    };
    auto issue_loads_b = [&](int64_t el, int set) {
      double* sQo = sm + set * kIn + ev(9 * I::n3);
      const double* t = io.Qf + el * 54 * I::n2;
      if (kBulk) {
        if (tid == 64) {
          fence_proxy_async();
          mbar_expect_tx(&mbar, (unsigned)(sizeof(double) * 54 * I::n2));
          tma_load(sQo, t, sizeof(double) * 54 * I::n2, &mbar);
        }
      } else {
        for (int k = tid; k < 54 * I::n2; k += H) cp_async8(sQo + k, t + k);
      }
      cp_async_commit();
    };
    fetch_nbr(blockIdx.x);
    if ((int64_t)blockIdx.x < E) {
      issue_loads_a(blockIdx.x, 0);
      issue_loads_b(blockIdx.x, 0);
      fetch_nbr((int64_t)blockIdx.x + gridDim.x);
    }
    const bool rk = io.Qout != nullptr;
    const bool g0 = rk && io.A0 != nullptr, g1 = rk && io.A1 != nullptr;

    double K[P2][9], w[P2];                     // sources and Runge-Kutta registers of this thread's points (set beside the chains)
    auto finish = [&](int64_t ef, int setf) {   // out = w * (div_xi F~) + K for element ef, whose tiles are input set setf
      double* sQ = sm + setf * kIn;
      double* sR = sQ + ev(9 * I::n3);
#pragma unroll
      for (int q = 0; q < P2; ++q) {
        const int s = tid + q * H;
        if (s < I::n3) {
          double R[9];
#pragma unroll
          for (int v = 0; v < 9; ++v) {
            double dv;
            if (kPre) dv = sR12[v * I::n3 + s] + sR12[kRS + v * I::n3 + s];          // the accumulators of the two waves
            else if (M::kFree) dv = sR[v * I::n3 + s] + sR12[v * I::n3 + s] + sR12[kRS + v * I::n3 + s];   // one per direction
            else dv = sR[v * I::n3 + s];
            R[v] = w[q] * dv + K[q][v];
          }
          if (DIFF) {                    // finished by the face kernel
#pragma unroll
            for (int v = 0; v < 9; ++v) io.Part[(ef * 9 + v) * I::n3 + s] = R[v];
          } else if (rk) {
#pragma unroll
            for (int v = 0; v < 9; ++v) {
              io.Qout[(ef * 9 + v) * I::n3 + s] = R[v];
              (kChainTraces ? sNew : sQ)[v * I::n3 + s] = R[v];   // this thread is the only reader and writer of point s in this phase
            }
          } else {
#pragma unroll
            for (int v = 0; v < 9; ++v) io.Rout[((int64_t)v * E + ef) * I::n3 + s] = R[v];
          }
        }
      }
      if (!DIFF && rk && !kChainTraces) {
        bar_sync(kBarHelp, H);
        emit_traces<N>(sQ, io.QfOut + ef * 54 * I::n2, tid, H);
      }
      bar_sync(kBarHelp, H);                   // every helper is done with this element's shared memory
    };
    // A8 sources and the Runge-Kutta registers of element es (state tile sQ), so that  out = w * (div_xi F~) + K  is all that is left
    auto sources = [&](int64_t e, const double* sQ, const double* sG) {
#pragma unroll
      for (int q = 0; q < P2; ++q) {
        const int s = tid + q * H;
        const int sc = s < I::n3 ? s : 0;
        double Q[9];
#pragma unroll
        for (int v = 0; v < 9; ++v) Q[v] = sQ[v * I::n3 + sc];
        double divB = 0.0;
        if (GRADV == 2) divB = sG[15 * I::n3 + sc] + sG[19 * I::n3 + sc] + sG[23 * I::n3 + sc];
        if (GRADV == 1) divB = sG[0 * I::n3 + sc] + sG[4 * I::n3 + sc] + sG[8 * I::n3 + sc];
        {
          const PrimD p = primitives(ph, Q);
#pragma unroll
          for (int v = 0; v < 9; ++v) K[q][v] = 0.0;
          add_sources(ph, p, divB, geo.xsol[(e * 3 + 0) * I::n3 + sc], geo.xsol[(e * 3 + 1) * I::n3 + sc],
                      geo.xsol[(e * 3 + 2) * I::n3 + sc], K[q]);                                      // K = M (Eq. 5)
        }
        w[q] = -1.0 / geo.detJ[e * I::n3 + sc];              // R = w * div_xi F~ + M  (Eq. 16)
        if (rk) {                                            // step mode: out = cq Q + c0 A0 + c1 A1 + bdt R
          w[q] *= io.bdt;
#pragma unroll
          for (int v = 0; v < 9; ++v) K[q][v] = io.bdt * K[q][v] + io.cq * Q[v];
          if (g0) {
#pragma unroll
            for (int v = 0; v < 9; ++v) K[q][v] += io.c0 * io.A0[(e * 9 + v) * I::n3 + sc];
          }
          if (g1) {
#pragma unroll
            for (int v = 0; v < 9; ++v) K[q][v] += io.c1 * io.A1[(e * 9 + v) * I::n3 + sc];
          }
        }
      }
    };
    // kPre: walls and common inviscid fluxes of element el (input set `set`) an element ahead: the common SOLUTION (BR1 average
    // or wall state Q_b) replaces the neighbour traces, the common FLUX (Rusanov / wall, scaled by sigma |S|) the own traces
    auto face_pass = [&](int64_t el, int set) {
      double* sQo = sm + set * kIn + ev(9 * I::n3);
      double* sQn = kPre ? sQn1 : sQo + ev(kOwn);
      const ElemNbr& nb = nbs[set];
      for (int t = tid; t < 6 * I::n2; t += H) {
        const int f = t / I::n2, ab = t % I::n2;
        const double* nf_ = geo.nfc + (el * 6 + f) * 4 * I::n2 + ab;
        const double nx = nf_[0], ny = nf_[I::n2], nz = nf_[2 * I::n2], sa = nf_[3 * I::n2];
        double Qi[9], Qc[9], F[9];
#pragma unroll
        for (int v = 0; v < 9; ++v) Qi[v] = sQo[(f * 9 + v) * I::n2 + ab];
        if (nb.ne[f] >= 0) {
          double Qo[9];
#pragma unroll
          for (int v = 0; v < 9; ++v) Qo[v] = sQn[(f * 9 + v) * I::n2 + ab];
          flux_rusanov(ph, Qi, Qo, nx, ny, nz, F);
#pragma unroll
          for (int v = 0; v < 9; ++v) Qc[v] = 0.5 * Qi[v] + 0.5 * Qo[v];          // BR1
        } else {
          wall_state(ph, nb.ne[f], Qi, nx, ny, nz, Qc);
          const PrimD sb_ = primitives(ph, Qc);
          flux_inviscid<true>(ph, sb_, nx, ny, nz, F);
        }
#pragma unroll
        for (int v = 0; v < 9; ++v) {
          sQn[(f * 9 + v) * I::n2 + ab] = Qc[v];
          sQo[(f * 9 + v) * I::n2 + ab] = sa * F[v];
        }
      }
    };
    unsigned ld_phase = 0;
    int it = 0;
    int64_t e_last = -1;
    if constexpr (kPre) {
      // ---- two input sets: everything the chain warps need of element e -- inputs, wall states, common fluxes -- is made
      //      while they work on element e - 1; the finish of e - 1 happens after e has been handed over
      if ((int64_t)blockIdx.x < E) {
        cp_async_wait_all();
        mbar_wait(&mbar, ld_phase);
        ld_phase ^= 1u;
        bar_sync(kBarHelp, H);
        face_pass(blockIdx.x, 0);
        bar_sync(kBarIn, kMainThreads);              // the first element is handed over: inputs, common solution, common fluxes
      }
      for (int64_t e = blockIdx.x; e < E; e += gridDim.x, ++it) {
        const int cur = it & 1;
        const bool more = e + gridDim.x < E;
        e_last = e;
        // The chain warps are done with the previous element (RES): its input set is free, and its finish touches no input tile
        // (it reads the accumulators and writes global memory, without diffusion also sNew).  With diffusion the next loads go
        // first, so that the proxy fence of their issuing threads does not wait for the finish's global stores (the chain warps
        // need the accumulators only after the streamed viscous flux of their first task); without it the chain warps need them
        // almost at once, and the finish goes first.  The single neighbour tile is free as well: the chain warps report RES after
        // the gradient tasks that read it -- except before the first element, whose gradient is awaited here.
        if (it == 0) bar_sync(kBarGrad, kMainThreads);
        if (DIFF && more) {
          issue_loads_a(e + gridDim.x, cur ^ 1);
          issue_loads_b(e + gridDim.x, cur ^ 1);
          fetch_nbr(e + 2 * (int64_t)gridDim.x);
        }
        if (it > 0) finish(e - gridDim.x, cur ^ 1);  // previous element: reads the accumulators
        bar_arrive(kBarFaces, kMainThreads);         // the accumulators are free for this element's chains
        if (!DIFF && more) {
          issue_loads_a(e + gridDim.x, cur ^ 1);
          issue_loads_b(e + gridDim.x, cur ^ 1);
          fetch_nbr(e + 2 * (int64_t)gridDim.x);
        }
        if (e + 2 * (int64_t)gridDim.x < E) prefetch_next<N, GRADV>(io, geo, e + 2 * (int64_t)gridDim.x, pn_e, pn_f, tid, H);
        if (more) {
          cp_async_wait_all();
          mbar_wait(&mbar, ld_phase);
          ld_phase ^= 1u;
          bar_sync(kBarHelp, H);
          face_pass(e + gridDim.x, cur ^ 1);
        }
        if (it > 0) bar_sync(kBarGrad, kMainThreads);   // the gradient of e is complete (the chain warps arrived an element ago)
        if (more) bar_arrive(kBarNext, H + 32 * (M::kFreeWarps - (M::kTasks - M::kFreeWarps)));   // next element handed over
        sources(e, sm + cur * kIn, sG + cur * kGS);
        bar_sync(kBarRes, kMainThreads);             // every chain warp is done with element e
      }
      if (e_last >= 0) {
        finish(e_last, (it - 1) & 1);
        if (kChainTraces && rk) bar_arrive(kBarIn, kMainThreads);      // the chain warps make the last element's traces
      }
    } else

    for (int64_t e = blockIdx.x; e < E; e += gridDim.x, ++it) {
      const int cur = kPre ? (it & 1) : 0;
      double* sQ = sm + cur * kIn;
      double* sQo = sQ + ev(9 * I::n3);
      double* sQn = sQo + ev(kOwn);
      e_last = e;
      const ElemNbr& nb = nbs[cur];
      const bool more = e + gridDim.x < E;
      cp_async_wait_all();
      if (kBulk) mbar_wait(&mbar, ld_phase);   // the bulk copies have landed ...
      ld_phase ^= 1u;
      bar_sync(kBarHelp, H);                   // ... and every helper's gathered copies
      for (int t = tid; t < 6 * I::n2; t += H) {     // wall faces: the boundary state Q_b takes the neighbour's place
        const int f = t / I::n2, ab = t % I::n2;
        const int ne = nb.ne[f];
        if (ne < 0) {
          double own[9], out[9];
#pragma unroll
          for (int v = 0; v < 9; ++v) own[v] = sQo[(f * 9 + v) * I::n2 + ab];
          const double* nf_ = geo.nfc + ((e * 6 + f) * 4) * I::n2 + ab;
          wall_state(ph, ne, own, nf_[0], nf_[I::n2], nf_[2 * I::n2], out);
#pragma unroll
          for (int v = 0; v < 9; ++v) sQn[(f * 9 + v) * I::n2 + ab] = out[v];
        }
      }
      bar_sync(kBarIn, kMainThreads);

      // ---- A6: common INVISCID fluxes at the 6 n^2 face points (Rusanov / wall), scaled by sigma |S|.  They replace the
      //      neighbour traces in sQn, which the gradient is still reading: computed now, stored after the GRAD barrier.
      auto face_flux = [&](int t, double* F) {
        const int f = t / I::n2, ab = t % I::n2;
        const double* nf_ = geo.nfc + (e * 6 + f) * 4 * I::n2 + ab;
        const double nx = nf_[0], ny = nf_[I::n2], nz = nf_[2 * I::n2], sa = nf_[3 * I::n2];
        double Qo[9];
#pragma unroll
        for (int v = 0; v < 9; ++v) Qo[v] = sQn[(f * 9 + v) * I::n2 + ab];
        if (nb.ne[f] >= 0) {
          double Qi[9];
#pragma unroll
          for (int v = 0; v < 9; ++v) Qi[v] = sQo[(f * 9 + v) * I::n2 + ab];
          flux_rusanov(ph, Qi, Qo, nx, ny, nz, F);
        } else {
          const PrimD sb_ = primitives(ph, Qo);          // Qo holds the wall state Q_b
          flux_inviscid<true>(ph, sb_, nx, ny, nz, F);
        }
#pragma unroll
        for (int v = 0; v < 9; ++v) F[v] *= sa;
      };
      {
        double Ff[9];                              // one face point per helper thread beside the gradient DMMAs ...
        if (tid < 6 * I::n2) face_flux(tid, Ff);
        bar_sync(kBarGrad, kMainThreads);
        if (tid < 6 * I::n2) {
          const int f = tid / I::n2, ab = tid % I::n2;
#pragma unroll
          for (int v = 0; v < 9; ++v) sQn[(f * 9 + v) * I::n2 + ab] = Ff[v];
        }
        for (int t = tid + H; t < 6 * I::n2; t += H) {   // ... the rest beside the chain rule, in place (own face point only)
          double F[9];
          face_flux(t, F);
          const int f = t / I::n2, ab = t % I::n2;
#pragma unroll
          for (int v = 0; v < 9; ++v) sQn[(f * 9 + v) * I::n2 + ab] = F[v];
        }
      }
      bar_sync(kBarFaces, kMainThreads);

      if constexpr (DIFF && kFaceOutOrder(N)) {
        // Own-side viscous flux at the 3 n^2 points of the faces m = 0 (not in the chains' tiles): Q and grad Q interpolated to the
        // face point (Eq. 19), evaluated on Q_in (interior face) or on the wall state Q_b, along the outward unit normal.  The
        // gradient is complete: the chain warps reached FACES after their chain rule.
        const OpsC& op = c_ops[N];
        for (int t = tid; t < 3 * I::n2; t += H) {
          const int d = t / I::n2, ab = t % I::n2, f = 2 * d;
          const int st = I::stride(d), sb = I::sbase(d, ab);
          // The lines of a warp's 32 face points start 8 or 64 doubles apart: read in the same order they would meet in two
          // (direction 0) or eight (direction 1) shared-memory banks.  Each lane walks its line from its own starting point
          // instead (l = (j + rot) mod 8), which spreads a half-warp over all 32 banks.
          static_assert(N == 8, "bank rotation written for n = 8");
          const int rot = d == 0 ? ((((ab & 7) >> 1) + 4 * ((ab >> 3) & 1)) & 7) : d == 1 ? ((ab >> 3) & 1) : 0;
          double wI[N];
          int lo[N];
#pragma unroll
          for (int j = 0; j < N; ++j) {
            const int l = (j + rot) & 7;
            wI[j] = op.Isf[((f & 1) ? N * N : 0) + l];
            lo[j] = sb + l * st;
          }
          double q[9];
#pragma unroll
          for (int v = 0; v < 9; ++v) {
            double a = 0.0;
#pragma unroll
            for (int j = 0; j < N; ++j) a += wI[j] * sQ[v * I::n3 + lo[j]];
            q[v] = a;
          }
          const double* nf_ = geo.nfc + ((e * 6 + f) * 4) * I::n2 + ab;
          const double nx = nf_[0], ny = nf_[I::n2], nz = nf_[2 * I::n2];
          const int ne = nb.ne[f];
          if (ne < 0) {
            double qb[9];
            wall_state(ph, ne, q, nx, ny, nz, qb);
#pragma unroll
            for (int v = 0; v < 9; ++v) q[v] = qb[v];
          }
          const PrimD p = primitives(ph, q);
          VStream vs;
#define CHORUS_FACE_VAR(V)                                                              \
  {                                                                                     \
    double g0 = 0.0, g1 = 0.0, g2 = 0.0;                                                \
    const double* G = sG + (3 * (V)) * I::n3;                                           \
    _Pragma("unroll") for (int j = 0; j < N; ++j) {                                     \
      const double wl = wI[j];                                                          \
      g0 += wl * G[lo[j]];                                                              \
      g1 += wl * G[I::n3 + lo[j]];                                                      \
      g2 += wl * G[2 * I::n3 + lo[j]];                                                  \
    }                                                                                   \
    vs_fold<V>(vs, p, nx, ny, nz, g0, g1, g2);                                          \
  }
          CHORUS_FACE_VAR(0) CHORUS_FACE_VAR(1) CHORUS_FACE_VAR(2) CHORUS_FACE_VAR(3) CHORUS_FACE_VAR(4)
          CHORUS_FACE_VAR(5) CHORUS_FACE_VAR(6) CHORUS_FACE_VAR(7) CHORUS_FACE_VAR(8)
#undef CHORUS_FACE_VAR
          const double kr = geo.krfl ? geo.krfl[(e * 3 + d) * I::nf + I::fbase(d, ab) + ((f & 1) ? N : 0) * st] : 0.0;
          double Fv[7];
          if (ne < 0) vs_flux_wall(ph, ne, vs, p, nx, ny, nz, kr, Fv);
          else vs_flux(ph, vs, p, nx, ny, nz, kr, Fv);
          double* o = io.Vf + ((e * 6 + f) * 7) * I::n2 + ab;
#pragma unroll
          for (int k = 0; k < 7; ++k) o[k * I::n2] = Fv[k];
        }
      }
      sources(e, sQ, sG);                      // beside the chains
      // measured: -0.9k cycles of the 6.2k the chain warps wait for the next element's inputs
      if (e + (kPre ? 2 : 1) * (int64_t)gridDim.x < E)
        prefetch_next<N, GRADV>(io, geo, e + (kPre ? 2 : 1) * (int64_t)gridDim.x, pn_e, pn_f, tid, H);
      bar_sync(kBarRes, kMainThreads);

      // ---- A9: finish the element.  The next element's state, metrics and neighbour traces start streaming in first
      //      (except when this element's new state still has to pass through sQ for its traces).  With two input sets the
      //      finish is deferred until the NEXT element's inputs have been handed to the chain warps (top of the loop).
      constexpr bool kEarlyLoads = DIFF;
      if (!kPre && kEarlyLoads && more) issue_loads_a(e + gridDim.x, 0);
      if (!kPre) finish(e, 0);
      if (!kPre && more) {
        if (!kEarlyLoads) issue_loads_a(e + gridDim.x, 0);
        issue_loads_b(e + gridDim.x, 0);
        fetch_nbr(e + 2 * (int64_t)gridDim.x);
      }
    }

  }
}

template <int N, int GRADV>
constexpr size_t stage_main_smem_bytes() {
  using I = Ix<N>;
  constexpr int NGV = GRADV == 2 ? 9 : GRADV == 1 ? 3 : 0;
  constexpr int kOwn = 54 * I::n2 > 9 * I::n3 ? 54 * I::n2 : 9 * I::n3;
  constexpr auto ev = [](int x) { return (x + 1) & ~1; };
  constexpr int kST = kSglobalOrder(N) ? 0 : kSintOrder(N) ? 9 * I::n2 * (N - 1) : 9 * I::nf;
  if (kPrefetchOrder(N))   // two sets of (state, own traces / fluxes, S^d), one neighbour tile, two gradients, two accumulators
    return sizeof(double) * (size_t)(2 * (ev(9 * I::n3) + ev(kOwn) + kST) + ev(54 * I::n2) + 2 * ev(3 * NGV * I::n3) + 2 * ev(9 * I::n3) +
                                     (GRADV != 2 ? ev(9 * I::n3) : 0));      // without diffusion: the new-state tile sNew
  return sizeof(double) * (size_t)((kPrefetchOrder(N) ? 2 : 1) * (ev(9 * I::n3) + ev(kOwn) + ev(54 * I::n2) + kST) +
                                   (kPrefetchOrder(N) ? 2 : 1) * ev(3 * NGV * I::n3) + (Mma<N>::kFree ? 2 * ev(9 * I::n3) : 0));
}

// ---------------------------------------------------------------------------------------------------------
// stage_face_kernel (diffusion): value = Part + scale/|J| * sum_faces l'_{m_f}(X_s,i) sigma_f |S_f| Fv_common,
//   Fv_common = 1/2 (own - neighbour's along its own, opposite, normal)  on interior faces, the wall flux on walls
//   (R = -(1/|J|) div_xi F~ and the viscous part of F~ at a face point is sigma |S| (-Fv_common); Eq. 16).
// scale = bdt (step mode: Part is the new state, finished in place, and its face traces are emitted) or 1 (residual
// mode: written to Rout in the interface layout).
// ---------------------------------------------------------------------------------------------------------
template <int N>
__global__ void __launch_bounds__(256) stage_face_kernel(int64_t E, StageIO io, Geo geo) {
  using I = Ix<N>;
  extern __shared__ double sm[];
  double* sP = sm;                    // [9][n3]
  double* sV = sP + 9 * I::n3;        // [6][7][n2]  sigma |S| Fv_common
  __shared__ ElemNbr nb;
  const OpsC& op = c_ops[N];
  const bool step = io.Qout != nullptr;
  const double scale = step ? io.bdt : 1.0;
  for (int64_t e = blockIdx.x; e < E; e += gridDim.x) {
    __syncthreads();
    load_nbr(nb, e, geo.nbr_elem, geo.nbr_face, geo.nbr_orient);
    for (int t = threadIdx.x; t < 9 * I::n3; t += blockDim.x) sP[t] = io.Part[e * 9 * I::n3 + t];
    __syncthreads();
    for (int t = threadIdx.x; t < 6 * I::n2; t += blockDim.x) {
      const int f = t / I::n2, ab = t % I::n2;
      const double sa = geo.nfc[((e * 6 + f) * 4 + 3) * I::n2 + ab];
      const int ne = nb.ne[f];
      const double* mine = io.Vf + ((e * 6 + f) * 7) * I::n2 + ab;
      if (ne >= 0) {
        const int ab2 = I::orient(nb.no[f], ab);
        const double* theirs = io.Vf + (((int64_t)ne * 6 + nb.nf[f]) * 7) * I::n2 + ab2;
#pragma unroll
        for (int k = 0; k < 7; ++k) sV[(f * 7 + k) * I::n2 + ab] = sa * (0.5 * (mine[k * I::n2] - theirs[k * I::n2]));
      } else {
#pragma unroll
        for (int k = 0; k < 7; ++k) sV[(f * 7 + k) * I::n2 + ab] = sa * mine[k * I::n2];
      }
    }
    __syncthreads();
    for (int s = threadIdx.x; s < I::n3; s += blockDim.x) {
      const int i = s % N, j = (s / N) % N, k = s / I::n2;
      const double w = scale / geo.detJ[e * I::n3 + s];
      const int ab0 = k * N + j, ab1 = k * N + i, ab2 = j * N + i;      // face point of the xi-, eta-, zeta-line through s
      const double d00 = op.Dfs[i * (N + 1)], d01 = op.Dfs[i * (N + 1) + N];
      const double d10 = op.Dfs[j * (N + 1)], d11 = op.Dfs[j * (N + 1) + N];
      const double d20 = op.Dfs[k * (N + 1)], d21 = op.Dfs[k * (N + 1) + N];
#pragma unroll
      for (int c = 0; c < 7; ++c) {
        const double div = d00 * sV[(0 * 7 + c) * I::n2 + ab0] + d01 * sV[(1 * 7 + c) * I::n2 + ab0] +
                           d10 * sV[(2 * 7 + c) * I::n2 + ab1] + d11 * sV[(3 * 7 + c) * I::n2 + ab1] +
                           d20 * sV[(4 * 7 + c) * I::n2 + ab2] + d21 * sV[(5 * 7 + c) * I::n2 + ab2];
        sP[(1 + c) * I::n3 + s] += w * div;
      }
      if (step) {
#pragma unroll
        for (int v = 0; v < 9; ++v) io.Qout[(e * 9 + v) * I::n3 + s] = sP[v * I::n3 + s];
      } else {
#pragma unroll
        for (int v = 0; v < 9; ++v) io.Rout[((int64_t)v * E + e) * I::n3 + s] = sP[v * I::n3 + s];
      }
    }
    if (step) {
      __syncthreads();
      emit_traces<N>(sP, io.QfOut + e * 54 * I::n2, threadIdx.x, blockDim.x);
    }
  }
}

template <int N>
constexpr size_t stage_face_smem_bytes() {
  using I = Ix<N>;
  return sizeof(double) * (size_t)(9 * I::n3 + 42 * I::n2);
}

}  // namespace chorus
