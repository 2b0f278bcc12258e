// kernels_stage.cuh -- the production pipeline of one residual evaluation / Runge-Kutta stage (orders 4..7).
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

template <int N>
struct Mma {
  static_assert(N >= 4 && N <= 7, "DMMA chain kernel: orders 4..7");
  using I = Ix<N>;
  static constexpr int kGroups = (I::n2 + 7) / 8;      // line groups per direction
  static constexpr int kWarps = kGroups;               // one warp per group
  static constexpr int kThreads = 32 * kWarps;
  // column j of the 8-wide tile -> flux point index m, or -1 (padding).
  // interior points first; the two face points share the SECOND column of their thread pairs so that one divergent
  // pass serves both (cols 2c+1 of the last two thread columns that hold anything).
  __device__ __forceinline__ static int col_m(int j) {
    // 4 bits per column, value m + 1 (0 = padding).  N = 4: {1,2,3,0,-,4,-,-}; 5: {1,2,3,4,-,0,-,5}; 6: {1,2,3,4,5,0,-,6};
    // 7: {1,2,3,4,5,0,6,7}
    constexpr uint32_t tbl = N == 4 ? 0x00501432u : N == 5 ? 0x60105432u : N == 6 ? 0x70165432u : 0x87165432u;
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
  double* Qout;          // new state (step mode), or nullptr:  Qout = c0*A0 + c1*A1 + c2*A2 + bdt * R
  double* QfOut;         // face traces of Qout (step mode)
  const double* A0;      // stage registers; a null pointer contributes nothing
  const double* A1;
  const double* A2;
  double c0, c1, c2, bdt;
};

struct Geo {
  const double* Sfl;     // [E][3 fam][3 comp][nf]
  const double* detJ;    // [E][n3]
  const double* jinv;    // [E][3 d][3 p][n3]
  const double* xsol;    // [E][3][n3]
  const double* krfl;    // [E][3 fam][nf] or nullptr
  const int32_t* nbr_elem;
  const uint8_t* nbr_face;
  const uint8_t* nbr_orient;
};

// Face traces of the element-resident state sQ [9][n3] -> Qf_e [6][9][n2]  (A1 restricted to the faces; Eq. 19, 21)
template <int N>
__device__ __forceinline__ void emit_traces(const double* sQ, double* __restrict__ Qf_e) {
  using I = Ix<N>;
  const OpsC& op = c_ops[N];
  for (int t = threadIdx.x; t < 3 * 9 * I::n2; t += blockDim.x) {
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
  const double ir = 1.0 / p.rho;
  const double grS = Sx * s.gr0 + Sy * s.gr1 + Sz * s.gr2;
  const double uS = p.u * Sx + p.v * Sy + p.w * Sz;
  const double mu = p.rho * ph.nu;
  const double divu = (s.divm - (p.u * s.gr0 + p.v * s.gr1 + p.w * s.gr2)) * ir;
  const double lam = -(2.0 / 3.0) * mu * divu;                                     // Stokes
  const double mi = mu * ir;
  t0 = mi * ((s.mS0 - p.u * grS) + (s.W0 - uS * s.gr0)) + lam * Sx;                // Eq. 8 contracted with S
  t1 = mi * ((s.mS1 - p.v * grS) + (s.W1 - uS * s.gr1)) + lam * Sy;
  t2 = mi * ((s.mS2 - p.w * grS) + (s.W2 - uS * s.gr2)) + lam * Sz;
  const double u2 = p.u * p.u + p.v * p.v + p.w * p.w;
  const double dpS = ph.gm1 * (s.acc - (p.u * s.mS0 + p.v * s.mS1 + p.w * s.mS2) + 0.5 * u2 * grS);
  const double Tt = p.p * ir / ph.R;
  const double dTS = (dpS - p.p * ir * grS) * ir / ph.R;
  const double dSS = ph.Cp * (dpS / (ph.gamma * p.p) - grS * ir);                  // gradient of Eq. 10
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

#ifndef CHORUS_MAIN_MINBLOCKS
#define CHORUS_MAIN_MINBLOCKS 2
#endif

// GRADV: 0 no gradient needed, 1 gradient of B only (Powell sources without diffusion), 2 all nine variables.
template <int N, bool DIFF, int GRADV>
__global__ void __launch_bounds__(Mma<N>::kThreads, CHORUS_MAIN_MINBLOCKS)
stage_main_kernel(int64_t E, PhysD ph, StageIO io, Geo geo) {
  using I = Ix<N>;
  using M = Mma<N>;
  static_assert(!DIFF || GRADV == 2, "diffusion needs the gradient of all variables");
  constexpr int NGV = GRADV == 2 ? 9 : GRADV == 1 ? 3 : 0;
  constexpr int GV0 = GRADV == 1 ? 5 : 0;
  extern __shared__ double sm[];
  double* sQ = sm;                       // [9][n3]
  constexpr int kOwn = 54 * I::n2 > 9 * I::n3 ? 54 * I::n2 : 9 * I::n3;
  double* sQo = sQ + 9 * I::n3;          // [6][9][n2] own traces; the region is reused as sR [9][n3] after the face pass
  double* sQn = sQo + kOwn;              // [6][9][n2] neighbour traces / wall states; overwritten by the face fluxes
  double* sG = sQn + 54 * I::n2;         // [3*NGV][n3]
  double* sR = sQo;
  __shared__ ElemNbr nb;
  const OpsC& op = c_ops[N];
  const int lane = threadIdx.x & 31, r = lane >> 2, c = lane & 3, warp = threadIdx.x >> 5;

  // ---- per-lane operator fragments (B operands), fixed for the whole kernel
  // interpolation: B[k = l][n = col r] = h_l(X_f,m(r));  k-step s covers l = 4s + c
  const int mB = M::col_m(r);
  double bI0 = 0.0, bI1 = 0.0;
  if (mB >= 0) {
    bI0 = op.Isf[mB * N + c];
    if (4 + c < N) bI1 = op.Isf[mB * N + 4 + c];
  }
  // derivative: B[k = col][n = l_out r] = l'_{m(col)}(X_s,l_out);  k-step s covers col = 2c + s  (the C -> A reuse)
  const int m0 = M::col_m(2 * c), m1 = M::col_m(2 * c + 1);
  double bD0 = 0.0, bD1 = 0.0;
  if (r < N) {
    if (m0 >= 0) bD0 = op.Dfs[r * (N + 1) + m0];
    if (m1 >= 0) bD1 = op.Dfs[r * (N + 1) + m1];
  }
  // BR1 gradient: x = (q_0..q_{N-1}, common value at m = 0, at m = N), K = N + 2 -> up to 3 k-steps of 4
  // B[k][n = l_out r]: k < N: Dss[l_out][k]; k = N: Dfs[l_out][0]; k = N+1: Dfs[l_out][N]
  double bG[3] = {0.0, 0.0, 0.0};
  if (r < N) {
#pragma unroll
    for (int s = 0; s < 3; ++s) {
      const int k = 4 * s + c;
      if (k < N) bG[s] = op.Dss[r * N + k];
      else if (k == N) bG[s] = op.Dfs[r * (N + 1)];
      else if (k == N + 1) bG[s] = op.Dfs[r * (N + 1) + N];
    }
  }
  constexpr int KG = (N + 2 + 3) / 4;    // k-steps of the gradient product

  for (int64_t e = blockIdx.x; e < E; e += gridDim.x) {
    __syncthreads();
    load_nbr(nb, e, geo.nbr_elem, geo.nbr_face, geo.nbr_orient);
    for (int t = threadIdx.x; t < 9 * I::n3; t += blockDim.x) sQ[t] = io.Qe[e * 9 * I::n3 + t];
    __syncthreads();
    const double* Sfl_e = geo.Sfl + e * 9 * I::nf;
    stage_traces<N>(e, nb, ph, io.Qf, Sfl_e, sQo, sQn);
    __syncthreads();

    // ---- A3: BR1 gradient.  d/dxi_d by DMMA (warp = line group, all directions), then the chain rule per point.
    if constexpr (GRADV != 0) {
      const int line = warp * 8 + r;
      const bool lv = line < I::n2;
      const int ln = lv ? line : 0;
#pragma unroll 1
      for (int d = 0; d < 3; ++d) {
        const int st = I::stride(d), sb = I::sbase(d, ln);
        const int f0 = 2 * d, f1 = 2 * d + 1;
        const bool w0 = nb.ne[f0] < 0, w1 = nb.ne[f1] < 0;
#pragma unroll
        for (int vv = 0; vv < NGV; ++vv) {
          const int v = GV0 + vv;
          double d0 = 0.0, d1 = 0.0;
#pragma unroll
          for (int s = 0; s < KG; ++s) {
            const int k = 4 * s + c;
            double a = 0.0;
            if (k < N) a = sQ[v * I::n3 + sb + k * st];
            else if (k == N) {
              const double o = sQo[(f0 * 9 + v) * I::n2 + ln], nn = sQn[(f0 * 9 + v) * I::n2 + ln];
              a = w0 ? nn : 0.5 * (o + nn);
            } else if (k == N + 1) {
              const double o = sQo[(f1 * 9 + v) * I::n2 + ln], nn = sQn[(f1 * 9 + v) * I::n2 + ln];
              a = w1 ? nn : 0.5 * (o + nn);
            }
            dmma884(d0, d1, a, bG[s]);
          }
          if (lv) {
            if (2 * c < N) sG[(vv * 3 + d) * I::n3 + sb + (2 * c) * st] = d0;
            if (2 * c + 1 < N) sG[(vv * 3 + d) * I::n3 + sb + (2 * c + 1) * st] = d1;
          }
        }
      }
      __syncthreads();
      for (int s = threadIdx.x; s < I::n3; s += blockDim.x) {
        double j[9];
#pragma unroll
        for (int k = 0; k < 9; ++k) j[k] = geo.jinv[e * 9 * I::n3 + k * I::n3 + s];
#pragma unroll
        for (int vv = 0; vv < NGV; ++vv) {
          const double g0 = sG[(vv * 3 + 0) * I::n3 + s], g1 = sG[(vv * 3 + 1) * I::n3 + s], g2 = sG[(vv * 3 + 2) * I::n3 + s];
#pragma unroll
          for (int p = 0; p < 3; ++p) sG[(vv * 3 + p) * I::n3 + s] = j[p] * g0 + j[3 + p] * g1 + j[6 + p] * g2;
        }
      }
    }

    // ---- A6: common INVISCID fluxes at the 6 n^2 face points (Rusanov / wall), scaled by sigma |S|, in place over sQn
    for (int t = threadIdx.x; t < 6 * I::n2; t += blockDim.x) {
      const int f = t / I::n2, ab = t % I::n2;
      double nx, ny, nz, area, sg;
      face_normal<N>(Sfl_e, f, ab, nx, ny, nz, area, sg);
      double Qo[9], F[9];
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
      const double sa = sg * area;
#pragma unroll
      for (int v = 0; v < 9; ++v) sQn[(f * 9 + v) * I::n2 + ab] = sa * F[v];
    }
    __syncthreads();   // own traces (sQo) are dead from here on: the region becomes the divergence accumulator sR

    // ---- A1, A4, A5, A7: one DMMA chain per warp and direction
    {
      const int line = warp * 8 + r;
      const bool lv = line < I::n2;
      const int ln = lv ? line : 0;
#pragma unroll 1
      for (int d = 0; d < 3; ++d) {
        const int st = I::stride(d), sb = I::sbase(d, ln);
        // A1: Q at the two flux points of this thread
        double q0[9], q1[9];
#pragma unroll
        for (int v = 0; v < 9; ++v) {
          const double a0 = sQ[v * I::n3 + sb + c * st];
          const double a1 = (4 + c < N) ? sQ[v * I::n3 + sb + (4 + c) * st] : 0.0;
          q0[v] = 0.0; q1[v] = 0.0;
          dmma884(q0[v], q1[v], a0, bI0);
          if (N > 4) dmma884(q0[v], q1[v], a1, bI1);
        }
        // per-slot setup: area vector and the state the fluxes are evaluated on
        const bool int0 = m0 > 0 && m0 < N, int1 = m1 > 0 && m1 < N;
        const bool face0 = m0 == 0 || m0 == N, face1 = m1 == 0 || m1 == N;     // m = -1: padding
        double S0x = 0.0, S0y = 0.0, S0z = 0.0, S1x = 0.0, S1y = 0.0, S1z = 0.0, kr0 = 0.0, kr1 = 0.0;
        int fc0 = 0, fc1 = 0;
        if (int0) {
          const int ix = I::fbase(d, ln) + m0 * st;
          S0x = Sfl_e[(d * 3 + 0) * I::nf + ix]; S0y = Sfl_e[(d * 3 + 1) * I::nf + ix]; S0z = Sfl_e[(d * 3 + 2) * I::nf + ix];
          if (DIFF && geo.krfl) kr0 = geo.krfl[(e * 3 + d) * I::nf + ix];
        }
        if (int1) {
          const int ix = I::fbase(d, ln) + m1 * st;
          S1x = Sfl_e[(d * 3 + 0) * I::nf + ix]; S1y = Sfl_e[(d * 3 + 1) * I::nf + ix]; S1z = Sfl_e[(d * 3 + 2) * I::nf + ix];
          if (DIFF && geo.krfl) kr1 = geo.krfl[(e * 3 + d) * I::nf + ix];
        }
        if (DIFF) {   // face columns: the own-side viscous flux along the outward unit normal, on Q_in (interior) or Q_b (wall)
          if (face0) {
            fc0 = 2 * d + (m0 == N ? 1 : 0);
            double area, sg;
            face_normal<N>(Sfl_e, fc0, ln, S0x, S0y, S0z, area, sg);
            if (geo.krfl) kr0 = geo.krfl[(e * 3 + d) * I::nf + I::fbase(d, ln) + m0 * st];
            if (nb.ne[fc0] < 0) {
              double qb[9];
              wall_state(ph, nb.ne[fc0], q0, S0x, S0y, S0z, qb);
#pragma unroll
              for (int v = 0; v < 9; ++v) q0[v] = qb[v];
            }
          }
          if (face1) {
            fc1 = 2 * d + (m1 == N ? 1 : 0);
            double area, sg;
            face_normal<N>(Sfl_e, fc1, ln, S1x, S1y, S1z, area, sg);
            if (geo.krfl) kr1 = geo.krfl[(e * 3 + d) * I::nf + I::fbase(d, ln) + m1 * st];
            if (nb.ne[fc1] < 0) {
              double qb[9];
              wall_state(ph, nb.ne[fc1], q1, S1x, S1y, S1z, qb);
#pragma unroll
              for (int v = 0; v < 9; ++v) q1[v] = qb[v];
            }
          }
        }
        PrimD p0, p1;
        if (DIFF || int0) p0 = primitives(ph, q0);
        if (DIFF || int1) p1 = primitives(ph, q1);
        double Fv0[7], Fv1[7];
        if (DIFF) {
          // A4 + Eq. 7-10: stream the gradients of the nine variables through the tensor core, three components at a time
          VStream s0, s1;
#define CHORUS_STREAM_VAR(V)                                                                            \
  {                                                                                                     \
    double ga0 = 0.0, ga1 = 0.0, gb0 = 0.0, gb1 = 0.0, gc0 = 0.0, gc1 = 0.0;                              \
    const double* gp = sG + (3 * (V)) * I::n3 + sb + c * st;                                            \
    dmma884(ga0, ga1, gp[0], bI0);                                                                      \
    dmma884(gb0, gb1, gp[I::n3], bI0);                                                                  \
    dmma884(gc0, gc1, gp[2 * I::n3], bI0);                                                              \
    if (N > 4) {                                                                                        \
      const bool hi = 4 + c < N;                                                                        \
      dmma884(ga0, ga1, hi ? gp[4 * st] : 0.0, bI1);                                                    \
      dmma884(gb0, gb1, hi ? gp[I::n3 + 4 * st] : 0.0, bI1);                                            \
      dmma884(gc0, gc1, hi ? gp[2 * I::n3 + 4 * st] : 0.0, bI1);                                        \
    }                                                                                                   \
    vs_fold<V>(s0, p0, S0x, S0y, S0z, ga0, gb0, gc0);                                                   \
    vs_fold<V>(s1, p1, S1x, S1y, S1z, ga1, gb1, gc1);                                                   \
  }
          CHORUS_STREAM_VAR(0) CHORUS_STREAM_VAR(1) CHORUS_STREAM_VAR(2) CHORUS_STREAM_VAR(3) CHORUS_STREAM_VAR(4)
          CHORUS_STREAM_VAR(5) CHORUS_STREAM_VAR(6) CHORUS_STREAM_VAR(7) CHORUS_STREAM_VAR(8)
#undef CHORUS_STREAM_VAR
          // slot 0
          if (face0 && nb.ne[fc0] < 0) vs_flux_wall(ph, nb.ne[fc0], s0, p0, S0x, S0y, S0z, kr0, Fv0);
          else vs_flux(ph, s0, p0, S0x, S0y, S0z, kr0, Fv0);
          if (face1 && nb.ne[fc1] < 0) vs_flux_wall(ph, nb.ne[fc1], s1, p1, S1x, S1y, S1z, kr1, Fv1);
          else vs_flux(ph, s1, p1, S1x, S1y, S1z, kr1, Fv1);
          if (lv) {
            if (face0) {
              double* o = io.Vf + ((e * 6 + fc0) * 7) * I::n2 + ln;
#pragma unroll
              for (int k = 0; k < 7; ++k) o[k * I::n2] = Fv0[k];
            }
            if (face1) {
              double* o = io.Vf + ((e * 6 + fc1) * 7) * I::n2 + ln;
#pragma unroll
              for (int k = 0; k < 7; ++k) o[k * I::n2] = Fv1[k];
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
          const int f = 2 * d + (m0 == N ? 1 : 0);
#pragma unroll
          for (int v = 0; v < 9; ++v) q0[v] = sQn[(f * 9 + v) * I::n2 + ln];
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
          const int f = 2 * d + (m1 == N ? 1 : 0);
#pragma unroll
          for (int v = 0; v < 9; ++v) q1[v] = sQn[(f * 9 + v) * I::n2 + ln];
        } else {
#pragma unroll
          for (int v = 0; v < 9; ++v) q1[v] = 0.0;
        }
        // A7: derivative of the flux polynomial at the solution points of the line: C fragments reused as A fragments
#pragma unroll
        for (int v = 0; v < 9; ++v) {
          double r0 = 0.0, r1 = 0.0;
          dmma884(r0, r1, q0[v], bD0);
          dmma884(r0, r1, q1[v], bD1);
          if (lv) {
            if (2 * c < N) {
              double* p = sR + v * I::n3 + sb + (2 * c) * st;
              *p = (d == 0) ? r0 : (*p + r0);
            }
            if (2 * c + 1 < N) {
              double* p = sR + v * I::n3 + sb + (2 * c + 1) * st;
              *p = (d == 0) ? r1 : (*p + r1);
            }
          }
        }
        __syncthreads();
      }
    }

    // ---- A8 + A9
    for (int s = threadIdx.x; s < I::n3; s += blockDim.x) {
      double Q[9], R[9];
#pragma unroll
      for (int v = 0; v < 9; ++v) Q[v] = sQ[v * I::n3 + s];
      const double rj = -1.0 / geo.detJ[e * I::n3 + s];
#pragma unroll
      for (int v = 0; v < 9; ++v) R[v] = sR[v * I::n3 + s] * rj;
      double divB = 0.0;
      if (GRADV == 2) divB = sG[15 * I::n3 + s] + sG[19 * I::n3 + s] + sG[23 * I::n3 + s];
      if (GRADV == 1) divB = sG[0 * I::n3 + s] + sG[4 * I::n3 + s] + sG[8 * I::n3 + s];
      const PrimD p = primitives(ph, Q);
      const double* xe = geo.xsol + e * 3 * I::n3;
      add_sources(ph, p, divB, xe[s], xe[I::n3 + s], xe[2 * I::n3 + s], R);
      if (io.Qout != nullptr) {        // step mode: Runge-Kutta combination
#pragma unroll
        for (int v = 0; v < 9; ++v) {
          const int64_t ix = (e * 9 + v) * I::n3 + s;
          double a = io.bdt * R[v];
          if (io.A0 != nullptr) a += io.c0 * io.A0[ix];
          if (io.A1 != nullptr) a += io.c1 * io.A1[ix];
          if (io.A2 != nullptr) a += io.c2 * io.A2[ix];
          R[v] = a;
        }
      }
      if (DIFF) {                      // finished by the face kernel
#pragma unroll
        for (int v = 0; v < 9; ++v) io.Part[(e * 9 + v) * I::n3 + s] = R[v];
      } else if (io.Qout != nullptr) {
#pragma unroll
        for (int v = 0; v < 9; ++v) {
          io.Qout[(e * 9 + v) * I::n3 + s] = R[v];
          sQ[v * I::n3 + s] = R[v];     // this thread is the only reader and writer of point s in this phase
        }
      } else {
#pragma unroll
        for (int v = 0; v < 9; ++v) io.Rout[((int64_t)v * E + e) * I::n3 + s] = R[v];
      }
    }
    if (!DIFF && io.Qout != nullptr) {
      __syncthreads();
      emit_traces<N>(sQ, io.QfOut + e * 54 * I::n2);
    }
  }
}

template <int N, int GRADV>
constexpr size_t stage_main_smem_bytes() {
  using I = Ix<N>;
  constexpr int NGV = GRADV == 2 ? 9 : GRADV == 1 ? 3 : 0;
  constexpr int kOwn = 54 * I::n2 > 9 * I::n3 ? 54 * I::n2 : 9 * I::n3;
  return sizeof(double) * (size_t)(9 * I::n3 + kOwn + 54 * I::n2 + 3 * NGV * I::n3);
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
    const double* Sfl_e = geo.Sfl + e * 9 * I::nf;
    for (int t = threadIdx.x; t < 6 * I::n2; t += blockDim.x) {
      const int f = t / I::n2, ab = t % I::n2;
      double nx, ny, nz, area, sg;
      face_normal<N>(Sfl_e, f, ab, nx, ny, nz, area, sg);
      const double sa = sg * area;
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
      emit_traces<N>(sP, io.QfOut + e * 54 * I::n2);
    }
  }
}

template <int N>
constexpr size_t stage_face_smem_bytes() {
  using I = Ix<N>;
  return sizeof(double) * (size_t)(9 * I::n3 + 42 * I::n2);
}

}  // namespace chorus
