// kernels_residual.cuh -- the element kernel of the hot path: A1 (interpolate Q to the three flux families),
// A4 (interpolate grad Q), A5 (fluxes at interior flux points), A6 (Rusanov / wall fluxes at face flux points),
// A7 (derivative of the flux polynomials at the solution points), A8 (sources), A9 (fused RK stage update).
//   procedure PAPER.md:123; bases Eq. 19-20; reconstruction Eq. 21-24; transformed equations Eq. 16-17;
//   fluxes Eq. 6-10; sources Eq. 5; common fluxes PAPER.md:149; SSPRK(5,3) PAPER.md:151.
#pragma once
#include "kernels_grad.cuh"

namespace chorus {

struct StageOut {
  double* Rout;          // residual in the interface layout [9][E][n3], or nullptr
  double* Qout;          // new state, element-major, or nullptr:  Qout = c0*A0 + c1*A1 + c2*A2 + bdt * R
  const double* A0;      // stage registers (element-major); a null pointer contributes nothing
  const double* A1;
  const double* A2;
  double c0, c1, c2, bdt;
};

// GRADV: 0 no gradient needed, 1 gradient of B only (Powell sources without diffusion), 2 all nine variables.
// SPILL: orders whose tiles exceed the shared memory of an SM (n = 8, 9 with diffusion) keep the neighbour traces, the gradient
// and its interpolant in a per-CTA scratch area in global memory (L2-resident: the grid is persistent) instead.
template <int N, bool DIFF, int GRADV, bool SPILL = false>
__global__ void __launch_bounds__(ScalarCfg<N>::kThreads, 1)
residual_kernel(int64_t E, PhysD ph, const double* __restrict__ Qe, const double* __restrict__ Qf, const double* __restrict__ Vf,
                const double* __restrict__ Sfl, const double* __restrict__ detJ, const double* __restrict__ jinv,
                const double* __restrict__ xsol, const double* __restrict__ krfl, const int32_t* __restrict__ nbr_elem,
                const uint8_t* __restrict__ nbr_face, const uint8_t* __restrict__ nbr_orient, StageOut out, double* scratch) {
  using I = Ix<N>;
  static_assert(!DIFF || GRADV == 2, "diffusion needs the gradient of all variables");
  constexpr int NGV = GRADV == 2 ? 9 : GRADV == 1 ? 3 : 0;
  constexpr int GV0 = GRADV == 1 ? 5 : 0;
  extern __shared__ double sm[];
  double* sQ = sm;                                // [9][n3]
  double* sR = sQ + 9 * I::n3;                    // [9][n3]        xi-divergence accumulator
  double* sH = sR + 9 * I::n3;                    // [9][N+1][n2]   Q^ then F~ of the current family, line-major
  double* sQo = sH + 9 * I::nf;                   // [6][9][n2]
  constexpr size_t kScratch = (size_t)54 * I::n2 + 3 * NGV * I::n3 + (DIFF ? 27 * (N - 1) * I::n2 : 0);
  double* sQn = SPILL ? scratch + blockIdx.x * kScratch : sQo + 54 * I::n2;      // [6][9][n2]
  double* sG = sQn + 54 * I::n2;                  // [3*NGV][n3]
  double* sGh = sG + 3 * NGV * I::n3;             // [27][N-1][n2]  (DIFF only)
  __shared__ ElemNbr nb;
  const OpsC& op = c_ops[N];

  for (int64_t e = blockIdx.x; e < E; e += gridDim.x) {
    __syncthreads();
    load_nbr(nb, e, nbr_elem, nbr_face, nbr_orient);
    for (int t = threadIdx.x; t < 9 * I::n3; t += blockDim.x) sQ[t] = Qe[e * 9 * I::n3 + t];
    __syncthreads();
    const double* Sfl_e = Sfl + e * 9 * I::nf;
    stage_traces<N>(e, nb, ph, Qf, Sfl_e, sQo, sQn);
    __syncthreads();
    if constexpr (GRADV != 0) br1_gradient<N, GV0, NGV>(nb, sQ, sQo, sQn, jinv + e * 9 * I::n3, sG);

    for (int d = 0; d < 3; ++d) {
      const int st = I::stride(d);
      // ---- A1: Q at the d-family flux points (all m; the end values equal the own traces)
      for (int t = threadIdx.x; t < 9 * I::n2; t += blockDim.x) {
        const int ab = t % I::n2, v = t / I::n2;
        const int sb = I::sbase(d, ab);
        double q[N];
#pragma unroll
        for (int l = 0; l < N; ++l) q[l] = sQ[v * I::n3 + sb + l * st];
#pragma unroll
        for (int m = 0; m <= N; ++m) {
          double s = 0.0;
#pragma unroll
          for (int l = 0; l < N; ++l) s += op.Isf[m * N + l] * q[l];
          sH[(v * (N + 1) + m) * I::n2 + ab] = s;
        }
      }
      // ---- A4: grad Q at the interior d-family flux points
      if (DIFF) {
        for (int t = threadIdx.x; t < 27 * I::n2; t += blockDim.x) {
          const int ab = t % I::n2, c = t / I::n2;
          const int sb = I::sbase(d, ab);
          double g[N];
#pragma unroll
          for (int l = 0; l < N; ++l) g[l] = sG[c * I::n3 + sb + l * st];
#pragma unroll
          for (int m = 1; m < N; ++m) {
            double s = 0.0;
#pragma unroll
            for (int l = 0; l < N; ++l) s += op.Isf[m * N + l] * g[l];
            sGh[(c * (N - 1) + m - 1) * I::n2 + ab] = s;
          }
        }
      }
      __syncthreads();
      // ---- A5 / A6: transformed flux F~ at every flux point of the family (in place over Q^)
      for (int t = threadIdx.x; t < (N + 1) * I::n2; t += blockDim.x) {
        const int ab = t % I::n2, m = t / I::n2;
        const int ix = I::fbase(d, ab) + m * st;
        double F[9];
        if (m > 0 && m < N) {
          double Q[9];
#pragma unroll
          for (int v = 0; v < 9; ++v) Q[v] = sH[(v * (N + 1) + m) * I::n2 + ab];
          const double Sx = Sfl_e[(d * 3 + 0) * I::nf + ix], Sy = Sfl_e[(d * 3 + 1) * I::nf + ix], Sz = Sfl_e[(d * 3 + 2) * I::nf + ix];
          const PrimD s = primitives(ph, Q);
          flux_inviscid<false>(ph, s, Sx, Sy, Sz, F);
          if (DIFF) {
            double G[27], Fv[7];
#pragma unroll
            for (int c = 0; c < 27; ++c) G[c] = sGh[(c * (N - 1) + m - 1) * I::n2 + ab];
            const double kr = krfl ? krfl[(e * 3 + d) * I::nf + ix] : 0.0;
            flux_viscous(ph, s, G, Sx, Sy, Sz, kr, Fv);
#pragma unroll
            for (int c = 0; c < 7; ++c) F[1 + c] -= Fv[c];
          }
        } else {
          const int f = 2 * d + (m == N ? 1 : 0);
          const int ne = nb.ne[f];
          double nx, ny, nz, area, sg;
          face_normal<N>(Sfl_e, f, ab, nx, ny, nz, area, sg);
          double Qo[9];
#pragma unroll
          for (int v = 0; v < 9; ++v) Qo[v] = sQn[(f * 9 + v) * I::n2 + ab];
          double Fv[7];
#pragma unroll
          for (int c = 0; c < 7; ++c) Fv[c] = 0.0;
          if (ne >= 0) {
            double Qi[9];
#pragma unroll
            for (int v = 0; v < 9; ++v) Qi[v] = sQo[(f * 9 + v) * I::n2 + ab];
            flux_rusanov(ph, Qi, Qo, nx, ny, nz, F);
            if (DIFF) {   // average of the two sides' viscous fluxes; the neighbour's is along its own (opposite) normal
              const int ab2 = I::orient(nb.no[f], ab);
              const double* mine = Vf + ((e * 6 + f) * 7) * I::n2 + ab;
              const double* theirs = Vf + (((int64_t)ne * 6 + nb.nf[f]) * 7) * I::n2 + ab2;
#pragma unroll
              for (int c = 0; c < 7; ++c) Fv[c] = 0.5 * (mine[c * I::n2] - theirs[c * I::n2]);
            }
          } else {
            const PrimD sb_ = primitives(ph, Qo);            // Qo holds the wall state Q_b
            flux_inviscid<true>(ph, sb_, nx, ny, nz, F);
            if (DIFF) {
              const double* mine = Vf + ((e * 6 + f) * 7) * I::n2 + ab;
#pragma unroll
              for (int c = 0; c < 7; ++c) Fv[c] = mine[c * I::n2];
            }
          }
          const double sa = sg * area;
          F[0] *= sa;
#pragma unroll
          for (int c = 0; c < 7; ++c) F[1 + c] = sa * (F[1 + c] - Fv[c]);
          F[8] *= sa;
        }
#pragma unroll
        for (int v = 0; v < 9; ++v) sH[(v * (N + 1) + m) * I::n2 + ab] = F[v];
      }
      __syncthreads();
      // ---- A7: derivative of the flux polynomial at the solution points, accumulated over the three families
      for (int t = threadIdx.x; t < 9 * I::n2; t += blockDim.x) {
        const int ab = t % I::n2, v = t / I::n2;
        const int sb = I::sbase(d, ab);
        double fl[N + 1];
#pragma unroll
        for (int m = 0; m <= N; ++m) fl[m] = sH[(v * (N + 1) + m) * I::n2 + ab];
#pragma unroll
        for (int l = 0; l < N; ++l) {
          double s = 0.0;
#pragma unroll
          for (int m = 0; m <= N; ++m) s += op.Dfs[l * (N + 1) + m] * fl[m];
          double* r = sR + v * I::n3 + sb + l * st;
          *r = (d == 0) ? s : (*r + s);
        }
      }
      __syncthreads();
    }

    // ---- A8 + A9: R = -(1/|J|) div_xi F~ + M (Eq. 16, Eq. 5); residual output and / or fused RK combination
    for (int s = threadIdx.x; s < I::n3; s += blockDim.x) {
      double Q[9], R[9];
#pragma unroll
      for (int v = 0; v < 9; ++v) Q[v] = sQ[v * I::n3 + s];
      const double rj = -1.0 / detJ[e * I::n3 + s];
#pragma unroll
      for (int v = 0; v < 9; ++v) R[v] = sR[v * I::n3 + s] * rj;
      double divB = 0.0;
      if (GRADV == 2) divB = sG[15 * I::n3 + s] + sG[19 * I::n3 + s] + sG[23 * I::n3 + s];
      if (GRADV == 1) divB = sG[0 * I::n3 + s] + sG[4 * I::n3 + s] + sG[8 * I::n3 + s];
      const PrimD p = primitives(ph, Q);
      const double* xe = xsol + e * 3 * I::n3;
      add_sources(ph, p, divB, xe[s], xe[I::n3 + s], xe[2 * I::n3 + s], R);
      if (out.Rout != nullptr) {
#pragma unroll
        for (int v = 0; v < 9; ++v) out.Rout[((int64_t)v * E + e) * I::n3 + s] = R[v];
      }
      if (out.Qout != nullptr) {
#pragma unroll
        for (int v = 0; v < 9; ++v) {
          const int64_t ix = (e * 9 + v) * I::n3 + s;
          double a = out.bdt * R[v];
          if (out.A0 != nullptr) a += out.c0 * out.A0[ix];
          if (out.A1 != nullptr) a += out.c1 * out.A1[ix];
          if (out.A2 != nullptr) a += out.c2 * out.A2[ix];
          out.Qout[ix] = a;
        }
      }
    }
  }
}

template <int N, bool DIFF, int GRADV>
constexpr size_t residual_scratch_doubles() {     // per CTA, SPILL only
  using I = Ix<N>;
  constexpr int NGV = GRADV == 2 ? 9 : GRADV == 1 ? 3 : 0;
  return (size_t)54 * I::n2 + 3 * NGV * I::n3 + (DIFF ? 27 * (N - 1) * I::n2 : 0);
}
template <int N, bool DIFF, int GRADV, bool SPILL = false>
constexpr size_t residual_smem_bytes() {
  using I = Ix<N>;
  return sizeof(double) * ((size_t)(18 * I::n3 + 9 * I::nf + 54 * I::n2) + (SPILL ? 0 : residual_scratch_doubles<N, DIFF, GRADV>()));
}
template <int N, bool SPILL = false>
constexpr size_t grad_smem_bytes() {
  using I = Ix<N>;
  return sizeof(double) * (size_t)((SPILL ? 9 : 36) * I::n3 + 108 * I::n2);
}

}  // namespace chorus
