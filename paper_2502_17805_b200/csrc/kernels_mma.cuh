// kernels_mma.cuh -- the element kernel as register-resident FP64 tensor-core chains (orders 4..7).
//
// Same mathematics as kernels_residual.cuh (A1, A3-A9 of the hot path; Eq. 19-24), different mapping:
// one warp owns a group of 8 lines of one direction.  With mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4)
//   Q^, grad Q^ [line][col]  = A[line][l] * B[l][col]      A = solution values of the line (from shared memory),
//                                                         B = h_l(X_f,m(col))  (Eq. 19 evaluated at the flux points)
// land in the C fragment: thread (r = lane/4, c = lane%4) holds columns 2c and 2c+1 of line r, i.e. ALL 36 interpolated
// quantities of two flux points -- exactly what the pointwise fluxes (Eq. 6-10) need, with no shared-memory round trip.
// The fluxes F~ stay in those registers, and because the C layout of m8n8k4 (row = lane/4, cols 2c, 2c+1) is the A
// layout of two k-steps once the contraction index is permuted, they feed the derivative product
//   dF~/dxi [line][l]        = F~[line][col] * B'[col][l]    B' = l'_{m(col)}(X_s,l)  (Eq. 20, 22-24)
// directly.  Columns: the interior flux points first, then the two face points (whose common fluxes come from the
// face pass), then padding.  FP64 DMMA on B200 runs at the DFMA pipe's peak (measured 37.1 vs 34.0 TFLOP/s) but
// needs 1/8 of the issue slots and none of the shared-memory traffic for the intermediates (profiles/).
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
  // column j of the 8-wide tile -> flux point index m, or -1 (padding).  interior m = 1..N-1, then m = 0, m = N.
  __device__ __forceinline__ static int col_m(int j) { return j < N - 1 ? j + 1 : j == N - 1 ? 0 : j == N ? N : -1; }
};

// GRADV as in residual_kernel.  kThreads threads per CTA.
#ifndef CHORUS_MMA_MINBLOCKS
#define CHORUS_MMA_MINBLOCKS 1
#endif
template <int N, bool DIFF, int GRADV>
__global__ void __launch_bounds__(Mma<N>::kThreads, CHORUS_MMA_MINBLOCKS)
residual_mma_kernel(int64_t E, PhysD ph, const double* __restrict__ Qe, const double* __restrict__ Qf, const double* __restrict__ Vf,
                    const double* __restrict__ Sfl, const double* __restrict__ detJ, const double* __restrict__ jinv,
                    const double* __restrict__ xsol, const double* __restrict__ krfl, const int32_t* __restrict__ nbr_elem,
                    const uint8_t* __restrict__ nbr_face, const uint8_t* __restrict__ nbr_orient, StageOut out) {
  using I = Ix<N>;
  using M = Mma<N>;
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
  double bD0 = 0.0, bD1 = 0.0;
  if (r < N) {
    const int m0 = M::col_m(2 * c), m1 = M::col_m(2 * c + 1);
    if (m0 >= 0) bD0 = op.Dfs[r * (N + 1) + m0];
    if (m1 >= 0) bD1 = op.Dfs[r * (N + 1) + m1];
  }
  // BR1 gradient: x = (q_0..q_{N-1}, common value at m = 0, at m = N), K = N + 2 <= 12 -> up to 3 k-steps of 4
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
    load_nbr(nb, e, nbr_elem, nbr_face, nbr_orient);
    for (int t = threadIdx.x; t < 9 * I::n3; t += blockDim.x) sQ[t] = Qe[e * 9 * I::n3 + t];
    __syncthreads();
    const double* Sfl_e = Sfl + e * 9 * I::nf;
    stage_traces<N>(e, nb, ph, Qf, Sfl_e, sQo, sQn);
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
        for (int k = 0; k < 9; ++k) j[k] = jinv[e * 9 * I::n3 + k * I::n3 + s];
#pragma unroll
        for (int vv = 0; vv < NGV; ++vv) {
          const double g0 = sG[(vv * 3 + 0) * I::n3 + s], g1 = sG[(vv * 3 + 1) * I::n3 + s], g2 = sG[(vv * 3 + 2) * I::n3 + s];
#pragma unroll
          for (int p = 0; p < 3; ++p) sG[(vv * 3 + p) * I::n3 + s] = j[p] * g0 + j[3 + p] * g1 + j[6 + p] * g2;
        }
      }
    }

    // ---- A6: common fluxes at the 6 n^2 face points (Rusanov / wall, viscous average), scaled by sigma |S|, in place over sQn
    for (int t = threadIdx.x; t < 6 * I::n2; t += blockDim.x) {
      const int f = t / I::n2, ab = t % I::n2;
      const int ne = nb.ne[f];
      double nx, ny, nz, area, sg;
      face_normal<N>(Sfl_e, f, ab, nx, ny, nz, area, sg);
      double Qo[9], F[9], Fv[7];
#pragma unroll
      for (int v = 0; v < 9; ++v) Qo[v] = sQn[(f * 9 + v) * I::n2 + ab];
#pragma unroll
      for (int k = 0; k < 7; ++k) Fv[k] = 0.0;
      if (ne >= 0) {
        double Qi[9];
#pragma unroll
        for (int v = 0; v < 9; ++v) Qi[v] = sQo[(f * 9 + v) * I::n2 + ab];
        flux_rusanov(ph, Qi, Qo, nx, ny, nz, F);
        if (DIFF) {
          const int ab2 = I::orient(nb.no[f], ab);
          const double* mine = Vf + ((e * 6 + f) * 7) * I::n2 + ab;
          const double* theirs = Vf + (((int64_t)ne * 6 + nb.nf[f]) * 7) * I::n2 + ab2;
#pragma unroll
          for (int k = 0; k < 7; ++k) Fv[k] = 0.5 * (mine[k * I::n2] - theirs[k * I::n2]);
        }
      } else {
        const PrimD sb_ = primitives(ph, Qo);
        flux_inviscid<true>(ph, sb_, nx, ny, nz, F);
        if (DIFF) {
          const double* mine = Vf + ((e * 6 + f) * 7) * I::n2 + ab;
#pragma unroll
          for (int k = 0; k < 7; ++k) Fv[k] = mine[k * I::n2];
        }
      }
      const double sa = sg * area;
      sQn[(f * 9 + 0) * I::n2 + ab] = sa * F[0];
#pragma unroll
      for (int k = 0; k < 7; ++k) sQn[(f * 9 + 1 + k) * I::n2 + ab] = sa * (F[1 + k] - Fv[k]);
      sQn[(f * 9 + 8) * I::n2 + ab] = sa * F[8];
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
        double q0[9], q1[9];
#pragma unroll
        for (int v = 0; v < 9; ++v) {
          const double a0 = sQ[v * I::n3 + sb + c * st];
          const double a1 = (4 + c < N) ? sQ[v * I::n3 + sb + (4 + c) * st] : 0.0;
          q0[v] = 0.0; q1[v] = 0.0;
          dmma884(q0[v], q1[v], a0, bI0);
          if (N > 4) dmma884(q0[v], q1[v], a1, bI1);
        }
        double g0[DIFF ? 27 : 1], g1[DIFF ? 27 : 1];
        if (DIFF) {
#pragma unroll
          for (int k = 0; k < 27; ++k) {
            const double a0 = sG[k * I::n3 + sb + c * st];
            const double a1 = (4 + c < N) ? sG[k * I::n3 + sb + (4 + c) * st] : 0.0;
            g0[k] = 0.0; g1[k] = 0.0;
            dmma884(g0[k], g1[k], a0, bI0);
            if (N > 4) dmma884(g0[k], g1[k], a1, bI1);
          }
        }
        // pointwise fluxes on the two columns this thread holds; results overwrite q0 / q1
#pragma unroll
        for (int slot = 0; slot < 2; ++slot) {
          double* q = slot ? q1 : q0;
          double* g = slot ? g1 : g0;
          const int m = M::col_m(2 * c + slot);
          if (m > 0 && m < N) {                                   // interior flux point
            const int ix = I::fbase(d, ln) + m * st;
            const double Sx = Sfl_e[(d * 3 + 0) * I::nf + ix], Sy = Sfl_e[(d * 3 + 1) * I::nf + ix], Sz = Sfl_e[(d * 3 + 2) * I::nf + ix];
            const PrimD s = primitives(ph, q);
            double F[9];
            flux_inviscid<false>(ph, s, Sx, Sy, Sz, F);
            if (DIFF) {
              double Fv[7];
              const double kr = krfl ? krfl[(e * 3 + d) * I::nf + ix] : 0.0;
              flux_viscous(ph, s, g, Sx, Sy, Sz, kr, Fv);
#pragma unroll
              for (int k = 0; k < 7; ++k) F[1 + k] -= Fv[k];
            }
#pragma unroll
            for (int v = 0; v < 9; ++v) q[v] = F[v];
          } else if (m >= 0) {                                    // face flux point: the common flux from the face pass
            const int f = 2 * d + (m == N ? 1 : 0);
#pragma unroll
            for (int v = 0; v < 9; ++v) q[v] = sQn[(f * 9 + v) * I::n2 + ln];
          } else {
#pragma unroll
            for (int v = 0; v < 9; ++v) q[v] = 0.0;
          }
        }
        // derivative of the flux polynomial at the solution points of the line: C fragments reused as A fragments
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

template <int N, int GRADV>
constexpr size_t residual_mma_smem_bytes() {
  using I = Ix<N>;
  constexpr int NGV = GRADV == 2 ? 9 : GRADV == 1 ? 3 : 0;
  constexpr int kOwn = 54 * I::n2 > 9 * I::n3 ? 54 * I::n2 : 9 * I::n3;
  return sizeof(double) * (size_t)(9 * I::n3 + kOwn + 54 * I::n2 + 3 * NGV * I::n3);
}

}  // namespace chorus
