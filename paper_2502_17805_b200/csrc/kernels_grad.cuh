// kernels_grad.cuh -- A2 (face gather + BR1 common solution), A3 (gradient at the solution points) and the
// face part of A4 (own-side viscous flux at the face points) of the hot path.
//   PAPER.md:123 "the solutions and solution gradient are then extrapolated to their respective families of flux points"
//   PAPER.md:149 BR1: the common solution on an interface is the average of the two polynomials; "a similar
//   procedure is used for the viscous flux"; walls PAPER.md:190-198.
#pragma once
#include "kernels_common.cuh"

namespace chorus {

// CTA size of the scalar three-kernel path (grad_kernel, residual_kernel): orders 8 and 9 fit one CTA per SM (their tiles fill the
// shared memory), which carries 16 warps instead of 8 to hide the latency of its shared-memory passes (measured on the sweep
// meshes: 384 / 512 / 640 / 768 / 1024 threads give 8.6 / 8.8 / 7.5 / 6.1 / 4.7e9 DOF-updates/s at n = 8 against 7.6e9 with 256).
template <int N> struct ScalarCfg { static constexpr int kThreads = N >= 8 ? 512 : 256; };


// Stage the own traces and the neighbours' traces of one element in shared memory.
//   sQo[f][v][ab] = own polynomial at the face point;  sQn[f][v][ab] = neighbour's polynomial there, or, on a
//   wall face, the boundary state Q_b (so that "common solution" = Q_b and "outer state" = Q_b both read sQn).
template <int N>
__device__ __forceinline__ void stage_traces(int64_t e, const ElemNbr& nb, const PhysD& ph, const double* __restrict__ Qf,
                                             const double* __restrict__ Sfl_e, double* sQo, double* sQn) {
  using I = Ix<N>;
  for (int t = threadIdx.x; t < 6 * I::n2; t += blockDim.x) {
    const int f = t / I::n2, ab = t % I::n2;
    double own[9], out[9];
#pragma unroll
    for (int v = 0; v < 9; ++v) own[v] = Qf[((e * 6 + f) * 9 + v) * I::n2 + ab];
    const int ne = nb.ne[f];
    if (ne >= 0) {
      const int ab2 = I::orient(nb.no[f], ab);
      const double* src = Qf + (((int64_t)ne * 6 + nb.nf[f]) * 9) * I::n2 + ab2;
#pragma unroll
      for (int v = 0; v < 9; ++v) out[v] = src[v * I::n2];
    } else {
      double nx, ny, nz, area, sg;
      face_normal<N>(Sfl_e, f, ab, nx, ny, nz, area, sg);
      wall_state(ph, ne, own, nx, ny, nz, out);
    }
#pragma unroll
    for (int v = 0; v < 9; ++v) {
      sQo[(f * 9 + v) * I::n2 + ab] = own[v];
      sQn[(f * 9 + v) * I::n2 + ab] = out[v];
    }
  }
}

// BR1 gradient of variables V0 .. V0+NV-1 at the solution points:  sG[((v-V0)*3 + p)*n3 + s] = d Q_v / d x_p.
// d/dxi_d of the degree-n polynomial through the d-family values (interior: own polynomial at the interior flux
// points, folded into Dss = Dfs*Isf; ends: the common face values), then the chain rule with grad xi_d (G9).
// Must be called by all threads; contains __syncthreads().
template <int N, int V0, int NV>
__device__ __forceinline__ void br1_gradient(const ElemNbr& nb, const double* sQ, const double* sQo, const double* sQn,
                                             const double* __restrict__ jinv_e, double* sG) {
  using I = Ix<N>;
  const OpsC& op = c_ops[N];
  for (int t = threadIdx.x; t < 3 * NV * I::n2; t += blockDim.x) {
    const int ab = t % I::n2, vv = (t / I::n2) % NV, d = t / (NV * I::n2);
    const int v = V0 + vv;
    const int st = I::stride(d), sb = I::sbase(d, ab);
    double q[N];
#pragma unroll
    for (int l = 0; l < N; ++l) q[l] = sQ[v * I::n3 + sb + l * st];
    const int f0 = 2 * d, f1 = 2 * d + 1;
    const double o0 = sQo[(f0 * 9 + v) * I::n2 + ab], n0 = sQn[(f0 * 9 + v) * I::n2 + ab];
    const double o1 = sQo[(f1 * 9 + v) * I::n2 + ab], n1 = sQn[(f1 * 9 + v) * I::n2 + ab];
    const double c0 = nb.ne[f0] >= 0 ? 0.5 * (o0 + n0) : n0;      // BR1 average, or the wall state
    const double c1 = nb.ne[f1] >= 0 ? 0.5 * (o1 + n1) : n1;
#pragma unroll
    for (int l = 0; l < N; ++l) {
      double s = op.Dfs[l * (N + 1)] * c0 + op.Dfs[l * (N + 1) + N] * c1;
#pragma unroll
      for (int k = 0; k < N; ++k) s += op.Dss[l * N + k] * q[k];
      sG[(vv * 3 + d) * I::n3 + sb + l * st] = s;
    }
  }
  __syncthreads();
  for (int s = threadIdx.x; s < I::n3; s += blockDim.x) {
    double j[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) j[k] = jinv_e[k * I::n3 + s];     // j[d*3+p] = (grad xi_d)_p
#pragma unroll
    for (int vv = 0; vv < NV; ++vv) {
      const double g0 = sG[(vv * 3 + 0) * I::n3 + s], g1 = sG[(vv * 3 + 1) * I::n3 + s], g2 = sG[(vv * 3 + 2) * I::n3 + s];
#pragma unroll
      for (int p = 0; p < 3; ++p) sG[(vv * 3 + p) * I::n3 + s] = j[p] * g0 + j[3 + p] * g1 + j[6 + p] * g2;
    }
  }
  __syncthreads();
}

// ---------------------------------------------------------------------------------------------------------
// grad_kernel: per element, BR1 gradient of all 9 variables, extrapolated to the 6 faces, and the own-side
// viscous flux along the outward unit normal at every face point -> Vf[e][f][7][ab].
// On wall faces the final wall viscous flux (stress-free, thermal and magnetic wall options) is stored instead.
// Optionally writes the gradient itself (test accessor chorus_get_gradient): Gout [E][27][n3].
// ---------------------------------------------------------------------------------------------------------
// SPILL: the gradient lives in a per-CTA scratch area in global memory (n = 9: 36 n^3 doubles do not fit in shared memory)
template <int N, bool SPILL = false>
__global__ void __launch_bounds__(ScalarCfg<N>::kThreads) grad_kernel(int64_t E, PhysD ph, const double* __restrict__ Qe, const double* __restrict__ Qf,
                                                   const double* __restrict__ Sfl, const double* __restrict__ jinv,
                                                   const double* __restrict__ krfl, const int32_t* __restrict__ nbr_elem,
                                                   const uint8_t* __restrict__ nbr_face, const uint8_t* __restrict__ nbr_orient,
                                                   double* __restrict__ Vf, double* __restrict__ Gout, double* scratch) {
  using I = Ix<N>;
  extern __shared__ double sm[];
  double* sQ = sm;                       // [9][n3]
  double* sG = SPILL ? scratch + blockIdx.x * (size_t)27 * I::n3 : sQ + 9 * I::n3;   // [27][n3]
  double* sQo = sQ + (SPILL ? 9 : 36) * I::n3;                                        // [6][9][n2]
  double* sQn = sQo + 54 * I::n2;        // [6][9][n2]
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
    br1_gradient<N, 0, 9>(nb, sQ, sQo, sQn, jinv + e * 9 * I::n3, sG);
    if (Gout != nullptr)
      for (int t = threadIdx.x; t < 27 * I::n3; t += blockDim.x) Gout[e * 27 * I::n3 + t] = sG[t];
    if (Vf == nullptr) continue;
    for (int t = threadIdx.x; t < 6 * I::n2; t += blockDim.x) {
      const int f = t / I::n2, ab = t % I::n2;
      const int d = f >> 1, st = I::stride(d), sb = I::sbase(d, ab);
      const double* w = op.Isf + ((f & 1) ? N * N : 0);
      double G[27];
#pragma unroll
      for (int c = 0; c < 27; ++c) {
        double s = 0.0;
#pragma unroll
        for (int l = 0; l < N; ++l) s += w[l] * sG[c * I::n3 + sb + l * st];
        G[c] = s;
      }
      double nx, ny, nz, area, sg;
      face_normal<N>(Sfl_e, f, ab, nx, ny, nz, area, sg);
      const int m = (f & 1) ? N : 0;
      const double kr = krfl ? krfl[(e * 3 + d) * I::nf + I::fbase(d, ab) + m * st] : 0.0;
      double Q[9], Fv[7];
      const int ne = nb.ne[f];
      const double* src = (ne >= 0 ? sQo : sQn) + f * 9 * I::n2 + ab;      // interior: Q_in; wall: Q_b
#pragma unroll
      for (int v = 0; v < 9; ++v) Q[v] = src[v * I::n2];
      const PrimD s = primitives(ph, Q);
      if (ne >= 0) flux_viscous(ph, s, G, nx, ny, nz, kr, Fv);
      else flux_wall_viscous(ph, ne, s, G, nx, ny, nz, kr, Fv);
#pragma unroll
      for (int c = 0; c < 7; ++c) Vf[((e * 6 + f) * 7 + c) * I::n2 + ab] = Fv[c];
    }
  }
}

}  // namespace chorus
