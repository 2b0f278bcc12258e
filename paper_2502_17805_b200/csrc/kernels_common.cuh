// kernels_common.cuh -- shared pieces of the hot-path kernels: operator tables in constant memory, index maps,
// per-element face information, the face-trace kernel (A1 restricted to the faces), layout transposes and the
// max-wave-speed reduction (A10).
//
// Device data layout ("element-major"):
//   state       Qe  [E][9][n3]            one contiguous 9*n^3 block per element
//   S^d         Sfl [E][3 fam][3 comp][nf] natural family layout (see include/chorus.h)
//   |J|, grad xi, x at solution points:  detJ [E][n3], jinv [E][9][n3], xsol [E][3][n3]
//   face traces Qf  [E][6][9][n2]         own polynomial extrapolated to the element's 6 faces
//   viscous face fluxes Vf [E][6][7][n2]  own-side viscous flux along the own outward unit normal (wall: the wall flux)
#pragma once
#include <cstdint>
#include "physics.cuh"

namespace chorus {

constexpr int kMaxN = 9;

struct OpsC {
  double Isf[(kMaxN + 1) * kMaxN];   // [(n+1)][n]
  double Dfs[kMaxN * (kMaxN + 1)];   // [n][(n+1)]
  double Dss[kMaxN * kMaxN];         // [n][n]
};
__constant__ OpsC c_ops[kMaxN + 1];   // indexed by the order n

template <int N>
struct Ix {
  static constexpr int N1 = N + 1, n2 = N * N, n3 = N * N * N, nf = N * N * (N + 1);
  // a "line" along direction d is labelled ab = b*N + a, (a,b) = the two other solution indices in increasing axis order
  __device__ __forceinline__ static int sbase(int d, int ab) {
    const int a = ab % N, b = ab / N;
    return d == 0 ? ab * N : d == 1 ? b * n2 + a : ab;
  }
  __device__ __forceinline__ static int stride(int d) { return d == 0 ? 1 : d == 1 ? N : n2; }
  __device__ __forceinline__ static int fbase(int d, int ab) {      // index into the natural family-d layout
    const int a = ab % N, b = ab / N;
    return d == 0 ? ab * N1 : d == 1 ? b * N1 * N + a : ab;
  }
  // own face point ab -> neighbour's face point under orientation `code`
  __device__ __forceinline__ static int orient(int code, int ab) {
    int a = ab % N, b = ab / N;
    if (code & 1) { const int t = a; a = b; b = t; }
    if (code & 2) a = N - 1 - a;
    if (code & 4) b = N - 1 - b;
    return b * N + a;
  }
};

struct ElemNbr {   // connectivity of one element, staged in shared memory
  int ne[6];
  int nf[6];
  int no[6];
};

__device__ __forceinline__ void load_nbr(ElemNbr& s, int64_t e, const int32_t* nbr_elem, const uint8_t* nbr_face,
                                         const uint8_t* nbr_orient) {
  if (threadIdx.x < 6) {
    s.ne[threadIdx.x] = nbr_elem[e * 6 + threadIdx.x];
    s.nf[threadIdx.x] = nbr_face[e * 6 + threadIdx.x];
    s.no[threadIdx.x] = nbr_orient[e * 6 + threadIdx.x];
  }
}

// unit outward normal and area at face point ab of face f, from S^d at the face flux points
template <int N>
__device__ __forceinline__ void face_normal(const double* __restrict__ Sfl_e, int f, int ab, double& nx, double& ny, double& nz,
                                            double& area, double& sg) {
  using I = Ix<N>;
  const int d = f >> 1, m = (f & 1) ? N : 0;
  const int ix = I::fbase(d, ab) + m * I::stride(d);
  const double sx = Sfl_e[(d * 3 + 0) * I::nf + ix], sy = Sfl_e[(d * 3 + 1) * I::nf + ix], sz = Sfl_e[(d * 3 + 2) * I::nf + ix];
  area = sqrt(sx * sx + sy * sy + sz * sz);
  sg = (f & 1) ? 1.0 : -1.0;
  const double inv = sg / area;
  nx = sx * inv; ny = sy * inv; nz = sz * inv;
}

// ---------------------------------------------------------------------------------------------------------
// A1 (faces): Qf[e][f][v][ab] = sum_l h_l(X_f at the face) Q[e][v][line(ab), l]       (Eq. 19, 21)
// ---------------------------------------------------------------------------------------------------------
template <int N>
__global__ void __launch_bounds__(256) trace_kernel(int64_t E, const double* __restrict__ Qe, double* __restrict__ Qf) {
  using I = Ix<N>;
  extern __shared__ double sm[];
  double* sQ = sm;   // [9][n3]
  const OpsC& op = c_ops[N];
  for (int64_t e = blockIdx.x; e < E; e += gridDim.x) {
    __syncthreads();
    for (int t = threadIdx.x; t < 9 * I::n3; t += blockDim.x) sQ[t] = Qe[e * 9 * I::n3 + t];
    __syncthreads();
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
      Qf[((e * 6 + 2 * d) * 9 + v) * I::n2 + ab] = lo;
      Qf[((e * 6 + 2 * d + 1) * 9 + v) * I::n2 + ab] = hi;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// layout transposes between the interface layout [V][E][n3] and the element-major layout [E][V][n3]
// ---------------------------------------------------------------------------------------------------------
__global__ void to_element_major(int64_t E, int n3, int nv, const double* __restrict__ in, double* __restrict__ out) {
  const int64_t total = E * nv * n3;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int s = t % n3;
    const int64_t r = t / n3;
    const int v = r % nv;
    const int64_t e = r / nv;
    out[t] = in[((int64_t)v * E + e) * n3 + s];
  }
}
__global__ void from_element_major(int64_t E, int n3, int nv, const double* __restrict__ in, double* __restrict__ out) {
  const int64_t total = E * nv * n3;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int s = t % n3;
    const int64_t r = t / n3;
    const int64_t e = r % E;
    const int v = r / E;
    out[t] = in[(e * nv + v) * n3 + s];
  }
}

// ---------------------------------------------------------------------------------------------------------
// A10: max over solution points of |U| + sqrt((gamma p + |B|^2)/rho): warp shuffle -> block -> atomic max.
// Wave speeds are non-negative, so the IEEE bit pattern orders like the value; NaN is propagated as +inf bits | 1.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) wavespeed_kernel(int64_t E, int n3, PhysD ph, const double* __restrict__ Qe,
                                                       unsigned long long* __restrict__ out) {
  double mx = 0.0;
  bool bad = false;
  const int64_t total = E * n3;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t e = t / n3;
    const int s = t % n3;
    double Q[9];
#pragma unroll
    for (int v = 0; v < 9; ++v) Q[v] = Qe[(e * 9 + v) * n3 + s];
    const double c = wavespeed(ph, Q);
    if (!(c == c) || isinf(c)) bad = true;
    mx = fmax(mx, c);
  }
  if (bad) mx = __longlong_as_double(0x7ff8000000000000LL);
  unsigned long long bits = (unsigned long long)__double_as_longlong(mx);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long other = __shfl_xor_sync(0xffffffffu, bits, o);
    bits = other > bits ? other : bits;
  }
  __shared__ unsigned long long wmax[8];
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = bits;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (blockDim.x >> 5); ++w) bits = wmax[w] > bits ? wmax[w] : bits;
    atomicMax(out, bits);
  }
}

// ---------------------------------------------------------------------------------------------------------
// Volume integrals of Eq. 34-35 by the solution-point quadrature  int f dV = sum w_i w_j w_k |J| f:
// sum |J| w, sum |J| w 1/2 rho U.U, sum |J| w 1/2 B.B.  Deterministic: one partial per block (warp shuffle tree, then the
// block's warps in order), then one block adds the partials in a fixed tree -- no atomics, bit-reproducible.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void block_sum3(double& a, double& b, double& c, double (*sh)[3]) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
    c += __shfl_xor_sync(0xffffffffu, c, o);
  }
  const int warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) { sh[warp][0] = a; sh[warp][1] = b; sh[warp][2] = c; }
  __syncthreads();
  if (threadIdx.x == 0) {
    a = sh[0][0]; b = sh[0][1]; c = sh[0][2];
    for (int w = 1; w < nw; ++w) { a += sh[w][0]; b += sh[w][1]; c += sh[w][2]; }
  }
}
__global__ void __launch_bounds__(256) diagnostics_kernel(int64_t E, int n, const double* __restrict__ wq, const double* __restrict__ detJ,
                                                         const double* __restrict__ Qe, double* __restrict__ partial /*[grid][3]*/) {
  __shared__ double sh[8][3];
  const int n3 = n * n * n;
  double V = 0.0, KE = 0.0, EB = 0.0;
  const int64_t total = E * n3;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t e = t / n3;
    const int s = (int)(t % n3);
    const int i = s % n, j = (s / n) % n, k = s / (n * n);
    const double wJ = wq[i] * wq[j] * wq[k] * detJ[t];
    const double* q = Qe + e * 9 * n3 + s;
    const double rho = q[0], m1 = q[n3], m2 = q[2 * n3], m3 = q[3 * n3];
    const double b1 = q[5 * n3], b2 = q[6 * n3], b3 = q[7 * n3];
    V += wJ;
    KE += wJ * (0.5 * (m1 * m1 + m2 * m2 + m3 * m3) / rho);
    EB += wJ * (0.5 * (b1 * b1 + b2 * b2 + b3 * b3));
  }
  block_sum3(V, KE, EB, sh);
  if (threadIdx.x == 0) { partial[blockIdx.x * 3 + 0] = V; partial[blockIdx.x * 3 + 1] = KE; partial[blockIdx.x * 3 + 2] = EB; }
}
// sums != 0: the raw integrals (a partition's share; the caller adds the partitions' and divides)
__global__ void __launch_bounds__(256) diagnostics_final_kernel(int nparts, const double* __restrict__ partial, double* __restrict__ out /*[3]*/,
                                                               int sums) {
  __shared__ double sh[8][3];
  double V = 0.0, KE = 0.0, EB = 0.0;
  for (int t = threadIdx.x; t < nparts; t += blockDim.x) { V += partial[t * 3]; KE += partial[t * 3 + 1]; EB += partial[t * 3 + 2]; }
  block_sum3(V, KE, EB, sh);
  if (threadIdx.x == 0) { out[0] = V; out[1] = sums ? KE : KE / V; out[2] = sums ? EB : EB / V; }
}

// ---------------------------------------------------------------------------------------------------------
// Halo of a partition: item k is face fc[k] of element el[k]; its block of w doubles (9 n^2 face traces or
// 7 n^2 viscous face fluxes) at base[(el*6 + fc) * w] is copied to (pack) or from (unpack) buf[k * w].
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) halo_copy_kernel(int64_t cnt, int w, const int32_t* __restrict__ el, const uint8_t* __restrict__ fc,
                                                       double* __restrict__ base, double* __restrict__ buf, int pack) {
  const int64_t total = cnt * w;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t k = t / w;
    const int j = (int)(t % w);
    double* p = base + ((int64_t)el[k] * 6 + fc[k]) * w + j;
    if (pack) buf[t] = *p;
    else *p = buf[t];
  }
}

}  // namespace chorus
