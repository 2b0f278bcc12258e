// geometry.cuh -- A0: geometry precompute kernel (once per mesh).
// Element map P (Eq. 13) -> Jacobi matrix (Eq. 15), |J| and |J| J^-1 (Eq. 17).
// The metrics are the conservative curl form of the degree-n interpolant of the map on the (n+1)^3 grid of
// flux-point abscissae:  S^d_p = -[curl_xi( X_l grad_xi X_m )]_d, (p,m,l) cyclic, so that sum_d d/dxi_d S^d_p = 0
// holds discretely (free-stream preservation on curved elements; reading G4).  All coordinates are taken
// relative to the element's mean node so that rounding scales with the element size.
#pragma once
#include <cstdint>

namespace chorus {

struct GeomOps {          // device pointers, row-major
  const double* Gm;       // [(n+1)][ng]      geometry nodes -> flux-point grid
  const double* Dff;      // [(n+1)][(n+1)]
  const double* Efs;      // [n][(n+1)]
  const double* Dfs;      // [n][(n+1)]
};

// out = M applied along `axis` of in[n2][n1][n0] (axis extent = cols); out extent along axis = rows.
__device__ inline void apply_axis(const double* in, int n0, int n1, int n2, int axis, const double* M, int rows, int cols,
                                  double* out) {
  const int m0 = axis == 0 ? rows : n0, m1 = axis == 1 ? rows : n1, m2 = axis == 2 ? rows : n2;
  const int total = m0 * m1 * m2;
  const int stride = axis == 0 ? 1 : axis == 1 ? n0 : n0 * n1;
  for (int t = threadIdx.x; t < total; t += blockDim.x) {
    const int i = t % m0, j = (t / m0) % m1, k = t / (m0 * m1);
    const int r = axis == 0 ? i : axis == 1 ? j : k;
    const int base = (axis == 0 ? 0 : i) + n0 * ((axis == 1 ? 0 : j) + n1 * (axis == 2 ? 0 : k));
    double s = 0.0;
    for (int q = 0; q < cols; ++q) s += M[r * cols + q] * in[base + q * stride];
    out[t] = s;
  }
}

// One CTA per element.  Dynamic shared memory: 22 * max(ng,n+1)^3 doubles.
__global__ void geometry_kernel(int n, int ng, int64_t E, GeomOps op, const double* __restrict__ xyz,
                                double* __restrict__ Sfl,     // [E][3 fam][3 comp][nf]
                                double* __restrict__ detJ,    // [E][n3]
                                double* __restrict__ jinv,    // [E][3 d][3 p][n3]
                                double* __restrict__ xsol,    // [E][3][n3]
                                double* __restrict__ krfl,    // [E][3 fam][nf] or nullptr
                                double kr_scale, double kr_c0, double kr_c1, double kr_c2, double kr_wscale) {
  extern __shared__ double sm[];
  const int N1 = n + 1, G3 = N1 * N1 * N1, n2 = n * n, n3 = n2 * n, nf = n2 * N1, ng3 = ng * ng * ng;
  const int cap = (ng > N1 ? ng : N1);
  const int C3 = cap * cap * cap;
  double* Xc = sm;               // [3][G3]   centred grid coordinates
  double* dX = Xc + 3 * C3;      // [9][G3]   dX[(j*3+c)] = d X_c / d xi_j
  double* V = dX + 9 * C3;       // [3][G3]
  double* t0 = V + 3 * C3;       // scratch
  double* t1 = t0 + C3;
  double* t2 = t1 + C3;
  double* Js = t2 + C3;          // [3][C3] reused: S at solution points for one d (3 comps) / Jacobi entries
  __shared__ double x0[3], xbar[3];
  const int64_t e = blockIdx.x;
  const int tid = threadIdx.x;

  // 0. mean node
  if (tid < 3) {
    double s = 0.0;
    for (int g = 0; g < ng3; ++g) s += xyz[(e * 3 + tid) * ng3 + g];
    x0[tid] = s / ng3;
  }
  __syncthreads();
  // 1. offsets, interpolated to the flux-point grid (three 1-D passes)
  for (int c = 0; c < 3; ++c) {
    for (int g = tid; g < ng3; g += blockDim.x) t0[g] = xyz[(e * 3 + c) * ng3 + g] - x0[c];
    __syncthreads();
    apply_axis(t0, ng, ng, ng, 0, op.Gm, N1, ng, t1);
    __syncthreads();
    apply_axis(t1, N1, ng, ng, 1, op.Gm, N1, ng, t2);
    __syncthreads();
    apply_axis(t2, N1, N1, ng, 2, op.Gm, N1, ng, Xc + c * C3);
    __syncthreads();
  }
  // 2. centre on the grid mean (exactly representable shift; the curl of a gradient vanishes discretely)
  if (tid < 3) {
    double s = 0.0;
    for (int g = 0; g < G3; ++g) s += Xc[tid * C3 + g];
    xbar[tid] = s / G3;
  }
  __syncthreads();
  for (int t = tid; t < 3 * G3; t += blockDim.x) Xc[(t / G3) * C3 + t % G3] -= xbar[t / G3];
  __syncthreads();
  // 3. derivatives of the interpolant on the grid
  for (int j = 0; j < 3; ++j)
    for (int c = 0; c < 3; ++c) apply_axis(Xc + c * C3, N1, N1, N1, j, op.Dff, N1, N1, dX + (j * 3 + c) * C3);
  __syncthreads();
  // 4. curl-form metrics
  for (int p = 0; p < 3; ++p) {
    const int mm = (p + 1) % 3, ll = (p + 2) % 3;
    for (int t = tid; t < 3 * G3; t += blockDim.x) {
      const int j = t / G3, g = t % G3;
      V[j * C3 + g] = Xc[ll * C3 + g] * dX[(j * 3 + mm) * C3 + g];
    }
    __syncthreads();
    for (int d = 0; d < 3; ++d) {
      const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
      apply_axis(V + d2 * C3, N1, N1, N1, d1, op.Dff, N1, N1, t0);
      apply_axis(V + d1 * C3, N1, N1, N1, d2, op.Dff, N1, N1, t1);
      __syncthreads();
      for (int g = tid; g < G3; g += blockDim.x) t0[g] = t1[g] - t0[g];      // S^d_p on the grid
      __syncthreads();
      // evaluate at the d-family flux points: Efs along the two other axes (in increasing axis order)
      int dims[3] = {N1, N1, N1};
      const int oa = d == 0 ? 1 : 0, ob = d == 2 ? 1 : 2;
      apply_axis(t0, dims[0], dims[1], dims[2], oa, op.Efs, n, N1, t1);
      dims[oa] = n;
      __syncthreads();
      apply_axis(t1, dims[0], dims[1], dims[2], ob, op.Efs, n, N1, t2);
      dims[ob] = n;
      __syncthreads();
      for (int g = tid; g < nf; g += blockDim.x) Sfl[((e * 3 + d) * 3 + p) * nf + g] = t2[g];
      // ... and at the solution points: Efs along d as well
      apply_axis(t2, dims[0], dims[1], dims[2], d, op.Efs, n, N1, Js + (d * 3 + p) % 3 * 0 + 0 * C3 + 0);
      __syncthreads();
      for (int g = tid; g < n3; g += blockDim.x) jinv[((e * 3 + d) * 3 + p) * n3 + g] = Js[g];   // S^d_p at sol pts; /|J| below
      __syncthreads();
    }
  }
  // 5. |J| at the solution points = det of the interpolant's Jacobi matrix there
  //    J[c][j]: Dfs along j, Efs along the other two axes.  9 entries -> dX region reused as [9][n3]
  for (int c = 0; c < 3; ++c)
    for (int j = 0; j < 3; ++j) {
      apply_axis(Xc + c * C3, N1, N1, N1, 0, j == 0 ? op.Dfs : op.Efs, n, N1, t0);
      __syncthreads();
      apply_axis(t0, n, N1, N1, 1, j == 1 ? op.Dfs : op.Efs, n, N1, t1);
      __syncthreads();
      apply_axis(t1, n, n, N1, 2, j == 2 ? op.Dfs : op.Efs, n, N1, dX + (c * 3 + j) * C3);
      __syncthreads();
    }
  for (int s = tid; s < n3; s += blockDim.x) {
    auto J = [&](int c, int j) { return dX[(c * 3 + j) * C3 + s]; };
    const double det = J(0, 0) * (J(1, 1) * J(2, 2) - J(1, 2) * J(2, 1)) - J(0, 1) * (J(1, 0) * J(2, 2) - J(1, 2) * J(2, 0)) +
                       J(0, 2) * (J(1, 0) * J(2, 1) - J(1, 1) * J(2, 0));
    detJ[e * n3 + s] = det;
    for (int dp = 0; dp < 9; ++dp) jinv[(e * 9 + dp) * n3 + s] /= det;
  }
  // 6. coordinates of the solution points; kappa_r at the flux points
  for (int c = 0; c < 3; ++c) {
    __syncthreads();
    apply_axis(Xc + c * C3, N1, N1, N1, 0, op.Efs, n, N1, t0);
    __syncthreads();
    apply_axis(t0, n, N1, N1, 1, op.Efs, n, N1, t1);
    __syncthreads();
    apply_axis(t1, n, n, N1, 2, op.Efs, n, N1, t2);
    __syncthreads();
    for (int s = tid; s < n3; s += blockDim.x) xsol[(e * 3 + c) * n3 + s] = t2[s] + xbar[c] + x0[c];
  }
  if (krfl != nullptr) {
    for (int d = 0; d < 3; ++d) {
      const int oa = d == 0 ? 1 : 0, ob = d == 2 ? 1 : 2;
      for (int c = 0; c < 3; ++c) {
        int dims[3] = {N1, N1, N1};
        __syncthreads();
        apply_axis(Xc + c * C3, dims[0], dims[1], dims[2], oa, op.Efs, n, N1, t0);
        dims[oa] = n;
        __syncthreads();
        apply_axis(t0, dims[0], dims[1], dims[2], ob, op.Efs, n, N1, V + c * C3);
      }
      __syncthreads();
      for (int g = tid; g < nf; g += blockDim.x) {
        const double px = V[g] + xbar[0] + x0[0], py = V[C3 + g] + xbar[1] + x0[1], pz = V[2 * C3 + g] + xbar[2] + x0[2];
        const double w = sqrt(px * px + py * py + pz * pz) * kr_wscale;
        krfl[(e * 3 + d) * nf + g] = kr_scale * (kr_c0 + kr_c1 * w + kr_c2 * w * w);
      }
    }
  }
}

// Outward unit normal and signed area at the face points, from S^d at the face flux points (O3):
//   nfc[e][f][0..2][ab] = sigma S/|S|,  nfc[e][f][3][ab] = sigma |S|,  sigma = +1 on the "1" faces, -1 on the "0" faces.
__global__ void face_geometry_kernel(int n, int64_t E, const double* __restrict__ Sfl, double* __restrict__ nfc) {
  const int n2 = n * n, nf = n2 * (n + 1);
  const int64_t total = E * 6 * n2;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int ab = (int)(t % n2), f = (int)((t / n2) % 6);
    const int64_t e = t / (6 * n2);
    const int d = f >> 1, m = (f & 1) ? n : 0;
    const int a = ab % n, b = ab / n;
    const int fb = d == 0 ? ab * (n + 1) : d == 1 ? b * (n + 1) * n + a : ab;
    const int ix = fb + m * (d == 0 ? 1 : d == 1 ? n : n2);
    const double* S = Sfl + (e * 3 + d) * 3 * nf + ix;
    const double sx = S[0], sy = S[nf], sz = S[2 * nf];
    const double area = sqrt(sx * sx + sy * sy + sz * sz);
    const double sg = (f & 1) ? 1.0 : -1.0;
    const double inv = sg / area;
    double* o = nfc + (e * 6 + f) * 4 * n2 + ab;
    o[0] = sx * inv; o[n2] = sy * inv; o[2 * n2] = sz * inv; o[3 * n2] = sg * area;
  }
}

// S^d at the INTERIOR flux points only (m = 1 .. n-1), the part of Sfl that the element kernel's chains read (the face points go
// through nfc): Sint[e][fam d][comp][.] in the natural family layout with n - 1 points per line,
//   d = 0: ab (n-1) + (m-1);   d = 1: b (n-1) n + (m-1) n + a;   d = 2: (m-1) n^2 + ab.
__global__ void interior_S_kernel(int n, int64_t E, const double* __restrict__ Sfl, double* __restrict__ Sint) {
  const int n2 = n * n, nf = n2 * (n + 1), nfi = n2 * (n - 1);
  const int64_t total = E * 9 * nfi;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int idx = (int)(t % nfi), fc = (int)((t / nfi) % 9);
    const int64_t e = t / (9 * (int64_t)nfi);
    const int d = fc / 3;
    int ab, m;
    if (d == 0) { ab = idx / (n - 1); m = idx % (n - 1) + 1; }
    else if (d == 1) { const int b = idx / ((n - 1) * n), r = idx % ((n - 1) * n); m = r / n + 1; ab = b * n + r % n; }
    else { m = idx / n2 + 1; ab = idx % n2; }
    const int a = ab % n, b = ab / n;
    const int fb = d == 0 ? ab * (n + 1) : d == 1 ? b * (n + 1) * n + a : ab;
    Sint[t] = Sfl[(e * 9 + fc) * nf + fb + m * (d == 0 ? 1 : d == 1 ? n : n2)];
  }
}

}  // namespace chorus
