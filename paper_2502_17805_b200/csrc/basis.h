// basis.h -- host-side 1-D node sets and operators of the SD method for the CUDA library.
// Written independently of oracle/ (barycentric Lagrange formulas, long double).
//   solution points  Eq. 18         Chebyshev-Gauss on [0,1]
//   flux points      PAPER.md:115 (reading G1)     0, roots of Legendre P_{n-1} mapped to [0,1], 1
//   h_i, l_i         Eq. 19-20  Lagrange bases on the solution / flux points
#pragma once
#include <cmath>
#include <vector>

namespace chorus {

constexpr int kMaxOrder = 9;

struct Basis {
  int n = 0;
  std::vector<double> xs, xf;   // [n], [n+1]
  std::vector<double> Isf;      // [(n+1)][n]    h_i(xf_m)              solution -> flux interpolation
  std::vector<double> Dfs;      // [n][(n+1)]    l'_m(xs_i)             derivative of the flux polynomial at solution points
  std::vector<double> Efs;      // [n][(n+1)]    l_m(xs_i)              flux polynomial evaluated at solution points (geometry)
  std::vector<double> Dff;      // [(n+1)][(n+1)] l'_m(xf_a)            derivative on the flux-point grid (geometry)
  std::vector<double> Dss;      // [n][n]        sum_{m interior} Dfs[i][m] Isf[m][l]   (BR1 gradient, interior part)
  std::vector<double> wq;       // [n]           quadrature weights at the solution points (volume integrals, Eq. 34-35)
};

namespace detail {
typedef long double real;

inline std::vector<real> bary_weights(const std::vector<real>& x) {
  std::vector<real> w(x.size());
  for (size_t i = 0; i < x.size(); ++i) {
    real p = 1;
    for (size_t s = 0; s < x.size(); ++s)
      if (s != i) p *= (x[i] - x[s]);
    w[i] = 1 / p;
  }
  return w;
}
// value of every basis function of the node set x at X (barycentric second form; exact delta at a node)
inline std::vector<real> basis_at(const std::vector<real>& x, const std::vector<real>& w, real X) {
  std::vector<real> v(x.size(), 0);
  for (size_t i = 0; i < x.size(); ++i)
    if (X == x[i]) {
      v[i] = 1;
      return v;
    }
  real den = 0;
  for (size_t i = 0; i < x.size(); ++i) {
    v[i] = w[i] / (X - x[i]);
    den += v[i];
  }
  for (auto& t : v) t /= den;
  return v;
}
// derivative of every basis function of the node set x at X
inline std::vector<real> dbasis_at(const std::vector<real>& x, const std::vector<real>& w, real X) {
  const size_t N = x.size();
  std::vector<real> d(N, 0);
  for (size_t a = 0; a < N; ++a)
    if (X == x[a]) {   // at a node: D[a][m] = (w_m / w_a) / (x_a - x_m), diagonal by the zero row sum
      real diag = 0;
      for (size_t m = 0; m < N; ++m)
        if (m != a) {
          d[m] = (w[m] / w[a]) / (x[a] - x[m]);
          diag -= d[m];
        }
      d[a] = diag;
      return d;
    }
  std::vector<real> v = basis_at(x, w, X);
  // l_m'(X) = l_m(X) * ( sum_{q != m} 1/(X - x_q) )
  real tot = 0;
  for (size_t q = 0; q < N; ++q) tot += 1 / (X - x[q]);
  for (size_t m = 0; m < N; ++m) d[m] = v[m] * (tot - 1 / (X - x[m]));
  return d;
}
// roots of the Legendre polynomial of degree m in (-1,1), ascending (Newton on the three-term recurrence)
inline std::vector<real> legendre_roots(int m) {
  std::vector<real> r(m);
  const real pi = acosl(-1.0L);
  for (int k = 0; k < m; ++k) {
    real z = cosl(pi * (m - k - 0.25L) / (m + 0.5L));
    for (int it = 0; it < 200; ++it) {
      real pkm1 = 1, pk = z;
      for (int l = 1; l < m; ++l) {
        real pkp1 = ((2 * l + 1) * z * pk - l * pkm1) / (l + 1);
        pkm1 = pk;
        pk = pkp1;
      }
      real dp = m * (pkm1 - z * pk) / (1 - z * z);
      real dz = pk / dp;
      z -= dz;
      if (fabsl(dz) < 1e-19L) break;
    }
    r[k] = z;
  }
  // enforce exact symmetry about 0
  for (int k = 0; k < m / 2; ++k) {
    real s = 0.5L * (r[m - 1 - k] - r[k]);
    r[k] = -s;
    r[m - 1 - k] = s;
  }
  if (m % 2) r[m / 2] = 0;
  return r;
}
}  // namespace detail

inline Basis make_basis(int n) {
  using detail::real;
  Basis B;
  B.n = n;
  const int N1 = n + 1;
  const real pi = acosl(-1.0L);
  std::vector<real> xs(n), xf(N1);
  for (int k = 1; k <= n; ++k) xs[k - 1] = 0.5L * (1 - cosl((2 * k - 1) * pi / (2 * n)));
  std::vector<real> gl = detail::legendre_roots(n - 1);
  xf[0] = 0;
  xf[n] = 1;
  for (int k = 1; k < n; ++k) xf[k] = 0.5L * (1 + gl[k - 1]);
  std::vector<real> ws = detail::bary_weights(xs), wf = detail::bary_weights(xf);
  std::vector<real> Isf(N1 * n), Dfs(n * N1), Efs(n * N1), Dff(N1 * N1), Dss(n * n, 0);
  for (int m = 0; m < N1; ++m) {
    std::vector<real> h = detail::basis_at(xs, ws, xf[m]);
    for (int i = 0; i < n; ++i) Isf[m * n + i] = h[i];
    std::vector<real> d = detail::dbasis_at(xf, wf, xf[m]);
    for (int q = 0; q < N1; ++q) Dff[m * N1 + q] = d[q];
  }
  for (int i = 0; i < n; ++i) {
    std::vector<real> l = detail::basis_at(xf, wf, xs[i]);
    std::vector<real> d = detail::dbasis_at(xf, wf, xs[i]);
    for (int m = 0; m < N1; ++m) {
      Efs[i * N1 + m] = l[m];
      Dfs[i * N1 + m] = d[m];
    }
  }
  for (int i = 0; i < n; ++i)
    for (int l = 0; l < n; ++l) {
      real s = 0;
      for (int m = 1; m < n; ++m) s += Dfs[i * N1 + m] * Isf[m * n + l];
      Dss[i * n + l] = s;
    }
  auto cvt = [](const std::vector<real>& a) { return std::vector<double>(a.begin(), a.end()); };
  B.xs = cvt(xs);
  B.xf = cvt(xf);
  B.Isf = cvt(Isf);
  B.Dfs = cvt(Dfs);
  B.Efs = cvt(Efs);
  B.Dff = cvt(Dff);
  B.Dss = cvt(Dss);
  // Interpolatory quadrature on the Chebyshev-Gauss points of [0,1] = Fejer's first rule, closed form:
  // w_k = (1/n) [1 - 2 sum_{j=1}^{n/2} cos(2 j theta_k) / (4 j^2 - 1)], theta_k = (2k - 1) pi / (2n)
  B.wq.resize(n);
  for (int k = 1; k <= n; ++k) {
    const real th = (2 * k - 1) * pi / (2 * n);
    real w = 1;
    for (int q = 1; q <= n / 2; ++q) w -= 2 * cosl(2 * q * th) / (4.0L * q * q - 1);
    B.wq[k - 1] = (double)(w / n);
  }
  return B;
}

// Lagrange interpolation matrix from arbitrary abscissae g[ng] to the flux points: Gm[(n+1)][ng]
inline std::vector<double> geometry_interp(const Basis& B, const double* g, int ng) {
  using detail::real;
  std::vector<real> x(g, g + ng);
  std::vector<real> w = detail::bary_weights(x);
  std::vector<double> Gm((size_t)(B.n + 1) * ng);
  for (int m = 0; m <= B.n; ++m) {
    std::vector<real> v = detail::basis_at(x, w, (real)B.xf[m]);
    for (int q = 0; q < ng; ++q) Gm[(size_t)m * ng + q] = (double)v[q];
  }
  return Gm;
}

}  // namespace chorus
