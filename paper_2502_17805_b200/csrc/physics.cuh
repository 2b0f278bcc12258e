// physics.cuh -- pointwise physics of the CHORUS-MHD hot path as device functions (fp64).
//   conserved state / ideal gas   Eq. 2-4
//   source vector M               Eq. 5
//   inviscid ideal-MHD+GLM flux   Eq. 6
//   viscous/resistive/thermal     Eq. 7-10
//   Rusanov common flux
//   impenetrable stress-free walls, magnetic / thermal wall options  PAPER.md:190-198 (Eq. 32-33)
// Readings of the points where the paper is silent or garbled are listed in DESIGN.md (G1..G28).
#pragma once
#include <cstdint>

namespace chorus {

enum : uint32_t {
  kFlagDiffusion = 1u, kFlagGravity = 2u, kFlagCoriolis = 4u, kFlagPowell = 8u, kFlagGlmDamp = 16u,
  kFlagFixedTOuter = 32u, kFlagFixedFluxInner = 64u, kFlagCentrifugal = 128u
};

struct PhysD {
  double gamma, gm1, R, Cp, GM, Omega, nu, kappa, eta, c_h, a_psi, q_bottom, T_top;
  double iR, igamma;   // 1/R, 1/gamma
  int bc_inner, bc_outer;
  uint32_t flags;
};

struct PrimD {
  double rho, u, v, w, p, Bx, By, Bz, psi, E;
  double ir;   // 1/rho
};

__device__ __forceinline__ PrimD primitives(const PhysD& ph, const double* Q) {
  PrimD s;
  s.rho = Q[0];
  const double ir = 1.0 / Q[0];
  s.ir = ir;
  s.u = Q[1] * ir; s.v = Q[2] * ir; s.w = Q[3] * ir;
  s.E = Q[4];
  s.Bx = Q[5]; s.By = Q[6]; s.Bz = Q[7];
  s.psi = Q[8];
  const double ke = 0.5 * s.rho * (s.u * s.u + s.v * s.v + s.w * s.w);
  const double me = 0.5 * (s.Bx * s.Bx + s.By * s.By + s.Bz * s.Bz);
  s.p = ph.gm1 * (s.E - ke - me - 0.5 * s.psi * s.psi);        // Eq. 3
  return s;
}

// F~ = S . F_inv (Eq. 6 contracted with an area vector, Eq. 17).  WALL: u.S is literally zero.
template <bool WALL>
__device__ __forceinline__ void flux_inviscid(const PhysD& ph, const PrimD& s, double Sx, double Sy, double Sz, double* F) {
  const double uS = WALL ? 0.0 : s.u * Sx + s.v * Sy + s.w * Sz;
  const double BS = s.Bx * Sx + s.By * Sy + s.Bz * Sz;
  const double pstar = s.p + 0.5 * (s.Bx * s.Bx + s.By * s.By + s.Bz * s.Bz);
  const double e = s.E - 0.5 * s.psi * s.psi;
  const double uB = s.u * s.Bx + s.v * s.By + s.w * s.Bz;
  const double chpsi = ph.c_h * s.psi;
  const double ruS = s.rho * uS;
  F[0] = ruS;
  F[1] = ruS * s.u + pstar * Sx - s.Bx * BS;
  F[2] = ruS * s.v + pstar * Sy - s.By * BS;
  F[3] = ruS * s.w + pstar * Sz - s.Bz * BS;
  F[4] = (e + pstar) * uS - uB * BS + chpsi * BS;
  F[5] = s.Bx * uS - s.u * BS + chpsi * Sx;
  F[6] = s.By * uS - s.v * BS + chpsi * Sy;
  F[7] = s.Bz * uS - s.w * BS + chpsi * Sz;
  F[8] = ph.c_h * BS;
}

// Stress tensor, heat flux, B x J and grad B from (prims, grad Q);  G[3*v+j] = d Q_v / d x_j  (Eq. 7-10)
struct ViscD {
  double tau[3][3], q[3], BxJ[3], dB[3][3];
};
__device__ __forceinline__ void viscous_terms(const PhysD& ph, const PrimD& s, const double* G, double kr, ViscD& V) {
  const double uu[3] = {s.u, s.v, s.w}, BB[3] = {s.Bx, s.By, s.Bz};
  const double ir = 1.0 / s.rho;
  double du[3][3];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      du[i][j] = (G[(1 + i) * 3 + j] - uu[i] * G[j]) * ir;       // d_j u_i
      V.dB[i][j] = G[(5 + i) * 3 + j];
    }
  const double u2 = s.u * s.u + s.v * s.v + s.w * s.w;
  const double Tt = s.p * ir / ph.R;
  const double mu = s.rho * ph.nu;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    const double udm = s.u * G[3 + j] + s.v * G[6 + j] + s.w * G[9 + j];
    const double BdB = s.Bx * V.dB[0][j] + s.By * V.dB[1][j] + s.Bz * V.dB[2][j];
    const double dp = ph.gm1 * (G[12 + j] - udm + 0.5 * u2 * G[j] - BdB - s.psi * G[24 + j]);
    const double dT = (dp - s.p * ir * G[j]) * ir / ph.R;
    const double dS = ph.Cp * (dp / (ph.gamma * s.p) - G[j] * ir);                 // gradient of Eq. 10
    V.q[j] = -ph.kappa * s.rho * Tt * dS - kr * s.rho * ph.Cp * dT;                  // Eq. 9
  }
  const double divu = du[0][0] + du[1][1] + du[2][2];
  const double lamdiv = -(2.0 / 3.0) * mu * divu;                                     // Stokes
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) V.tau[i][j] = mu * (du[i][j] + du[j][i]) + (i == j ? lamdiv : 0.0);   // Eq. 8
  const double J0 = V.dB[2][1] - V.dB[1][2], J1 = V.dB[0][2] - V.dB[2][0], J2 = V.dB[1][0] - V.dB[0][1];
  V.BxJ[0] = BB[1] * J2 - BB[2] * J1;
  V.BxJ[1] = BB[2] * J0 - BB[0] * J2;
  V.BxJ[2] = BB[0] * J1 - BB[1] * J0;
}
// F~_vis = S . F_vis; only rows 1..7 are non-zero: Fv[0..2] momentum, Fv[3] energy, Fv[4..6] induction
__device__ __forceinline__ void flux_viscous(const PhysD& ph, const PrimD& s, const double* G, double Sx, double Sy, double Sz,
                                             double kr, double* Fv) {
  ViscD V;
  viscous_terms(ph, s, G, kr, V);
  const double S[3] = {Sx, Sy, Sz}, uu[3] = {s.u, s.v, s.w};
#pragma unroll
  for (int c = 0; c < 7; ++c) Fv[c] = 0.0;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
#pragma unroll
    for (int i = 0; i < 3; ++i) Fv[i] += S[j] * V.tau[j][i];
    const double work = uu[0] * V.tau[j][0] + uu[1] * V.tau[j][1] + uu[2] * V.tau[j][2];
    Fv[3] += S[j] * (work - V.q[j] + ph.eta * V.BxJ[j]);
#pragma unroll
    for (int i = 0; i < 3; ++i) Fv[4 + i] += S[j] * ph.eta * (V.dB[i][j] - V.dB[j][i]);
  }
}

__device__ __forceinline__ double fast_speed(const PhysD& ph, const PrimD& s, double nx, double ny, double nz) {
  const double ir = s.ir;
  const double a2 = ph.gamma * s.p * ir;
  const double Bn = s.Bx * nx + s.By * ny + s.Bz * nz;
  const double b2 = (s.Bx * s.Bx + s.By * s.By + s.Bz * s.Bz) * ir, bn2 = Bn * Bn * ir;
  const double t = a2 + b2;
  const double disc = fmax(t * t - 4.0 * a2 * bn2, 0.0);
  return sqrt(0.5 * (t + sqrt(disc)));
}

// Rusanov flux along the unit normal (nx,ny,nz):  1/2 (F(Qi)+F(Qo)) - 1/2 lambda (Qo - Qi)
__device__ __forceinline__ void flux_rusanov(const PhysD& ph, const double* Qi, const double* Qo, double nx, double ny, double nz,
                                             double* F) {
  const PrimD si = primitives(ph, Qi), so = primitives(ph, Qo);
  const double li = fabs(si.u * nx + si.v * ny + si.w * nz) + fast_speed(ph, si, nx, ny, nz);
  const double lo = fabs(so.u * nx + so.v * ny + so.w * nz) + fast_speed(ph, so, nx, ny, nz);
  const double lam = fmax(fmax(li, lo), ph.c_h);
  double Fi[9], Fo[9];
  flux_inviscid<false>(ph, si, nx, ny, nz, Fi);
  flux_inviscid<false>(ph, so, nx, ny, nz, Fo);
#pragma unroll
  for (int c = 0; c < 9; ++c) F[c] = 0.5 * (Fi[c] + Fo[c]) - 0.5 * lam * (Qo[c] - Qi[c]);
}

// Boundary state at a wall (wall = -1 inner, -2 outer) with outward unit normal n
__device__ __forceinline__ void wall_state(const PhysD& ph, int wall, const double* Q, double nx, double ny, double nz, double* Qb) {
  const PrimD s = primitives(ph, Q);
  const double un = s.u * nx + s.v * ny + s.w * nz;
  const double Bn = s.Bx * nx + s.By * ny + s.Bz * nz;
  const int bc = (wall == -1) ? ph.bc_inner : ph.bc_outer;
  const double ub = s.u - un * nx, vb = s.v - un * ny, wb = s.w - un * nz;               // Eq. 33
  double bx, by, bz;
  if (bc == 0) { bx = s.Bx - Bn * nx; by = s.By - Bn * ny; bz = s.Bz - Bn * nz; }        // conducting: B_r = 0
  else { bx = Bn * nx; by = Bn * ny; bz = Bn * nz; }                                     // radial: B_theta = B_phi = 0
  double pb = s.p;
  if (wall == -2 && (ph.flags & kFlagFixedTOuter)) pb = s.rho * ph.R * ph.T_top;
  Qb[0] = s.rho;
  Qb[1] = s.rho * ub; Qb[2] = s.rho * vb; Qb[3] = s.rho * wb;
  Qb[5] = bx; Qb[6] = by; Qb[7] = bz;
  Qb[8] = s.psi;
  Qb[4] = pb / ph.gm1 + 0.5 * s.rho * (ub * ub + vb * vb + wb * wb) + 0.5 * (bx * bx + by * by + bz * bz) + 0.5 * s.psi * s.psi;
}

// Viscous wall flux along the outward unit normal from (Q_b, grad Q_in): stress-free (normal traction only), no
// viscous work, prescribed or computed heat flux, resistive terms only on a radial-field wall.  Fv as flux_viscous.
__device__ __forceinline__ void flux_wall_viscous(const PhysD& ph, int wall, const PrimD& sb, const double* G, double nx, double ny,
                                                  double nz, double kr, double* Fv) {
  ViscD V;
  viscous_terms(ph, sb, G, kr, V);
  const double nh[3] = {nx, ny, nz};
  const int bc = (wall == -1) ? ph.bc_inner : ph.bc_outer;
  double tn = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) tn += (V.tau[i][0] * nx + V.tau[i][1] * ny + V.tau[i][2] * nz) * nh[i];
#pragma unroll
  for (int i = 0; i < 3; ++i) Fv[i] = tn * nh[i];
  double qn = V.q[0] * nx + V.q[1] * ny + V.q[2] * nz;
  if (wall == -1 && (ph.flags & kFlagFixedFluxInner)) qn = -ph.q_bottom;                 // Eq. 32
  double res = 0.0;
  Fv[4] = Fv[5] = Fv[6] = 0.0;
  if (bc != 0) {
    res = ph.eta * (V.BxJ[0] * nx + V.BxJ[1] * ny + V.BxJ[2] * nz);
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = 0; j < 3; ++j) Fv[4 + i] += nh[j] * ph.eta * (V.dB[i][j] - V.dB[j][i]);
  }
  Fv[3] = -qn + res;
}

// Source vector M of Eq. 5 added to R[9]; divB from the BR1 gradient
__device__ __forceinline__ void add_sources(const PhysD& ph, const PrimD& s, double divB, double x, double y, double z, double* R) {
  if (ph.flags & kFlagGravity) {
    const double r2 = x * x + y * y + z * z;
    const double f = -ph.GM / (r2 * sqrt(r2));
    const double gx = f * x, gy = f * y, gz = f * z;
    R[1] += s.rho * gx; R[2] += s.rho * gy; R[3] += s.rho * gz;
    R[4] += s.rho * (s.u * gx + s.v * gy + s.w * gz);
  }
  if (ph.flags & kFlagCoriolis) {
    R[1] += 2.0 * s.rho * ph.Omega * s.v;
    R[2] -= 2.0 * s.rho * ph.Omega * s.u;
  }
  if (ph.flags & kFlagCentrifugal) {
    const double cx = s.rho * ph.Omega * ph.Omega * x, cy = s.rho * ph.Omega * ph.Omega * y;
    R[1] += cx; R[2] += cy;
    R[4] += s.u * cx + s.v * cy;
  }
  if (ph.flags & kFlagPowell) {
    const double uB = s.u * s.Bx + s.v * s.By + s.w * s.Bz;
    R[1] -= divB * s.Bx; R[2] -= divB * s.By; R[3] -= divB * s.Bz;
    R[4] -= divB * uB;
    R[5] -= divB * s.u; R[6] -= divB * s.v; R[7] -= divB * s.w;
  }
  if (ph.flags & kFlagGlmDamp) R[8] -= ph.a_psi * s.psi;
}

__device__ __forceinline__ double wavespeed(const PhysD& ph, const double* Q) {
  const PrimD s = primitives(ph, Q);
  const double B2 = s.Bx * s.Bx + s.By * s.By + s.Bz * s.Bz;
  return sqrt(s.u * s.u + s.v * s.v + s.w * s.w) + sqrt((ph.gamma * s.p + B2) / s.rho);
}

}  // namespace chorus
