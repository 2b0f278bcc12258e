// sd_mhd_oracle.cpp -- CPU ORACLE for the CHORUS-MHD hot path (TEST INFRASTRUCTURE, NOT PRODUCT CODE).
//
// A plain, slow, literal implementation of the spectral-difference (SD) residual of the compressible
// MHD + GLM equations on curved hexahedra, and of the SSPRK(5,3) step, written step by step from
// /root/reference/PAPER.md (arxiv 2502.17805) in the paper's order and notation.  No blocking, no
// fusion, no reordering beyond what the paper's procedure states; OpenMP only over whole elements.
// Shares no code with the CUDA library.  Citations: PAPER.md:<line> (section / equation).
// Where the paper is silent or garbled the readings G1..G28 of DESIGN.md ("Readings") are taken.
//
// Parity status of the readings the paper cannot pin: wall details
// G16-G19, the Rusanov wave-speed estimate G14, mu = rho*nu G11, C_h and a (inputs) G21.
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC   (see oracle/build.py)
#include "sd_mhd_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <vector>

namespace {

enum : uint32_t { F_DIFF = 1u, F_GRAV = 2u, F_CORI = 4u, F_POWELL = 8u, F_GLMDAMP = 16u, F_TTOP = 32u, F_QBOT = 64u, F_CENTRI = 128u };

template <class T>
struct Phys {
  T gamma, R, Cp, GM, Omega, nu, kappa, eta, kr_scale, kr_c[3], kr_wscale, c_h, a_psi, q_bottom, T_top;
  int bc_inner, bc_outer;
  uint32_t flags;
  explicit Phys(const oracle_physics& p)
      : gamma(p.gamma), R(p.R_gas), Cp(p.Cp), GM(p.GM), Omega(p.Omega), nu(p.nu), kappa(p.kappa), eta(p.eta),
        kr_scale(p.kr_scale), kr_wscale(p.kr_wscale), c_h(p.c_h), a_psi(p.a_psi), q_bottom(p.q_bottom),
        T_top(p.T_top), bc_inner(p.bc_mag_inner), bc_outer(p.bc_mag_outer), flags(p.flags) {
    for (int i = 0; i < 3; ++i) kr_c[i] = p.kr_c[i];
  }
};

// ------------------------------------------------------------------------------------------------
// O4  primitives: U = m/rho;  p from Eq. 3;  T = p/(rho R) (Eq. 4)
// ------------------------------------------------------------------------------------------------
template <class T>
struct Prim {
  T rho, u[3], p, B[3], psi, E;
};
template <class T>
Prim<T> primitives(const Phys<T>& ph, const T* Q) {
  Prim<T> w;
  w.rho = Q[0];
  for (int i = 0; i < 3; ++i) w.u[i] = Q[1 + i] / Q[0];
  w.E = Q[4];
  for (int i = 0; i < 3; ++i) w.B[i] = Q[5 + i];
  w.psi = Q[8];
  T ke = T(0.5) * w.rho * (w.u[0] * w.u[0] + w.u[1] * w.u[1] + w.u[2] * w.u[2]);
  T me = T(0.5) * (w.B[0] * w.B[0] + w.B[1] * w.B[1] + w.B[2] * w.B[2]);
  w.p = (ph.gamma - T(1)) * (w.E - ke - me - T(0.5) * w.psi * w.psi);
  return w;
}

// ------------------------------------------------------------------------------------------------
// O10  inviscid flux of Eq. 6 contracted with an area vector S  (readings G6, G7)
// ------------------------------------------------------------------------------------------------
template <class T>
void flux_inviscid(const Phys<T>& ph, const T* Q, const T* S, T* F, bool wall = false) {
  Prim<T> w = primitives(ph, Q);
  T uS = wall ? T(0) : w.u[0] * S[0] + w.u[1] * S[1] + w.u[2] * S[2];   // wall: u.S is literal 0 (G16)
  T BS = w.B[0] * S[0] + w.B[1] * S[1] + w.B[2] * S[2];
  T B2 = w.B[0] * w.B[0] + w.B[1] * w.B[1] + w.B[2] * w.B[2];
  T pstar = w.p + T(0.5) * B2;                       // p + |B|^2/2
  T e = w.E - T(0.5) * w.psi * w.psi;                // e of Eq. 3
  T uB = w.u[0] * w.B[0] + w.u[1] * w.B[1] + w.u[2] * w.B[2];
  F[0] = w.rho * uS;
  for (int i = 0; i < 3; ++i) F[1 + i] = w.rho * w.u[i] * uS + pstar * S[i] - w.B[i] * BS;
  F[4] = (e + pstar) * uS - uB * BS + ph.c_h * w.psi * BS;
  for (int i = 0; i < 3; ++i) F[5 + i] = w.B[i] * uS - w.u[i] * BS + ph.c_h * w.psi * S[i];
  F[8] = ph.c_h * BS;
}

// The same expression with every product replaced by its modulus and every sum by a sum of moduli:
// the forward-error scale of the inviscid flux (used only for the magnitude residual of reading G24).
template <class T>
void flux_inviscid_abs(const Phys<T>& ph, const T* Q, const T* S, T* F, bool wall = false) {
  Prim<T> w = primitives(ph, Q);
  auto ab = [](T x) { return std::fabs(x); };
  T uS = wall ? T(0) : ab(w.u[0] * S[0]) + ab(w.u[1] * S[1]) + ab(w.u[2] * S[2]);
  T BS = ab(w.B[0] * S[0]) + ab(w.B[1] * S[1]) + ab(w.B[2] * S[2]);
  T B2 = w.B[0] * w.B[0] + w.B[1] * w.B[1] + w.B[2] * w.B[2];
  T pstar = ab(w.p) + T(0.5) * B2;
  T e = ab(w.E) + T(0.5) * w.psi * w.psi;
  T uB = ab(w.u[0] * w.B[0]) + ab(w.u[1] * w.B[1]) + ab(w.u[2] * w.B[2]);
  F[0] = ab(w.rho) * uS;
  for (int i = 0; i < 3; ++i) F[1 + i] = ab(w.rho * w.u[i]) * uS + pstar * ab(S[i]) + ab(w.B[i]) * BS;
  F[4] = (e + pstar) * uS + uB * BS + ab(ph.c_h * w.psi) * BS;
  for (int i = 0; i < 3; ++i) F[5 + i] = ab(w.B[i]) * uS + ab(w.u[i]) * BS + ab(ph.c_h * w.psi * S[i]);
  F[8] = ab(ph.c_h) * BS;
}

// ------------------------------------------------------------------------------------------------
// O9  viscous / resistive / thermal flux of Eq. 7-10 from (Q, grad Q)  (G8, G10, G11)
//     G[3*v+j] = d Q_v / d x_j.
// ------------------------------------------------------------------------------------------------
template <class T>
struct Visc {
  T tau[3][3], q[3], BxJ[3], dB[3][3];   // dB[i][j] = d_j B_i
  T dT[3];                                 // grad T
};
template <class T>
Visc<T> viscous_terms(const Phys<T>& ph, const Prim<T>& w, const T* G, T kr) {
  Visc<T> v;
  T drho[3], dm[3][3], dE[3], dpsi[3];
  for (int j = 0; j < 3; ++j) {
    drho[j] = G[0 * 3 + j];
    for (int i = 0; i < 3; ++i) dm[i][j] = G[(1 + i) * 3 + j];
    dE[j] = G[4 * 3 + j];
    for (int i = 0; i < 3; ++i) v.dB[i][j] = G[(5 + i) * 3 + j];
    dpsi[j] = G[8 * 3 + j];
  }
  T du[3][3];   // du[i][j] = d_j u_i = (d_j m_i - u_i d_j rho)/rho
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) du[i][j] = (dm[i][j] - w.u[i] * drho[j]) / w.rho;
  T u2 = w.u[0] * w.u[0] + w.u[1] * w.u[1] + w.u[2] * w.u[2];
  T dp[3], dT[3], dS[3];
  for (int j = 0; j < 3; ++j) {
    T udm = w.u[0] * dm[0][j] + w.u[1] * dm[1][j] + w.u[2] * dm[2][j];
    T BdB = w.B[0] * v.dB[0][j] + w.B[1] * v.dB[1][j] + w.B[2] * v.dB[2][j];
    dp[j] = (ph.gamma - T(1)) * (dE[j] - udm + T(0.5) * u2 * drho[j] - BdB - w.psi * dpsi[j]);
    dT[j] = (dp[j] - (w.p / w.rho) * drho[j]) / (w.rho * ph.R);
    dS[j] = ph.Cp * (dp[j] / (ph.gamma * w.p) - drho[j] / w.rho);          // gradient of Eq. 10
  }
  T mu = w.rho * ph.nu;                      // G11
  T lam = -(T(2) / T(3)) * mu;               // Stokes
  T divu = du[0][0] + du[1][1] + du[2][2];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) v.tau[i][j] = mu * (du[i][j] + du[j][i]) + (i == j ? lam * divu : T(0));   // Eq. 8
  T Tt = w.p / (w.rho * ph.R);
  for (int j = 0; j < 3; ++j) v.q[j] = -ph.kappa * w.rho * Tt * dS[j] - kr * w.rho * ph.Cp * dT[j];      // Eq. 9
  for (int j = 0; j < 3; ++j) v.dT[j] = dT[j];
  T J[3] = {v.dB[2][1] - v.dB[1][2], v.dB[0][2] - v.dB[2][0], v.dB[1][0] - v.dB[0][1]};                  // J = curl B
  v.BxJ[0] = w.B[1] * J[2] - w.B[2] * J[1];
  v.BxJ[1] = w.B[2] * J[0] - w.B[0] * J[2];
  v.BxJ[2] = w.B[0] * J[1] - w.B[1] * J[0];
  return v;
}
template <class T>
void flux_viscous(const Phys<T>& ph, const T* Q, const T* G, const T* S, T kr, T* F) {
  Prim<T> w = primitives(ph, Q);
  Visc<T> v = viscous_terms(ph, w, G, kr);
  for (int c = 0; c < 9; ++c) F[c] = T(0);
  for (int j = 0; j < 3; ++j) {   // F~ = sum_j S_j F_vis,j  (Eq. 7 rows; Eq. 17)
    for (int i = 0; i < 3; ++i) F[1 + i] += S[j] * v.tau[j][i];
    T work = w.u[0] * v.tau[j][0] + w.u[1] * v.tau[j][1] + w.u[2] * v.tau[j][2];
    F[4] += S[j] * (work - v.q[j] + ph.eta * v.BxJ[j]);
    for (int i = 0; i < 3; ++i) F[5 + i] += S[j] * ph.eta * (v.dB[i][j] - v.dB[j][i]);   // G10
  }
}

// ------------------------------------------------------------------------------------------------
// O11  Rusanov common flux (ref [7]) along a unit normal  (reading G14)
// ------------------------------------------------------------------------------------------------
template <class T>
T fast_speed(const Phys<T>& ph, const Prim<T>& w, const T* nh) {
  T a2 = ph.gamma * w.p / w.rho;
  T B2 = w.B[0] * w.B[0] + w.B[1] * w.B[1] + w.B[2] * w.B[2];
  T Bn = w.B[0] * nh[0] + w.B[1] * nh[1] + w.B[2] * nh[2];
  T b2 = B2 / w.rho, bn2 = Bn * Bn / w.rho;
  T s = a2 + b2;
  T disc = s * s - T(4) * a2 * bn2;
  if (disc < T(0)) disc = T(0);
  return std::sqrt(T(0.5) * (s + std::sqrt(disc)));
}
template <class T>
void flux_rusanov(const Phys<T>& ph, const T* Qi, const T* Qo, const T* nh, T* F, T* Fabs = nullptr) {
  Prim<T> wi = primitives(ph, Qi), wo = primitives(ph, Qo);
  T uni = wi.u[0] * nh[0] + wi.u[1] * nh[1] + wi.u[2] * nh[2];
  T uno = wo.u[0] * nh[0] + wo.u[1] * nh[1] + wo.u[2] * nh[2];
  T li = std::fabs(uni) + fast_speed(ph, wi, nh), lo = std::fabs(uno) + fast_speed(ph, wo, nh);
  T lam = std::max(std::max(li, lo), ph.c_h);
  T Fi[9], Fo[9];
  flux_inviscid(ph, Qi, nh, Fi);
  flux_inviscid(ph, Qo, nh, Fo);
  for (int c = 0; c < 9; ++c) F[c] = T(0.5) * (Fi[c] + Fo[c]) - T(0.5) * lam * (Qo[c] - Qi[c]);
  if (Fabs) {   // moduli of the terms, for the magnitude residual (G24)
    flux_inviscid_abs(ph, Qi, nh, Fi);
    flux_inviscid_abs(ph, Qo, nh, Fo);
    for (int c = 0; c < 9; ++c)
      Fabs[c] = T(0.5) * (Fi[c] + Fo[c]) + T(0.5) * lam * (std::fabs(Qo[c]) + std::fabs(Qi[c]));
  }
}

// ------------------------------------------------------------------------------------------------
// O12  walls (Eq. 32-33)  (readings G16-G19; parity unpinned by the paper)
// ------------------------------------------------------------------------------------------------
template <class T>
void wall_state(const Phys<T>& ph, int wall, const T* Q, const T* nh, T* Qb) {
  Prim<T> w = primitives(ph, Q);
  T un = w.u[0] * nh[0] + w.u[1] * nh[1] + w.u[2] * nh[2];
  T Bn = w.B[0] * nh[0] + w.B[1] * nh[1] + w.B[2] * nh[2];
  int bc = (wall == -1) ? ph.bc_inner : ph.bc_outer;
  T ub[3], Bb[3];
  for (int i = 0; i < 3; ++i) {
    ub[i] = w.u[i] - un * nh[i];                               // Eq. 33: U.r = 0
    Bb[i] = (bc == 0) ? (w.B[i] - Bn * nh[i]) : (Bn * nh[i]);   // conducting: B_r = 0; radial: B_theta = B_phi = 0
  }
  T pb = w.p;
  if (wall == -2 && (ph.flags & F_TTOP)) pb = w.rho * ph.R * ph.T_top;   // constant-temperature outer surface
  Qb[0] = w.rho;
  for (int i = 0; i < 3; ++i) Qb[1 + i] = w.rho * ub[i];
  for (int i = 0; i < 3; ++i) Qb[5 + i] = Bb[i];
  Qb[8] = w.psi;
  Qb[4] = pb / (ph.gamma - T(1)) + T(0.5) * w.rho * (ub[0] * ub[0] + ub[1] * ub[1] + ub[2] * ub[2]) +
          T(0.5) * (Bb[0] * Bb[0] + Bb[1] * Bb[1] + Bb[2] * Bb[2]) + T(0.5) * w.psi * w.psi;   // Eq. 3
}
// Wall viscous flux along the outward unit normal nh from (Q_b, grad Q_in), with the wall conditions applied to the WALL
// GRADIENTS as PAPER.md:198 describes ("transforming the Jacobian of the magnetic field into spherical coordinates and
// setting the appropriate derivatives to zero"; stress tensor "converted to spherical coordinates, and the angular components
// are set to zero"), reading G29 of DESIGN.md:
//   frame     (e_r, t_1, t_2) at the wall point, e_r = the wall's radial direction = +nh on the outer wall, -nh on the inner
//             wall (on the paper's spherical shells this is the spherical frame), r = rw = distance of the point from the origin;
//             in this frame the spherical component derivatives are  d_r B_a = e_a.(dB/dr)  and, along a tangent t,
//             d_t B_r = e_r.(dB/dt) + B_t/r,  d_s B_t = e_t.(dB/ds) - delta_st B_r/r  (the unit vectors turn with the position);
//   conductor B_r = 0 on the whole surface, d_r(r B_t) = 0:   D[r][t] = -B_t/r (so that d_t B_r = 0),  D[t][r] = -B_t/r;
//   radial    B_t = 0 on the whole surface, d_r(r^2 B_r) = 0:  D[s][t] = delta_st B_r/r (d_s B_t = 0),  D[r][r] = -2 B_r/r
//             (the conditioned Jacobian is divergence free: "to maintain the divergence-free magnetic field");
//   where D[a][b] = e_a.(grad B).e_b is the Cartesian Jacobian in the wall frame and B is the wall state's field.  The
//   conditioned Jacobian gives the current J = curl B of the resistive terms only: grad p, grad T, grad S come from the
//   unconditioned conserved gradients (conditioning grad B without grad E would change grad p);
//   stress    tau_rt = tau_tr = 0 (stress-free);
//   thermal   constant-temperature outer wall: T is uniform on the surface, the tangential part of grad T is zero;
//             constant-flux inner wall: q.r_hat = q_bottom (Eq. 32).
// rw <= 0 stands for a plane wall (1/r = 0).
template <class T>
void wall_frame(const T* er, T R[3][3]) {          // columns of R: e_r, t_1, t_2 (right-handed, orthonormal)
  int k = 0;                                       // Cartesian axis least aligned with e_r
  for (int i = 1; i < 3; ++i)
    if (std::fabs(er[i]) < std::fabs(er[k])) k = i;
  T a[3] = {T(0), T(0), T(0)};
  a[k] = T(1);
  T t1[3] = {er[1] * a[2] - er[2] * a[1], er[2] * a[0] - er[0] * a[2], er[0] * a[1] - er[1] * a[0]};
  T nrm = std::sqrt(t1[0] * t1[0] + t1[1] * t1[1] + t1[2] * t1[2]);
  for (int i = 0; i < 3; ++i) t1[i] /= nrm;
  T t2[3] = {er[1] * t1[2] - er[2] * t1[1], er[2] * t1[0] - er[0] * t1[2], er[0] * t1[1] - er[1] * t1[0]};
  for (int i = 0; i < 3; ++i) { R[i][0] = er[i]; R[i][1] = t1[i]; R[i][2] = t2[i]; }
}
template <class T>
void to_frame(const T R[3][3], const T A[3][3], T D[3][3]) {      // D = R^T A R
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) {
      T s = T(0);
      for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) s += R[i][a] * A[i][j] * R[j][b];
      D[a][b] = s;
    }
}
template <class T>
void from_frame(const T R[3][3], const T D[3][3], T A[3][3]) {    // A = R D R^T
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      T s = T(0);
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) s += R[i][a] * D[a][b] * R[j][b];
      A[i][j] = s;
    }
}
// the conditioned Jacobian of B (dBc[i][j] = d_j B_i, Cartesian) of a wall with magnetic condition bc (0 conductor, 1 radial)
template <class T>
void wall_condition_gradB(int bc, const T dB[3][3], const T* Bb, const T* er, T rw, T dBc[3][3]) {
  T R[3][3], D[3][3];
  wall_frame(er, R);
  to_frame(R, dB, D);
  T ir = rw > T(0) ? T(1) / rw : T(0);
  T Bl[3];                                         // wall-state field in the frame: (B_r, B_1, B_2)
  for (int a = 0; a < 3; ++a) Bl[a] = Bb[0] * R[0][a] + Bb[1] * R[1][a] + Bb[2] * R[2][a];
  if (bc == 0) {
    for (int t = 1; t < 3; ++t) {
      D[0][t] = -Bl[t] * ir;                       // d_t B_r = 0 on the surface
      D[t][0] = -Bl[t] * ir;                       // d_r (r B_t) = 0
    }
  } else {
    for (int s_ = 1; s_ < 3; ++s_)
      for (int t = 1; t < 3; ++t) D[t][s_] = (s_ == t) ? Bl[0] * ir : T(0);   // d_s B_t = 0 on the surface
    D[0][0] = -T(2) * Bl[0] * ir;                  // d_r (r^2 B_r) = 0
  }
  from_frame(R, D, dBc);
}
template <class T>
void flux_wall_viscous(const Phys<T>& ph, int wall, const T* Qb, const T* G, const T* nh, T rw, T kr, T* F) {
  Prim<T> w = primitives(ph, Qb);
  Visc<T> v = viscous_terms(ph, w, G, kr);
  int bc = (wall == -1) ? ph.bc_inner : ph.bc_outer;
  T sgn = (wall == -1) ? T(-1) : T(1);
  T er[3] = {sgn * nh[0], sgn * nh[1], sgn * nh[2]};
  T R[3][3];
  wall_frame(er, R);
  // stress-free: angular components of the stress tensor in the wall frame set to zero
  T tl[3][3], tc[3][3];
  to_frame(R, v.tau, tl);
  for (int t = 1; t < 3; ++t) tl[0][t] = tl[t][0] = T(0);
  from_frame(R, tl, tc);
  // magnetic wall: conditioned Jacobian of B, its current density
  T dBc[3][3];
  wall_condition_gradB(bc, v.dB, w.B, er, rw, dBc);
  T J[3] = {dBc[2][1] - dBc[1][2], dBc[0][2] - dBc[2][0], dBc[1][0] - dBc[0][1]};
  T BxJ[3] = {w.B[1] * J[2] - w.B[2] * J[1], w.B[2] * J[0] - w.B[0] * J[2], w.B[0] * J[1] - w.B[1] * J[0]};
  // thermal walls
  T q[3] = {v.q[0], v.q[1], v.q[2]};
  if (wall == -2 && (ph.flags & F_TTOP)) {         // uniform T on the surface: only the radial part of grad T conducts
    T dTr = v.dT[0] * er[0] + v.dT[1] * er[1] + v.dT[2] * er[2];
    for (int j = 0; j < 3; ++j) q[j] += kr * w.rho * ph.Cp * (v.dT[j] - dTr * er[j]);
  }
  T qn = q[0] * nh[0] + q[1] * nh[1] + q[2] * nh[2];
  if (wall == -1 && (ph.flags & F_QBOT)) qn = -ph.q_bottom;     // Eq. 32: q = q_b r_hat, outward normal = -r_hat
  for (int c = 0; c < 9; ++c) F[c] = T(0);
  T work = T(0);
  for (int i = 0; i < 3; ++i) {
    T ti = tc[i][0] * nh[0] + tc[i][1] * nh[1] + tc[i][2] * nh[2];     // traction of the conditioned stress
    F[1 + i] = ti;
    work += w.u[i] * ti;                                               // U_b . t (U_b is tangent, t is normal: round-off)
  }
  F[4] = work - qn + ph.eta * (BxJ[0] * nh[0] + BxJ[1] * nh[1] + BxJ[2] * nh[2]);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) F[5 + i] += nh[j] * ph.eta * (dBc[i][j] - dBc[j][i]);
}

// ------------------------------------------------------------------------------------------------
// O13  source vector M of Eq. 5; Mabs = sum of the moduli of the individual terms
// ------------------------------------------------------------------------------------------------
template <class T>
void source(const Phys<T>& ph, const T* Q, const T* G, const T* x, T* M, T* Mabs) {
  Prim<T> w = primitives(ph, Q);
  for (int c = 0; c < 9; ++c) M[c] = Mabs[c] = T(0);
  auto add = [&](int c, T v) { M[c] += v; Mabs[c] += std::fabs(v); };
  if (ph.flags & F_GRAV) {
    T r2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
    T r = std::sqrt(r2);
    T g[3];
    for (int i = 0; i < 3; ++i) g[i] = -ph.GM * x[i] / (r2 * r);         // g = -GM r_hat / r^2
    for (int i = 0; i < 3; ++i) add(1 + i, w.rho * g[i]);
    for (int i = 0; i < 3; ++i) add(4, w.rho * w.u[i] * g[i]);
  }
  if (ph.flags & F_CORI) {                                                 // -2 rho Omega x U, Omega = Omega z_hat
    add(1, T(2) * w.rho * ph.Omega * w.u[1]);
    add(2, -T(2) * w.rho * ph.Omega * w.u[0]);
  }
  if (ph.flags & F_CENTRI) {                                               // optional, not in Eq. 5 (G22)
    T cx = w.rho * ph.Omega * ph.Omega * x[0], cy = w.rho * ph.Omega * ph.Omega * x[1];
    add(1, cx);
    add(2, cy);
    add(4, w.u[0] * cx + w.u[1] * cy);
  }
  if (ph.flags & F_POWELL) {
    T divB = G[5 * 3 + 0] + G[6 * 3 + 1] + G[7 * 3 + 2];
    T uB = w.u[0] * w.B[0] + w.u[1] * w.B[1] + w.u[2] * w.B[2];
    for (int i = 0; i < 3; ++i) add(1 + i, -divB * w.B[i]);
    add(4, -divB * uB);
    for (int i = 0; i < 3; ++i) add(5 + i, -divB * w.u[i]);
  }
  if (ph.flags & F_GLMDAMP) add(8, -ph.a_psi * w.psi);
}

// O15  max over directions of |U| + c_f  (reading G20)
template <class T>
T wavespeed(const Phys<T>& ph, const T* Q) {
  Prim<T> w = primitives(ph, Q);
  T u = std::sqrt(w.u[0] * w.u[0] + w.u[1] * w.u[1] + w.u[2] * w.u[2]);
  T B2 = w.B[0] * w.B[0] + w.B[1] * w.B[1] + w.B[2] * w.B[2];
  return u + std::sqrt((ph.gamma * w.p + B2) / w.rho);
}

// ------------------------------------------------------------------------------------------------
// O1, O2  node sets and 1-D operators (Eq. 18-20; readings G1, G2)
// ------------------------------------------------------------------------------------------------
template <class T>
T lagrange(const std::vector<T>& x, int i, T X) {          // Eq. 19 / 20: prod_{s != i} (X - x_s)/(x_i - x_s)
  T v = T(1);
  for (int s = 0; s < (int)x.size(); ++s)
    if (s != i) v *= (X - x[s]) / (x[i] - x[s]);
  return v;
}
template <class T>
T lagrange_deriv(const std::vector<T>& x, int i, T X) {    // d/dX of the above, product rule written out
  T sum = T(0);
  for (int q = 0; q < (int)x.size(); ++q) {
    if (q == i) continue;
    T v = T(1) / (x[i] - x[q]);
    for (int s = 0; s < (int)x.size(); ++s)
      if (s != i && s != q) v *= (X - x[s]) / (x[i] - x[s]);
    sum += v;
  }
  return sum;
}
template <class T>
struct Ops {
  int n;
  std::vector<T> xs, xf;
  std::vector<T> Isf, Dfs, Efs, Dff;
  std::vector<T> wq;   // [n] quadrature weights at the solution points: w_i = int_0^1 h_i(X) dX (volume integrals, Eq. 34-35)
  explicit Ops(int n_) : n(n_), xs(n_), xf(n_ + 1), wq(n_, T(0)) {
    const T pi = std::acos(T(-1));
    for (int k = 1; k <= n; ++k) xs[k - 1] = T(0.5) * (T(1) - std::cos(T(2 * k - 1) * pi / T(2 * n)));   // Eq. 18
    // flux points: 0, roots of the Legendre polynomial P_{n-1} mapped to [0,1], 1  (G1)
    xf[0] = T(0);
    xf[n] = T(1);
    int m = n - 1;
    std::vector<T> gw(n + 1, T(0));   // weights of the (n-1)-point Gauss-Legendre rule on [0,1] at the interior flux points
    for (int k = 1; k <= m; ++k) {
      T z = -std::cos(pi * (T(k) - T(0.25)) / (T(m) + T(0.5)));          // ascending initial guesses
      for (int it = 0; it < 100; ++it) {
        T p0 = T(1), p1 = z;                                               // Bonnet recurrence
        for (int l = 2; l <= m; ++l) {
          T p2 = (T(2 * l - 1) * z * p1 - T(l - 1) * p0) / T(l);
          p0 = p1;
          p1 = p2;
        }
        T pm = (m == 0) ? T(1) : p1, pm1 = (m == 1) ? T(1) : p0;
        T dp = T(m) * (z * pm - pm1) / (z * z - T(1));
        T dz = pm / dp;
        z -= dz;
        if (std::fabs(dz) < T(4) * std::numeric_limits<T>::epsilon()) break;
      }
      xf[k] = T(0.5) * (T(1) + z);
      {   // Gauss weight 2 / ((1 - z^2) P_m'(z)^2) on [-1,1], halved for [0,1]
        T p0 = T(1), p1 = z;
        for (int l = 2; l <= m; ++l) {
          T p2 = (T(2 * l - 1) * z * p1 - T(l - 1) * p0) / T(l);
          p0 = p1;
          p1 = p2;
        }
        T pm = (m == 0) ? T(1) : p1, pm1 = (m == 1) ? T(1) : p0;
        T dp = T(m) * (z * pm - pm1) / (z * z - T(1));
        gw[k] = T(1) / ((T(1) - z * z) * dp * dp);
      }
    }
    int N1 = n + 1;
    Isf.resize(N1 * n);
    Dfs.resize(n * N1);
    Efs.resize(n * N1);
    Dff.resize(N1 * N1);
    for (int m2 = 0; m2 < N1; ++m2)
      for (int i = 0; i < n; ++i) Isf[m2 * n + i] = lagrange(xs, i, xf[m2]);          // h_i(X_f,m)
    for (int i = 0; i < n; ++i)
      for (int m2 = 0; m2 < N1; ++m2) {
        Dfs[i * N1 + m2] = lagrange_deriv(xf, m2, xs[i]);                              // l'_m(X_s,i)
        Efs[i * N1 + m2] = lagrange(xf, m2, xs[i]);                                    // l_m(X_s,i)
      }
    for (int a = 0; a < N1; ++a)
      for (int m2 = 0; m2 < N1; ++m2) Dff[a * N1 + m2] = lagrange_deriv(xf, m2, xf[a]);   // l'_m(X_f,a)
    // w_i = int_0^1 h_i: h_i has degree n-1 and the (n-1)-point Gauss rule is exact to degree 2n-3 >= n-1, so the integral is
    // the Gauss sum of h_i over the interior flux points (n = 2: one point, exact to degree 1)
    for (int i = 0; i < n; ++i)
      for (int k = 1; k <= m; ++k) wq[i] += gw[k] * Isf[k * n + i];
  }
};

// ------------------------------------------------------------------------------------------------
// O14  SSPRK(5,3) of Ruuth [8] Table 1 in Shu-Osher form (reading G23), plus test aids
// ------------------------------------------------------------------------------------------------
void rk_tableau(int nstages, double alpha[5][5], double beta[5][5]) {
  for (int i = 0; i < 5; ++i)
    for (int k = 0; k < 5; ++k) alpha[i][k] = beta[i][k] = 0.0;
  if (nstages == 5) {
    alpha[0][0] = 1.0;                beta[0][0] = 0.37726891511710;
    alpha[1][1] = 1.0;                beta[1][1] = 0.37726891511710;
    alpha[2][0] = 0.56656131914033;   alpha[2][2] = 0.43343868085967;   beta[2][2] = 0.16352294089771;
    alpha[3][0] = 0.09299483444413;   alpha[3][1] = 0.00002090369620;   alpha[3][3] = 0.90698426185967;
    beta[3][0] = 0.00071997378654;    beta[3][3] = 0.34217696850008;
    alpha[4][0] = 0.00736132260920;   alpha[4][1] = 0.20127980325145;   alpha[4][2] = 0.00182955389682;
    alpha[4][4] = 0.78952932024253;
    beta[4][0] = 0.00277719819460;    beta[4][1] = 0.00001567934613;    beta[4][4] = 0.29786487010104;
  } else if (nstages == 3) {          // Shu-Osher SSPRK(3,3)
    alpha[0][0] = 1.0;          beta[0][0] = 1.0;
    alpha[1][0] = 0.75;         alpha[1][1] = 0.25;        beta[1][1] = 0.25;
    alpha[2][0] = 1.0 / 3.0;    alpha[2][2] = 2.0 / 3.0;   beta[2][2] = 2.0 / 3.0;
  } else {                            // forward Euler
    alpha[0][0] = 1.0;          beta[0][0] = 1.0;
  }
}

// ------------------------------------------------------------------------------------------------
// the whole-mesh solver
// ------------------------------------------------------------------------------------------------
struct MeshCopy {
  int64_t E;
  int ng;
  std::vector<double> gnodes, xyz;
  std::vector<int32_t> nbr_elem;
  std::vector<uint8_t> nbr_face, nbr_orient;
};

template <class T>
struct Solver {
  int n, N1, n2, n3, nf;   // nf = n^2 (n+1) points per flux family
  int64_t E;
  Ops<T> op;
  Phys<T> ph;
  MeshCopy mesh;
  // geometry (O3)
  std::vector<T> Sfl;    // [E][3 fam][3 comp][nf]     S^d = |J| grad xi_d at the d-family flux points (Eq. 17)
  std::vector<T> detJ;   // [E][n3]
  std::vector<T> jinv;   // [E][3 d][3 p][n3]          (grad xi_d)_p at the solution points
  std::vector<T> xsol;   // [E][3][n3]
  std::vector<T> krfl;   // [E][3 fam][nf]             kappa_r at the flux points (only if kr_scale != 0)
  std::vector<T> rfl;    // [E][3 fam][nf]             distance of the flux points from the origin (wall frame, kappa_r)
  // state and work arrays
  std::vector<T> Q;      // [9][E][n3]
  bool have_state = false;

  Solver(const oracle_mesh& m, int order, const oracle_physics& p) : n(order), op(order), ph(p) {
    N1 = n + 1; n2 = n * n; n3 = n2 * n; nf = n2 * N1;
    E = m.n_elem;
    mesh.E = E; mesh.ng = m.n_geom;
    int ng3 = m.n_geom * m.n_geom * m.n_geom;
    mesh.gnodes.assign(m.geom_nodes, m.geom_nodes + m.n_geom);
    mesh.xyz.assign(m.xyz, m.xyz + E * 3 * (int64_t)ng3);
    mesh.nbr_elem.assign(m.nbr_elem, m.nbr_elem + E * 6);
    mesh.nbr_face.assign(m.nbr_face, m.nbr_face + E * 6);
    mesh.nbr_orient.assign(m.nbr_orient, m.nbr_orient + E * 6);
    Q.assign((size_t)9 * E * n3, T(0));
    geometry();
  }

  // ---- index helpers.  A "line" along direction d is labelled by (a,b) = the two remaining solution
  //      indices in increasing axis order; l = solution index along d, m = flux index along d.
  int sidx(int d, int l, int a, int b) const {
    if (d == 0) return (b * n + a) * n + l;
    if (d == 1) return (b * n + l) * n + a;
    return (l * n + b) * n + a;
  }
  int fidx(int d, int m, int a, int b) const {
    if (d == 0) return (b * n + a) * N1 + m;
    if (d == 1) return (b * N1 + m) * n + a;
    return (m * n + b) * n + a;
  }
  void orient(int code, int a, int b, int& a2, int& b2) const {   // own (a,b) -> neighbour (a',b')
    if (code & 1) std::swap(a, b);
    if (code & 2) a = n - 1 - a;
    if (code & 4) b = n - 1 - b;
    a2 = a; b2 = b;
  }

  // out[r2][r1][r0] = sum M2[r2][c] M1[r1][b] M0[r0][a] g[c][b][a] on the (N1)^3 grid; Mk = nullptr means identity.
  void tensor_eval(const T* g, const T* M0, int r0, const T* M1, int r1, const T* M2, int r2, T* out) const {
    for (int k = 0; k < r2; ++k)
      for (int j = 0; j < r1; ++j)
        for (int i = 0; i < r0; ++i) {
          T s = T(0);
          for (int c = 0; c < N1; ++c) {
            T w2 = M2 ? M2[k * N1 + c] : (c == k ? T(1) : T(0));
            if (w2 == T(0)) continue;
            for (int b = 0; b < N1; ++b) {
              T w1 = M1 ? M1[j * N1 + b] : (b == j ? T(1) : T(0));
              if (w1 == T(0)) continue;
              for (int a = 0; a < N1; ++a) {
                T w0 = M0 ? M0[i * N1 + a] : (a == i ? T(1) : T(0));
                if (w0 == T(0)) continue;
                s += w2 * w1 * w0 * g[(c * N1 + b) * N1 + a];
              }
            }
          }
          out[(k * r1 + j) * r0 + i] = s;
        }
  }

  // ---- O3 geometry: free-stream preserving curl-form metrics of the degree-n interpolant (Eq. 13-17; G3, G4)
  void geometry() {
    Sfl.assign((size_t)E * 9 * nf, T(0));
    detJ.assign((size_t)E * n3, T(0));
    jinv.assign((size_t)E * 9 * n3, T(0));
    xsol.assign((size_t)E * 3 * n3, T(0));
    bool need_kr = (ph.kr_scale != T(0));
    if (need_kr) krfl.assign((size_t)E * 3 * nf, T(0));
    else krfl.clear();
    rfl.assign((size_t)E * 3 * nf, T(0));
    const int ng = mesh.ng, ng3 = ng * ng * ng, G3 = N1 * N1 * N1;
    std::vector<T> gn(ng);
    for (int q = 0; q < ng; ++q) gn[q] = T(mesh.gnodes[q]);
    std::vector<T> Gm(N1 * ng);                    // geometry nodes -> flux-point grid
    for (int m = 0; m < N1; ++m)
      for (int q = 0; q < ng; ++q) Gm[m * ng + q] = lagrange(gn, q, op.xf[m]);
    const T* Dff = op.Dff.data();
    const T* Efs = op.Efs.data();
    const T* Dfs = op.Dfs.data();
#pragma omp parallel for schedule(static) if (E >= 1024)
    for (int64_t e = 0; e < E; ++e) {
      std::vector<T> X(3 * G3), t1, t2;
      // 0. work with offsets from the element's mean node, X := x - x0: derivatives and the curl form below do not
      //    see a constant, and rounding then scales with the element size instead of the distance from the origin
      T x0[3];
      for (int c = 0; c < 3; ++c) {
        T s = T(0);
        for (int g = 0; g < ng3; ++g) s += T(mesh.xyz[((size_t)e * 3 + c) * ng3 + g]);
        x0[c] = s / T(ng3);
      }
      // 1. geometry nodes -> (n+1)^3 grid of flux-point abscissae (three 1-D passes)
      for (int c = 0; c < 3; ++c) {
        const double* src = &mesh.xyz[((size_t)e * 3 + c) * ng3];
        t1.assign((size_t)ng * ng * N1, T(0));     // [c][b][m]
        for (int cc = 0; cc < ng; ++cc)
          for (int b = 0; b < ng; ++b)
            for (int m = 0; m < N1; ++m) {
              T s = T(0);
              for (int a = 0; a < ng; ++a) s += Gm[m * ng + a] * (T(src[(cc * ng + b) * ng + a]) - x0[c]);
              t1[(cc * ng + b) * N1 + m] = s;
            }
        t2.assign((size_t)ng * N1 * N1, T(0));     // [c][m2][m]
        for (int cc = 0; cc < ng; ++cc)
          for (int m2 = 0; m2 < N1; ++m2)
            for (int m = 0; m < N1; ++m) {
              T s = T(0);
              for (int b = 0; b < ng; ++b) s += Gm[m2 * ng + b] * t1[(cc * ng + b) * N1 + m];
              t2[(cc * N1 + m2) * N1 + m] = s;
            }
        for (int m3 = 0; m3 < N1; ++m3)
          for (int m2 = 0; m2 < N1; ++m2)
            for (int m = 0; m < N1; ++m) {
              T s = T(0);
              for (int cc = 0; cc < ng; ++cc) s += Gm[m3 * ng + cc] * t2[(cc * N1 + m2) * N1 + m];
              X[c * G3 + (m3 * N1 + m2) * N1 + m] = s;
            }
      }
      T Xbar[3];
      for (int c = 0; c < 3; ++c) {
        T s = T(0);
        for (int g = 0; g < G3; ++g) s += X[c * G3 + g];
        Xbar[c] = s / T(G3);
      }
      // centred coordinates: every derivative below is taken of X - Xbar (the derivative of a constant is
      // zero; removing it first removes a cancellation of size |X| / (element size) from the metrics)
      std::vector<T> Xc(3 * G3);
      for (int c = 0; c < 3; ++c)
        for (int g = 0; g < G3; ++g) Xc[c * G3 + g] = X[c * G3 + g] - Xbar[c];
      auto gi = [&](int a, int b, int c) { return (c * N1 + b) * N1 + a; };
      auto deriv = [&](const T* f, int j, T* out) {     // derivative of the interpolant along grid direction j
        for (int c = 0; c < N1; ++c)
          for (int b = 0; b < N1; ++b)
            for (int a = 0; a < N1; ++a) {
              T s = T(0);
              for (int q = 0; q < N1; ++q) {
                int row = (j == 0 ? a : j == 1 ? b : c);
                int src = (j == 0 ? gi(q, b, c) : j == 1 ? gi(a, q, c) : gi(a, b, q));
                s += Dff[row * N1 + q] * f[src];
              }
              out[gi(a, b, c)] = s;
            }
      };
      std::vector<T> dX(9 * G3);                       // dX[(j*3+c)*G3] = d X_c / d xi_j
      for (int j = 0; j < 3; ++j)
        for (int c = 0; c < 3; ++c) deriv(&Xc[c * G3], j, &dX[(j * 3 + c) * G3]);
      // 2. S^d_p = -[curl_xi ( (X_l - Xbar_l) grad_xi X_m )]_d,  (p,m,l) cyclic   (conservative curl form)
      std::vector<T> V(3 * G3), dV(G3), dW(G3), Sg(G3), tmp(nf);
      std::vector<T> Ssol(9 * n3);
      for (int p = 0; p < 3; ++p) {
        int mm = (p + 1) % 3, ll = (p + 2) % 3;
        for (int j = 0; j < 3; ++j)
          for (int g = 0; g < G3; ++g) V[j * G3 + g] = Xc[ll * G3 + g] * dX[(j * 3 + mm) * G3 + g];
        for (int d = 0; d < 3; ++d) {
          int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
          deriv(&V[d2 * G3], d1, dV.data());
          deriv(&V[d1 * G3], d2, dW.data());
          for (int g = 0; g < G3; ++g) Sg[g] = -(dV[g] - dW[g]);
          // at the d-family flux points: identity along d, Efs along the other two
          tensor_eval(Sg.data(), d == 0 ? nullptr : Efs, d == 0 ? N1 : n, d == 1 ? nullptr : Efs, d == 1 ? N1 : n,
                      d == 2 ? nullptr : Efs, d == 2 ? N1 : n, &Sfl[(((size_t)e * 3 + d) * 3 + p) * nf]);
          // at the solution points
          tensor_eval(Sg.data(), Efs, n, Efs, n, Efs, n, &Ssol[(d * 3 + p) * n3]);
        }
      }
      // 3. |J| at the solution points: determinant of the interpolant's Jacobi matrix (Eq. 15)
      std::vector<T> Jm(9 * n3);                       // Jm[(c*3+j)*n3] = d X_c / d xi_j at solution points
      for (int c = 0; c < 3; ++c)
        for (int j = 0; j < 3; ++j)
          tensor_eval(&Xc[c * G3], j == 0 ? Dfs : Efs, n, j == 1 ? Dfs : Efs, n, j == 2 ? Dfs : Efs, n, &Jm[(c * 3 + j) * n3]);
      for (int s = 0; s < n3; ++s) {
        auto J = [&](int c, int j) { return Jm[(c * 3 + j) * n3 + s]; };
        T det = J(0, 0) * (J(1, 1) * J(2, 2) - J(1, 2) * J(2, 1)) - J(0, 1) * (J(1, 0) * J(2, 2) - J(1, 2) * J(2, 0)) +
                J(0, 2) * (J(1, 0) * J(2, 1) - J(1, 1) * J(2, 0));
        detJ[(size_t)e * n3 + s] = det;
        for (int dp = 0; dp < 9; ++dp) jinv[((size_t)e * 9 + dp) * n3 + s] = Ssol[dp * n3 + s] / det;
      }
      for (int c = 0; c < 3; ++c) {
        tensor_eval(&X[c * G3], Efs, n, Efs, n, Efs, n, &xsol[((size_t)e * 3 + c) * n3]);
        for (int s = 0; s < n3; ++s) xsol[((size_t)e * 3 + c) * n3 + s] += x0[c];
      }
      {
        std::vector<T> xf3(3 * nf);
        for (int d = 0; d < 3; ++d) {
          for (int c = 0; c < 3; ++c)
            tensor_eval(&X[c * G3], d == 0 ? nullptr : Efs, d == 0 ? N1 : n, d == 1 ? nullptr : Efs, d == 1 ? N1 : n,
                        d == 2 ? nullptr : Efs, d == 2 ? N1 : n, &xf3[c * nf]);
          for (int g = 0; g < nf; ++g) {
            T px = xf3[g] + x0[0], py = xf3[nf + g] + x0[1], pz = xf3[2 * nf + g] + x0[2];
            T r = std::sqrt(px * px + py * py + pz * pz);
            rfl[((size_t)e * 3 + d) * nf + g] = r;
            T w = r * ph.kr_wscale;
            if (need_kr) krfl[((size_t)e * 3 + d) * nf + g] = ph.kr_scale * (ph.kr_c[0] + ph.kr_c[1] * w + ph.kr_c[2] * w * w);
          }
        }
      }
    }
  }

  // area vector, unit outward normal and |S| at face point (a,b) of face f of element e
  void face_normal(int64_t e, int f, int a, int b, T* nh, T& area, T& sigma) const {
    int d = f / 2, m = (f & 1) ? n : 0;
    sigma = (f & 1) ? T(1) : T(-1);
    T S[3];
    for (int p = 0; p < 3; ++p) S[p] = Sfl[(((size_t)e * 3 + d) * 3 + p) * nf + fidx(d, m, a, b)];
    area = std::sqrt(S[0] * S[0] + S[1] * S[1] + S[2] * S[2]);
    for (int p = 0; p < 3; ++p) nh[p] = sigma * S[p] / area;
  }

  // ---- O5: Q at the three flux families, Qh [E][3][9][nf]  (Eq. 21 with Eq. 19)
  void interpolate_state(const std::vector<T>& Qs, std::vector<T>& Qh) const {
    Qh.assign((size_t)E * 27 * nf, T(0));
#pragma omp parallel for schedule(static) if (E >= 1024)
    for (int64_t e = 0; e < E; ++e)
      for (int d = 0; d < 3; ++d)
        for (int v = 0; v < 9; ++v)
          for (int b = 0; b < n; ++b)
            for (int a = 0; a < n; ++a)
              for (int m = 0; m < N1; ++m) {
                T s = T(0);
                for (int l = 0; l < n; ++l) s += op.Isf[m * n + l] * Qs[((size_t)v * E + e) * n3 + sidx(d, l, a, b)];
                Qh[(((size_t)e * 3 + d) * 9 + v) * nf + fidx(d, m, a, b)] = s;
              }
  }

  // ---- O6 + O7: BR1 common solution on faces, gradient at solution points  G [27][E][n3]
  void gradient(const std::vector<T>& Qh, std::vector<T>& G) const {
    G.assign((size_t)27 * E * n3, T(0));
#pragma omp parallel for schedule(static) if (E >= 1024)
    for (int64_t e = 0; e < E; ++e) {
      std::vector<T> Qc((size_t)27 * nf);     // own flux-point values with the face values replaced by the common ones
      for (size_t i = 0; i < Qc.size(); ++i) Qc[i] = Qh[(size_t)e * 27 * nf + i];
      for (int f = 0; f < 6; ++f) {
        int d = f / 2, m = (f & 1) ? n : 0;
        int32_t ne = mesh.nbr_elem[e * 6 + f];
        for (int b = 0; b < n; ++b)
          for (int a = 0; a < n; ++a) {
            T Qi[9], Qcm[9];
            for (int v = 0; v < 9; ++v) Qi[v] = Qh[(((size_t)e * 3 + d) * 9 + v) * nf + fidx(d, m, a, b)];
            if (ne >= 0) {                      // BR1: average of the two polynomials
              int nfc = mesh.nbr_face[e * 6 + f], dn = nfc / 2, mn = (nfc & 1) ? n : 0, a2, b2;
              orient(mesh.nbr_orient[e * 6 + f], a, b, a2, b2);
              for (int v = 0; v < 9; ++v) {
                T Qo = Qh[(((size_t)ne * 3 + dn) * 9 + v) * nf + fidx(dn, mn, a2, b2)];
                Qcm[v] = T(0.5) * (Qi[v] + Qo);
              }
            } else {                            // wall: the boundary state (O12)
              T nh[3], area, sg;
              face_normal(e, f, a, b, nh, area, sg);
              wall_state(ph, ne, Qi, nh, Qcm);
            }
            for (int v = 0; v < 9; ++v) Qc[((size_t)d * 9 + v) * nf + fidx(d, m, a, b)] = Qcm[v];
          }
      }
      for (int s3 = 0; s3 < n3; ++s3) {
        int i = s3 % n, j = (s3 / n) % n, k = s3 / n2;
        for (int v = 0; v < 9; ++v) {
          T dxi[3];
          for (int d = 0; d < 3; ++d) {
            int l = (d == 0 ? i : d == 1 ? j : k), a = (d == 0 ? j : i), b = (d == 2 ? j : k);
            T s = T(0);
            for (int m = 0; m < N1; ++m) s += op.Dfs[l * N1 + m] * Qc[((size_t)d * 9 + v) * nf + fidx(d, m, a, b)];
            dxi[d] = s;
          }
          for (int p = 0; p < 3; ++p) {          // chain rule with grad xi_d (reading G9)
            T s = T(0);
            for (int d = 0; d < 3; ++d) s += jinv[((size_t)e * 9 + d * 3 + p) * n3 + s3] * dxi[d];
            G[((size_t)(3 * v + p) * E + e) * n3 + s3] = s;
          }
        }
      }
    }
  }

  // ---- O8 (faces): own gradient at own face points, Gf [E][6][27][n2]
  void gradient_traces(const std::vector<T>& G, std::vector<T>& Gf) const {
    Gf.assign((size_t)E * 6 * 27 * n2, T(0));
#pragma omp parallel for schedule(static) if (E >= 1024)
    for (int64_t e = 0; e < E; ++e)
      for (int f = 0; f < 6; ++f) {
        int d = f / 2, m = (f & 1) ? n : 0;
        for (int c = 0; c < 27; ++c)
          for (int b = 0; b < n; ++b)
            for (int a = 0; a < n; ++a) {
              T s = T(0);
              for (int l = 0; l < n; ++l) s += op.Isf[m * n + l] * G[((size_t)c * E + e) * n3 + sidx(d, l, a, b)];
              Gf[(((size_t)e * 6 + f) * 27 + c) * n2 + b * n + a] = s;
            }
      }
  }

  // ---- the residual (O5 .. O13): R = -(1/|J|) div_xi F~ + M  (Eq. 16), A = magnitude residual (G24)
  void residual(const std::vector<T>& Qs, std::vector<T>& R, std::vector<T>* A, std::vector<T>* Gout = nullptr) const {
    const bool diff = (ph.flags & F_DIFF) != 0;
    const bool have_kr = !krfl.empty();
    std::vector<T> Qh, G, Gf;
    interpolate_state(Qs, Qh);
    gradient(Qh, G);
    gradient_traces(G, Gf);
    R.assign((size_t)9 * E * n3, T(0));
    if (A) A->assign((size_t)9 * E * n3, T(0));
#pragma omp parallel for schedule(static) if (E >= 1024)
    for (int64_t e = 0; e < E; ++e) {
      std::vector<T> Fh((size_t)27 * nf);       // F~ of the three families, [3][9][nf]
      std::vector<T> FhA((size_t)27 * nf);      // sum of the moduli of the terms of F~ (magnitude residual, G24)
      for (int d = 0; d < 3; ++d)
        for (int b = 0; b < n; ++b)
          for (int a = 0; a < n; ++a)
            for (int m = 0; m < N1; ++m) {
              int ix = fidx(d, m, a, b);
              T S[3], Fi[9], Fv[9];
              for (int p = 0; p < 3; ++p) S[p] = Sfl[(((size_t)e * 3 + d) * 3 + p) * nf + ix];
              T kr = have_kr ? krfl[((size_t)e * 3 + d) * nf + ix] : T(0);
              T Qi[9];
              for (int v = 0; v < 9; ++v) Qi[v] = Qh[(((size_t)e * 3 + d) * 9 + v) * nf + ix];
              if (m > 0 && m < n) {             // interior flux point: flux of the element's own polynomial
                flux_inviscid(ph, Qi, S, Fi);
                { T Fa0[9]; flux_inviscid_abs(ph, Qi, S, Fa0); for (int v = 0; v < 9; ++v) FhA[((size_t)d * 9 + v) * nf + ix] = Fa0[v]; }
                if (diff) {
                  T Gi[27];
                  for (int c = 0; c < 27; ++c) {   // O8: gradient interpolated to the flux point
                    T s = T(0);
                    for (int l = 0; l < n; ++l) s += op.Isf[m * n + l] * G[((size_t)c * E + e) * n3 + sidx(d, l, a, b)];
                    Gi[c] = s;
                  }
                  flux_viscous(ph, Qi, Gi, S, kr, Fv);
                  for (int v = 0; v < 9; ++v) Fi[v] -= Fv[v];
                  for (int v = 0; v < 9; ++v) FhA[((size_t)d * 9 + v) * nf + ix] += std::fabs(Fv[v]);
                }
                for (int v = 0; v < 9; ++v) Fh[((size_t)d * 9 + v) * nf + ix] = Fi[v];
                continue;
              }
              // face flux point: common fluxes (O11) or wall fluxes (O12)
              int f = 2 * d + (m == n ? 1 : 0);
              int32_t ne = mesh.nbr_elem[e * 6 + f];
              T nh[3], area, sg;
              face_normal(e, f, a, b, nh, area, sg);
              const T* Gin = &Gf[(((size_t)e * 6 + f) * 27) * n2 + b * n + a];   // stride n2
              T Gi[27];
              for (int c = 0; c < 27; ++c) Gi[c] = Gin[(size_t)c * n2];
              T Fc[9], Fa[9];
              for (int v = 0; v < 9; ++v) Fv[v] = T(0);
              if (ne >= 0) {
                int nfc = mesh.nbr_face[e * 6 + f], dn = nfc / 2, mn = (nfc & 1) ? n : 0, a2, b2;
                orient(mesh.nbr_orient[e * 6 + f], a, b, a2, b2);
                T Qo[9], Go[27];
                for (int v = 0; v < 9; ++v) Qo[v] = Qh[(((size_t)ne * 3 + dn) * 9 + v) * nf + fidx(dn, mn, a2, b2)];
                flux_rusanov(ph, Qi, Qo, nh, Fc, Fa);
                if (diff) {                     // "a similar procedure": average of the two sides' viscous fluxes (G15)
                  for (int c = 0; c < 27; ++c) Go[c] = Gf[(((size_t)ne * 6 + nfc) * 27 + c) * n2 + b2 * n + a2];
                  T F1[9], F2[9];
                  flux_viscous(ph, Qi, Gi, nh, kr, F1);
                  flux_viscous(ph, Qo, Go, nh, kr, F2);
                  for (int v = 0; v < 9; ++v) Fv[v] = T(0.5) * (F1[v] + F2[v]);
                  for (int v = 0; v < 9; ++v) Fa[v] += T(0.5) * (std::fabs(F1[v]) + std::fabs(F2[v]));
                }
              } else {
                T Qb[9];
                wall_state(ph, ne, Qi, nh, Qb);
                flux_inviscid(ph, Qb, nh, Fc, /*wall=*/true);
                if (diff) flux_wall_viscous(ph, ne, Qb, Gi, nh, rfl[((size_t)e * 3 + d) * nf + ix], kr, Fv);
                flux_inviscid_abs(ph, Qb, nh, Fa, /*wall=*/true);
                for (int v = 0; v < 9; ++v) Fa[v] += std::fabs(Fv[v]);
              }
              for (int v = 0; v < 9; ++v) Fh[((size_t)d * 9 + v) * nf + ix] = sg * area * (Fc[v] - Fv[v]);
              for (int v = 0; v < 9; ++v) FhA[((size_t)d * 9 + v) * nf + ix] = area * Fa[v];
            }
      // O13: derivative of the flux polynomials at the solution points (Eq. 20, 22-24) and sources
      for (int s3 = 0; s3 < n3; ++s3) {
        int i = s3 % n, j = (s3 / n) % n, k = s3 / n2;
        T Qp[9], Gp[27], M[9], Mabs[9];
        for (int v = 0; v < 9; ++v) Qp[v] = Qs[((size_t)v * E + e) * n3 + s3];
        for (int c = 0; c < 27; ++c) Gp[c] = G[((size_t)c * E + e) * n3 + s3];
        T x[3] = {xsol[((size_t)e * 3 + 0) * n3 + s3], xsol[((size_t)e * 3 + 1) * n3 + s3], xsol[((size_t)e * 3 + 2) * n3 + s3]};
        source(ph, Qp, Gp, x, M, Mabs);
        T dj = detJ[(size_t)e * n3 + s3];
        for (int v = 0; v < 9; ++v) {
          T div = T(0), adiv = T(0);
          for (int d = 0; d < 3; ++d) {
            int l = (d == 0 ? i : d == 1 ? j : k), a = (d == 0 ? j : i), b = (d == 2 ? j : k);
            for (int m = 0; m < N1; ++m) {
              int ix = fidx(d, m, a, b);
              div += op.Dfs[l * N1 + m] * Fh[((size_t)d * 9 + v) * nf + ix];
              adiv += std::fabs(op.Dfs[l * N1 + m]) * FhA[((size_t)d * 9 + v) * nf + ix];
            }
          }
          R[((size_t)v * E + e) * n3 + s3] = -div / dj + M[v];
          if (A) (*A)[((size_t)v * E + e) * n3 + s3] = adiv / std::fabs(dj) + Mabs[v];
        }
      }
    }
    if (Gout) Gout->swap(G);
  }

  // ---- O14: one time step, literal Shu-Osher form
  void step(T dt, int nstages) {
    double al[5][5], be[5][5];
    rk_tableau(nstages, al, be);
    std::vector<std::vector<T>> u(nstages + 1), Fu(nstages);
    u[0] = Q;
    for (int i = 1; i <= nstages; ++i) {
      residual(u[i - 1], Fu[i - 1], nullptr);
      u[i].assign(Q.size(), T(0));
      for (int k = 0; k < i; ++k) {
        T a = T(al[i - 1][k]), b = T(be[i - 1][k]);
        if (a == T(0) && b == T(0)) continue;
        for (size_t s = 0; s < Q.size(); ++s) u[i][s] += a * u[k][s] + dt * b * Fu[k][s];
      }
    }
    Q = u[nstages];
  }

  // Eq. 34-35: V = int dV, KE = (1/V) int 1/2 rho U.U dV, E_B = (1/V) int 1/2 B.B dV, with the
  // interpolatory quadrature of the solution points: int f dV = sum_e sum_ijk w_i w_j w_k |J| f.  Sums are kept in long double.
  void diagnostics(double out[3]) const {
    long double V = 0, KE = 0, EB = 0;
    for (int64_t e = 0; e < E; ++e)
      for (int k = 0; k < n; ++k)
        for (int j = 0; j < n; ++j)
          for (int i = 0; i < n; ++i) {
            int s = (k * n + j) * n + i;
            T Qp[9];
            for (int v = 0; v < 9; ++v) Qp[v] = Q[((size_t)v * E + e) * n3 + s];
            long double wJ = (long double)(op.wq[i] * op.wq[j] * op.wq[k]) * (long double)detJ[(size_t)e * n3 + s];
            V += wJ;
            KE += wJ * (long double)(T(0.5) * (Qp[1] * Qp[1] + Qp[2] * Qp[2] + Qp[3] * Qp[3]) / Qp[0]);
            EB += wJ * (long double)(T(0.5) * (Qp[5] * Qp[5] + Qp[6] * Qp[6] + Qp[7] * Qp[7]));
          }
    out[0] = (double)V;
    out[1] = (double)(KE / V);
    out[2] = (double)(EB / V);
  }

  T max_wavespeed() const {
    T mx = T(0);
    for (int64_t e = 0; e < E; ++e)
      for (int s = 0; s < n3; ++s) {
        T Qp[9];
        for (int v = 0; v < 9; ++v) Qp[v] = Q[((size_t)v * E + e) * n3 + s];
        mx = std::max(mx, wavespeed(ph, Qp));
      }
    return mx;
  }
};

template <class T>
void to_double(const std::vector<T>& a, double* out) {
  for (size_t i = 0; i < a.size(); ++i) out[i] = (double)a[i];
}

}  // namespace

struct oracle_ctx {
  Solver<double>* d = nullptr;
  Solver<long double>* l = nullptr;
};

#define DISPATCH(ctx, call) ((ctx)->d ? (ctx)->d->call : (ctx)->l->call)

extern "C" {

oracle_ctx* oracle_init(const oracle_mesh* mesh, int order, const oracle_physics* phys, int prec) {
  if (!mesh || !phys || order < 2 || order > 9 || mesh->n_elem <= 0 || mesh->n_geom < 2) return nullptr;
  oracle_ctx* c = new oracle_ctx;
  if (prec == 0) c->d = new Solver<double>(*mesh, order, *phys);
  else c->l = new Solver<long double>(*mesh, order, *phys);
  return c;
}
void oracle_free(oracle_ctx* c) {
  if (!c) return;
  delete c->d;
  delete c->l;
  delete c;
}
int oracle_set_physics(oracle_ctx* c, const oracle_physics* p) {
  if (!c || !p) return -1;
  bool regeo;
  if (c->d) { regeo = (c->d->ph.kr_scale != p->kr_scale) || p->kr_scale != 0.0; c->d->ph = Phys<double>(*p); if (regeo) c->d->geometry(); }
  else { regeo = (c->l->ph.kr_scale != (long double)p->kr_scale) || p->kr_scale != 0.0; c->l->ph = Phys<long double>(*p); if (regeo) c->l->geometry(); }
  return 0;
}
int oracle_set_state(oracle_ctx* c, const double* q) {
  if (!c || !q) return -1;
  if (c->d) { for (size_t i = 0; i < c->d->Q.size(); ++i) c->d->Q[i] = q[i]; c->d->have_state = true; }
  else { for (size_t i = 0; i < c->l->Q.size(); ++i) c->l->Q[i] = q[i]; c->l->have_state = true; }
  return 0;
}
int oracle_get_state(oracle_ctx* c, double* q) {
  if (!c || !q) return -1;
  if (c->d) to_double(c->d->Q, q); else to_double(c->l->Q, q);
  return 0;
}
int oracle_residual(oracle_ctx* c, double* r, double* a) {
  if (!c || !r) return -1;
  if (c->d) {
    std::vector<double> R, A;
    c->d->residual(c->d->Q, R, a ? &A : nullptr);
    to_double(R, r);
    if (a) to_double(A, a);
  } else {
    std::vector<long double> R, A;
    c->l->residual(c->l->Q, R, a ? &A : nullptr);
    to_double(R, r);
    if (a) to_double(A, a);
  }
  return 0;
}
int oracle_step(oracle_ctx* c, double dt, int nstages) {
  if (!c || (nstages != 1 && nstages != 3 && nstages != 5)) return -1;
  if (c->d) c->d->step(dt, nstages); else c->l->step((long double)dt, nstages);
  return 0;
}
int oracle_max_wavespeed(oracle_ctx* c, double* out) {
  if (!c || !out) return -1;
  *out = c->d ? c->d->max_wavespeed() : (double)c->l->max_wavespeed();
  return 0;
}
int oracle_diagnostics(oracle_ctx* c, double* out) {
  if (!c || !out) return -1;
  if (c->d) c->d->diagnostics(out); else c->l->diagnostics(out);
  return 0;
}
int oracle_quadrature_weights(int order, double* w) {
  if (order < 2 || order > 12 || !w) return -1;
  Ops<long double> o(order);
  for (int i = 0; i < order; ++i) w[i] = (double)o.wq[i];
  return 0;
}
int oracle_get_gradient(oracle_ctx* c, double* g) {
  if (!c || !g) return -1;
  if (c->d) {
    std::vector<double> R, G;
    c->d->residual(c->d->Q, R, nullptr, &G);
    to_double(G, g);
  } else {
    std::vector<long double> R, G;
    c->l->residual(c->l->Q, R, nullptr, &G);
    to_double(G, g);
  }
  return 0;
}
int oracle_get_geometry(oracle_ctx* c, double* detJ, double* S, double* xsol, double* jinv) {
  if (!c) return -1;
  auto put = [&](auto* s) {
    if (detJ) to_double(s->detJ, detJ);
    if (S) to_double(s->Sfl, S);
    if (jinv) to_double(s->jinv, jinv);
    if (xsol)   // internal [E][3][n3] -> interface [3][E][n3]
      for (int64_t e = 0; e < s->E; ++e)
        for (int cc = 0; cc < 3; ++cc)
          for (int i = 0; i < s->n3; ++i) xsol[((size_t)cc * s->E + e) * s->n3 + i] = (double)s->xsol[((size_t)e * 3 + cc) * s->n3 + i];
  };
  if (c->d) put(c->d); else put(c->l);
  return 0;
}

int oracle_nodes(int order, double* xs, double* xf) {
  if (order < 2 || order > 9) return -1;
  Ops<long double> op(order);
  if (xs) to_double(op.xs, xs);
  if (xf) to_double(op.xf, xf);
  return 0;
}
int oracle_operators(int order, double* Isf, double* Dfs, double* Efs, double* Dff) {
  if (order < 2 || order > 9) return -1;
  Ops<double> op(order);
  if (Isf) to_double(op.Isf, Isf);
  if (Dfs) to_double(op.Dfs, Dfs);
  if (Efs) to_double(op.Efs, Efs);
  if (Dff) to_double(op.Dff, Dff);
  return 0;
}
int oracle_rk_tableau(int nstages, double* alpha, double* beta) {
  if (nstages != 1 && nstages != 3 && nstages != 5) return -1;
  double al[5][5], be[5][5];
  rk_tableau(nstages, al, be);
  std::memcpy(alpha, al, sizeof al);
  std::memcpy(beta, be, sizeof be);
  return 0;
}

void oracle_flux_inviscid(const oracle_physics* p, const double* Q, const double* S, double* F) {
  flux_inviscid(Phys<double>(*p), Q, S, F);
}
void oracle_flux_viscous(const oracle_physics* p, const double* Q, const double* G, const double* S, double kr, double* F) {
  flux_viscous(Phys<double>(*p), Q, G, S, kr, F);
}
void oracle_flux_rusanov(const oracle_physics* p, const double* Qi, const double* Qo, const double* nh, double* F) {
  flux_rusanov(Phys<double>(*p), Qi, Qo, nh, F);
}
double oracle_fast_speed(const oracle_physics* p, const double* Q, const double* nh) {
  Phys<double> ph(*p);
  return fast_speed(ph, primitives(ph, Q), nh);
}
double oracle_wavespeed(const oracle_physics* p, const double* Q) { return wavespeed(Phys<double>(*p), Q); }
void oracle_wall_state(const oracle_physics* p, int wall, const double* Q, const double* nh, double* Qb) {
  wall_state(Phys<double>(*p), wall, Q, nh, Qb);
}
void oracle_flux_wall_inviscid(const oracle_physics* p, const double* Qb, const double* nh, double* F) {
  flux_inviscid(Phys<double>(*p), Qb, nh, F, true);
}
void oracle_flux_wall_viscous(const oracle_physics* p, int wall, const double* Qb, const double* G, const double* nh, double rw,
                              double kr, double* F) {
  flux_wall_viscous(Phys<double>(*p), wall, Qb, G, nh, rw, kr, F);
}
void oracle_wall_condition_gradB(int bc, const double* dB, const double* Bb, const double* er, double rw, double* dBc) {
  double a[3][3], c[3][3];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) a[i][j] = dB[i * 3 + j];
  wall_condition_gradB<double>(bc, a, Bb, er, rw, c);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) dBc[i * 3 + j] = c[i][j];
}
void oracle_source(const oracle_physics* p, const double* Q, const double* G, const double* x, double* M, double* Mabs) {
  source(Phys<double>(*p), Q, G, x, M, Mabs);
}

}  // extern "C"
