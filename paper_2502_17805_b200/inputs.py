"""Seeded synthetic inputs: meshes, physics parameter sets and states.

This module is the ONLY code shared by the CUDA path and the CPU oracle.  It holds
none of the method's arithmetic (no SD nodes, operators, metrics, fluxes or RK):
it builds hexahedral meshes (geometry nodes + connectivity), evaluates analytic
background / perturbation fields at point coordinates *handed in by the caller*,
and names the BASELINE.json workload configurations.  numpy only.

Citations are to /root/reference/PAPER.md (line : section / equation).
  * cubed-sphere shell      PAPER.md:70-80   (SIII, Eq. 11-12)
  * polytropic background   PAPER.md:155-169 (SV, Eq. 25-27)
  * conserved state         PAPER.md:27-36   (SII, Eq. 2-4)
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field, asdict

import numpy as np

# --------------------------------------------------------------------------------------
# physics-parameter record (plain data; each binding marshals it into its own C struct)
# --------------------------------------------------------------------------------------
FLAG_DIFFUSION = 1 << 0
FLAG_GRAVITY = 1 << 1
FLAG_CORIOLIS = 1 << 2
FLAG_POWELL = 1 << 3
FLAG_GLM_DAMP = 1 << 4
FLAG_FIXED_T_OUTER = 1 << 5
FLAG_FIXED_FLUX_INNER = 1 << 6
FLAG_CENTRIFUGAL = 1 << 7

BC_CONDUCTING = 0
BC_RADIAL = 1


@dataclass
class Physics:
    """Physical parameters of Eq. 3-10 and the wall options of SVI."""
    gamma: float = 5.0 / 3.0
    R_gas: float = 1.0
    Cp: float = 2.5
    GM: float = 1.0
    Omega: float = 0.0
    nu: float = 0.0
    kappa: float = 0.0
    eta: float = 0.0
    kr_scale: float = 0.0
    kr_c: tuple = (0.0, 0.0, 0.0)
    kr_wscale: float = 1.0
    c_h: float = 0.0
    a_psi: float = 0.0
    q_bottom: float = 0.0
    T_top: float = 0.0
    bc_mag_inner: int = BC_CONDUCTING
    bc_mag_outer: int = BC_RADIAL
    flags: int = 0

    def copy(self, **kw) -> "Physics":
        d = asdict(self)
        d.update(kw)
        return Physics(**d)


# --------------------------------------------------------------------------------------
# geometry-node abscissae
# --------------------------------------------------------------------------------------
def lobatto_abscissae(ng: int) -> np.ndarray:
    """ng Chebyshev-Lobatto abscissae on [0,1] (end points included).

    These are where the mesh generators sample the element map; they are a property of
    the *mesh file*, not of the SD discretisation (both implementations re-interpolate
    the geometry onto their own flux-point grid).
    """
    if ng < 2:
        raise ValueError("need at least 2 geometry nodes per direction")
    k = np.arange(ng)
    x = 0.5 * (1.0 - np.cos(np.pi * k / (ng - 1)))
    x[0], x[-1] = 0.0, 1.0
    return x


# --------------------------------------------------------------------------------------
# connectivity of a conforming hexahedral mesh, by matching face corners
# --------------------------------------------------------------------------------------
def _face_corners(c: np.ndarray, f: int) -> np.ndarray:
    """c [3,2,2,2] element corners (axes xi,eta,zeta) -> [3,2,2] corners of local face f,
    indexed (a,b) = the two remaining axes in increasing order.
    Faces 0..5 = xi0, xi1, eta0, eta1, zeta0, zeta1."""
    ax, side = divmod(f, 2)
    return np.take(c, side, axis=1 + ax)


def orient_map(code: int, a, b, n: int):
    """Face-point index map of orientation `code` (bit0 swap, bit1 reverse a, bit2 reverse b):
    own face point (a,b) coincides with the neighbour's face point (a',b') returned here."""
    if code & 1:
        a, b = b, a
    if code & 2:
        a = n - 1 - a
    if code & 4:
        b = n - 1 - b
    return a, b


def hex_connectivity(corners: np.ndarray, wall_tag=None, decimals: int = 8):
    """corners [E,3,2,2,2] -> (nbr_elem int32[E,6], nbr_face uint8[E,6], nbr_orient uint8[E,6]).

    Faces are paired by their (rounded) centres; unpaired faces get nbr_elem =
    wall_tag(centres[M,3]) (negative ints; default -1).  Orientation codes follow
    `orient_map` and are found by comparing the 4 corners under each of the 8 codes.
    """
    E = corners.shape[0]
    faces = np.stack([_face_corners_all(corners, f) for f in range(6)], axis=1)      # [E,6,3,2,2]
    cen = faces.reshape(E, 6, 3, 4).mean(-1).reshape(E * 6, 3)
    key = np.round(cen * 10.0 ** decimals).astype(np.int64)
    _, inv, cnt = np.unique(key, axis=0, return_inverse=True, return_counts=True)
    inv = inv.reshape(-1)
    if cnt.max() > 2:
        raise ValueError("non-manifold face")
    order = np.argsort(inv, kind="stable")
    sorted_inv = inv[order]
    first = np.flatnonzero((sorted_inv[1:] == sorted_inv[:-1])) if order.size > 1 else np.zeros(0, np.int64)
    A, B = order[first], order[first + 1]                # paired global face ids (e*6+f)
    nbr_elem = np.full(E * 6, -1, np.int32)
    nbr_face = np.zeros(E * 6, np.uint8)
    nbr_orient = np.zeros(E * 6, np.uint8)
    single = order[np.flatnonzero(cnt[sorted_inv] == 1)]
    if wall_tag is not None and single.size:
        nbr_elem[single] = wall_tag(cen[single])
    F = faces.reshape(E * 6, 3, 2, 2)
    scale = np.abs(corners).max()
    tol = scale * 10.0 ** (-decimals + 1)
    for me, other in ((A, B), (B, A)):
        P1, P2 = F[me], F[other]
        code_found = np.full(me.size, 255, np.int64)
        for code in range(7, -1, -1):
            ok = np.ones(me.size, bool)
            for a, b in itertools.product((0, 1), (0, 1)):
                a2, b2 = orient_map(code, a, b, 2)
                ok &= np.abs(P1[:, :, a, b] - P2[:, :, a2, b2]).max(axis=1) <= tol
            code_found[ok] = code
        if (code_found == 255).any():
            raise ValueError("faces share a centre but no orientation code matches")
        nbr_elem[me] = other // 6
        nbr_face[me] = other % 6
        nbr_orient[me] = code_found
    return nbr_elem.reshape(E, 6), nbr_face.reshape(E, 6), nbr_orient.reshape(E, 6)


def _face_corners_all(corners: np.ndarray, f: int) -> np.ndarray:
    """corners [E,3,2,2,2] -> [E,3,2,2] corners of local face f for every element."""
    ax, side = divmod(f, 2)
    return np.take(corners, side, axis=2 + ax)


# --------------------------------------------------------------------------------------
# cubed-sphere shell (Eq. 11-12)
# --------------------------------------------------------------------------------------
def _panel_dir(p: int, al, be):
    """Unit direction of panel p at equiangular coordinates (alpha, beta) (Eq. 11-12).
    Panel 0 is the +x face with alpha = atan(y/x), beta = atan(z/x); the
    other five are its rotations: +y, -x, -y, +z, -z (all right-handed in (alpha,beta,r))."""
    X, Y = np.tan(al), np.tan(be)
    d = np.sqrt(1.0 + X * X + Y * Y)
    one = np.ones_like(d)
    v = [(one, X, Y), (-X, one, Y), (-one, -X, Y), (X, -one, Y), (-Y, X, one), (Y, X, -one)][p]
    return np.stack([c / d for c in v])


def cubed_sphere_shell(n_z: int, n_r: int, r_b: float, r_t: float, gnodes: np.ndarray, oblateness: float = 0.0):
    """Mesh dict of the 6*n_r*n_z^2 element shell (N_cells of PAPER.md:80).

    Element order: panel-major, then radial k, then j (beta), then i (alpha).
    (xi,eta,zeta) = (alpha,beta,r) scaled to [0,1] per element; uniform radial spacing.
    xyz [E,3,ng^3] holds the map sampled at gnodes^3 (xi fastest).  Inner wall faces get
    nbr_elem = -1, outer wall faces -2.  `oblateness` e>0 scales z by (1-e) (oblate shells,
    PAPER.md:70 "It is also possible to generate oblate meshes").
    """
    g = np.asarray(gnodes, np.float64)
    ng = g.size
    E = 6 * n_r * n_z * n_z
    h = 0.5 * np.pi / n_z
    dr = (r_t - r_b) / n_r

    def sample(gs):
        m = gs.size
        out = np.empty((6, n_r, n_z, n_z, 3, m, m, m))           # [p,k,j,i,comp,c,b,a]
        al = -0.25 * np.pi + (np.arange(n_z)[:, None] + gs[None, :]) * h      # [i,a]
        r = r_b + (np.arange(n_r)[:, None] + gs[None, :]) * dr                # [k,c]
        A = al[None, None, :, None, None, :]
        B = al[None, :, None, None, :, None]
        R = r[:, None, None, :, None, None]
        A, B, R = np.broadcast_arrays(A, B, R)
        for p in range(6):
            out[p] = np.moveaxis(R * _panel_dir(p, A, B), 0, 3)
        return out.reshape(E, 3, m, m, m)

    xyz = sample(g)                                               # [E,3,c,b,a]
    corners = np.transpose(sample(np.array([0.0, 1.0])), (0, 1, 4, 3, 2))   # -> [E,3,xi,eta,zeta]
    r_mid = 0.5 * (r_b + r_t)

    def wall_tag(c):
        return np.where(np.linalg.norm(c, axis=1) < r_mid, -1, -2).astype(np.int32)

    nbr_elem, nbr_face, nbr_orient = hex_connectivity(corners, wall_tag)
    if oblateness != 0.0:
        xyz[:, 2] *= (1.0 - oblateness)
    return dict(n_elem=E, n_geom=ng, geom_nodes=g.copy(), xyz=np.ascontiguousarray(xyz.reshape(E, 3, ng ** 3)),
                nbr_elem=nbr_elem, nbr_face=nbr_face, nbr_orient=nbr_orient,
                kind="shell", n_z=n_z, n_r=n_r, r_b=r_b, r_t=r_t)


# --------------------------------------------------------------------------------------
# periodic (optionally curvilinear) box -- used by the oracle pins (Alfven wave, decay tests)
# --------------------------------------------------------------------------------------
def periodic_box(nx: int, ny: int, nz: int, lengths, gnodes: np.ndarray, distort: float = 0.0,
                 walls_z: bool = False):
    """nx*ny*nz hexes on [0,Lx]x[0,Ly]x[0,Lz], periodic in all directions (or with walls at
    z=0 (tag -1) and z=Lz (tag -2) if walls_z).  distort>0 displaces the nodes by a smooth
    periodic field of amplitude distort*min(h) whose z-component vanishes on z=0,Lz, so the
    elements are genuinely curved, conforming, and the walls stay planar.
    Element order k, j, i (i fastest); orientation codes are all 0."""
    g = np.asarray(gnodes, np.float64)
    ng = g.size
    Lx, Ly, Lz = lengths
    hx, hy, hz = Lx / nx, Ly / ny, Lz / nz
    E = nx * ny * nz
    xyz = np.empty((E, 3, ng, ng, ng))
    nbr_elem = np.empty((E, 6), np.int32)
    nbr_face = np.empty((E, 6), np.uint8)
    nbr_orient = np.zeros((E, 6), np.uint8)
    amp = distort * min(hx, hy, hz)
    eid = lambda i, j, k: ((k % nz) * ny + (j % ny)) * nx + (i % nx)
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                e = eid(i, j, k)
                Z, Y, X = np.meshgrid((k + g) * hz, (j + g) * hy, (i + g) * hx, indexing="ij")
                if amp != 0.0:
                    sx, sy, sz = np.sin(2 * np.pi * X / Lx), np.sin(2 * np.pi * Y / Ly), np.sin(2 * np.pi * Z / Lz)
                    cx, cy, cz = np.cos(2 * np.pi * X / Lx), np.cos(2 * np.pi * Y / Ly), np.cos(2 * np.pi * Z / Lz)
                    X, Y, Z = X + amp * sx * cy * cz, Y + 0.7 * amp * cx * sy * cz, Z + 0.5 * amp * cx * cy * sz
                xyz[e, 0], xyz[e, 1], xyz[e, 2] = X, Y, Z
                nbr_elem[e] = [eid(i - 1, j, k), eid(i + 1, j, k), eid(i, j - 1, k), eid(i, j + 1, k),
                               eid(i, j, k - 1), eid(i, j, k + 1)]
                nbr_face[e] = [1, 0, 3, 2, 5, 4]
                if walls_z:
                    if k == 0:
                        nbr_elem[e, 4] = -1
                    if k == nz - 1:
                        nbr_elem[e, 5] = -2
    return dict(n_elem=E, n_geom=ng, geom_nodes=g.copy(), xyz=np.ascontiguousarray(xyz.reshape(E, 3, ng ** 3)),
                nbr_elem=nbr_elem, nbr_face=nbr_face, nbr_orient=nbr_orient,
                kind="box", lengths=(Lx, Ly, Lz), shape=(nx, ny, nz))


# --------------------------------------------------------------------------------------
# polytropic hydrostatic background (Eq. 25-27)
# --------------------------------------------------------------------------------------
@dataclass
class Shell:
    """Nondimensional shell of SURVEY.md S8(d): r_b/r_t = 0.70/0.95 (Table 1 aspect 4.87/6.61,
    PAPER.md:206), gamma = 5/3, R = 1, GM = 1, rho_b = 1."""
    r_b: float = 0.70
    r_t: float = 0.95
    gamma: float = 5.0 / 3.0
    R_gas: float = 1.0
    GM: float = 1.0
    rho_b: float = 1.0
    N_rho: float = 3.0

    @property
    def Cp(self):
        return self.gamma * self.R_gas / (self.gamma - 1.0)

    @property
    def T_b(self):
        """Eq. 27."""
        phi_b, phi_t = -self.GM / self.r_b, -self.GM / self.r_t
        return (phi_t - phi_b) / (self.Cp * (1.0 - np.exp(-(self.gamma - 1.0) * self.N_rho)))

    def profile(self, r):
        """rho, p, T at radius r (Eq. 26)."""
        theta = 1.0 - (-self.GM / r + self.GM / self.r_b) / (self.Cp * self.T_b)
        T = self.T_b * theta
        rho = self.rho_b * theta ** (1.0 / (self.gamma - 1.0))
        p = self.rho_b * self.R_gas * self.T_b * theta ** (self.gamma / (self.gamma - 1.0))
        return rho, p, T


def flux_balanced_profile(shell: "Shell", L: float, kappa: float, kr=None, n_grid: int = 4001):
    """The "almost flux-balanced" initial stratification of PAPER.md:169-186 (SV, Eq. 28-31), radial profiles on a uniform grid.

    1. polytrope of Eq. 26-27: rho0(r), T0(r), dT0/dr = -g/Cp;
    2. entropy gradient that carries the luminosity L through every radial layer (Eq. 28 with q_r = L/(4 pi r^2), "the total
       heat flux from the shell is constant through each radial layer"), on the polytrope's rho0, T0 (Eq. 29):
           dS/dr = -(L/(4 pi r^2) + kr(r) rho0 Cp dT0/dr) / (kappa rho0 T0)
       (Eq. 29 as printed lacks the minus sign that its own derivation from Eq. 28 gives: reading G30 of DESIGN.md);
    3. S(r) = S_b + int_{r_b}^{r} dS/dr (Eq. 30), S_b = Cp ln(p_b^{1/gamma}/rho_b) (Eq. 10), by Simpson's rule;
    4. new density from hydrostatic balance dp/dr = -rho g (Eq. 25) with p = rho^gamma exp(gamma S/Cp) (Eq. 10 inverted):
           d rho/dr = -(rho/Cp dS/dr + (g/gamma) rho^(2-gamma) exp(-gamma S/Cp))          (Eq. 31; the printed exponent has
       the opposite sign, which contradicts Eq. 10 and 25: reading G31), integrated from rho(r_b) = rho_b by classical RK4;
    5. p = rho^gamma exp(gamma S/Cp), T = p/(rho R).
    kr: None, or a function r -> kappa_r(r).  Returns dict(r, rho, p, T, S, dSdr) of n_grid points.
    With L = 0 and kr = None the result is the polytrope itself (isentropic)."""
    if n_grid < 3 or n_grid % 2 == 0:
        raise ValueError("n_grid must be odd and >= 3")
    g_, Cp, gam, R = shell.GM, shell.Cp, shell.gamma, shell.R_gas
    krf = (lambda r: 0.0 * r) if kr is None else kr

    def dSdr(r):
        rho0, _, T0 = shell.profile(r)
        dT0 = -g_ / (Cp * r * r)
        return -(L / (4.0 * np.pi * r * r) + krf(r) * rho0 * Cp * dT0) / (kappa * rho0 * T0)

    r = np.linspace(shell.r_b, shell.r_t, n_grid)
    h = r[1] - r[0]
    rm = 0.5 * (r[:-1] + r[1:])                       # interval mid points
    f, fm = dSdr(r), dSdr(rm)
    rho_b, p_b, _ = shell.profile(shell.r_b)
    S_b = Cp * np.log(p_b ** (1.0 / gam) / rho_b)
    S = S_b + np.concatenate([[0.0], np.cumsum(h / 6.0 * (f[:-1] + 4.0 * fm + f[1:]))])       # Simpson on every interval
    # S at the mid points (for RK4): Simpson on the half interval with the quarter point
    rq = 0.5 * (r[:-1] + rm)
    Sm = S[:-1] + 0.5 * h / 6.0 * (f[:-1] + 4.0 * dSdr(rq) + fm)

    def rhs(rr, rho, Sv, dS):
        return -(rho / Cp * dS + (g_ / (rr * rr)) / gam * rho ** (2.0 - gam) * np.exp(-gam * Sv / Cp))

    rho = np.empty(n_grid)
    rho[0] = rho_b
    for k in range(n_grid - 1):
        k1 = rhs(r[k], rho[k], S[k], f[k])
        k2 = rhs(rm[k], rho[k] + 0.5 * h * k1, Sm[k], fm[k])
        k3 = rhs(rm[k], rho[k] + 0.5 * h * k2, Sm[k], fm[k])
        k4 = rhs(r[k + 1], rho[k] + h * k3, S[k + 1], f[k + 1])
        rho[k + 1] = rho[k] + h / 6.0 * (k1 + 2.0 * k2 + 2.0 * k3 + k4)
    pr = rho ** gam * np.exp(gam * S / Cp)
    return dict(r=r, rho=rho, p=pr, T=pr / (rho * R), S=S, dSdr=f)


def conserved(rho, U, p, B, psi, gamma):
    """Q = (rho, rho U, E, B, psi) with E of Eq. 3.  U, B: [3,...]."""
    E = p / (gamma - 1.0) + 0.5 * rho * (U ** 2).sum(0) + 0.5 * (B ** 2).sum(0) + 0.5 * psi ** 2
    return np.stack([rho, rho * U[0], rho * U[1], rho * U[2], E, B[0], B[1], B[2], psi])


def shell_state(x_sol: np.ndarray, shell: Shell, seed: int, u_amp: float = 1e-4, b_amp: float = 1e-3,
                dipole: bool = True, b_random: float = 0.1, flatten: float = 0.0, background: dict | None = None) -> np.ndarray:
    """Seeded stratified-shell state at the solution-point coordinates x_sol [3,E,n^3].

    Recipe (BASELINE.json configs): polytrope of Eq. 26-27; velocity
    = u_amp * c_s(r) * uniform(-1,1)^3; B = B0*(dipole + b_random*uniform(-1,1)^3) with
    B0 = b_amp*sqrt(gamma p_top) ("equipartition" read as B^2 = rho c_s^2 at the top) --
    or B0*uniform(-1,1)^3 alone when dipole=False ("weak random B seed"); psi = 0.
    `flatten` in [0,1] blends the background towards its shell-mean (non-equilibrium inputs
    for the naive-relative-error parity check).  `background`: the flux-balanced
    stratification of Eq. 28-31 (flux_balanced_profile) in place of the polytrope.
    Draw order: pu = uniform(-1,1,(3,E,n^3)) then pb = uniform(-1,1,(3,E,n^3)).
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    shp = x_sol.shape[1:]
    pu = rng.uniform(-1.0, 1.0, (3,) + shp)
    pb = rng.uniform(-1.0, 1.0, (3,) + shp)
    r = np.sqrt((x_sol ** 2).sum(0))
    if background is not None:      # radial profiles of flux_balanced_profile (Eq. 28-31) instead of the polytrope of Eq. 26
        rho = np.exp(np.interp(r, background["r"], np.log(background["rho"])))
        p = np.exp(np.interp(r, background["r"], np.log(background["p"])))
    else:
        rho, p, _ = shell.profile(r)
    if flatten:
        rho = (1 - flatten) * rho + flatten * rho.mean()
        p = (1 - flatten) * p + flatten * p.mean()
    cs = np.sqrt(shell.gamma * p / rho)
    U = u_amp * cs * pu
    _, p_t, _ = shell.profile(shell.r_t)
    B0 = b_amp * np.sqrt(shell.gamma * p_t)
    if dipole:
        x, y, z = x_sol
        dip = shell.r_b ** 3 * np.stack([3 * z * x / r ** 5, 3 * z * y / r ** 5, 3 * z * z / r ** 5 - 1.0 / r ** 3])
        B = B0 * (dip + b_random * pb)
    else:
        B = B0 * pb
    return np.ascontiguousarray(conserved(rho, U, p, B, np.zeros(shp), shell.gamma))


# --------------------------------------------------------------------------------------
# BASELINE.json workload configurations
# --------------------------------------------------------------------------------------
OMEGA_ND = 0.129   # paper's Omega * sqrt(L^3/GM_sun), Table 1


@dataclass
class Workload:
    name: str
    order: int
    n_z: int
    n_r: int
    N_rho: float
    seed: int
    diffusion: float            # nu = kappa = eta (0 => diffusion flag off)
    dipole: bool = True
    n_steps: int = 2
    shell: Shell = field(default_factory=Shell)

    @property
    def n_elem(self):
        return 6 * self.n_r * self.n_z ** 2

    def physics(self, c_h: float) -> Physics:
        sh = self.shell
        flags = FLAG_GRAVITY | FLAG_CORIOLIS | FLAG_POWELL | FLAG_GLM_DAMP
        if self.diffusion > 0:
            flags |= FLAG_DIFFUSION
        return Physics(gamma=sh.gamma, R_gas=sh.R_gas, Cp=sh.Cp, GM=sh.GM, Omega=OMEGA_ND,
                       nu=self.diffusion, kappa=self.diffusion, eta=self.diffusion,
                       c_h=c_h, a_psi=c_h / (0.18 * (sh.r_t - sh.r_b)),
                       bc_mag_inner=BC_CONDUCTING, bc_mag_outer=BC_RADIAL, flags=flags)

    def mesh(self, gnodes=None):
        g = lobatto_abscissae(self.order + 1) if gnodes is None else gnodes
        return cubed_sphere_shell(self.n_z, self.n_r, self.shell.r_b, self.shell.r_t, g)

    def state(self, x_sol):
        return shell_state(x_sol, self.shell, self.seed, dipole=self.dipole)

    def dt(self, wavespeed: float, dxi_min: float) -> float:
        """CFL step of SURVEY.md S8(d): Delta = min(dr, r_b*(pi/2)/N_z) * (X_f1 - X_f0)."""
        sh = self.shell
        delta = min((sh.r_t - sh.r_b) / self.n_r, sh.r_b * 0.5 * np.pi / self.n_z) * dxi_min
        dt = 0.4 * delta / wavespeed
        if self.diffusion > 0:
            dt = min(dt, 0.05 * delta ** 2 / self.diffusion)
        return dt


def workload(name: str) -> Workload:
    """configs[0..3] of BASELINE.json and the order sweep configs[4] ('sweep_n4' .. 'sweep_n9' at N_rho = 3, 'sweep1_n4' ..
    'sweep1_n9' at N_rho = 1)."""
    sh1, sh3 = Shell(N_rho=1.0), Shell(N_rho=3.0)
    table = {
        "config0": Workload("config0", 6, 4, 2, 1.0, 0, 0.0, True, 2, sh1),
        "config1": Workload("config1", 6, 8, 4, 3.0, 1, 1e-3, True, 20, sh3),
        "config2": Workload("config2", 6, 16, 8, 3.0, 2, 0.0, False, 10, sh3),
        "config3": Workload("config3", 6, 32, 12, 3.0, 3, 1e-3, True, 10, sh3),
        "sweep_n4": Workload("sweep_n4", 4, 48, 16, 3.0, 4, 1e-3, True, 2, sh3),
        "sweep_n5": Workload("sweep_n5", 5, 34, 12, 3.0, 4, 1e-3, True, 2, sh3),
        "sweep_n6": Workload("sweep_n6", 6, 28, 10, 3.0, 4, 1e-3, True, 2, sh3),
        "sweep_n7": Workload("sweep_n7", 7, 24, 8, 3.0, 4, 1e-3, True, 2, sh3),
        # orders 8 and 9 run on the scalar three-kernel path (with diffusion its gradient tiles live in a global scratch area)
        "sweep_n8": Workload("sweep_n8", 8, 22, 7, 3.0, 4, 1e-3, True, 2, sh3),
        "sweep_n9": Workload("sweep_n9", 9, 18, 7, 3.0, 4, 1e-3, True, 2, sh3),
    }
    # configs[4] asks for N_rho = 1 and 3: the same meshes on the shallower polytrope
    for n in range(4, 10):
        w3_ = table[f"sweep_n{n}"]
        table[f"sweep1_n{n}"] = Workload(f"sweep1_n{n}", n, w3_.n_z, w3_.n_r, 1.0, 4, 1e-3, True, 2, sh1)
    return table[name]


# --------------------------------------------------------------------------------------
# a walled box whose elements have randomly rotated local axes: exercises every face pairing
# (xi<->eta<->zeta) and every orientation code; test input only
# --------------------------------------------------------------------------------------
def _proper_rotations():
    rots = []
    for perm in itertools.permutations(range(3)):
        for flips in itertools.product((False, True), repeat=3):
            sign = 1
            p = list(perm)                      # parity of the permutation
            for i in range(3):
                for j in range(i + 1, 3):
                    if p[i] > p[j]:
                        sign = -sign
            for f in flips:
                if f:
                    sign = -sign
            if sign > 0:
                rots.append((perm, flips))
    return rots


def scrambled_box(nx: int, ny: int, nz: int, lengths, gnodes: np.ndarray, seed: int, distort: float = 0.0):
    """nx*ny*nz hexes on a box with walls on every outer face (z-low faces tagged -1, all others -2); every
    element's local (xi,eta,zeta) axes are rotated by a random proper rotation, so neighbours meet through
    arbitrary local faces and orientations.  gnodes must be symmetric under x -> 1-x."""
    g = np.asarray(gnodes, np.float64)
    if np.abs(g + g[::-1] - 1.0).max() > 1e-14:
        raise ValueError("gnodes must be symmetric")
    base = periodic_box(nx, ny, nz, lengths, g, distort=distort, walls_z=True)
    ng, E = g.size, base["n_elem"]
    xyz = base["xyz"].reshape(E, 3, ng, ng, ng)          # [E,comp,c,b,a]
    rng = np.random.Generator(np.random.PCG64(seed))
    rots = _proper_rotations()
    out = np.empty_like(xyz)
    for e in range(E):
        perm, flips = rots[rng.integers(len(rots))]
        A = np.transpose(xyz[e], (0, 3, 2, 1))             # [comp,a,b,c] = axes (xi,eta,zeta)
        A = np.transpose(A, (0,) + tuple(1 + p for p in perm))
        for ax, f in enumerate(flips):
            if f:
                A = np.flip(A, axis=1 + ax)
        out[e] = np.transpose(A, (0, 3, 2, 1))             # back to [comp,c,b,a]
    corners = np.transpose(out[:, :, ::ng - 1, ::ng - 1, ::ng - 1], (0, 1, 4, 3, 2))   # [E,3,xi,eta,zeta]
    Lz = lengths[2]

    def wall_tag(c):
        return np.where(c[:, 2] < 1e-9 * Lz, -1, -2).astype(np.int32)

    nbr_elem, nbr_face, nbr_orient = hex_connectivity(corners, wall_tag)
    return dict(n_elem=E, n_geom=ng, geom_nodes=g.copy(), xyz=np.ascontiguousarray(out.reshape(E, 3, ng ** 3)),
                nbr_elem=nbr_elem, nbr_face=nbr_face, nbr_orient=nbr_orient, kind="scrambled_box",
                lengths=tuple(lengths), shape=(nx, ny, nz))


# --------------------------------------------------------------------------------------
# patch extraction: the sub-mesh of all elements within `rings` face-neighbour steps of `center`.
# The SD residual of an element depends on its neighbours' states (Rusanov, BR1 common solution) and, with
# diffusion, on its neighbours' gradients, i.e. on two rings; a 2-ring patch therefore reproduces the residual of
# its centre element exactly, whatever closes the patch.  Used for parity at full benchmark sizes, where the CPU
# oracle cannot run the whole mesh.  Pure indexing: no arithmetic of the method.
# --------------------------------------------------------------------------------------
def extract_patch(mesh: dict, center: int, rings: int = 2):
    """Returns (patch_mesh, elems): elems[i] = index in `mesh` of patch element i (elems[0] == center).
    Faces whose neighbour lies outside the patch are closed with an outer wall (-2); wall faces keep their tag."""
    nbr = mesh["nbr_elem"]
    elems, seen, frontier = [int(center)], {int(center)}, [int(center)]
    for _ in range(rings):
        nxt = []
        for e in frontier:
            for f in range(6):
                ne = int(nbr[e, f])
                if ne >= 0 and ne not in seen:
                    seen.add(ne)
                    elems.append(ne)
                    nxt.append(ne)
        frontier = nxt
    elems = np.asarray(elems, np.int64)
    local = {int(g): i for i, g in enumerate(elems)}
    pe = np.empty((elems.size, 6), np.int32)
    for i, g in enumerate(elems):
        for f in range(6):
            ne = int(nbr[g, f])
            pe[i, f] = ne if ne < 0 else local.get(ne, -2)
    out = dict(n_elem=int(elems.size), n_geom=mesh["n_geom"], geom_nodes=mesh["geom_nodes"].copy(),
               xyz=np.ascontiguousarray(mesh["xyz"][elems]), nbr_elem=pe,
               nbr_face=np.ascontiguousarray(mesh["nbr_face"][elems]), nbr_orient=np.ascontiguousarray(mesh["nbr_orient"][elems]),
               kind="patch")
    return out, elems


# --------------------------------------------------------------------------------------
# element partitions for multi-GPU runs: contiguous blocks of the element order; every rank's local
# mesh = its owned elements followed by ghost copies of their off-rank face neighbours, plus the lists of faces whose
# data cross between ranks.  Pure indexing: no arithmetic of the method.
# --------------------------------------------------------------------------------------
def partition_mesh(mesh: dict, n_parts: int, rank: int | None = None):
    """Split `mesh` into n_parts partitions (rank p owns the global elements [E p / P, E (p+1) / P)).

    Returns a list of partition dicts (or the one of `rank`), each with
      mesh        local mesh dict: owned elements [0, n_owned) then ghosts; nbr_elem of owned elements holds local indices
                  (ghost faces of ghosts are closed with -2 and never used)
      n_owned     number of owned elements
      elems       int64[n_local]: global element of every local element (owned then ghosts, ghosts in increasing order)
      send_elem, send_face, send_counts   faces of owned elements whose data other ranks need, grouped by destination rank
                  in increasing rank order (send_counts[q] items go to rank q), each group sorted by (global element, face)
      recv_elem, recv_face, recv_counts   the matching faces of ghost elements, grouped by source rank, same order
    The face (g, f) of an element g owned by q is needed by p when the element across f is owned by p != q."""
    E = int(mesh["n_elem"])
    P = int(n_parts)
    if P < 1 or P > E:
        raise ValueError("need 1 <= n_parts <= n_elem")
    bounds = [E * p // P for p in range(P + 1)]
    owner = np.empty(E, np.int64)
    for p in range(P):
        owner[bounds[p]:bounds[p + 1]] = p
    nbr, nface = mesh["nbr_elem"], mesh["nbr_face"]
    parts = []
    for p in (range(P) if rank is None else [int(rank)]):
        lo, hi = bounds[p], bounds[p + 1]
        own = np.arange(lo, hi)
        ne = nbr[lo:hi]                                             # [n_owned, 6]
        off = (ne >= 0) & ((ne < lo) | (ne >= hi))
        ghosts = np.unique(ne[off])
        elems = np.concatenate([own, ghosts]).astype(np.int64)
        local = {int(g): i for i, g in enumerate(elems)}
        pe = np.full((elems.size, 6), -2, np.int32)
        for i in range(hi - lo):
            for f in range(6):
                v = int(ne[i, f])
                pe[i, f] = v if v < 0 else local[v]
        pm = dict(n_elem=int(elems.size), n_geom=mesh["n_geom"], geom_nodes=mesh["geom_nodes"].copy(),
                  xyz=np.ascontiguousarray(mesh["xyz"][elems]), nbr_elem=pe,
                  nbr_face=np.ascontiguousarray(mesh["nbr_face"][elems]), nbr_orient=np.ascontiguousarray(mesh["nbr_orient"][elems]),
                  kind="partition")
        # faces crossing the partition boundary, seen from the owned side: (e, f) with the neighbour on another rank
        ei, fi = np.nonzero(off)
        nb_glob = ne[ei, fi]
        nb_rank = owner[nb_glob]
        # what WE send to rank q: our face (e, f); sorted by (destination, global e, f)
        order = np.lexsort((fi, ei + lo, nb_rank))
        send_elem, send_face = ei[order].astype(np.int32), fi[order].astype(np.uint8)
        send_counts = np.bincount(nb_rank, minlength=P).astype(np.int64)
        # what we RECEIVE from rank q: the neighbour's face (g, f'), f' = nbr_face[e, f]; sorted by (source, global g, f')
        nb_face = nface[ei + lo, fi]
        order = np.lexsort((nb_face, nb_glob, nb_rank))
        recv_elem = np.array([local[int(g)] for g in nb_glob[order]], np.int32)
        recv_face = nb_face[order].astype(np.uint8)
        # a ghost face can be reached from one owned face only (conforming mesh), but be safe against duplicates
        key = recv_elem.astype(np.int64) * 6 + recv_face
        if np.unique(key).size != key.size:
            raise ValueError("a ghost face is referenced twice: the mesh is not conforming")
        parts.append(dict(mesh=pm, n_owned=int(hi - lo), elems=elems, rank=p, n_parts=P,
                          send_elem=send_elem, send_face=send_face, send_counts=send_counts,
                          recv_elem=recv_elem, recv_face=recv_face, recv_counts=send_counts.copy()))
    return parts if rank is None else parts[0]
