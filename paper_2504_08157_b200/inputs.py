"""Seeded synthetic input generators (meshes, reference states, initial states, forcing).

This module is INPUT DATA ONLY.  It holds none of the method's arithmetic (no derivative
matrix, no metric terms, no DSS, no tendencies, no time stepping) and is the one module
that both the CPU oracle tests (``oracle/``) and the CUDA path use, so that the two see
bit-identical inputs.  It imports neither of them.

The paper's own workloads (observed Hurricane-Guillermo heating; the Jordan
sounding, L298; the Nolan-type vortex of Eq. 17) are not available here; the
generators below take their *shape* -- limited-area box of column-preserving hexahedra
(L162-L168, L256), N = 3..8, 25-300 M nodes, localised heating near the vortex core -- and
stand in for them ("Input recipe").

Layout conventions (shared by oracle and CUDA path, see include/numa_b200.h):
  * Nq = N+1, Mn = Nq**3, local node index  n = i + Nq*(j + Nq*k)  (i = xi fastest),
  * arrays are element-local SoA:  field[m][e][n]  (``q_e(i,j,k,e,m)``),
  * element order is column-major: e = ez + nz*(ex + nx*ey)  (whole columns contiguous,
    PAPER.md:L164 "keep the grid columns within a partition"),
  * faces 0..5 = xi-, xi+, eta-, eta+, zeta-, zeta+.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np
from numpy.polynomial import legendre as _leg

SEED_BASE = 250408157  # seed = 250408157 + 1000*config + refresh_index

# Physical constants passed to both sides through numa_params (reading Q6).
CONSTANTS = dict(g=9.81, p_a=1.0e5, c_p=1004.67, c_v=717.5, R_gas=1004.67 - 717.5)


def lgl_points(N: int) -> np.ndarray:
    """Legendre-Gauss-Lobatto points on [-1,1] (generator's own copy: only used to PLACE
    nodes; the oracle and the CUDA library each compute their own tables)."""
    if N < 1:
        raise ValueError("N >= 1")
    c = np.zeros(N + 1)
    c[N] = 1.0
    interior = _leg.legroots(_leg.legder(c)) if N > 1 else np.array([])
    x = np.concatenate(([-1.0], np.sort(interior.real), [1.0]))
    # two Newton steps on P'_N to polish the interior roots
    d1 = _leg.legder(c)
    d2 = _leg.legder(c, 2)
    for _ in range(2):
        xi = x[1:-1]
        x[1:-1] = xi - _leg.legval(xi, d1) / _leg.legval(xi, d2)
    x = 0.5 * (x - x[::-1])  # enforce symmetry exactly
    return x


@dataclass
class Mesh:
    N: int
    nx: int
    ny: int
    nz: int
    xyz: np.ndarray          # [3][Ne][Mn] float64
    intma_cg: np.ndarray     # [Ne][Mn]    int32, unique CG node id
    face_bc: np.ndarray      # [Ne][6]     uint8, 0 interior / periodic, 1 no-flux wall
    n_global: int
    extent: tuple            # (Lx, Ly, Lz)
    origin: tuple = (0.0, 0.0, 0.0)
    periodic: tuple = (False, False, False)

    @property
    def Nq(self):
        return self.N + 1

    @property
    def Mn(self):
        return (self.N + 1) ** 3

    @property
    def n_elem(self):
        return self.nx * self.ny * self.nz

    @property
    def n_local(self):
        return self.n_elem * self.Mn


def geometric_heights(Lz: float, nz: int, ratio: float) -> np.ndarray:
    """Element heights growing geometrically by `ratio` (config 3: 1.1), summing to Lz."""
    if abs(ratio - 1.0) < 1e-14:
        return np.full(nz, Lz / nz)
    h0 = Lz * (ratio - 1.0) / (ratio ** nz - 1.0)
    return h0 * ratio ** np.arange(nz)


def box_mesh(N, nx, ny, nz, extent, origin=(0.0, 0.0, 0.0), z_ratio=1.0, perturb=0.0,
             seed=0, periodic=(False, False, False)) -> Mesh:
    """Box of nx*ny*nz hexahedra with trilinear (vertex-defined) geometry.

    perturb: element VERTICES are moved by uniform +-perturb*h per component (h = local
    element size in that direction), with the wall-normal component left at zero on
    non-periodic boundary vertices so walls stay planar (reading Q13; config 1:
    "seed perturbs the node coordinates by <=5% of the element size").  LGL nodes are
    placed by trilinear interpolation and made bit-identical across element copies.
    """
    Nq = N + 1
    Lx, Ly, Lz = extent
    x0, y0, z0 = origin
    px, py, pz = periodic
    rng = np.random.default_rng(seed)
    vx = x0 + np.linspace(0.0, Lx, nx + 1)
    vy = y0 + np.linspace(0.0, Ly, ny + 1)
    hz = geometric_heights(Lz, nz, z_ratio)
    vz = z0 + np.concatenate(([0.0], np.cumsum(hz)))
    vz[-1] = z0 + Lz
    VX, VY, VZ = np.meshgrid(vx, vy, vz, indexing="ij")  # [nx+1][ny+1][nz+1]
    VX = VX.copy(); VY = VY.copy(); VZ = VZ.copy()
    if perturb > 0.0:
        hx = Lx / nx
        hy = Ly / ny
        hzv = np.minimum(np.concatenate((hz[:1], hz)), np.concatenate((hz, hz[-1:])))
        dx = rng.uniform(-perturb, perturb, VX.shape) * hx
        dy = rng.uniform(-perturb, perturb, VY.shape) * hy
        dz = rng.uniform(-perturb, perturb, VZ.shape) * hzv[None, None, :]
        if px:
            dx[-1] = dx[0]; dy[-1] = dy[0]; dz[-1] = dz[0]
        else:
            dx[0] = 0.0; dx[-1] = 0.0
        if py:
            dx[:, -1] = dx[:, 0]; dy[:, -1] = dy[:, 0]; dz[:, -1] = dz[:, 0]
        else:
            dy[:, 0] = 0.0; dy[:, -1] = 0.0
        if pz:
            dx[:, :, -1] = dx[:, :, 0]; dy[:, :, -1] = dy[:, :, 0]; dz[:, :, -1] = dz[:, :, 0]
        else:
            dz[:, :, 0] = 0.0; dz[:, :, -1] = 0.0
        VX += dx; VY += dy; VZ += dz

    xi = lgl_points(N)
    a = 0.5 * (1.0 - xi)      # weight of the "low" vertex along one direction
    b = 0.5 * (1.0 + xi)

    Ne = nx * ny * nz
    Mn = Nq ** 3
    # element (ex,ey,ez) -> e = ez + nz*(ex + nx*ey)
    EY, EX, EZ = np.meshgrid(np.arange(ny), np.arange(nx), np.arange(nz), indexing="ij")
    ex = EX.reshape(-1); ey = EY.reshape(-1); ez = EZ.reshape(-1)  # order: ey slowest, ez fastest
    assert np.array_equal(ez + nz * (ex + nx * ey), np.arange(Ne))

    # trilinear weights for local node n = i + Nq*(j + Nq*k): W[c][n], c = corner (dx,dy,dz)
    wi = np.stack((a, b))  # [2][Nq]
    xyz = np.empty((3, Ne, Mn))
    if perturb == 0.0:
        # separable (axis-aligned) mesh: each coordinate depends on one index only, so that it
        # is bit-identical along the other two reference directions
        lx = vx[ex][:, None] * a[None, :] + vx[ex + 1][:, None] * b[None, :]   # [Ne][Nq]
        ly = vy[ey][:, None] * a[None, :] + vy[ey + 1][:, None] * b[None, :]
        lz = vz[ez][:, None] * a[None, :] + vz[ez + 1][:, None] * b[None, :]
        shape = (Ne, Nq, Nq, Nq)
        xyz[0] = np.broadcast_to(lx[:, None, None, :], shape).reshape(Ne, Mn)
        xyz[1] = np.broadcast_to(ly[:, None, :, None], shape).reshape(Ne, Mn)
        xyz[2] = np.broadcast_to(lz[:, :, None, None], shape).reshape(Ne, Mn)
    for comp, V in enumerate((VX, VY, VZ)):
        if perturb == 0.0:
            break
        acc = np.zeros((Ne, Nq, Nq, Nq))  # [e][k][j][i]
        for cz in (0, 1):
            for cy in (0, 1):
                for cx in (0, 1):
                    corner = V[ex + cx, ey + cy, ez + cz]  # [Ne]
                    w = (wi[cz][:, None, None] * wi[cy][None, :, None] * wi[cx][None, None, :])
                    acc += corner[:, None, None, None] * w[None]
        xyz[comp] = acc.reshape(Ne, Mn)

    # unique CG numbering on the global LGL lattice (x fastest); periodic wraps.
    ngx = nx * N + (0 if px else 1)
    ngy = ny * N + (0 if py else 1)
    ngz = nz * N + (0 if pz else 1)
    ii = np.arange(Nq)
    gx = (ex[:, None] * N + ii[None, :]) % ngx     # [Ne][Nq]
    gy = (ey[:, None] * N + ii[None, :]) % ngy
    gz = (ez[:, None] * N + ii[None, :]) % ngz
    g = (gx[:, None, None, :].astype(np.int64)
         + ngx * (gy[:, None, :, None].astype(np.int64)
                  + ngy * gz[:, :, None, None].astype(np.int64)))      # [e][k][j][i]
    n_global = ngx * ngy * ngz
    if n_global >= 2 ** 31:
        raise ValueError("n_global exceeds int32")
    intma_cg = g.reshape(Ne, Mn).astype(np.int32)

    # make coordinates of coincident copies bit-identical (not across periodic seams,
    # where the physical coordinates legitimately differ by the period).
    if not (px or py or pz):
        for comp in range(3):
            glob = np.empty(n_global)
            glob[intma_cg.reshape(-1)] = xyz[comp].reshape(-1)
            xyz[comp] = glob[intma_cg]

    face_bc = np.zeros((Ne, 6), dtype=np.uint8)
    if not px:
        face_bc[ex == 0, 0] = 1; face_bc[ex == nx - 1, 1] = 1
    if not py:
        face_bc[ey == 0, 2] = 1; face_bc[ey == ny - 1, 3] = 1
    if not pz:
        face_bc[ez == 0, 4] = 1; face_bc[ez == nz - 1, 5] = 1
    return Mesh(N=N, nx=nx, ny=ny, nz=nz, xyz=xyz, intma_cg=intma_cg, face_bc=face_bc,
                n_global=int(n_global), extent=tuple(extent), origin=tuple(origin),
                periodic=tuple(periodic))


def node_levels(mesh: Mesh):
    """Horizontal level of every local node: level[e][n] = ez*N + k (int32) and the number of
    levels.  Index data only (like intma_cg): the nodes "at a height z" over which the RI
    diagnostic integrates and averages (Eq. 19, 22; reading Q25)."""
    N, Nq = mesh.N, mesh.N + 1
    ez = np.arange(mesh.n_elem) % mesh.nz                       # e = ez + nz*(ex + nx*ey)
    k = np.arange(mesh.Mn) // (Nq * Nq)
    n_lev = mesh.nz * N + (0 if mesh.periodic[2] else 1)
    lev = (ez[:, None] * N + k[None, :]) % n_lev
    return np.ascontiguousarray(lev, dtype=np.int32), int(n_lev)


# --------------------------------------------------------------------------------------
# reference (background) states: hydrostatic, functions of z only
# --------------------------------------------------------------------------------------
def reference_neutral(z, theta0=300.0, c=CONSTANTS):
    """Neutral atmosphere theta0 = const (configs 1-2; reading Q17)."""
    g, p_a, c_p, c_v, R = c["g"], c["p_a"], c["c_p"], c["c_v"], c["R_gas"]
    pi0 = 1.0 - g * z / (c_p * theta0)
    rho0 = p_a * pi0 ** (c_v / R) / (R * theta0)
    return rho0, np.full_like(z, theta0)


def reference_stable(z, theta_s=300.0, N_bv=0.01, c=CONSTANTS):
    """Constant Brunt-Vaisala-frequency sounding (configs 3-5; stands in for the Jordan
    sounding of PAPER.md:L298, which is not available; reading Q17)."""
    g, p_a, c_p, c_v, R = c["g"], c["p_a"], c["c_p"], c["c_v"], c["R_gas"]
    s = N_bv ** 2 / g
    theta0 = theta_s * np.exp(s * z)
    pi0 = 1.0 + g * g / (c_p * theta_s * N_bv ** 2) * (np.exp(-s * z) - 1.0)
    rho0 = p_a * pi0 ** (c_v / R) / (R * theta0)
    return rho0, theta0


def reference_uniform(z, rho0=1.2, theta0=300.0):
    """Uniform background (used with g=0 by the free-stream / manufactured-solution pins)."""
    return np.full_like(z, rho0), np.full_like(z, theta0)


# --------------------------------------------------------------------------------------
# initial states
# --------------------------------------------------------------------------------------
def bubble_state(mesh: Mesh, rho0, theta0, centre, radius, amp=0.5):
    """Cosine warm bubble theta' = amp/2*(1+cos(pi r/radius)), r<radius; rho' chosen so
    that p' = 0 (pressure-balanced): (1+rho'/rho0)(1+theta'/theta0) = 1.  u = 0."""
    x, y, z = mesh.xyz
    r = np.sqrt((x - centre[0]) ** 2 + (y - centre[1]) ** 2 + (z - centre[2]) ** 2)
    thp = np.where(r < radius, 0.5 * amp * (1.0 + np.cos(np.pi * r / radius)), 0.0)
    rhop = -rho0 * thp / (theta0 + thp)
    q = np.zeros((5,) + x.shape)
    q[0] = rhop
    q[4] = thp
    return q


def sinusoidal_velocity(mesh: Mesh, seed, amplitude=0.1, n_modes=3):
    """Config 2: random smooth 3-mode sinusoidal velocity, integer wave numbers 1..3 per
    direction, scaled to max |component| = amplitude, times wall-vanishing envelopes so
    u.n = 0 on the (planar) walls."""
    rng = np.random.default_rng(seed)
    x, y, z = mesh.xyz
    Lx, Ly, Lz = mesh.extent
    x0, y0, z0 = mesh.origin
    X = (x - x0) / Lx; Y = (y - y0) / Ly; Z = (z - z0) / Lz
    vel = np.zeros((3,) + x.shape)
    for c in range(3):
        for _ in range(n_modes):
            k = rng.integers(1, 4, size=3)
            ph = rng.uniform(0, 2 * np.pi)
            A = rng.uniform(0.5, 1.0)
            vel[c] += A * np.sin(2 * np.pi * (k[0] * X + k[1] * Y + k[2] * Z) + ph)
    env = (np.sin(np.pi * X), np.sin(np.pi * Y), np.sin(np.pi * Z))
    for c in range(3):
        if not mesh.periodic[c]:
            vel[c] *= env[c]
        vel[c] *= amplitude / np.max(np.abs(vel[c]))
    return vel


def smooth_random_state(mesh: Mesh, rho0, theta0, seed, scales=(1e-2, 5.0, 5.0, 0.5, 2.0)):
    """Seeded smooth state with ALL five fields non-zero (parity protocol, reading Q19):
    a few low sinusoidal modes per field; velocity vanishes normal to non-periodic walls."""
    rng = np.random.default_rng(seed)
    x, y, z = mesh.xyz
    Lx, Ly, Lz = mesh.extent
    x0, y0, z0 = mesh.origin
    X = (x - x0) / Lx; Y = (y - y0) / Ly; Z = (z - z0) / Lz
    q = np.zeros((5,) + x.shape)
    for m in range(5):
        f = np.zeros_like(x)
        for _ in range(3):
            k = rng.integers(1, 3, size=3)
            ph = rng.uniform(0, 2 * np.pi)
            f += rng.uniform(0.5, 1.0) * np.sin(2 * np.pi * (k[0] * X + k[1] * Y + k[2] * Z) + ph)
        q[m] = scales[m] * f / np.max(np.abs(f))
    q[0] *= rho0  # rho' relative to the local background density
    env = (np.sin(np.pi * X), np.sin(np.pi * Y), np.sin(np.pi * Z))
    for c in range(3):
        if not mesh.periodic[c]:
            q[1 + c] *= env[c]
    return q


def vortex_state(mesh: Mesh, rho0_fun, f_cor, vmax=20.0, r_m=100e3, z_top=15e3, c=CONSTANTS):
    """Config 3: warm-core axisymmetric vortex in gradient-wind + hydrostatic balance
    (reading Q16; stands in for PAPER.md Eq. 17).

    v_t(r,z) = V(r) s(z),  V = vmax (r/r_m) exp((1-(r/r_m)^2)/2),  s = max(0, 1 - z/z_top)
    p'(r,z)  = -rho0(z) [ s^2 A(r) + f s B(r) ],  A = int_r^inf V^2/r' dr',  B = int_r^inf V dr'
    rho'     = -(1/g) dp'/dz ;  theta' from the equation of state.
    """
    g, p_a, c_p, c_v, R = c["g"], c["p_a"], c["c_p"], c["c_v"], c["R_gas"]
    gamma = c_p / c_v
    x, y, z = mesh.xyz
    Lx, Ly, _ = mesh.extent
    xc = mesh.origin[0] + 0.5 * Lx
    yc = mesh.origin[1] + 0.5 * Ly
    rx = x - xc; ry = y - yc
    r = np.sqrt(rx * rx + ry * ry)
    # radial tables by fine quadrature
    rt = np.linspace(0.0, 12.0 * r_m, 240001)
    Vt = vmax * (rt / r_m) * np.exp(0.5 * (1.0 - (rt / r_m) ** 2))
    with np.errstate(invalid="ignore", divide="ignore"):
        ia = np.where(rt > 0, Vt * Vt / rt, 0.0)
    def tail_integral(fv):
        seg = 0.5 * (fv[1:] + fv[:-1]) * np.diff(rt)
        out = np.zeros_like(rt)
        out[:-1] = np.cumsum(seg[::-1])[::-1]
        return out
    At = tail_integral(ia)
    Bt = tail_integral(Vt)
    V = np.interp(r, rt, Vt); A = np.interp(r, rt, At); B = np.interp(r, rt, Bt)
    s = np.clip(1.0 - z / z_top, 0.0, None)
    ds = np.where(z < z_top, -1.0 / z_top, 0.0)
    rho0, theta0 = rho0_fun(z)
    eps = 1.0
    rho0p, _ = rho0_fun(z + eps)
    rho0m, _ = rho0_fun(z - eps)
    drho0 = (rho0p - rho0m) / (2 * eps)
    pp = -rho0 * (s * s * A + f_cor * s * B)
    dppdz = -drho0 * (s * s * A + f_cor * s * B) - rho0 * (2 * s * ds * A + f_cor * ds * B)
    rhop = -dppdz / g
    p0 = p_a * (rho0 * R * theta0 / p_a) ** gamma
    theta = p_a * ((p0 + pp) / p_a) ** (1.0 / gamma) / ((rho0 + rhop) * R)
    vt = V * s
    with np.errstate(invalid="ignore", divide="ignore"):
        cs = np.where(r > 0, rx / r, 0.0)
        sn = np.where(r > 0, ry / r, 0.0)
    q = np.zeros((5,) + x.shape)
    q[0] = rhop
    q[1] = -vt * sn
    q[2] = vt * cs
    q[4] = theta - theta0
    return q


# --------------------------------------------------------------------------------------
# forcing
# --------------------------------------------------------------------------------------
def heating_field(mesh: Mesh, seed, n_cells=8, r_disc=150e3, peak=20.0 / 3600.0,
                  z_top=15e3, sigma_range=(5e3, 20e3)):
    """Prescribed latent heating S_theta [K/s]: sum of `n_cells`
    seeded rotated anisotropic Gaussians within r < r_disc of the domain centre, field
    maximum `peak` (20 K/h), vertical profile sin(pi z / z_top) below z_top."""
    rng = np.random.default_rng(seed)
    x, y, z = mesh.xyz
    Lx, Ly, _ = mesh.extent
    xc = mesh.origin[0] + 0.5 * Lx
    yc = mesh.origin[1] + 0.5 * Ly
    horiz = np.zeros_like(x)
    for _ in range(n_cells):
        rr = r_disc * np.sqrt(rng.uniform())
        ang = rng.uniform(0, 2 * np.pi)
        cx = xc + rr * np.cos(ang); cy = yc + rr * np.sin(ang)
        sa, sb = rng.uniform(*sigma_range, size=2)
        rot = rng.uniform(0, np.pi)
        amp = rng.uniform(0.25, 1.0)
        dx = x - cx; dy = y - cy
        xa = np.cos(rot) * dx + np.sin(rot) * dy
        xb = -np.sin(rot) * dx + np.cos(rot) * dy
        horiz += amp * np.exp(-0.5 * ((xa / sa) ** 2 + (xb / sb) ** 2))
    prof = np.where(z < z_top, np.sin(np.pi * z / z_top), 0.0)
    f = horiz * prof
    m = np.max(np.abs(f))
    return f * (peak / m) if m > 0 else f


def sponge_coefficient(mesh: Mesh, top=5e3, lateral=50e3, beta_max=0.05):
    """Rayleigh damping coefficient beta(x) [1/s] (reading Q9): top `top` metres
    and lateral `lateral` metres; beta = beta_max*min(1, s(d_top)+s(d_x)+s(d_y)),
    s(d) = sin^2(pi d / 2), d = fractional depth into the layer."""
    x, y, z = mesh.xyz
    Lx, Ly, Lz = mesh.extent
    x0, y0, z0 = mesh.origin
    def s(d):
        d = np.clip(d, 0.0, 1.0)
        return np.sin(0.5 * np.pi * d) ** 2
    dtop = (z - (z0 + Lz - top)) / top
    dx = np.maximum((x0 + lateral - x), (x - (x0 + Lx - lateral))) / lateral
    dy = np.maximum((y0 + lateral - y), (y - (y0 + Ly - lateral))) / lateral
    return beta_max * np.minimum(1.0, s(dtop) + s(dx) + s(dy))


# --------------------------------------------------------------------------------------
# the BASELINE.json configurations
# --------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    mesh: Mesh
    ref: np.ndarray               # [2][Ne][Mn]: rho0, theta0
    q: np.ndarray                 # [5][Ne][Mn]: rho', u, v, w, theta'
    dt: float
    n_steps: int
    f_cor: float = 0.0
    heating: Optional[np.ndarray] = None   # [Ne][Mn] K/s
    sponge: Optional[np.ndarray] = None    # [Ne][Mn] 1/s
    heating_refresh_steps: int = 0         # 0 = never refreshed
    config: int = 0
    constants: dict = field(default_factory=lambda: dict(CONSTANTS))
    notes: str = ""

    def heating_at(self, refresh_index: int) -> Optional[np.ndarray]:
        if self.heating is None:
            return None
        if refresh_index == 0:
            return self.heating
        return heating_field(self.mesh, SEED_BASE + 1000 * self.config + refresh_index)


def _tc_workload(config, name, N, nx, ny, nz, dt, n_steps, Lxy=1000e3, Lz=20e3, z_ratio=1.1):
    mesh = box_mesh(N, nx, ny, nz, (Lxy, Lxy, Lz), z_ratio=z_ratio)
    z = mesh.xyz[2]
    rho0, theta0 = reference_stable(z)
    f_cor = 5e-5
    q = vortex_state(mesh, reference_stable, f_cor)
    heat = heating_field(mesh, SEED_BASE + 1000 * config + 0)
    beta = sponge_coefficient(mesh)
    return Workload(name=name, mesh=mesh, ref=np.stack((rho0, theta0)), q=q, dt=dt,
                    n_steps=n_steps, f_cor=f_cor, heating=heat, sponge=beta,
                    heating_refresh_steps=60, config=config,
                    notes="dt reduced from the stated 1 s: explicit RK3 is unstable there "
                          "(DESIGN.md reading Q12)")


def paper_table1_workload(scale: float = 1.0) -> Workload:
    """The grid of the paper's Table 1 / Section 5.2: 800 km x 800 km x
    20 km, 80 x 80 x 24 elements at N = 5 (dx = 2 km, dz = 167 m uniform), 165,888,000 DOF, IMEX
    dt = 0.5 s -- with the synthetic vortex / heating / sponge of config 3 standing in for the
    paper's Nolan vortex, Jordan sounding and observed heating (not available here)."""
    nx = max(2, int(round(80 * scale)))
    return _tc_workload(3, "table1_tc_%dx%dx24_N5" % (nx, nx), 5, nx, nx, 24, dt=0.5, n_steps=100,
                        Lxy=800e3 * nx / 80.0, Lz=20e3, z_ratio=1.0)


# config 4: ~32 M local nodes for every N (reading Q14), 20 stretched layers
CFG4_NXY = {3: 158, 4: 113, 5: 86, 6: 68, 7: 56, 8: 47}
CFG4_DT = {3: 0.15, 4: 0.10, 5: 0.07, 6: 0.055, 7: 0.043, 8: 0.034}


# config 4's two literal examples (BASELINE.json: "N=4: 200x200x20 elements; N=7: 125x125x16"), which
# contradict its "~32M local nodes" (100 M and 128 M nodes; reading Q14): run as extra rows
CFG4_LITERAL = {4: (200, 20), 7: (125, 16)}


def make_workload(config: int, N: Optional[int] = None, scale: float = 1.0,
                  literal: bool = False) -> Workload:
    """Build BASELINE.json config 1..5.  `scale` < 1 shrinks the horizontal element counts
    (used by tests and by the bounded CPU-baseline sample); the physics is unchanged.
    literal=True (config 4, N = 4 or 7): the element counts BASELINE.json gives as examples."""
    if config == 1:
        N = 4 if N is None else N
        mesh = box_mesh(N, 4, 4, 4, (1000.0, 1000.0, 1000.0), perturb=0.05,
                        seed=SEED_BASE + 1000 * 1)
        rho0, theta0 = reference_neutral(mesh.xyz[2])
        q = bubble_state(mesh, rho0, theta0, (500.0, 500.0, 350.0), 250.0, 0.5)
        return Workload("cfg1_bubble_4x4x4_N%d" % N, mesh, np.stack((rho0, theta0)), q,
                        dt=0.01, n_steps=100, config=1)
    if config == 2:
        N = 4 if N is None else N
        nx = max(2, int(round(20 * scale))); nz = max(2, int(round(10 * scale)))
        mesh = box_mesh(N, nx, nx, nz, (2000.0, 2000.0, 1000.0), perturb=0.05,
                        seed=SEED_BASE + 1000 * 2)
        rho0, theta0 = reference_neutral(mesh.xyz[2])
        q = bubble_state(mesh, rho0, theta0, (1000.0, 1000.0, 350.0), 250.0, 0.5)
        q[1:4] = sinusoidal_velocity(mesh, SEED_BASE + 1000 * 2 + 1, 0.1)
        return Workload("cfg2_bubble_%dx%dx%d_N%d" % (nx, nx, nz, N), mesh,
                        np.stack((rho0, theta0)), q, dt=0.01, n_steps=1000, config=2)
    if config == 3:
        N = 4 if N is None else N
        nx = max(2, int(round(100 * scale)))
        return _tc_workload(3, "cfg3_tc_%dx%dx20_N%d" % (nx, nx, N), N, nx, nx, 20,
                            dt=0.1, n_steps=200)
    if config == 4:
        N = 4 if N is None else N
        if literal:
            nxy, nz = CFG4_LITERAL[N]
            nx = max(2, int(round(nxy * scale)))
            return _tc_workload(4, "cfg4_literal_%dx%dx%d_N%d" % (nx, nx, nz, N), N, nx, nx, nz,
                                dt=CFG4_DT[N], n_steps=20)
        nx = max(2, int(round(CFG4_NXY[N] * scale)))
        return _tc_workload(4, "cfg4_sweep_%dx%dx20_N%d" % (nx, nx, N), N, nx, nx, 20,
                            dt=CFG4_DT[N], n_steps=20)
    if config == 5:
        N = 7 if N is None else N
        nx = max(2, int(round(160 * scale)))
        return _tc_workload(5, "cfg5_tc_%dx%dx24_N%d" % (nx, nx, N), N, nx, nx, 24,
                            dt=0.025, n_steps=50)
    raise ValueError("config must be 1..5")
