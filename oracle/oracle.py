"""ctypes front end of the CPU FP64 oracle (oracle/numa_oracle.c).

TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` leg may import this.  It imports nothing from the product package
``paper_2504_08157_b200`` and shares no code with the CUDA path.

`Oracle` strings the C functions together in the order of SURVEY.md 8(a) / DESIGN.md:
A0 setup -> (A2-A6 tendency + weight) -> A7 DSS -> A8 sources -> A9 walls -> A10 RK stage,
A11 = SSP-RK3 (Shu-Osher) driver (reading Q11).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "numa_oracle.c")
_LIB = os.path.join(_HERE, "libnuma_oracle.so")

# SSP-RK3 (Shu-Osher) as (a0, a1, b):  q_out = a0 q0 + a1 qs + b dt L(qs)
SSP_RK3 = ((1.0, 0.0, 1.0), (0.75, 0.25, 0.25), (1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0))

# ARK2 of Giraldo, Kelly & Constantinescu 2013 ("the second-order additive
# Runge-Kutta (ARK2) scheme proposed in (Giraldo et al. 2013)"; the paper does not print the
# tableau: reading Q35 of DESIGN.md).  Three stages, gamma = 1 - 1/sqrt(2); explicit A, implicit
# At (singly diagonally implicit, first stage explicit), b shared.  Pinned by the order conditions
# and by measured second-order convergence (tests/test_oracle_imex.py).
_G = 1.0 - 1.0 / np.sqrt(2.0)
_A32 = (3.0 + 2.0 * np.sqrt(2.0)) / 6.0
_B = 1.0 / (2.0 * np.sqrt(2.0))
ARK2_A = ((0.0, 0.0, 0.0), (2.0 * _G, 0.0, 0.0), (1.0 - _A32, _A32, 0.0))
ARK2_AT = ((0.0, 0.0, 0.0), (_G, _G, 0.0), (_B, _B, _G))
ARK2_B = (_B, _B, _G)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, OpenMP over elements, no FP contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-std=c99", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None
_dp = C.POINTER(C.c_double)


def _p(a, typ=C.c_double):
    if a is None:
        return None
    return a.ctypes.data_as(C.POINTER(typ))


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_lgl.argtypes = [C.c_int, _dp, _dp]
        L.orc_dmat.argtypes = [C.c_int, _dp, _dp]
        L.orc_metrics.argtypes = [C.c_int, C.c_long, _dp, _dp, _dp]
        L.orc_metrics.restype = C.c_long
        L.orc_mass.argtypes = [C.c_int, C.c_long, C.c_long, C.POINTER(C.c_int32), _dp, _dp, _dp, _dp]
        L.orc_wall_list.argtypes = [C.c_int, C.c_long, C.POINTER(C.c_uint8), _dp,
                                    C.POINTER(C.c_int64), _dp]
        L.orc_wall_list.restype = C.c_long
        L.orc_tendency.argtypes = [C.c_int, C.c_long, _dp, _dp, _dp, _dp, _dp, _dp]
        L.orc_weight.argtypes = [C.c_long, C.c_int, _dp, _dp, _dp]
        L.orc_dss.argtypes = [C.c_long, C.c_long, C.c_int, C.POINTER(C.c_int32), _dp]
        L.orc_sources.argtypes = [C.c_long, _dp, _dp, _dp, C.c_double, _dp]
        L.orc_walls.argtypes = [C.c_long, C.c_long, C.POINTER(C.c_int64), _dp, _dp]
        L.orc_rk_stage.argtypes = [C.c_long, C.c_double, C.c_double, C.c_double, _dp, _dp, _dp, _dp]
        L.orc_hd_laplacian.argtypes = [C.c_int, C.c_long, C.c_int, _dp, _dp, _dp, _dp]
        L.orc_linear_tendency.argtypes = [C.c_int, C.c_long, _dp, _dp, _dp, _dp, _dp]
        _ip = C.POINTER(C.c_int32)
        L.orc_ri_area.argtypes = [C.c_int, C.c_long, _dp, _dp]
        L.orc_ri_velocity.argtypes = [C.c_long, C.c_long, _ip, _ip, C.c_int, C.c_int, C.c_double,
                                      _dp, _dp, _dp, _dp, _ip, _dp, _ip, _dp]
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def lgl(N):
    xi = np.empty(N + 1); w = np.empty(N + 1)
    lib().orc_lgl(N, _p(xi), _p(w))
    return xi, w


def dmat(N):
    xi, _ = lgl(N)
    D = np.empty((N + 1, N + 1))
    lib().orc_dmat(N, _p(xi), _p(D))
    return D


def metrics(N, xyz):
    xyz = _f64(xyz)
    Ne = xyz.shape[1]
    met = np.empty((9,) + xyz.shape[1:])
    jac = np.empty(xyz.shape[1:])
    bad = lib().orc_metrics(N, Ne, _p(xyz), _p(met), _p(jac))
    return met, jac, int(bad)


def mass(N, intma_cg, n_global, jac):
    intma_cg = np.ascontiguousarray(intma_cg, dtype=np.int32)
    Ne = intma_cg.shape[0]
    wJ = np.empty(jac.shape); M = np.empty(n_global); om = np.empty(jac.shape)
    lib().orc_mass(N, Ne, n_global, _p(intma_cg, C.c_int32), _p(_f64(jac)), _p(wJ), _p(M), _p(om))
    return wJ, M, om


def wall_list(N, face_bc, met):
    face_bc = np.ascontiguousarray(face_bc, dtype=np.uint8)
    Ne = face_bc.shape[0]
    cnt = lib().orc_wall_list(N, Ne, _p(face_bc, C.c_uint8), _p(met), None, None)
    node = np.empty(cnt, dtype=np.int64); nrm = np.empty((cnt, 3))
    if cnt:
        lib().orc_wall_list(N, Ne, _p(face_bc, C.c_uint8), _p(met), _p(node, C.c_int64), _p(nrm))
    return node, nrm


def tendency(N, par, q, ref, met, want_T=False):
    q = _f64(q); ref = _f64(ref)
    Ne = q.shape[1]
    S = np.empty_like(q)
    T = np.empty_like(q) if want_T else None
    par = _f64(par)
    lib().orc_tendency(N, Ne, _p(par), _p(q), _p(ref), _p(met), _p(S), _p(T))
    return (S, T) if want_T else S


def weight(omega, S):
    r = np.empty_like(S)
    lib().orc_weight(omega.size, S.shape[0], _p(omega), _p(_f64(S)), _p(r))
    return r


def dss(intma_cg, n_global, r):
    """In place on r[nf][Ne][Mn]."""
    assert r.flags.c_contiguous and r.dtype == np.float64
    intma_cg = np.ascontiguousarray(intma_cg, dtype=np.int32)
    lib().orc_dss(intma_cg.size, n_global, r.shape[0], _p(intma_cg, C.c_int32), _p(r))
    return r


def sources(q, heat, beta, f_cor, r):
    assert r.flags.c_contiguous
    NL = q[0].size
    lib().orc_sources(NL, _p(_f64(q)), _p(None if heat is None else _f64(heat)),
                      _p(None if beta is None else _f64(beta)), float(f_cor), _p(r))
    return r


def walls(node, nrm, r):
    assert r.flags.c_contiguous
    NL = r[0].size
    lib().orc_walls(NL, node.size, _p(node, C.c_int64), _p(nrm), _p(r))
    return r


def rk_stage(a0, a1, b_dt, q0, qs, r, out=None):
    if out is None:
        out = np.empty_like(q0)
    lib().orc_rk_stage(q0.size, a0, a1, b_dt, _p(q0), _p(qs), _p(r), _p(out))
    return out


def linear_tendency(N, par, q, ref, met):
    """Element-local linear operator L_loc(q) of the IMEX splitting (Eq. 13; reading Q34)."""
    q = _f64(q)
    out = np.empty_like(q)
    lib().orc_linear_tendency(N, q.shape[1], _p(_f64(par)), _p(q), _p(_f64(ref)), _p(met), _p(out))
    return out


def gmres(apply_A, b, x0, dot, tol, m, max_restarts):
    """Restarted GMRES(m) of Saad & Schultz 1986, written out: Arnoldi with
    modified Gram-Schmidt, Givens rotations on the Hessenberg matrix, no preconditioner.
    Stops when ||r|| <= tol ||b|| (residual norm from the rotated right-hand side).
    Returns (x, inner iterations, relative residual estimate)."""
    x = x0.copy()
    bnorm = np.sqrt(dot(b, b))
    if bnorm == 0.0:
        return np.zeros_like(b), 0, 0.0
    its = 0
    rel = np.inf
    for _ in range(max_restarts + 1):
        r = b - apply_A(x)
        beta = np.sqrt(dot(r, r))
        rel = beta / bnorm
        if rel <= tol:
            break
        V = [r / beta]
        H = np.zeros((m + 1, m))
        cs = np.zeros(m); sn = np.zeros(m)
        g = np.zeros(m + 1); g[0] = beta
        k_used = 0
        for k in range(m):
            w = apply_A(V[k])
            for i in range(k + 1):
                H[i, k] = dot(w, V[i])
                w = w - H[i, k] * V[i]
            hn = np.sqrt(dot(w, w))
            H[k + 1, k] = hn
            for i in range(k):
                t = cs[i] * H[i, k] + sn[i] * H[i + 1, k]
                H[i + 1, k] = -sn[i] * H[i, k] + cs[i] * H[i + 1, k]
                H[i, k] = t
            d = np.hypot(H[k, k], H[k + 1, k])
            cs[k] = H[k, k] / d; sn[k] = H[k + 1, k] / d
            H[k, k] = d; H[k + 1, k] = 0.0
            g[k + 1] = -sn[k] * g[k]; g[k] = cs[k] * g[k]
            its += 1
            k_used = k + 1
            rel = abs(g[k + 1]) / bnorm
            if rel <= tol or d == 0.0:
                break
            V.append(w / hn)
        y = np.zeros(k_used)
        for i in range(k_used - 1, -1, -1):
            y[i] = (g[i] - H[i, i + 1:k_used] @ y[i + 1:]) / H[i, i]
        for i in range(k_used):
            x = x + y[i] * V[i]
        if rel <= tol:
            break
    return x, its, rel


def hd_tau(met, c, dt):
    """Viscosity tensor of the hyper-diffusion (Eq. 15-16) at every local
    node, from the metric terms met[9][Ne][Mn] (row a = grad xi_a, i.e. the matrix J^-1):
        G = J^-1 J^-T (L149);  eigenvalues of G ascending = (1/lambda_1, 1/lambda_2, 1/lambda_3),
        E = eigenvectors in columns (LAPACK dsyevd through numpy.linalg.eigh: the library step);
        nu_i = c_i^(1/alpha) dx_i^2 / dt^(1/alpha), alpha = 2 (Eq. 16), with the element size in
        the i-th principal direction taken as dx_i = 2 lambda_i^(1/2) (reading Q31: the
        reference element [-1,1] has length 2, so an axis-aligned brick gets dx_i = h_i);
        tau = J E diag(nu_i / lambda_i) (J E)^T (Eq. 15).
    Returns tau[6][Ne][Mn] = (xx, xy, xz, yy, yz, zz)."""
    met = _f64(met)
    shp = met.shape[1:]
    Jinv = np.moveaxis(met.reshape(3, 3, -1), 2, 0)          # [node][a][c] = d xi_a / d x_c
    J = np.linalg.inv(Jinv)                                   # d x_c / d xi_a  ([node][c][a])
    G = Jinv @ np.swapaxes(Jinv, 1, 2)                        # J^-1 J^-T
    ev, E = np.linalg.eigh(G)                                 # ascending eigenvalues 1/lambda_i
    lam = 1.0 / ev
    dx = 2.0 * np.sqrt(lam)
    nu = np.sqrt(np.asarray(c, dtype=np.float64))[None, :] * dx ** 2 / np.sqrt(dt)
    JE = J @ E
    T = (JE * (nu / lam)[:, None, :]) @ np.swapaxes(JE, 1, 2)
    T = 0.5 * (T + np.swapaxes(T, 1, 2))
    out = np.stack([T[:, 0, 0], T[:, 0, 1], T[:, 0, 2], T[:, 1, 1], T[:, 1, 2], T[:, 2, 2]])
    return np.ascontiguousarray(out.reshape((6,) + shp))


def hd_laplacian(N, met, tau, f):
    """Element-local L f = div(tau grad f) for f[nf][Ne][Mn] (strong form, Q30)."""
    f = _f64(f)
    out = np.empty_like(f)
    lib().orc_hd_laplacian(N, f.shape[1], f.shape[0], _p(_f64(met)), _p(_f64(tau)), _p(f), _p(out))
    return out


def ri_area(N, xyz):
    """Horizontal quadrature weight a[Ne][Mn] of the RI diagnostic (Q26)."""
    xyz = _f64(xyz)
    a = np.empty(xyz.shape[1:])
    lib().orc_ri_area(N, xyz.shape[1], _p(xyz), _p(a))
    return a


def ri_velocity(N, xyz, intma_cg, n_global, level, n_lev, q, r_max, n_strip=50, area=None):
    """RI-velocity diagnostic (Eq. 18-22): dict with u_ri, umax_h, centroid[n_lev][2],
    valid[n_lev], ubar[n_lev][n_strip], count[n_lev][n_strip]."""
    xyz = _f64(xyz); q = _f64(q)
    intma_cg = np.ascontiguousarray(intma_cg, dtype=np.int32)
    level = np.ascontiguousarray(level, dtype=np.int32)
    a = ri_area(N, xyz) if area is None else _f64(area)
    cen = np.empty((n_lev, 2)); valid = np.empty(n_lev, dtype=np.int32)
    ubar = np.empty((n_lev, n_strip)); cnt = np.empty((n_lev, n_strip), dtype=np.int32)
    sc = np.empty(2)
    lib().orc_ri_velocity(intma_cg.size, int(n_global), _p(intma_cg, C.c_int32), _p(level, C.c_int32),
                          int(n_lev), int(n_strip), float(r_max), _p(xyz), _p(a), _p(q), _p(cen),
                          _p(valid, C.c_int32), _p(ubar), _p(cnt, C.c_int32), _p(sc))
    return dict(u_ri=float(sc[0]), umax_h=float(sc[1]), centroid=cen, valid=valid, ubar=ubar,
                count=cnt, area=a)


class Oracle:
    """A0 once, then rhs()/step_rk3() on element-local SoA arrays [m][Ne][Mn]."""

    def __init__(self, N, xyz, intma_cg, n_global, face_bc, ref, constants, f_cor=0.0,
                 sponge=None, hd_c=None, hd_dt=1.0):
        self.N = N
        self.intma_cg = np.ascontiguousarray(intma_cg, dtype=np.int32)
        self.n_global = int(n_global)
        self.ref = _f64(ref)
        self.par = np.array([constants["g"], constants["p_a"], constants["R_gas"],
                             constants["c_p"], constants["c_v"]], dtype=np.float64)
        self.f_cor = float(f_cor)
        self.sponge = None if sponge is None else _f64(sponge)
        self.met, self.jac, bad = metrics(N, xyz)
        if bad:
            raise ValueError("non-positive Jacobian at %d nodes" % bad)
        self.wJ, self.M, self.omega = mass(N, self.intma_cg, self.n_global, self.jac)
        self.wall_node, self.wall_normal = wall_list(N, face_bc, self.met)
        # NEXT-1: tensor hyper-diffusion (Eq. 14-16), off unless coefficients are given
        self.tau = None
        if hd_c is not None and any(float(x) != 0.0 for x in hd_c):
            self.tau = hd_tau(self.met, hd_c, hd_dt)

    @classmethod
    def from_workload(cls, wl, hd_c=None, hd_dt=1.0):
        m = wl.mesh
        return cls(m.N, m.xyz, m.intma_cg, m.n_global, m.face_bc, wl.ref, wl.constants,
                   f_cor=wl.f_cor, sponge=wl.sponge, hd_c=hd_c, hd_dt=hd_dt)

    def hyperdiffusion(self, q):
        """H_q = -L(L(q)) on u, v, w, theta' (Eq. 14 with alpha = 2; Eq. 1b-1c), L = M^-1 DSS(wJ
        div(tau grad .)) (Eq. 11-12): two applications with the assembly after each.  [4][Ne][Mn]."""
        f = np.ascontiguousarray(_f64(q)[1:5])
        l1 = weight(self.omega, hd_laplacian(self.N, self.met, self.tau, f))
        dss(self.intma_cg, self.n_global, l1)
        l2 = weight(self.omega, hd_laplacian(self.N, self.met, self.tau, l1))
        dss(self.intma_cg, self.n_global, l2)
        return -l2

    # --- the separate calls of the C-ABI boundary -------------------------------------
    def rhs_local(self, q, want_T=False):
        """numa_rhs: A2-A6, weighted element-local contributions (before DSS)."""
        out = tendency(self.N, self.par, q, self.ref, self.met, want_T)
        if want_T:
            S, T = out
            return weight(self.omega, S), weight(self.omega, T)
        return weight(self.omega, out)

    def dss(self, r):
        """numa_dss_or_flux (CG): A7, in place."""
        return dss(self.intma_cg, self.n_global, r)

    def apply_sources(self, q, heat, r):
        """numa_apply_sources: A8 (+ H_q of Eq. 1b-1c when enabled) then A9, in place."""
        sources(q, heat, self.sponge, self.f_cor, r)
        if self.tau is not None:
            r[1:5] += self.hyperdiffusion(q)
        walls(self.wall_node, self.wall_normal, r)
        return r

    def rhs(self, q, heat=None):
        """Full assembled tendency L(q) = walls(sources(DSS(omega * S(q))))."""
        r = self.rhs_local(q)
        self.dss(r)
        self.apply_sources(q, heat, r)
        return r

    # --- NEXT-3: IMEX (Eq. 13), ARK2 + matrix-free GMRES (L127-L137) --------------------------
    def linear(self, q):
        """L_h(q) = walls(DSS(omega * L_loc(q))): the linear operator assembled like S (Eq. 11-12),
        with the no-flux projection; no sources (they stay in the explicit part)."""
        r = weight(self.omega, linear_tendency(self.N, self.par, q, self.ref, self.met))
        self.dss(r)
        walls(self.wall_node, self.wall_normal, r)
        return r

    def dot(self, a, b):
        """Euclidean inner product over the unique global nodes (each local copy weighted by
        1 / multiplicity), all five fields: the inner product of the GMRES (reading Q36)."""
        if not hasattr(self, "_inv_mult"):
            cnt = np.bincount(self.intma_cg.reshape(-1), minlength=self.n_global)
            self._inv_mult = (1.0 / cnt[self.intma_cg]).reshape(1, *self.intma_cg.shape)
        return float(np.sum(self._inv_mult * a * b))

    def step_ark2(self, q, dt, heat=None, tol=1e-10, m=20, max_restarts=10, stats=None):
        """One IMEX ARK2 step (Eq. 13): explicit part N = S - L, implicit part L, stages
            Q_i = q + dt sum_{j<i} (a_ij N(Q_j) + at_ij L(Q_j)) + dt at_ii L(Q_i),
        the linear systems (I - dt at_ii L) Q_i = R_i solved by GMRES(m) from the initial guess R_i;
        q_new = q + dt sum b_i S(Q_i)."""
        q = _f64(q)
        Nq, Lq, Sq = [], [], []
        for i in range(3):
            R = q.copy()
            for j in range(i):
                R = R + dt * (ARK2_A[i][j] * Nq[j] + ARK2_AT[i][j] * Lq[j])
            aii = ARK2_AT[i][i]
            if aii == 0.0:
                Q = R
            else:
                Q, its, rel = gmres(lambda x: x - dt * aii * self.linear(x), R, R, self.dot, tol, m, max_restarts)
                if stats is not None:
                    stats.append((its, rel))
            S = self.rhs(Q, heat)
            L = self.linear(Q)
            Sq.append(S); Lq.append(L); Nq.append(S - L)
        out = q.copy()
        for i in range(3):
            out = out + dt * ARK2_B[i] * Sq[i]
        return out

    def step_rk3(self, q, dt, heat=None):
        """A11: one SSP-RK3 step (Q11)."""
        q0 = _f64(q)
        qs = q0
        for (a0, a1, b) in SSP_RK3:
            r = self.rhs(qs, heat)
            qs = rk_stage(a0, a1, b * dt, q0, qs, r)
        return qs
