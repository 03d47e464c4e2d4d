"""ORACLE (test infrastructure, not the product).  Problem families of BASELINE.json as plain
parametric NLPs  min f(x,theta) s.t. c(x,theta)=0, x_L<x<x_U  (eqs 1a-1c), with general
inequalities turned into equalities by slack variables.

Everything is DENSE and written for readability: c is a vector of length m, A = dc/dx an m-by-n array,
W = sigma_f*Hess f + sum_j y_j Hess c_j an n-by-n array (notation of PAPER.md:90).  Dynamics derivatives
come from running the ODE formula on second-order jets (oracle/jets.py); nothing here is shared with
the CUDA path.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline/reference legs may
import this package.

Decision vector, stage order (same layout the C ABI documents in include/jipm.h):
    x = [ x_0 | u_0 x_1 s_1 | ... | u_{N-1} x_N s_N ],   c = [ x_0 - xhat0 | dyn_1 g_1 | ... | dyn_N g_N ]
    dyn_k = x_k - F(x_{k-1},u_{k-1}),   g_k = h(x_k) - s_k  (h >= 0 are the obstacle / separation inequalities)
Quadrotor model: SURVEY.md Appendix C (12 states: p, ZYX Euler (phi,theta,psi), world velocity v, body rates w).
Family 4 is the paper's own vehicle: 13 states (p, quaternion q, BODY velocity v, body rates w), four
rotor speeds as inputs; the paper gives no parameters, the ones used are DESIGN.md reading N3.
"""
from __future__ import annotations

import numpy as np

from .jets import Jet

FAM_POINTMASS2D, FAM_QUAD_TRACK, FAM_MULTIQUAD, FAM_QUAD_CLUTTER, FAM_QUAT_NAV = 0, 1, 2, 3, 4

G_ACC = 9.81
MASS = 1.0
ARM = 0.2
JX, JY, JZ = 0.01, 0.01, 0.02
KTAU = 0.02
REF_SPEED = 1.5
SEP2 = 0.25  # 0.5 m minimum separation, squared


def _sin(a):
    return a.sin() if isinstance(a, Jet) else np.sin(a)


def _cos(a):
    return a.cos() if isinstance(a, Jet) else np.cos(a)


def quad_ode(x, u):
    """Continuous-time rigid-body quadrotor, xdot = f(x,u).  x: 12 scalars (arrays or jets), u: 4."""
    ph, th, ps = x[3], x[4], x[5]
    vx, vy, vz = x[6], x[7], x[8]
    wp, wq, wr = x[9], x[10], x[11]
    sph, cph, sth, cth, sps, cps = _sin(ph), _cos(ph), _sin(th), _cos(th), _sin(ps), _cos(ps)
    T = u[0] + u[1] + u[2] + u[3]
    tan_th = sth / cth
    qr = wq * sph + wr * cph
    dph = wp + qr * tan_th
    dth = wq * cph - wr * sph
    dps = qr / cth
    a = T * (1.0 / MASS)
    dvx = a * (cps * sth * cph + sps * sph)
    dvy = a * (sps * sth * cph - cps * sph)
    dvz = a * (cth * cph) - G_ACC
    tx = ARM * (u[1] - u[3])
    ty = ARM * (u[2] - u[0])
    tz = KTAU * (u[0] - u[1] + u[2] - u[3])
    dwp = (tx - (JZ - JY) * wq * wr) * (1.0 / JX)
    dwq = (ty - (JX - JZ) * wr * wp) * (1.0 / JY)
    dwr = (tz - (JY - JX) * wp * wq) * (1.0 / JZ)
    return [vx, vy, vz, dph, dth, dps, dvx, dvy, dvz, dwp, dwq, dwr]


KF_ROTOR = 1.0      # thrust of rotor i = KF_ROTOR * u_i^2 (rotor speeds in units that make this 1)
KM_ROTOR = 0.02     # drag torque of rotor i = KM_ROTOR * u_i^2


def quat_ode(x, u):
    """13-state rigid body: p world position, q = (w, x, y, z) attitude (body -> world), v BODY linear
    velocity, w body angular velocity; u = four rotor speeds.
        pdot = R(q) v;  qdot = 1/2 q (x) (0, w);  vdot = -w x v + R(q)^T (0,0,-g) + (0,0,T/m);  wdot = J^-1 (tau - w x J w)."""
    qw, qx, qy, qz = x[3], x[4], x[5], x[6]
    vx, vy, vz = x[7], x[8], x[9]
    wx, wy, wz = x[10], x[11], x[12]
    # rotation matrix of the (unnormalised) quaternion, row by row
    r00, r01, r02 = 1.0 - 2.0 * (qy * qy + qz * qz), 2.0 * (qx * qy - qw * qz), 2.0 * (qx * qz + qw * qy)
    r10, r11, r12 = 2.0 * (qx * qy + qw * qz), 1.0 - 2.0 * (qx * qx + qz * qz), 2.0 * (qy * qz - qw * qx)
    r20, r21, r22 = 2.0 * (qx * qz - qw * qy), 2.0 * (qy * qz + qw * qx), 1.0 - 2.0 * (qx * qx + qy * qy)
    dp = [r00 * vx + r01 * vy + r02 * vz, r10 * vx + r11 * vy + r12 * vz, r20 * vx + r21 * vy + r22 * vz]
    dq = [(qx * wx + qy * wy + qz * wz) * (-0.5), (qw * wx + qy * wz - qz * wy) * 0.5,
          (qw * wy + qz * wx - qx * wz) * 0.5, (qw * wz + qx * wy - qy * wx) * 0.5]
    f = [KF_ROTOR * (ui * ui) for ui in u]
    T = f[0] + f[1] + f[2] + f[3]
    # gravity seen from the body: R^T (0, 0, -g) = -g * (third ROW of R)
    dv = [-(wy * vz - wz * vy) - G_ACC * r20, -(wz * vx - wx * vz) - G_ACC * r21,
          -(wx * vy - wy * vx) - G_ACC * r22 + T * (1.0 / MASS)]
    tx = ARM * (f[1] - f[3])
    ty = ARM * (f[2] - f[0])
    tz = (KM_ROTOR / KF_ROTOR) * (f[0] - f[1] + f[2] - f[3])
    dw = [(tx - (JZ - JY) * wy * wz) * (1.0 / JX), (ty - (JX - JZ) * wz * wx) * (1.0 / JY),
          (tz - (JY - JX) * wx * wy) * (1.0 / JZ)]
    return dp + dq + dv + dw


def rk4(ode, x, u, h):
    """One classical RK4 step with zero-order-hold input."""
    k1 = ode(x, u)
    k2 = ode([xi + (0.5 * h) * ki for xi, ki in zip(x, k1)], u)
    k3 = ode([xi + (0.5 * h) * ki for xi, ki in zip(x, k2)], u)
    k4 = ode([xi + h * ki for xi, ki in zip(x, k3)], u)
    return [xi + (h / 6.0) * (a + 2.0 * b + 2.0 * c + d) for xi, a, b, c, d in zip(x, k1, k2, k3, k4)]


def quad_rk4(x, u, h):
    return rk4(quad_ode, x, u, h)


class Problem:
    """One family with fixed dimensions; theta is passed to every call."""

    def __init__(self, family: int, horizon_N: int, n_agents: int, n_obstacles: int, dt: float):
        self.family, self.N, self.na, self.nobs, self.dt = family, horizon_N, n_agents, n_obstacles, dt
        self.ax, self.au = (4, 2) if family == FAM_POINTMASS2D else ((13, 4) if family == FAM_QUAT_NAV else (12, 4))
        self.ode = quat_ode if family == FAM_QUAT_NAV else quad_ode
        if family == FAM_POINTMASS2D:
            self.nx, self.nu, self.pdim, self.ru = 4, 2, 2, 0.1
        else:
            self.nx, self.nu, self.pdim, self.ru = self.ax * n_agents, self.au * n_agents, 3, 0.01
        self.ng = n_agents * (n_agents - 1) // 2 if family == FAM_MULTIQUAD else n_obstacles
        N = self.N
        self.blk = self.nu + self.nx + self.ng
        self.n = (N + 1) * self.nx + N * self.nu + N * self.ng
        self.m = (N + 1) * self.nx + N * self.ng
        self.pairs = [(i, j) for i in range(n_agents) for j in range(i + 1, n_agents)]

    # ---- layout --------------------------------------------------------------------------------
    def ix(self, k):
        return 0 if k == 0 else self.nx + (k - 1) * self.blk + self.nu

    def iu(self, k):
        return self.nx + k * self.blk

    def islack(self, k):
        return self.nx + (k - 1) * self.blk + self.nu + self.nx

    def ic_dyn(self, k):
        return 0 if k == 0 else self.nx + (k - 1) * (self.nx + self.ng)

    def ic_g(self, k):
        return self.ic_dyn(k) + self.nx

    def bounds(self):
        xL, xU = np.full(self.n, -np.inf), np.full(self.n, np.inf)
        lo, hi = (-1.0, 1.0) if self.family == FAM_POINTMASS2D else (0.0, MASS * G_ACC / 2.0)
        if self.family == FAM_QUAT_NAV:   # rotor speeds: thrust per rotor KF u^2 <= m g / 2
            hi = float(np.sqrt(MASS * G_ACC / 2.0 / KF_ROTOR))
        for k in range(self.N):
            xL[self.iu(k):self.iu(k) + self.nu] = lo
            xU[self.iu(k):self.iu(k) + self.nu] = hi
        for k in range(1, self.N + 1):
            xL[self.islack(k):self.islack(k) + self.ng] = 0.0
        return xL, xU

    # ---- parameters ----------------------------------------------------------------------------
    def xhat0(self, th):
        return th[:self.nx]

    def target(self, th, k, agent=0):
        """Position the cost pulls knot k (of one agent) towards."""
        if self.family == FAM_POINTMASS2D:
            return th[4:6]
        if self.family == FAM_QUAD_TRACK:
            rho, phase = th[12], th[13]
            ang = phase + REF_SPEED * (k * self.dt) / rho
            return np.array([rho * np.cos(ang), rho * np.sin(ang), 0.0])
        if self.family == FAM_MULTIQUAD:
            o = 12 * self.na + 3 * agent
            return th[o:o + 3]
        if self.family == FAM_QUAT_NAV:
            return th[13:16]
        return th[12:15]

    def obstacle(self, th, j):
        if self.family == FAM_POINTMASS2D:
            o = 6 + 3 * j
            return th[o:o + 2], th[o + 2]
        o = {FAM_QUAD_TRACK: 14, FAM_QUAD_CLUTTER: 15, FAM_QUAT_NAV: 16}[self.family] + 4 * j
        return th[o:o + 3], th[o + 3]

    def pos_index(self, k, agent=0):
        """Index in x of the position of one agent at knot k."""
        return self.ix(k) + (self.ax * agent if self.family != FAM_POINTMASS2D else 0)

    # ---- objective (quadratic) -----------------------------------------------------------------
    def f(self, x, th):
        val = 0.0
        for k in range(self.N + 1):
            for a in range(self.na):
                i = self.pos_index(k, a)
                d = x[i:i + self.pdim] - self.target(th, k, a)
                val += float(d @ d)
        for k in range(self.N):
            u = x[self.iu(k):self.iu(k) + self.nu]
            val += self.ru * float(u @ u)
        return val

    def grad_f(self, x, th):
        g = np.zeros(self.n)
        for k in range(self.N + 1):
            for a in range(self.na):
                i = self.pos_index(k, a)
                g[i:i + self.pdim] = 2.0 * (x[i:i + self.pdim] - self.target(th, k, a))
        for k in range(self.N):
            i = self.iu(k)
            g[i:i + self.nu] = 2.0 * self.ru * x[i:i + self.nu]
        return g

    def hess_f(self):
        h = np.zeros(self.n)
        for k in range(self.N + 1):
            for a in range(self.na):
                i = self.pos_index(k, a)
                h[i:i + self.pdim] = 2.0
        for k in range(self.N):
            h[self.iu(k):self.iu(k) + self.nu] = 2.0 * self.ru
        return np.diag(h)

    # ---- dynamics ------------------------------------------------------------------------------
    def _stack_xu(self, x):
        """[N, nx+nu] rows (x_k, u_k), k = 0..N-1."""
        return np.array([np.concatenate([x[self.ix(k):self.ix(k) + self.nx],
                                         x[self.iu(k):self.iu(k) + self.nu]]) for k in range(self.N)])

    def dynamics(self, x, order=0):
        """F(x_k,u_k) for k=0..N-1: values [N,nx]; order>=1 also Jacobians [N,nx,nx+nu]; order 2 also
        Hessians [N,nx,nx+nu,nx+nu]."""
        Z = self._stack_xu(x)
        N, nx, nu, h = self.N, self.nx, self.nu, self.dt
        if self.family == FAM_POINTMASS2D:
            # exact zero-order hold of the double integrator: p+ = p + h v + h^2/2 u, v+ = v + h u
            J = np.zeros((nx, nx + nu))
            J[:, :nx] = np.eye(4)
            J[0, 2] = J[1, 3] = h
            J[0, 4] = J[1, 5] = 0.5 * h * h
            J[2, 4] = J[3, 5] = h
            F = Z @ J.T
            if order == 0:
                return F
            Jac = np.broadcast_to(J, (N, nx, nx + nu)).copy()
            return (F, Jac) if order == 1 else (F, Jac, np.zeros((N, nx, nx + nu, nx + nu)))
        F = np.zeros((N, nx))
        Jac = np.zeros((N, nx, nx + nu))
        Hes = np.zeros((N, nx, nx + nu, nx + nu))
        ax, au = self.ax, self.au
        for a in range(self.na):
            cols = list(range(ax * a, ax * a + ax)) + list(range(nx + au * a, nx + au * a + au))
            za = Z[:, cols]
            if order == 0:
                out = rk4(self.ode, [za[:, i] for i in range(ax)], [za[:, ax + i] for i in range(au)], h)
                F[:, ax * a:ax * a + ax] = np.stack(out, axis=1)
                continue
            v = Jet.variables(za)
            out = rk4(self.ode, v[:ax], v[ax:], h)
            for i, o in enumerate(out):
                F[:, ax * a + i] = o.v
                Jac[:, ax * a + i, cols] = o.g
                if order == 2:
                    Hes[np.ix_(range(N), [ax * a + i], cols, cols)] = o.H[:, None, :, :]
        if order == 0:
            return F
        return (F, Jac) if order == 1 else (F, Jac, Hes)

    # ---- inequalities h(x_k) >= 0 -----------------------------------------------------------------
    def ineq(self, x, th, k):
        """Values h [ng], list of (positions index list, gradient pieces) for knot k (1..N)."""
        out = np.zeros(self.ng)
        if self.family == FAM_MULTIQUAD:
            for q, (i, j) in enumerate(self.pairs):
                pi, pj = self.pos_index(k, i), self.pos_index(k, j)
                d = x[pi:pi + 3] - x[pj:pj + 3]
                out[q] = float(d @ d) - SEP2
        else:
            p0 = self.pos_index(k)
            for j in range(self.nobs):
                c, r = self.obstacle(th, j)
                d = x[p0:p0 + self.pdim] - c
                out[j] = float(d @ d) - r * r
        return out

    # ---- constraints ---------------------------------------------------------------------------
    def c(self, x, th):
        cv = np.zeros(self.m)
        cv[0:self.nx] = x[0:self.nx] - self.xhat0(th)
        F = self.dynamics(x, 0)
        for k in range(1, self.N + 1):
            cv[self.ic_dyn(k):self.ic_dyn(k) + self.nx] = x[self.ix(k):self.ix(k) + self.nx] - F[k - 1]
            s = x[self.islack(k):self.islack(k) + self.ng]
            cv[self.ic_g(k):self.ic_g(k) + self.ng] = self.ineq(x, th, k) - s
        return cv

    def jac(self, x, th):
        A = np.zeros((self.m, self.n))
        nx, nu, pd = self.nx, self.nu, self.pdim
        A[0:nx, 0:nx] = np.eye(nx)
        _, J = self.dynamics(x, 1)
        for k in range(1, self.N + 1):
            r = self.ic_dyn(k)
            A[r:r + nx, self.ix(k):self.ix(k) + nx] = np.eye(nx)
            A[r:r + nx, self.ix(k - 1):self.ix(k - 1) + nx] = -J[k - 1][:, :nx]
            A[r:r + nx, self.iu(k - 1):self.iu(k - 1) + nu] = -J[k - 1][:, nx:]
            rg = self.ic_g(k)
            for q in range(self.ng):
                A[rg + q, self.islack(k) + q] = -1.0
                if self.family == FAM_MULTIQUAD:
                    i, j = self.pairs[q]
                    pi, pj = self.pos_index(k, i), self.pos_index(k, j)
                    d = x[pi:pi + 3] - x[pj:pj + 3]
                    A[rg + q, pi:pi + 3] = 2.0 * d
                    A[rg + q, pj:pj + 3] = -2.0 * d
                else:
                    c, _ = self.obstacle(th, q)
                    p0 = self.pos_index(k)
                    A[rg + q, p0:p0 + pd] = 2.0 * (x[p0:p0 + pd] - c)
        return A

    def hess_lag(self, x, th, y, sigma_f=1.0):
        """W = sigma_f Hess f + sum_j y_j Hess c_j."""
        W = sigma_f * self.hess_f()
        nx, nu, pd = self.nx, self.nu, self.pdim
        if self.family != FAM_POINTMASS2D:
            _, _, H = self.dynamics(x, 2)
            for k in range(1, self.N + 1):
                lam = y[self.ic_dyn(k):self.ic_dyn(k) + nx]
                Hk = -np.tensordot(lam, H[k - 1], axes=(0, 0))  # dyn_k = x_k - F(...)
                ia, ib = self.ix(k - 1), self.iu(k - 1)
                W[ia:ia + nx, ia:ia + nx] += Hk[:nx, :nx]
                W[ia:ia + nx, ib:ib + nu] += Hk[:nx, nx:]
                W[ib:ib + nu, ia:ia + nx] += Hk[nx:, :nx]
                W[ib:ib + nu, ib:ib + nu] += Hk[nx:, nx:]
        I = np.eye(pd)
        for k in range(1, self.N + 1):
            rg = self.ic_g(k)
            for q in range(self.ng):
                if self.family == FAM_MULTIQUAD:
                    i, j = self.pairs[q]
                    pi, pj = self.pos_index(k, i), self.pos_index(k, j)
                    W[pi:pi + 3, pi:pi + 3] += 2.0 * y[rg + q] * I
                    W[pj:pj + 3, pj:pj + 3] += 2.0 * y[rg + q] * I
                    W[pi:pi + 3, pj:pj + 3] -= 2.0 * y[rg + q] * I
                    W[pj:pj + 3, pi:pi + 3] -= 2.0 * y[rg + q] * I
                else:
                    p0 = self.pos_index(k)
                    W[p0:p0 + pd, p0:p0 + pd] += 2.0 * y[rg + q] * I
        return W

    def init_slacks(self, x, th):
        """Step I-2: s_k <- h(x_k) so that the slack-defining equalities hold at x0."""
        x = x.copy()
        for k in range(1, self.N + 1):
            x[self.islack(k):self.islack(k) + self.ng] = self.ineq(x, th, k)
        return x
