"""Pins for oracle/families.py and oracle/jets.py: every derivative function against central finite
differences of the function it differentiates (SURVEY.md 8(c) "Derivatives"), the jets against a
closed-form example, the RK4 step against a tiny-step reference integration, and hover as a fixed point."""
import numpy as np
import pytest

from oracle import families as fam
from oracle.jets import Jet
from paper_2606_26341_b200 import workloads as wl
from helpers import fd_grad, fd_jac

CASES = [(0, {}), (1, dict(horizon_N=3)), (2, dict(horizon_N=2, n_agents=2)), (3, dict(horizon_N=3, n_obstacles=4)),
         (5, dict(horizon_N=3))]


def make(cfg, kw, P=2):
    d = wl.config_dims(cfg, **kw)
    d, th, x0 = wl.generate(cfg, P, d)
    p = fam.Problem(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt)
    return d, p, th, x0


def test_jet_closed_form():
    # h(a,b) = sin(a)*b/cos(b) + a*a ; derivatives by hand
    z = np.array([[0.3, -0.7], [1.1, 0.4]])
    a, b = Jet.variables(z)
    h = a.sin() * b / b.cos() + a * a
    A, B = z[:, 0], z[:, 1]
    np.testing.assert_allclose(h.v, np.sin(A) * B / np.cos(B) + A * A, rtol=1e-14)
    ha = np.cos(A) * B / np.cos(B) + 2 * A
    q = 1 / np.cos(B) + B * np.sin(B) / np.cos(B) ** 2          # d/db (b / cos b)
    hb = np.sin(A) * q
    np.testing.assert_allclose(h.g, np.stack([ha, hb], 1), rtol=1e-13)
    haa = -np.sin(A) * B / np.cos(B) + 2
    hab = np.cos(A) * q
    qb = 2 * np.sin(B) / np.cos(B) ** 2 + B * (np.cos(B) ** 2 + 2 * np.sin(B) ** 2) / np.cos(B) ** 3
    hbb = np.sin(A) * qb
    np.testing.assert_allclose(h.H[:, 0, 0], haa, rtol=1e-13)
    np.testing.assert_allclose(h.H[:, 0, 1], hab, rtol=1e-13)
    np.testing.assert_allclose(h.H[:, 1, 0], hab, rtol=1e-13)
    np.testing.assert_allclose(h.H[:, 1, 1], hbb, rtol=1e-12)


def test_quad_hover_is_equilibrium_and_free_fall():
    x = [np.array([v]) for v in [1.0, 2.0, 3.0, 0, 0, 0.7, 0, 0, 0, 0, 0, 0]]
    hover = [np.array([fam.MASS * fam.G_ACC / 4])] * 4
    xd = fam.quad_ode(x, hover)
    assert max(abs(float(np.ravel(v)[0])) for v in xd) < 1e-14
    # zero thrust: p_z(t) = -g t^2/2 exactly for RK4 (quadratic in t)
    zero = [np.array([0.0])] * 4
    x1 = fam.quad_rk4(x, zero, 0.05)
    assert abs(float(x1[2][0]) - (3.0 - 0.5 * fam.G_ACC * 0.05 ** 2)) < 1e-14
    assert abs(float(x1[8][0]) + fam.G_ACC * 0.05) < 1e-14


def test_quad_yaw_torque_and_roll_axis():
    # pure roll torque (u2 > u4): wdot_p = l (u2-u4)/Jx ; thrust along body z rotates with roll
    x = [np.array([0.0])] * 12
    u = [np.array([1.0]), np.array([1.5]), np.array([1.0]), np.array([0.5])]
    xd = fam.quad_ode(x, u)
    assert abs(float(xd[9][0]) - fam.ARM * 1.0 / fam.JX) < 1e-12
    assert abs(float(xd[11][0])) < 1e-12 + abs(fam.KTAU * (1.0 - 1.5 + 1.0 - 0.5) / fam.JZ)
    x = [np.array([v]) for v in [0, 0, 0, 0.3, 0, 0, 0, 0, 0, 0, 0, 0]]   # roll 0.3: a_y = -T sin(phi)
    xd = fam.quad_ode(x, u)
    assert abs(float(xd[7][0]) + 4.0 * np.sin(0.3)) < 1e-12
    assert abs(float(xd[8][0]) - (4.0 * np.cos(0.3) - fam.G_ACC)) < 1e-12


def test_rk4_against_fine_integration():
    """One RK4 step vs a 400-substep reference: small error, and 4th-order global convergence (x16 per halving)."""
    rng = np.random.default_rng(0)
    x = rng.uniform(-0.3, 0.3, 12)
    u = rng.uniform(1.0, 4.0, 4)
    xs = [np.array([v]) for v in x]
    us = [np.array([v]) for v in u]

    def integrate(nsub, T=0.2):
        cur = xs
        for _ in range(nsub):
            cur = fam.quad_rk4(cur, us, T / nsub)
        return np.array([float(v[0]) for v in cur])

    fine = integrate(400)
    e1, e2, e4 = (np.max(np.abs(integrate(k) - fine)) for k in (1, 2, 4))
    assert e4 < 1e-4
    assert 8.0 < e1 / e2 < 40.0 and 8.0 < e2 / e4 < 40.0


@pytest.mark.parametrize("cfg,kw", CASES)
def test_gradient_jacobian_hessian_fd(cfg, kw):
    d, p, th, x0 = make(cfg, kw)
    rng = np.random.default_rng(cfg)
    x = x0[0] + rng.uniform(-0.1, 0.1, p.n)
    t = th[0]
    assert p.n == d.n and p.m == d.m
    g = p.grad_f(x, t)
    np.testing.assert_allclose(g, fd_grad(lambda v: p.f(v, t), x), rtol=1e-6, atol=1e-6)
    A = p.jac(x, t)
    np.testing.assert_allclose(A, fd_jac(lambda v: p.c(v, t), x), rtol=1e-6, atol=2e-7)
    y = rng.normal(size=p.m)
    W = p.hess_lag(x, t, y, 1.0)
    np.testing.assert_allclose(W, W.T, atol=1e-12)
    Wfd = fd_jac(lambda v: p.grad_f(v, t) + p.jac(v, t).T @ y, x, h=1e-5)
    np.testing.assert_allclose(W, Wfd, rtol=2e-5, atol=2e-6)
    W0 = p.hess_lag(x, t, y, 0.0)
    np.testing.assert_allclose(W - W0, p.hess_f(), atol=1e-12)


@pytest.mark.parametrize("cfg,kw", CASES)
def test_layout_matches_workloads(cfg, kw):
    d, p, th, x0 = make(cfg, kw)
    for k in range(d.horizon_N + 1):
        assert p.ix(k) == d.ix(k)
        assert p.ic_dyn(k) == d.ic_dyn(k)
    for k in range(d.horizon_N):
        assert p.iu(k) == d.iu(k)
    for k in range(1, d.horizon_N + 1):
        assert p.islack(k) == d.islack(k) and p.ic_g(k) == d.ic_g(k)
    xL, xU = p.bounds()
    wL, wU = wl.bounds(d)
    np.testing.assert_array_equal(xL, wL)
    np.testing.assert_array_equal(xU, wU)
    # stay-put initial guess satisfies the initial condition, slack init makes the slack rows vanish
    x = p.init_slacks(x0[0], th[0])
    c = p.c(x, th[0])
    assert np.max(np.abs(c[:p.nx])) == 0.0
    for k in range(1, p.N + 1):
        assert np.max(np.abs(c[p.ic_g(k):p.ic_g(k) + p.ng])) < 1e-12


def test_quat_ode_against_rotation_library_and_cross_products():
    """The 13-state vehicle of PAPER.md:174 (family 4) against an independent statement: R(q) from
    scipy.spatial.transform.Rotation; pdot = R v_body; vdot = -w x v + R^T (0,0,-g) + (0,0,T/m) with numpy.cross;
    wdot = J^-1 (tau - w x J w); and the quaternion kinematics through the rotation it generates:
    R(q + eps qdot) = R(q) (I + eps [w]x) + O(eps^2) for a unit quaternion."""
    from scipy.spatial.transform import Rotation
    rng = np.random.default_rng(3)
    for _ in range(10):
        q = rng.normal(size=4)
        q /= np.linalg.norm(q)
        x = np.concatenate([rng.uniform(-1, 1, 3), q, rng.uniform(-2, 2, 3), rng.uniform(-3, 3, 3)])
        u = rng.uniform(0.3, 2.0, 4)
        got = np.array(fam.quat_ode(list(x), list(u)), dtype=float)
        R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()      # scipy order: (x, y, z, w)
        v, w = x[7:10], x[10:13]
        f = u ** 2
        T = f.sum()
        Jm = np.diag([0.01, 0.01, 0.02])
        tau = np.array([0.2 * (f[1] - f[3]), 0.2 * (f[2] - f[0]), 0.02 * (f[0] - f[1] + f[2] - f[3])])
        np.testing.assert_allclose(got[0:3], R @ v, rtol=1e-12, atol=1e-12)
        np.testing.assert_allclose(got[7:10], -np.cross(w, v) + R.T @ np.array([0, 0, -9.81]) + np.array([0, 0, T]), rtol=1e-12,
                                   atol=1e-12)
        np.testing.assert_allclose(got[10:13], np.linalg.solve(Jm, tau - np.cross(w, Jm @ w)), rtol=1e-12, atol=1e-12)
        eps = 1e-6
        q2 = q + eps * got[3:7]
        R2 = Rotation.from_quat([q2[1], q2[2], q2[3], q2[0]]).as_matrix()
        wx = np.array([[0, -w[2], w[1]], [w[2], 0, -w[0]], [-w[1], w[0], 0]])
        np.testing.assert_allclose(R2, R @ (np.eye(3) + eps * wx), atol=5e-11)
    # hover: level, at rest, rotor speed sqrt(m g / 4): an equilibrium
    xh = np.array([1.0, 2.0, 3.0, 1, 0, 0, 0, 0, 0, 0, 0, 0, 0])
    assert np.max(np.abs(fam.quat_ode(list(xh), [np.sqrt(9.81 / 4)] * 4))) < 1e-14
