"""Pins for oracle/ipm.py against closed forms, textbook special cases, brute force and an independent
library (SURVEY.md section 8(c) "What pins the oracle").  None of these re-types the oracle's own formula."""
import math
import os

import numpy as np
import pytest

from oracle import ipm
from oracle import families as fam
from paper_2606_26341_b200 import workloads as wl
from helpers import SmallNLP

INF = np.inf
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def golden_mu():
    rows = [l.split() for l in open(os.path.join(GOLD, "mu_schedule.txt")) if l.strip() and not l.startswith("#")]
    return np.array([[float(a), float(b)] for a, b in rows])


def test_one_dim_barrier_trajectory_and_mu_schedule():
    """min x s.t. x >= 0 from x0 = 0.5, z0 = 1, no damping, no bound relaxation.  By (6)-(7): Sigma = z/x,
    Newton gives x+ = mu/z with z == 1, so x_k equals the barrier parameter of iteration k; mu follows the
    golden schedule two steps at a time (the update loop fires twice while E_mu <= 10 mu);
    SOLVED in 4 iterations.  First step: Sigma = 2, grad phi = 0.96, dx = -0.48, dz = 0."""
    p = SmallNLP(1, 0, lambda x: x[0], lambda x: [1.0], lambda x: [[0.0]])
    o = ipm.Options(kappa_d=0.0, bound_relax_factor=0.0)
    s = ipm.Solver(p, [0.0], [INF], o)
    st = s.initialise([0.5], None)
    assert st.x[0] == 0.5 and st.zL[0] == 1.0 and st.mu == 0.1
    g = golden_mu()
    expect_mu = [g[1, 0], g[3, 0], g[4, 0], g[5, 0]]
    tr = s.iterate(st, None)
    np.testing.assert_allclose(tr["step"][0], [-0.48], rtol=1e-12)
    np.testing.assert_allclose(tr["step"][2], [0.0], atol=1e-12)
    assert tr["alpha"] == 1.0 and tr["alpha_z"] == 1.0
    xs, mus = [st.x[0]], [st.mu]
    while st.status == ipm.ST_NOT_RUN:
        s.iterate(st, None)
        if st.status == ipm.ST_NOT_RUN:
            xs.append(st.x[0])
            mus.append(st.mu)
    assert st.status == ipm.ST_SOLVED and st.k == 4
    np.testing.assert_allclose(mus, expect_mu, rtol=2e-6)
    np.testing.assert_allclose(xs, expect_mu, rtol=2e-6)
    np.testing.assert_allclose(st.zL, [1.0], rtol=1e-9)


def test_mu_schedule_golden():
    """The monotone update rule alone, against the printed schedule (tests/golden/mu_schedule.txt)."""
    g = golden_mu()
    p = SmallNLP(1, 0, lambda x: x[0], lambda x: [1.0], lambda x: [[0.0]])
    o = ipm.Options(kappa_d=0.0, bound_relax_factor=0.0, max_mu_updates=1, kappa_eps=1e30, tol=1e-8)
    s = ipm.Solver(p, [0.0], [INF], o)
    st = s.initialise([0.5], None)
    got = [(st.mu, st.tau)]
    for _ in range(6):
        st.x[:] = 0.5                  # keeps E0 above tol so that the floor row is reached
        s.iterate(st, None)       # kappa_eps huge: exactly one mu update per iteration
        got.append((st.mu, st.tau))
    np.testing.assert_allclose(np.array(got), g, rtol=2e-6)


def test_two_sided_barrier_minimiser_at_fixed_mu():
    """min x on [0,1]: the barrier problem (3) has the closed-form minimiser
    x(mu) = ((1+2mu) - sqrt(1+4mu^2))/2  (root of 1 - mu/x + mu/(1-x) = 0)."""
    p = SmallNLP(1, 0, lambda x: x[0], lambda x: [1.0], lambda x: [[0.0]])
    for mu, xstar in ((0.1, 0.0900980486), (0.02, 0.0196001599)):
        o = ipm.Options(mu_init=mu, max_mu_updates=0, bound_relax_factor=0.0, tol=1e-30, max_iter=60)
        s = ipm.Solver(p, [0.0], [1.0], o)
        st = s.initialise([0.5], None)
        for _ in range(40):
            s.iterate(st, None)
        assert abs(st.x[0] - xstar) < 1e-9
        assert abs(st.x[0] - ((1 + 2 * mu) - math.sqrt(1 + 4 * mu * mu)) / 2) < 1e-12
        assert abs(st.zL[0] * st.x[0] - mu) < 1e-12 and abs(st.zU[0] * (1 - st.x[0]) - mu) < 1e-12


def test_equality_qp_one_newton_step():
    """No bounds: (7) is the KKT system of the QP, so one full step from any x0 lands on
    [[Q, A^T],[A, 0]]^{-1} [-q; b]  -- pins assembly, the solve and the sign of y_c (eq 4, 5a)."""
    rng = np.random.default_rng(3)
    n, m = 6, 3
    M = rng.normal(size=(n, n))
    Q = M @ M.T + n * np.eye(n)
    q = rng.normal(size=n)
    A = rng.normal(size=(m, n))
    b = rng.normal(size=m)
    p = SmallNLP(n, m, lambda x: 0.5 * x @ Q @ x + q @ x, lambda x: Q @ x + q, lambda x: Q,
                 lambda x: A @ x - b, lambda x: A, None)
    s = ipm.Solver(p, np.full(n, -INF), np.full(n, INF))
    st = s.initialise(rng.normal(size=n), None)
    tr = s.iterate(st, None)
    sol = np.linalg.solve(np.block([[Q, A.T], [A, np.zeros((m, m))]]), np.concatenate([-q, b]))
    assert tr["alpha"] == 1.0 and tr["kind"] == "newton"
    np.testing.assert_allclose(st.x, sol[:n], rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(st.y, sol[n:], rtol=1e-9, atol=1e-11)
    s.iterate(st, None)
    assert st.status == ipm.ST_SOLVED and st.k == 1


def test_box_qp_clip_and_multiplier_signs():
    """min 1/2||x-a||^2, l<=x<=u: x* = clip(a,l,u), z_L* = max(0, l-a), z_U* = max(0, a-u)."""
    a = np.array([-2.0, 0.3, 5.0, 0.9, -0.5])
    l, u = np.full(5, -1.0), np.full(5, 1.0)
    p = SmallNLP(5, 0, lambda x: 0.5 * (x - a) @ (x - a), lambda x: x - a, lambda x: np.eye(5))
    s = ipm.Solver(p, l, u)
    st = s.solve(np.zeros(5), None)
    assert st.status == ipm.ST_SOLVED
    np.testing.assert_allclose(st.x, np.clip(a, l, u), atol=2e-7)
    np.testing.assert_allclose(st.zL, np.maximum(0, l - a), atol=2e-7)
    np.testing.assert_allclose(st.zU, np.maximum(0, a - u), atol=2e-7)


def test_newton_step_satisfies_unreduced_system_6():
    """Solve through (7) + the Delta z recovery; the result must satisfy all four block rows
    of (6), assembled here independently as one dense (n+m+2n) matrix."""
    d, th, x0 = wl.generate(0, 1)
    p = fam.Problem(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt)
    xL, xU = p.bounds()
    s = ipm.Solver(p, xL, xU)
    st = s.initialise(x0[0], th[0])
    for _ in range(3):
        s.iterate(st, th[0])
    x, y, zL, zU = st.x.copy(), st.y.copy(), st.zL.copy(), st.zU.copy()
    tr = s.iterate(st, th[0])
    mu = st.mu                          # the direction uses mu AFTER the A-3 update of this iteration
    dx, dy, dzL, dzU = tr["step"]
    n, m = p.n, p.m
    W, A = p.hess_lag(x, th[0], y), p.jac(x, th[0])
    iL, iU = np.where(s.hasL)[0], np.where(s.hasU)[0]
    EL, EU = np.eye(n)[:, iL], np.eye(n)[:, iU]
    SL, SU = np.diag((x - s.xL)[iL]), np.diag((s.xU - x)[iU])
    M = np.block([
        [W + tr["dw"] * np.eye(n), A.T, -EL, EU],
        [A, -tr["dc"] * np.eye(m), np.zeros((m, len(iL))), np.zeros((m, len(iU)))],
        [np.diag(zL[iL]) @ EL.T, np.zeros((len(iL), m)), SL, np.zeros((len(iL), len(iU)))],
        [-np.diag(zU[iU]) @ EU.T, np.zeros((len(iU), m)), np.zeros((len(iU), len(iL))), SU]])
    kd = s.damping(mu)
    rhs = -np.concatenate([p.grad_f(x, th[0]) + A.T @ y - zL + zU + kd, p.c(x, th[0]),
                           (x - s.xL)[iL] * zL[iL] - mu, (s.xU - x)[iU] * zU[iU] - mu])
    step = np.concatenate([dx, dy, dzL[iL], dzU[iU]])
    res = M @ step - rhs
    assert np.max(np.abs(res)) <= 1e-10 * (np.max(np.abs(rhs)) + np.max(np.abs(step)))
    np.testing.assert_allclose(step, np.linalg.solve(M, rhs), rtol=1e-7, atol=1e-9)


def test_lqr_special_case_riccati():
    """C0 without obstacle and with inactive input bounds is a finite-horizon LQR; the textbook backward
    Riccati recursion gives the optimal inputs/states.  Pins stage ordering and the dynamics Jacobians."""
    d = wl.config_dims(0, n_obstacles=0)
    p = fam.Problem(d.family, d.horizon_N, 1, 0, d.dt)
    xh = np.array([0.05, -0.04, 0.0, 0.0])
    goal = np.array([0.12, 0.02])
    th = np.concatenate([xh, goal])
    x0 = np.zeros(p.n)
    xL, xU = p.bounds()
    st = ipm.Solver(p, xL, xU).solve(x0, th)
    assert st.status == ipm.ST_SOLVED
    h, N = d.dt, d.horizon_N
    Ad = np.eye(4); Ad[0, 2] = Ad[1, 3] = h
    Bd = np.array([[h * h / 2, 0], [0, h * h / 2], [h, 0], [0, h]])
    Q = np.diag([2.0, 2.0, 0, 0]); R = 0.2 * np.eye(2)
    xg = np.array([goal[0], goal[1], 0, 0])
    # cost sum (x-xg)'Q/2(x-xg)*... with affine term: track via value function V_k(x) = 1/2 x'P x + p'x
    P = Q.copy(); pv = -Q @ xg
    Ks, ks = [], []
    for k in range(N - 1, -1, -1):
        Huu = R + Bd.T @ P @ Bd
        Hux = Bd.T @ P @ Ad
        K = -np.linalg.solve(Huu, Hux); kk = -np.linalg.solve(Huu, Bd.T @ pv)
        Ks.append(K); ks.append(kk)
        Pn = Q + Ad.T @ P @ Ad + Hux.T @ K
        pv = -Q @ xg + Ad.T @ pv + Hux.T @ kk
        P = Pn
    Ks.reverse(); ks.reverse()
    x = xh.copy()
    for k in range(N):
        u = Ks[k] @ x + ks[k]
        assert np.all(np.abs(u) < 0.9)        # bounds inactive (barrier shifts the solution by O(mu_min))
        np.testing.assert_allclose(st.x[p.iu(k):p.iu(k) + 2], u, atol=1e-6)
        x = Ad @ x + Bd @ u
        np.testing.assert_allclose(st.x[p.ix(k + 1):p.ix(k + 1) + 4], x, atol=1e-6)


def test_inertia_correction_sequence():
    """Concave 1-D objective -25 x^2 on [-1,1] from x0 = 0.2: W + Sigma < 0 so IC must fire; the first-ever
    sequence is delta_w = 1e-4, 1e-2, 1, 100 (x100 while delta_w_last = 0) and the next iteration starts from
    delta_w_last/3 and multiplies by 8 ([7] Algorithm IC, recalled)."""
    p = SmallNLP(1, 0, lambda x: -25.0 * x[0] ** 2, lambda x: [-50.0 * x[0]], lambda x: [[-50.0]])
    s = ipm.Solver(p, [-1.0], [1.0])
    st = s.initialise([0.2], None)
    tr = s.iterate(st, None)
    assert tr["nfact"] == 5 and tr["dw"] == pytest.approx(100.0) and tr["dc"] == 0.0
    assert st.delta_w_last == pytest.approx(100.0)
    tr = s.iterate(st, None)
    # Sigma grows as x approaches the bound; whichever of 100/3, 800/3 first exceeds 50 - Sigma is taken
    assert tr["dw"] in (pytest.approx(100.0 / 3.0), pytest.approx(800.0 / 3.0))
    st = s.solve([0.2], None)
    assert st.status == ipm.ST_SOLVED and abs(abs(st.x[0]) - 1.0) < 1e-6


def test_delta_c_value():
    o = ipm.Options()
    assert o.delta_c_bar * 0.1 ** o.kappa_c == pytest.approx(5.6234e-9, rel=1e-4)


def test_nonconvex_two_variable_bruteforce():
    """min (x^2-1)^2 + y^2 + 0.3x + 0.5xy, s.t. x*y <= 0.5 (slack), box [-2,2]^2.  The returned point must be
    feasible, satisfy E0 <= tol, and be a grid-local minimiser of f over the feasible set."""
    def f3(v):
        x, y = v[0], v[1]
        return (x * x - 1) ** 2 + y * y + 0.3 * x + 0.5 * x * y

    def g3(v):
        x, y = v[0], v[1]
        return [4 * x * (x * x - 1) + 0.3 + 0.5 * y, 2 * y + 0.5 * x, 0.0]

    def h3(v):
        x = v[0]
        return [[12 * x * x - 4, 0.5, 0], [0.5, 2, 0], [0, 0, 0]]
    p = SmallNLP(3, 1, f3, g3, h3, lambda v: [0.5 - v[0] * v[1] - v[2]], lambda v: [[-v[1], -v[0], -1.0]],
                 lambda v, j: [[0, -1, 0], [-1, 0, 0], [0, 0, 0]])
    s = ipm.Solver(p, [-2, -2, 0], [2, 2, INF])
    for start in ([1.5, 1.5, 0.1], [-1.5, 0.5, 1.0], [0.1, -1.0, 0.5]):
        st = s.solve(np.array(start), None)
        assert st.status == ipm.ST_SOLVED
        x, y = st.x[0], st.x[1]
        assert x * y <= 0.5 + 1e-7 and abs(x) <= 2 + 1e-7 and abs(y) <= 2 + 1e-7
        hgrid = 2e-3
        best = f3(st.x)
        for dxg in np.arange(-10, 11) * hgrid:
            for dyg in np.arange(-10, 11) * hgrid:
                xx, yy = x + dxg, y + dyg
                if xx * yy <= 0.5 and abs(xx) <= 2 and abs(yy) <= 2:
                    assert f3([xx, yy]) >= best - 1e-6


def test_c0_against_scipy_trust_constr():
    """Independent library cross-check on reduced point-mass instances (N=3)."""
    from scipy.optimize import minimize, NonlinearConstraint, Bounds
    d = wl.config_dims(0, horizon_N=3)
    d, th, x0 = wl.generate(0, 4, d)
    p = fam.Problem(d.family, d.horizon_N, 1, 1, d.dt)
    xL, xU = p.bounds()
    s = ipm.Solver(p, xL, xU)
    ncmp = 0
    for i in range(4):
        st = s.solve(x0[i], th[i])
        if st.status != ipm.ST_SOLVED:
            continue
        t = th[i]
        res = minimize(lambda v: p.f(v, t), st.x + 1e-3, jac=lambda v: p.grad_f(v, t), method="trust-constr",
                       constraints=[NonlinearConstraint(lambda v: p.c(v, t), 0, 0, jac=lambda v: p.jac(v, t))],
                       bounds=Bounds(xL, xU), options=dict(xtol=1e-12, gtol=1e-10, maxiter=3000))
        assert abs(res.fun - p.f(st.x, t)) <= 1e-6 * max(1.0, abs(res.fun))
        np.testing.assert_allclose(res.x, st.x, atol=5e-5)
        ncmp += 1
    assert ncmp >= 3


def test_invariants_along_c0_solves():
    """x strictly inside the bounds and z > 0 at every iterate; E0 <= tol, complementarity and stationarity
    recomputed here at SOLVED; filter entries only added on non-f-type steps; iteration counts do not depend on
    the order problems are solved in."""
    d, th, x0 = wl.generate(0, 24)
    p = fam.Problem(d.family, d.horizon_N, 1, 1, d.dt)
    xL, xU = p.bounds()
    s = ipm.Solver(p, xL, xU)
    iters = []
    for i in range(24):
        st = s.initialise(x0[i], th[i])
        while st.status == ipm.ST_NOT_RUN:
            nf = len(st.filt) if st.resto is None else None
            tr = s.iterate(st, th[i])
            if st.resto is None and tr["mode"] == 0 and tr["kind"] in ("newton", "soc") and tr["nmu"] == 0:
                assert len(st.filt) == nf + (0 if tr["ftype"] else 1)
            assert np.all(st.x[s.hasL] > s.xL[s.hasL]) and np.all(st.x[s.hasU] < s.xU[s.hasU])
            assert np.all(st.zL[s.hasL] > 0) and np.all(st.zU[s.hasU] > 0)
        iters.append(st.k)
        if st.status == ipm.ST_SOLVED:
            t = th[i]
            rd = p.grad_f(st.x, t) + p.jac(st.x, t).T @ st.y - st.zL + st.zU
            assert np.max(np.abs(rd)) <= 1e-8 * max(1.0, (np.abs(st.y).sum() + st.zL.sum() + st.zU.sum()) / (p.m + s.nL + s.nU) / 100)
            assert np.max(np.abs(p.c(st.x, t))) <= 1e-8
            assert np.max(np.abs((st.x - s.xL)[s.hasL] * st.zL[s.hasL])) <= 1e-8 * max(1.0, (st.zL.sum() + st.zU.sum()) / (s.nL + s.nU) / 100)
    again = [s.solve(x0[i], th[i]).k for i in reversed(range(24))][::-1]
    assert again == iters


def test_ftb_limits_exactly():
    p = SmallNLP(2, 0, lambda x: 0.0, lambda x: [0.0, 0.0], lambda x: np.zeros((2, 2)))
    s = ipm.Solver(p, [0.0, -INF], [1.0, INF], ipm.Options(bound_relax_factor=0.0))
    x = np.array([0.25, 3.0])
    a = s.ftb_primal(x, np.array([-1.0, -100.0]), 0.99)
    assert a == pytest.approx(0.99 * 0.25)                 # x + a dx = x_L + (1-tau)(x - x_L)
    assert x[0] + a * (-1.0) == pytest.approx(0.01 * 0.25)
    assert s.ftb_primal(x, np.array([3.0, 5.0]), 0.99) == pytest.approx(0.99 * 0.75 / 3.0)
    assert s.ftb_primal(x, np.array([0.1, 5.0]), 0.99) == 1.0
    assert s.ftb_dual(np.array([2.0, 0.0]), np.array([1.0, 0.0]), np.array([-4.0, -9.0]), np.array([0.5, -9.0]), 0.9) \
        == pytest.approx(0.9 * 2.0 / 4.0)


def test_restoration_infeasible_toy():
    """c(x) = x^2 + 1 = 0 has no solution: the solver must end LOCALLY_INFEASIBLE near the minimiser of |c|, x=0.
    Also pins the closed-form (p, n) initialisation: c - p + n = 0 and the barrier stationarity
    rho - mu/p - lam = 0, rho - mu/n + lam = 0 eliminated -> n solves 2 rho n^2 - (2 mu - 2 rho c) n ... ."""
    p = SmallNLP(1, 1, lambda x: x[0], lambda x: [1.0], lambda x: [[0.0]],
                 lambda x: [x[0] ** 2 + 1.0], lambda x: [[2 * x[0]]], lambda x, j: [[2.0]])
    s = ipm.Solver(p, [-INF], [INF])
    st = s.initialise([0.7], None)
    saw_resto = False
    while st.status == ipm.ST_NOT_RUN:
        tr = s.iterate(st, None)
        if tr.get("enter_resto"):
            saw_resto = True
            rs = st.resto.state
            x, pp, nn = rs.x[0], rs.x[1], rs.x[2]
            cval = x * x + 1.0
            assert abs(cval - pp + nn) < 1e-12
            mu_bar, rho = rs.mu, 1000.0
            # stationarity of rho(p+n) - mu ln p - mu ln n on the line p = c + n:  2 rho - mu/p - mu/n = 0
            assert abs(2 * rho - mu_bar / pp - mu_bar / nn) < 1e-9 * rho
            assert pp > 0 and nn > 0
    assert saw_resto
    assert st.status == ipm.ST_LOCALLY_INFEASIBLE
    assert abs(st.x[0]) < 1e-3


def test_restoration_recovers_on_feasible_problem():
    """C0 instances whose start lies inside the obstacle disc go through restoration; whatever the path, a
    SOLVED result must be feasible and the exit point must have satisfied theta <= 0.9 theta_entry."""
    d, th, x0 = wl.generate(0, 256)
    p = fam.Problem(d.family, d.horizon_N, 1, 1, d.dt)
    xL, xU = p.bounds()
    s = ipm.Solver(p, xL, xU)
    inside = [i for i in range(256) if np.linalg.norm(th[i, 0:2] - th[i, 6:8]) < th[i, 8]]
    assert inside
    nresto = 0
    for i in inside[:6]:
        st = s.initialise(x0[i], th[i])
        while st.status == ipm.ST_NOT_RUN:
            entry = st.resto.theta_entry if st.resto is not None else None
            tr = s.iterate(st, th[i])
            if tr.get("exit_resto"):
                nresto += 1
                assert np.abs(p.c(st.x, th[i])).sum() <= 0.9 * entry + 1e-15
                assert np.all(st.y == 0)
        assert st.status in (ipm.ST_SOLVED, ipm.ST_LOCALLY_INFEASIBLE, ipm.ST_RESTORATION_FAILED)
        if st.status == ipm.ST_SOLVED:
            assert np.max(np.abs(p.c(st.x, th[i]))) <= 1e-8
