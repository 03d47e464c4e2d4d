"""Pins for the oracle functions VERDICT round 1 listed as unpinned: the scaled optimality error, the filter
acceptance rules and alpha_min (A-5), the second-order correction, the interior push, the least-squares
multipliers, the z safeguard, the rigid-body model with non-zero body rates and pitch, and the mechanics of the
restoration problem.  Every expected number below is worked by hand in the docstring of its test (or comes from
an independent library routine); none re-types the oracle's formula."""
import math

import numpy as np
import pytest

from oracle import families as fam
from oracle import ipm
from helpers import SmallNLP

INF = np.inf
EPS = 2.220446049250313e-16


def plain_solver(n=1, m=0, xL=None, xU=None, **opt):
    p = SmallNLP(n, m, lambda x: 0.0, lambda x: np.zeros(n), lambda x: np.zeros((n, n)),
                 (lambda x: np.zeros(m)) if m else None, (lambda x: np.zeros((m, n))) if m else None, None)
    xL = np.full(n, -INF) if xL is None else xL
    xU = np.full(n, INF) if xU is None else xU
    return ipm.Solver(p, xL, xU, ipm.Options(bound_relax_factor=0.0, **opt))


# ---- optimality error (A-2; reading S-3) ---------------------------------------------------------------------
def test_opt_error_hand_computed_scalings():
    """n = 3, m = 1; bounds x1 >= 0, 0 <= x2 <= 4, x3 free  ->  n_L = 2, n_U = 1 multipliers exist.
    x = (1, 1, 5), z_L = (300, 600, 0), z_U = (0, 900, 0), y = 1200, grad f = (10, -20, 30), A = [0.5 -1 2], c = 7.
      s_d = max(100, (1200 + 1800)/(1 + 3))/100 = 750/100 = 7.5        s_c = max(100, 1800/3)/100 = 6
      dual residual = (10 + 600 - 300, -20 - 1200 - 600 + 900, 30 + 2400) = (310, -920, 2430)  ->  2430/7.5 = 324
      complementarity = (1*300, 1*600, (4-1)*900) = (300, 600, 2700)                             ->  2700/6 = 450
      E_0 = max(324, 7, 450) = 450.
    With mu = 0.5: complementarity 2699.5/6 = 449.91666..., the damping kappa_d*mu = 5e-6 on x1 (bounded below only)
    leaves the dual maximum at 2430: E_mu = 449.916666...
    With y = 12000: s_d = max(100, 13800/4)/100 = 34.5, dual residual (5710, -11720, 24030) -> 24030/34.5 = 696.5217...
    which now exceeds 450."""
    p = SmallNLP(3, 1, lambda x: 0.0, lambda x: np.zeros(3), lambda x: np.zeros((3, 3)),
                 lambda x: [7.0], lambda x: [[0.5, -1.0, 2.0]], None)
    s = ipm.Solver(p, [0.0, 0.0, -INF], [INF, 4.0, INF], ipm.Options(bound_relax_factor=0.0))
    x = np.array([1.0, 1.0, 5.0])
    zL, zU = np.array([300.0, 600.0, 0.0]), np.array([0.0, 900.0, 0.0])
    g, cv, A = np.array([10.0, -20.0, 30.0]), np.array([7.0]), np.array([[0.5, -1.0, 2.0]])
    assert s.opt_error(x, np.array([1200.0]), zL, zU, g, cv, A, 0.0) == pytest.approx(450.0, rel=1e-14)
    assert s.opt_error(x, np.array([1200.0]), zL, zU, g, cv, A, 0.5) == pytest.approx(2699.5 / 6.0, rel=1e-14)
    assert s.opt_error(x, np.array([12000.0]), zL, zU, g, cv, A, 0.0) == pytest.approx(24030.0 / 34.5, rel=1e-14)
    # small multipliers: both scalings are 1 and the constraint violation is the maximum
    assert s.opt_error(x, np.array([1.0]), zL / 1e3, zU / 1e3, g / 1e3, cv, A / 1e3, 0.0) == pytest.approx(7.0)


# ---- filter acceptance (A-5) ---------------------------------------------------------------------------------
def test_filter_membership_hand_made():
    """F = {(1, 10), (0.5, 20)}, theta_max = 100.  A point is forbidden iff theta >= theta_max or it is
    dominated by an entry in BOTH coordinates."""
    s = plain_solver()
    st = ipm.State(x=np.zeros(1), y=np.zeros(0), zL=np.zeros(1), zU=np.zeros(1), mu=0.1, tau=0.99)
    st.filt, st.theta_max = [(1.0, 10.0), (0.5, 20.0)], 100.0
    assert s.in_filter(st, 1.0, 10.0)            # on the corner of entry 1 (>= in both)
    assert not s.in_filter(st, 0.99, 10.0)       # left of entry 1; above entry 2 in theta only
    assert s.in_filter(st, 0.6, 25.0)            # dominated by entry 2
    assert not s.in_filter(st, 0.6, 19.999)      # below entry 2 in phi
    assert s.in_filter(st, 150.0, -1e9)          # theta >= theta_max whatever phi
    assert not s.in_filter(st, 0.4, 1e9)         # left of every entry


def test_switching_and_armijo_hand_numbers():
    """Switching condition g < 0 and alpha (-g)^2.3 > theta^1.1 (delta = 1):
        g = -2, alpha = 0.5: 0.5 * 2^2.3 = 0.5 * 4.924578 = 2.462289;  2^1.1 = 2.143547 -> holds at theta = 2,
        2.3^1.1 = 2.499773 -> fails at theta = 2.3;  g > 0 never.
    Armijo phi_t - phi_k - 10 eps |phi_k| <= 1e-8 alpha g:
        phi_k = 100, alpha = 1, g = -1: needs a decrease of 1e-8 (relaxed by 2.2e-13): -1.01e-8 passes, -0.99e-8 fails;
        phi_k = 1e6, g = -1e-3: NO decrease at all still passes because 10 eps 1e6 = 2.2e-9 > 1e-11 (the relaxation)."""
    s = plain_solver()
    assert s.switching(0.5, -2.0, 2.0) and not s.switching(0.5, -2.0, 2.3) and not s.switching(0.5, 1.0, 1e-9)
    assert 0.5 * 2.0 ** 2.3 == pytest.approx(2.462289, rel=1e-6) and 2.3 ** 1.1 == pytest.approx(2.499773, rel=1e-6)
    assert s.armijo(100.0 - 1.01e-8, 100.0, 1.0, -1.0)
    assert not s.armijo(100.0 - 0.99e-8, 100.0, 1.0, -1.0)
    assert s.armijo(1e6, 1e6, 1.0, -1e-3)
    assert not s.armijo(1e6 + 1e-8, 1e6, 1.0, -1e-3)


def test_acceptance_h_type_and_f_type_sides():
    """theta_min = 1e-4, empty filter, theta_max = 1e4.
    h-type (theta_k = 1 > theta_min, phi_k = 5): accept iff theta_t <= (1 - 1e-5) or phi_t <= 5 - 1e-8 (both relaxed
    only by 10 eps*5 = 1.1e-14):  (0.99998, 7) yes; (0.999995, 7) no; (1.5, 5 - 2e-8) yes; (1.5, 5 - 0.5e-8) no.
    f-type (theta_k = 1e-6 <= theta_min, g = -1, alpha = 1: switching 1 > (1e-6)^1.1 holds): ONLY Armijo counts:
    (0.5, 5 - 2e-8) yes although theta grew; (0, 5 - 0.5e-8) no although theta vanished.
    A filter entry (0.4, 4.0) then rejects (0.5, 5 - 2e-8)."""
    s = plain_solver()
    st = ipm.State(x=np.zeros(1), y=np.zeros(0), zL=np.zeros(1), zU=np.zeros(1), mu=0.1, tau=0.99)
    st.theta_min, st.theta_max = 1e-4, 1e4
    assert s.acceptable(st, 0.99998, 7.0, 1.0, 5.0, 1.0, -1.0)
    assert not s.acceptable(st, 0.999995, 7.0, 1.0, 5.0, 1.0, -1.0)
    assert s.acceptable(st, 1.5, 5.0 - 2e-8, 1.0, 5.0, 1.0, -1.0)
    assert not s.acceptable(st, 1.5, 5.0 - 0.5e-8, 1.0, 5.0, 1.0, -1.0)
    assert s.acceptable(st, 0.5, 5.0 - 2e-8, 1e-6, 5.0, 1.0, -1.0)
    assert not s.acceptable(st, 0.0, 5.0 - 0.5e-8, 1e-6, 5.0, 1.0, -1.0)
    assert not s.acceptable(st, math.nan, 1.0, 1.0, 5.0, 1.0, -1.0) and not s.acceptable(st, 0.1, math.inf, 1.0, 5.0, 1.0, -1.0)
    st.filt = [(0.4, 4.0)]
    assert not s.acceptable(st, 0.5, 5.0 - 2e-8, 1e-6, 5.0, 1.0, -1.0)


def test_alpha_min_three_cases():
    """alpha_min = 0.05 * { min(1e-5, 1e-8 theta/(-g), theta^1.1/(-g)^2.3)  if g < 0 and theta <= theta_min
                          { min(1e-5, 1e-8 theta/(-g))                       if g < 0 and theta > theta_min
                          { 1e-5                                             otherwise.
    (a) theta = 1e-3 <= theta_min = 1e-2, g = -1e-4: 1e-8*1e-3/1e-4 = 1e-7; (1e-3)^1.1/(1e-4)^2.3 = 5.0e-4/6.3e-10 ~ 8e5
        -> min = 1e-7 -> 5e-9.
    (a') theta = 1e-10, g = -1e6: second 1e-8*1e-10/1e6 = 1e-24; third 1e-11/10^13.8 = 10^-24.8 = 1.584893e-25
        -> 0.05 * 1.584893e-25 = 7.924466e-27.
    (b) theta = 50 > theta_min, g = -0.01: 1e-8*50/0.01 = 5e-5 > 1e-5 -> 5e-7;   theta = 2, g = -1: 2e-8 -> 1e-9.
    (c) g = +3: 5e-7."""
    s = plain_solver()
    assert s.alpha_min(-1e-4, 1e-3, 1e-2) == pytest.approx(5e-9, rel=1e-12)
    assert s.alpha_min(-1e6, 1e-10, 1e-2) == pytest.approx(7.924466e-27, rel=1e-6)
    assert s.alpha_min(-0.01, 50.0, 1e-2) == pytest.approx(5e-7, rel=1e-12)
    assert s.alpha_min(-1.0, 2.0, 1e-2) == pytest.approx(1e-9, rel=1e-12)
    assert s.alpha_min(3.0, 2.0, 1e-2) == pytest.approx(5e-7, rel=1e-12)
    assert s.alpha_min(0.0, 1e-9, 1e-2) == pytest.approx(5e-7, rel=1e-12)


def test_accepted_points_are_outside_the_filter_and_alpha_min_is_respected():
    """Along real solves: every point accepted by the line search is not in the filter it was tested against, and a
    backtracked step length is never below alpha_min."""
    from paper_2606_26341_b200 import workloads as wl
    d, th, x0 = wl.generate(0, 12)
    p = fam.Problem(d.family, d.horizon_N, 1, 1, d.dt)
    xL, xU = p.bounds()
    s = ipm.Solver(p, xL, xU)
    checked = 0
    for i in range(12):
        st = s.initialise(x0[i], th[i])
        while st.status == ipm.ST_NOT_RUN and st.resto is None:
            filt_before, thmax, mu_before = list(st.filt), st.theta_max, st.mu
            tr = s.iterate(st, th[i])
            if tr["kind"] in ("newton", "soc") and tr["mode"] == 0 and st.resto is None and not tr["wd"]:
                fil = filt_before if tr["nmu"] == 0 else []
                tmp = ipm.State(x=st.x, y=st.y, zL=st.zL, zU=st.zU, mu=st.mu, tau=st.tau, filt=fil, theta_max=thmax)
                theta_t = np.abs(p.c(st.x, th[i])).sum()
                phi_t = s.phi(st.x, p.f(st.x, th[i]), st.mu)
                assert not s.in_filter(tmp, theta_t, phi_t)
                if tr["kind"] == "newton":
                    assert tr["alpha"] >= tr["a_min"]
                checked += 1
    assert checked > 50


# ---- second-order correction (Table I row 2) -----------------------------------------------------------------
def maratos():
    """min 2(x^2+y^2-1) - x  s.t.  x^2+y^2 = 1  (the textbook example where full Newton steps from feasible points
    increase both f and |c|)."""
    return SmallNLP(2, 1, lambda v: 2 * (v[0] ** 2 + v[1] ** 2 - 1) - v[0], lambda v: [4 * v[0] - 1, 4 * v[1]],
                    lambda v: [[4, 0], [0, 4]], lambda v: [v[0] ** 2 + v[1] ** 2 - 1],
                    lambda v: [[2 * v[0], 2 * v[1]]], lambda v, j: [[2, 0], [0, 2]])


def test_second_order_correction_fires_and_solves_the_corrected_system():
    """From (0.8, 0.7) (c = 0.13) the full step is rejected with theta+ >= theta, so the correction must fire:
    c_soc = alpha c(x) + c(x + alpha dx) with alpha = 1 (no bounds), and the corrected step solves (7) with the
    same matrix and c replaced by c_soc -- checked against numpy.linalg.solve on a matrix assembled here."""
    p = maratos()
    s = ipm.Solver(p, [-INF, -INF], [INF, INF])
    st = s.initialise(np.array([0.8, 0.7]), None)
    x, y = st.x.copy(), st.y.copy()
    tr = s.iterate(st, None)
    assert tr["kind"] == "soc" and tr["soc"] == 1 and tr["ls"] == 0 and tr["alpha"] == 1.0
    dx = tr["step"][0]
    c0 = x[0] ** 2 + x[1] ** 2 - 1
    xt = x + dx
    ct = xt[0] ** 2 + xt[1] ** 2 - 1
    assert abs(ct) >= abs(c0)                                   # why the correction was tried
    np.testing.assert_allclose(tr["soc_rhs"][0], [1.0 * c0 + ct], rtol=1e-14)
    W = np.array([[4.0, 0], [0, 4.0]]) + y[0] * 2 * np.eye(2)
    A = np.array([[2 * x[0], 2 * x[1]]])
    K = np.block([[W, A.T], [A, np.zeros((1, 1))]])
    rhs = -np.concatenate([np.array([4 * x[0] - 1, 4 * x[1]]) + A.T @ y, [c0 + ct]])
    sol = np.linalg.solve(K, rhs)
    np.testing.assert_allclose(tr["soc_steps"][0][0], sol[:2], rtol=1e-10)
    np.testing.assert_allclose(tr["soc_steps"][0][1], sol[2:], rtol=1e-10)
    np.testing.assert_allclose(st.x, x + sol[:2], rtol=1e-10)   # alpha_soc = 1: the corrected point was taken
    np.testing.assert_allclose(st.y, y + sol[2:], rtol=1e-10)


def test_second_order_correction_recursion_with_short_steps_and_abort():
    """backtrack() called with a fraction-to-boundary limit alpha_max = 0.6: the first correction's right-hand side
    is 0.6 c(x) + c(x + 0.6 dx); if it is rejected with theta_soc <= 0.99 theta_old the next one is
    alpha_soc c_soc + c(x_soc); a correction that does not reduce theta by kappa_soc aborts the sequence."""
    p = maratos()
    s = ipm.Solver(p, [-INF, -INF], [INF, INF])
    st = s.initialise(np.array([0.6, 0.9]), None)
    x, y = st.x.copy(), st.y.copy()
    fv, g, cv, A = p.f(x, None), p.grad_f(x, None), p.c(x, None), p.jac(x, None)
    W = p.hess_lag(x, None, y)
    fac, dw, dc, _ = s.inertia_correction(W, np.zeros(2), A, st.mu, 0.0)
    b = [-(g + A.T @ y), -cv, np.zeros(2), np.zeros(2)]
    d, _, failed = s.solve_full(fac, W, A, x, st.zL, st.zU, dw, dc, b)
    assert not failed
    theta_k, phi_k, gd = abs(cv[0]), fv, float(g @ d[0])
    tr = dict(soc=0)
    acc = s.backtrack(st, None, tr, x, tuple(d), cv, (fac, W, A, dw, dc, b), st.mu, st.tau, theta_k, phi_k, gd, 0.6, False)
    assert tr["soc"] >= 1
    xt = x + 0.6 * d[0]
    c_first = 0.6 * cv[0] + (xt[0] ** 2 + xt[1] ** 2 - 1)
    np.testing.assert_allclose(tr["soc_rhs"][0], [c_first], rtol=1e-14)
    K = np.block([[W, A.T], [A, np.zeros((1, 1))]])
    sol = np.linalg.solve(K, -np.concatenate([g + A.T @ y, [c_first]]))
    np.testing.assert_allclose(tr["soc_steps"][0][0], sol[:2], rtol=1e-10)
    if tr["soc"] >= 2:
        xs = x + sol[:2]                                        # alpha_soc = 1 without bounds
        np.testing.assert_allclose(tr["soc_rhs"][1], [1.0 * c_first + (xs[0] ** 2 + xs[1] ** 2 - 1)], rtol=1e-12)
    else:
        xs = x + sol[:2]
        th_s = abs(xs[0] ** 2 + xs[1] ** 2 - 1)
        assert acc is not None and acc["kind"] == "soc" or th_s > 0.99 * theta_k or tr["ls"] > 0
    assert acc is not None


# ---- Step I --------------------------------------------------------------------------------------------------
def test_push_interior_hand_values():
    """kappa_1 = kappa_2 = 1e-2.
      [0, 10]:      p_L = min(0.01*max(1,0), 0.01*10) = 0.01, p_U = min(0.01*10, 0.1) = 0.1   -> clip to [0.01, 9.9]
      [5, 5.001]:   p_L = p_U = min(0.05, 1e-5) = 1e-5                                        -> [5.00001, 5.00099]
      [-200, inf):  x >= -200 + 0.01*200 = -198          (-inf, 3]: x <= 3 - 0.03 = 2.97      free: unchanged."""
    s = plain_solver(6, 0, np.array([0.0, 0.0, 5.0, -200.0, -INF, -INF]), np.array([10.0, 10.0, 5.001, INF, 3.0, INF]))
    out = s.push_interior(np.array([-3.0, 9.99, 7.0, -500.0, 2.99, 123.0]))
    np.testing.assert_allclose(out, [0.01, 9.9, 5.00099, -198.0, 2.97, 123.0], rtol=1e-14)
    out = s.push_interior(np.array([4.0, 0.001, 5.0, -100.0, -7.0, -1e9]))
    np.testing.assert_allclose(out, [4.0, 0.01, 5.00001, -100.0, -7.0, -1e9], rtol=1e-14)


def test_least_squares_multipliers_against_lstsq_and_cutoff():
    """I-5: y minimises || A^T y + (grad f - z_L + z_U) ||_2 (numpy.linalg.lstsq, an independent routine); if its
    max-norm exceeds 1e3 the multipliers start at zero."""
    rng = np.random.default_rng(11)
    n, m = 7, 3
    A = rng.normal(size=(m, n))
    g = rng.normal(size=n)
    p = SmallNLP(n, m, lambda x: g @ x, lambda x: g, lambda x: np.zeros((n, n)), lambda x: A @ x, lambda x: A, None)
    xL = np.full(n, -INF); xL[0] = -5.0
    xU = np.full(n, INF); xU[1] = 5.0
    s = ipm.Solver(p, xL, xU)
    zL = np.zeros(n); zL[0] = 1.0
    zU = np.zeros(n); zU[1] = 1.0
    y = s.least_squares_multipliers(np.zeros(n), None, zL, zU)
    ref = np.linalg.lstsq(A.T, -(g - zL + zU), rcond=None)[0]
    np.testing.assert_allclose(y, ref, rtol=1e-10, atol=1e-12)
    big = SmallNLP(n, m, lambda x: 1e5 * g @ x, lambda x: 1e5 * g, lambda x: np.zeros((n, n)), lambda x: A @ x,
                   lambda x: A, None)
    y2 = ipm.Solver(big, xL, xU).least_squares_multipliers(np.zeros(n), None, zL, zU)
    assert np.max(np.abs(np.linalg.lstsq(A.T, -(1e5 * g - zL + zU), rcond=None)[0])) > 1e3
    assert np.all(y2 == 0.0)


def test_safeguard_z_both_clamps():
    """[7] eq (16) with kappa_Sigma = 1e10, mu = 0.1: slack 2 -> z in [0.1/(2e10), 1e10*0.1/2] = [5e-12, 5e8];
    upper slack 0.5 -> [2e-11, 2e9]."""
    s = plain_solver(3, 0, np.array([0.0, 0.0, 0.0]), np.array([INF, INF, 2.5]))
    st = ipm.State(x=np.array([2.0, 2.0, 2.0]), y=np.zeros(0), zL=np.array([1e9, 1e-13, 3.0]),
                   zU=np.array([0.0, 0.0, 1e10]), mu=0.1, tau=0.99)
    s.safeguard_z(st, 0.1)
    np.testing.assert_allclose(st.zL, [5e8, 5e-12, 3.0], rtol=1e-14)
    np.testing.assert_allclose(st.zU, [0.0, 0.0, 2e9], rtol=1e-14)


# ---- rigid-body model away from hover --------------------------------------------------
def test_quad_ode_against_rotation_matrices_and_cross_products():
    """xdot from an independent statement of the model: thrust direction = Rz(psi) Ry(theta) Rx(phi) e3 (explicit
    rotation-matrix product), Euler rates from solving E(eta) etadot = omega with
    E = [[1, 0, -sin th], [0, cos ph, sin ph cos th], [0, -sin ph, cos ph cos th]] (numpy.linalg.solve), and
    omegadot = J^-1 (tau - omega x J omega) with numpy.cross; '+' rotor layout."""
    rng = np.random.default_rng(7)
    for _ in range(20):
        x = rng.uniform(-1, 1, 12)
        x[3:6] = rng.uniform(-1.2, 1.2, 3)
        x[9:12] = rng.uniform(-3, 3, 3)
        u = rng.uniform(0.5, 4.5, 4)
        ph, th, ps = x[3:6]
        Rx = np.array([[1, 0, 0], [0, math.cos(ph), -math.sin(ph)], [0, math.sin(ph), math.cos(ph)]])
        Ry = np.array([[math.cos(th), 0, math.sin(th)], [0, 1, 0], [-math.sin(th), 0, math.cos(th)]])
        Rz = np.array([[math.cos(ps), -math.sin(ps), 0], [math.sin(ps), math.cos(ps), 0], [0, 0, 1]])
        T = u.sum()
        vdot = (Rz @ Ry @ Rx) @ np.array([0, 0, T / 1.0]) - np.array([0, 0, 9.81])
        E = np.array([[1, 0, -math.sin(th)], [0, math.cos(ph), math.sin(ph) * math.cos(th)],
                      [0, -math.sin(ph), math.cos(ph) * math.cos(th)]])
        etadot = np.linalg.solve(E, x[9:12])
        Jm = np.diag([0.01, 0.01, 0.02])
        tau = np.array([0.2 * (u[1] - u[3]), 0.2 * (u[2] - u[0]), 0.02 * (u[0] - u[1] + u[2] - u[3])])
        wdot = np.linalg.solve(Jm, tau - np.cross(x[9:12], Jm @ x[9:12]))
        ref = np.concatenate([x[6:9], etadot, vdot, wdot])
        got = np.array(fam.quad_ode(list(x), list(u)), dtype=float)
        np.testing.assert_allclose(got, ref, rtol=1e-12, atol=1e-12)


# ---- restoration problem mechanics (Step R; readings R-1, R-2, S-15) -----------------------------------------
def test_restoration_nlp_values_by_hand():
    """RestoNLP on a base problem with n = 2, m = 1, c(x) = x1 x2 - 1, x_R = (2, 0.5):
       D_R = (min(1, 1/2), min(1, 1/0.5)) = (0.5, 1);  zeta = sqrt(mu) = 0.2 at mu = 0.04.
       X = (x; p; n) = (3, 1; 0.3; 0.1):  f_R = 1000 (0.3 + 0.1) + 0.2/2 * (0.25*1^2 + 1*0.5^2) = 400 + 0.1*0.5 = 400.05
       grad = (0.2*0.25*1, 0.2*1*0.5, 1000, 1000) = (0.05, 0.1, 1000, 1000);  c_R = (3*1 - 1) - 0.3 + 0.1 = 1.8
       Jacobian = [x2, x1, -1, +1] = [1, 3, -1, 1];  the Lagrangian Hessian drops f (sigma_f = 0 in the base call) and adds
       zeta D_R^2 on x: y = 2 -> [[0.05, 2], [2, 0.2]] on x, zero on p, n."""
    base = SmallNLP(2, 1, lambda x: 99.0 * x[0], lambda x: [99.0, 0.0], lambda x: np.zeros((2, 2)),
                    lambda x: [x[0] * x[1] - 1.0], lambda x: [[x[1], x[0]]], lambda x, j: [[0, 1.0], [1.0, 0]])
    r = ipm.RestoNLP(base, np.array([2.0, 0.5]), 1000.0, 0.04)
    X = np.array([3.0, 1.0, 0.3, 0.1])
    assert r.f(X, None) == pytest.approx(400.05, rel=1e-14)
    np.testing.assert_allclose(r.grad_f(X, None), [0.05, 0.1, 1000.0, 1000.0], rtol=1e-14)
    np.testing.assert_allclose(r.c(X, None), [1.8], rtol=1e-14)
    np.testing.assert_allclose(r.jac(X, None), [[1.0, 3.0, -1.0, 1.0]], rtol=1e-14)
    Wr = r.hess_lag(X, None, np.array([2.0]), 1.0)
    np.testing.assert_allclose(Wr, [[0.05, 2.0, 0, 0], [2.0, 0.2, 0, 0], [0, 0, 0, 0], [0, 0, 0, 0]], atol=1e-15)
    r.set_mu(0.01)                                           # reading R-1: zeta follows the restoration mu
    assert r.f(X, None) == pytest.approx(400.0 + 0.05 * 0.5, rel=1e-14)


def test_restoration_entry_exit_mechanics():
    """A line search that must fail (the regular filter holds the entry (0.004, -1e9): every point with theta >= 0.004 is
    forbidden, and backtracking from theta_k = 0.17 never gets there; no correction, no soft phase): Step R entry and
    exit are then checked against their definitions: entry adds ((1-gamma_theta) theta, phi - gamma_phi theta) to the
    REGULAR filter, mu_bar = max(mu, ||c||_inf), z_L, z_U = min(rho, z), lambda_bar = 0, z_p = mu_bar/p, z_n = mu_bar/n;
    the exit happens at the first restoration iterate with theta <= 0.9 theta_entry outside the regular filter, and
    resets y to 0 and z to 1 when some z exceeds 1e3 (reading S-15)."""
    p = maratos()
    o = ipm.Options(max_soc=0, soft_resto_factor=0.0, bound_relax_factor=0.0)
    s = ipm.Solver(p, [-INF, -5.0], [INF, INF], o)
    st = s.initialise(np.array([0.6, 0.9]), None)
    st.zL[1] = 5000.0                                        # a large bound multiplier: capped at rho on entry
    st.filt = [(0.004, -1e9)]
    x_e, mu_e = st.x.copy(), st.mu
    tr = s.iterate(st, None)
    assert tr.get("enter_resto") and tr["kind"] == "ls_fail" and st.k == 1
    theta_e = abs(x_e[0] ** 2 + x_e[1] ** 2 - 1)
    phi_e = p.f(x_e, None) - mu_e * math.log(x_e[1] + 5.0) + o.kappa_d * mu_e * (x_e[1] + 5.0)
    assert st.filt[-1] == pytest.approx(((1 - 1e-5) * theta_e, phi_e - 1e-8 * theta_e), rel=1e-13)
    rs = st.resto.state
    assert rs.mu == max(mu_e, theta_e) and np.all(rs.y == 0.0)
    assert rs.zL[1] == 1000.0 and rs.zL[0] == 0.0
    pp, nn = rs.x[2], rs.x[3]
    assert rs.zL[2] == pytest.approx(rs.mu / pp) and rs.zL[3] == pytest.approx(rs.mu / nn)
    np.testing.assert_array_equal(rs.x[:2], x_e)
    # run the restoration phase until it hands back
    while st.status == ipm.ST_NOT_RUN and st.resto is not None:
        before = st.resto.state.x[:2].copy()
        tr = s.iterate(st, None)
        if st.resto is not None and st.status == ipm.ST_NOT_RUN:
            xr = st.resto.state.x[:2]
            th_r = abs(xr[0] ** 2 + xr[1] ** 2 - 1)
            phi_r = s.phi(xr, p.f(xr, None), st.mu)
            assert th_r > 0.9 * theta_e or s.in_filter(st, th_r, phi_r)     # else it would have left
    assert tr.get("exit_resto")
    th_x = abs(st.x[0] ** 2 + st.x[1] ** 2 - 1)
    assert th_x <= 0.9 * theta_e and th_x < 0.004 and not s.in_filter(st, th_x, s.phi(st.x, p.f(st.x, None), st.mu))
    assert np.all(st.y == 0.0) and st.mu == mu_e
    assert st.zL[1] <= 1e3 or st.zL[1] == 1.0
