"""Pins for the fallbacks of Table I rows 3-5 (watchdog, tiny-step rule, soft feasibility
restoration) and for the "pretend singular" reaction to a failed iterative refinement (reading S-7).  Each case is
small enough that the expected iterates are worked by hand in the docstring or recomputed here with independent
numpy code."""
import math

import numpy as np
import pytest

from oracle import ipm
from helpers import SmallNLP

INF = np.inf
EPS = 2.220446049250313e-16


def sqrt_problem():
    """f(x) = sqrt(1 + x^2): f' = x / sqrt(1+x^2), f'' = (1+x^2)^(-3/2), so the Newton step is -x (1 + x^2) and the
    full step lands on -x^3: it converges for |x| < 1 and diverges for |x| > 1."""
    return SmallNLP(1, 0, lambda x: math.sqrt(1 + x[0] ** 2), lambda x: [x[0] / math.sqrt(1 + x[0] ** 2)],
                    lambda x: [[(1 + x[0] ** 2) ** -1.5]])


# ---- watchdog (Table I row 3) --------------------------------------------------------------------------------
def test_watchdog_reverts_to_entry_iterate_after_three_unconditional_steps():
    """Entry x_e = 1.5 with 10 shortened steps on the counter.  Newton direction d_e = -1.5 (1 + 2.25) = -4.875.
    The watchdog takes the full steps x -> -x^3 without any test: -3.375, 38.443359375, -56815.1286...; none is
    acceptable to the ENTRY iterate (f only grows), so the fourth iteration gives up, returns to x_e and backtracks
    along d_e, skipping the full step that was already tried: alpha = 1/2 -> x = 1.5 - 2.4375 = -0.9375 (f = 1.3707
    < f(1.5) = 1.8028: Armijo holds)."""
    s = ipm.Solver(sqrt_problem(), [-INF], [INF], ipm.Options(max_mu_updates=0))
    st = s.initialise(np.array([1.5]), None)
    st.n_short = 10
    tr = s.iterate(st, None)
    assert tr["wd"] == 1 and st.wd is not None and st.wd.trials == 1 and tr["ls"] == 0
    assert st.wd.x[0] == 1.5 and st.wd.d[0][0] == pytest.approx(-4.875, rel=1e-14) and st.wd.alpha == 1.0
    assert st.x[0] == pytest.approx(-3.375, rel=1e-14)
    nfilt = len(st.filt)
    tr = s.iterate(st, None)
    assert tr["wd"] == 2 and st.x[0] == pytest.approx(38.443359375, rel=1e-13) and st.wd.trials == 2
    tr = s.iterate(st, None)
    assert tr["wd"] == 2 and st.x[0] == pytest.approx(-(38.443359375 ** 3), rel=1e-12) and st.wd.trials == 3
    assert len(st.filt) == nfilt                     # unconditional steps leave the filter alone
    tr = s.iterate(st, None)
    assert tr["wd"] == 4 and st.wd is None
    assert st.x[0] == -0.9375                        # exactly: 1.5 + 0.5 * (-4.875)
    assert tr["ls"] == 1 and tr["alpha"] == 0.5 and tr["step"][0][0] == pytest.approx(-4.875, rel=1e-14)
    assert st.k == 4 and st.n_short == 1
    # from -0.9375 the full steps converge (|x| < 1): no more backtracking
    tr = s.iterate(st, None)
    assert tr["wd"] == 0 and tr["ls"] == 0 and st.x[0] == pytest.approx(0.9375 ** 3, rel=1e-13)


def test_watchdog_succeeds_when_a_full_step_is_acceptable_to_the_entry_iterate():
    """From x = 2 the line search needs two halvings (full step -8, then -3, then -0.5: the first with f below f(2)),
    which brings the counter from 9 to 10; the next iteration starts the watchdog at x_e = -0.5 and its full step to
    0.125 is acceptable at once: success, counter back to 0, no unconditional step taken."""
    s = ipm.Solver(sqrt_problem(), [-INF], [INF], ipm.Options(max_mu_updates=0))
    st = s.initialise(np.array([2.0]), None)
    st.n_short = 9
    tr = s.iterate(st, None)
    assert tr["ls"] == 2 and st.x[0] == -0.5 and st.n_short == 10 and tr["wd"] == 0
    tr = s.iterate(st, None)
    assert tr["wd"] == 3 and st.wd is None and st.n_short == 0 and st.x[0] == pytest.approx(0.125, rel=1e-14)
    # below the trigger nothing wakes up
    st = s.initialise(np.array([2.0]), None)
    st.n_short = 8
    s.iterate(st, None)
    tr = s.iterate(st, None)
    assert tr["wd"] == 0 and st.n_short == 0


def test_watchdog_success_is_measured_against_the_entry_not_the_previous_iterate():
    """Entry x_e = 1.05 (f = 1.45): unconditional steps -1.157625, 1.551328..., then -3.7334...: each is worse than its
    predecessor AND than the entry, so the watchdog reverts.  With entry 0.98 instead the second full step
    (-0.941192 -> 0.8337...) has f below the entry's: the FIRST trial is already acceptable (|x| < 1 contracts)."""
    s = ipm.Solver(sqrt_problem(), [-INF], [INF], ipm.Options(max_mu_updates=0))
    st = s.initialise(np.array([1.05]), None)
    st.n_short = 10
    codes = []
    for _ in range(4):
        codes.append(s.iterate(st, None)["wd"])
    assert codes == [1, 2, 2, 4]
    assert st.x[0] == pytest.approx(1.05 + 0.5 * (-1.05 * (1 + 1.05 ** 2)), rel=1e-14)
    st = s.initialise(np.array([0.98]), None)
    st.n_short = 10
    assert s.iterate(st, None)["wd"] == 3


def test_barrier_decrease_cancels_the_watchdog():
    s = ipm.Solver(sqrt_problem(), [-INF], [INF])          # default options: mu decreases as soon as E_mu <= 10 mu
    st = s.initialise(np.array([1.5]), None)
    st.n_short = 10
    tr = s.iterate(st, None)
    assert tr["nmu"] >= 1 and tr["wd"] == 0 and st.wd is None


# ---- tiny step (Table I row 4) -------------------------------------------------------------------------------
def stiff_quadratic():
    return SmallNLP(1, 0, lambda x: 0.5e12 * (x[0] - 1) ** 2, lambda x: [1e12 * (x[0] - 1)], lambda x: [[1e12]])


def test_tiny_step_is_accepted_without_any_test():
    """f = 1e12/2 (x-1)^2 at x = 1 + 4 eps: E_0 = 1e12 * 8.9e-16 = 8.9e-4 > tol, but the Newton step -8.9e-16 is below
    10 eps (1 + |x|) = 4.4e-15.  The filter is rigged to forbid EVERY point (entry (0, -inf)), so an ordinary line
    search would fail; the tiny-step rule accepts x + alpha_max dx = 1 exactly, leaves the filter alone and does not
    touch the watchdog counter."""
    s = ipm.Solver(stiff_quadratic(), [-INF], [INF], ipm.Options(max_mu_updates=0))
    st = s.initialise(np.array([1.0 + 4 * EPS]), None)
    st.filt = [(0.0, -INF)]
    st.n_short = 7
    tr = s.iterate(st, None)
    assert tr["tiny"] == 1 and tr["kind"] == "tiny" and tr["alpha"] == 1.0 and tr["ls"] == 0
    assert st.x[0] == 1.0 and st.filt == [(0.0, -INF)] and st.n_short == 7 and st.k == 1
    assert st.tiny_last and not st.tiny_flag
    # the same start with a step that is NOT tiny (x = 1 + 1e-9) goes through the (rigged) line search and fails
    st = s.initialise(np.array([1.0 + 1e-9]), None)
    st.filt = [(0.0, -INF)]
    tr = s.iterate(st, None)
    assert tr["tiny"] == 0 and tr["kind"] != "tiny"


def test_two_tiny_steps_force_a_barrier_decrease_then_stop():
    """Two tiny steps in a row (with a small multiplier step: there are no constraints here) raise the flag; the next
    barrier update decreases mu ONCE although E_mu > kappa_eps mu (0.1 -> 0.02, the golden schedule's first rung);
    when mu already sits at its floor the solver stops with TINY_STEP."""
    o = ipm.Options(kappa_eps=1e-30)                       # the ordinary update rule can never fire
    s = ipm.Solver(stiff_quadratic(), [-INF], [INF], o)
    st = s.initialise(np.array([1.0 + 4 * EPS]), None)
    s.iterate(st, None)
    assert st.tiny_last and not st.tiny_flag and st.mu == 0.1
    st.x[:] = 1.0 + 4 * EPS
    tr = s.iterate(st, None)
    assert tr["tiny"] == 1 and st.tiny_flag and st.mu == 0.1
    st.x[:] = 1.0 + 4 * EPS
    tr = s.iterate(st, None)
    assert tr["nmu"] == 1 and st.mu == pytest.approx(0.02, rel=1e-14)
    # a normal step in between clears the memory
    st.x[:] = 1.0 + 1e-9
    s.iterate(st, None)
    assert not st.tiny_last and not st.tiny_flag
    # at the floor of mu the forced decrease is impossible: TINY_STEP
    st = s.initialise(np.array([1.0 + 4 * EPS]), None)
    st.mu = o.mu_min
    for _ in range(2):
        st.x[:] = 1.0 + 4 * EPS
        s.iterate(st, None)
    assert st.tiny_flag
    st.x[:] = 1.0 + 4 * EPS
    tr = s.iterate(st, None)
    assert st.status == ipm.ST_TINY_STEP and tr["status"] == ipm.ST_TINY_STEP


def test_tiny_step_needs_small_constraint_violation():
    """The rule does not apply while ||c||_inf > 1e-4 (a vanishing step at an infeasible point is a different failure)."""
    p = SmallNLP(1, 1, lambda x: 0.5e12 * (x[0] - 1) ** 2, lambda x: [1e12 * (x[0] - 1)], lambda x: [[1e12]],
                 lambda x: [1e-12 * x[0] + 1e-3], lambda x: [[1e-12]], None)
    s = ipm.Solver(p, [-INF], [INF], ipm.Options(max_mu_updates=0))
    st = s.initialise(np.array([1.0 + 4 * EPS]), None)
    st.y[:] = 0.0
    tr = s.iterate(st, None)
    assert tr["tiny"] == 0


# ---- soft restoration (Table I row 5) ------------------------------------------------------------------------
def box_qp():
    rng = np.random.default_rng(3)
    n, m = 4, 2
    M = rng.normal(size=(n, n))
    Q = M @ M.T + n * np.eye(n)
    q, A, b = rng.normal(size=n), rng.normal(size=(m, n)), rng.normal(size=m)
    p = SmallNLP(n, m, lambda x: 0.5 * x @ Q @ x + q @ x, lambda x: Q @ x + q, lambda x: Q, lambda x: A @ x - b,
                 lambda x: A, None)
    return p, Q, q, A, b


def pd_error_by_hand(x, y, zL, zU, Q, q, A, b, mu, lo, hi):
    """(||grad L||_1 / n) + (||c||_1 / m) + (||complementarity - mu||_1 / #bounds), typed out independently."""
    rd = Q @ x + q + A.T @ y - zL + zU
    comp = np.concatenate([(x - lo) * zL - mu, (hi - x) * zU - mu])
    return np.abs(rd).sum() / x.size + np.abs(A @ x - b).sum() / b.size + np.abs(comp).sum() / comp.size


def test_soft_restoration_step_and_return_to_the_original_criterion():
    """Convex QP with two linear equalities and the box [-2, 2]^4, mu fixed at 0.1.  Iteration 1: the regular filter is
    rigged with the entry (0, -inf), which forbids EVERY point, so the line search fails.  The soft phase takes ONE step
    length alpha = min(alpha_max, alpha_z_max) for x, y, z_L and z_U (here the dual limit 0.7697 binds); the point is
    forbidden like all others, but the primal-dual error (recomputed here independently) drops by more than the factor
    0.9999: accepted, phase continues ('s').  Iteration 2: the rigged entry is replaced by (1e-6, -inf); the full step
    reaches theta+ ~ 1e-16 < 1e-6 with theta reduced, so the original criterion holds again: accepted, phase over ('S')."""
    p, Q, q, A, b = box_qp()
    lo, hi = np.full(4, -2.0), np.full(4, 2.0)
    s = ipm.Solver(p, lo, hi, ipm.Options(max_mu_updates=0, bound_relax_factor=0.0))
    st = s.initialise(np.zeros(4), None)
    st.filt = [(0.0, -INF)]
    x, y, zL, zU = st.x.copy(), st.y.copy(), st.zL.copy(), st.zU.copy()
    tr = s.iterate(st, None)
    assert tr["kind"] == "soft" and tr["soft"] == 1 and st.soft and st.soft_count == 0 and tr["ls"] > 5
    dx, dy, dzL, dzU = tr["step"]
    a = min(s.ftb_primal(x, dx, st.tau), s.ftb_dual(zL, zU, dzL, dzU, st.tau))
    assert a < 1.0 and tr["alpha"] == a and tr["alpha_z"] == a
    np.testing.assert_allclose(st.x, x + a * dx, rtol=1e-15)
    np.testing.assert_allclose(st.y, y + a * dy, rtol=1e-15)
    np.testing.assert_allclose(st.zL, zL + a * dzL, rtol=1e-15)
    np.testing.assert_allclose(st.zU, zU + a * dzU, rtol=1e-15)
    e_k = pd_error_by_hand(x, y, zL, zU, Q, q, A, b, 0.1, lo, hi)
    e_t = pd_error_by_hand(st.x, st.y, st.zL, st.zU, Q, q, A, b, 0.1, lo, hi)
    assert e_t <= (1 - 1e-4) * e_k
    assert len(st.filt) == 2                                 # the phase starts by adding the current point to the filter
    theta_k = np.abs(A @ x - b).sum()
    assert st.filt[-1][0] == pytest.approx((1 - 1e-5) * theta_k, rel=1e-13)
    st.filt[0] = (1e-6, -INF)
    tr = s.iterate(st, None)
    assert tr["kind"] == "soft" and tr["soft"] == 2 and not st.soft and st.soft_count == 0
    assert np.abs(A @ st.x - b).sum() < 1e-6 and len(st.filt) == 2
    tr = s.iterate(st, None)
    assert tr["soft"] == 0 and tr["kind"] in ("newton", "soc", "tiny")


def test_soft_restoration_gives_way_to_hard_restoration():
    """(a) a soft step that does not reduce the primal-dual error is refused: hard restoration starts in the same
    iteration; (b) the phase lasts at most max_soft_resto_iters iterations."""
    p, Q, q, A, b = box_qp()
    lo, hi = np.full(4, -2.0), np.full(4, 2.0)
    o = ipm.Options(max_mu_updates=0, bound_relax_factor=0.0, soft_resto_factor=1e-12)   # asks for an impossible reduction
    s = ipm.Solver(p, lo, hi, o)
    st = s.initialise(np.zeros(4), None)
    st.filt = [(0.0, -INF)]
    tr = s.iterate(st, None)
    assert tr["kind"] == "ls_fail" and tr.get("enter_resto") and not st.soft and st.resto is not None
    # (b): everything forbidden, error reduction easy -> soft steps until the limit, then hard restoration
    o2 = ipm.Options(max_mu_updates=0, bound_relax_factor=0.0, soft_resto_factor=1.0 - 1e-15, max_soft_resto_iters=3,
                     tiny_step_tol=0.0)
    s = ipm.Solver(p, lo, hi, o2)
    st = s.initialise(np.zeros(4), None)
    st.filt = [(0.0, -INF)]
    kinds = []
    for _ in range(6):
        tr = s.iterate(st, None)
        kinds.append((tr["kind"], tr["soft"]))
        if st.resto is not None or st.status != ipm.ST_NOT_RUN:
            break
    assert [k for k, _ in kinds[:-1]] == ["soft"] * (len(kinds) - 1) and len(kinds) <= 5
    assert kinds[-1][0] == "ls_fail" or st.status != ipm.ST_NOT_RUN


# ---- pretend singular (reading S-7) --------------------------------------------------------------------------
def test_refinement_failure_is_treated_as_a_singular_matrix():
    """The reaction to a failed refinement, with the failure SIMULATED (Bunch-Kaufman on small dense systems does not
    fail by itself: a nearly dependent pair of rows shows up as a wrong inertia first): solve_full is wrapped so that
    its first call -- and, in the second scenario, its first two calls -- report failure.  The solver must act as if a
    zero eigenvalue had been found: delta_c = 1e-8 mu^0.25 = 5.6234e-9, delta_w = first rung 1e-4 (then x100 = 1e-2),
    one more factorisation per reaction, and the step finally taken solves the PERTURBED system (numpy.linalg.solve)."""
    n, m = 3, 2
    A = np.array([[1.0, 2.0, -1.0], [0.0, 1.0, 1.0]])
    bvec = np.array([0.0, 1.0])
    Q = np.diag([2.0, 3.0, 4.0])
    p = SmallNLP(n, m, lambda x: 0.5 * x @ Q @ x, lambda x: Q @ x, lambda x: Q, lambda x: A @ x - bvec, lambda x: A, None)

    class Flaky(ipm.Solver):
        fail_first = 1
        calls = 0

        def solve_full(self, *a, **k):
            d, nref, failed = super().solve_full(*a, **k)
            self.calls += 1
            return d, nref, failed or self.calls <= self.fail_first

    for nfail, dw_expect in ((1, 1e-4), (2, 1e-2)):
        s = Flaky(p, np.full(n, -INF), np.full(n, INF), ipm.Options(max_mu_updates=0))
        s.fail_first = nfail
        st = s.initialise(np.array([1.0, 1.0, 1.0]), None)
        x, y = st.x.copy(), st.y.copy()
        tr = s.iterate(st, None)
        assert tr["npsing"] == nfail and tr["nfact"] == 1 + nfail
        assert tr["dc"] == pytest.approx(5.6234e-9, rel=1e-4) and tr["dw"] == pytest.approx(dw_expect, rel=1e-14)
        assert st.delta_w_last == pytest.approx(dw_expect, rel=1e-14)
        K = np.block([[Q + tr["dw"] * np.eye(n), A.T], [A, -tr["dc"] * np.eye(m)]])
        sol = np.linalg.solve(K, -np.concatenate([Q @ x + A.T @ y, A @ x - bvec]))
        np.testing.assert_allclose(tr["step"][0], sol[:n], rtol=1e-9)
        np.testing.assert_allclose(tr["step"][1], sol[n:], rtol=1e-9)
    # with delta_w_last = 0.3 from an earlier iteration the ladder starts at 0.3/3 and multiplies by 8
    s = Flaky(p, np.full(n, -INF), np.full(n, INF), ipm.Options(max_mu_updates=0))
    s.fail_first = 2
    st = s.initialise(np.array([1.0, 1.0, 1.0]), None)
    st.delta_w_last = 0.3
    tr = s.iterate(st, None)
    assert tr["dw"] == pytest.approx(0.8, rel=1e-14) and tr["nfact"] == 3
    # failures without end climb the ladder to delta_w_max and end in restoration (IC-6)
    s = Flaky(p, np.full(n, -INF), np.full(n, INF), ipm.Options(max_mu_updates=0))
    s.fail_first = 10 ** 9
    st = s.initialise(np.array([1.0, 1.0, 1.0]), None)
    tr = s.iterate(st, None)
    assert tr["kind"] == "ic_fail" and tr.get("enter_resto")
    # the honest solver never triggers it on this well-conditioned system
    s = ipm.Solver(p, np.full(n, -INF), np.full(n, INF))
    tr = s.iterate(s.initialise(np.ones(3), None), None)
    assert tr["npsing"] == 0 and tr["nfact"] == 1 and tr["dw"] == 0.0


def test_solve_full_reports_failure_only_above_the_singular_ratio():
    """solve_full() with a deliberately WRONG factor (the factor of a perturbed matrix): refinement stalls.  If the
    stalled ratio is below residual_ratio_singular (1e-5) the solution is kept, else the failure flag is raised."""
    rng = np.random.default_rng(5)
    n, m = 5, 2
    M = rng.normal(size=(n, n))
    W = M @ M.T + n * np.eye(n)
    A = rng.normal(size=(m, n))
    p = SmallNLP(n, m, lambda x: 0.0, lambda x: np.zeros(n), lambda x: W, lambda x: np.zeros(m), lambda x: A, None)
    s = ipm.Solver(p, np.full(n, -INF), np.full(n, INF))
    x, z = np.zeros(n), np.zeros(n)
    b = [rng.normal(size=n), rng.normal(size=m), np.zeros(n), np.zeros(n)]
    from oracle.linsolve import DenseLDL
    good = DenseLDL(s.kkt_matrix(W, np.zeros(n), A, 0.0, 0.0))
    d, nref, failed = s.solve_full(good, W, A, x, z, z, 0.0, 0.0, b)
    assert not failed and nref == 1
    # factor of a DIFFERENT matrix (W scaled by -1 in one entry): refinement with it diverges -> failure
    Wbad = W.copy()
    Wbad[0, 0] = -W[0, 0]
    bad = DenseLDL(s.kkt_matrix(Wbad, np.zeros(n), A, 0.0, 0.0))
    d, nref, failed = s.solve_full(bad, W, A, x, z, z, 0.0, 0.0, b)
    assert failed and nref >= 2
    # same wrong factor, but the bar for 'singular' raised above the stalled ratio: the solution is kept
    s.o.residual_ratio_singular = 1e300
    d, nref, failed = s.solve_full(bad, W, A, x, z, z, 0.0, 0.0, b)
    assert not failed


# ---- adaptive barrier parameter with the switch to the monotone schedule (Table I row 7) ------------------------
def one_dim_bound_problem():
    return SmallNLP(1, 0, lambda x: x[0], lambda x: [1.0], lambda x: [[0.0]])


def test_adaptive_mu_probing_by_hand():
    """min x s.t. x >= 0 at x = 0.5, z = 2 (no damping, no bound relaxation).  Affine-scaling step = Newton step on (5)
    with mu = 0:  row 1 of (6): -dz = -(1 - 2) -> dz = -1;  row 3: z dx + s dz = -s z -> 2 dx - 0.5 = -1 -> dx = -0.25.
    Both reach at most half-way to their bounds, so the step lengths to the boundary are 1:
    mu_aff = (0.5 - 0.25)(2 - 1) = 0.25, average complementarity s z = 1, sigma = 0.25^3 = 1/64, mu = 0.015625;
    the upper bound of mu is 1e3 x the first average complementarity = 1000; the filter is reset."""
    o = ipm.Options(mu_strategy=1, kappa_d=0.0, bound_relax_factor=0.0)
    s = ipm.Solver(one_dim_bound_problem(), [0.0], [INF], o)
    st = s.initialise([0.5], None)
    st.zL[:] = 2.0
    st.filt = [(1.0, 1.0)]
    tr = s.iterate(st, None)
    assert tr["mu_mode"] == 1 and tr["mu_switch"] == 0
    np.testing.assert_allclose(tr["aff_step"][0], [-0.25], rtol=1e-13)
    np.testing.assert_allclose(tr["aff_step"][2], [-1.0], rtol=1e-13)
    assert tr["mu_aff"] == pytest.approx(0.25, rel=1e-13) and tr["sigma"] == pytest.approx(1.0 / 64.0, rel=1e-13)
    assert st.mu == pytest.approx(0.015625, rel=1e-13) and st.mu_max == pytest.approx(1000.0)
    assert st.tau == max(0.99, 1.0 - st.mu) and st.kkt_hist and len(st.kkt_hist) == 1
    # the Newton step of the iteration used the NEW mu: Sigma = 4, grad phi = 1 - mu/0.5, dx = -(1 - 2 mu)/4
    np.testing.assert_allclose(tr["step"][0], [-(1.0 - 2.0 * 0.015625) / 4.0], rtol=1e-12)
    # mu is clipped at its floor: from z = 1 the affine step reaches the bound exactly, mu_aff = 0
    st = s.initialise([0.5], None)
    s.iterate(st, None)
    assert st.mu == o.mu_min


def test_adaptive_mu_switches_to_monotone_and_back():
    """Free mode keeps the KKT errors of the last 4 accepted iterates; an iterate whose error exceeds 0.9999 x the largest
    of them sends the solver to the monotone schedule with mu = 0.8 x average complementarity (filter reset, no probing);
    it returns to the adaptive rule once the barrier problem is solved (E_mu <= 10 mu)."""
    o = ipm.Options(mu_strategy=1, kappa_d=0.0, bound_relax_factor=0.0)
    s = ipm.Solver(one_dim_bound_problem(), [0.0], [INF], o)
    st = s.initialise([0.5], None)
    st.zL[:] = 2.0
    # KKT error here: |1 - z| / 1 + |s z - 0| / 1 = 1 + 1 = 2
    st.kkt_hist = [9.0, 1.5, 1.9, 1.0, 1.2]          # only the last four count: max 1.9 < 2 -> no progress
    tr = s.iterate(st, None)
    assert tr["mu_switch"] == 1 and tr["mu_mode"] == 2 and not st.mu_free and "sigma" not in tr
    assert st.mu == pytest.approx(0.8, rel=1e-14)
    # with the same history but its largest recent value 2.1 the iterate counts as progress and is appended
    st = s.initialise([0.5], None)
    st.zL[:] = 2.0
    st.kkt_hist = [9.0, 1.5, 2.1, 1.0, 1.2]
    tr = s.iterate(st, None)
    assert tr["mu_switch"] == 0 and st.mu_free and st.kkt_hist[:4] == [1.5, 2.1, 1.0, 1.2] and len(st.kkt_hist) == 5
    # monotone phase: mu stays until E_mu <= kappa_eps mu, then the adaptive rule is back with a fresh history
    st = s.initialise([0.5], None)
    st.zL[:] = 2.0
    st.mu_free, st.mu, st.mu_max = False, 1e-3, 1000.0   # E_mu = max(|1-2|, |1 - 1e-3|) = 1 > 10 * 1e-3: stay
    tr = s.iterate(st, None)
    assert tr["mu_mode"] == 2 and tr["mu_switch"] == 0 and st.mu == 1e-3 and tr["nmu"] == 0
    st = s.initialise([0.5], None)
    st.zL[:] = 2.0
    st.mu_free, st.mu, st.mu_max = False, 0.8, 1000.0    # E_mu = 1 <= 8: solved -> free mode, probing in the same iteration
    tr = s.iterate(st, None)
    assert tr["mu_switch"] == 2 and tr["mu_mode"] == 1 and st.mu_free and "sigma" in tr and len(st.kkt_hist) == 1


def test_adaptive_mu_solves_the_same_problems():
    """The adaptive strategy reaches the same solutions as the monotone one on box QPs (closed form: clip)."""
    a = np.array([-2.0, 0.3, 5.0, 0.9, -0.5])
    l, u = np.full(5, -1.0), np.full(5, 1.0)
    p = SmallNLP(5, 0, lambda x: 0.5 * (x - a) @ (x - a), lambda x: x - a, lambda x: np.eye(5))
    st = ipm.Solver(p, l, u, ipm.Options(mu_strategy=1)).solve(np.zeros(5), None)
    assert st.status == ipm.ST_SOLVED
    np.testing.assert_allclose(st.x, np.clip(a, l, u), atol=2e-7)


# ---- acceptable-level termination (NEXT-4, reading AT) --------------------------------------------------------
def one_dim_barrier(**opt):
    """min x s.t. x >= 0 from x0 = 0.5, z == 1 (test_oracle_ipm.py): x_k = the barrier parameter of iteration k-1, so
    E_0 at the start of iterations 0..4 is the complementarity x_k z = 0.5, 0.02, 1.504241e-4, 1.844914e-6, 2.505904e-9
    (tests/golden/mu_schedule.txt) and the dual residual 1 - z is 0."""
    p = SmallNLP(1, 0, lambda x: x[0], lambda x: [1.0], lambda x: [[0.0]])
    s = ipm.Solver(p, [0.0], [INF], ipm.Options(kappa_d=0.0, bound_relax_factor=0.0, **opt))
    return s, s.initialise([0.5], None)


def run(s, st):
    acc = []
    while st.status == ipm.ST_NOT_RUN:
        acc.append(s.iterate(st, None).get("acc"))
    return acc


def test_acceptable_level_termination_counts_consecutive_iterations():
    """acceptable_tol = 1e-3: E_0 = 1.5e-4 at iteration 2 is the first acceptable one, 1.8e-6 at iteration 3 the second:
    with acceptable_iter = 2 the solve stops THERE (k = 3, status ACCEPTABLE) instead of SOLVED at k = 4; with
    acceptable_iter = 3 the third acceptable iterate already meets tol = 1e-8 and SOLVED wins (it is tested first)."""
    s, st = one_dim_barrier(acceptable_tol=1e-3, acceptable_iter=2)
    assert run(s, st) == [0, 0, 1, 2] and st.status == ipm.ST_ACCEPTABLE and st.k == 3
    assert st.x[0] == pytest.approx(1.844914e-6, rel=2e-6)
    s, st = one_dim_barrier(acceptable_tol=1e-3, acceptable_iter=3)
    assert run(s, st) == [0, 0, 1, 2, None] and st.status == ipm.ST_SOLVED and st.k == 4
    # off by default: the pinned trajectory is untouched
    s, st = one_dim_barrier()
    assert run(s, st) == [None] * 5 and st.status == ipm.ST_SOLVED and st.k == 4


def test_acceptable_level_needs_every_component_bound_and_resets():
    """The complementarity bound is on the UNSCALED product: with acceptable_compl_inf_tol = 1e-5 iteration 2
    (x z = 1.5e-4) is not acceptable although E_0 <= acceptable_tol, iteration 3 is the first, and the solve ends SOLVED.
    A dual bound of 0 can never hold on a problem whose dual residual is not exactly 0 (x0 away from z = 1 is not needed:
    here it IS exactly 0, so the bound 0 still passes -- the constraint bound is the one that fails below).  A counter
    left over from earlier iterations is cleared by one iteration that is not acceptable."""
    s, st = one_dim_barrier(acceptable_tol=1e-3, acceptable_iter=2, acceptable_compl_inf_tol=1e-5)
    assert run(s, st) == [0, 0, 0, 1, None] and st.status == ipm.ST_SOLVED
    s, st = one_dim_barrier(acceptable_tol=1e-3, acceptable_iter=2, acceptable_dual_inf_tol=0.0)
    assert run(s, st) == [0, 0, 1, 2] and st.status == ipm.ST_ACCEPTABLE          # dual residual 1 - z == 0 exactly
    s, st = one_dim_barrier(acceptable_tol=1e-3, acceptable_iter=50)
    st.acc_count = 7
    assert s.iterate(st, None)["acc"] == 0 and st.acc_count == 0                     # E_0 = 0.5 at iteration 0
    # with an equality constraint the violation bound counts: c = x1 + x2 - 1 at a point with |c| = 0.2 > 1e-2
    p = SmallNLP(2, 1, lambda x: 0.0, lambda x: np.zeros(2), lambda x: np.zeros((2, 2)),
                 lambda x: [x[0] + x[1] - 1.0], lambda x: [[1.0, 1.0]], None)
    s2 = ipm.Solver(p, [-INF, -INF], [INF, INF], ipm.Options(acceptable_tol=1.0, acceptable_iter=1))
    x = np.array([0.5, 0.7])
    assert s2.error_parts(x, np.array([3.0]), np.zeros(2), np.zeros(2), np.zeros(2), np.array([0.2]),
                          np.array([[1.0, 1.0]])) == (3.0, 0.2, 0.0)
    st2 = s2.initialise(x, None)
    tr = s2.iterate(st2, None)
    assert tr["E0"] <= 1.0 and tr["acc"] == 0 and st2.status == ipm.ST_NOT_RUN   # E_0 = 0.2 acceptable, |c| = 0.2 is not
    s3 = ipm.Solver(p, [-INF, -INF], [INF, INF], ipm.Options(acceptable_tol=1.0, acceptable_iter=1, acceptable_constr_viol_tol=0.5))
    st3 = s3.initialise(x, None)
    s3.iterate(st3, None)
    assert st3.status == ipm.ST_ACCEPTABLE and st3.k == 0
