"""ORACLE (test infrastructure, not the product).  A plain, slow, sequential fp64 implementation of the
interior-point iteration of arxiv 2606.26341 section IV: barrier problem (3), iterate
(x, y_c, z_L, z_U) and Lagrangian (4), Newton system (6), augmented system (7) with inertia-correcting
perturbations (delta_w, delta_c), and the Table I fallbacks the hot path covers
(PAPER.md:118-142): backtracking line search (row 1), second-order correction (row 2), watchdog (row 3),
tiny-step rule (row 4), soft feasibility restoration (row 5), hard feasibility restoration (row 6),
monotone barrier update (row 7).  The paper defers every constant and the filter/restoration details to
its reference [7] (Waechter & Biegler 2006); the readings taken are listed in DESIGN.md "Readings" and
all constants live in ``Options``.

The oracle follows the algorithm step by step (Step I = initialise, Step A = one iteration, Step R =
restoration) on DENSE matrices: the Newton step is the solution of the dense
system (7) by Bunch-Kaufman LDL^T (oracle/linsolve.py), Delta z from PAPER.md:110, refinement on the full
unreduced system (6).  Restoration is the same iteration applied, recursively, to the restoration NLP
written out as an NLP (no elimination of p, n).  Nothing here is shared with the CUDA path.

Parity status: every function below is pinned by tests/test_oracle_*.py (closed forms, hand-computed cases,
independent library routines).  What stays "parity unpinned": the VALUES of the constants
recalled from IPOPT's release (gamma_phi, eta_phi, kappa_d, the watchdog / soft-restoration / tiny-step
thresholds) and the choice of readings R-1, R-2, S-15 of Step R -- the mechanics of each reading are pinned,
that IPOPT takes the same reading cannot be checked here ([7] and IPOPT are not available).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

from .linsolve import DenseLDL

ST_NOT_RUN, ST_SOLVED, ST_MAXITER, ST_LOCALLY_INFEASIBLE = -1, 0, 1, 2
ST_RESTORATION_FAILED, ST_RESTO_AT_FEASIBLE_POINT, ST_NONFINITE, ST_TINY_STEP = 3, 4, 5, 6
ST_ACCEPTABLE = 7
EPS = 2.220446049250313e-16


@dataclass
class Options:
    tol: float = 1e-8
    max_iter: int = 3000
    mu_init: float = 0.1
    kappa_eps: float = 10.0
    kappa_mu: float = 0.2
    theta_mu: float = 1.5
    tau_min: float = 0.99
    s_max: float = 100.0
    kappa_sigma: float = 1e10
    kappa_1: float = 1e-2
    kappa_2: float = 1e-2
    bound_relax_factor: float = 1e-8
    bound_mult_init: float = 1.0
    lam_init_max: float = 1e3
    kappa_d: float = 1e-5
    gamma_theta: float = 1e-5
    gamma_phi: float = 1e-8
    eta_phi: float = 1e-8
    delta: float = 1.0
    s_theta: float = 1.1
    s_phi: float = 2.3
    gamma_alpha: float = 0.05
    theta_max_fact: float = 1e4
    theta_min_fact: float = 1e-4
    alpha_red: float = 0.5
    max_backtrack: int = 64
    max_soc: int = 4
    kappa_soc: float = 0.99
    delta_w_min: float = 1e-20
    delta_w_0: float = 1e-4
    delta_w_max: float = 1e40
    kappa_w_minus: float = 1.0 / 3.0
    kappa_w_plus: float = 8.0
    kappa_w_plus_first: float = 100.0
    delta_c_bar: float = 1e-8
    kappa_c: float = 0.25
    refine_min: int = 1
    refine_max: int = 10
    residual_ratio_max: float = 1e-10
    rho_resto: float = 1000.0
    kappa_resto: float = 0.9
    z_reset_threshold: float = 1e3
    max_mu_updates: int = 8
    zero_pivot_tol: float = 0.0
    init_slacks: int = 1
    enable_restoration: int = 1
    # iterative refinement / "pretend singular" (reading S-7)
    residual_ratio_singular: float = 1e-5
    residual_improvement_factor: float = 0.999999999
    # Table I rows 3-5 (readings W, T, SR of DESIGN.md section 3)
    watchdog_trigger: int = 10        # consecutive shortened steps that wake the watchdog (0 = off)
    watchdog_trial_max: int = 3       # trial steps accepted unconditionally before reverting
    tiny_step_tol: float = 10.0 * 2.220446049250313e-16
    tiny_step_y_tol: float = 1e-2
    tiny_step_cviol: float = 1e-4
    soft_resto_factor: float = 1.0 - 1e-4   # required reduction of the primal-dual error (0 = off)
    max_soft_resto_iters: int = 10
    # Table I row 7 (reading AM of DESIGN.md section 3): 0 = monotone schedule (IPOPT's default),
    # 1 = adaptive barrier parameter (Mehrotra probing) with the switch to the monotone schedule
    mu_strategy: int = 0
    adaptive_red_fact: float = 0.9999       # required reduction of the KKT error w.r.t. the last adaptive_red_iters
    adaptive_red_iters: int = 4
    adaptive_monotone_init: float = 0.8     # mu of the monotone phase = this x average complementarity
    adaptive_sigma_max: float = 100.0
    adaptive_mu_max_fact: float = 1e3       # mu never exceeds this x the first average complementarity
    # acceptable-level termination (NEXT-4; IPOPT feature, not in the paper: reading AT, off by default): stop after
    # acceptable_iter consecutive regular iterations whose E_0 <= acceptable_tol and whose unscaled dual residual,
    # constraint violation and complementarity stay below the three bounds
    acceptable_tol: float = 1e-6
    acceptable_dual_inf_tol: float = 1e10
    acceptable_constr_viol_tol: float = 1e-2
    acceptable_compl_inf_tol: float = 1e-2
    acceptable_iter: int = 0                # IPOPT's default is 15; 0 = off

    @property
    def mu_min(self) -> float:
        return self.tol / 10.0


@dataclass
class State:
    x: np.ndarray
    y: np.ndarray
    zL: np.ndarray
    zU: np.ndarray
    mu: float
    tau: float
    delta_w_last: float = 0.0
    filt: list = field(default_factory=list)
    theta_min: float = 0.0
    theta_max: float = 0.0
    k: int = 0
    status: int = ST_NOT_RUN
    resto: "RestoContext | None" = None
    n_short: int = 0                  # consecutive iterations whose accepted step needed backtracking
    wd: "Watchdog | None" = None      # watchdog in progress (Table I row 3)
    soft: bool = False                # in the soft restoration phase (Table I row 5)
    soft_count: int = 0
    tiny_last: bool = False           # the previous iteration took a tiny step (Table I row 4)
    tiny_flag: bool = False           # two tiny steps in a row: force a barrier decrease at the next A-3
    mu_free: bool = True              # adaptive strategy (Table I row 7): free mode (True) or monotone phase
    kkt_hist: list = field(default_factory=list)   # KKT errors of the last accepted free-mode iterates
    mu_max: float = -1.0              # upper bound of the adaptive mu (set at the first iteration)
    acc_count: int = 0                # consecutive acceptable iterations (reading AT)


@dataclass
class Watchdog:
    """Entry iterate of the watchdog, its search direction and the reference values of the acceptance test."""
    x: np.ndarray
    y: np.ndarray
    zL: np.ndarray
    zU: np.ndarray
    d: tuple
    theta: float
    phi: float
    gd: float
    alpha: float
    trials: int = 0


def relax_bounds(xL, xU, o: Options):
    """Step I-1: finite bounds relaxed by bound_relax_factor*max(1,|b|) ([7] sec 3.5, recalled)."""
    xL, xU = np.array(xL, dtype=np.float64), np.array(xU, dtype=np.float64)
    fl, fu = np.isfinite(xL), np.isfinite(xU)
    xL[fl] -= o.bound_relax_factor * np.maximum(1.0, np.abs(xL[fl]))
    xU[fu] += o.bound_relax_factor * np.maximum(1.0, np.abs(xU[fu]))
    return xL, xU


class Solver:
    """Holds one NLP (duck-typed: n, m, f, grad_f, c, jac, hess_lag, optional set_mu) with its bounds."""

    def __init__(self, prob, xL, xU, opts: Options | None = None, relax: bool = True):
        self.p = prob
        self.o = opts or Options()
        self.xL, self.xU = relax_bounds(xL, xU, self.o) if relax else (np.array(xL, float), np.array(xU, float))
        if np.any(self.xL >= self.xU):
            raise ValueError("x_L >= x_U")  # PAPER.md:63 requires a strict interior
        self.hasL, self.hasU = np.isfinite(self.xL), np.isfinite(self.xU)
        self.onlyL, self.onlyU = self.hasL & ~self.hasU, self.hasU & ~self.hasL
        self.nL, self.nU = int(self.hasL.sum()), int(self.hasU.sum())
        self.n, self.m = prob.n, prob.m

    # ---- barrier objective (3) and its gradient, with the one-sided damping of [7] sec 3.7 ------------
    def slacks(self, x):
        sL = np.where(self.hasL, x - np.where(self.hasL, self.xL, 0.0), 1.0)
        sU = np.where(self.hasU, np.where(self.hasU, self.xU, 0.0) - x, 1.0)
        return sL, sU

    def phi(self, x, fval, mu):
        sL, sU = self.slacks(x)
        if np.any(sL <= 0) or np.any(sU <= 0):
            return math.nan
        val = fval
        val -= mu * float(np.sum(np.log(sL[self.hasL])))
        val -= mu * float(np.sum(np.log(sU[self.hasU])))
        val += self.o.kappa_d * mu * float(np.sum(sL[self.onlyL]))
        val += self.o.kappa_d * mu * float(np.sum(sU[self.onlyU]))
        return val

    def damping(self, mu):
        return self.o.kappa_d * mu * (self.onlyL.astype(float) - self.onlyU.astype(float))

    def grad_phi(self, x, g, mu):
        sL, sU = self.slacks(x)
        return g - mu * self.hasL / sL + mu * self.hasU / sU + self.damping(mu)

    # ---- optimality error E_mu ([7] eq 5, recalled; reading S-3 for the denominators) -----------------
    def opt_error(self, x, y, zL, zU, g, cval, A, mu):
        o = self.o
        sL, sU = self.slacks(x)
        rd = g + A.T @ y - zL + zU + self.damping(mu)
        comp = np.concatenate([(sL * zL - mu)[self.hasL], (sU * zU - mu)[self.hasU]])
        nz = self.nL + self.nU
        zsum = float(np.sum(np.abs(zL)) + np.sum(np.abs(zU)))
        sd = max(o.s_max, (float(np.sum(np.abs(y))) + zsum) / (self.m + nz)) / o.s_max if self.m + nz > 0 else 1.0
        sc = max(o.s_max, zsum / nz) / o.s_max if nz > 0 else 1.0
        e_d = float(np.max(np.abs(rd))) / sd if rd.size else 0.0
        e_c = float(np.max(np.abs(cval))) if cval.size else 0.0
        e_s = float(np.max(np.abs(comp))) / sc if comp.size else 0.0
        return max(e_d, e_c, e_s)

    def error_parts(self, x, y, zL, zU, g, cval, A):
        """Unscaled max-norms of the three blocks of (5) at mu = 0: dual residual, constraint
        violation, complementarity."""
        sL, sU = self.slacks(x)
        rd = g + A.T @ y - zL + zU
        comp = np.concatenate([(sL * zL)[self.hasL], (sU * zU)[self.hasU]])
        return (float(np.max(np.abs(rd))) if rd.size else 0.0, float(np.max(np.abs(cval))) if cval.size else 0.0,
                float(np.max(np.abs(comp))) if comp.size else 0.0)

    # ---- fraction to the boundary (PAPER.md:148 fn 2; [7] eq 15) --------------------------------------
    def ftb_primal(self, x, dx, tau):
        sL, sU = self.slacks(x)
        a = 1.0
        for i in range(self.n):
            if self.hasL[i] and dx[i] < 0:
                a = min(a, -tau * sL[i] / dx[i])
            if self.hasU[i] and dx[i] > 0:
                a = min(a, tau * sU[i] / dx[i])
        return a

    def ftb_dual(self, zL, zU, dzL, dzU, tau):
        a = 1.0
        for i in range(self.n):
            if self.hasL[i] and dzL[i] < 0:
                a = min(a, -tau * zL[i] / dzL[i])
            if self.hasU[i] and dzU[i] < 0:
                a = min(a, -tau * zU[i] / dzU[i])
        return a

    # ---- Step I ------------------------------------------------------------------------------------
    def initialise(self, x0, th) -> State:
        o, p = self.o, self.p
        x = np.array(x0, dtype=np.float64)
        if o.init_slacks and hasattr(p, "init_slacks"):
            x = p.init_slacks(x, th)  # I-2
        x = self.push_interior(x)  # I-3
        zL = np.where(self.hasL, o.bound_mult_init, 0.0)  # I-4
        zU = np.where(self.hasU, o.bound_mult_init, 0.0)
        if hasattr(p, "set_mu"):
            p.set_mu(o.mu_init)
        y = self.least_squares_multipliers(x, th, zL, zU)  # I-5
        mu = o.mu_init  # I-6
        st = State(x=x, y=y, zL=zL, zU=zU, mu=mu, tau=max(o.tau_min, 1.0 - mu))
        theta0 = float(np.sum(np.abs(p.c(x, th)))) if self.m else 0.0  # I-7
        st.theta_max = o.theta_max_fact * max(1.0, theta0)
        st.theta_min = o.theta_min_fact * max(1.0, theta0)
        return st

    def push_interior(self, x):
        o = self.o
        x = x.copy()
        for i in range(self.n):
            l, u = self.xL[i], self.xU[i]
            if self.hasL[i] and self.hasU[i]:
                pl = min(o.kappa_1 * max(1.0, abs(l)), o.kappa_2 * (u - l))
                pu = min(o.kappa_1 * max(1.0, abs(u)), o.kappa_2 * (u - l))
                x[i] = min(max(x[i], l + pl), u - pu)
            elif self.hasL[i]:
                x[i] = max(x[i], l + o.kappa_1 * max(1.0, abs(l)))
            elif self.hasU[i]:
                x[i] = min(x[i], u - o.kappa_1 * max(1.0, abs(u)))
        return x

    def least_squares_multipliers(self, x, th, zL, zU):
        """I-5: [[I, A^T],[A, 0]] [w; y] = -[grad f - z_L + z_U; 0]; y <- 0 if too large ([7] sec 3.6)."""
        if self.m == 0:
            return np.zeros(0)
        n, m = self.n, self.m
        A = self.p.jac(x, th)
        K = np.zeros((n + m, n + m))
        K[:n, :n] = np.eye(n)
        K[n:, :n] = A
        K[:n, n:] = A.T
        rhs = np.concatenate([-(self.p.grad_f(x, th) - zL + zU), np.zeros(m)])
        fac = DenseLDL(K, self.o.zero_pivot_tol)
        if fac.inertia != (n, m, 0):
            return np.zeros(m)
        y = fac.solve(rhs)[n:]
        if not np.all(np.isfinite(y)) or np.max(np.abs(y)) > self.o.lam_init_max:
            return np.zeros(m)
        return y

    # ---- the linear algebra of one iteration ---------------------------------------------------------
    def kkt_matrix(self, W, Sigma, A, dw, dc):
        """Augmented matrix of eq (7) with the perturbations of PAPER.md:114."""
        n, m = self.n, self.m
        K = np.zeros((n + m, n + m))
        K[:n, :n] = W + np.diag(Sigma + dw)
        K[n:, :n] = A
        K[:n, n:] = A.T
        K[n:, n:] = -dc * np.eye(m)
        return K

    def inertia_correction(self, W, Sigma, A, mu, dw_last, resume=None):
        """Algorithm IC ([7] sec 3.1, recalled).  Returns (factor, dw, dc, nfact) or None.

        ``resume=(dw, dc)``: the factorisation with these perturbations had the right inertia but the solve with it
        failed the refinement test ("pretend singular", reading S-7): the matrix is treated like one with a zero
        eigenvalue -- delta_c takes its IC-2 value, delta_w moves to the next rung of the ladder (IC-3 from 0,
        else IC-5) -- and the loop IC-4..IC-6 continues from there."""
        o, n, m = self.o, self.n, self.m
        nfact = 0
        tried = self.ic_tried = getattr(self, "ic_tried", [])   # (delta_w, delta_c) of every factorisation, for tests
        if resume is None:
            tried.clear()
            fac = DenseLDL(self.kkt_matrix(W, Sigma, A, 0.0, 0.0), o.zero_pivot_tol)  # IC-1
            nfact = 1
            tried.append((0.0, 0.0))
            if fac.inertia == (n, m, 0):
                return fac, 0.0, 0.0, nfact
            dc = o.delta_c_bar * mu ** o.kappa_c if fac.inertia[2] > 0 else 0.0  # IC-2
            dw = o.delta_w_0 if dw_last == 0.0 else max(o.delta_w_min, o.kappa_w_minus * dw_last)  # IC-3
        else:
            dw, dc = resume
            dc = o.delta_c_bar * mu ** o.kappa_c
            if dw == 0.0:
                dw = o.delta_w_0 if dw_last == 0.0 else max(o.delta_w_min, o.kappa_w_minus * dw_last)
            else:
                dw = (o.kappa_w_plus_first if dw_last == 0.0 else o.kappa_w_plus) * dw
                if dw > o.delta_w_max:
                    return None
        while True:
            fac = DenseLDL(self.kkt_matrix(W, Sigma, A, dw, dc), o.zero_pivot_tol)  # IC-4
            nfact += 1
            tried.append((dw, dc))
            if fac.inertia == (n, m, 0):
                return fac, dw, dc, nfact
            dw = (o.kappa_w_plus_first if dw_last == 0.0 else o.kappa_w_plus) * dw  # IC-5
            if dw > o.delta_w_max:  # IC-6
                return None

    def full_matvec(self, W, A, x, zL, zU, dw, dc, d):
        """Left-hand side of the unreduced Newton system (6) applied to d."""
        dx, dy, dzL, dzU = d
        sL, sU = self.slacks(x)
        r1 = W @ dx + dw * dx + A.T @ dy - dzL + dzU
        r2 = A @ dx - dc * dy
        r3 = np.where(self.hasL, zL * dx + sL * dzL, 0.0)
        r4 = np.where(self.hasU, -zU * dx + sU * dzU, 0.0)
        return r1, r2, r3, r4

    def solve_full(self, fac, W, A, x, zL, zU, dw, dc, b):
        """Solve (6) for right-hand side b=(b1,b2,b3,b4) through the augmented system (7) and the Delta z
        recovery of PAPER.md:110, then refine on (6) (reading S-7)."""
        o = self.o
        sL, sU = self.slacks(x)
        n = self.n

        def reduced_solve(b1, b2, b3, b4):
            r = b1 + np.where(self.hasL, b3 / sL, 0.0) - np.where(self.hasU, b4 / sU, 0.0)
            s = fac.solve(np.concatenate([r, b2]))
            dx, dy = s[:n], s[n:]
            dzL = np.where(self.hasL, (b3 - zL * dx) / sL, 0.0)
            dzU = np.where(self.hasU, (b4 + zU * dx) / sU, 0.0)
            return [dx, dy, dzL, dzU]

        def ratio(d):
            lhs = self.full_matvec(W, A, x, zL, zU, dw, dc, d)
            res = [bi - li for bi, li in zip(b, lhs)]
            rnorm = max(float(np.max(np.abs(v))) if v.size else 0.0 for v in res)
            dnorm = max(float(np.max(np.abs(v))) if v.size else 0.0 for v in d)
            den = bnorm + dnorm
            return res, (rnorm / den if den > 0.0 else rnorm)

        d = reduced_solve(*b)
        bnorm = max(float(np.max(np.abs(v))) if v.size else 0.0 for v in b)
        res, rat = ratio(d)
        nref, failed = 0, False
        # at least refine_min steps; stop at ratio <= residual_ratio_max; give up when refine_max is exceeded or
        # a step no longer improves the ratio -- then the solution is kept if the ratio is below
        # residual_ratio_singular, else the solve is reported as FAILED (the caller pretends the matrix is singular)
        while rat > o.residual_ratio_max or nref < o.refine_min:
            if not math.isfinite(rat):
                failed = True
                break
            corr = reduced_solve(*res)
            d = [di + ci for di, ci in zip(d, corr)]
            nref += 1
            rat_old = rat
            res, rat = ratio(d)
            if rat > o.residual_ratio_max and nref > o.refine_min and (
                    nref >= o.refine_max or rat > o.residual_improvement_factor * rat_old):
                failed = not (rat < o.residual_ratio_singular)
                break
        return d, nref, failed

    # ---- filter acceptance ([7] sec 2.3) -----------------------------------------
    def switching(self, alpha, g, theta_k):
        o = self.o
        return g < 0.0 and alpha * (-g) ** o.s_phi > o.delta * theta_k ** o.s_theta

    def armijo(self, phi_t, phi_k, alpha, g):
        return phi_t - phi_k - 10.0 * EPS * abs(phi_k) <= self.o.eta_phi * alpha * g

    def in_filter(self, st: State, theta_t, phi_t):
        if theta_t >= st.theta_max:
            return True
        return any(theta_t >= tj and phi_t >= pj for (tj, pj) in st.filt)

    def acceptable(self, st: State, theta_t, phi_t, theta_k, phi_k, alpha, g):
        o = self.o
        if not (math.isfinite(theta_t) and math.isfinite(phi_t)):
            return False
        if self.in_filter(st, theta_t, phi_t):
            return False
        if theta_k <= st.theta_min and self.switching(alpha, g, theta_k):
            return self.armijo(phi_t, phi_k, alpha, g)
        return (theta_t <= (1.0 - o.gamma_theta) * theta_k
                or phi_t - phi_k - 10.0 * EPS * abs(phi_k) <= -o.gamma_phi * theta_k)

    def trial_point(self, x, th, mu):
        fv = self.p.f(x, th)
        cv = self.p.c(x, th)
        theta = float(np.sum(np.abs(cv))) if cv.size else 0.0
        return fv, cv, theta, self.phi(x, fv, mu)

    def alpha_min(self, gd, theta_k, theta_min):
        """Smallest step length the backtracking line search tries before it gives up (A-5; [7] eq 23, recalled)."""
        o = self.o
        if gd < 0.0 and theta_k <= theta_min:
            return o.gamma_alpha * min(o.gamma_theta, o.gamma_phi * theta_k / (-gd),
                                       o.delta * theta_k ** o.s_theta / (-gd) ** o.s_phi)
        if gd < 0.0:
            return o.gamma_alpha * min(o.gamma_theta, o.gamma_phi * theta_k / (-gd))
        return o.gamma_alpha * o.gamma_theta

    def pd_error(self, x, y, zL, zU, g, cval, A, mu):
        """Error of the primal-dual system (5a-d) as the soft restoration phase measures it:
        the 1-norm of each block divided by its length, summed (reading SR)."""
        sL, sU = self.slacks(x)
        rd = g + A.T @ y - zL + zU + self.damping(mu)
        comp = np.concatenate([(sL * zL - mu)[self.hasL], (sU * zU - mu)[self.hasU]])
        e = float(np.sum(np.abs(rd))) / self.n
        if self.m:
            e += float(np.sum(np.abs(cval))) / self.m
        if comp.size:
            e += float(np.sum(np.abs(comp))) / comp.size
        return e

    # ---- Step A: one iteration ------------------------------------------------------------------------
    def iterate(self, st: State, th) -> dict:
        """Advance ``st`` by one iteration (regular or restoration mode); returns the decision trace."""
        if st.resto is not None:
            return self.iterate_resto(st, th)
        o, p, n, m = self.o, self.p, self.n, self.m
        tr = dict(mode=0, nfact=0, dw=0.0, dc=0.0, nref=0, kind="", ls=0, soc=0, alpha=0.0, alpha_z=0.0,
                  ftype=False, augment=False, nmu=0, status=ST_NOT_RUN, npsing=0, wd=0, soft=0, tiny=0)
        x, y = st.x, st.y
        # A-1 evaluate
        fv, g, cv, A = p.f(x, th), p.grad_f(x, th), p.c(x, th), p.jac(x, th)
        if not (math.isfinite(fv) and np.all(np.isfinite(g)) and np.all(np.isfinite(cv)) and np.all(np.isfinite(A))):
            st.status = tr["status"] = ST_NONFINITE
            return tr
        # A-2 termination
        e0 = self.opt_error(x, y, st.zL, st.zU, g, cv, A, 0.0)
        tr["E0"] = e0
        if e0 <= o.tol:
            st.status = tr["status"] = ST_SOLVED
            return tr
        if o.acceptable_iter > 0 and not hasattr(p, "set_mu"):   # reading AT; never inside the restoration sub-solver
            d_inf, c_inf, s_inf = self.error_parts(x, y, st.zL, st.zU, g, cv, A)
            ok = (e0 <= o.acceptable_tol and d_inf <= o.acceptable_dual_inf_tol and c_inf <= o.acceptable_constr_viol_tol
                  and s_inf <= o.acceptable_compl_inf_tol)
            st.acc_count = st.acc_count + 1 if ok else 0
            tr["acc"] = st.acc_count
            if st.acc_count >= o.acceptable_iter:
                st.status = tr["status"] = ST_ACCEPTABLE
                return tr
        if st.k >= o.max_iter:
            st.status = tr["status"] = ST_MAXITER
            return tr
        # A-3 monotone barrier update (Table I row 7: the monotone schedule).  Two tiny steps in a
        # row (Table I row 4) force one decrease; if mu cannot decrease any more the search direction has become
        # too small to make progress: TINY_STEP.
        force = st.tiny_flag
        st.tiny_flag = False
        adaptive = o.mu_strategy == 1 and not hasattr(p, "set_mu") and (self.nL + self.nU) > 0
        tr["mu_mode"], tr["mu_switch"] = 0, 0
        if adaptive:
            # Table I row 7: the adaptive rule runs while the KKT error keeps falling ("free mode");
            # when an iterate fails to reduce it below adaptive_red_fact x the largest of the last adaptive_red_iters
            # values, the monotone schedule takes over from mu = adaptive_monotone_init x average complementarity
            # until its barrier problem is solved; then the adaptive rule returns.
            sLc, sUc = self.slacks(x)
            avg = (float(np.sum((sLc * st.zL)[self.hasL])) + float(np.sum((sUc * st.zU)[self.hasU]))) / (self.nL + self.nU)
            kkt = self.pd_error(x, y, st.zL, st.zU, g, cv, A, 0.0)
            if st.mu_max < 0.0:
                st.mu_max = o.adaptive_mu_max_fact * avg
            if st.mu_free:
                hist = st.kkt_hist[-o.adaptive_red_iters:]
                if hist and kkt > o.adaptive_red_fact * max(hist):
                    st.mu_free = False
                    st.mu = min(st.mu_max, max(o.mu_min, o.adaptive_monotone_init * avg))
                    st.tau = max(o.tau_min, 1.0 - st.mu)
                    st.filt = []
                    st.wd, st.n_short, st.soft, st.soft_count = None, 0, False, 0
                    tr["mu_switch"] = 1
                else:
                    st.kkt_hist = hist + [kkt]
            elif self.opt_error(x, y, st.zL, st.zU, g, cv, A, st.mu) <= o.kappa_eps * st.mu:
                st.mu_free = True
                st.kkt_hist = [kkt]
                tr["mu_switch"] = 2
            tr["mu_mode"] = 1 if st.mu_free else 2
        while not adaptive and tr["nmu"] < o.max_mu_updates and (
                force or self.opt_error(x, y, st.zL, st.zU, g, cv, A, st.mu) <= o.kappa_eps * st.mu):
            if not st.mu > o.mu_min:
                if force:
                    st.status = tr["status"] = ST_TINY_STEP
                    return tr
                break
            force = False
            st.mu = max(o.mu_min, min(o.kappa_mu * st.mu, st.mu ** o.theta_mu))
            st.tau = max(o.tau_min, 1.0 - st.mu)
            st.filt = []
            # a new barrier problem: the watchdog, its counter and the soft restoration phase start afresh
            st.wd, st.n_short, st.soft, st.soft_count = None, 0, False, 0
            tr["nmu"] += 1
            if hasattr(p, "set_mu"):
                p.set_mu(st.mu)
                fv, g = p.f(x, th), p.grad_f(x, th)
        W = p.hess_lag(x, th, y, 1.0)
        # A-4 search direction
        sL, sU = self.slacks(x)
        Sigma = np.where(self.hasL, st.zL / sL, 0.0) + np.where(self.hasU, st.zU / sU, 0.0)
        resume, probed = None, False
        while True:
            ic = self.inertia_correction(W, Sigma, A, st.mu, st.delta_w_last, resume)
            if ic is None:
                tr["kind"] = "ic_fail"
                tr["nfact"] = tr["nref"] = 0
                tr["dw"] = tr["dc"] = 0.0
                return self.enter_restoration(st, th, tr, fv, cv)
            fac, dw, dc, nf = ic
            tr["nfact"] += nf
            if adaptive and st.mu_free and not probed:
                # Mehrotra's probing with the factorisation of this iteration (it does not depend on mu): the
                # affine-scaling step is the Newton step on (5) with mu = 0; mu_aff = average complementarity after
                # the largest step that stays feasible; sigma = (mu_aff / average complementarity)^3; mu = sigma x avg.
                probed = True
                b_aff = [-(g + A.T @ y - st.zL + st.zU), -cv, np.where(self.hasL, -sL * st.zL, 0.0),
                         np.where(self.hasU, -sU * st.zU, 0.0)]
                da, _, _ = self.solve_full(fac, W, A, x, st.zL, st.zU, dw, dc, b_aff)
                a_p = self.ftb_primal(x, da[0], 1.0)
                a_d = self.ftb_dual(st.zL, st.zU, da[2], da[3], 1.0)
                mu_aff = (float(np.sum(((sL + a_p * da[0]) * (st.zL + a_d * da[2]))[self.hasL]))
                          + float(np.sum(((sU - a_p * da[0]) * (st.zU + a_d * da[3]))[self.hasU]))) / (self.nL + self.nU)
                sigma = min(o.adaptive_sigma_max, (mu_aff / avg) ** 3) if avg > 0.0 else 1.0
                tr["sigma"], tr["mu_aff"], tr["aff_step"] = sigma, mu_aff, da
                st.mu = min(st.mu_max, max(o.mu_min, sigma * avg))
                st.tau = max(o.tau_min, 1.0 - st.mu)
                st.filt = []
                st.wd, st.n_short, st.soft, st.soft_count = None, 0, False, 0
            mu, tau = st.mu, st.tau
            gphi = self.grad_phi(x, g, mu)
            b = [-(g + A.T @ y - st.zL + st.zU + self.damping(mu)), -cv,
                 np.where(self.hasL, mu - sL * st.zL, 0.0), np.where(self.hasU, mu - sU * st.zU, 0.0)]
            (dx, dy, dzL, dzU), tr["nref"], failed = self.solve_full(fac, W, A, x, st.zL, st.zU, dw, dc, b)
            if not failed:
                break
            tr["npsing"] += 1          # refinement failed: pretend the matrix is singular (reading S-7)
            resume = (dw, dc)
        tr["dw"], tr["dc"] = dw, dc
        if dw > 0.0:
            st.delta_w_last = dw
        tr["step"] = (dx, dy, dzL, dzU)
        # the linear system this step solved, for tests that want a second opinion on it (nothing below reads it)
        tr["lin"] = dict(W=W, A=A, Sigma=Sigma, b=b, x=x, y=y, th=th, tau=tau, zL=st.zL, zU=st.zU, d=(dx, dy, dzL, dzU),
                         tried=list(self.ic_tried))
        d = (dx, dy, dzL, dzU)
        # A-5 line search
        theta_k = float(np.sum(np.abs(cv))) if m else 0.0
        phi_k = self.phi(x, fv, mu)
        gd = float(gphi @ dx)
        a_max = self.ftb_primal(x, dx, tau)
        tr["theta"], tr["phi"], tr["gd"], tr["a_max"] = theta_k, phi_k, gd, a_max

        # Table I row 4: a step too small for backtracking to refine is accepted as it is
        xmax = float(np.max(np.abs(dx) / (1.0 + np.abs(x)))) if n else 0.0
        cmax = float(np.max(np.abs(cv))) if m else 0.0
        if xmax <= o.tiny_step_tol and cmax <= o.tiny_step_cviol:
            tr["tiny"] = 1
            if st.tiny_last and (float(np.max(np.abs(dy))) if m else 0.0) < o.tiny_step_y_tol:
                st.tiny_flag = True
            st.tiny_last = True
            xt = x + a_max * dx
            return self.accept(st, tr, dict(x=xt, d=d, alpha=a_max, kind="tiny"), mu, tau, ftype=True)
        st.tiny_last = False

        # Table I row 5: in the soft restoration phase the acceptance criterion is a
        # reduction of the primal-dual error, until the original criterion holds again or the limit is reached
        if st.soft:
            st.soft_count += 1
            if st.soft_count > o.max_soft_resto_iters:
                st.soft = False
                tr["kind"] = "ls_fail"
                return self.enter_restoration(st, th, tr, fv, cv)
            return self.soft_step(st, th, tr, d, mu, tau, fv, g, cv, A, theta_k, phi_k, gd)

        # Table I row 3: after watchdog_trigger shortened steps in a row the watchdog wakes up
        if st.wd is None and o.watchdog_trigger > 0 and st.n_short >= o.watchdog_trigger:
            st.wd = Watchdog(x=x.copy(), y=y.copy(), zL=st.zL.copy(), zU=st.zU.copy(), d=d,
                             theta=theta_k, phi=phi_k, gd=gd, alpha=a_max)
            tr["wd"] = 1
        if st.wd is not None:
            wd = st.wd
            xt = x + a_max * dx
            ft, ct, theta_t, phi_t = self.trial_point(xt, th, mu)
            if self.acceptable(st, theta_t, phi_t, wd.theta, wd.phi, wd.alpha, wd.gd):
                # the watchdog succeeded: the point is acceptable to the entry iterate's criterion
                ftype = self.switching(wd.alpha, wd.gd, wd.theta) and self.armijo(phi_t, wd.phi, wd.alpha, wd.gd)
                if not ftype:
                    st.filt.append(((1.0 - o.gamma_theta) * wd.theta, wd.phi - o.gamma_phi * wd.theta))
                st.wd, st.n_short = None, 0
                tr["wd"] = 3
                tr["augment"] = not ftype
                return self.accept(st, tr, dict(x=xt, d=d, alpha=a_max, kind="newton"), mu, tau, ftype=ftype)
            wd.trials += 1
            if wd.trials <= o.watchdog_trial_max and math.isfinite(theta_t) and math.isfinite(phi_t):
                if tr["wd"] == 0:
                    tr["wd"] = 2       # accepted unconditionally
                return self.accept(st, tr, dict(x=xt, d=d, alpha=a_max, kind="newton"), mu, tau, ftype=True)
            # the watchdog gives up: back to its entry iterate and direction, ordinary backtracking from there
            # (the full step of the entry iterate was tried when the watchdog started: skip it; no correction)
            st.x, st.y, st.zL, st.zU = wd.x, wd.y, wd.zL, wd.zU
            x, y, d = st.x, st.y, wd.d
            dx, dy, dzL, dzU = d
            theta_k, phi_k, gd, a_max = wd.theta, wd.phi, wd.gd, wd.alpha
            st.wd, st.n_short = None, 0
            tr["wd"] = 4
            tr["step"] = d
            fv, g, cv, A = p.f(x, th), p.grad_f(x, th), p.c(x, th), p.jac(x, th)
            acc = self.backtrack(st, th, tr, x, d, cv, None, mu, tau, theta_k, phi_k, gd, a_max, skip_first=True)
        else:
            acc = self.backtrack(st, th, tr, x, d, cv, (fac, W, A, dw, dc, b), mu, tau, theta_k, phi_k, gd, a_max,
                                 skip_first=False)
        if acc is None:
            # the line search failed: first the soft restoration phase (row 5), then the hard one (row 6)
            if o.soft_resto_factor > 0.0:
                st.soft, st.soft_count = True, 0
                st.filt.append(((1.0 - o.gamma_theta) * theta_k, phi_k - o.gamma_phi * theta_k))
                return self.soft_step(st, th, tr, d, mu, tau, fv, g, cv, A, theta_k, phi_k, gd)
            tr["kind"] = "ls_fail"
            return self.enter_restoration(st, th, tr, fv, cv)
        # A-6 accept, A-7 filter
        ftype = self.switching(acc["alpha_test"], gd, theta_k) and self.armijo(acc["phi"], phi_k, acc["alpha_test"], gd)
        if not ftype:
            st.filt.append(((1.0 - o.gamma_theta) * theta_k, phi_k - o.gamma_phi * theta_k))
        st.n_short = st.n_short + 1 if tr["ls"] > 0 else 0
        tr["augment"] = not ftype
        return self.accept(st, tr, acc, mu, tau, ftype=ftype)

    def backtrack(self, st, th, tr, x, d, cv, lin, mu, tau, theta_k, phi_k, gd, a_max, skip_first):
        """Backtracking line search with the second-order correction (Table I rows 1-2; A-5).
        ``lin`` = (factor, W, A, dw, dc, b) for the correction solves, or None (no correction).  Returns the
        accepted trial (dict) or None when alpha falls below alpha_min."""
        o = self.o
        dx = d[0]
        a_min = self.alpha_min(gd, theta_k, st.theta_min)
        tr["a_min"] = a_min
        alpha, ntrial = a_max, 0
        if skip_first:
            alpha *= o.alpha_red
            ntrial = 1
            if alpha < a_min:
                tr["ls"] = ntrial
                return None
        acc = None
        while True:
            xt = x + alpha * dx
            ft, ct, theta_t, phi_t = self.trial_point(xt, th, mu)
            if self.acceptable(st, theta_t, phi_t, theta_k, phi_k, alpha, gd):
                acc = dict(x=xt, d=d, alpha=alpha, alpha_test=alpha, phi=phi_t, kind="newton")
                break
            if (ntrial == 0 and lin is not None and math.isfinite(theta_t) and theta_t >= theta_k
                    and o.max_soc > 0):
                # second-order correction (Table I row 2; [7] sec 2.4)
                fac, W, A, dw, dc, b = lin
                c_soc = alpha * cv + ct
                theta_old = theta_k
                tr["soc_rhs"], tr["soc_steps"] = [], []
                for psoc in range(1, o.max_soc + 1):
                    bs = [b[0], -c_soc, b[2], b[3]]
                    ds, _, _ = self.solve_full(fac, W, A, x, st.zL, st.zU, dw, dc, bs)
                    a_soc = self.ftb_primal(x, ds[0], tau)
                    xs = x + a_soc * ds[0]
                    fs, cs, theta_s, phi_s = self.trial_point(xs, th, mu)
                    tr["soc"] = psoc
                    tr["soc_rhs"].append(c_soc.copy())
                    tr["soc_steps"].append(tuple(ds))
                    if self.acceptable(st, theta_s, phi_s, theta_k, phi_k, alpha, gd):
                        acc = dict(x=xs, d=tuple(ds), alpha=a_soc, alpha_test=alpha, phi=phi_s, kind="soc")
                        break
                    if not math.isfinite(theta_s) or theta_s > o.kappa_soc * theta_old:
                        break
                    theta_old = theta_s
                    c_soc = a_soc * c_soc + cs
                if acc is not None:
                    break
            alpha *= o.alpha_red
            ntrial += 1
            if alpha < a_min or ntrial > o.max_backtrack:
                break
        tr["ls"] = ntrial
        return acc

    def soft_step(self, st, th, tr, d, mu, tau, fv, g, cv, A, theta_k, phi_k, gd):
        """One step of the soft restoration phase (Table I row 5; reading SR): the same step
        length for primal and dual variables; accepted if the original criterion holds (then the phase ends) or
        if the primal-dual error drops by the factor soft_resto_factor; otherwise hard restoration."""
        o, p = self.o, self.p
        x, y = st.x, st.y
        dx, dy, dzL, dzU = d
        alpha = min(self.ftb_primal(x, dx, tau), self.ftb_dual(st.zL, st.zU, dzL, dzU, tau))
        xt = x + alpha * dx
        ft, ct, theta_t, phi_t = self.trial_point(xt, th, mu)
        ok = math.isfinite(theta_t) and math.isfinite(phi_t)
        orig = ok and self.acceptable(st, theta_t, phi_t, theta_k, phi_k, 0.0, gd)
        if ok and not orig:
            yt, zLt, zUt = y + alpha * dy, st.zL + alpha * dzL, st.zU + alpha * dzU
            gt, At = p.grad_f(xt, th), p.jac(xt, th)
            e_t = self.pd_error(xt, yt, zLt, zUt, gt, ct, At, mu)
            e_k = self.pd_error(x, y, st.zL, st.zU, g, cv, A, mu)
            ok = math.isfinite(e_t) and e_t <= o.soft_resto_factor * e_k
        if not ok:
            st.soft = False
            tr["kind"] = "ls_fail"
            return self.enter_restoration(st, th, tr, fv, cv)
        tr["soft"] = 2 if orig else 1
        if orig:
            st.soft, st.soft_count = False, 0
        st.n_short = 0
        return self.accept(st, tr, dict(x=xt, d=d, alpha=alpha, kind="soft"), mu, tau, ftype=True, alpha_z=alpha)

    def accept(self, st, tr, acc, mu, tau, ftype, alpha_z=None):
        """A-6 / A-8: move to the accepted trial point, step the multipliers, safeguard z, count the iteration."""
        dxa, dya, dzLa, dzUa = acc["d"]
        a_z = self.ftb_dual(st.zL, st.zU, dzLa, dzUa, tau) if alpha_z is None else alpha_z
        st.x = acc["x"]
        st.y = st.y + acc["alpha"] * dya
        st.zL = st.zL + a_z * dzLa
        st.zU = st.zU + a_z * dzUa
        self.safeguard_z(st, mu)
        st.k += 1  # A-8
        tr.update(kind=acc["kind"], alpha=acc["alpha"], alpha_z=a_z, ftype=ftype)
        return tr

    def safeguard_z(self, st: State, mu):
        """[7] eq (16): keep z within [mu/(kappa_Sigma s), kappa_Sigma mu / s]."""
        ks = self.o.kappa_sigma
        sL, sU = self.slacks(st.x)
        st.zL = np.where(self.hasL, np.maximum(np.minimum(st.zL, ks * mu / sL), mu / (ks * sL)), 0.0)
        st.zU = np.where(self.hasU, np.maximum(np.minimum(st.zU, ks * mu / sU), mu / (ks * sU)), 0.0)

    # ---- driver ----------------------------------------------------------------------------------------
    def solve(self, x0, th, trace: list | None = None):
        st = self.initialise(x0, th)
        while st.status == ST_NOT_RUN:
            tr = self.iterate(st, th)
            if trace is not None:
                trace.append(tr)
        return st

    # ---- Step R: hard feasibility restoration (Table I row 6; [7] sec 3.3) -----------
    def enter_restoration(self, st: State, th, tr, fv, cv):
        o = self.o
        theta_k = float(np.sum(np.abs(cv))) if self.m else 0.0
        if not o.enable_restoration or isinstance(self.p, RestoNLP):  # no nested restoration (A20)
            st.status = tr["status"] = ST_RESTORATION_FAILED
            return tr
        if theta_k < o.tol:
            st.status = tr["status"] = ST_RESTO_AT_FEASIBLE_POINT
            return tr
        phi_k = self.phi(st.x, fv, st.mu)
        st.filt.append(((1.0 - o.gamma_theta) * theta_k, phi_k - o.gamma_phi * theta_k))
        # the regular problem's line-search memory does not survive a restoration phase
        st.wd, st.n_short, st.soft, st.soft_count, st.tiny_last, st.tiny_flag = None, 0, False, 0, False, False
        st.acc_count = 0   # acceptable iterations must be consecutive REGULAR iterations
        mu_bar = max(st.mu, float(np.max(np.abs(cv))))
        rp = RestoNLP(self.p, st.x, o.rho_resto, mu_bar)
        n, m, rho = self.n, self.m, o.rho_resto
        # closed-form minimiser of the restoration barrier problem in (p, n) at fixed x ([7] eq 32-33)
        t = (mu_bar - rho * cv) / (2.0 * rho)
        nn = t + np.sqrt(t * t + mu_bar * cv / (2.0 * rho))
        pp = cv + nn
        X = np.concatenate([st.x, pp, nn])
        XL = np.concatenate([self.xL, np.zeros(2 * m)])
        XU = np.concatenate([self.xU, np.full(2 * m, np.inf)])
        sub = Solver(rp, XL, XU, o, relax=False)
        zL = np.concatenate([np.minimum(rho, st.zL), mu_bar / pp, mu_bar / nn])
        zU = np.concatenate([np.minimum(rho, st.zU), np.zeros(2 * m)])
        zL = np.where(sub.hasL, zL, 0.0)
        zU = np.where(sub.hasU, zU, 0.0)
        rs = State(x=X, y=np.zeros(m), zL=zL, zU=zU, mu=mu_bar, tau=max(o.tau_min, 1.0 - mu_bar))
        theta0 = float(np.sum(np.abs(rp.c(X, th))))
        rs.theta_max = o.theta_max_fact * max(1.0, theta0)
        rs.theta_min = o.theta_min_fact * max(1.0, theta0)
        st.resto = RestoContext(sub=sub, state=rs, theta_entry=theta_k)
        tr["status"] = ST_NOT_RUN
        tr["enter_resto"] = True
        st.k += 1  # the failed regular iteration counts (it did a factorisation and a line search)
        return tr

    def iterate_resto(self, st: State, th):
        o, rc = self.o, st.resto
        rs = rc.state
        rs.k = st.k  # so that max_iter applies to the total count (reading S-19)
        tr = rc.sub.iterate(rs, th)
        tr["mode"] = 1
        st.k = rs.k
        if rs.status == ST_SOLVED:
            # restoration problem converged without an acceptable point: local minimiser of the violation
            x = rs.x[:self.n]
            theta = float(np.sum(np.abs(self.p.c(x, th))))
            st.x = x
            st.status = tr["status"] = ST_LOCALLY_INFEASIBLE if theta > o.tol else ST_RESTO_AT_FEASIBLE_POINT
            return tr
        if rs.status != ST_NOT_RUN:
            st.status = tr["status"] = rs.status if rs.status in (ST_MAXITER, ST_NONFINITE) else ST_RESTORATION_FAILED
            st.x = rs.x[:self.n]
            return tr
        # exit test after an accepted restoration step
        x = rs.x[:self.n]
        fv, cv, theta, phi = self.trial_point(x, th, st.mu)
        if (math.isfinite(phi) and theta <= o.kappa_resto * rc.theta_entry
                and not self.in_filter(st, theta, phi)):
            st.x = x.copy()
            st.y = np.zeros(self.m)  # reading S-15 (parity unpinned)
            zL, zU = rs.zL[:self.n].copy(), rs.zU[:self.n].copy()
            if max(float(np.max(zL, initial=0.0)), float(np.max(zU, initial=0.0))) > o.z_reset_threshold:
                zL = np.where(self.hasL, 1.0, 0.0)
                zU = np.where(self.hasU, 1.0, 0.0)
            st.zL, st.zU = zL, zU
            st.resto = None
            tr["exit_resto"] = True
        return tr


@dataclass
class RestoContext:
    sub: Solver
    state: State
    theta_entry: float


class RestoNLP:
    """The restoration problem of [7] sec 3.3 written out as an NLP in X = [x; p; n]:
        min rho*sum(p+n) + zeta/2 * ||D_R (x - x_R)||^2   s.t.  c(x) - p + n = 0,  p, n >= 0,  x_L <= x <= x_U
    with zeta = sqrt(mu) following the restoration barrier parameter."""

    def __init__(self, base, x_R, rho, mu):
        self.base, self.xR, self.rho = base, np.array(x_R), rho
        self.DR2 = np.minimum(1.0, 1.0 / np.maximum(np.abs(self.xR), 1e-300)) ** 2
        self.nb, self.m = base.n, base.m
        self.n = base.n + 2 * base.m
        self.zeta = math.sqrt(mu)

    def set_mu(self, mu):
        self.zeta = math.sqrt(mu)

    def split(self, X):
        return X[:self.nb], X[self.nb:self.nb + self.m], X[self.nb + self.m:]

    def f(self, X, th):
        x, p, n = self.split(X)
        d = x - self.xR
        return self.rho * float(np.sum(p) + np.sum(n)) + 0.5 * self.zeta * float(np.sum(self.DR2 * d * d))

    def grad_f(self, X, th):
        x, p, n = self.split(X)
        return np.concatenate([self.zeta * self.DR2 * (x - self.xR), np.full(2 * self.m, self.rho)])

    def c(self, X, th):
        x, p, n = self.split(X)
        return self.base.c(x, th) - p + n

    def jac(self, X, th):
        x, p, n = self.split(X)
        I = np.eye(self.m)
        return np.hstack([self.base.jac(x, th), -I, I])

    def hess_lag(self, X, th, y, sigma_f=1.0):
        x, p, n = self.split(X)
        W = np.zeros((self.n, self.n))
        W[:self.nb, :self.nb] = self.base.hess_lag(x, th, y, 0.0) + sigma_f * self.zeta * np.diag(self.DR2)
        return W
