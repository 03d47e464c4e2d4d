"""Helpers of the GPU-vs-oracle parity tests: run the oracle on seeded problems, decode the GPU decision trace,
and compare the two with the metrics of BASELINE.json's north_star (SURVEY.md 8(c) "Parity metrics"):
  (i)   KKT step residual of the unreduced system (6) <= 1e-10 relative,
  (ii)  step parity e_v of eq (8) <= 1e-8,
  (iii) identical iteration counts and acceptance decisions on >= 99 % of problems,
  (iv)  x* within 1e-6 relative and scaled KKT error E_0 <= 1e-8 on every converged problem.
Nothing here is imported by the product path."""
from __future__ import annotations

import numpy as np

from oracle import families as ofam
from oracle import ipm as oipm

KIND_CODE = {"newton": 0, "soc": 1, "ls_fail": 2, "ic_fail": 3, "": 4, "tiny": 5, "soft": 6}
# GPU trace record columns (include/jipm.h)
T_MODE, T_NFACT, T_DW, T_DC, T_NREF, T_KIND, T_LS, T_SOC, T_ALPHA, T_ALPHAZ, T_FTYPE, T_NMU, T_E0, T_MU = range(14)
T_THETA, T_PHI, T_WD, T_SOFT, T_TINY, T_NPSING, T_MUMODE, T_MUSWITCH = 14, 15, 16, 17, 18, 19, 20, 21


def oracle_for(d, xL, xU, opts=None):
    prob = ofam.Problem(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt)
    return prob, oipm.Solver(prob, xL, xU, opts)


def oracle_solve(d, xL, xU, x0, theta, opts=None):
    """Solve every row with the oracle; returns list of (State, trace)."""
    prob, s = oracle_for(d, xL, xU, opts)
    out = []
    for i in range(x0.shape[0]):
        tr = []
        st = s.solve(x0[i], theta[i], tr)
        out.append((st, tr))
    return out


def e_v(v, vref):
    """Step-parity metric of eq (8): max_i |v_i - vref_i| / (1 + |vref_i|)."""
    v, vref = np.asarray(v, float), np.asarray(vref, float)
    if v.size == 0:
        return 0.0
    return float(np.max(np.abs(v - vref) / (1.0 + np.abs(vref))))


def decisions_equal(gpu_rec: np.ndarray, otr: dict) -> tuple[bool, str]:
    """One iteration: every integer decision must be identical -- step kind, mode, #mu updates, #factorisations, the
    perturbations delta_w AND delta_c, #refinement failures treated as singular, #backtracks, #corrections, the
    watchdog / soft-restoration / tiny-step codes, f- or h-type -- and the step lengths agree to 1e-4 relative (the
    iterates are compared tightly by the step-parity tests; here the reals only guard against a different branch).
    The NUMBER of refinement steps is a property of the linear solver, not a decision of the method (two LAPACK
    solvers differ in it too): it is reported by the tests, not asserted."""
    kind = KIND_CODE[otr["kind"]]
    if int(gpu_rec[T_KIND]) != kind:
        return False, f"kind {int(gpu_rec[T_KIND])} vs {kind}"
    if int(gpu_rec[T_MODE]) != int(otr.get("mode", 0)):
        return False, "mode"
    if kind == 4:
        return True, ""
    if int(gpu_rec[T_NMU]) != otr["nmu"]:
        return False, f"nmu {int(gpu_rec[T_NMU])} vs {otr['nmu']}"
    for col, key in ((T_MUMODE, "mu_mode"), (T_MUSWITCH, "mu_switch")):
        if int(gpu_rec[col]) != int(otr.get(key, 0)):
            return False, f"{key} {int(gpu_rec[col])} vs {otr.get(key, 0)}"
    if kind == 3:
        return True, ""
    if int(gpu_rec[T_NFACT]) != otr["nfact"]:
        return False, f"nfact {int(gpu_rec[T_NFACT])} vs {otr['nfact']}"
    if int(gpu_rec[T_NPSING]) != otr.get("npsing", 0):
        return False, f"npsing {int(gpu_rec[T_NPSING])} vs {otr.get('npsing', 0)}"
    if not np.isclose(gpu_rec[T_DW], otr["dw"], rtol=1e-9, atol=0.0):
        return False, f"dw {gpu_rec[T_DW]} vs {otr['dw']}"
    if not np.isclose(gpu_rec[T_DC], otr["dc"], rtol=1e-9, atol=0.0):
        return False, f"dc {gpu_rec[T_DC]} vs {otr['dc']}"
    for col, key in ((T_WD, "wd"), (T_SOFT, "soft"), (T_TINY, "tiny")):
        if int(gpu_rec[col]) != int(otr.get(key, 0)):
            return False, f"{key} {int(gpu_rec[col])} vs {otr.get(key, 0)}"
    if int(gpu_rec[T_LS]) != otr["ls"]:
        return False, f"ls {int(gpu_rec[T_LS])} vs {otr['ls']}"
    if int(gpu_rec[T_SOC]) != otr["soc"]:
        return False, f"soc {int(gpu_rec[T_SOC])} vs {otr['soc']}"
    if kind == 2:
        return True, ""
    if bool(gpu_rec[T_FTYPE]) != bool(otr["ftype"]):
        return False, "ftype"
    if not np.isclose(gpu_rec[T_ALPHA], otr["alpha"], rtol=1e-4, atol=1e-12):
        return False, f"alpha {gpu_rec[T_ALPHA]} vs {otr['alpha']}"
    if not np.isclose(gpu_rec[T_ALPHAZ], otr["alpha_z"], rtol=1e-4, atol=1e-12):
        return False, f"alpha_z {gpu_rec[T_ALPHAZ]} vs {otr['alpha_z']}"
    return True, ""


def iterate_gap(solver, lin, d):
    """e_v (eq 8) between the iterates two solutions of the same step produce when each takes ITS OWN
    largest step the line search considers: x + alpha_max(d) dx and y + alpha_max(d) dy with alpha_max from the
    fraction-to-the-boundary rule (the step length inherits the rounding of dx, and y moves by alpha_max dy)."""
    ref, x, tau = lin["d"], lin["x"], lin["tau"]
    a_ref = solver.ftb_primal(x, ref[0], tau)
    a_new = solver.ftb_primal(x, d[0], tau)
    gap = e_v(x + a_new * d[0], x + a_ref * ref[0])
    if solver.m:
        gap = max(gap, e_v(a_new * d[1], a_ref * ref[1]))
    return gap if np.isfinite(gap) else np.inf


class LUFactor:
    """numpy/scipy LU with partial pivoting behind the interface of oracle.linsolve.DenseLDL.solve."""

    def __init__(self, K):
        import scipy.linalg
        self._sl = scipy.linalg
        self.lu = scipy.linalg.lu_factor(K)

    def solve(self, b):
        return self._sl.lu_solve(self.lu, b)


def second_opinion_gap(solver, tr):
    """How far two LAPACK solvers disagree on the linear system of this iteration: the oracle's Bunch-Kaufman LDL^T
    against an LU with partial pivoting, both followed by the same refinement on (6) (reading S-7).  Measured with
    iterate_gap: e_v of eq (8) on the iterates the largest step the line search considers would produce.  A step on which two backward-stable library solvers already differ by more than the parity
    tolerance cannot be asked of a third one: such steps are reported, not asserted."""
    lin = tr.get("lin")
    if lin is None:
        return 0.0
    K = solver.kkt_matrix(lin["W"], lin["Sigma"], lin["A"], tr["dw"], tr["dc"])
    if not np.all(np.isfinite(K)):
        return np.inf
    try:
        d, _, _ = solver.solve_full(LUFactor(K), lin["W"], lin["A"], lin["x"], lin["zL"], lin["zU"], tr["dw"], tr["dc"],
                                    lin["b"])
    except Exception:
        return np.inf
    return iterate_gap(solver, lin, d)


def perturbed_derivatives(solver, lin, rel, rng):
    """W, A with the error two independent fp64 derivative codes leave in them.  A: relative `rel` per structural
    non-zero (e_v style: rel (1 + |A_ij|)).  W = sigma_f Hess f + sum_j y_j Hess c_j is a SUM of terms weighted by the
    multipliers: each TERM carries a relative rounding error, so the error of an entry scales with the multipliers that
    feed it, whatever the size of the entry (terms cancel).  Modelled exactly that way: the oracle's Hessian is
    re-evaluated with every multiplier y_j replaced by y_j (1 + rel u_j), u_j ~ U(-1, 1), and every entry gets a relative
    `rel` on top."""
    W, A = lin["W"], lin["A"]
    y = lin["y"]
    yp = y * (1.0 + rel * rng.uniform(-1.0, 1.0, y.shape))
    Wy = solver.p.hess_lag(lin["x"], lin["th"], yp, 1.0)
    E = rng.uniform(-1.0, 1.0, W.shape)
    Wp = Wy * (1.0 + rel * (E + E.T) / 2.0)
    Ap = A + rel * (1.0 + np.abs(A)) * rng.uniform(-1.0, 1.0, A.shape) * (A != 0.0)
    return Wp, Ap


def sensitivity_gap(solver, tr, rel=1e-12, seed=1):
    """How far the step of this iteration moves when the computed derivative blocks W and A carry the rounding error of
    another fp64 derivative code (perturbed_derivatives with rel = 1e-12: every multiplier-weighted term of W and every
    entry of A off by a relative 1e-12; the oracle's jets and the kernel's analytic RK4 chain agree to 1e-11 in A and
    1e-10 max(1, ||y||) in W: test_derivative_blocks_against_oracle asserts that, a hundred times looser).
    Same solver (Bunch-Kaufman + refinement), same right-hand side; measured like second_opinion_gap.  Where this
    exceeds the parity tolerance the step amplifies differences below the resolution of the derivatives by more than
    1e4: no implementation with its own derivative code can reproduce it to 1e-8."""
    from oracle.linsolve import DenseLDL
    lin = tr.get("lin")
    if lin is None:
        return 0.0
    rng = np.random.default_rng(seed)
    Wp, Ap = perturbed_derivatives(solver, lin, rel, rng)
    K = solver.kkt_matrix(Wp, lin["Sigma"], Ap, tr["dw"], tr["dc"])
    if not np.all(np.isfinite(K)):
        return np.inf
    try:
        d, _, _ = solver.solve_full(DenseLDL(K), Wp, Ap, lin["x"], lin["zL"], lin["zU"], tr["dw"], tr["dc"], lin["b"])
    except Exception:
        return np.inf
    return iterate_gap(solver, lin, d)


def residual_rounding_gap(solver, tr, ulps=4.0, seed=2):
    """How far the step moves when the right-hand side of (6) carries the rounding error ANY fp64 evaluation leaves in
    it: the constraint residual c(x) is a difference of numbers of size |A| |x| and the dual residual grad f + A^T y - z_L
    + z_U a sum of terms of size |A|^T |y| + z_L + z_U, so each component is known to a few ulps of those magnitudes, not of
    its own (the standard componentwise model, `ulps` = 4).  Same matrix, same solver, right-hand side perturbed by
    ulps eps u (|A| |x| + |c|) and ulps eps u (|A|^T |y| + z_L + z_U + |b_1|), u ~ U(-1, 1); measured like
    second_opinion_gap.  Matters when the primal iterate has converged to rounding level (theta = 2e-13) while delta_w
    is 1e12 ... 1e16: dy = delta_w (A A^T)^-1 c + ... then IS the rounding noise of c times delta_w (seen with the adaptive
    barrier strategy on the reduced workload-3 problem 2, iterations 178-187: the two codes evaluate theta = 2.39e-13 and
    2.82e-13 at the same point and the multiplier steps differ by 1e3)."""
    from oracle.linsolve import DenseLDL
    lin = tr.get("lin")
    if lin is None:
        return 0.0
    rng = np.random.default_rng(seed)
    eps = 2.220446049250313e-16
    A, b = lin["A"], lin["b"]
    s1 = np.abs(A).T @ np.abs(lin["y"]) + lin["zL"] + lin["zU"] + np.abs(b[0]) if solver.m else lin["zL"] + lin["zU"] + np.abs(b[0])
    bp = [b[0] + ulps * eps * s1 * rng.uniform(-1.0, 1.0, b[0].shape)]
    if solver.m:
        s2 = np.abs(A) @ np.abs(lin["x"]) + np.abs(b[1])
        bp.append(b[1] + ulps * eps * s2 * rng.uniform(-1.0, 1.0, b[1].shape))
    else:
        bp.append(b[1])
    bp += [b[2], b[3]]
    K = solver.kkt_matrix(lin["W"], lin["Sigma"], A, tr["dw"], tr["dc"])
    if not np.all(np.isfinite(K)):
        return np.inf
    try:
        d, _, _ = solver.solve_full(DenseLDL(K), lin["W"], A, lin["x"], lin["zL"], lin["zU"], tr["dw"], tr["dc"], bp)
    except Exception:
        return np.inf
    return iterate_gap(solver, lin, d)


def step_is_well_posed(solver, tr, tol):
    """(well-posed?, text): the criteria above with the parity tolerance, plus the rounding floor of the step itself:
    e_v (eq 8) is a COMPONENTWISE measure, and a solver that is backward stable in the usual normwise sense delivers every
    component of the step to within a few ulps of the LARGEST component of (dx, dy, dz_L, dz_U) -- the refinement of
    reading S-7 stops on the common max-norm of the four blocks.  When 8 eps alpha_max ||step||_inf already exceeds the
    tolerance, the small components of the next iterate cannot be asked to 1e-8 (seen on restoration steps with delta_w
    1e9: ||dy||_inf = 5e8, differences of 2e-6 on multipliers of size 200, i.e. 4e-14 of ||dy||; and on steps with an
    active slack, Sigma = 1e10: dz = 1e10, the multiplier of the inequality is a difference of nearly equal numbers
    times 1e10)."""
    lin = tr.get("lin")
    if lin is not None:
        a_ref = solver.ftb_primal(lin["x"], lin["d"][0], lin["tau"])
        big = max(float(np.max(np.abs(v))) if v.size else 0.0 for v in lin["d"])   # all four blocks: the refinement of
        floor = 8.0 * 2.220446049250313e-16 * a_ref * big                          # reading S-7 stops on their common norm
        if not np.isfinite(floor) or floor > tol:
            return False, f"8 eps alpha_max ||step||_inf = {floor:.1e}"
    g1 = second_opinion_gap(solver, tr)
    if g1 > tol:
        return False, f"LAPACK LU vs Bunch-Kaufman {g1:.1e}"
    g2 = sensitivity_gap(solver, tr)
    if g2 > tol:
        return False, f"rounding-level perturbation of W, A moves the step by {g2:.1e}"
    g3 = residual_rounding_gap(solver, tr)
    if g3 > tol:
        return False, f"rounding of the residuals c, grad L (4 ulps of their terms) moves the step by {g3:.1e}"
    if len((tr.get("lin") or {}).get("tried", [])) > 1 and not inertia_is_stable(solver, tr):
        return False, "inertia changes under a rounding-level perturbation of W, A"
    return True, f"{max(g1, g2, g3):.1e}"


class WithGpuDerivatives:
    """A problem that answers like `base` except that, AT THE POINT x_at, the dynamics blocks of its Jacobian and the
    stage blocks of its Lagrangian Hessian are the ones the GPU evaluated (taken from the debug state).  Lets the oracle's
    iteration run on exactly the matrices the kernel factorised: what is left between the two results is linear
    algebra and line-search logic, with the rounding of the two derivative codes (asserted separately, block by block,
    in test_derivative_blocks_against_oracle) taken out."""

    def __init__(self, base, x_at, Jg, Wg, WNg):
        self.base, self.x_at, self.Jg, self.Wg, self.WNg = base, np.array(x_at), Jg, Wg, WNg
        for name in ("n", "m", "N", "nx", "nu", "ng", "na", "family", "dt", "ax", "au", "pdim"):
            if hasattr(base, name):
                setattr(self, name, getattr(base, name))

    def __getattr__(self, name):
        return getattr(self.base, name)

    def _here(self, x):
        return x.shape == self.x_at.shape and np.array_equal(x, self.x_at)

    def jac(self, x, th):
        A = self.base.jac(x, th)
        if self._here(x):
            b, nx, nu = self.base, self.base.nx, self.base.nu
            for k in range(1, b.N + 1):
                r = b.ic_dyn(k)
                A[r:r + nx, b.ix(k - 1):b.ix(k - 1) + nx] = -self.Jg[k - 1][:, :nx]
                A[r:r + nx, b.iu(k - 1):b.iu(k - 1) + nu] = -self.Jg[k - 1][:, nx:]
        return A

    def hess_lag(self, x, th, y, sigma_f=1.0):
        W = self.base.hess_lag(x, th, y, sigma_f)
        if self._here(x):
            b, nx, nu = self.base, self.base.nx, self.base.nu
            for k in range(b.N):
                rows = list(range(b.ix(k), b.ix(k) + nx)) + list(range(b.iu(k), b.iu(k) + nu))
                W[np.ix_(rows, rows)] = self.Wg[k]
            rows = list(range(b.ix(b.N), b.ix(b.N) + nx))
            W[np.ix_(rows, rows)] = self.WNg
        return W


def oracle_step_with_gpu_derivatives(osol, st_copy, theta, gpu_state, lay, d):
    """Run ONE oracle iteration from st_copy (a deep copy of the oracle's state before the step) with the GPU's
    derivative blocks substituted at the current point; returns (trace, state after)."""
    import copy
    n, N, nx, nz = d.n, d.horizon_N, d.nx, d.nx + d.nu
    Jg = gpu_state[lay["J"]:lay["J"] + N * nx * nz].reshape(N, nx, nz)
    Wg = gpu_state[lay["W"]:lay["W"] + N * nz * nz].reshape(N, nz, nz)
    WNg = gpu_state[lay["W"] + N * nz * nz:lay["W"] + N * nz * nz + nx * nx].reshape(nx, nx)
    sol = copy.copy(osol)
    if st_copy.resto is None:
        sol.p = WithGpuDerivatives(osol.p, st_copy.x, Jg, Wg, WNg)
    else:
        sub = copy.copy(st_copy.resto.sub)
        rp = copy.copy(sub.p)
        rp.base = WithGpuDerivatives(rp.base, st_copy.resto.state.x[:n], Jg, Wg, WNg)
        sub.p = rp
        st_copy.resto.sub = sub
    tr = sol.iterate(st_copy, theta)
    return tr, st_copy


def inertia_is_stable(solver, tr, rel=1e-12, seed=0):
    """Is every inertia Algorithm IC read in this iteration (one per factorisation it tried) the same for a matrix whose
    derivative blocks carry another code's rounding error (perturbed_derivatives)?  If not, the sequence of
    perturbations delta_w is not a property of the problem but of the rounding."""
    from oracle.linsolve import DenseLDL
    lin = tr.get("lin")
    if lin is None:
        return True
    rng = np.random.default_rng(seed)
    W, A = lin["W"], lin["A"]
    Wp, Ap = perturbed_derivatives(solver, lin, rel, rng)
    for dw, dc in lin["tried"]:
        K0 = solver.kkt_matrix(W, lin["Sigma"], A, dw, dc)
        K1 = solver.kkt_matrix(Wp, lin["Sigma"], Ap, dw, dc)
        if not (np.all(np.isfinite(K0)) and np.all(np.isfinite(K1))):
            return False
        if DenseLDL(K0).inertia != DenseLDL(K1).inertia:
            return False
    return True


def compare_problem(gpu_trace: np.ndarray, gpu_status: int, gpu_iters: int, st, otr: list):
    """Returns (same, first_diverging_iteration, reason).  gpu_trace: [max_records, TRACE_W]."""
    if gpu_status != st.status:
        reason = f"status {gpu_status} vs {st.status}"
    elif gpu_iters != st.k:
        reason = f"iters {gpu_iters} vs {st.k}"
    else:
        reason = ""
    nrec = min(len(otr), gpu_trace.shape[0])
    for j in range(nrec):
        ok, why = decisions_equal(gpu_trace[j], otr[j])
        if not ok:
            return False, j, why
    if reason:
        return False, nrec, reason
    return True, -1, ""


def rel_x_err(xg, xo):
    return float(np.max(np.abs(xg - xo)) / max(1.0, np.max(np.abs(xo))))


def oracle_E0(prob, osol, x, y, zL, zU, theta):
    """Scaled KKT error E_0 recomputed by the oracle's functions at a (GPU) point."""
    return osol.opt_error(x, y, zL, zU, prob.grad_f(x, theta), prob.c(x, theta), prob.jac(x, theta), 0.0)


def full_system_residual(prob, osol, x, y, zL, zU, theta, mu, dw, dc, step):
    """Relative residual of the four block rows of (6) (with the perturbations of PAPER.md:114)
    at the iterate (x, y, z), with W, A, c, grad f from the ORACLE and the step from the GPU."""
    dx, dy, dzL, dzU = step
    W, A = prob.hess_lag(x, theta, y, 1.0), prob.jac(x, theta)
    g, cv = prob.grad_f(x, theta), prob.c(x, theta)
    sL, sU = osol.slacks(x)
    b = [-(g + A.T @ y - zL + zU + osol.damping(mu)), -cv,
         np.where(osol.hasL, mu - sL * zL, 0.0), np.where(osol.hasU, mu - sU * zU, 0.0)]
    lhs = osol.full_matvec(W, A, x, zL, zU, dw, dc, (dx, dy, dzL, dzU))
    rn = max(float(np.max(np.abs(bi - li))) for bi, li in zip(b, lhs))
    bn = max(float(np.max(np.abs(v))) for v in b)
    sn = max(float(np.max(np.abs(v))) for v in (dx, dy, dzL, dzU))
    return rn / (bn + sn)


def prune_filter(filt):
    """Drop entries dominated by a later one (decision-neutral, reading S-10) so that the oracle's unbounded list
    fits the GPU filter capacity (256)."""
    out = []
    for (t, p) in filt:
        out = [(a, b) for (a, b) in out if not (a >= t and b >= p)]
        out.append((t, p))
    return out


def snapshot_state(lay, st, n, m):
    """Full state of the oracle before an iteration, in the layout of jipm_debug_state_layout (either mode)."""
    snap = np.zeros(lay["len"])

    def put_filter(key, filt):
        f = prune_filter(filt)
        assert len(f) <= 256, len(f)
        for j, (t, p) in enumerate(f):
            snap[lay[key] + 2 * j], snap[lay[key] + 2 * j + 1] = t, p
        return len(f)

    nreg = put_filter("filt", st.filt)
    if st.resto is None:
        cur = st
        snap[lay["x"]:lay["x"] + n], snap[lay["zL"]:lay["zL"] + n], snap[lay["zU"]:lay["zU"] + n] = st.x, st.zL, st.zU
        nf = nreg
    else:  # Step R: the restoration iterate X = [x; p; n] with its own scalars and filter, the regular ones parked
        cur, rp = st.resto.state, st.resto.sub.p
        snap[lay["x"]:lay["x"] + n], snap[lay["pn"]:lay["pn"] + 2 * m] = cur.x[:n], cur.x[n:]
        snap[lay["zL"]:lay["zL"] + n], snap[lay["zpn"]:lay["zpn"] + 2 * m] = cur.zL[:n], cur.zL[n:]
        snap[lay["zU"]:lay["zU"] + n] = cur.zU[:n]
        snap[lay["xR"]:lay["xR"] + n] = rp.xR
        snap[lay["rs"]:lay["rs"] + 9] = [1, st.mu, st.tau, st.delta_w_last, st.theta_min, st.theta_max, nreg,
                                         st.resto.theta_entry, rp.zeta]
        nf = put_filter("filtR", cur.filt)
    snap[lay["y"]:lay["y"] + m] = cur.y
    snap[lay["sc"]:lay["sc"] + 8] = [cur.mu, cur.tau, cur.delta_w_last, cur.theta_min, cur.theta_max, st.k, -1, nf]
    # line-search memory of the active problem (Table I rows 3-5) and the watchdog's entry iterate and direction
    wd = cur.wd
    snap[lay["ls"]:lay["ls"] + 11] = [cur.n_short, int(wd is not None), wd.trials if wd else 0, wd.theta if wd else 0.0,
                                      wd.phi if wd else 0.0, wd.gd if wd else 0.0, wd.alpha if wd else 0.0,
                                      int(cur.soft), cur.soft_count, int(cur.tiny_last), int(cur.tiny_flag)]
    hist = list(cur.kkt_hist)
    snap[lay["ls"] + 11:lay["ls"] + 14] = [int(cur.mu_free), cur.mu_max, len(hist)]
    for j in range(max(0, len(hist) - 4), len(hist)):
        snap[lay["ls"] + 14 + (j & 3)] = hist[j]
    snap[lay["ls"] + 18] = cur.acc_count
    if wd is not None:
        nw, o = n + 2 * m, lay["wd"]
        for q, v in enumerate((wd.x, wd.zL, wd.zU, wd.d[0], wd.d[2], wd.d[3])):
            snap[o + q * nw:o + q * nw + v.size] = v
        snap[o + 6 * nw:o + 6 * nw + m] = wd.y
        snap[o + 6 * nw + m:o + 6 * nw + 2 * m] = wd.d[1]
    return snap


def ls_memory(st):
    """(n_short, watchdog active, watchdog trials, soft, soft_count, tiny_last, tiny_flag, acceptable count) of the active problem."""
    cur = st if st.resto is None else st.resto.state
    return [cur.n_short, int(cur.wd is not None), cur.wd.trials if cur.wd else 0, int(cur.soft), cur.soft_count,
            int(cur.tiny_last), int(cur.tiny_flag), cur.acc_count]
