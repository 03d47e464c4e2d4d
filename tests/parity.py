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

KIND_CODE = {"newton": 0, "soc": 1, "ls_fail": 2, "ic_fail": 3, "": 4}
# GPU trace record columns (include/jipm.h)
T_MODE, T_NFACT, T_DW, T_DC, T_NREF, T_KIND, T_LS, T_SOC, T_ALPHA, T_ALPHAZ, T_FTYPE, T_NMU, T_E0, T_MU = range(14)


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
    """One iteration: the integer decisions must be identical; the step lengths agree to 1e-4 relative (iterates
    are compared tightly by the step-parity tests; here the reals only guard against a different branch)."""
    kind = KIND_CODE[otr["kind"]]
    if int(gpu_rec[T_KIND]) != kind:
        return False, f"kind {int(gpu_rec[T_KIND])} vs {kind}"
    if int(gpu_rec[T_MODE]) != int(otr.get("mode", 0)):
        return False, "mode"
    if kind == 4:
        return True, ""
    if int(gpu_rec[T_NMU]) != otr["nmu"]:
        return False, f"nmu {int(gpu_rec[T_NMU])} vs {otr['nmu']}"
    if kind == 3:
        return True, ""
    if int(gpu_rec[T_NFACT]) != otr["nfact"]:
        return False, f"nfact {int(gpu_rec[T_NFACT])} vs {otr['nfact']}"
    if not np.isclose(gpu_rec[T_DW], otr["dw"], rtol=1e-9, atol=0.0):
        return False, f"dw {gpu_rec[T_DW]} vs {otr['dw']}"
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
    return snap
