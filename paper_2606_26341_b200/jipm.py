"""Thin ctypes binding of the C ABI in include/jipm.h (argument marshalling only).

PyTorch is used for device memory and the CUDA stream, nothing else: every step of the interior-point
iteration runs in the hand-written kernels of ``csrc/``.  There is no CPU fallback: if ``libjipm.so`` is
missing, importing the symbols raises; if no CUDA device is present, ``jipm_create`` returns JIPM_ERR_CUDA.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libjipm.so")

TRACE_W = 22
ST_NOT_RUN, ST_SOLVED, ST_MAXITER, ST_LOCALLY_INFEASIBLE = -1, 0, 1, 2
ST_RESTORATION_FAILED, ST_RESTO_AT_FEASIBLE_POINT, ST_NONFINITE, ST_TINY_STEP = 3, 4, 5, 6
ST_ACCEPTABLE = 7

_DOUBLE_FIELDS = [
    "tol", "mu_init", "kappa_eps", "kappa_mu", "theta_mu", "tau_min", "s_max", "kappa_sigma",
    "kappa_1", "kappa_2", "bound_relax_factor", "bound_mult_init", "lam_init_max", "kappa_d",
    "gamma_theta", "gamma_phi", "eta_phi", "delta", "s_theta", "s_phi", "gamma_alpha",
    "theta_max_fact", "theta_min_fact", "alpha_red", "kappa_soc",
    "delta_w_min", "delta_w_0", "delta_w_max", "kappa_w_minus", "kappa_w_plus", "kappa_w_plus_first",
    "delta_c_bar", "kappa_c", "residual_ratio_max", "rho_resto", "kappa_resto", "z_reset_threshold",
    "residual_ratio_singular", "residual_improvement_factor",
    "tiny_step_tol", "tiny_step_y_tol", "tiny_step_cviol", "soft_resto_factor",
    "adaptive_red_fact", "adaptive_monotone_init", "adaptive_sigma_max", "adaptive_mu_max_fact",
    "acceptable_tol", "acceptable_dual_inf_tol", "acceptable_constr_viol_tol", "acceptable_compl_inf_tol"]
_INT_FIELDS = ["max_iter", "max_backtrack", "max_soc", "refine_min", "refine_max", "max_mu_updates",
               "init_slacks", "enable_restoration", "watchdog_trigger", "watchdog_trial_max", "max_soft_resto_iters",
               "mu_strategy", "adaptive_red_iters", "acceptable_iter"]
_INT_LAYOUT = _INT_FIELDS[:-3] + ["polish_max"] + _INT_FIELDS[-3:]   # order of the int32 members in jipm_options


class Options(C.Structure):
    _fields_ = [(f, C.c_double) for f in _DOUBLE_FIELDS] + [(f, C.c_int32) for f in _INT_LAYOUT]


class FamilyDims(C.Structure):
    _fields_ = [("horizon_N", C.c_int32), ("n_agents", C.c_int32), ("n_obstacles", C.c_int32), ("dt", C.c_double)]


_lib = None

EXPORTS = ["jipm_default_options", "jipm_family_sizes", "jipm_create", "jipm_solve_batch",
           "jipm_solve_batch_host", "jipm_destroy", "jipm_last_error", "jipm_last_stats",
           "jipm_debug_set_trace", "jipm_debug_state_layout", "jipm_debug_step", "jipm_debug_init",
           "jipm_bench_fp64_peak", "jipm_residency", "jipm_solve_batch_static"]

STATIC_SCRATCH_BYTES = 64 << 20   # JIPM_STATIC_SCRATCH_BYTES of include/jipm.h


def lib():
    """Load libjipm.so (built by __graft_entry__.build()); fails loudly when it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                               "(jipm has no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i64, dp, ip = C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p
        L.jipm_default_options.argtypes = [C.POINTER(Options)]
        L.jipm_family_sizes.argtypes = [C.c_int, C.POINTER(FamilyDims), C.POINTER(i64), C.POINTER(i64), C.POINTER(i64)]
        L.jipm_create.argtypes = [C.POINTER(vp), C.c_int, C.POINTER(FamilyDims), i64, i64, dp, dp,
                                  C.POINTER(Options), i64, vp]
        L.jipm_solve_batch.argtypes = [vp, i64, dp, dp, dp, dp, dp, dp, ip, ip]
        L.jipm_solve_batch_host.argtypes = [vp, i64, dp, dp, dp, dp, dp, dp, ip, ip]
        L.jipm_destroy.argtypes = [vp]
        L.jipm_last_error.restype = C.c_char_p
        L.jipm_last_stats.argtypes = [vp, C.POINTER(i64), i64]
        L.jipm_debug_set_trace.argtypes = [vp, dp, i64]
        L.jipm_debug_state_layout.argtypes = [vp, C.POINTER(i64), i64]
        L.jipm_debug_step.argtypes = [vp, i64, dp, dp, i64]
        L.jipm_debug_init.argtypes = [vp, i64, dp, dp, dp]
        L.jipm_bench_fp64_peak.argtypes = [vp, C.POINTER(C.c_double)]
        L.jipm_residency.argtypes = [vp, C.POINTER(i64)]
        L.jipm_solve_batch_static.argtypes = [C.c_int, C.POINTER(FamilyDims), i64, i64, dp, dp, C.POINTER(Options), vp,
                                              i64, dp, dp, dp, dp, dp, dp, ip, ip]
        _lib = L
    return _lib


class JipmError(RuntimeError):
    pass


def _check(rc):
    if rc != 0:
        raise JipmError(f"jipm error {rc}: {lib().jipm_last_error().decode()}")


def default_options() -> Options:
    o = Options()
    _check(lib().jipm_default_options(C.byref(o)))
    return o


def family_sizes(family: int, horizon_N: int, n_agents: int, n_obstacles: int, dt: float):
    d = FamilyDims(horizon_N, n_agents, n_obstacles, dt)
    n, m, nt = C.c_int64(), C.c_int64(), C.c_int64()
    _check(lib().jipm_family_sizes(family, C.byref(d), C.byref(n), C.byref(m), C.byref(nt)))
    return n.value, m.value, nt.value


def fp64_peak_tflops() -> float:
    import torch
    v = C.c_double()
    _check(lib().jipm_bench_fp64_peak(C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(v)))
    return v.value


def solve_batch_static(family, horizon_N, n_agents, n_obstacles, dt, xL, xU, x0, params, out, opts: Options | None = None):
    """jipm_solve_batch_static: the solve without any allocation inside the library (scratch in a static device array
    of STATIC_SCRATCH_BYTES).  x0 [P,n], params [P,n_theta] and the tensors of `out` (x, lam, status, iters and
    optionally zL, zU) are CUDA tensors the caller owns; xL, xU host arrays."""
    import torch
    d = FamilyDims(horizon_N, n_agents, n_obstacles, dt)
    n, m, _ = family_sizes(family, horizon_N, n_agents, n_obstacles, dt)
    xL = np.ascontiguousarray(xL, dtype=np.float64)
    xU = np.ascontiguousarray(xU, dtype=np.float64)
    assert xL.shape == (n,) and xU.shape == (n,)
    zl = out["zL"].data_ptr() if "zL" in out else None
    zu = out["zU"].data_ptr() if "zU" in out else None
    _check(lib().jipm_solve_batch_static(family, C.byref(d), n, m, xL.ctypes.data, xU.ctypes.data,
                                         C.byref(opts) if opts is not None else None,
                                         C.c_void_p(torch.cuda.current_stream().cuda_stream), x0.shape[0],
                                         x0.data_ptr(), params.data_ptr(), out["x"].data_ptr(), out["lam"].data_ptr(),
                                         zl, zu, out["status"].data_ptr(), out["iters"].data_ptr()))


class Solver:
    """jipm_create / jipm_solve_batch / jipm_destroy with torch tensors for device memory."""

    LAY_NAMES = ["len", "x", "y", "zL", "zU", "sc", "filt", "dx", "dy", "dzL", "dzU", "g", "c", "J", "W",
                 "rs", "pn", "zpn", "xR", "filtR", "ls", "wd"]

    def __init__(self, family, horizon_N, n_agents, n_obstacles, dt, xL, xU, opts: Options | None = None,
                 resident_slots: int = 0):
        import torch
        self.torch = torch
        self.dims = FamilyDims(horizon_N, n_agents, n_obstacles, dt)
        self.n, self.m, self.n_theta = family_sizes(family, horizon_N, n_agents, n_obstacles, dt)
        xL = np.ascontiguousarray(xL, dtype=np.float64)
        xU = np.ascontiguousarray(xU, dtype=np.float64)
        self._h = C.c_void_p()
        stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
        _check(lib().jipm_create(C.byref(self._h), family, C.byref(self.dims), self.n, self.m,
                                 xL.ctypes.data, xU.ctypes.data, C.byref(opts) if opts is not None else None,
                                 resident_slots, C.c_void_p(stream)))
        self._trace = None

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value and _lib is not None:
            _lib.jipm_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def _dev(self, a, dtype=None):
        t = self.torch
        if not isinstance(a, t.Tensor):
            a = t.as_tensor(np.ascontiguousarray(a))
        a = a.to(device="cuda", dtype=dtype or t.float64).contiguous()
        return a

    def solve_batch(self, x0, params, want_z=True):
        """x0 [P,n], params [P,n_theta] (numpy or cuda tensors) -> dict of cuda tensors."""
        t = self.torch
        x0, params = self._dev(x0), self._dev(params)
        P = x0.shape[0]
        assert x0.shape == (P, self.n) and params.shape == (P, self.n_theta)
        out = dict(x=t.empty((P, self.n), dtype=t.float64, device="cuda"),
                   lam=t.empty((P, self.m), dtype=t.float64, device="cuda"),
                   status=t.full((P,), -1, dtype=t.int32, device="cuda"),
                   iters=t.zeros((P,), dtype=t.int32, device="cuda"))
        if want_z:
            out["zL"] = t.empty((P, self.n), dtype=t.float64, device="cuda")
            out["zU"] = t.empty((P, self.n), dtype=t.float64, device="cuda")
        self.solve_batch_into(x0, params, out)
        return out

    def solve_batch_into(self, x0, params, out):
        """Same, with caller-provided device tensors (no allocation: the form bench.py times)."""
        P = x0.shape[0]
        zl = out["zL"].data_ptr() if "zL" in out else None
        zu = out["zU"].data_ptr() if "zU" in out else None
        _check(lib().jipm_solve_batch(self._h, P, x0.data_ptr(), params.data_ptr(), out["x"].data_ptr(),
                                      out["lam"].data_ptr(), zl, zu, out["status"].data_ptr(),
                                      out["iters"].data_ptr()))

    def solve_batch_host(self, x0, params, out=None):
        """HOST numpy buffers in and out (host<->device copies inside the call)."""
        x0 = np.ascontiguousarray(x0, dtype=np.float64)
        params = np.ascontiguousarray(params, dtype=np.float64)
        P = x0.shape[0]
        if out is None:
            out = dict(x=np.empty((P, self.n)), lam=np.empty((P, self.m)), zL=np.empty((P, self.n)),
                       zU=np.empty((P, self.n)), status=np.empty(P, np.int32), iters=np.empty(P, np.int32))
        _check(lib().jipm_solve_batch_host(self._h, P, x0.ctypes.data, params.ctypes.data, out["x"].ctypes.data,
                                           out["lam"].ctypes.data, out["zL"].ctypes.data, out["zU"].ctypes.data,
                                           out["status"].ctypes.data, out["iters"].ctypes.data))
        return out

    def stats(self):
        a = (C.c_int64 * 24)()
        _check(lib().jipm_last_stats(self._h, a, 24))
        names = ["iterations", "factorisations", "kkt_solves", "deriv_evals", "fc_evals", "slots", "launches",
                 "resto_iterations", "cyc_derivs", "cyc_factor", "cyc_solve", "cyc_residual", "cyc_trial_eval",
                 "cyc_iterations", "cyc_init", "cyc_speculative_trials",
                 "cycf_TJ", "cycf_M", "cycf_pivots", "cycf_phi_store", "cycf_dc_extra", "cycx_solve_full_first", "cycx_line_search", "cycx_iteration_head"]
        d = dict(zip(names, list(a)))
        d["co_resident_slots"] = min(d["slots"], self.co_resident_slots())
        return d

    def co_resident_slots(self):
        """Problem slots (CTAs) the device holds at once for this family: SMs x teams per SM."""
        a = (C.c_int64 * 2)()
        _check(lib().jipm_residency(self._h, a))
        return int(a[0] * a[1])

    # ---- debug / parity entries ------------------------------------------------------------------------
    def set_trace(self, P, max_records):
        t = self.torch
        if P == 0:
            self._trace = None
            _check(lib().jipm_debug_set_trace(self._h, None, 0))
            return None
        self._trace = t.zeros((P, max_records, TRACE_W), dtype=t.float64, device="cuda")
        _check(lib().jipm_debug_set_trace(self._h, self._trace.data_ptr(), max_records))
        return self._trace

    def state_layout(self):
        a = (C.c_int64 * 22)()
        _check(lib().jipm_debug_state_layout(self._h, a, 22))
        return dict(zip(self.LAY_NAMES, list(a)))

    def debug_init(self, x0, params):
        t = self.torch
        x0, params = self._dev(x0), self._dev(params)
        P = x0.shape[0]
        st = t.zeros((P, self.state_layout()["len"]), dtype=t.float64, device="cuda")
        _check(lib().jipm_debug_init(self._h, P, x0.data_ptr(), params.data_ptr(), st.data_ptr()))
        return st

    def debug_step(self, params, state, n_steps=1):
        params = self._dev(params)
        assert state.is_cuda and state.is_contiguous()
        _check(lib().jipm_debug_step(self._h, state.shape[0], params.data_ptr(), state.data_ptr(), n_steps))
        return state
