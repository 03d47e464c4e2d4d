"""The smallest run that takes every code path of the slot kernel, for compute-sanitizer (racecheck / synccheck /
memcheck):  compute-sanitizer --tool racecheck python tests/sanitizer_case.py
C0 batch 8, C1 batch 2 (full dimensions), reduced C1 with the watchdog forced, reduced C3 (restoration), the quaternion
family -- a few iterations each.  Prints one line per case; exits non-zero if a call fails."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from paper_2606_26341_b200 import jipm, workloads as wl  # noqa: E402

CASES = [("C0 batch 8", 0, {}, 8, 5, {}),
         ("C1 batch 2", 1, {}, 2, 5, {}),
         ("C1 reduced, watchdog after one shortened step", 1, dict(horizon_N=7), 4, 40, dict(watchdog_trigger=1)),
         ("C3 reduced (restoration phases)", 3, dict(horizon_N=6, n_obstacles=5), 2, 120, {}),
         ("C2 reduced (2 agents)", 2, dict(horizon_N=5, n_agents=2), 2, 6, {}),
         ("N3 quaternion family reduced", 5, dict(horizon_N=8), 2, 6, {})]


def main():
    for name, cfg, kw, P, max_iter, opt in CASES:
        d = wl.config_dims(cfg, **kw)
        d, theta, x0 = wl.generate(cfg, P, d)
        xL, xU = wl.bounds(d)
        o = jipm.default_options()
        o.max_iter = max_iter
        for k, v in opt.items():
            setattr(o, k, v)
        s = jipm.Solver(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt, xL, xU, o)
        out = s.solve_batch(x0, theta)
        st = s.stats()
        print(name, "status", out["status"].cpu().tolist(), "iters", out["iters"].cpu().tolist(),
              "resto iterations", st["resto_iterations"], flush=True)
        s.close()


if __name__ == "__main__":
    main()
