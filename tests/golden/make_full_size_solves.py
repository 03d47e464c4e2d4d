"""Writes tests/golden/full_size_c{1,2,3,5}.json: the ORACLE's results on the first problems of BASELINE.json configs[1..3]
(and of workload 5, the paper's own 13-state quaternion vehicle) at their FULL dimensions (status, iteration count, objective, positions of every knot of x*, and the largest pitch angle
the iterates reached -- the 12-state Euler model of SURVEY.md Appendix C is singular at |pitch| = pi/2).  The GPU tests
compare against these files instead of re-running the dense oracle (minutes per problem at n = 1448 / 1452).

    python tests/golden/make_full_size_solves.py [cfg ...]        (imports only oracle/ and the seeded input generator)

Nothing here touches the CUDA path: every stored value is the oracle's."""
from __future__ import annotations

import json
import os
import sys
import time
from multiprocessing import get_context

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
os.environ.setdefault("OMP_NUM_THREADS", "1")

import numpy as np  # noqa: E402

from oracle import families as ofam, ipm as oipm  # noqa: E402
from paper_2606_26341_b200 import workloads as wl  # noqa: E402

COUNT = {1: 48, 2: 8, 3: 8, 5: 16}
MAX_ITER = {1: 3000, 2: 300, 3: 600, 5: 3000}   # the oracle is cut here; a problem that reaches the cap is stored as such


def solve_one(args):
    cfg, idx = args
    d, theta, x0 = wl.generate(cfg, 1, first_id=idx)
    xL, xU = wl.bounds(d)
    prob = ofam.Problem(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt)
    o = oipm.Options()
    o.max_iter = MAX_ITER[cfg]
    s = oipm.Solver(prob, xL, xU, o)
    th = theta[0]
    st = s.initialise(x0[0], th)
    t0 = time.time()
    pitch, n_resto, kinds = 0.0, 0, {}
    while st.status == oipm.ST_NOT_RUN:
        x = st.x if st.resto is None else st.resto.state.x[:d.n]
        if d.family in (wl.FAM_QUAD_TRACK, wl.FAM_MULTIQUAD, wl.FAM_QUAD_CLUTTER):   # the Euler-angle families
            pitch = max(pitch, max(abs(x[prob.ix(k) + 12 * a + 4]) for k in range(d.horizon_N + 1) for a in range(d.n_agents)))
        tr = s.iterate(st, th)
        n_resto += int(tr.get("mode", 0) == 1)
        for key in ("wd", "soft", "tiny", "npsing"):
            if tr.get(key):
                kinds[key] = kinds.get(key, 0) + 1
    pos = [[float(v) for v in st.x[prob.ix(k) + prob.ax * a: prob.ix(k) + prob.ax * a + 3]]
           for k in range(d.horizon_N + 1) for a in range(d.n_agents)]
    return dict(id=idx, status=int(st.status), iters=int(st.k), f=float(prob.f(st.x, th)), max_pitch=float(pitch),
                resto_iters=n_resto, fallbacks=kinds, positions=pos, seconds=round(time.time() - t0, 1))


def main():
    cfgs = [int(a) for a in sys.argv[1:]] or [1, 3, 2]
    for cfg in cfgs:
        with get_context("fork").Pool(os.cpu_count() or 1) as pool:
            rows = pool.map(solve_one, [(cfg, i) for i in range(COUNT[cfg])], chunksize=1)
        out = dict(config=cfg, oracle_max_iter=MAX_ITER[cfg], note="written by tests/golden/make_full_size_solves.py "
                   "(oracle/ only); positions = p_k of every knot and agent of x*", problems=rows)
        with open(os.path.join(HERE, f"full_size_c{cfg}.json"), "w") as f:
            json.dump(out, f, indent=0)
        print(cfg, [(r["id"], r["status"], r["iters"]) for r in rows], flush=True)


if __name__ == "__main__":
    main()
