"""How far the ORACLE is from ITSELF when its inputs move by one rounding error: the yardstick for the whole-trajectory
parity of the CUDA path (tests/test_gpu_parity.py).  x0 and theta of the batches the GPU tests use
are perturbed by a relative 1e-15 (seeded) and every trajectory is compared decision by decision with the unperturbed
one.  On the well-conditioned families (the point mass; the paper's quaternion vehicle) nothing changes: there the
>= 99 % bar on whole trajectories can be asked of a second implementation, and is.  On the Euler-angle families a
trajectory or two of twelve part after 10-190 identical iterations (measured here: reduced C1 11/12, C2 10/12, C3
11/12; the GPU against the oracle: 11/12, 10/12, 8/12): no implementation with its own rounding can do better, which is
why those tests ask for an EXPLANATION of every parting instead of a fraction."""
import numpy as np
import pytest

import parity as par
from paper_2606_26341_b200 import workloads as wl

REDUCED = {0: dict(), 1: dict(horizon_N=7), 2: dict(horizon_N=5, n_agents=2), 3: dict(horizon_N=6, n_obstacles=5),
           5: dict(horizon_N=8)}
KEYS = ("kind", "mode", "nfact", "ls", "soc", "nmu", "wd", "soft", "tiny", "npsing")


def decisions(trace):
    return [tuple(t.get(k, 0) for k in KEYS) for t in trace]


def identical_under_perturbation(cfg, P, rel=1e-15, seed=7):
    d = wl.config_dims(cfg, **REDUCED[cfg])
    d, theta, x0 = wl.generate(cfg, P, d)
    xL, xU = wl.bounds(d)
    rng = np.random.default_rng(seed)
    x0p = x0 * (1.0 + rel * rng.uniform(-1, 1, x0.shape))
    thp = theta * (1.0 + rel * rng.uniform(-1, 1, theta.shape))
    same, partings = 0, []
    for (s0, t0), (s1, t1) in zip(par.oracle_solve(d, xL, xU, x0, theta), par.oracle_solve(d, xL, xU, x0p, thp)):
        a, b = decisions(t0), decisions(t1)
        if s0.status == s1.status and s0.k == s1.k and a == b:
            same += 1
        else:
            first = next((i for i, (u, v) in enumerate(zip(a, b)) if u != v), min(len(a), len(b)))
            partings.append((first, s0.status, s0.k, s1.status, s1.k))
    return same, partings


@pytest.mark.parametrize("cfg,P", [(0, 48), (5, 12)])
def test_well_conditioned_families_are_insensitive(cfg, P):
    same, partings = identical_under_perturbation(cfg, P)
    print(f"cfg {cfg}: oracle vs oracle with inputs moved by 1e-15: {same}/{P} trajectories identical {partings}")
    assert same >= 0.99 * P, partings


@pytest.mark.parametrize("cfg,P", [(1, 12), (2, 12), (3, 12)])
def test_euler_angle_families_part_only_after_a_common_prefix(cfg, P):
    """Reported, not asserted: the fraction (it depends on the LAPACK build).  Asserted: a parting is never immediate --
    the first iterations agree -- and most trajectories still agree completely."""
    same, partings = identical_under_perturbation(cfg, P)
    print(f"cfg {cfg}: oracle vs oracle with inputs moved by 1e-15: {same}/{P} trajectories identical; partings "
          f"(first differing iteration, status, iterations | status, iterations): {partings}")
    assert all(p[0] >= 3 for p in partings), partings
    assert same >= P // 2, partings
