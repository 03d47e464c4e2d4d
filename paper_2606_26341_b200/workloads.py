"""Seeded synthetic input generators for the BASELINE.json configs (C0..C3).

This module is shared by the tests, ``bench.py`` and ``__graft_entry__.smoke()``; it feeds the
SAME arrays to the CUDA path and to the oracle.  It holds none of the method's arithmetic: no
objective, constraint, derivative, KKT or line-search code lives here, only (a) the index layout of
the stage-ordered decision vector, (b) the bounds, and (c) the random draws of the per-problem
parameter vector theta and of the initial guess x0.  It imports neither ``oracle`` nor the CUDA
binding.

Inputs stand in for the paper's quadrotor task generator (Tables II-IV), which is
not available; the recipe is the one of SURVEY.md section 8(d) / DESIGN.md "Input recipe".

Layout of the decision vector (n entries) -- "stage order":
    [ x_0 | u_0 x_1 s_1 | u_1 x_2 s_2 | ... | u_{N-1} x_N s_N ]
and of the equality vector (m entries):
    [ x_0 - xhat0 | dyn_1 g_1 | dyn_2 g_2 | ... | dyn_N g_N ]
with dyn_k = x_k - F(x_{k-1}, u_{k-1}) and g_k = (inequality residuals at knot k) - s_k.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

FAM_POINTMASS2D = 0
FAM_QUAD_TRACK = 1
FAM_MULTIQUAD = 2
FAM_QUAD_CLUTTER = 3
FAM_QUAT_NAV = 4        # the paper's own vehicle: 13-state quaternion quadrotor, rotor-speed inputs

GRAV = 9.81
QUAD_MASS = 1.0


@dataclass(frozen=True)
class Dims:
    """Mirror of ``jipm_family_dims`` plus the derived sizes."""
    family: int
    horizon_N: int
    n_agents: int
    n_obstacles: int
    dt: float

    @property
    def nx(self) -> int:
        if self.family == FAM_QUAT_NAV:
            return 13
        return 4 if self.family == FAM_POINTMASS2D else 12 * self.n_agents

    @property
    def nu(self) -> int:
        return 2 if self.family == FAM_POINTMASS2D else 4 * self.n_agents

    @property
    def ng(self) -> int:
        if self.family == FAM_MULTIQUAD:
            return self.n_agents * (self.n_agents - 1) // 2
        return self.n_obstacles

    @property
    def n(self) -> int:
        N = self.horizon_N
        return (N + 1) * self.nx + N * self.nu + N * self.ng

    @property
    def m(self) -> int:
        N = self.horizon_N
        return (N + 1) * self.nx + N * self.ng

    @property
    def n_theta(self) -> int:
        if self.family == FAM_POINTMASS2D:
            return 4 + 2 + 3 * self.n_obstacles
        if self.family == FAM_QUAD_TRACK:
            return 12 + 2 + 4 * self.n_obstacles
        if self.family == FAM_MULTIQUAD:
            return 12 * self.n_agents + 3 * self.n_agents
        if self.family == FAM_QUAT_NAV:
            return 13 + 3 + 4 * self.n_obstacles
        return 12 + 3 + 4 * self.n_obstacles

    # index helpers (stage order) -------------------------------------------------------------
    @property
    def blk(self) -> int:
        return self.nu + self.nx + self.ng

    def ix(self, k: int) -> int:
        return 0 if k == 0 else self.nx + (k - 1) * self.blk + self.nu

    def iu(self, k: int) -> int:
        return self.nx + k * self.blk

    def islack(self, k: int) -> int:  # k = 1..N
        return self.nx + (k - 1) * self.blk + self.nu + self.nx

    def ic_dyn(self, k: int) -> int:  # k = 1..N ; k = 0 is the initial condition at 0
        return 0 if k == 0 else self.nx + (k - 1) * (self.nx + self.ng)

    def ic_g(self, k: int) -> int:  # k = 1..N
        return self.nx + (k - 1) * (self.nx + self.ng) + self.nx


def config_dims(cfg: int, horizon_N: int | None = None, n_obstacles: int | None = None,
                n_agents: int | None = None) -> Dims:
    """BASELINE.json configs; the optional overrides give the reduced instances used in tests."""
    if cfg == 0:
        d = Dims(FAM_POINTMASS2D, 10, 1, 1, 0.1)
    elif cfg == 1:
        d = Dims(FAM_QUAD_TRACK, 20, 1, 3, 0.05)
    elif cfg == 2:
        d = Dims(FAM_MULTIQUAD, 20, 4, 0, 0.05)
    elif cfg == 3:
        d = Dims(FAM_QUAD_CLUTTER, 30, 1, 32, 0.05)
    elif cfg == 5:   # NEXT-3: the paper's own formulation: dt 0.1, 30 knots (29 intervals), 506 variables
        d = Dims(FAM_QUAT_NAV, 29, 1, 3, 0.1)
    else:
        raise ValueError(cfg)
    return Dims(d.family,
                d.horizon_N if horizon_N is None else horizon_N,
                d.n_agents if n_agents is None else n_agents,
                d.n_obstacles if n_obstacles is None else n_obstacles,
                d.dt)


CONFIG_BATCH = {0: 256, 1: 4096, 2: 2048, 3: 8192, 5: 2000}


# ------------------------------------------------------------------------------------------------
# counter-based generator: splitmix64 of (seed, problem, draw) -> 53-bit uniform in [0,1)
# ------------------------------------------------------------------------------------------------
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(z: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = (z + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def uniform01(seed: int, problem: np.ndarray, draw: np.ndarray) -> np.ndarray:
    """u[problem, draw] in [0,1); independent of batch size and order (counter based)."""
    with np.errstate(over="ignore"):
        key = _splitmix64(np.uint64(seed) + np.zeros_like(problem, dtype=np.uint64))
        key = _splitmix64(key ^ (problem.astype(np.uint64) * np.uint64(0xD1342543DE82EF95)))
        key = _splitmix64(key ^ (draw.astype(np.uint64) * np.uint64(0x2545F4914F6CDD1D)))
    return (key >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


class _Draws:
    def __init__(self, seed: int, ids: np.ndarray):
        self.seed, self.ids, self.count = seed, ids, 0

    def u(self, lo: float, hi: float, k: int = 1) -> np.ndarray:
        """[P, k] uniforms in [lo, hi), consuming k counters per problem."""
        d = np.arange(self.count, self.count + k, dtype=np.uint64)
        self.count += k
        r = uniform01(self.seed, self.ids[:, None], d[None, :])
        return lo + (hi - lo) * r


def bounds(d: Dims) -> tuple[np.ndarray, np.ndarray]:
    """Shared bounds x_L, x_U: inputs boxed, slacks >= 0, states free."""
    xL = np.full(d.n, -np.inf)
    xU = np.full(d.n, np.inf)
    if d.family == FAM_POINTMASS2D:
        ulo, uhi = -1.0, 1.0
    elif d.family == FAM_QUAT_NAV:   # rotor speeds, thrust per rotor u^2 <= m g / 2
        ulo, uhi = 0.0, math.sqrt(QUAD_MASS * GRAV / 2.0)
    else:
        ulo, uhi = 0.0, QUAD_MASS * GRAV / 2.0
    for k in range(d.horizon_N):
        xL[d.iu(k):d.iu(k) + d.nu] = ulo
        xU[d.iu(k):d.iu(k) + d.nu] = uhi
    for k in range(1, d.horizon_N + 1):
        xL[d.islack(k):d.islack(k) + d.ng] = 0.0
    return xL, xU


def generate(cfg: int, P: int, d: Dims | None = None, first_id: int = 0, stream: int = 0):
    """Return (dims, theta[P, n_theta], x0[P, n]) for problems first_id .. first_id+P-1 of config cfg."""
    d = config_dims(cfg) if d is None else d
    seed = 26341 + 1000 * cfg + stream
    ids = np.arange(first_id, first_id + P, dtype=np.uint64)
    dr = _Draws(seed, ids)
    N, nx, nu = d.horizon_N, d.nx, d.nu
    theta = np.zeros((P, d.n_theta))
    x0 = np.zeros((P, d.n))
    if d.family == FAM_POINTMASS2D:
        xh = np.zeros((P, 4))
        xh[:, 0:2] = dr.u(-2, 2, 2)
        goal = dr.u(-2, 2, 2)
        theta[:, 0:4] = xh
        theta[:, 4:6] = goal
        for j in range(d.n_obstacles):
            theta[:, 6 + 3 * j:8 + 3 * j] = dr.u(-1, 1, 2)
            theta[:, 8 + 3 * j] = dr.u(0.3, 0.5, 1)[:, 0]
        for k in range(N + 1):
            x0[:, d.ix(k):d.ix(k) + 4] = xh
        return d, theta, x0

    hover = QUAD_MASS * GRAV / 4.0
    if d.family == FAM_QUAT_NAV:
        # Sector navigation (stands in for PAPER.md:186-205, whose generator is not given): every vehicle flies to a
        # common goal (0, 0, 1) from a start on a 6 m arc around it, angle ~ U(-90, 90) degrees (the 180-degree sector),
        # altitude 1 + U(-0.5, 0.5); the obstacles sit in the central 90 degrees between arc and goal: centre at
        # distance U(2, 4) and angle U(-45, 45) degrees, altitude 1 + U(-0.5, 0.5), radius U(0.3, 0.6).  Level attitude
        # (q = (1, 0, 0, 0)), at rest; initial guess: stay put with the hover rotor speed sqrt(m g / 4).
        xh = np.zeros((P, 13))
        ang = dr.u(-0.5 * math.pi, 0.5 * math.pi, 1)[:, 0]
        xh[:, 0], xh[:, 1] = 6.0 * np.cos(ang), 6.0 * np.sin(ang)
        xh[:, 2] = 1.0 + dr.u(-0.5, 0.5, 1)[:, 0]
        xh[:, 3] = 1.0
        theta[:, 0:13] = xh
        theta[:, 13:16] = np.array([0.0, 0.0, 1.0])
        for j in range(d.n_obstacles):
            rad = dr.u(2.0, 4.0, 1)[:, 0]
            a2 = dr.u(-0.25 * math.pi, 0.25 * math.pi, 1)[:, 0]
            theta[:, 16 + 4 * j] = rad * np.cos(a2)
            theta[:, 17 + 4 * j] = rad * np.sin(a2)
            theta[:, 18 + 4 * j] = 1.0 + dr.u(-0.5, 0.5, 1)[:, 0]
            theta[:, 19 + 4 * j] = dr.u(0.3, 0.6, 1)[:, 0]
        for k in range(N + 1):
            x0[:, d.ix(k):d.ix(k) + 13] = xh
        for k in range(N):
            x0[:, d.iu(k):d.iu(k) + nu] = math.sqrt(hover)
        return d, theta, x0
    if d.family == FAM_QUAD_TRACK:
        xh = np.zeros((P, 12))
        xh[:, 0:3] = dr.u(-3, 3, 3)
        xh[:, 3:6] = dr.u(-0.2, 0.2, 3)
        rho = dr.u(1, 3, 1)[:, 0]
        theta[:, 0:12] = xh
        theta[:, 12] = rho
        theta[:, 13] = np.arctan2(xh[:, 1], xh[:, 0])
        for j in range(d.n_obstacles):
            theta[:, 14 + 4 * j:17 + 4 * j] = dr.u(-3, 3, 3)
            theta[:, 17 + 4 * j] = dr.u(0.3, 0.6, 1)[:, 0]
        for k in range(N + 1):
            x0[:, d.ix(k):d.ix(k) + 12] = xh
    elif d.family == FAM_MULTIQUAD:
        na = d.n_agents
        start = np.zeros((P, na, 3))
        goal = np.zeros((P, na, 3))
        todo = np.ones(P, dtype=bool)
        # reject-and-resample the whole problem until all start pairs are >= 1 m apart (D-3)
        for _attempt in range(64):
            ang = dr.u(0.0, 2.0 * math.pi, na)
            js = dr.u(-0.3, 0.3, 3 * na).reshape(P, na, 3)
            jg = dr.u(-0.3, 0.3, 3 * na).reshape(P, na, 3)
            c = np.stack([4 * np.cos(ang), 4 * np.sin(ang), np.zeros_like(ang)], axis=-1)
            s_new, g_new = c + js, -c + jg
            start[todo], goal[todo] = s_new[todo], g_new[todo]
            ok = np.ones(P, dtype=bool)
            for i in range(na):
                for j in range(i + 1, na):
                    ok &= np.linalg.norm(start[:, i] - start[:, j], axis=1) >= 1.0
            todo = ~ok
            if not todo.any():
                break
        xh = np.zeros((P, 12 * na))
        for a in range(na):
            xh[:, 12 * a:12 * a + 3] = start[:, a]
        theta[:, 0:12 * na] = xh
        theta[:, 12 * na:] = goal.reshape(P, 3 * na)
        for k in range(N + 1):
            x0[:, d.ix(k):d.ix(k) + nx] = xh
    else:  # FAM_QUAD_CLUTTER
        xh = np.zeros((P, 12))
        xh[:, 0:3] = dr.u(-0.5, 0.5, 3)
        goal = 10.0 + dr.u(-0.5, 0.5, 3)
        theta[:, 0:12] = xh
        theta[:, 12:15] = goal
        for j in range(d.n_obstacles):
            c = dr.u(0, 10, 3)
            r = dr.u(0.2, 0.5, 1)[:, 0]
            for _attempt in range(32):  # resample individually if within r+0.5 m of start or goal
                bad = (np.linalg.norm(c - xh[:, 0:3], axis=1) < r + 0.5) | \
                      (np.linalg.norm(c - goal, axis=1) < r + 0.5)
                c2 = dr.u(0, 10, 3)
                r2 = dr.u(0.2, 0.5, 1)[:, 0]
                c[bad], r[bad] = c2[bad], r2[bad]
                if not bad.any():
                    break
            theta[:, 15 + 4 * j:18 + 4 * j] = c
            theta[:, 18 + 4 * j] = r
        for k in range(N + 1):  # straight-line initial guess start -> goal
            w = k / N
            x0[:, d.ix(k):d.ix(k) + 3] = (1 - w) * xh[:, 0:3] + w * goal
    for k in range(N):
        x0[:, d.iu(k):d.iu(k) + nu] = hover
    return d, theta, x0
