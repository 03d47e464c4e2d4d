"""Pins for oracle/linsolve.py: inertia against eigenvalue sign counts (Sylvester's law of inertia,
PAPER.md:114 "inertia (n_x, n_c, 0)"), solves against numpy.linalg.solve."""
import numpy as np

from oracle.linsolve import DenseLDL


def eig_inertia(K):
    w = np.linalg.eigvalsh(K)
    return int((w > 0).sum()), int((w < 0).sum()), int((w == 0).sum())


def test_inertia_random_indefinite():
    rng = np.random.default_rng(1)
    for n in (1, 2, 3, 7, 20, 55):
        for _ in range(20):
            M = rng.normal(size=(n, n))
            K = M + M.T
            assert DenseLDL(K).inertia == eig_inertia(K)


def test_inertia_kkt_structured():
    rng = np.random.default_rng(2)
    for n, m in ((5, 2), (12, 7), (30, 30)):
        for trial in range(10):
            H = rng.normal(size=(n, n))
            H = H @ H.T if trial % 2 == 0 else H + H.T      # convex / nonconvex Hessian
            A = rng.normal(size=(m, n))
            K = np.block([[H, A.T], [A, np.zeros((m, m))]])
            f = DenseLDL(K)
            assert f.inertia == eig_inertia(K)
            if trial % 2 == 0:
                assert f.inertia == (n, m, 0)
            b = rng.normal(size=n + m)
            np.testing.assert_allclose(f.solve(b), np.linalg.solve(K, b), rtol=1e-8, atol=1e-10)


def test_exact_singularity_is_reported():
    K = np.array([[1.0, 0.0, 1.0], [0.0, 0.0, 0.0], [1.0, 0.0, 0.0]])
    assert DenseLDL(K).inertia[2] >= 1
    K = np.zeros((2, 2))
    assert DenseLDL(K).inertia == (0, 0, 2)
