"""Small NLPs with closed-form answers, used to pin the oracle (and, on the GPU box, nothing else)."""
import numpy as np


class SmallNLP:
    """Duck-typed problem for oracle.ipm.Solver built from callables (dense)."""

    def __init__(self, n, m, f, grad, hess_f, c=None, jac=None, hess_c=None):
        self.n, self.m = n, m
        self._f, self._g, self._hf, self._c, self._j, self._hc = f, grad, hess_f, c, jac, hess_c

    def f(self, x, th):
        return float(self._f(x))

    def grad_f(self, x, th):
        return np.asarray(self._g(x), float)

    def c(self, x, th):
        return np.asarray(self._c(x), float) if self.m else np.zeros(0)

    def jac(self, x, th):
        return np.asarray(self._j(x), float).reshape(self.m, self.n) if self.m else np.zeros((0, self.n))

    def hess_lag(self, x, th, y, sigma_f=1.0):
        W = sigma_f * np.asarray(self._hf(x), float)
        if self.m and self._hc is not None:
            for j in range(self.m):
                W = W + y[j] * np.asarray(self._hc(x, j), float)
        return W


def fd_grad(fun, x, h=1e-6):
    g = np.zeros_like(x)
    for i in range(x.size):
        e = np.zeros_like(x)
        e[i] = h
        g[i] = (fun(x + e) - fun(x - e)) / (2 * h)
    return g


def fd_jac(fun, x, h=1e-6):
    f0 = fun(x)
    J = np.zeros((f0.size, x.size))
    for i in range(x.size):
        e = np.zeros_like(x)
        e[i] = h
        J[:, i] = (fun(x + e) - fun(x - e)) / (2 * h)
    return J
