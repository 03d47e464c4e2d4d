"""ORACLE (test infrastructure, not the product).  Second-order Taylor "jets" in numpy, fp64.

A Jet carries (value, gradient, Hessian) of a scalar function of d inputs, batched over a leading
axis B.  Arithmetic on jets applies the textbook sum / product / chain rules

    (ab)'  = a'b + ab'            (ab)'' = a''b + a'b'^T + b'a'^T + ab''
    g(a)'  = g'(a) a'             g(a)'' = g''(a) a'a'^T + g'(a) a''

so that running a plain formula (here: the quadrotor ODE of SURVEY.md Appendix C pushed through one
classical RK4 step) on jets yields the exact Jacobian and Hessian the KKT system (7) of
PAPER.md:110-112 needs (W = Hessian of the Lagrangian, A = Jacobian of c).
Pinned by central finite differences in tests/test_oracle_derivatives.py.
"""
from __future__ import annotations

import numpy as np


class Jet:
    __slots__ = ("v", "g", "H")

    def __init__(self, v, g, H):
        self.v, self.g, self.H = v, g, H

    @staticmethod
    def variables(z: np.ndarray) -> list["Jet"]:
        """z[B, d] -> d jets, jet i being the coordinate function z_i."""
        B, d = z.shape
        out = []
        for i in range(d):
            g = np.zeros((B, d))
            g[:, i] = 1.0
            out.append(Jet(z[:, i].copy(), g, np.zeros((B, d, d))))
        return out

    @staticmethod
    def const_like(ref: "Jet", c) -> "Jet":
        return Jet(np.zeros_like(ref.v) + c, np.zeros_like(ref.g), np.zeros_like(ref.H))

    def _lift(self, o) -> "Jet":
        return o if isinstance(o, Jet) else Jet.const_like(self, o)

    def __add__(self, o):
        o = self._lift(o)
        return Jet(self.v + o.v, self.g + o.g, self.H + o.H)

    __radd__ = __add__

    def __neg__(self):
        return Jet(-self.v, -self.g, -self.H)

    def __sub__(self, o):
        return self + (-self._lift(o))

    def __rsub__(self, o):
        return self._lift(o) - self

    def __mul__(self, o):
        if not isinstance(o, Jet):
            return Jet(self.v * o, self.g * o, self.H * o)
        a, b = self, o
        cross = a.g[:, :, None] * b.g[:, None, :]
        H = a.H * b.v[:, None, None] + cross + np.swapaxes(cross, 1, 2) + b.H * a.v[:, None, None]
        return Jet(a.v * b.v, a.g * b.v[:, None] + b.g * a.v[:, None], H)

    __rmul__ = __mul__

    def _chain(self, g0, g1, g2):
        """Compose with a scalar function whose value / 1st / 2nd derivative at self.v are g0,g1,g2."""
        outer = self.g[:, :, None] * self.g[:, None, :]
        return Jet(g0, g1[:, None] * self.g, g2[:, None, None] * outer + g1[:, None, None] * self.H)

    def recip(self):
        r = 1.0 / self.v
        return self._chain(r, -r * r, 2.0 * r * r * r)

    def __truediv__(self, o):
        if not isinstance(o, Jet):
            return self * (1.0 / o)
        return self * o.recip()

    def sin(self):
        s, c = np.sin(self.v), np.cos(self.v)
        return self._chain(s, c, -s)

    def cos(self):
        s, c = np.sin(self.v), np.cos(self.v)
        return self._chain(c, -s, -c)
