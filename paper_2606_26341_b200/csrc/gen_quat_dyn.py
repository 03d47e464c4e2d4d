#!/usr/bin/env python
"""Writes dyn_quat_gen.cuh: device functions of the 13-state quaternion quadrotor of the paper's own experiments
(x = (p, q, v, omega) in R^3 x R^4 x R^3 x R^3, body linear and angular velocities, four rotor speed
inputs), derived symbolically with sympy from the model equations below and emitted as straight-line CUDA with common
sub-expressions factored out:

    quat_ode   xdot = f(x, u)
    quat_jvp   K    = Df_x(x,u) y + Df_u(x,u) w                      (one column of the RK4 Jacobian chain)
    quat_vjp   out  = Df_x(x,u)^T mu                                 (adjoint recursion through the RK4 points)
    quat_hvp   t    = (sum_j mu_j Hess f_j(x,u)) v,  v in R^17       (adjoint-contracted Hessian times a column)

Model (textbook rigid body, the paper cites its ref. [40]; the paper gives no parameters -- DESIGN.md reading N3):
    pdot = R(q) v                         R(q) = rotation body -> world of q = (w, x, y, z) (not normalised)
    qdot = 1/2 q (x) (0, omega)
    vdot = -omega x v - g R(q)^T e3 + (T/m) e3,      T = kf sum u_i^2
    omegadot = J^-1 (tau - omega x J omega),         tau = (l kf (u2^2 - u4^2), l kf (u3^2 - u1^2), km (u1^2 - u2^2 + u3^2 - u4^2))
with m = 1, g = 9.81, l = 0.2, J = diag(0.01, 0.01, 0.02), kf = 1, km = 0.02 (rotor speeds in units with kf = 1).

Run:  python paper_2606_26341_b200/csrc/gen_quat_dyn.py     (rewrites dyn_quat_gen.cuh next to this file)
The oracle does NOT use this: it differentiates its own plain formula with second-order jets (oracle/families.py)."""
import os
import re

import sympy as sp

M, G, L, JX, JY, JZ, KF, KM = 1.0, 9.81, 0.2, 0.01, 0.01, 0.02, 1.0, 0.02


def model():
    x = sp.symbols("x0:13", real=True)
    u = sp.symbols("u0:4", real=True)
    p, q, v, w = x[0:3], x[3:7], x[7:10], x[10:13]
    qw, qx, qy, qz = q
    R = sp.Matrix([[1 - 2 * (qy * qy + qz * qz), 2 * (qx * qy - qw * qz), 2 * (qx * qz + qw * qy)],
                   [2 * (qx * qy + qw * qz), 1 - 2 * (qx * qx + qz * qz), 2 * (qy * qz - qw * qx)],
                   [2 * (qx * qz - qw * qy), 2 * (qy * qz + qw * qx), 1 - 2 * (qx * qx + qy * qy)]])
    vv, ww = sp.Matrix(v), sp.Matrix(w)
    pdot = R * vv
    qdot = sp.Rational(1, 2) * sp.Matrix([-(qx * w[0] + qy * w[1] + qz * w[2]),
                                          qw * w[0] + qy * w[2] - qz * w[1],
                                          qw * w[1] + qz * w[0] - qx * w[2],
                                          qw * w[2] + qx * w[1] - qy * w[0]])
    T = KF * sum(ui * ui for ui in u)
    vdot = -ww.cross(vv) - G * (R.T * sp.Matrix([0, 0, 1])) + sp.Matrix([0, 0, T / M])
    tau = sp.Matrix([L * KF * (u[1] ** 2 - u[3] ** 2), L * KF * (u[2] ** 2 - u[0] ** 2),
                     KM * (u[0] ** 2 - u[1] ** 2 + u[2] ** 2 - u[3] ** 2)])
    Jm = sp.diag(JX, JY, JZ)
    wdot = Jm.inv() * (tau - ww.cross(Jm * ww))
    f = sp.Matrix(list(pdot) + list(qdot) + list(vdot) + list(wdot))
    return x, u, f


def emit(name, args, outname, exprs, doc):
    repl, red = sp.cse(list(exprs), symbols=sp.numbered_symbols("t_"), optimizations="basic")
    lines = [f"// {doc}", f"__device__ __forceinline__ void {name}({args}) {{"]
    for s, e in repl:
        lines.append(f"    const double {s} = {sp.ccode(e)};")
    for i, e in enumerate(red):
        lines.append(f"    {outname}[{i}] = {sp.ccode(e)};")
    lines.append("}")
    txt = "\n".join(lines)
    # pow(a, 2) -> (a*a): no call into the math library for a square
    txt = re.sub(r"pow\(([A-Za-z_0-9\[\]]+), 2\)", r"(\1*\1)", txt)
    assert "pow(" not in txt, "unexpected power in the generated code"
    return txt


def main():
    x, u, f = model()
    z = list(x) + list(u)
    y = sp.symbols("y0:13", real=True)
    w = sp.symbols("w0:4", real=True)
    mu = sp.symbols("mu0:13", real=True)
    v = sp.symbols("v0:17", real=True)
    Dx, Du = f.jacobian(list(x)), f.jacobian(list(u))
    jvp = Dx * sp.Matrix(y) + Du * sp.Matrix(w)
    vjp = Dx.T * sp.Matrix(mu)
    lag = sum(mu[j] * f[j] for j in range(13))
    H = sp.hessian(lag, z)
    hvp = H * sp.Matrix(v)

    def sub(e, names):
        m = {}
        for arr, base in names:
            for i, s_ in enumerate(arr):
                m[s_] = sp.Symbol(f"{base}[{i}]")
        return [sp.simplify(ei).xreplace(m) for ei in e]

    xs = [(x, "x"), (u, "u")]
    parts = [
        emit("quat_ode", "const double* x, const double* u, double* d", "d", sub(f, xs), "xdot = f(x, u)"),
        emit("quat_jvp", "const double* x, const double* u, const double* y, const double* w, double* K", "K",
             sub(jvp, xs + [(y, "y"), (w, "w")]), "K = Df_x y + Df_u w"),
        emit("quat_vjp", "const double* x, const double* u, const double* mu, double* out", "out",
             sub(vjp, xs + [(mu, "mu")]), "out = Df_x^T mu"),
        emit("quat_hvp", "const double* x, const double* u, const double* mu, const double* v, double* t", "t",
             sub(hvp, xs + [(mu, "mu"), (v, "v")]), "t = (sum_j mu_j Hess f_j) v over z = (x, u)"),
    ]
    hdr = ("// dyn_quat_gen.cuh -- GENERATED by gen_quat_dyn.py (sympy) from the 13-state quaternion quadrotor model of\n"
           "// PAPER.md:174-180; do not edit by hand.  Parameters: m 1, g 9.81, l 0.2, J diag(0.01,0.01,0.02), kf 1, km 0.02.\n"
           "#pragma once\n\nnamespace jipm {\n\n")
    out = hdr + "\n\n".join(parts) + "\n\n}  // namespace jipm\n"
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "dyn_quat_gen.cuh"), "w") as fh:
        fh.write(out)
    print("wrote dyn_quat_gen.cuh:", out.count("\n"), "lines")


if __name__ == "__main__":
    main()
