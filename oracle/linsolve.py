"""ORACLE (test infrastructure, not the product).  Dense symmetric-indefinite LDL^T of the augmented
matrix of eq (7) by LAPACK's Bunch-Kaufman routine (dsytrf, a library primitive
used as one step), the inertia (n+, n-, n0) read from the 1x1 / 2x2 blocks of D (Sylvester's law),
and solves with the same factor (dsytrs).  No band, no condensation, no structure exploited.
Pinned against numpy.linalg.eigvalsh / numpy.linalg.solve in tests/test_oracle_linsolve.py.
"""
from __future__ import annotations

import numpy as np
from scipy.linalg import lapack


class DenseLDL:
    def __init__(self, K: np.ndarray, zero_tol: float = 0.0):
        K = np.asarray(K, dtype=np.float64)
        self.n = K.shape[0]
        ldu, ipiv, info = lapack.dsytrf(K, lower=1)
        if info < 0:
            raise ValueError(f"dsytrf argument {-info}")
        self.ldu, self.ipiv, self.info = ldu, ipiv, info
        # reading S-6: a pivot counts as a zero eigenvalue only if |d| <= zero_tol (ABSOLUTE,
        # default 0 = exactly singular).  A threshold relative to max|K_ii| misfires late in the solve, when
        # Sigma = z/s of active bounds reaches 1e8+ and legitimately small pivots would be flagged.
        thr = zero_tol
        npos = nneg = nzero = 0
        i = 0
        n = self.n
        while i < n:
            if ipiv[i] > 0:  # 1x1 block (LAPACK 1-based pivots)
                d = ldu[i, i]
                if abs(d) <= thr:
                    nzero += 1
                elif d > 0:
                    npos += 1
                else:
                    nneg += 1
                i += 1
            else:  # 2x2 block in rows i, i+1 (lower storage: off-diagonal at [i+1, i])
                a, b, c = ldu[i, i], ldu[i + 1, i], ldu[i + 1, i + 1]
                det = a * c - b * b
                if abs(det) <= thr * thr:
                    # singular 2x2: one zero eigenvalue, the other has the sign of the trace
                    nzero += 1
                    tr = a + c
                    if tr > 0:
                        npos += 1
                    elif tr < 0:
                        nneg += 1
                    else:
                        nzero += 1
                elif det < 0:
                    npos += 1
                    nneg += 1
                elif a + c > 0:
                    npos += 2
                else:
                    nneg += 2
                i += 2
        self.inertia = (npos, nneg, nzero)

    def solve(self, b: np.ndarray) -> np.ndarray:
        x, info = lapack.dsytrs(self.ldu, self.ipiv, np.asarray(b, dtype=np.float64), lower=1)
        if info != 0:
            raise ValueError(f"dsytrs info {info}")
        return x
