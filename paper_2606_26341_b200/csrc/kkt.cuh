// kkt.cuh -- stage-ordered block LDL^T of the augmented system (7)
//        [ W + Sigma + Hd   A^T ] [dx]   [rp]
//        [ A               -Dc  ] [dy] = [rc]
// with an inertia count from the pivot blocks, and the solve with that factor.
//
// Elimination order (a block LDL^T of the stage-ordered KKT matrix):
//   1. every (slack s_kj, multiplier y_g,kj) pair as a 2x2 block [[sig,-1],[-1,-dc]] -- inertia (1,1,0) always;
//      its Schur complement adds G^T Dg G, Dg = 1/(1/sig + dc), to the position block of stage k;
//   2. backwards over stages k = N..1: the pair (x_k, y_dyn,k) as the block [[P_k, I],[I, -D_k]] whose inertia is
//      (0,nx,0) + In(I + E P_k E), E = sqrt(D_k) (equal to (nx,nx,0) when D_k = 0, for any P_k); its Schur complement
//      adds [A B]^T T_k [A B] to stage k-1 with T_k = (I + P_k D_k)^{-1} P_k;
//   3. the control block Rt_k = R_k + B^T T_{k+1} B by an unpivoted LDL^T: its pivot signs carry the inertia test.
// By Haynsworth additivity the KKT matrix has inertia (n, m, 0) iff every Rt_k pivot (and every pivot of
// I + E P E when D != 0) is positive.
#pragma once
#include "core.cuh"

namespace jipm {

template <class C>
struct Kkt {
    static constexpr int NX = C::NX, NU = C::NU, NZ = C::NZ, PD = C::PD, AX = C::AX, NA = C::NA;
    using X = Ctx<C>;

    // Dg weights of the condensed (slack, multiplier) pairs of stage k into sv-style scratch: returns for (k,j)
    __device__ static __forceinline__ double Dg(const X& c, int k, int j) {
        const double sig = c.ws[c.L.Sig + c.is(k) + j], dcg = c.ws[c.L.Dc + c.icg(k) + j];
        return 1.0 / (1.0 / sig + dcg);
    }

    // add sum_j Dg_j G_j^T G_j of stage k (k>=1) to the position entries of the tile M (leading dim ld)
    __device__ static void add_cond(const X& c, int k, double* M, int ld) {
        const Pb& pb = c.pb;
        const double* gv = c.ws + c.L.gv + (k - 1) * pb.ng * PD;
        constexpr int NPOS = NA * PD;
        for (int e = c.lane; e < NPOS * NPOS; e += 32) {
            const int r = e / NPOS, q = e % NPOS;
            const int a = r / PD, i = r % PD, b = q / PD, i2 = q % PD;
            double s = 0.0;
            if (pb.family == JIPM_FAM_MULTIQUAD) {
                for (int j = 0; j < pb.ng; ++j) {
                    int pa, pb2; c.pair_ab(j, pa, pb2);
                    const double sa = (pa == a) ? 1.0 : (pb2 == a ? -1.0 : 0.0);
                    const double sb = (pa == b) ? 1.0 : (pb2 == b ? -1.0 : 0.0);
                    if (sa != 0.0 && sb != 0.0) s += sa * sb * Dg(c, k, j) * gv[j * PD + i] * gv[j * PD + i2];
                }
            } else {
                for (int j = 0; j < pb.ng; ++j) s += Dg(c, k, j) * gv[j * PD + i] * gv[j * PD + i2];
            }
            M[(AX * a + i) * ld + AX * b + i2] += s;
        }
        __syncwarp();
    }

    // T <- (I + P D)^{-1} P in place on the NX x NX tile sT (symmetric), D = Dc at rows [row0, row0+NX).
    // Returns the number of non-positive pivots of I + E P E (0 when D == 0).  Uses sM as scratch.
    __device__ static int transform_T(const X& c, double* sT, double* sM, int row0) {
        const double* Dc = c.ws + c.L.Dc + row0;
        double dmax = 0.0;
        for (int i = c.lane; i < NX; i += 32) dmax = fmax(dmax, Dc[i]);
        dmax = wmax(dmax);
        if (dmax == 0.0) return 0;
        // G = I + E P E -> sM (NX x NX), E = sqrt(D);   Y = E P -> rows scaled copy in sM second half is avoided:
        // solve G Z = E P by LDL^T of G, then T = P - (P E) Z.
        double* G = sM;              // NX*NX
        double* Z = sM + NX * NX;    // NX*NX  (needs NZ*NZ >= 2 NX*NX; guaranteed by SM layout check at launch)
        for (int e = c.lane; e < NX * NX; e += 32) {
            const int r = e / NX, q = e % NX;
            const double er = sqrt(Dc[r]), eq = sqrt(Dc[q]);
            G[e] = er * sT[e] * eq + (r == q ? 1.0 : 0.0);
            Z[e] = er * sT[e];
        }
        __syncwarp();
        int bad = 0;
        // unpivoted LDL^T of G applied to the right-hand sides Z (column q of Z handled by lane q)
        for (int p = 0; p < NX; ++p) {
            double d = G[p * NX + p];
            if (!(d > 0.0)) { bad++; if (d == 0.0) d = 1.0; }
            for (int q = c.lane; q < 2 * NX; q += 32) {
                double* Mx = (q < NX) ? G : Z;
                const int qq = (q < NX) ? q : q - NX;
                if (q < NX && qq <= p) continue;
                const double lpq = Mx[p * NX + qq] / d;
                for (int r = p + 1; r < NX; ++r) Mx[r * NX + qq] -= G[r * NX + p] * lpq;
            }
            __syncwarp();
        }
        // now G holds (in its lower part, column p rows r>p) L*d ... Z holds L^{-1} E P; finish Z <- L^{-T} D^{-1} Z
        for (int p = NX - 1; p >= 0; --p) {
            double d = G[p * NX + p];
            if (d == 0.0) d = 1.0;
            for (int q = c.lane; q < NX; q += 32) {
                double v = Z[p * NX + q] / d;
                for (int r = p + 1; r < NX; ++r) v -= (G[r * NX + p] / d) * Z[r * NX + q];
                Z[p * NX + q] = v;
            }
            __syncwarp();
        }
        // T = P - (P E) Z ; (P E)[i][l] = P[i][l] e_l
        for (int q = c.lane; q < NX; q += 32) {
            double acc[NX];
#pragma unroll
            for (int i = 0; i < NX; ++i) acc[i] = 0.0;
            for (int l = 0; l < NX; ++l) {
                const double zl = sqrt(Dc[l]) * Z[l * NX + q];
#pragma unroll
                for (int i = 0; i < NX; ++i) acc[i] += sT[l * NX + i] * zl;
            }
            // write into G region first to avoid overwriting P while other lanes read it
#pragma unroll
            for (int i = 0; i < NX; ++i) G[i * NX + q] = sT[i * NX + q] - acc[i];
        }
        __syncwarp();
        for (int e = c.lane; e < NX * NX; e += 32) {
            const int r = e / NX, q = e % NX;
            sT[e] = 0.5 * (G[e] + G[q * NX + r]);
        }
        __syncwarp();
        return bad;
    }

    // Factor.  Reads W, J, Sig, Dc, gv from the workspace; writes T, Xf, Lf.  Returns the number of pivots with
    // the wrong sign (0 <=> inertia (n, m, 0)); nzero counts exactly-zero pivots.
    __device__ static int factor(const X& c, int& nzero, bool useW = true) {
        const Pb& pb = c.pb;
        const int N = pb.N, lane = c.lane;
        double* sT = c.sm + C::SM_T;
        double* sJ = c.sm + C::SM_J;
        double* sM = c.sm + C::SM_M;
        const double* Sig = c.ws + c.L.Sig;
        int bad = 0;
        nzero = 0;
        // terminal block
        {
            const double* WN = c.Wk(N);
            for (int e = lane; e < NX * NX; e += 32) {
                const int r = e / NX, q = e % NX;
                sT[e] = (useW ? WN[e] : 0.0) + (r == q ? Sig[c.ix(N) + r] : 0.0);
            }
            __syncwarp();
            if (pb.ng > 0) add_cond(c, N, sT, NX);
            bad += transform_T(c, sT, sM, c.icd(N));
            double* TN = c.ws + c.L.T + N * NX * NX;
            for (int e = lane; e < NX * NX; e += 32) TN[e] = sT[e];
            __syncwarp();
        }
        for (int k = N - 1; k >= 0; --k) {
            const double* Jg = c.Jk(k);
            for (int e = lane; e < NX * NZ; e += 32) sJ[e] = Jg[e];
            __syncwarp();
            const double* Wg = c.Wk(k);
            for (int j = lane; j < NZ; j += 32) {
                double acc[NX];
#pragma unroll
                for (int i = 0; i < NX; ++i) acc[i] = 0.0;
                for (int l = 0; l < NX; ++l) {
                    const double jl = sJ[l * NZ + j];
#pragma unroll
                    for (int i = 0; i < NX; ++i) acc[i] += sT[l * NX + i] * jl;
                }
                double mcol[NZ];
                const double sg = Sig[c.zidx(k, j)];
#pragma unroll
                for (int a = 0; a < NZ; ++a) mcol[a] = (useW ? Wg[a * NZ + j] : 0.0) + (a == j ? sg : 0.0);
#pragma unroll
                for (int l = 0; l < NX; ++l) {
                    const double t = acc[l];
#pragma unroll
                    for (int a = 0; a < NZ; ++a) mcol[a] += sJ[l * NZ + a] * t;
                }
#pragma unroll
                for (int a = 0; a < NZ; ++a) sM[a * NZ + j] = mcol[a];
            }
            __syncwarp();
            if (k >= 1 && pb.ng > 0) add_cond(c, k, sM, NZ);
            // eliminate the controls: pivots NX .. NZ-1
            for (int p = 0; p < NU; ++p) {
                const int pp = NX + p;
                double d = sM[pp * NZ + pp];
                if (!(d > 0.0)) { bad++; if (d == 0.0) { nzero++; d = 1.0; } }
                for (int b = lane; b < NZ; b += 32) {
                    if (b < NX || b > pp) {
                        const double lb = sM[pp * NZ + b] / d;
                        for (int a = 0; a < NX; ++a) sM[a * NZ + b] -= sM[a * NZ + pp] * lb;
                        for (int a = pp + 1; a < NZ; ++a) sM[a * NZ + b] -= sM[a * NZ + pp] * lb;
                    }
                }
                __syncwarp();
            }
            // store L (unit lower, D on the diagonal) and X = Mxu-columns scaled
            double* Lg = c.ws + c.L.Lf + k * NU * NU;
            double* Xg = c.ws + c.L.Xf + k * NX * NU;
            for (int e = lane; e < NU * NU; e += 32) {
                const int r = e / NU, p = e % NU;
                double d = sM[(NX + p) * NZ + NX + p];
                const double dd = (d == 0.0) ? 1.0 : d;
                Lg[e] = (r == p) ? dd : (r > p ? sM[(NX + r) * NZ + NX + p] / dd : 0.0);
            }
            for (int e = lane; e < NX * NU; e += 32) {
                const int r = e / NU, p = e % NU;
                double d = sM[(NX + p) * NZ + NX + p];
                if (d == 0.0) d = 1.0;
                Xg[e] = sM[r * NZ + NX + p] / d;
            }
            for (int e = lane; e < NX * NX; e += 32) {
                const int r = e / NX, q = e % NX;
                sT[e] = 0.5 * (sM[r * NZ + q] + sM[q * NZ + r]);
            }
            __syncwarp();
            bad += transform_T(c, sT, sM, c.icd(k));
            double* Tg = c.ws + c.L.T + k * NX * NX;
            for (int e = lane; e < NX * NX; e += 32) Tg[e] = sT[e];
            __syncwarp();
        }
        return bad;
    }

    // condensed right-hand side contribution to x_k position entry (agent a, coordinate i), k >= 1:
    //   sum_j G_j^T Dg_j (rc_g,j + rp_s,j / sig_j)
    __device__ static double cond_rhs(const X& c, const double* rp, const double* rc, int k, int a, int i) {
        const Pb& pb = c.pb;
        const double* gv = c.ws + c.L.gv + (k - 1) * pb.ng * PD;
        double s = 0.0;
        for (int j = 0; j < pb.ng; ++j) {
            double sgn = 1.0;
            if (pb.family == JIPM_FAM_MULTIQUAD) {
                int pa, pb2; c.pair_ab(j, pa, pb2);
                sgn = (pa == a) ? 1.0 : (pb2 == a ? -1.0 : 0.0);
                if (sgn == 0.0) continue;
            }
            const double sig = c.ws[c.L.Sig + c.is(k) + j];
            s += sgn * gv[j * PD + i] * Dg(c, k, j) * (rc[c.icg(k) + j] + rp[c.is(k) + j] / sig);
        }
        return s;
    }

    // Solve with the current factor: [dx; dy] = K^{-1} [rp; rc].
    __device__ static void solve(const X& c, const double* rp, const double* rc, double* dx, double* dy) {
        const Pb& pb = c.pb;
        const int N = pb.N, lane = c.lane;
        double* sp = c.sm + C::SM_V;        // p vector  [NX]
        double* sw = sp + NX;               // w         [NX]
        double* sv = sw + NX;               // temp      [NX]
        double* sx = sv + NX;               // x_k       [NX]
        double* st = sx + NX;               // t / u     [NU]
        const double* Dc = c.ws + c.L.Dc;
        double* wv = c.ws + c.L.wv;
        double* tv = c.ws + c.L.tv;
        // ---- backward vector pass ----
        for (int i = lane; i < NX; i += 32) {
            double v = rp[c.ix(N) + i];
            const int ag = i / AX, ii = i % AX;
            if (ii < PD && pb.ng > 0) v += cond_rhs(c, rp, rc, N, ag, ii);
            sp[i] = v;
        }
        __syncwarp();
        for (int k = N - 1; k >= 0; --k) {
            const double* Tn = c.ws + c.L.T + (k + 1) * NX * NX;
            const double* Jg = c.Jk(k);
            const double* Lg = c.ws + c.L.Lf + k * NU * NU;
            const double* Xg = c.ws + c.L.Xf + k * NX * NU;
            const int r0 = c.icd(k + 1);
            for (int i = lane; i < NX; i += 32) sv[i] = rc[r0 + i] + Dc[r0 + i] * sp[i];
            __syncwarp();
            for (int i = lane; i < NX; i += 32) {
                double s = -sp[i];
#pragma unroll 4
                for (int l = 0; l < NX; ++l) s += Tn[l * NX + i] * sv[l];
                sw[i] = s; wv[k * NX + i] = s;
            }
            __syncwarp();
            for (int p = lane; p < NU; p += 32) {
                double s = rp[c.iu(k) + p];
#pragma unroll 4
                for (int l = 0; l < NX; ++l) s -= Jg[l * NZ + NX + p] * sw[l];
                st[p] = s;
            }
            __syncwarp();
            // t = L^{-1} rhat (column-oriented forward substitution)
            for (int p = 0; p < NU - 1; ++p) {
                const double tp = st[p];
                __syncwarp();
                for (int q = p + 1 + lane; q < NU; q += 32) st[q] -= Lg[q * NU + p] * tp;
                __syncwarp();
            }
            for (int i = lane; i < NX; i += 32) {
                double s = rp[c.ix(k) + i];
                const int ag = i / AX, ii = i % AX;
                if (k >= 1 && ii < PD && pb.ng > 0) s += cond_rhs(c, rp, rc, k, ag, ii);
#pragma unroll 4
                for (int l = 0; l < NX; ++l) s -= Jg[l * NZ + i] * sw[l];
#pragma unroll 4
                for (int p = 0; p < NU; ++p) s -= Xg[i * NU + p] * st[p];
                sv[i] = s;
            }
            for (int p = lane; p < NU; p += 32) tv[k * NU + p] = st[p] / Lg[p * NU + p];
            __syncwarp();
            for (int i = lane; i < NX; i += 32) sp[i] = sv[i];
            __syncwarp();
        }
        // ---- stage 0: nu_0 = T_0 (rc_0 + D_0 p_0) - p_0, x_0 = rc_0 - D_0 nu_0 ----
        {
            const double* T0 = c.ws + c.L.T;
            for (int i = lane; i < NX; i += 32) sv[i] = rc[i] + Dc[i] * sp[i];
            __syncwarp();
            for (int i = lane; i < NX; i += 32) {
                double s = -sp[i];
#pragma unroll 4
                for (int l = 0; l < NX; ++l) s += T0[l * NX + i] * sv[l];
                const double x0 = rc[i] - Dc[i] * s;
                sx[i] = x0; dx[i] = x0; dy[i] = -s;
            }
            __syncwarp();
        }
        // ---- forward pass ----
        for (int k = 0; k < N; ++k) {
            const double* Tn = c.ws + c.L.T + (k + 1) * NX * NX;
            const double* Jg = c.Jk(k);
            const double* Lg = c.ws + c.L.Lf + k * NU * NU;
            const double* Xg = c.ws + c.L.Xf + k * NX * NU;
            for (int p = lane; p < NU; p += 32) {
                double s = tv[k * NU + p];
#pragma unroll 4
                for (int i = 0; i < NX; ++i) s -= Xg[i * NU + p] * sx[i];
                st[p] = s;
            }
            __syncwarp();
            // u = L^{-T} q (backward substitution)
            for (int p = NU - 1; p > 0; --p) {
                const double up = st[p];
                __syncwarp();
                for (int q = lane; q < p; q += 32) st[q] -= Lg[p * NU + q] * up;
                __syncwarp();
            }
            for (int p = lane; p < NU; p += 32) dx[c.iu(k) + p] = st[p];
            for (int i = lane; i < NX; i += 32) {
                const double* Jr = Jg + i * NZ;
                double s = 0.0;
#pragma unroll 4
                for (int a = 0; a < NX; ++a) s += Jr[a] * sx[a];
#pragma unroll 4
                for (int a = 0; a < NU; ++a) s += Jr[NX + a] * st[a];
                sv[i] = s;
            }
            __syncwarp();
            const int r0 = c.icd(k + 1);
            for (int i = lane; i < NX; i += 32) {
                double nu = wv[k * NX + i];
#pragma unroll 4
                for (int l = 0; l < NX; ++l) nu += Tn[l * NX + i] * sv[l];
                const double xn = sv[i] - Dc[r0 + i] * nu + rc[r0 + i];
                dx[c.ix(k + 1) + i] = xn; dy[r0 + i] = -nu; sp[i] = xn;
            }
            __syncwarp();
            for (int i = lane; i < NX; i += 32) sx[i] = sp[i];
            __syncwarp();
        }
        // ---- slack / inequality-multiplier recovery ----
        const double* gv = c.ws + c.L.gv;
        for (int it = lane; it < N * pb.ng; it += 32) {
            const int k = it / pb.ng + 1, j = it % pb.ng;
            const double sig = c.ws[c.L.Sig + c.is(k) + j];
            const double rps = rp[c.is(k) + j];
            const double dyg = Dg(c, k, j) * (c.G_dot(gv, dx, k, j) - rc[c.icg(k) + j] - rps / sig);
            dy[c.icg(k) + j] = dyg;
            dx[c.is(k) + j] = (rps + dyg) / sig;
        }
        __syncwarp();
    }
};

}  // namespace jipm
