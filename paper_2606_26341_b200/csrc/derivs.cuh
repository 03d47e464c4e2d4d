// derivs.cuh -- batched derivative evaluation: grad f, Jacobian stage blocks J_k = dF/d(x_k,u_k), inequality
// gradient vectors, and the Lagrangian Hessian stage blocks W_k = sigma_f Hess f + sum_j y_j Hess c_j
// ("sparse derivative evaluation").
#pragma once
#include <type_traits>
#include "core.cuh"

namespace jipm {

template <class C>
__device__ void Ctx<C>::dyn_derivs(const double* x, const double* y) {
    const int N = pb->N;
    if constexpr (std::is_same<typename C::Dyn, PointmassDyn>::value) {
        // linear dynamics: constant Jacobian, zero Hessian
        const double h = pb->dt;
        for (int it = lane; it < N * NX * NZ; it += NT) {
            const int k = it / (NX * NZ), e = it % (NX * NZ), r = e / NZ, cidx = e % NZ;
            double v = 0.0;
            if (cidx == r) v = 1.0;
            else if (r < 2 && cidx == r + 2) v = h;
            else if (r < 2 && cidx == r + 4) v = 0.5 * h * h;
            else if (r >= 2 && cidx == r + 2) v = h;
            Jk(k)[r * LDJ + cidx] = v;
        }
        for (int it = lane; it < N * NZ * NZ + NX * NX; it += NT) vh(L->W)[it] = 0.0;
        tm.sync();
    } else if constexpr (std::is_same<typename C::Dyn, QuatDyn>::value) {
        // 13-state quaternion vehicle: the same RK4 chain as below, matrix-free: the products with Df and with the
        // adjoint-contracted Hessian at each RK point come from the generated functions of dyn_quat_gen.cuh.
        //   xi_1 = x, xi_{s+1} = x + a_{s+1} h f(xi_s);   mu_4 = b_4 lam, mu_{s-1} = b_{s-1} lam + a_s h Df_x(xi_s)^T mu_s
        //   column j of the chain: Y_1 = e_j, K_s = Df(xi_s) (Y_s, e_u), Y_{s+1} = e_j + a_{s+1} h K_s, J e_j = e_j + h sum b_s K_s
        //   lam^T Hess F = sum_s (Y_s, e_u)^T [sum_i mu_s,i Hess f_i(xi_s)] (Y_s, e_u)
        const double h = pb->dt;
        double* rk = v(L->rk);
        // ---- phase 1: thread <-> stage: the RK points and their adjoint weights ----
        for (int k = lane; k < N; k += NT) {
            double xa[13], ua[4], lam[13], kk[13], xi[13];
#pragma unroll
            for (int i = 0; i < 13; ++i) { xa[i] = x[ix(k) + i]; lam[i] = -y[icd(k + 1) + i]; }
#pragma unroll
            for (int i = 0; i < 4; ++i) ua[i] = x[iu(k) + i];
            double* out = rk + (k * 4) * RKW;
#pragma unroll
            for (int i = 0; i < 13; ++i) { xi[i] = xa[i]; out[i] = xi[i]; }
#pragma unroll 1
            for (int s = 1; s < 4; ++s) {
                quat_ode(xi, ua, kk);
                const double as = (s == 3) ? h : 0.5 * h;
#pragma unroll
                for (int i = 0; i < 13; ++i) { xi[i] = xa[i] + as * kk[i]; out[s * RKW + i] = xi[i]; }
            }
            double mu[13], t[13];
#pragma unroll
            for (int i = 0; i < 13; ++i) mu[i] = (h / 6.0) * lam[i];
#pragma unroll 1
            for (int s = 3; s >= 0; --s) {
#pragma unroll
                for (int i = 0; i < 13; ++i) out[s * RKW + 13 + i] = mu[i];
                if (s > 0) {
#pragma unroll
                    for (int i = 0; i < 13; ++i) xi[i] = out[s * RKW + i];
                    quat_vjp(xi, ua, mu, t);
                    const double as = (s == 3) ? h : 0.5 * h;
                    const double bprev = (s == 1) ? h / 6.0 : h / 3.0;
#pragma unroll
                    for (int i = 0; i < 13; ++i) mu[i] = bprev * lam[i] + as * t[i];
                }
            }
        }
        tm.sync();
        // ---- phase 2: warp <-> stage, lane j < 17 <-> column j of z = (x(13), u(4)) ----
        constexpr int NWP = NT / 32;
        const int wid = lane >> 5, j = lane & 31;
        const bool act = j < 17;
        double* sV = smt(C::SM_G) + wid * (17 * 17);
        for (int k0 = 0; k0 < N; k0 += NWP) {
            const int k = k0 + wid;
            const bool valid = k < N;
            const int kc = valid ? k : N - 1;
            double Y[13], Jc[13], Hc[17], uj[4], ua[4];
#pragma unroll
            for (int i = 0; i < 13; ++i) { Y[i] = (i == j) ? 1.0 : 0.0; Jc[i] = Y[i]; }
#pragma unroll
            for (int i = 0; i < 4; ++i) { uj[i] = (j == 13 + i) ? 1.0 : 0.0; ua[i] = x[iu(kc) + i]; }
#pragma unroll
            for (int i = 0; i < 17; ++i) Hc[i] = 0.0;
#pragma unroll 1
            for (int s = 0; s < 4; ++s) {
                const double* in = rk + (kc * 4 + s) * RKW;
                double xi[13], mu[13], K[13], V[17], t[17];
#pragma unroll
                for (int i = 0; i < 13; ++i) { xi[i] = in[i]; mu[i] = in[13 + i]; K[i] = 0.0; }
#pragma unroll
                for (int i = 0; i < 13; ++i) V[i] = Y[i];
#pragma unroll
                for (int i = 0; i < 4; ++i) V[13 + i] = uj[i];
                if (act) {
#pragma unroll
                    for (int e = 0; e < 17; ++e) sV[e * 17 + j] = V[e];
                    quat_hvp(xi, ua, mu, V, t);
                    quat_jvp(xi, ua, Y, uj, K);
                }
                __syncwarp();
                if (act) {
#pragma unroll
                    for (int c2 = 0; c2 < 17; ++c2) {
                        double acc = Hc[c2];
#pragma unroll
                        for (int e = 0; e < 17; ++e) acc += sV[e * 17 + c2] * t[e];
                        Hc[c2] = acc;
                    }
                }
                __syncwarp();
                const double bw = (s == 0 || s == 3) ? h / 6.0 : h / 3.0;
                const double an = (s == 2) ? h : 0.5 * h;
#pragma unroll
                for (int i = 0; i < 13; ++i) {
                    Jc[i] += bw * K[i];
                    Y[i] = ((i == j) ? 1.0 : 0.0) + an * K[i];
                }
            }
            if (valid && act) {
                double* Jb = Jk(k);
#pragma unroll
                for (int i = 0; i < 13; ++i) Jb[i * LDJ + j] = Jc[i];
                double* Wb = Wk(k);
#pragma unroll
                for (int c2 = 0; c2 < 17; ++c2) Wb[c2 * NZ + j] = Hc[c2];
            }
        }
        for (int it = lane; it < NX * NX; it += NT) Wk(N)[it] = 0.0;
        tm.sync();
    } else {
        const double h = pb->dt;
        double* rk = v(L->rk);
        if (NA > 1) {
            for (int it = lane; it < N * NZ * NZ; it += NT) vh(L->W)[it] = 0.0;
        }
        // ---- phase 1: lane <-> (stage, agent): RK points, Df entries, adjoints, contracted 7x7 Hessians ----
        for (int it = lane; it < N * NA; it += NT) {
            const int k = it / NA, a = it % NA;
            double xa[12], ua[4], lam[12], kk[12], xi[12];
            QuadBasics bs[4];
#pragma unroll
            for (int i = 0; i < 12; ++i) { xa[i] = x[ix(k) + 12 * a + i]; lam[i] = -y[icd(k + 1) + 12 * a + i]; }
#pragma unroll
            for (int i = 0; i < 4; ++i) ua[i] = x[iu(k) + 4 * a + i];
            QuadDyn::ode(xa, ua, kk, bs[0]);
#pragma unroll
            for (int i = 0; i < 12; ++i) xi[i] = xa[i] + (0.5 * h) * kk[i];
            QuadDyn::ode(xi, ua, kk, bs[1]);
#pragma unroll
            for (int i = 0; i < 12; ++i) xi[i] = xa[i] + (0.5 * h) * kk[i];
            QuadDyn::ode(xi, ua, kk, bs[2]);
#pragma unroll
            for (int i = 0; i < 12; ++i) xi[i] = xa[i] + h * kk[i];
            QuadDyn::ode(xi, ua, kk, bs[3]);
            // backward: mu_4 = b_4 lam; mu_{i-1} = b_{i-1} lam + a_i h Df_x(xi_i)^T mu_i
            double mu[12], t[12];
#pragma unroll
            for (int i = 0; i < 12; ++i) mu[i] = (h / 6.0) * lam[i];
#pragma unroll
            for (int s = 3; s >= 0; --s) {
                double* out = rk + (it * 4 + s) * RKW;
                double D[26], H[16];
                QuadDyn::dentries(bs[s], D);
                quad_hentries(bs[s], mu, H);
#pragma unroll
                for (int i = 0; i < 26; ++i) out[i] = D[i];
#pragma unroll
                for (int i = 0; i < 16; ++i) out[26 + i] = H[i];
                if (s > 0) {
                    quad_dfxT(D, mu, t);
                    const double as = (s == 3) ? h : 0.5 * h;
                    const double bprev = (s == 1) ? h / 6.0 : h / 3.0;
#pragma unroll
                    for (int i = 0; i < 12; ++i) mu[i] = bprev * lam[i] + as * t[i];
                }
            }
        }
        tm.sync();
        // ---- phase 2: 16-thread group <-> (stage, agent), thread <-> column j of z = (x(12), u(4)) ----------
        // (two groups share a warp and run the same instruction stream: __syncwarp orders the staging)
        const int grp = lane >> 4, j = lane & 15;
        constexpr int NGRP = C::NGRP;  // threads beyond 16 * NGRP idle through this phase
        double* sV = smt(C::SM_G) + grp * (7 * 16);
        const int nit = N * NA;
        for (int it0 = 0; it0 < nit && grp < NGRP; it0 += NGRP) {
            const int it = it0 + grp;
            const bool valid = it < nit;
            const int itc = valid ? it : nit - 1;
            const int k = itc / NA, a = itc % NA;
            double Y[12], Jc[12], Hc[16], uj[4];
#pragma unroll
            for (int i = 0; i < 12; ++i) { Y[i] = (i == j) ? 1.0 : 0.0; Jc[i] = Y[i]; }
#pragma unroll
            for (int i = 0; i < 4; ++i) uj[i] = (j == 12 + i) ? 1.0 : 0.0;
#pragma unroll
            for (int i = 0; i < 16; ++i) Hc[i] = 0.0;
            const double Tj = (j >= 12) ? 1.0 : 0.0;
#pragma unroll 1
            for (int s = 0; s < 4; ++s) {
                const double* in = rk + (itc * 4 + s) * RKW;
                double D[26], H[16], K[12], V[7], t[7];
#pragma unroll
                for (int i = 0; i < 26; ++i) D[i] = in[i];
#pragma unroll
                for (int i = 0; i < 16; ++i) H[i] = in[26 + i];
                V[0] = Y[3]; V[1] = Y[4]; V[2] = Y[5]; V[3] = Y[9]; V[4] = Y[10]; V[5] = Y[11]; V[6] = Tj;
#pragma unroll
                for (int e = 0; e < 7; ++e) sV[e * 16 + j] = V[e];
                quad_hmul(H, V, t);
                quad_dfcol(D, Y, uj, K);
                __syncwarp();
#pragma unroll
                for (int c2 = 0; c2 < 16; ++c2) {
                    double acc = Hc[c2];
#pragma unroll
                    for (int e = 0; e < 7; ++e) acc += sV[e * 16 + c2] * t[e];
                    Hc[c2] = acc;
                }
                __syncwarp();
                const double bw = (s == 0 || s == 3) ? h / 6.0 : h / 3.0;
                const double an = (s == 2) ? h : 0.5 * h;  // a_{s+2} h for the next point
#pragma unroll
                for (int i = 0; i < 12; ++i) {
                    Jc[i] += bw * K[i];
                    Y[i] = ((i == j) ? 1.0 : 0.0) + an * K[i];
                }
            }
            if (valid) {
                const int col = (j < 12) ? 12 * a + j : NX + 4 * a + (j - 12);
                double* Jb = Jk(k);
#pragma unroll
                for (int i = 0; i < 12; ++i) Jb[(12 * a + i) * LDJ + col] = Jc[i];
                double* Wb = Wk(k);
#pragma unroll
                for (int c2 = 0; c2 < 16; ++c2) {
                    const int row = (c2 < 12) ? 12 * a + c2 : NX + 4 * a + (c2 - 12);
                    Wb[row * NZ + col] = Hc[c2];
                }
            }
        }
        for (int it = lane; it < NX * NX; it += NT) Wk(N)[it] = 0.0;
        tm.sync();
    }
}

// grad f, J, W (+ objective and inequality curvature), inequality gradient vectors gv
template <class C>
__device__ void Ctx<C>::eval_derivs(const double* x, const double* y, double sigma_f) {
    const int N = pb->N;
    double* g = v(L->g);
    const double* tgt = vh(L->tgt);
    for (int i = lane; i < pb->n; i += NT) g[i] = 0.0;
    tm.sync();
    for (int it = lane; it < (N + 1) * NA * PD; it += NT) {
        const int ka = it / PD, i = it % PD, k = ka / NA, a = ka % NA;
        g[ix(k) + AX * a + i] = sigma_f * 2.0 * (x[ix(k) + AX * a + i] - tgt[it]);
    }
    for (int it = lane; it < N * NU; it += NT) {
        const int idx = iu(it / NU) + it % NU;
        g[idx] = sigma_f * 2.0 * pb->ru * x[idx];
    }
    // inequality gradient vectors
    double* gv = vh(L->gv);
    for (int it = lane; it < N * pb->ng; it += NT) {
        const int k = it / pb->ng + 1, j = it % pb->ng;
        if (pb->family == JIPM_FAM_MULTIQUAD) {
            int a, b; pair_ab(j, a, b);
#pragma unroll
            for (int i = 0; i < PD; ++i) gv[it * PD + i] = 2.0 * (x[ix(k) + AX * a + i] - x[ix(k) + AX * b + i]);
        } else {
            const double* ob = th + pb->th_obs + (PD + 1) * j;
#pragma unroll
            for (int i = 0; i < PD; ++i) gv[it * PD + i] = 2.0 * (x[ix(k) + i] - ob[i]);
        }
    }
    dyn_derivs(x, y);
    // objective curvature (diagonal) and inequality curvature 2 y_g I on positions
    for (int it = lane; it < (N + 1) * NA * PD; it += NT) {
        const int ka = it / PD, i = it % PD, k = ka / NA, a = ka % NA;
        const int r = AX * a + i, ld = (k < N) ? NZ : NX;
        double add = sigma_f * 2.0;
        if (k >= 1) {
            const double* yg = y + icg(k);
            if (pb->family == JIPM_FAM_MULTIQUAD) {
                for (int q = 0; q < pb->ng; ++q) {
                    int pa, pb2; pair_ab(q, pa, pb2);
                    if (pa == a || pb2 == a) {
                        add += 2.0 * yg[q];
                        const int other = (pa == a) ? pb2 : pa;
                        Wk(k)[r * ld + AX * other + i] -= 2.0 * yg[q];
                    }
                }
            } else {
                for (int q = 0; q < pb->ng; ++q) add += 2.0 * yg[q];
            }
        }
        Wk(k)[r * ld + r] += add;
    }
    for (int it = lane; it < N * NU; it += NT) {
        const int k = it / NU, r = NX + it % NU;
        Wk(k)[r * NZ + r] += sigma_f * 2.0 * pb->ru;
    }
    tm.sync();
}

}  // namespace jipm
