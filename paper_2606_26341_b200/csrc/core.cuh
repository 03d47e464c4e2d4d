// core.cuh -- solver context of one problem slot (= one team = one CTA): indexing, evaluation of f / c / derivatives,
// products with the stage-structured A and W of PAPER.md:90.  Everything here is a team-collective device function.
#pragma once
#include "common.cuh"
#include "dyn.cuh"

namespace jipm {

template <class Dyn_, int NA_, int NT_, bool HOT_SM_>
struct Cfg {
    using Dyn = Dyn_;
    static constexpr int NA = NA_;
    static constexpr int NT = NT_;  // threads per problem slot (team size)
    // the host guarantees that the "hot" group of the layout (factor blocks, sweep vectors, J, W, m-vectors) is
    // shared-memory resident: its accessor then yields pointers the compiler knows to be shared (LDS, not generic LD)
    static constexpr bool HOT_SM = HOT_SM_;
    static constexpr int AX = Dyn::AX, AU = Dyn::AU, PD = Dyn::PD;
    static constexpr int NX = AX * NA, NU = AU * NA, NZ = NX + NU;
    // fixed shared memory per team (doubles): T, J, M, TJ/Phi, Kf/Linv tiles of the stage sweep, the staging of the
    // quadrotor Hessian columns (7 x 16 per 16-thread group), the reduction scratch
    // row stride of the stage Jacobians J_k = [A B] (NX x NZ): odd in doubles, so that row-wise AND column-wise
    // accesses by consecutive threads fall on distinct shared-memory banks (stride NZ = 16 made every row-wise
    // product a 16-way bank conflict)
    static constexpr int LDJ = NZ + 1;
    static constexpr int SM_MSZ = (NZ * NZ > 2 * NX * NX) ? NZ * NZ : 2 * NX * NX;
    static constexpr int SM_T = 0, SM_J = SM_T + NX * NX, SM_M = SM_J + ((NX * LDJ + 1) & ~1), SM_M2 = SM_M + SM_MSZ, SM_TJ = SM_M2 + SM_MSZ;
    static constexpr int SM_K = SM_TJ + NX * NZ, SM_TILE_END = SM_K + NU * NX + NU * NU;
    static constexpr int NGRP = (NT / 16 < 16) ? NT / 16 : 16;  // 16-thread groups of the Hessian column propagation
    // the staging of the Hessian columns aliases the factorisation tiles M, M2, TJ, K (derivative evaluation and
    // factorisation are never live at the same time)
    static constexpr int SM_G = SM_M;
    static constexpr int SM_G_END = SM_G + (Dyn::AX == 12 ? NGRP * 7 * 16 : (Dyn::AX == 13 ? (NT / 32) * 17 * 17 : 0));
    static constexpr int SM_RED = (SM_TILE_END > SM_G_END) ? SM_TILE_END : SM_G_END;
    static constexpr int SM_SPEC = SM_RED + 2 * (NT / 32) + 2;  // (theta, phi) of the speculative trials, one pair per warp
    static constexpr int SM_CNT = SM_SPEC + 2 * (NT / 32);  // 16 diagnostic cycle counters (64-bit), written by thread 0
    static constexpr int SM_TOTAL = SM_CNT + 16;
};

template <class C>
struct Ctx {
    static constexpr int NX = C::NX, NU = C::NU, NZ = C::NZ, PD = C::PD, AX = C::AX, AU = C::AU, NA = C::NA, LDJ = C::LDJ;
    static constexpr int NT = C::NT;
    PbProxy pb;        // launch arguments: constant memory (common.cuh)
    LayProxy L;
    OptProxy o;
    double* ws;        // this team's global workspace, shifted so that ws + off is valid for off >= L->nsm
    double* sm;        // this team's fixed shared memory (tiles, staging, reduction scratch)
    double* smd;       // this team's shared-memory part of the workspace layout (offsets < L->nsm)
    const double* th;  // theta of the current problem
    int lane;          // thread index inside the team, 0 .. NT-1
    mutable Team<NT> tm;
    // index maps built once per kernel (no runtime integer division in the hot loops):
    //   imap[i] of primal entry i: (k << 16) | (j << 8) | a   a < NZ: entry a of z_k = (x_k, u_k); a = 255: slack j of knot k
    //   cmap[r] of equality row r: (k << 16) | (j << 8) | rr  rr < NX: row rr of dyn_{k+1}; 255: inequality j of knot k; 254: x_0 row
    const int* imap; const int* cmap;
    // Diagnostic cycle counters live in shared memory and only thread 0 updates them (as registers of every thread they
    // cost 32 registers of a kernel that is register-bound): 0-7 = phases of the iteration (stats[8..15]), 8-15 = the
    // factorisation's sub-phases and iteration blocks (stats[16..23]).
    __device__ __forceinline__ void tick(int idx, long long cycles) const {
        if (lane == 0) reinterpret_cast<unsigned long long*>(jipm_smem + C::SM_CNT)[idx] += (unsigned long long)cycles;
    }
    __device__ __forceinline__ unsigned long long counter(int idx) const {
        return reinterpret_cast<unsigned long long*>(jipm_smem + C::SM_CNT)[idx];
    }

    __device__ Ctx(double* ws_, double* sm_, int tid_)
        : ws(ws_ - g_A.L.nsm), sm(sm_), smd(sm_ + C::SM_TOTAL), th(nullptr), lane(tid_) {
        if (tid_ < 16) reinterpret_cast<unsigned long long*>(jipm_smem + C::SM_CNT)[tid_] = 0ull;
        tm.tid = tid_; tm.flip = 0; tm.red = sm_ + C::SM_RED;
    }

    __device__ void build_maps() {
        int* im = reinterpret_cast<int*>(vh(L->imap));
        int* cm = reinterpret_cast<int*>(vh(L->cmap));
        for (int idx = lane; idx < pb->n; idx += NT) {
            int v;
            if (idx < NX) v = idx;
            else {
                const int q = idx - NX, kk = q / pb->blk, r = q % pb->blk;
                if (r < NU) v = (kk << 16) | (NX + r);
                else if (r < NU + NX) v = ((kk + 1) << 16) | (r - NU);
                else v = ((kk + 1) << 16) | ((r - NU - NX) << 8) | 255;
            }
            im[idx] = v;
        }
        for (int r = lane; r < pb->m; r += NT) {
            int v;
            if (r < NX) v = 254;
            else {
                const int q = r - NX, k = q / pb->cblk, rr = q % pb->cblk;
                v = (rr < NX) ? ((k << 16) | rr) : (((k + 1) << 16) | ((rr - NX) << 8) | 255);
            }
            cm[r] = v;
        }
        imap = im; cmap = cm;
        tm.sync();
    }

    // ---- stage-order index helpers (same layout as include/jipm.h) -----------------------------------
    __device__ __forceinline__ int ix(int k) const { return k == 0 ? 0 : NX + (k - 1) * pb->blk + NU; }
    __device__ __forceinline__ int iu(int k) const { return NX + k * pb->blk; }
    __device__ __forceinline__ int is(int k) const { return NX + (k - 1) * pb->blk + NU + NX; }
    __device__ __forceinline__ int icd(int k) const { return k == 0 ? 0 : NX + (k - 1) * pb->cblk; }
    __device__ __forceinline__ int icg(int k) const { return NX + (k - 1) * pb->cblk + NX; }
    __device__ __forceinline__ int zidx(int k, int a) const { return a < NX ? ix(k) + a : iu(k) + a - NX; }
    __device__ __forceinline__ double* Jk(int k) const { return vh(L->J) + k * (NX * LDJ); }
    __device__ __forceinline__ double* Wk(int k) const { return vh(L->W) + k * (NZ * NZ); }  // k == N: NX x NX
    // workspace array at layout offset off: the first L->nsm doubles of the layout live in shared memory (the
    // hot vectors and factor blocks), the rest in this slot's global workspace (L2-resident scratch)
    __device__ __forceinline__ double* v(int off) const { return off < L->nsm ? smd + off : ws + off; }
    // same for an array of the hot group: addressed off the CTA's shared array itself (one team per CTA), so that
    // the compiler emits shared loads/stores (LDS/STS) instead of generic ones
    __device__ __forceinline__ double* vh(int off) const {
        if constexpr (C::HOT_SM) return jipm_smem + C::SM_TOTAL + off;
        else return v(off);
    }
    // fixed tile at offset off of this team's shared memory
    __device__ __forceinline__ double* smt(int off) const { return jipm_smem + off; }

    // pair q -> agents (a,b), a<b, row-major enumeration
    __device__ __forceinline__ void pair_ab(int q, int& a, int& b) const {
        int aa = 0, rem = q;
        while (rem >= NA - 1 - aa) { rem -= NA - 1 - aa; ++aa; }
        a = aa; b = aa + 1 + rem;
    }

    // inequality h_j(x_k) >= 0 (obstacle or pair separation), value
    __device__ double ineq_val(const double* x, int k, int j) const {
        double s = 0.0;
        if (pb->family == JIPM_FAM_MULTIQUAD) {
            int a, b; pair_ab(j, a, b);
            const double* pa = x + ix(k) + AX * a; const double* pb_ = x + ix(k) + AX * b;
#pragma unroll
            for (int i = 0; i < PD; ++i) { double d = pa[i] - pb_[i]; s += d * d; }
            return s - 0.25;
        }
        const double* p = x + ix(k);
        const double* ob = th + pb->th_obs + (PD + 1) * j;
#pragma unroll
        for (int i = 0; i < PD; ++i) { double d = p[i] - ob[i]; s += d * d; }
        return s - ob[PD] * ob[PD];
    }
    // G_{k,j} . d  with the gradient vector stored in gv (2*(p-c) or 2*(p_a-p_b))
    __device__ double G_dot(const double* gv, const double* d, int k, int j) const {
        const double* g = gv + ((k - 1) * pb->ng + j) * PD;
        double s = 0.0;
        if (pb->family == JIPM_FAM_MULTIQUAD) {
            int a, b; pair_ab(j, a, b);
            const double* da = d + ix(k) + AX * a; const double* db = d + ix(k) + AX * b;
#pragma unroll
            for (int i = 0; i < PD; ++i) s += g[i] * (da[i] - db[i]);
        } else {
            const double* dp = d + ix(k);
#pragma unroll
            for (int i = 0; i < PD; ++i) s += g[i] * dp[i];
        }
        return s;
    }
    // (G_k^T s)_(agent a, coordinate i) for a per-constraint weight vector sv (indexed [j], stage k)
    __device__ double GT_entry(const double* gv, const double* sv, int k, int a, int i) const {
        const double* g = gv + (k - 1) * pb->ng * PD;
        double s = 0.0;
        if (pb->family == JIPM_FAM_MULTIQUAD) {
            for (int j = 0; j < pb->ng; ++j) {
                int pa, pb2; pair_ab(j, pa, pb2);
                if (pa == a) s += g[j * PD + i] * sv[j];
                else if (pb2 == a) s -= g[j * PD + i] * sv[j];
            }
        } else {
            for (int j = 0; j < pb->ng; ++j) s += g[j * PD + i] * sv[j];
        }
        return s;
    }

    // ---- f, c at a point (line-search trial evaluation) --------------------------------
    // returns f; writes c[m]; theta = ||c||_1, cmax = ||c||_inf; fin = all finite
    __device__ __noinline__ double eval_fc(const double* x, double* c, double& theta, double& cmax, bool& fin) const {
        const int N = pb->N;
        double f = 0.0;
        const double* tgt = vh(L->tgt);
        for (int it = lane; it < (N + 1) * NA; it += NT) {
            const int k = it / NA, a = it % NA;
            const double* p = x + ix(k) + AX * a;
            double s = 0.0;
#pragma unroll
            for (int i = 0; i < PD; ++i) { double d = p[i] - tgt[it * PD + i]; s += d * d; }
            f += s;
        }
        for (int it = lane; it < N * NU; it += NT) {
            const double u = x[iu(it / NU) + it % NU];
            f += pb->ru * (u * u);
        }
        f = tm.sum(f);
        double th1 = 0.0, cm = 0.0;
        for (int i = lane; i < NX; i += NT) {
            const double v = x[i] - th[i];
            c[i] = v; th1 += fabs(v); cm = fmax(cm, fabs(v));
        }
        for (int it = lane; it < N * NA; it += NT) {
            const int k = it / NA, a = it % NA;
            double xa[AX], ua[AU], Fv[AX];
#pragma unroll
            for (int i = 0; i < AX; ++i) xa[i] = x[ix(k) + AX * a + i];
#pragma unroll
            for (int i = 0; i < AU; ++i) ua[i] = x[iu(k) + AU * a + i];
            C::Dyn::F(xa, ua, pb->dt, Fv);
#pragma unroll
            for (int i = 0; i < AX; ++i) {
                const double v = x[ix(k + 1) + AX * a + i] - Fv[i];
                c[icd(k + 1) + AX * a + i] = v; th1 += fabs(v); cm = fmax(cm, fabs(v));
            }
        }
        for (int it = lane; it < N * pb->ng; it += NT) {
            const int k = it / pb->ng + 1, j = it % pb->ng;
            const double v = ineq_val(x, k, j) - x[is(k) + j];
            c[icg(k) + j] = v; th1 += fabs(v); cm = fmax(cm, fabs(v));
        }
        theta = tm.sum(th1);
        cmax = tm.max(cm);
        fin = isfinite(f) && isfinite(theta);
        tm.sync();
        return f;
    }

    // ---- A d (m-vector) and A^T y (n-vector) with the stage blocks J_k and the inequality gradients -----
    __device__ void A_mul(const double* d, double* out) const {
        const double* gv = vh(L->gv);
        for (int r = lane; r < pb->m; r += NT) {
            double s;
            const int cmv = cmap[r], rr = cmv & 255, k = cmv >> 16;
            if (rr == 254) s = d[r];
            else if (rr < NX) {
                const double* Jr = Jk(k) + rr * LDJ;
                s = d[ix(k + 1) + rr];
                const int ar = (NA == 1) ? 0 : rr / AX;  // J_k is block diagonal over the agents
                const double* dxk = d + ix(k) + AX * ar; const double* duk = d + iu(k) + AU * ar;
#pragma unroll 4
                for (int a = 0; a < AX; ++a) s -= Jr[AX * ar + a] * dxk[a];
#pragma unroll 4
                for (int a = 0; a < AU; ++a) s -= Jr[NX + AU * ar + a] * duk[a];
            } else {
                const int j = (cmv >> 8) & 255;
                s = G_dot(gv, d, k, j) - d[is(k) + j];
            }
            out[r] = s;
        }
        tm.sync();
    }
    __device__ double AT_entry(const double* y, int idx) const {
        const double* gv = vh(L->gv);
        const int imv = imap[idx], k = imv >> 16, a = imv & 255;  // x_k[a] or u_k[a-NX]
        if (a == 255) return -y[icg(k) + ((imv >> 8) & 255)];
        double s = 0.0;
        if (k < pb->N) {
            const int ac = (NA == 1) ? 0 : (a < NX ? a / AX : (a - NX) / AU);  // J_k is block diagonal over the agents
            const double* Jc = Jk(k) + AX * ac * LDJ + a; const double* yn = y + icd(k + 1) + AX * ac;
#pragma unroll 4
            for (int l = 0; l < AX; ++l) s -= Jc[l * LDJ] * yn[l];
        }
        if (a < NX) {
            s += y[icd(k) + a];
            const int ag = a / AX, i = a % AX;
            if (k >= 1 && i < PD) s += GT_entry(gv, y + icg(k), k, ag, i);
        }
        return s;
    }
    // (W d)_idx.  W is symmetric: column idx is read instead of row idx, so that consecutive threads read consecutive
    // addresses (row access with stride NZ is a 16-way shared-memory bank conflict)
    __device__ double W_entry(const double* d, int idx) const {
        const int imv = imap[idx], k = imv >> 16, a = imv & 255;
        if (a == 255) return 0.0;
        double s0 = 0.0, s1 = 0.0;
        if (k < pb->N) {
            const double* Wc = Wk(k) + a; const double* dxk = d + ix(k); const double* duk = d + iu(k);
#pragma unroll 4
            for (int b = 0; b + 1 < NX; b += 2) { s0 += Wc[b * NZ] * dxk[b]; s1 += Wc[(b + 1) * NZ] * dxk[b + 1]; }
            if constexpr (NX & 1) s0 += Wc[(NX - 1) * NZ] * dxk[NX - 1];
#pragma unroll 4
            for (int b = 0; b + 1 < NU; b += 2) { s0 += Wc[(NX + b) * NZ] * duk[b]; s1 += Wc[(NX + b + 1) * NZ] * duk[b + 1]; }
            if constexpr (NU & 1) s0 += Wc[(NX + NU - 1) * NZ] * duk[NU - 1];
        } else {
            const double* Wc = Wk(k) + a; const double* dxk = d + ix(k);
#pragma unroll 4
            for (int b = 0; b + 1 < NX; b += 2) { s0 += Wc[b * NX] * dxk[b]; s1 += Wc[(b + 1) * NX] * dxk[b + 1]; }
            if constexpr (NX & 1) s0 += Wc[(NX - 1) * NX] * dxk[NX - 1];
        }
        return s0 + s1;
    }

    __device__ __noinline__ void eval_derivs(const double* x, const double* y, double sigma_f);
    __device__ void dyn_derivs(const double* x, const double* y);
};

}  // namespace jipm
