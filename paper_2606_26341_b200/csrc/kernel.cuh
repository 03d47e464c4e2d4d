// kernel.cuh -- the persistent slot kernel: one team (CTA) per resident slot; a slot pops problem ids from the queue
// until it is empty (iteration-level batching: a finished problem is replaced at once, no
// slot ever waits for a straggler).  Also the debug load/store used by the parity tests.
#pragma once
#include "iter_impl.cuh"

namespace jipm {

template <class C>
__device__ void Solver<C>::dbg_load(const double* st) {
    const DbgLay D = make_dbglay(pb->n, pb->m, pb->N, NX, NZ);
    double* x = V(L->x); double* y = VH(L->y); double* zL = V(L->zL); double* zU = V(L->zU);
    for (int i = lane; i < pb->n; i += NT) { x[i] = st[D.x + i]; zL[i] = st[D.zL + i]; zU[i] = st[D.zU + i]; }
    for (int i = lane; i < pb->m; i += NT) y[i] = st[D.y + i];
    for (int i = lane; i < 2 * MAX_FILTER; i += NT) VH(L->filt)[i] = st[D.filt + i];
    mode = (int)st[D.rs + 0]; nX = mode ? pb->n + 2 * pb->m : pb->n;
    mu = st[D.sc + 0]; tau = st[D.sc + 1]; dw_last = st[D.sc + 2];
    theta_min = st[D.sc + 3]; theta_max = st[D.sc + 4];
    k = (int)st[D.sc + 5]; status = (int)st[D.sc + 6]; nfilt = (int)st[D.sc + 7];
    if (mode) {  // restoration state: regular scalars parked, (p, n), (z_p, z_n), x_R, D_R, the restoration filter
        mu_reg = st[D.rs + 1]; tau_reg = st[D.rs + 2]; dw_last_reg = st[D.rs + 3];
        theta_min_reg = st[D.rs + 4]; theta_max_reg = st[D.rs + 5]; nfilt_reg = (int)st[D.rs + 6];
        theta_entry = st[D.rs + 7]; zeta = st[D.rs + 8];
        Vec xv = VX(L->x); Vec zLv = VX(L->zL); Vec zUv = VX(L->zU);
        for (int j = lane; j < 2 * pb->m; j += NT) {
            xv[pb->n + j] = st[D.pn + j]; zLv[pb->n + j] = st[D.zpn + j]; zUv[pb->n + j] = 0.0;
        }
        double* xR = V(L->xR); double* DR2 = V(L->DR2);
        for (int i = lane; i < pb->n; i += NT) {
            const double xi = st[D.xR + i];
            xR[i] = xi;
            const double dr = fmin(1.0, 1.0 / fmax(fabs(xi), 1e-300));
            DR2[i] = dr * dr;
        }
        for (int i = lane; i < 2 * MAX_FILTER; i += NT) V(L->filtR)[i] = st[D.filtR + i];
    }
    // line-search memory of the active problem (Table I rows 3-5) and the watchdog's entry iterate / direction
    n_short = (int)st[D.ls + 0]; wd_active = (int)st[D.ls + 1]; wd_trials = (int)st[D.ls + 2];
    wd_theta = st[D.ls + 3]; wd_phi = st[D.ls + 4]; wd_gd = st[D.ls + 5]; wd_alpha = st[D.ls + 6];
    soft = (int)st[D.ls + 7]; soft_count = (int)st[D.ls + 8]; tiny_last = (int)st[D.ls + 9]; tiny_flag = (int)st[D.ls + 10];
    mu_free = (int)st[D.ls + 11]; mu_max = st[D.ls + 12]; nhist = (int)st[D.ls + 13];
    for (int q = 0; q < 4; ++q) hist[q] = st[D.ls + 14 + q];   // hist[j & 3] = j-th remembered KKT error
    acc_count = (int)st[D.ls + 18];
    if (wd_active) {
        const int nw = pb->n + 2 * pb->m;
        Vec w[6] = {VX(L->wx), VX(L->wzL), VX(L->wzU), VX(L->wdx), VX(L->wdzL), VX(L->wdzU)};
        for (int q = 0; q < 6; ++q)
            for (int i = lane; i < nX; i += NT) w[q][i] = st[D.wd + q * nw + i];
        for (int i = lane; i < pb->m; i += NT) { V(L->wy)[i] = st[D.wd + 6 * nw + i]; V(L->wdy)[i] = st[D.wd + 6 * nw + pb->m + i]; }
    }
    c.tm.sync();
    f = eval_point(VX(L->x), VH(L->c), theta, cmax, f_base, theta_base, cmax_base, f_pn, f_q);
}

template <class C>
__device__ void Solver<C>::dbg_store(double* st) {
    const DbgLay D = make_dbglay(pb->n, pb->m, pb->N, NX, NZ);
    c.tm.sync();
    for (int i = lane; i < pb->n; i += NT) {
        st[D.x + i] = V(L->x)[i]; st[D.zL + i] = V(L->zL)[i]; st[D.zU + i] = V(L->zU)[i];
        st[D.dx + i] = V(L->dx)[i]; st[D.dzL + i] = V(L->dzL)[i]; st[D.dzU + i] = V(L->dzU)[i];
        st[D.g + i] = V(L->g)[i];
    }
    for (int i = lane; i < pb->m; i += NT) {
        st[D.y + i] = VH(L->y)[i]; st[D.dy + i] = VH(L->dy)[i]; st[D.c + i] = VH(L->c)[i];
    }
    for (int i = lane; i < 2 * MAX_FILTER; i += NT) st[D.filt + i] = VH(L->filt)[i];
    for (int i = lane; i < pb->N * NX * NZ; i += NT) st[D.J + i] = VH(L->J)[(i / NZ) * C::LDJ + i % NZ];  // dense in the debug state
    for (int i = lane; i < pb->N * NZ * NZ + NX * NX; i += NT) st[D.W + i] = VH(L->W)[i];
    if (lane == 0) {
        st[D.sc + 0] = mu; st[D.sc + 1] = tau; st[D.sc + 2] = dw_last; st[D.sc + 3] = theta_min;
        st[D.sc + 4] = theta_max; st[D.sc + 5] = k; st[D.sc + 6] = status; st[D.sc + 7] = nfilt;
        st[D.rs + 0] = mode; st[D.rs + 1] = mu_reg; st[D.rs + 2] = tau_reg; st[D.rs + 3] = dw_last_reg;
        st[D.rs + 4] = theta_min_reg; st[D.rs + 5] = theta_max_reg; st[D.rs + 6] = nfilt_reg;
        st[D.rs + 7] = theta_entry; st[D.rs + 8] = zeta;
        st[D.ls + 0] = n_short; st[D.ls + 1] = wd_active; st[D.ls + 2] = wd_trials; st[D.ls + 3] = wd_theta;
        st[D.ls + 4] = wd_phi; st[D.ls + 5] = wd_gd; st[D.ls + 6] = wd_alpha; st[D.ls + 7] = soft;
        st[D.ls + 8] = soft_count; st[D.ls + 9] = tiny_last; st[D.ls + 10] = tiny_flag;
        st[D.ls + 11] = mu_free; st[D.ls + 12] = mu_max; st[D.ls + 13] = nhist;
        for (int q = 0; q < 4; ++q) st[D.ls + 14 + q] = hist[q];
        st[D.ls + 18] = acc_count;
    }
    if (wd_active) {
        const int nw = pb->n + 2 * pb->m;
        Vec w[6] = {VX(L->wx), VX(L->wzL), VX(L->wzU), VX(L->wdx), VX(L->wdzL), VX(L->wdzU)};
        for (int q = 0; q < 6; ++q)
            for (int i = lane; i < nX; i += NT) st[D.wd + q * nw + i] = w[q][i];
        for (int i = lane; i < pb->m; i += NT) { st[D.wd + 6 * nw + i] = V(L->wy)[i]; st[D.wd + 6 * nw + pb->m + i] = V(L->wdy)[i]; }
    }
    if (mode) {
        Vec xv = VX(L->x); Vec zLv = VX(L->zL);
        for (int j = lane; j < 2 * pb->m; j += NT) { st[D.pn + j] = xv[pb->n + j]; st[D.zpn + j] = zLv[pb->n + j]; }
        for (int i = lane; i < pb->n; i += NT) st[D.xR + i] = V(L->xR)[i];
        for (int i = lane; i < 2 * MAX_FILTER; i += NT) st[D.filtR + i] = V(L->filtR)[i];
    }
}

template <class C, int MINB>
__global__ void __launch_bounds__(C::NT, MINB) jipm_slot_kernel() {
    constexpr int NT = C::NT;
    const ArgsProxy A;
    const int lane = threadIdx.x;  // one team per CTA
    // claim one of this SM's workspaces (see Args::sm_mask)
    __shared__ int s_ws_id;
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    if (lane == 0) {
        int got = -1;
        while (got < 0) {
            for (int b = 0; b < A->teams_per_sm && got < 0; ++b) {
                const unsigned old = atomicOr(A->sm_mask + smid, 1u << b);
                if (!(old & (1u << b))) got = b;
            }
            if (got < 0) __nanosleep(500);
        }
        __threadfence();
        s_ws_id = (int)smid * A->teams_per_sm + got;
    }
    __syncthreads();
    const int ws_id = s_ws_id;
    double* ws = A->ws + (int64_t)ws_id * A->ws_stride;
    Ctx<C> ctx(ws, jipm_smem, lane);
    Solver<C> S(ctx);
    while (true) {
        int id = 0;
        if (lane == 0) id = atomicAdd(A->queue, 1);
        id = ctx.tm.bcast0(id);
        if (id >= A->P) break;
        if (A->dbg_mode == 2) {
            S.pid = id; S.nrec = 0;
            ctx.th = A->th + (int64_t)id * A->pb.nth;
            // targets and J zeroing as in init
            {
                const PbProxy pb;
                double* tgt = ctx.vh(A->L.tgt);
                for (int it = lane; it < (pb->N + 1) * C::NA; it += NT) {
                    const int kk = it / C::NA, a = it % C::NA;
                    if (pb->family == JIPM_FAM_QUAD_TRACK) {
                        const double rho = ctx.th[12], phase = ctx.th[13];
                        const double ang = phase + 1.5 * (kk * pb->dt) / rho;
                        tgt[it * C::PD + 0] = rho * cos(ang); tgt[it * C::PD + 1] = rho * sin(ang);
                        if (C::PD > 2) tgt[it * C::PD + 2] = 0.0;
                    } else {
                        for (int i = 0; i < C::PD; ++i) tgt[it * C::PD + i] = ctx.th[pb->th_goal + C::PD * a + i];
                    }
                }
                if (C::NA > 1)
                    for (int it = lane; it < pb->N * C::NX * C::LDJ; it += NT) ctx.vh(A->L.J)[it] = 0.0;
                ctx.tm.sync();
            }
            ctx.tm.sync();
            S.dbg_load(A->dbg_state + (int64_t)id * A->dbg_len);
            for (int s = 0; s < A->dbg_steps && S.status == JIPM_ST_NOT_RUN; ++s) S.iterate();
            S.dbg_store(A->dbg_state + (int64_t)id * A->dbg_len);
        } else {
            const long long t0i = clock64();
            S.init_problem(id);
            if (A->dbg_mode == 1) {
                S.dbg_store(A->dbg_state + (int64_t)id * A->dbg_len);
            } else {
                const long long t1 = clock64();
                ctx.tick(6, t1 - t0i);
                while (S.status == JIPM_ST_NOT_RUN) S.iterate();
                ctx.tick(5, clock64() - t1);
                S.write_outputs();
            }
        }
        ctx.tm.sync();
    }
    if (lane == 0) {
        atomicAdd(&A->stats[0], (unsigned long long)S.n_iter);
        atomicAdd(&A->stats[1], (unsigned long long)S.n_fact);
        atomicAdd(&A->stats[2], (unsigned long long)S.n_solve);
        atomicAdd(&A->stats[3], (unsigned long long)S.n_deriv);
        atomicAdd(&A->stats[4], (unsigned long long)S.n_fc);
        atomicAdd(&A->stats[7], (unsigned long long)S.n_resto);
        for (int i = 0; i < 16; ++i) atomicAdd(&A->stats[8 + i], ctx.counter(i));
    }
    // release the workspace: all global-scratch accesses of this CTA are done
    __syncthreads();
    if (lane == 0) {
        __threadfence();
        atomicAnd(A->sm_mask + smid, ~(1u << (ws_id - (int)smid * A->teams_per_sm)));
    }
}

}  // namespace jipm
