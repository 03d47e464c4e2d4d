// iter_impl.cuh -- Step I (initialise), Step A (one iteration) and the persistent slot kernel.
#pragma once
#include "iter.cuh"

namespace jipm {

// ---- Step I: slack init, interior push, z0 = 1, least-squares y0, mu0, filter bounds ------
template <class C>
__device__ void Solver<C>::init_problem(long long id) {
    pid = id;
    mode = 0; nX = pb->n;
    c.th = A->th + id * pb->nth;
    const double* th = c.th;
    const int N = pb->N;
    Vec x = VX(L->x); double* y = VH(L->y); Vec zL = VX(L->zL); Vec zU = VX(L->zU);
    const double* x0 = A->x0 + id * pb->n;
    for (int i = lane; i < pb->n; i += NT) x[i] = x0[i];
    // cost targets per knot / agent
    double* tgt = V(L->tgt);
    for (int it = lane; it < (N + 1) * NA; it += NT) {
        const int kk = it / NA, a = it % NA;
        if (pb->family == JIPM_FAM_QUAD_TRACK) {
            const double rho = th[12], phase = th[13];
            const double ang = phase + 1.5 * (kk * pb->dt) / rho;
            tgt[it * PD + 0] = rho * cos(ang); tgt[it * PD + 1] = rho * sin(ang);
            if (PD > 2) tgt[it * PD + 2] = 0.0;
        } else {
            const double* gl = th + pb->th_goal + PD * a;
#pragma unroll
            for (int i = 0; i < PD; ++i) tgt[it * PD + i] = gl[i];
        }
    }
    if (NA > 1) {
        for (int it = lane; it < N * NX * C::LDJ; it += NT) V(L->J)[it] = 0.0;
    }
    c.tm.sync();
    if (o->init_slacks) {  // I-2
        for (int it = lane; it < N * pb->ng; it += NT) {
            const int kk = it / pb->ng + 1, j = it % pb->ng;
            x[c.is(kk) + j] = c.ineq_val(x, kk, j);
        }
        c.tm.sync();
    }
    for (int i = lane; i < pb->n; i += NT) {  // I-3 push into the interior, I-4 z0
        const double l = pb->xL[i], u = pb->xU[i];
        const bool hl = l > -INFINITY, hu = u < INFINITY;
        double xi = x[i];
        if (hl && hu) {
            const double pl = fmin(o->kappa_1 * fmax(1.0, fabs(l)), o->kappa_2 * (u - l));
            const double pu = fmin(o->kappa_1 * fmax(1.0, fabs(u)), o->kappa_2 * (u - l));
            xi = fmin(fmax(xi, l + pl), u - pu);
        } else if (hl) xi = fmax(xi, l + o->kappa_1 * fmax(1.0, fabs(l)));
        else if (hu) xi = fmin(xi, u - o->kappa_1 * fmax(1.0, fabs(u)));
        x[i] = xi;
        zL[i] = hl ? o->bound_mult_init : 0.0;
        zU[i] = hu ? o->bound_mult_init : 0.0;
    }
    for (int i = lane; i < pb->m; i += NT) y[i] = 0.0;
    c.tm.sync();
    // I-5 least-squares multipliers: [[I, A^T],[A, 0]] [w; y] = -[grad f - zL + zU; 0]
    c.eval_derivs(x, y, 1.0);
    n_deriv++;
    {
        Vec Sig = VX(L->Sig); Vec Hd = VX(L->Hd); double* Dc = VH(L->Dc);
        Vec rr = VX(L->rr); double* b2 = VH(L->b2); Vec g = VX(L->g);
        for (int i = lane; i < pb->n; i += NT) { Sig[i] = 1.0; Hd[i] = 0.0; rr[i] = -(g[i] - zL[i] + zU[i]); }
        for (int i = lane; i < pb->m; i += NT) { Dc[i] = 0.0; b2[i] = 0.0; }
        c.tm.sync();
        int nz;
        const int bad = K::factor(c, nz, false, false);
        n_fact++;
        K::solve(c, rr, b2, VX(L->dx), VH(L->dy), false);
        n_solve++;
        const double* dy = VH(L->dy);
        double ym = 0.0, ys = 0.0;
        for (int i = lane; i < pb->m; i += NT) { ym = fmax(ym, fabs(dy[i])); ys += dy[i]; }
        ym = c.tm.max(ym); ys = c.tm.sum(ys);
        const bool okls = bad == 0 && isfinite(ys) && ym <= o->lam_init_max;
        for (int i = lane; i < pb->m; i += NT) y[i] = okls ? dy[i] : 0.0;
        c.tm.sync();
    }
    mu = o->mu_init;  // I-6
    tau = fmax(o->tau_min, 1.0 - mu);
    dw_last = 0.0;
    bool fin;
    f = c.eval_fc(x, VH(L->c), theta, cmax, fin);  // I-7
    n_fc++;
    theta_max = o->theta_max_fact * fmax(1.0, theta);
    theta_min = o->theta_min_fact * fmax(1.0, theta);
    nfilt = 0; k = 0; nrec = 0;
    status = fin ? JIPM_ST_NOT_RUN : JIPM_ST_NONFINITE;
}

// f, c (and theta, ||c||_inf) of the active problem at a trial point.  Regular mode: the NLP itself.  Restoration
// mode ([7] sec 3.3): X = [x; p; n], f_R = rho sum(p+n) + zeta/2 ||D_R (x - x_R)||^2, c_R = c(x) - p + n; the base
// problem's f, theta, ||c||_inf come back too (the exit test of Step R needs them).
template <class C>
__device__ double Solver<C>::eval_point(const Vec xt, double* ct, double& th_t, double& cm_t, double& fb,
                                        double& thb, double& cmb, double& fpn, double& fq) {
    bool fin;
    const long long t0 = clock64();
    fb = c.eval_fc(xt.a, ct, thb, cmb, fin);
    tph[4] += clock64() - t0;
    n_fc++;
    if (!mode) { th_t = thb; cm_t = cmb; fpn = 0.0; fq = 0.0; return fb; }
    const int n = pb->n, m = pb->m;
    const double* xR = V(L->xR); const double* DR2 = V(L->DR2);
    double spn = 0.0, sq = 0.0, th1 = 0.0, cm = 0.0;
    for (int j = lane; j < m; j += NT) {
        const double pj = xt[n + j], nj = xt[n + m + j];
        const double v = (ct[j] - pj) + nj;
        ct[j] = v; th1 += fabs(v); cm = fmax(cm, fabs(v));
        spn += pj + nj;
    }
    for (int i = lane; i < n; i += NT) { const double d = xt[i] - xR[i]; sq += DR2[i] * d * d; }
    c.tm.sync();
    fpn = c.tm.sum(spn); fq = c.tm.sum(sq); th_t = c.tm.sum(th1); cm_t = c.tm.max(cm);
    return o->rho_resto * fpn + 0.5 * zeta * fq;
}

// Speculative trial evaluation ("compute the branch-unique work for all, then select"): ONE WARP
// computes theta = ||c||_1 and phi_mu of the active problem (either mode) at x + alpha dx, nothing is stored and only
// warp shuffles synchronise, so the NT/32 warps of the team evaluate NT/32 backtracking candidates at once.
template <class C>
__device__ void Solver<C>::trial_warp(const Vec x, const Vec dx, double alpha, double& th_t, double& ph_t) const {
    const int wl = lane & 31;
    const int N = pb->N, n = pb->n, m = pb->m, ng = pb->ng;
    const double* xa = x.a; const double* da = dx.a;
    const double* xt_ = x.t; const double* dt_ = dx.t;
    const double* th = c.th;
    const double* tgt = c.vh(L->tgt);
    auto X = [&](int i) { return xa[i] + alpha * da[i]; };
    // restoration rows: c_R = (c - p) + n with p, n at the tail entries n + r, n + m + r
    auto ROW = [&](int r, double v) {
        if (mode) v = (v - (xt_[n + r] + alpha * dt_[n + r])) + (xt_[n + m + r] + alpha * dt_[n + m + r]);
        return fabs(v);
    };
    double f = 0.0, th1 = 0.0, bar = 0.0;
    int badpt = 0;
    if (!mode) {
        for (int it = wl; it < (N + 1) * NA; it += 32) {
            const int k = it / NA, a = it % NA, p0 = c.ix(k) + AX * a;
            double s = 0.0;
#pragma unroll
            for (int i = 0; i < PD; ++i) { const double d = X(p0 + i) - tgt[it * PD + i]; s += d * d; }
            f += s;
        }
        for (int it = wl; it < N * NU; it += 32) { const double u = X(c.iu(it / NU) + it % NU); f += pb->ru * (u * u); }
    } else {
        const double* xR = V(L->xR); const double* DR2 = V(L->DR2);
        double sq = 0.0, spn = 0.0;
        for (int i = wl; i < n; i += 32) { const double d = X(i) - xR[i]; sq += DR2[i] * d * d; }
        for (int r = wl; r < 2 * m; r += 32) spn += xt_[n + r] + alpha * dt_[n + r];
        f = o->rho_resto * spn + 0.5 * zeta * sq;
    }
    for (int i = wl; i < NX; i += 32) th1 += ROW(i, X(i) - th[i]);
    for (int it = wl; it < N * NA; it += 32) {
        const int k = it / NA, a = it % NA;
        double xs[AX], us[C::AU], Fv[AX];
#pragma unroll
        for (int i = 0; i < AX; ++i) xs[i] = X(c.ix(k) + AX * a + i);
#pragma unroll
        for (int i = 0; i < C::AU; ++i) us[i] = X(c.iu(k) + C::AU * a + i);
        C::Dyn::F(xs, us, pb->dt, Fv);
#pragma unroll
        for (int i = 0; i < AX; ++i) th1 += ROW(c.icd(k + 1) + AX * a + i, X(c.ix(k + 1) + AX * a + i) - Fv[i]);
    }
    for (int it = wl; it < N * ng; it += 32) {
        const int k = it / ng + 1, j = it % ng;
        double s = 0.0;
        if (pb->family == JIPM_FAM_MULTIQUAD) {
            int a, b; c.pair_ab(j, a, b);
#pragma unroll
            for (int i = 0; i < PD; ++i) { const double d = X(c.ix(k) + AX * a + i) - X(c.ix(k) + AX * b + i); s += d * d; }
            s -= 0.25;
        } else {
            const double* ob = th + pb->th_obs + (PD + 1) * j;
#pragma unroll
            for (int i = 0; i < PD; ++i) { const double d = X(c.ix(k) + i) - ob[i]; s += d * d; }
            s -= ob[PD] * ob[PD];
        }
        th1 += ROW(c.icg(k) + j, s - X(c.is(k) + j));
    }
    // barrier terms of (3) with the one-sided damping, as in phi()
    // sum of log(slack) as ONE log per lane: slack = mant * 2^ex with mant in [1, 2); the mantissas are multiplied (a
    // lane sees nX / 32 + 1 < 1000 of them, far from overflow) and the exponents added as integers.  A slack that is
    // not a positive normal number marks the point as bad (phi_mu = inf), as log would.
    double mprod = 1.0;
    int esum = 0;
    auto LOGACC = [&](double sl) {
        if (!(sl >= 2.2250738585072014e-308) || !(sl < INFINITY)) { badpt = 1; return; }
        const int hi32 = __double2hiint(sl);
        esum += (hi32 >> 20) - 1023;
        mprod *= __hiloint2double((hi32 & 0x000fffff) | 0x3ff00000, __double2loint(sl));
    };
    for (int i = wl; i < nX; i += 32) {
        const double l = lo(i), u = hi(i);
        const bool hl = l > -INFINITY, hu = u < INFINITY;
        if (!hl && !hu) continue;
        const double xi = (i < n) ? X(i) : xt_[i] + alpha * dt_[i];
        if (hl) {
            const double sl = xi - l;
            LOGACC(sl);
            if (!hu) bar += o->kappa_d * mu * sl;
        }
        if (hu) {
            const double su = u - xi;
            LOGACC(su);
            if (!hl) bar += o->kappa_d * mu * su;
        }
    }
    bar -= mu * (log(mprod) + 0.6931471805599453 * (double)esum);
#pragma unroll
    for (int s = 16; s; s >>= 1) {
        f += __shfl_xor_sync(FULL, f, s);
        th1 += __shfl_xor_sync(FULL, th1, s);
        bar += __shfl_xor_sync(FULL, bar, s);
        badpt |= __shfl_xor_sync(FULL, badpt, s);
    }
    th_t = th1;
    ph_t = badpt ? NAN : f + bar;
}

// Restoration entry (Table I row 6; Step R of SURVEY.md 8(c), [7] sec 3.3).  The restoration
// problem  min rho e^T(p+n) + zeta/2 ||D_R(x-x_R)||^2  s.t. c(x) - p + n = 0, p, n >= 0, x_L <= x <= x_U  is iterated
// by the SAME iterate() with mode = 1 (same KKT sparsity after eliminating p, n: that is what lets it fuse).
template <class C>
__device__ void Solver<C>::enter_restoration(double* rec, int kind) {
    rec[5] = kind;
    if (!o->enable_restoration || mode == 1) { status = JIPM_ST_RESTORATION_FAILED; return; }  // no nesting (A20)
    if (theta < o->tol) { status = JIPM_ST_RESTO_AT_FEASIBLE_POINT; return; }
    const int n = pb->n, m = pb->m;
    Vec x = VX(L->x); double* y = VH(L->y); Vec zL = VX(L->zL); Vec zU = VX(L->zU); double* cv = VH(L->c);
    const double theta_k = theta;
    const double phi_k = phi(x, f, mu, n);
    filter_add((1.0 - o->gamma_theta) * theta_k, phi_k - o->gamma_phi * theta_k);
    const double mu_bar = fmax(mu, cmax);
    mu_reg = mu; tau_reg = tau; dw_last_reg = dw_last; theta_min_reg = theta_min; theta_max_reg = theta_max;
    nfilt_reg = nfilt;
    f_base = f; theta_base = theta_k; cmax_base = cmax;
    const double rho = o->rho_resto;
    double* xR = V(L->xR); double* DR2 = V(L->DR2);
    for (int i = lane; i < n; i += NT) {
        const double xi = x[i];
        xR[i] = xi;
        const double dr = fmin(1.0, 1.0 / fmax(fabs(xi), 1e-300));
        DR2[i] = dr * dr;
        zL[i] = hasL(i) ? fmin(rho, zL[i]) : 0.0;
        zU[i] = hasU(i) ? fmin(rho, zU[i]) : 0.0;
    }
    double th1 = 0.0, cm = 0.0, spn = 0.0;
    for (int j = lane; j < m; j += NT) {
        // closed-form minimiser of the restoration barrier function in (p, n) at fixed x ([7] eqs 32-33)
        const double cj = cv[j];
        const double t = (mu_bar - rho * cj) / (2.0 * rho);
        const double nn = t + sqrt(t * t + mu_bar * cj / (2.0 * rho));
        const double pp = cj + nn;
        x[n + j] = pp; x[n + m + j] = nn;
        zL[n + j] = mu_bar / pp; zL[n + m + j] = mu_bar / nn;
        zU[n + j] = 0.0; zU[n + m + j] = 0.0;
        y[j] = 0.0;
        const double v = (cj - pp) + nn;
        cv[j] = v; th1 += fabs(v); cm = fmax(cm, fabs(v));
        spn += pp + nn;
    }
    c.tm.sync();
    theta = c.tm.sum(th1); cmax = c.tm.max(cm); f_pn = c.tm.sum(spn); f_q = 0.0;
    mode = 1; nX = n + 2 * m;
    mu = mu_bar; tau = fmax(o->tau_min, 1.0 - mu_bar); dw_last = 0.0; nfilt = 0;
    zeta = sqrt(mu_bar);
    f = rho * f_pn + 0.5 * zeta * f_q;
    theta_max = o->theta_max_fact * fmax(1.0, theta);
    theta_min = o->theta_min_fact * fmax(1.0, theta);
    theta_entry = theta_k;
    k += 1;  // the failed regular iteration counts (reading S-19)
}

// Exit test after an accepted restoration step: theta(x) <= kappa_resto theta(x_R) and (theta, phi_mu) not in the
// REGULAR filter -> back to regular mode with y = 0 and the restoration z (reading S-15).
template <class C>
__device__ void Solver<C>::try_exit_restoration() {
    const int n = pb->n;
    Vec x = VX(L->x); double* y = VH(L->y); Vec zL = VX(L->zL); Vec zU = VX(L->zU);
    const double phi_b = phi(x, f_base, mu_reg, n);
    if (!isfinite(phi_b) || !(theta_base <= o->kappa_resto * theta_entry)) return;
    if (in_filter_of(V(L->filt), nfilt_reg, theta_max_reg, theta_base, phi_b)) return;
    double zm = 0.0;
    for (int i = lane; i < n; i += NT) zm = fmax(zm, fmax(zL[i], zU[i]));
    zm = c.tm.max(zm);
    if (zm > o->z_reset_threshold)
        for (int i = lane; i < n; i += NT) { zL[i] = hasL(i) ? 1.0 : 0.0; zU[i] = hasU(i) ? 1.0 : 0.0; }
    for (int j = lane; j < pb->m; j += NT) y[j] = 0.0;
    c.tm.sync();
    mode = 0; nX = n;
    mu = mu_reg; tau = tau_reg; dw_last = dw_last_reg; theta_min = theta_min_reg; theta_max = theta_max_reg;
    nfilt = nfilt_reg;
    bool fin;
    f = c.eval_fc(x, VH(L->c), theta, cmax, fin);  // base c back into the c vector (same point: same values)
    n_fc++;
}

// ---- Step A: one iteration (either mode) ---------------------------------------------------------------------
template <class C>
__device__ void Solver<C>::iterate() {
    Vec x = VX(L->x); double* y = VH(L->y); Vec zL = VX(L->zL); Vec zU = VX(L->zU);
    double* cv = VH(L->c); Vec g = VX(L->g);
    Vec b1 = VX(L->b1); double* b2 = VH(L->b2); Vec b3 = VX(L->b3); Vec b4 = VX(L->b4);
    Vec dx = VX(L->dx); double* dy = VH(L->dy); Vec dzL = VX(L->dzL); Vec dzU = VX(L->dzU);
    const int n = pb->n, m = pb->m;
    double rec[JIPM_TRACE_W];
#pragma unroll
    for (int i = 0; i < JIPM_TRACE_W; ++i) rec[i] = 0.0;
    rec[0] = mode;
    n_iter++;
    if (mode) n_resto++;
    // A-1 derivatives at (x, y): sigma_f = 0 in restoration mode (its objective is rho e^T(p+n) + zeta/2 ||D_R(x-x_R)||^2)
    const long long t_it = clock64();
    c.eval_derivs(x, y, mode ? 0.0 : 1.0);
    const long long t_hd = clock64();
    tph[0] += t_hd - t_it;
    n_deriv++;
    if (mode) {
        const double* xR = V(L->xR); const double* DR2 = V(L->DR2);
        for (int i = lane; i < n; i += NT) g[i] = zeta * DR2[i] * (x[i] - xR[i]);
        for (int i = n + lane; i < nX; i += NT) g[i] = o->rho_resto;
        c.tm.sync();
    }
    // dual residual base rdb = grad f + A^T y - zL + zU  (into b1), multiplier sums for the scaling s_d, s_c
    double ysum = 0.0, zsum = 0.0, chk = 0.0;
    for (int i = lane; i < nX; i += NT) {
        const double v = g[i] + ATx(y, i) - zL[i] + zU[i];
        b1[i] = v; chk += v;
        zsum += fabs(zL[i]) + fabs(zU[i]);
    }
    for (int i = lane; i < m; i += NT) ysum += fabs(y[i]);
    ysum = c.tm.sum(ysum); zsum = c.tm.sum(zsum); chk = c.tm.sum(chk);
    c.tm.sync();
    if (!isfinite(chk) || !isfinite(f) || !isfinite(theta)) {
        status = JIPM_ST_NONFINITE; rec[5] = KIND_TERMINAL; trace_put(rec); return;
    }
    const int nz = pb->nL + pb->nU + (mode ? 2 * m : 0);
    const double sd = (m + nz > 0) ? fmax(o->s_max, (ysum + zsum) / (m + nz)) / o->s_max : 1.0;
    const double sc = (nz > 0) ? fmax(o->s_max, zsum / nz) / o->s_max : 1.0;
    // A-2 termination
    const double e0 = opt_error(0.0, sd, sc);
    rec[12] = e0;
    if (e0 <= o->tol) {
        // restoration problem converged without an acceptable point: local minimiser of the violation
        if (mode) status = (theta_base > o->tol) ? JIPM_ST_LOCALLY_INFEASIBLE : JIPM_ST_RESTO_AT_FEASIBLE_POINT;
        else status = JIPM_ST_SOLVED;
        rec[5] = KIND_TERMINAL; trace_put(rec); return;
    }
    if (k >= o->max_iter) { status = JIPM_ST_MAXITER; rec[5] = KIND_TERMINAL; trace_put(rec); return; }
    // A-3 monotone barrier update (Table I row 7)
    int nmu = 0;
    const double mu_min = o->tol / 10.0;
    while (nmu < o->max_mu_updates && mu > mu_min && opt_error(mu, sd, sc) <= o->kappa_eps * mu) {
        mu = fmax(mu_min, fmin(o->kappa_mu * mu, pow(mu, o->theta_mu)));
        tau = fmax(o->tau_min, 1.0 - mu);
        nfilt = 0;
        nmu++;
        if (mode) {  // zeta = sqrt(mu) follows the restoration barrier parameter: objective, gradient, residual move
            const double zn = sqrt(mu);
            const double* xR = V(L->xR); const double* DR2 = V(L->DR2);
            for (int i = lane; i < n; i += NT) {
                const double gi = zn * DR2[i] * (x[i] - xR[i]);
                b1[i] += gi - g[i]; g[i] = gi;
            }
            c.tm.sync();
            zeta = zn;
            f = o->rho_resto * f_pn + 0.5 * zeta * f_q;
        }
    }
    rec[11] = nmu; rec[13] = mu;
    // A-4 search direction with inertia correction (Algorithm IC)
    int nfact = 0, nzero = 0;
    double dw = 0.0, dc = 0.0;
    bool ic_ok;
    set_sigma(0.0, 0.0);
    long long t_f = clock64();
    c.pc[7] += t_f - t_hd;
    int bad = K::factor(c, nzero, mode != 0, true); nfact++;  // IC-1
    ic_ok = (bad == 0);
    if (!ic_ok) {
        dc = (nzero > 0) ? o->delta_c_bar * pow(mu, o->kappa_c) : 0.0;                               // IC-2
        dw = (dw_last == 0.0) ? o->delta_w_0 : fmax(o->delta_w_min, o->kappa_w_minus * dw_last);      // IC-3
        while (true) {
            set_sigma(dw, dc);
            bad = K::factor(c, nzero, mode != 0 || dc != 0.0, true); nfact++;                       // IC-4
            if (bad == 0) { ic_ok = true; break; }
            dw *= (dw_last == 0.0) ? o->kappa_w_plus_first : o->kappa_w_plus;                         // IC-5
            if (dw > o->delta_w_max) break;                                                          // IC-6
        }
    }
    n_fact += nfact;
    tph[1] += clock64() - t_f;
    rec[1] = nfact; rec[2] = dw; rec[3] = dc; rec[14] = theta;
    if (!ic_ok) { rec[1] = 0; rec[2] = 0; rec[3] = 0; enter_restoration(rec, KIND_IC_FAIL); trace_put(rec); return; }
    if (dw > 0.0) dw_last = dw;
    // right-hand side of (6)
    for (int i = lane; i < nX; i += NT) {
        const double l = lo(i), u = hi(i);
        const bool hl = l > -INFINITY, hu = u < INFINITY;
        double dmp = 0.0;
        if (hl && !hu) dmp = o->kappa_d * mu;
        if (hu && !hl) dmp = -o->kappa_d * mu;
        b1[i] = -(b1[i] + dmp);
        b3[i] = hl ? mu - (x[i] - l) * zL[i] : 0.0;
        b4[i] = hu ? mu - (u - x[i]) * zU[i] : 0.0;
    }
    for (int i = lane; i < m; i += NT) b2[i] = -cv[i];
    c.tm.sync();
    const long long t_sf = clock64();
    const int nref = solve_full(b1, b2, b3, b4, dx, dy, dzL, dzU);
    c.pc[5] += clock64() - t_sf;
    rec[4] = nref;
    // A-5 filter line search
    double gd_part = 0.0;
    for (int i = lane; i < nX; i += NT) {
        const double l = lo(i), u = hi(i);
        const bool hl = l > -INFINITY, hu = u < INFINITY;
        double gp = g[i];
        if (hl) gp -= mu / (x[i] - l);
        if (hu) gp += mu / (u - x[i]);
        if (hl && !hu) gp += o->kappa_d * mu;
        if (hu && !hl) gp -= o->kappa_d * mu;
        gd_part += gp * dx[i];
    }
    const double gd = c.tm.sum(gd_part);
    const double theta_k = theta;
    const double phi_k = phi(x, f, mu, nX);
    rec[15] = phi_k;
    const double a_max = ftb_primal(x, dx, tau);
    double a_min;
    if (gd < 0.0 && theta_k <= theta_min)
        a_min = o->gamma_alpha * fmin(fmin(o->gamma_theta, o->gamma_phi * theta_k / (-gd)),
                                     o->delta * pow(theta_k, o->s_theta) / pow(-gd, o->s_phi));
    else if (gd < 0.0) a_min = o->gamma_alpha * fmin(o->gamma_theta, o->gamma_phi * theta_k / (-gd));
    else a_min = o->gamma_alpha * o->gamma_theta;
    const long long t_ls = clock64();
    Vec xt = VX(L->xt); double* ct = VH(L->ct);
    double alpha = a_max, alpha_acc = 0.0, phi_acc = 0.0, f_acc = 0.0, th_acc = 0.0, cm_acc = 0.0;
    double fb_acc = 0.0, thb_acc = 0.0, cmb_acc = 0.0, fpn_acc = 0.0, fq_acc = 0.0;
    int ntrial = 0, nsoc = 0, acc = -1;  // acc: 0 newton, 1 soc
    while (true) {
        for (int i = lane; i < nX; i += NT) xt[i] = x[i] + alpha * dx[i];
        c.tm.sync();
        double th_t, cm_t, fb, thb, cmb, fpn, fq;
        const double f_t = eval_point(xt, ct, th_t, cm_t, fb, thb, cmb, fpn, fq);
        const double ph_t = phi(xt, f_t, mu, nX);
        if (acceptable(th_t, ph_t, theta_k, phi_k, alpha, gd)) {
            acc = 0; alpha_acc = alpha; phi_acc = ph_t; f_acc = f_t; th_acc = th_t; cm_acc = cm_t;
            fb_acc = fb; thb_acc = thb; cmb_acc = cmb; fpn_acc = fpn; fq_acc = fq;
            break;
        }
        if (ntrial == 0 && isfinite(th_t) && th_t >= theta_k && o->max_soc > 0) {
            // second-order correction (Table I row 2)
            double* csoc = V(L->csoc); double* bs2 = V(L->bs2);
            Vec sx = VX(L->sx); double* sy = V(L->sy); Vec szL = VX(L->szL); Vec szU = VX(L->szU);
            for (int i = lane; i < m; i += NT) csoc[i] = alpha * cv[i] + ct[i];
            c.tm.sync();
            double theta_old = theta_k;
            for (int ps = 1; ps <= o->max_soc; ++ps) {
                for (int i = lane; i < m; i += NT) bs2[i] = -csoc[i];
                c.tm.sync();
                solve_full(b1, bs2, b3, b4, sx, sy, szL, szU);
                const double a_soc = ftb_primal(x, sx, tau);
                for (int i = lane; i < nX; i += NT) xt[i] = x[i] + a_soc * sx[i];
                c.tm.sync();
                double th_s, cm_s;
                const double f_s = eval_point(xt, ct, th_s, cm_s, fb, thb, cmb, fpn, fq);
                const double ph_s = phi(xt, f_s, mu, nX);
                nsoc = ps;
                if (acceptable(th_s, ph_s, theta_k, phi_k, alpha, gd)) {
                    acc = 1; alpha_acc = a_soc; phi_acc = ph_s; f_acc = f_s; th_acc = th_s; cm_acc = cm_s;
                    fb_acc = fb; thb_acc = thb; cmb_acc = cmb; fpn_acc = fpn; fq_acc = fq;
                    break;
                }
                if (!isfinite(th_s) || th_s > o->kappa_soc * theta_old) break;
                theta_old = th_s;
                for (int i = lane; i < m; i += NT) csoc[i] = a_soc * csoc[i] + ct[i];
                c.tm.sync();
            }
            if (acc >= 0) break;
        }
        alpha *= o->alpha_red;
        ntrial++;
        if (alpha < a_min || ntrial > o->max_backtrack) break;
        if constexpr (NT >= 64) {
            // Speculative backtracking: warp w evaluates the candidate alpha * alpha_red^w; the candidates
            // are then scanned in the sequential order with the sequential termination rule, so the decision is the one
            // of Step A-5.  The first acceptable candidate is re-evaluated by the regular path at the top of the loop
            // (it fills c, f and confirms the test); rejected ones only advance alpha and the trial counter.
            constexpr int NWP = NT / 32;
            double* spec = c.smt(C::SM_SPEC);
            bool exhausted = false, found = false;
            const long long t_sp = clock64();
            while (!found && !exhausted) {
                double aw = alpha;
                for (int w = 0; w < (lane >> 5); ++w) aw *= o->alpha_red;
                double th_w, ph_w;
                trial_warp(x, dx, aw, th_w, ph_w);
                const bool ok_w = acceptable_warp(th_w, ph_w, theta_k, phi_k, aw, gd);
                if ((lane & 31) == 0) spec[lane >> 5] = ok_w ? 1.0 : 0.0;
                c.tm.sync();
                for (int w = 0; w < NWP; ++w) {
                    if (spec[w] != 0.0) { found = true; break; }
                    n_fc++;
                    alpha *= o->alpha_red;
                    ntrial++;
                    if (alpha < a_min || ntrial > o->max_backtrack) { exhausted = true; break; }
                }
                c.tm.sync();
            }
            tph[7] += clock64() - t_sp;
            if (exhausted) break;
        }
    }
    rec[6] = ntrial; rec[7] = nsoc;
    c.pc[6] += clock64() - t_ls;
    if (acc < 0) { enter_restoration(rec, KIND_LS_FAIL); trace_put(rec); return; }
    // A-6 accept, A-7 filter augmentation
    const Vec ax = (acc == 1) ? VX(L->sx) : dx;
    const double* ay = (acc == 1) ? V(L->sy) : dy;
    const Vec azL = (acc == 1) ? VX(L->szL) : dzL;
    const Vec azU = (acc == 1) ? VX(L->szU) : dzU;
    (void)ax;
    const double a_z = ftb_dual(zL, zU, azL, azU, tau);
    const bool ftype = switching(alpha, gd, theta_k) && armijo(phi_acc, phi_k, alpha, gd);
    if (!ftype) filter_add((1.0 - o->gamma_theta) * theta_k, phi_k - o->gamma_phi * theta_k);
    const double ks = o->kappa_sigma;
    for (int i = lane; i < nX; i += NT) {
        const double l = lo(i), u = hi(i);
        const double xn = xt[i];
        x[i] = xn;
        double zl = 0.0, zu = 0.0;
        if (l > -INFINITY) {
            const double sl = xn - l;
            zl = fmax(fmin(zL[i] + a_z * azL[i], ks * mu / sl), mu / (ks * sl));
        }
        if (u < INFINITY) {
            const double su = u - xn;
            zu = fmax(fmin(zU[i] + a_z * azU[i], ks * mu / su), mu / (ks * su));
        }
        zL[i] = zl; zU[i] = zu;
    }
    for (int i = lane; i < m; i += NT) { y[i] += alpha_acc * ay[i]; cv[i] = ct[i]; }
    c.tm.sync();
    f = f_acc; theta = th_acc; cmax = cm_acc;
    f_base = fb_acc; theta_base = thb_acc; cmax_base = cmb_acc; f_pn = fpn_acc; f_q = fq_acc;
    k += 1;  // A-8
    rec[5] = (acc == 1) ? KIND_SOC : KIND_NEWTON;
    rec[8] = alpha_acc; rec[9] = a_z; rec[10] = ftype ? 1.0 : 0.0;
    trace_put(rec);
    if (mode) try_exit_restoration();
}

template <class C>
__device__ void Solver<C>::write_outputs() {
    Vec x = VX(L->x); const double* y = VH(L->y); Vec zL = VX(L->zL); Vec zU = VX(L->zU);
    if (A->x_out) for (int i = lane; i < pb->n; i += NT) A->x_out[pid * pb->n + i] = x[i];
    if (A->lam_out) for (int i = lane; i < pb->m; i += NT) A->lam_out[pid * pb->m + i] = y[i];
    if (A->zL_out) for (int i = lane; i < pb->n; i += NT) A->zL_out[pid * pb->n + i] = zL[i];
    if (A->zU_out) for (int i = lane; i < pb->n; i += NT) A->zU_out[pid * pb->n + i] = zU[i];
    if (lane == 0) {
        if (A->status_out) A->status_out[pid] = status;
        if (A->iters_out) A->iters_out[pid] = k;
    }
}

}  // namespace jipm
