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
    reset_ls_memory();
    reset_mu_memory();
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
    c.tick(4, clock64() - t0);
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
    reset_ls_memory();  // neither problem's line-search memory survives a change of mode
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
    reset_ls_memory();
    mu = mu_reg; tau = tau_reg; dw_last = dw_last_reg; theta_min = theta_min_reg; theta_max = theta_max_reg;
    nfilt = nfilt_reg;
    bool fin;
    f = c.eval_fc(x, VH(L->c), theta, cmax, fin);  // base c back into the c vector (same point: same values)
    n_fc++;
}

// ---- Algorithm IC (A-4) ---------------------------------------------------------------
// Factorises with (dw, dc) until the pivot signs give the inertia (n, m, 0).  resume: the factorisation at the
// incoming (dw, dc) had the right inertia but the solve with it failed the refinement test ("pretend singular",
// reading S-7): delta_c takes its IC-2 value, delta_w moves to the next rung (IC-3 from 0, else IC-5) and the loop
// IC-4..IC-6 continues.  Returns false when delta_w exceeds delta_w_max (IC-6).
template <class C>
__device__ bool Solver<C>::ic_loop(bool resume, double& dw, double& dc, int& nfact) {
    const long long t_f = clock64();
    const double grow = (dw_last == 0.0) ? o->kappa_w_plus_first : o->kappa_w_plus;
    const double first = (dw_last == 0.0) ? o->delta_w_0 : fmax(o->delta_w_min, o->kappa_w_minus * dw_last);  // IC-3
    int nzero = 0, nf = 0;
    bool ok = false, give_up = false;
    if (!resume) {
        set_sigma(0.0, 0.0);
        const int bad = K::factor(c, nzero, mode != 0, true); nf++;                       // IC-1
        if (bad == 0) { dw = 0.0; dc = 0.0; ok = true; }
        else {
            dc = (nzero > 0) ? o->delta_c_bar * pow(mu, o->kappa_c) : 0.0;                // IC-2
            dw = first;
        }
    } else {
        dc = o->delta_c_bar * pow(mu, o->kappa_c);
        if (dw == 0.0) dw = first;
        else { dw *= grow; if (dw > o->delta_w_max) give_up = true; }
    }
    while (!ok && !give_up) {
        set_sigma(dw, dc);
        const int bad = K::factor(c, nzero, mode != 0 || dc != 0.0, true); nf++;          // IC-4
        if (bad == 0) { ok = true; break; }
        dw *= grow;                                                                       // IC-5
        if (dw > o->delta_w_max) give_up = true;                                          // IC-6
    }
    nfact += nf; n_fact += nf;
    c.tick(1, clock64() - t_f);
    return ok;
}

// f, c, theta, phi_mu of the active problem at x + alpha d (into xt, ct)
template <class C>
__device__ void Solver<C>::trial(const Vec dxv, double alpha, Trial& t) {
    Vec x = VX(L->x); Vec xt = VX(L->xt); double* ct = VH(L->ct);
    for (int i = lane; i < nX; i += NT) xt[i] = x[i] + alpha * dxv[i];
    c.tm.sync();
    t.f = eval_point(xt, ct, t.th, t.cm, t.fb, t.thb, t.cmb, t.fpn, t.fq);
    t.ph = phi(xt, t.f, mu, nX);
}

// Backtracking line search with the second-order correction (Table I rows 1-2; A-5) along dxv from
// the current iterate.  acc: 0 = Newton step, 1 = corrected step (in sx, sy, szL, szU); alpha = the step length the
// acceptance test used, alpha_acc = the length of the accepted step; ta = the accepted trial.  rec[6], rec[7] get the
// numbers of backtracks and corrections.  Returns false when alpha falls below alpha_min.
template <class C>
__device__ bool Solver<C>::backtrack(const Vec dxv, double theta_k, double phi_k, double gd, double a_max,
                                     bool skip_first, bool allow_soc, double* rec, int& acc, double& alpha,
                                     double& alpha_acc, Trial& ta) {
    Vec x = VX(L->x); double* cv = VH(L->c);
    Vec b1 = VX(L->b1); Vec b3 = VX(L->b3); Vec b4 = VX(L->b4);
    const int m = pb->m;
    double a_min;
    if (gd < 0.0 && theta_k <= theta_min)
        a_min = o->gamma_alpha * fmin(fmin(o->gamma_theta, o->gamma_phi * theta_k / (-gd)),
                                     o->delta * pow(theta_k, o->s_theta) / pow(-gd, o->s_phi));
    else if (gd < 0.0) a_min = o->gamma_alpha * fmin(o->gamma_theta, o->gamma_phi * theta_k / (-gd));
    else a_min = o->gamma_alpha * o->gamma_theta;
    double* ct = VH(L->ct); Vec xt = VX(L->xt);
    alpha = a_max; alpha_acc = 0.0;
    int ntrial = 0, nsoc = 0;
    acc = -1;
    bool live = true;
    if (skip_first) {  // the full step was tried (and rejected) before: start one halving down, no correction
        alpha *= o->alpha_red;
        ntrial = 1;
        if (alpha < a_min) live = false;
    }
    while (live) {
        Trial t;
        trial(dxv, alpha, t);
        if (acceptable(t.th, t.ph, theta_k, phi_k, alpha, gd)) { acc = 0; alpha_acc = alpha; ta = t; break; }
        if (ntrial == 0 && allow_soc && isfinite(t.th) && t.th >= theta_k && o->max_soc > 0) {
            // second-order correction (Table I row 2)
            double* csoc = V(L->csoc); double* bs2 = V(L->bs2);
            Vec sx = VX(L->sx); double* sy = V(L->sy); Vec szL = VX(L->szL); Vec szU = VX(L->szU);
            for (int i = lane; i < m; i += NT) csoc[i] = alpha * cv[i] + ct[i];
            c.tm.sync();
            double theta_old = theta_k;
            for (int ps = 1; ps <= o->max_soc; ++ps) {
                for (int i = lane; i < m; i += NT) bs2[i] = -csoc[i];
                c.tm.sync();
                bool failed;
                solve_full(b1, bs2, b3, b4, sx, sy, szL, szU, failed);
                const double a_soc = ftb_primal(x, sx, tau);
                Trial ts;
                trial(sx, a_soc, ts);
                nsoc = ps;
                if (acceptable(ts.th, ts.ph, theta_k, phi_k, alpha, gd)) { acc = 1; alpha_acc = a_soc; ta = ts; break; }
                if (!isfinite(ts.th) || ts.th > o->kappa_soc * theta_old) break;
                theta_old = ts.th;
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
                trial_warp(x, dxv, aw, th_w, ph_w);
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
            c.tick(7, clock64() - t_sp);
            if (exhausted) break;
        }
    }
    rec[6] = ntrial; rec[7] = nsoc;
    (void)xt;
    return acc >= 0;
}

// A-6 / A-8: move to the accepted trial point (in xt, its c in ct), step the multipliers, safeguard z, count.
template <class C>
__device__ void Solver<C>::accept_step(int, const Vec, const double* ay, const Vec azL, const Vec azU, double,
                                       double alpha_y, double a_z, const Trial& t) {
    Vec x = VX(L->x); double* y = VH(L->y); Vec zL = VX(L->zL); Vec zU = VX(L->zU);
    Vec xt = VX(L->xt); double* ct = VH(L->ct); double* cv = VH(L->c);
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
    for (int i = lane; i < pb->m; i += NT) { y[i] += alpha_y * ay[i]; cv[i] = ct[i]; }
    c.tm.sync();
    f = t.f; theta = t.th; cmax = t.cm;
    f_base = t.fb; theta_base = t.thb; cmax_base = t.cmb; f_pn = t.fpn; f_q = t.fq;
    k += 1;  // A-8
}

// One step of the soft restoration phase (Table I row 5; reading SR): the same step length for
// primal and dual variables; accepted if the original criterion holds (the phase ends) or if the error of the
// primal-dual system (5a-d), measured as the sum of the 1-norms of its blocks divided by their lengths, drops by the
// factor soft_resto_factor.  Returns false when the step is refused (the caller starts the hard restoration).
template <class C>
__device__ bool Solver<C>::soft_step(double* rec, double theta_k, double phi_k, double gd) {
    Vec x = VX(L->x); double* y = VH(L->y); Vec zL = VX(L->zL); Vec zU = VX(L->zU);
    Vec b1 = VX(L->b1); Vec b3 = VX(L->b3); Vec b4 = VX(L->b4);
    Vec dx = VX(L->dx); double* dy = VH(L->dy); Vec dzL = VX(L->dzL); Vec dzU = VX(L->dzU);
    Vec xt = VX(L->xt); Vec g = VX(L->g);
    const int n = pb->n, m = pb->m;
    const double a_p = ftb_primal(x, dx, tau);
    const double a_d = ftb_dual(zL, zU, dzL, dzU, tau);
    const double alpha = fmin(a_p, a_d);
    // current error: -b1 is the dual residual (damping included), -b3 / -b4 the complementarity residuals
    double s1 = 0.0, s3 = 0.0;
    for (int i = lane; i < nX; i += NT) { s1 += fabs(b1[i]); s3 += fabs(b3[i]) + fabs(b4[i]); }
    s1 = c.tm.sum(s1); s3 = c.tm.sum(s3);
    const int ncomp = pb->nL + pb->nU + (mode ? 2 * m : 0);
    const double e_k = s1 / nX + (m > 0 ? theta_k / m : 0.0) + (ncomp > 0 ? s3 / ncomp : 0.0);
    Trial t;
    trial(dx, alpha, t);
    bool ok = isfinite(t.th) && isfinite(t.ph);
    const bool orig = ok && acceptable(t.th, t.ph, theta_k, phi_k, 0.0, gd);
    if (ok && !orig) {
        double* yt = V(L->sy);
        for (int i = lane; i < m; i += NT) yt[i] = y[i] + alpha * dy[i];
        c.tm.sync();
        c.eval_derivs(xt, yt, mode ? 0.0 : 1.0);  // J and grad f at the trial point (the next iteration re-evaluates)
        n_deriv++;
        const double* xR = V(L->xR); const double* DR2 = V(L->DR2);
        double t1 = 0.0, t3 = 0.0;
        for (int i = lane; i < nX; i += NT) {
            const double l = lo(i), u = hi(i);
            const bool hl = l > -INFINITY, hu = u < INFINITY;
            const double zl = hl ? zL[i] + alpha * dzL[i] : 0.0, zu = hu ? zU[i] + alpha * dzU[i] : 0.0;
            double gi;
            if (mode) gi = (i < n) ? zeta * DR2[i] * (xt[i] - xR[i]) : o->rho_resto;
            else gi = g[i];
            double v = gi + ATx(yt, i) - zl + zu;
            if (hl && !hu) v += o->kappa_d * mu;
            if (hu && !hl) v -= o->kappa_d * mu;
            t1 += fabs(v);
            if (hl) t3 += fabs((xt[i] - l) * zl - mu);
            if (hu) t3 += fabs((u - xt[i]) * zu - mu);
        }
        t1 = c.tm.sum(t1); t3 = c.tm.sum(t3);
        const double e_t = t1 / nX + (m > 0 ? t.th / m : 0.0) + (ncomp > 0 ? t3 / ncomp : 0.0);
        ok = isfinite(e_t) && e_t <= o->soft_resto_factor * e_k;
    }
    if (!ok) return false;
    rec[17] = orig ? 2.0 : 1.0;
    if (orig) { soft = 0; soft_count = 0; }
    n_short = 0;
    accept_step(0, dx, dy, dzL, dzU, alpha, alpha, alpha, t);
    rec[5] = KIND_SOFT; rec[8] = alpha; rec[9] = alpha; rec[10] = 1.0;
    return true;
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
    c.tick(0, t_hd - t_it);
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
    if (o->acceptable_iter > 0 && mode == 0) {   // acceptable-level termination (reading AT): regular problem only
        double ed, es;
        error_parts(ed, es);
        const bool okacc = e0 <= o->acceptable_tol && ed <= o->acceptable_dual_inf_tol &&
                           cmax <= o->acceptable_constr_viol_tol && es <= o->acceptable_compl_inf_tol;
        acc_count = okacc ? acc_count + 1 : 0;
        if (acc_count >= o->acceptable_iter) { status = JIPM_ST_ACCEPTABLE; rec[5] = KIND_TERMINAL; trace_put(rec); return; }
    }
    if (k >= o->max_iter) { status = JIPM_ST_MAXITER; rec[5] = KIND_TERMINAL; trace_put(rec); return; }
    // A-3 monotone barrier update (Table I row 7).  Two tiny steps in a row (Table I row 4) force one
    // decrease; when mu cannot decrease any more the search direction has become too small to make progress.
    int nmu = 0;
    const double mu_min = o->tol / 10.0;
    bool force = tiny_flag != 0;
    tiny_flag = 0;
    const int ncomp = pb->nL + pb->nU;
    const bool adaptive = o->mu_strategy == 1 && mode == 0 && ncomp > 0;
    double avg = 0.0;
    if (adaptive) {
        // Table I row 7: the adaptive rule runs while the KKT error keeps falling ("free mode"); an
        // iterate that fails to bring it below adaptive_red_fact x the largest of the last adaptive_red_iters values
        // hands over to the monotone schedule from mu = adaptive_monotone_init x average complementarity until its
        // barrier problem is solved; then the adaptive rule returns.  (b1 holds the dual residual without damping.)
        double s1 = 0.0, s3 = 0.0;
        for (int i = lane; i < nX; i += NT) {
            const double l = lo(i), u = hi(i);
            s1 += fabs(b1[i]);
            if (l > -INFINITY) s3 += (x[i] - l) * zL[i];
            if (u < INFINITY) s3 += (u - x[i]) * zU[i];
        }
        s1 = c.tm.sum(s1); s3 = c.tm.sum(s3);
        avg = s3 / ncomp;
        const double kkt = s1 / nX + (m > 0 ? theta / m : 0.0) + s3 / ncomp;
        if (mu_max < 0.0) mu_max = o->adaptive_mu_max_fact * avg;
        const int keep = o->adaptive_red_iters < 4 ? o->adaptive_red_iters : 4;
        if (mu_free) {
            double hmax = 0.0;
            const int nh = nhist < keep ? nhist : keep;
            for (int q = 0; q < nh; ++q) hmax = fmax(hmax, hist[(nhist - 1 - q) & 3]);
            if (nh > 0 && kkt > o->adaptive_red_fact * hmax) {
                mu_free = 0;
                mu = fmin(mu_max, fmax(mu_min, o->adaptive_monotone_init * avg));
                tau = fmax(o->tau_min, 1.0 - mu);
                nfilt = 0;
                wd_active = 0; wd_trials = 0; n_short = 0; soft = 0; soft_count = 0;
                rec[21] = 1.0;
            } else {
                hist[nhist & 3] = kkt; nhist++;
            }
        } else if (opt_error(mu, sd, sc) <= o->kappa_eps * mu) {
            mu_free = 1;
            hist[0] = kkt; nhist = 1;
            rec[21] = 2.0;
        }
        rec[20] = mu_free ? 1.0 : 2.0;
    }
    while (!adaptive && nmu < o->max_mu_updates && (force || opt_error(mu, sd, sc) <= o->kappa_eps * mu)) {
        if (!(mu > mu_min)) {
            if (force) {
                status = mode ? JIPM_ST_RESTORATION_FAILED : JIPM_ST_TINY_STEP;
                rec[5] = KIND_TERMINAL; rec[11] = nmu; trace_put(rec); return;
            }
            break;
        }
        force = false;
        mu = fmax(mu_min, fmin(o->kappa_mu * mu, pow(mu, o->theta_mu)));
        tau = fmax(o->tau_min, 1.0 - mu);
        nfilt = 0;
        nmu++;
        // a new barrier problem: the watchdog, its counter and the soft restoration phase start afresh
        wd_active = 0; wd_trials = 0; n_short = 0; soft = 0; soft_count = 0;
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
    rec[11] = nmu; rec[14] = theta;
    for (int i = lane; i < m; i += NT) b2[i] = -cv[i];
    c.tm.sync();
    // A-4 search direction with inertia correction (Algorithm IC); a solve whose refinement on (6) fails
    // sends the matrix back to Algorithm IC as if it were singular (reading S-7)
    int nfact = 0, npsing = 0, nref = 0;
    double dw = 0.0, dc = 0.0;
    bool resume = false, rhs_built = false;
    c.tick(15, clock64() - t_hd);
    while (true) {
        if (!ic_loop(resume, dw, dc, nfact)) { rec[13] = mu; enter_restoration(rec, KIND_IC_FAIL); trace_put(rec); return; }
        if (!rhs_built) {
            if (adaptive && mu_free) {
                // Mehrotra's probing with the factorisation of this iteration (it does not depend on mu): affine-scaling
                // step = Newton step on (5) with mu = 0 (into the correction's vectors, free at this point); mu_aff =
                // average complementarity after the largest feasible step; sigma = (mu_aff / average)^3; mu = sigma avg
                Vec a1 = VX(L->ab1); Vec a3 = VX(L->ab3); Vec a4 = VX(L->ab4);
                Vec sx = VX(L->sx); double* sy = V(L->sy); Vec szL = VX(L->szL); Vec szU = VX(L->szU);
                for (int i = lane; i < nX; i += NT) {
                    const double l = lo(i), u = hi(i);
                    a1[i] = -b1[i];
                    a3[i] = (l > -INFINITY) ? -(x[i] - l) * zL[i] : 0.0;
                    a4[i] = (u < INFINITY) ? -(u - x[i]) * zU[i] : 0.0;
                }
                c.tm.sync();
                bool failed_aff;
                solve_full(a1, b2, a3, a4, sx, sy, szL, szU, failed_aff);
                const double a_p = ftb_primal(x, sx, 1.0);
                const double a_d = ftb_dual(zL, zU, szL, szU, 1.0);
                double sa = 0.0;
                for (int i = lane; i < nX; i += NT) {
                    const double l = lo(i), u = hi(i);
                    if (l > -INFINITY) sa += ((x[i] - l) + a_p * sx[i]) * (zL[i] + a_d * szL[i]);
                    if (u < INFINITY) sa += ((u - x[i]) - a_p * sx[i]) * (zU[i] + a_d * szU[i]);
                }
                const double mu_aff = c.tm.sum(sa) / ncomp;
                const double r = mu_aff / avg;
                const double sigma = (avg > 0.0) ? fmin(o->adaptive_sigma_max, r * r * r) : 1.0;
                mu = fmin(mu_max, fmax(mu_min, sigma * avg));
                tau = fmax(o->tau_min, 1.0 - mu);
                nfilt = 0;
                wd_active = 0; wd_trials = 0; n_short = 0; soft = 0; soft_count = 0;
            }
            // right-hand side of (6) (it does not depend on the perturbations)
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
            c.tm.sync();
            rhs_built = true;
        }
        bool failed;
        const long long t_sf = clock64();
        nref = solve_full(b1, b2, b3, b4, dx, dy, dzL, dzU, failed);
        c.tick(13, clock64() - t_sf);
        if (!failed) break;
        npsing++;
        resume = true;
    }
    rec[13] = mu;
    rec[1] = nfact; rec[2] = dw; rec[3] = dc; rec[4] = nref; rec[19] = npsing;
    if (dw > 0.0) dw_last = dw;
    // A-5 line search
    double gd_part = 0.0, xm = 0.0, dym = 0.0;
    for (int i = lane; i < nX; i += NT) {
        const double l = lo(i), u = hi(i);
        const bool hl = l > -INFINITY, hu = u < INFINITY;
        double gp = g[i];
        if (hl) gp -= mu / (x[i] - l);
        if (hu) gp += mu / (u - x[i]);
        if (hl && !hu) gp += o->kappa_d * mu;
        if (hu && !hl) gp -= o->kappa_d * mu;
        gd_part += gp * dx[i];
        xm = fmax(xm, fabs(dx[i]) / (1.0 + fabs(x[i])));
    }
    for (int i = lane; i < m; i += NT) dym = fmax(dym, fabs(dy[i]));
    double gd = c.tm.sum(gd_part);
    xm = c.tm.max(xm); dym = c.tm.max(dym);
    double theta_k = theta;
    double phi_k = phi(x, f, mu, nX);
    rec[15] = phi_k;
    double a_max = ftb_primal(x, dx, tau);
    const long long t_ls = clock64();
    // Table I row 4: a step too small for backtracking to refine is accepted as it is
    if (xm <= o->tiny_step_tol && cmax <= o->tiny_step_cviol) {
        rec[18] = 1.0;
        if (tiny_last && dym < o->tiny_step_y_tol) tiny_flag = 1;
        tiny_last = 1;
        Trial t;
        trial(dx, a_max, t);
        const double a_z = ftb_dual(zL, zU, dzL, dzU, tau);
        accept_step(0, dx, dy, dzL, dzU, a_max, a_max, a_z, t);
        rec[5] = KIND_TINY; rec[8] = a_max; rec[9] = a_z; rec[10] = 1.0;
        trace_put(rec);
        if (mode) try_exit_restoration();
        return;
    }
    tiny_last = 0;
    // Table I row 5: in the soft restoration phase the acceptance criterion is a reduction of the
    // primal-dual error, until the original criterion holds again or the iteration limit is reached
    if (soft) {
        soft_count++;
        if (soft_count > o->max_soft_resto_iters || !soft_step(rec, theta_k, phi_k, gd)) {
            soft = 0;
            enter_restoration(rec, KIND_LS_FAIL); trace_put(rec); return;
        }
        trace_put(rec);
        if (mode) try_exit_restoration();
        return;
    }
    // Table I row 3: after watchdog_trigger shortened steps in a row the watchdog wakes up: it keeps
    // the entry iterate and direction, takes full steps without any test and either reaches a point acceptable to the
    // entry iterate's criterion or, after watchdog_trial_max trials, returns to the entry iterate
    if (!wd_active && o->watchdog_trigger > 0 && n_short >= o->watchdog_trigger) {
        Vec wx = VX(L->wx); Vec wzL = VX(L->wzL); Vec wzU = VX(L->wzU);
        Vec wdx = VX(L->wdx); Vec wdzL = VX(L->wdzL); Vec wdzU = VX(L->wdzU);
        double* wy = V(L->wy); double* wdy = V(L->wdy);
        for (int i = lane; i < nX; i += NT) {
            wx[i] = x[i]; wzL[i] = zL[i]; wzU[i] = zU[i]; wdx[i] = dx[i]; wdzL[i] = dzL[i]; wdzU[i] = dzU[i];
        }
        for (int i = lane; i < m; i += NT) { wy[i] = y[i]; wdy[i] = dy[i]; }
        c.tm.sync();
        wd_theta = theta_k; wd_phi = phi_k; wd_gd = gd; wd_alpha = a_max; wd_trials = 0; wd_active = 1;
        rec[16] = 1.0;
    }
    int acc = -1;
    double alpha = a_max, alpha_acc = 0.0;
    Trial ta;
    bool ok;
    if (wd_active) {
        Trial t;
        trial(dx, a_max, t);
        const bool good = acceptable(t.th, t.ph, wd_theta, wd_phi, wd_alpha, wd_gd);
        if (good || (wd_trials + 1 <= o->watchdog_trial_max && isfinite(t.th) && isfinite(t.ph))) {
            bool ftype = true;
            if (good) {  // acceptable to the entry iterate's criterion: the watchdog succeeded
                ftype = switching(wd_alpha, wd_gd, wd_theta) && armijo(t.ph, wd_phi, wd_alpha, wd_gd);
                if (!ftype) filter_add((1.0 - o->gamma_theta) * wd_theta, wd_phi - o->gamma_phi * wd_theta);
                wd_active = 0; wd_trials = 0; n_short = 0;
                rec[16] = 3.0;
            } else {     // taken unconditionally
                wd_trials++;
                if (rec[16] == 0.0) rec[16] = 2.0;
            }
            const double a_z = ftb_dual(zL, zU, dzL, dzU, tau);
            accept_step(0, dx, dy, dzL, dzU, a_max, a_max, a_z, t);
            rec[5] = KIND_NEWTON; rec[8] = a_max; rec[9] = a_z; rec[10] = ftype ? 1.0 : 0.0;
            c.tick(14, clock64() - t_ls);
            trace_put(rec);
            if (mode) try_exit_restoration();
            return;
        }
        // the watchdog gives up: back to its entry iterate and direction, ordinary backtracking from there (the full
        // step of the entry iterate was tried when the watchdog started: skipped; no correction)
        {
            Vec wx = VX(L->wx); Vec wzL = VX(L->wzL); Vec wzU = VX(L->wzU);
            Vec wdx = VX(L->wdx); Vec wdzL = VX(L->wdzL); Vec wdzU = VX(L->wdzU);
            const double* wy = V(L->wy); const double* wdy = V(L->wdy);
            for (int i = lane; i < nX; i += NT) {
                x[i] = wx[i]; zL[i] = wzL[i]; zU[i] = wzU[i]; dx[i] = wdx[i]; dzL[i] = wdzL[i]; dzU[i] = wdzU[i];
            }
            for (int i = lane; i < m; i += NT) { y[i] = wy[i]; dy[i] = wdy[i]; }
            c.tm.sync();
        }
        theta_k = wd_theta; phi_k = wd_phi; gd = wd_gd; a_max = wd_alpha;
        wd_active = 0; wd_trials = 0; n_short = 0;
        rec[16] = 4.0;
        // f, c, grad f, J and the residuals of (5a-d) at the entry iterate again (the soft phase may need them)
        f = eval_point(x, cv, theta, cmax, f_base, theta_base, cmax_base, f_pn, f_q);
        c.eval_derivs(x, y, mode ? 0.0 : 1.0);
        n_deriv++;
        if (mode) {
            const double* xR = V(L->xR); const double* DR2 = V(L->DR2);
            for (int i = lane; i < n; i += NT) g[i] = zeta * DR2[i] * (x[i] - xR[i]);
            for (int i = n + lane; i < nX; i += NT) g[i] = o->rho_resto;
            c.tm.sync();
        }
        for (int i = lane; i < nX; i += NT) {
            const double l = lo(i), u = hi(i);
            const bool hl = l > -INFINITY, hu = u < INFINITY;
            double dmp = 0.0;
            if (hl && !hu) dmp = o->kappa_d * mu;
            if (hu && !hl) dmp = -o->kappa_d * mu;
            b1[i] = -(g[i] + ATx(y, i) - zL[i] + zU[i] + dmp);
            b3[i] = hl ? mu - (x[i] - l) * zL[i] : 0.0;
            b4[i] = hu ? mu - (u - x[i]) * zU[i] : 0.0;
        }
        c.tm.sync();
        ok = backtrack(dx, theta_k, phi_k, gd, a_max, true, false, rec, acc, alpha, alpha_acc, ta);
    } else {
        ok = backtrack(dx, theta_k, phi_k, gd, a_max, false, true, rec, acc, alpha, alpha_acc, ta);
    }
    c.tick(14, clock64() - t_ls);
    if (!ok) {
        // the line search failed: first the soft restoration phase (row 5), then the hard one (row 6)
        if (o->soft_resto_factor > 0.0) {
            soft = 1; soft_count = 0;
            filter_add((1.0 - o->gamma_theta) * theta_k, phi_k - o->gamma_phi * theta_k);
            if (soft_step(rec, theta_k, phi_k, gd)) {
                trace_put(rec);
                if (mode) try_exit_restoration();
                return;
            }
            soft = 0;
        }
        enter_restoration(rec, KIND_LS_FAIL); trace_put(rec); return;
    }
    // A-6 accept, A-7 filter augmentation
    const double* ay = (acc == 1) ? V(L->sy) : dy;
    const Vec azL = (acc == 1) ? VX(L->szL) : dzL;
    const Vec azU = (acc == 1) ? VX(L->szU) : dzU;
    const double a_z = ftb_dual(zL, zU, azL, azU, tau);
    const bool ftype = switching(alpha, gd, theta_k) && armijo(ta.ph, phi_k, alpha, gd);
    if (!ftype) filter_add((1.0 - o->gamma_theta) * theta_k, phi_k - o->gamma_phi * theta_k);
    n_short = (rec[6] > 0.0) ? n_short + 1 : 0;
    accept_step(acc, dx, ay, azL, azU, alpha_acc, alpha_acc, a_z, ta);
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
