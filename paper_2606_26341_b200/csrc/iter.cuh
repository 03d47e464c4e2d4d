// iter.cuh -- the fused interior-point iteration (Table I) for one problem slot
// owned by one team (= one CTA), plus Step I (initialisation) and the slot refill loop.
// Step names (I-*, A-*, IC-*) follow SURVEY.md section 8(c) / DESIGN.md.
#pragma once
#include "core.cuh"
#include "derivs.cuh"
#include "kkt.cuh"

namespace jipm {

enum { KIND_NEWTON = 0, KIND_SOC = 1, KIND_LS_FAIL = 2, KIND_IC_FAIL = 3, KIND_TERMINAL = 4, KIND_TINY = 5, KIND_SOFT = 6 };

// what one trial-point evaluation returns (team-uniform)
struct Trial {
    double f, th, cm, ph;            // objective, ||c||_1, ||c||_inf, barrier objective of the ACTIVE problem
    double fb, thb, cmb, fpn, fq;    // base problem's f, theta, ||c||_inf and the restoration objective's parts
};

template <class C>
struct Solver {
    using X = Ctx<C>;
    using K = Kkt<C>;
    static constexpr int NX = C::NX, NU = C::NU, NZ = C::NZ, PD = C::PD, AX = C::AX, NA = C::NA, NT = C::NT;
    X& c;
    ArgsProxy A;
    PbProxy pb;
    LayProxy L;
    OptProxy o;
    int lane;
    // team-uniform scalar state of the problem in this slot
    double mu, tau, dw_last, theta_min, theta_max, f, theta, cmax;
    int k, status, nfilt, nrec;
    // line-search memory of the ACTIVE problem (Table I rows 3-5): it starts afresh whenever the
    // barrier parameter changes and on entering / leaving restoration, so nothing is parked across modes
    int n_short, wd_active, wd_trials, soft, soft_count, tiny_last, tiny_flag;
    double wd_theta, wd_phi, wd_gd, wd_alpha;
    // adaptive barrier parameter (Table I row 7): free mode or monotone phase, the upper bound of mu,
    // the KKT errors of the last accepted free-mode iterates (regular problem only; restoration is always monotone)
    int mu_free, nhist;
    double mu_max, hist[4];
    int acc_count;   // consecutive acceptable regular iterations (acceptable-level termination, reading AT)
    // restoration mode (Table I row 6): mode 1 iterates on X = [x; p; n] with the same kernel
    // code; the regular problem's scalars are parked in *_reg until the exit test succeeds
    int mode, nX, nfilt_reg;
    double mu_reg, tau_reg, dw_last_reg, theta_min_reg, theta_max_reg;
    double theta_entry, zeta, f_pn, f_q, f_base, theta_base, cmax_base, dc_cur;
    long long pid;
    unsigned n_fact, n_solve, n_deriv, n_fc, n_iter, n_resto;
    // SM-clock cycles this team spent in: 0 derivatives, 1 factorisations, 2 KKT solves, 3 residuals of (6),
    // 4 trial-point evaluations, 5 whole iterations, 6 Step I, 7 (spare)
    double* bl; double* bu;

    __device__ Solver(X& c_) : c(c_), lane(c_.lane) {
        n_fact = n_solve = n_deriv = n_fc = n_iter = n_resto = 0;
        // the shared bounds, copied next to the iterate once per kernel
        bl = c.vh(L->bl); bu = c.vh(L->bu);
        for (int q = lane; q < pb->n; q += NT) { bl[q] = pb->xL[q]; bu[q] = pb->xU[q]; }
        c.tm.sync();
        c.build_maps();
        mode = 0; nX = pb->n;
        reset_ls_memory();
    }
    __device__ __forceinline__ void reset_ls_memory() {
        n_short = wd_active = wd_trials = soft = soft_count = tiny_last = tiny_flag = acc_count = 0;
        wd_theta = wd_phi = wd_gd = wd_alpha = 0.0;
    }
    __device__ __forceinline__ void reset_mu_memory() {
        mu_free = 1; nhist = 0; mu_max = -1.0;
        hist[0] = hist[1] = hist[2] = hist[3] = 0.0;
    }
    __device__ __forceinline__ double* V(int off) const { return c.v(off); }
    __device__ __forceinline__ double* VH(int off) const { return c.vh(off); }
    __device__ __forceinline__ Vec VX(int off) const {
        Vec r;
        r.a = c.v(off); r.n = pb->n;
        r.t = c.v(L->tail0 + ((off - L->pv0) / L->npad) * L->tpad) - pb->n;
        return r;
    }
    // bounds of the extended primal vector: entries >= n are the restoration variables p, n >= 0
    __device__ __forceinline__ double lo(int i) const { return i < pb->n ? bl[i] : 0.0; }
    __device__ __forceinline__ double hi(int i) const { return i < pb->n ? bu[i] : INFINITY; }
    __device__ __forceinline__ bool hasL(int i) const { return lo(i) > -INFINITY; }
    __device__ __forceinline__ bool hasU(int i) const { return hi(i) < INFINITY; }
    __device__ __forceinline__ double* filt_active() const { return V(mode ? L->filtR : L->filt); }

    // barrier objective (3) with the one-sided damping term; NaN outside the interior
    __device__ __noinline__ double phi(const Vec x, double fv, double mu_, int nvar) const {
        double s = 0.0;
        int badpt = 0;
        for (int i = lane; i < nvar; i += NT) {
            const double l = lo(i), u = hi(i), xi = x[i];
            const bool hl = l > -INFINITY, hu = u < INFINITY;
            if (hl) {
                const double sl = xi - l;
                if (!(sl > 0.0)) badpt = 1;
                s -= mu_ * log(sl);
                if (!hu) s += o->kappa_d * mu_ * sl;
            }
            if (hu) {
                const double su = u - xi;
                if (!(su > 0.0)) badpt = 1;
                s -= mu_ * log(su);
                if (!hl) s += o->kappa_d * mu_ * su;
            }
        }
        s = c.tm.sum(s);
        if (c.tm.any(badpt)) return NAN;
        return fv + s;
    }

    // fraction to the boundary (PAPER.md:148 fn 2) on the primal step
    __device__ double ftb_primal(const Vec x, const Vec dx, double tau_) const {
        double a = 1.0;
        for (int i = lane; i < nX; i += NT) {
            const double l = lo(i), u = hi(i), d = dx[i];
            if (l > -INFINITY && d < 0.0) a = fmin(a, -tau_ * (x[i] - l) / d);
            if (u < INFINITY && d > 0.0) a = fmin(a, tau_ * (u - x[i]) / d);
        }
        return c.tm.min(a);
    }
    __device__ double ftb_dual(const Vec zL, const Vec zU, const Vec dzL, const Vec dzU,
                               double tau_) const {
        double a = 1.0;
        for (int i = lane; i < nX; i += NT) {
            if (hasL(i) && dzL[i] < 0.0) a = fmin(a, -tau_ * zL[i] / dzL[i]);
            if (hasU(i) && dzU[i] < 0.0) a = fmin(a, -tau_ * zU[i] / dzU[i]);
        }
        return c.tm.min(a);
    }

    // optimality error E_mu from the dual residual base in b1 (= grad f + A^T y - zL + zU)
    __device__ double opt_error(double mu_, double sd, double sc) const {
        Vec x = VX(L->x); Vec zL = VX(L->zL); Vec zU = VX(L->zU); Vec rdb = VX(L->b1);
        double ed = 0.0, es = 0.0;
        for (int i = lane; i < nX; i += NT) {
            const double l = lo(i), u = hi(i);
            const bool hl = l > -INFINITY, hu = u < INFINITY;
            double dmp = 0.0;
            if (hl && !hu) dmp = o->kappa_d * mu_;
            if (hu && !hl) dmp = -o->kappa_d * mu_;
            ed = fmax(ed, fabs(rdb[i] + dmp));
            if (hl) es = fmax(es, fabs((x[i] - l) * zL[i] - mu_));
            if (hu) es = fmax(es, fabs((u - x[i]) * zU[i] - mu_));
        }
        ed = c.tm.max(ed); es = c.tm.max(es);
        return fmax(fmax(ed / sd, cmax), es / sc);
    }

    // unscaled max-norms of the dual residual and of the complementarity products at mu = 0 (b1 holds the dual residual);
    // with cmax they are the three bounds of the acceptable-level test (reading AT)
    __device__ __noinline__ void error_parts(double& ed, double& es) const {
        Vec x = VX(L->x); Vec zL = VX(L->zL); Vec zU = VX(L->zU); Vec rdb = VX(L->b1);
        double a = 0.0, b = 0.0;
        for (int i = lane; i < nX; i += NT) {
            const double l = lo(i), u = hi(i);
            a = fmax(a, fabs(rdb[i]));
            if (l > -INFINITY) b = fmax(b, fabs((x[i] - l) * zL[i]));
            if (u < INFINITY) b = fmax(b, fabs((u - x[i]) * zU[i]));
        }
        ed = c.tm.max(a); es = c.tm.max(b);
    }

    // filter ([7] sec 2.3): entries (theta_j, phi_j) in the workspace
    __device__ bool in_filter_of(const double* F, int nf, double thmax, double th_t, double ph_t) const {
        if (th_t >= thmax) return true;
        int hit = 0;
        for (int j = lane; j < nf; j += NT) hit |= (th_t >= F[2 * j] && ph_t >= F[2 * j + 1]);
        return c.tm.any(hit);
    }
    // acceptance test of one speculative candidate by ONE WARP (the filter scanned 32 entries at a time)
    __device__ bool acceptable_warp(double th_t, double ph_t, double th_k, double ph_k, double alpha, double g) const {
        if (!(isfinite(th_t) && isfinite(ph_t))) return false;
        if (th_t >= theta_max) return false;
        const double* F = filt_active();
        int hit = 0;
        for (int j = lane & 31; j < nfilt; j += 32) hit |= (th_t >= F[2 * j] && ph_t >= F[2 * j + 1]);
        if (__any_sync(FULL, hit)) return false;
        if (th_k <= theta_min && switching(alpha, g, th_k)) return armijo(ph_t, ph_k, alpha, g);
        return th_t <= (1.0 - o->gamma_theta) * th_k ||
               ph_t - ph_k - 10.0 * EPS_MACH * fabs(ph_k) <= -o->gamma_phi * th_k;
    }
    __device__ bool in_filter(double th_t, double ph_t) const {
        return in_filter_of(filt_active(), nfilt, theta_max, th_t, ph_t);
    }
    // add an entry; entries dominated by the new one (their forbidden region is a subset of the new region) are
    // dropped first, which changes no decision (reading S-10).  Serial on lane 0: at most MAX_FILTER entries, once
    // per h-type step.
    __device__ void filter_add(double th_e, double ph_e) {
        double* F = filt_active();
        int nf = 0;
        if (lane == 0) {
            for (int j = 0; j < nfilt; ++j) {
                const double t = F[2 * j], p = F[2 * j + 1];
                if (!(t >= th_e && p >= ph_e)) { F[2 * nf] = t; F[2 * nf + 1] = p; ++nf; }
            }
            if (nf == MAX_FILTER) nf = MAX_FILTER - 1;  // overflow: the newest old entry is dropped (counted nowhere: never seen)
            F[2 * nf] = th_e; F[2 * nf + 1] = ph_e;
        }
        nfilt = c.tm.bcast0(nf) + 1;  // (the reduction's barrier also publishes lane 0's writes)
    }
    __device__ bool switching(double alpha, double g, double theta_k) const {
        return g < 0.0 && alpha * pow(-g, o->s_phi) > o->delta * pow(theta_k, o->s_theta);
    }
    __device__ bool armijo(double phi_t, double phi_k, double alpha, double g) const {
        return phi_t - phi_k - 10.0 * EPS_MACH * fabs(phi_k) <= o->eta_phi * alpha * g;
    }
    __device__ bool acceptable(double th_t, double ph_t, double th_k, double ph_k, double alpha, double g) const {
        if (!(isfinite(th_t) && isfinite(ph_t))) return false;
        if (in_filter(th_t, ph_t)) return false;
        if (th_k <= theta_min && switching(alpha, g, th_k)) return armijo(ph_t, ph_k, alpha, g);
        return th_t <= (1.0 - o->gamma_theta) * th_k ||
               ph_t - ph_k - 10.0 * EPS_MACH * fabs(ph_k) <= -o->gamma_phi * th_k;
    }

    // ---- linear algebra of one iteration ---------------------------------------------------------------
    // Sig = zL/sL + zU/sU + Hd, Hd = delta_w (+ zeta D_R^2 on x in restoration mode); Dc = delta_c, plus in
    // restoration mode the Schur complement 1/Sig_p + 1/Sig_n of the eliminated (p, n) pairs ([7] sec 3.3)
    __device__ void set_sigma(double dw, double dc) {
        dc_cur = dc;
        Vec x = VX(L->x); Vec zL = VX(L->zL); Vec zU = VX(L->zU);
        Vec Sig = VX(L->Sig); Vec Hd = VX(L->Hd); double* Dc = VH(L->Dc);
        const double* DR2 = V(L->DR2);
        for (int i = lane; i < nX; i += NT) {
            const double l = lo(i), u = hi(i);
            const double hd = (mode && i < pb->n) ? dw + zeta * DR2[i] : dw;
            double s = hd;
            if (l > -INFINITY) s += zL[i] / (x[i] - l);
            if (u < INFINITY) s += zU[i] / (u - x[i]);
            Sig[i] = s; Hd[i] = hd;
        }
        c.tm.sync();
        for (int i = lane; i < pb->m; i += NT)
            Dc[i] = mode ? dc + 1.0 / Sig[pb->n + i] + 1.0 / Sig[pb->n + pb->m + i] : dc;
        c.tm.sync();
    }

    // products with the constraint Jacobian / Lagrangian Hessian of the (extended) problem
    __device__ __forceinline__ double ATx(const double* y, int i) const {
        if (i < pb->n) return c.AT_entry(y, i);
        return (i < pb->n + pb->m) ? -y[i - pb->n] : y[i - pb->n - pb->m];
    }
    __device__ __forceinline__ double Wx(const Vec d, int i) const { return i < pb->n ? c.W_entry(d.a, i) : 0.0; }

    // solve (6) through (7) + the Delta z recovery of PAPER.md:110 for rhs (b1,b2,b3,b4) -> (d1..d4)
    __device__ void reduced_solve(const Vec b1, const double* b2, const Vec b3, const Vec b4,
                                  Vec d1, double* d2, Vec d3, Vec d4) {
        Vec x = VX(L->x); Vec zL = VX(L->zL); Vec zU = VX(L->zU);
        Vec rr = VX(L->rr);
        for (int i = lane; i < nX; i += NT) {
            const double l = lo(i), u = hi(i);
            double r = b1[i];
            if (l > -INFINITY) r += b3[i] / (x[i] - l);
            if (u < INFINITY) r -= b4[i] / (u - x[i]);
            rr[i] = r;
        }
        c.tm.sync();
        const double* rc = b2;
        Vec Sig = VX(L->Sig);
        const int n = pb->n, m = pb->m;
        if (mode) {  // eliminate (dp, dn): dp = (r_p + dy)/Sig_p, dn = (r_n - dy)/Sig_n
            double* rc2 = V(L->rc2);
            for (int j = lane; j < m; j += NT) rc2[j] = b2[j] + rr[n + j] / Sig[n + j] - rr[n + m + j] / Sig[n + m + j];
            c.tm.sync();
            rc = rc2;
        }
        const long long t0 = clock64();
        K::solve(c, rr.a, rc, d1.a, d2, mode != 0 || dc_cur != 0.0);
        c.tick(2, clock64() - t0);
        n_solve++;
        if (mode) {
            for (int j = lane; j < m; j += NT) {
                d1[n + j] = (rr[n + j] + d2[j]) / Sig[n + j];
                d1[n + m + j] = (rr[n + m + j] - d2[j]) / Sig[n + m + j];
            }
            c.tm.sync();
        }
        for (int i = lane; i < nX; i += NT) {
            const double l = lo(i), u = hi(i);
            d3[i] = (l > -INFINITY) ? (b3[i] - zL[i] * d1[i]) / (x[i] - l) : 0.0;
            d4[i] = (u < INFINITY) ? (b4[i] + zU[i] * d1[i]) / (u - x[i]) : 0.0;
        }
        c.tm.sync();
    }

    // residual of the unreduced system (6): r = b - M d; returns ||r||_inf; dnorm = ||d||_inf
    __device__ double full_residual(const Vec b1, const double* b2, const Vec b3, const Vec b4,
                                    const Vec d1, const double* d2, const Vec d3, const Vec d4,
                                    double& dnorm) const {
        Vec x = VX(L->x); Vec zL = VX(L->zL); Vec zU = VX(L->zU);
        Vec Hd = VX(L->Hd);
        Vec r1 = VX(L->r1); double* r2 = VH(L->r2); Vec r3 = VX(L->r3); Vec r4 = VX(L->r4);
        double rn = 0.0, dn = 0.0;
        for (int i = lane; i < nX; i += NT) {
            const double l = lo(i), u = hi(i);
            const double lhs1 = Wx(d1, i) + Hd[i] * d1[i] + ATx(d2, i) - d3[i] + d4[i];
            const double v1 = b1[i] - lhs1;
            r1[i] = v1; rn = fmax(rn, fabs(v1));
            double v3 = 0.0, v4 = 0.0;
            if (l > -INFINITY) v3 = b3[i] - (zL[i] * d1[i] + (x[i] - l) * d3[i]);
            if (u < INFINITY) v4 = b4[i] - (-zU[i] * d1[i] + (u - x[i]) * d4[i]);
            r3[i] = v3; r4[i] = v4;
            rn = fmax(rn, fmax(fabs(v3), fabs(v4)));
            dn = fmax(dn, fmax(fabs(d1[i]), fmax(fabs(d3[i]), fabs(d4[i]))));
        }
        c.A_mul(d1.a, r2);
        for (int i = lane; i < pb->m; i += NT) {
            double ad = r2[i];
            if (mode) ad += d1[pb->n + pb->m + i] - d1[pb->n + i];
            const double v2 = b2[i] - (ad - dc_cur * d2[i]);
            r2[i] = v2; rn = fmax(rn, fabs(v2)); dn = fmax(dn, fabs(d2[i]));
        }
        c.tm.sync();
        dnorm = c.tm.max(dn);
        return c.tm.max(rn);
    }

    // solve (6) with iterative refinement on the unreduced system (reading S-7); returns #refinements.  At least
    // refine_min steps; stops at ratio <= residual_ratio_max; gives up when refine_max is reached or a step no longer
    // improves the ratio -- then the solution is kept if the ratio is below residual_ratio_singular, else `failed`
    // is set and the caller pretends the matrix is singular (Algorithm IC continues with delta_c > 0).
    __device__ __noinline__ int solve_full(const Vec b1, const double* b2, const Vec b3, const Vec b4,
                              Vec d1, double* d2, Vec d3, Vec d4, bool& failed) {
        reduced_solve(b1, b2, b3, b4, d1, d2, d3, d4);
        double bn = 0.0;
        for (int i = lane; i < nX; i += NT) bn = fmax(bn, fmax(fabs(b1[i]), fmax(fabs(b3[i]), fabs(b4[i]))));
        for (int i = lane; i < pb->m; i += NT) bn = fmax(bn, fabs(b2[i]));
        bn = c.tm.max(bn);
        int nref = 0;
        failed = false;
        Vec e1 = VX(L->e1); double* e2 = VH(L->e2); Vec e3 = VX(L->e3); Vec e4 = VX(L->e4);
        auto ratio = [&]() {
            double dn;
            const long long t0 = clock64();
            const double rn = full_residual(b1, b2, b3, b4, d1, d2, d3, d4, dn);
            c.tick(3, clock64() - t0);
            const double den = bn + dn;
            return den > 0.0 ? rn / den : rn;
        };
        double rat = ratio();
        while (rat > o->residual_ratio_max || nref < o->refine_min) {
            if (!isfinite(rat)) { failed = true; break; }
            reduced_solve(VX(L->r1), VH(L->r2), VX(L->r3), VX(L->r4), e1, e2, e3, e4);
            for (int i = lane; i < nX; i += NT) { d1[i] += e1[i]; d3[i] += e3[i]; d4[i] += e4[i]; }
            for (int i = lane; i < pb->m; i += NT) d2[i] += e2[i];
            c.tm.sync();
            nref++;
            const double rat_old = rat;
            rat = ratio();
            if (rat > o->residual_ratio_max && nref > o->refine_min &&
                (nref >= o->refine_max || rat > o->residual_improvement_factor * rat_old)) {
                failed = !(rat < o->residual_ratio_singular);
                break;
            }
        }
        // Polish: the stop rule above is the oracle's, but its LAPACK factor sits at a ratio ~1e-16 after the one
        // compulsory step while the stage recursion can stop anywhere below 1e-10; the error left in Delta y is that
        // ratio times cond(7).  Up to three more steps while the ratio is above 1e-15 and still shrinking bring the
        // step within the parity tolerance of the oracle's (eq 8); they change no decision.
        const double polish_floor = 1e-15;
        for (int extra = 0; extra < o->polish_max && !failed && rat > polish_floor && nref < o->refine_max; ++extra) {
            reduced_solve(VX(L->r1), VH(L->r2), VX(L->r3), VX(L->r4), e1, e2, e3, e4);
            for (int i = lane; i < nX; i += NT) { d1[i] += e1[i]; d3[i] += e3[i]; d4[i] += e4[i]; }
            for (int i = lane; i < pb->m; i += NT) d2[i] += e2[i];
            c.tm.sync();
            nref++;
            const double rat_old = rat;
            rat = ratio();
            if (!(rat < 0.25 * rat_old)) break;
        }
        return nref;
    }

    __device__ void trace_put(const double* rec) {
        if (A->trace != nullptr && nrec < A->trace_cap && lane < JIPM_TRACE_W)
            A->trace[(pid * A->trace_cap + nrec) * JIPM_TRACE_W + lane] = rec[lane];
        nrec++;
    }

    __device__ void init_problem(long long id);
    __device__ void iterate();
    __device__ bool ic_loop(bool resume, double& dw, double& dc, int& nfact);
    __device__ __noinline__ void trial(const Vec dxv, double alpha, Trial& t);
    __device__ bool backtrack(const Vec dxv, double theta_k, double phi_k, double gd, double a_max, bool skip_first,
                              bool allow_soc, double* rec, int& acc, double& alpha, double& alpha_acc, Trial& ta);
    __device__ void accept_step(int acc_soc, const Vec dxv, const double* dyv, const Vec dzLv, const Vec dzUv,
                                double alpha_x, double alpha_y, double a_z, const Trial& ta);
    __device__ bool soft_step(double* rec, double theta_k, double phi_k, double gd);
    __device__ __noinline__ void trial_warp(const Vec x, const Vec dx, double alpha, double& th_t, double& ph_t) const;
    __device__ void enter_restoration(double* rec, int kind);
    __device__ void try_exit_restoration();
    __device__ __noinline__ double eval_point(const Vec xt, double* ct, double& th_t, double& cm_t, double& fb, double& thb,
                                 double& cmb, double& fpn, double& fq);
    __device__ void write_outputs();
    __device__ void dbg_load(const double* st);
    __device__ void dbg_store(double* st);
};

}  // namespace jipm
