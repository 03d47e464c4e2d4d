// jipm_api.cu -- host side of the C ABI declared in include/jipm.h.  No torch types, no CPU fallback.
#include <cstdio>
#include <cstring>
#include <cmath>
#include <string>
#include <vector>
#include <algorithm>
#include <mutex>
#include "launch.cuh"

using namespace jipm;

static thread_local std::string g_err = "";
static int fail(int code, const std::string& msg) { g_err = msg; return code; }
#define CUDA_TRY(expr)                                                                                   \
    do {                                                                                                 \
        cudaError_t e_ = (expr);                                                                         \
        if (e_ != cudaSuccess)                                                                           \
            return fail(e_ == cudaErrorMemoryAllocation ? JIPM_ERR_NOMEM : JIPM_ERR_CUDA,                \
                        std::string(#expr) + ": " + cudaGetErrorString(e_));                             \
    } while (0)


// Launch arguments live in ONE __constant__ block per family instantiation (inst.cuh): two solves of the same
// family must not overlap.  Every launch-to-completion section (run()) holds this lock.
static std::mutex g_launch_mutex;

// RAII switch to the solver's device for the duration of a call
struct DeviceGuard {
    int prev = -1; bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

struct jipm_solver {
    int family;
    int device = 0;
    jipm_family_dims dims;
    jipm_options o;
    Pb pb;
    Lay L;
    int NX, NU, NZ;
    Inst inst;
    int teams_per_sm;
    int n_slots;          // R: CTAs launched per solve (capped by the number of problems)
    int n_sm = 0;         // SMs of the solver's device; the global scratch holds n_sm * teams_per_sm workspaces
    unsigned* d_mask = nullptr;
    cudaStream_t stream;
    double *d_xL = nullptr, *d_xU = nullptr, *d_ws = nullptr;
    int* d_queue = nullptr;
    unsigned long long* d_stats = nullptr;
    double* trace = nullptr;
    int trace_cap = 0;
    long long stats[24] = {0};
    DbgLay dbg;
    // grow-only device staging of jipm_solve_batch_host
    double* d_stage = nullptr; size_t stage_doubles = 0;
    int32_t* d_istage = nullptr; size_t istage_ints = 0;
};

extern "C" const char* jipm_last_error(void) { return g_err.c_str(); }

extern "C" int jipm_default_options(jipm_options* o) {
    if (!o) return fail(JIPM_ERR_ARG, "options pointer is NULL");
    o->tol = 1e-8; o->mu_init = 0.1; o->kappa_eps = 10.0; o->kappa_mu = 0.2; o->theta_mu = 1.5; o->tau_min = 0.99;
    o->s_max = 100.0; o->kappa_sigma = 1e10; o->kappa_1 = 1e-2; o->kappa_2 = 1e-2; o->bound_relax_factor = 1e-8;
    o->bound_mult_init = 1.0; o->lam_init_max = 1e3; o->kappa_d = 1e-5; o->gamma_theta = 1e-5; o->gamma_phi = 1e-8;
    o->eta_phi = 1e-8; o->delta = 1.0; o->s_theta = 1.1; o->s_phi = 2.3; o->gamma_alpha = 0.05;
    o->theta_max_fact = 1e4; o->theta_min_fact = 1e-4; o->alpha_red = 0.5; o->kappa_soc = 0.99;
    o->delta_w_min = 1e-20; o->delta_w_0 = 1e-4; o->delta_w_max = 1e40; o->kappa_w_minus = 1.0 / 3.0;
    o->kappa_w_plus = 8.0; o->kappa_w_plus_first = 100.0; o->delta_c_bar = 1e-8; o->kappa_c = 0.25;
    o->residual_ratio_max = 1e-10; o->rho_resto = 1000.0; o->kappa_resto = 0.9; o->z_reset_threshold = 1e3;
    o->max_iter = 3000; o->max_backtrack = 64; o->max_soc = 4; o->refine_min = 1; o->refine_max = 10;
    o->max_mu_updates = 8; o->init_slacks = 1; o->enable_restoration = 1;
    o->residual_ratio_singular = 1e-5; o->residual_improvement_factor = 0.999999999;
    o->tiny_step_tol = 10.0 * 2.220446049250313e-16; o->tiny_step_y_tol = 1e-2; o->tiny_step_cviol = 1e-4;
    o->soft_resto_factor = 1.0 - 1e-4;
    o->watchdog_trigger = 10; o->watchdog_trial_max = 3; o->max_soft_resto_iters = 10; o->polish_max = 3;
    o->mu_strategy = 0; o->adaptive_red_iters = 4; o->adaptive_red_fact = 0.9999; o->adaptive_monotone_init = 0.8;
    o->adaptive_sigma_max = 100.0; o->adaptive_mu_max_fact = 1e3;
    o->acceptable_tol = 1e-6; o->acceptable_dual_inf_tol = 1e10; o->acceptable_constr_viol_tol = 1e-2;
    o->acceptable_compl_inf_tol = 1e-2; o->acceptable_iter = 0;
    return JIPM_OK;
}

static bool family_shape(int family, const jipm_family_dims* d, int& nx, int& nu, int& ng, int& nth, int& pd) {
    if (!d || d->horizon_N < 1 || d->horizon_N > 4096 || !(d->dt > 0.0)) return false;
    const int na = d->n_agents, nobs = d->n_obstacles;
    // core.cuh build_maps packs the inequality index of a knot into 8 bits with 254 / 255 as sentinels
    if (nobs > 254) return false;
    switch (family) {
        case JIPM_FAM_POINTMASS2D:
            if (na != 1 || nobs < 0) return false;
            nx = 4; nu = 2; ng = nobs; nth = 4 + 2 + 3 * nobs; pd = 2; return true;
        case JIPM_FAM_QUAD_TRACK:
            if (na != 1 || nobs < 0) return false;
            nx = 12; nu = 4; ng = nobs; nth = 12 + 2 + 4 * nobs; pd = 3; return true;
        case JIPM_FAM_QUAD_CLUTTER:
            if (na != 1 || nobs < 0) return false;
            nx = 12; nu = 4; ng = nobs; nth = 12 + 3 + 4 * nobs; pd = 3; return true;
        case JIPM_FAM_QUAT_NAV:
            if (na != 1 || nobs < 0) return false;
            nx = 13; nu = 4; ng = nobs; nth = 13 + 3 + 4 * nobs; pd = 3; return true;
        case JIPM_FAM_MULTIQUAD:
            if (na != 2 && na != 4) return false;
            nx = 12 * na; nu = 4 * na; ng = na * (na - 1) / 2; nth = 12 * na + 3 * na; pd = 3; return true;
        default: return false;
    }
}

extern "C" int jipm_family_sizes(int family, const jipm_family_dims* d, int64_t* n, int64_t* m, int64_t* n_theta) {
    int nx, nu, ng, nth, pd;
    if (!family_shape(family, d, nx, nu, ng, nth, pd)) return fail(JIPM_ERR_DIM, "bad family or dims");
    const int64_t N = d->horizon_N;
    if (n) *n = (N + 1) * nx + N * nu + N * ng;
    if (m) *m = (N + 1) * nx + N * ng;
    if (n_theta) *n_theta = nth;
    return JIPM_OK;
}

// Workspace layout of one slot.  Arrays are laid out in PRIORITY order; the first L.nsm doubles (as many whole
// arrays as the shared-memory budget holds) live in shared memory, the rest in the slot's global scratch.
static int build_layout(jipm_solver* s, int sm_budget_doubles) {
    const Pb& pb = s->pb;
    const int n = pb.n, m = pb.m, N = pb.N, NX = s->NX, NU = s->NU, NZ = s->NZ;
    const int pd = (pb.family == JIPM_FAM_POINTMASS2D) ? 2 : 3;
    Lay& L = s->L;
    struct Ent { int Lay::*f; int cnt; };
    const int rkn = pb.family == JIPM_FAM_POINTMASS2D ? 0 : N * pb.na * 4 * RKW;
    const int npad = (n + 1) & ~1, tpad = (2 * m + 1) & ~1;
    const Ent hot[] = {
        // the factor and what every solve streams through
        {&Lay::Psi, N * NX * NX}, {&Lay::pv, (N + 1) * NX}, {&Lay::qv, N * NX}, {&Lay::wv, N * NX}, {&Lay::sv, N * NX}, {&Lay::tv, N * NU},
        {&Lay::T, (N + 1) * NX * NX}, {&Lay::Kf, N * NU * NX}, {&Lay::Gf, N * NU * NU},
        {&Lay::J, N * NX * (NZ + 1)},  // row stride LDJ = NZ + 1 (core.cuh)
        {&Lay::Dc, m}, {&Lay::gv, N * pb.ng * pd}, {&Lay::dgv, N * pb.ng}, {&Lay::cnd, N * pb.na * pd * pb.na * pd}, {&Lay::tgt, (N + 1) * pb.na * pd},
        {&Lay::bl, n}, {&Lay::bu, n}, {&Lay::imap, (n + 1) / 2}, {&Lay::cmap, (m + 1) / 2},
        {&Lay::filt, 2 * MAX_FILTER},
        // m-vectors
        {&Lay::y, m}, {&Lay::c, m}, {&Lay::b2, m}, {&Lay::dy, m}, {&Lay::ct, m}, {&Lay::r2, m}, {&Lay::e2, m},
        {&Lay::W, N * NZ * NZ + NX * NX},
    };
    // primal-sized vectors: heads (n entries) contiguous with stride npad, in priority order; their restoration tails
    // (2m entries: p and n of Step R) live apart, always in the global scratch
    int Lay::*const primal[] = {
        &Lay::x, &Lay::rr, &Lay::dx, &Lay::Sig, &Lay::xt, &Lay::zL, &Lay::zU, &Lay::b1, &Lay::dzL, &Lay::dzU, &Lay::b3, &Lay::b4,
        &Lay::g, &Lay::Hd, &Lay::r1, &Lay::r3, &Lay::r4, &Lay::e1, &Lay::e3, &Lay::e4, &Lay::sx, &Lay::szL, &Lay::szU,
        &Lay::wx, &Lay::wzL, &Lay::wzU, &Lay::wdx, &Lay::wdzL, &Lay::wdzU, &Lay::ab1, &Lay::ab3, &Lay::ab4,
    };
    const Ent cold[] = {
        {&Lay::rk, rkn}, {&Lay::sy, m}, {&Lay::csoc, m}, {&Lay::bs2, m}, {&Lay::rc2, m},
        {&Lay::xR, n}, {&Lay::DR2, n}, {&Lay::filtR, 2 * MAX_FILTER}, {&Lay::wy, m}, {&Lay::wdy, m},
    };
    int o = 0;
    L.nsm = 0;
    L.pv0 = 0; L.npad = npad; L.tpad = tpad;
    const int n_primal = (int)(sizeof(primal) / sizeof(primal[0]));
    auto even = [](int c) { return (c + 1) & ~1; };  // keep 16-byte alignment
    int hot_total = 0;
    for (const Ent& e : hot) hot_total += even(e.cnt);
    const int hot_fits = hot_total <= sm_budget_doubles ? 1 : 0;  // the whole hot group is shared-memory resident
    // Arrays are placed in priority order; the first that does not fit ends the shared-memory part (everything after
    // it lives in the slot's L2 scratch).  A first-fit variant that keeps the small vectors on chip and sends the
    // factor blocks to L2 was measured on C2, C3 and the quaternion family and is 4-9 % SLOWER per slot-iteration
    // (DESIGN.md section 6): the factor blocks and J are the hotter data.
    bool in_sm = true;
    auto place = [&](int Lay::*f, int cnt0) {
        const int cnt = even(cnt0);
        if (in_sm && o + cnt > sm_budget_doubles) { in_sm = false; L.nsm = o; }
        L.*f = o;
        o += cnt;
    };
    for (const Ent& e : hot) place(e.f, e.cnt);
    L.pv0 = o;
    for (auto f : primal) place(f, n);
    for (const Ent& e : cold) place(e.f, e.cnt);
    if (in_sm) { in_sm = false; L.nsm = o; }
    L.tail0 = o;
    o += tpad * n_primal;
    L.total = o;
    return hot_fits;
}

static cudaError_t dispatch(jipm_solver* s, const Args& a) { return s->inst.launch(a, s->stream); }

extern "C" int jipm_create(jipm_solver** out, int family, const jipm_family_dims* d, int64_t n, int64_t m,
                           const double* x_L, const double* x_U, const jipm_options* opts, int64_t resident_slots,
                           void* cuda_stream) {
    if (!out || !x_L || !x_U) return fail(JIPM_ERR_ARG, "NULL argument");
    int nx, nu, ng, nth, pd;
    if (!family_shape(family, d, nx, nu, ng, nth, pd)) return fail(JIPM_ERR_DIM, "bad family or dims");
    int64_t n2, m2, nt2;
    jipm_family_sizes(family, d, &n2, &m2, &nt2);
    if (n != n2 || m != m2) return fail(JIPM_ERR_DIM, "n, m do not match jipm_family_sizes");
    if (resident_slots < 0) return fail(JIPM_ERR_ARG, "resident_slots < 0");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return fail(JIPM_ERR_CUDA, "no CUDA device (jipm has no CPU fallback)");
    jipm_solver* s = new jipm_solver();
    s->family = family; s->dims = *d;
    if (opts) s->o = *opts; else jipm_default_options(&s->o);
    s->stream = (cudaStream_t)cuda_stream;
    s->NX = nx; s->NU = nu; s->NZ = nx + nu;
    Pb& pb = s->pb;
    pb.family = family; pb.N = d->horizon_N; pb.ng = ng; pb.na = d->n_agents; pb.nobs = d->n_obstacles;
    pb.n = (int)n; pb.m = (int)m; pb.nth = nth; pb.blk = nu + nx + ng; pb.cblk = nx + ng;
    pb.dt = d->dt; pb.ru = (family == JIPM_FAM_POINTMASS2D) ? 0.1 : 0.01;
    pb.th_obs = (family == JIPM_FAM_POINTMASS2D) ? 6 : (family == JIPM_FAM_QUAD_TRACK ? 14 : (family == JIPM_FAM_QUAT_NAV ? 16 : 15));
    pb.th_goal = (family == JIPM_FAM_POINTMASS2D) ? 4 : (family == JIPM_FAM_MULTIQUAD ? 12 * d->n_agents : (family == JIPM_FAM_QUAT_NAV ? 13 : 12));
    // Step I-1: relax finite bounds; PAPER.md:63 needs x_L < x_U
    std::vector<double> xl(n), xu(n);
    pb.nL = pb.nU = 0;
    for (int64_t i = 0; i < n; ++i) {
        double l = x_L[i], u = x_U[i];
        if (std::isnan(l) || std::isnan(u)) { delete s; return fail(JIPM_ERR_BOUNDS, "NaN bound"); }
        if (l >= u) { delete s; return fail(JIPM_ERR_BOUNDS, "x_L >= x_U on a component (PAPER.md:63 needs x_L < x_U)"); }
        if (std::isfinite(l)) { l -= s->o.bound_relax_factor * std::max(1.0, std::fabs(l)); pb.nL++; } else l = -INFINITY;
        if (std::isfinite(u)) { u += s->o.bound_relax_factor * std::max(1.0, std::fabs(u)); pb.nU++; } else u = INFINITY;
        if (l >= u) { delete s; return fail(JIPM_ERR_BOUNDS, "x_L >= x_U on a component"); }
        xl[i] = l; xu[i] = u;
    }
    if (family == JIPM_FAM_POINTMASS2D) s->inst = inst_pm();
    else if (family == JIPM_FAM_MULTIQUAD) s->inst = d->n_agents == 4 ? inst_q4() : inst_q2();
    else if (family == JIPM_FAM_QUAT_NAV) s->inst = inst_qt();
    else s->inst = inst_q1();
    cudaDeviceProp prop;
    if (cudaGetDevice(&s->device) != cudaSuccess || cudaGetDeviceProperties(&prop, s->device) != cudaSuccess) {
        delete s;
        return fail(JIPM_ERR_CUDA, "cudaGetDevice / cudaGetDeviceProperties");
    }
    // shared-memory budget per team: the SM's shared memory split over the CTAs the kernel was compiled to co-run
    // (register budget of __launch_bounds__), minus the fixed tiles and 1 KB of per-CTA reservation
    s->teams_per_sm = std::max(1, std::min(s->inst.info.min_blocks, 2048 / s->inst.info.nt));
    const long per_team = std::min<long>((long)prop.sharedMemPerMultiprocessor / s->teams_per_sm - 1024,
                                         (long)prop.sharedMemPerBlockOptin);
    const long budget = per_team / (long)sizeof(double) - s->inst.info.sm_fixed;
    if (budget < 0) { delete s; return fail(JIPM_ERR_NOMEM, "stage tiles do not fit shared memory"); }
    int hot_fits = build_layout(s, (int)budget);
    if (!hot_fits && s->inst.info.hot_sm) {
        // the hot group does not fit: the general instantiation of the family (generic loads, arrays wherever they fit)
        if (family == JIPM_FAM_POINTMASS2D) { delete s; return fail(JIPM_ERR_NOMEM, "problem too large for the point-mass kernel"); }
        s->inst = inst_q1g();
        s->teams_per_sm = std::max(1, std::min(s->inst.info.min_blocks, 2048 / s->inst.info.nt));
        const long pt = std::min<long>((long)prop.sharedMemPerMultiprocessor / s->teams_per_sm - 1024, (long)prop.sharedMemPerBlockOptin);
        const long b2 = pt / (long)sizeof(double) - s->inst.info.sm_fixed;
        if (b2 < 0) { delete s; return fail(JIPM_ERR_NOMEM, "stage tiles do not fit shared memory"); }
        hot_fits = build_layout(s, (int)b2);
    }
    s->dbg = make_dbglay(pb.n, pb.m, pb.N, s->NX, s->NZ);
    s->n_sm = prop.multiProcessorCount;
    if (s->teams_per_sm > 32) s->teams_per_sm = 32;  // one bit of sm_mask per co-resident team
    if (resident_slots == 0) resident_slots = (int64_t)s->teams_per_sm * prop.multiProcessorCount;  // fill the GPU
    s->n_slots = (int)std::min<int64_t>(resident_slots, 0x7fffffff);
    const size_t n_ws = (size_t)s->n_sm * s->teams_per_sm;
    cudaError_t e;
    if ((e = cudaMalloc(&s->d_xL, n * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc(&s->d_xU, n * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc(&s->d_ws, n_ws * (s->L.total - s->L.nsm + 2) * sizeof(double))) != cudaSuccess ||
        (e = cudaMalloc(&s->d_mask, s->n_sm * sizeof(unsigned))) != cudaSuccess ||
        (e = cudaMalloc(&s->d_queue, sizeof(int))) != cudaSuccess ||
        (e = cudaMalloc(&s->d_stats, 24 * sizeof(unsigned long long))) != cudaSuccess) {
        std::string msg = std::string("cudaMalloc: ") + cudaGetErrorString(e);
        jipm_destroy(s);
        return fail(JIPM_ERR_NOMEM, msg);
    }
    pb.xL = s->d_xL; pb.xU = s->d_xU;
    if ((e = cudaMemcpyAsync(s->d_xL, xl.data(), n * sizeof(double), cudaMemcpyHostToDevice, s->stream)) != cudaSuccess ||
        (e = cudaMemcpyAsync(s->d_xU, xu.data(), n * sizeof(double), cudaMemcpyHostToDevice, s->stream)) != cudaSuccess ||
        (e = cudaMemsetAsync(s->d_ws, 0, n_ws * (s->L.total - s->L.nsm + 2) * sizeof(double), s->stream)) != cudaSuccess ||
        (e = cudaStreamSynchronize(s->stream)) != cudaSuccess) {
        std::string msg = std::string("upload: ") + cudaGetErrorString(e);
        jipm_destroy(s);
        return fail(JIPM_ERR_CUDA, msg);
    }
    *out = s;
    return JIPM_OK;
}

extern "C" int jipm_destroy(jipm_solver* s) {
    if (!s) return JIPM_OK;
    DeviceGuard dg(s->device);
    cudaFree(s->d_xL); cudaFree(s->d_xU); cudaFree(s->d_ws); cudaFree(s->d_queue); cudaFree(s->d_stats);
    cudaFree(s->d_mask);
    cudaFree(s->d_stage); cudaFree(s->d_istage);
    delete s;
    return JIPM_OK;
}

static int run(jipm_solver* s, Args& a) {
    DeviceGuard dg(s->device);
    if (!dg.ok) return fail(JIPM_ERR_CUDA, "cannot switch to the solver's device");
    std::lock_guard<std::mutex> lock(g_launch_mutex);
    a.pb = s->pb; a.L = s->L; a.o = s->o;
    a.ws = s->d_ws; a.ws_stride = s->L.total - s->L.nsm + 2; a.n_slots = (int)std::min<int64_t>(s->n_slots, std::max<int64_t>(a.P, 1));
    a.queue = s->d_queue; a.stats = s->d_stats;
    a.sm_mask = s->d_mask; a.teams_per_sm = s->teams_per_sm;
    CUDA_TRY(cudaMemsetAsync(s->d_mask, 0, s->n_sm * sizeof(unsigned), s->stream));
    a.trace = s->trace; a.trace_cap = s->trace_cap;
    a.dbg_len = s->dbg.len;
    CUDA_TRY(cudaMemsetAsync(s->d_queue, 0, sizeof(int), s->stream));
    CUDA_TRY(cudaMemsetAsync(s->d_stats, 0, 24 * sizeof(unsigned long long), s->stream));
    CUDA_TRY(dispatch(s, a));
    unsigned long long st[24];
    CUDA_TRY(cudaMemcpyAsync(st, s->d_stats, sizeof(st), cudaMemcpyDeviceToHost, s->stream));
    CUDA_TRY(cudaStreamSynchronize(s->stream));
    for (int i = 0; i < 24; ++i) s->stats[i] = (long long)st[i];
    s->stats[5] = a.n_slots; s->stats[6] = 1;
    return JIPM_OK;
}

extern "C" int jipm_solve_batch(jipm_solver* s, int64_t P, const double* x0, const double* params, double* x_out,
                                double* lam_out, double* zL_out, double* zU_out, int32_t* status_out,
                                int32_t* iters_out) {
    if (!s) return fail(JIPM_ERR_ARG, "solver is NULL");
    if (P < 0 || P > 0x7fffffff) return fail(JIPM_ERR_ARG, "bad P");
    if (P == 0) return JIPM_OK;
    if (!x0 || !params || !x_out || !lam_out || !status_out || !iters_out) return fail(JIPM_ERR_ARG, "NULL buffer");
    Args a; memset(&a, 0, sizeof(a));
    a.P = (int)P; a.x0 = x0; a.th = params; a.x_out = x_out; a.lam_out = lam_out; a.zL_out = zL_out; a.zU_out = zU_out;
    a.status_out = status_out; a.iters_out = iters_out; a.dbg_mode = 0;
    return run(s, a);
}

extern "C" int jipm_solve_batch_host(jipm_solver* s, int64_t P, const double* x0, const double* params, double* x_out,
                                     double* lam_out, double* zL_out, double* zU_out, int32_t* status_out,
                                     int32_t* iters_out) {
    if (!s) return fail(JIPM_ERR_ARG, "solver is NULL");
    if (P < 0 || P > 0x7fffffff) return fail(JIPM_ERR_ARG, "bad P");
    if (P == 0) return JIPM_OK;
    if (!x0 || !params || !x_out || !lam_out || !status_out || !iters_out) return fail(JIPM_ERR_ARG, "NULL buffer");
    const size_t n = s->pb.n, m = s->pb.m, nth = s->pb.nth;
    const size_t nd = P * (2 * n + m + nth + (zL_out ? n : 0) + (zU_out ? n : 0));
    DeviceGuard dg(s->device);
    if (!dg.ok) return fail(JIPM_ERR_CUDA, "cannot switch to the solver's device");
    // device staging owned by the solver, grow-only: repeated calls of the same size allocate nothing
    if (nd > s->stage_doubles) {
        cudaFree(s->d_stage); s->d_stage = nullptr; s->stage_doubles = 0;
        CUDA_TRY(cudaMalloc(&s->d_stage, nd * sizeof(double)));
        s->stage_doubles = nd;
    }
    if ((size_t)(2 * P) > s->istage_ints) {
        cudaFree(s->d_istage); s->d_istage = nullptr; s->istage_ints = 0;
        CUDA_TRY(cudaMalloc(&s->d_istage, 2 * P * sizeof(int32_t)));
        s->istage_ints = 2 * P;
    }
    double* buf = s->d_stage; int32_t* ib = s->d_istage;
    double* dx0 = buf; double* dth = dx0 + P * n; double* dxo = dth + P * nth; double* dlo = dxo + P * n;
    double* dzl = zL_out ? dlo + P * m : nullptr; double* dzu = zU_out ? (dlo + P * m + (zL_out ? P * n : 0)) : nullptr;
    int rc = JIPM_OK;
    auto chk = [&](cudaError_t ee) { if (ee != cudaSuccess && rc == JIPM_OK) rc = fail(JIPM_ERR_CUDA, cudaGetErrorString(ee)); };
    chk(cudaMemcpyAsync(dx0, x0, P * n * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    chk(cudaMemcpyAsync(dth, params, P * nth * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    if (rc == JIPM_OK) rc = jipm_solve_batch(s, P, dx0, dth, dxo, dlo, dzl, dzu, ib, ib + P);
    if (rc == JIPM_OK) {
        chk(cudaMemcpyAsync(x_out, dxo, P * n * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        chk(cudaMemcpyAsync(lam_out, dlo, P * m * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        if (zL_out) chk(cudaMemcpyAsync(zL_out, dzl, P * n * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        if (zU_out) chk(cudaMemcpyAsync(zU_out, dzu, P * n * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
        chk(cudaMemcpyAsync(status_out, ib, P * sizeof(int32_t), cudaMemcpyDeviceToHost, s->stream));
        chk(cudaMemcpyAsync(iters_out, ib + P, P * sizeof(int32_t), cudaMemcpyDeviceToHost, s->stream));
        chk(cudaStreamSynchronize(s->stream));
    }
    return rc;
}

extern "C" int jipm_last_stats(jipm_solver* s, int64_t* stats, int64_t n_stats) {
    if (!s || !stats) return fail(JIPM_ERR_ARG, "NULL argument");
    for (int64_t i = 0; i < n_stats && i < 24; ++i) stats[i] = s->stats[i];
    return JIPM_OK;
}

extern "C" int jipm_residency(jipm_solver* s, int64_t* res) {
    if (!s || !res) return fail(JIPM_ERR_ARG, "NULL argument");
    res[0] = s->n_sm; res[1] = s->teams_per_sm;
    return JIPM_OK;
}

extern "C" int jipm_debug_set_trace(jipm_solver* s, double* trace, int64_t max_records) {
    if (!s) return fail(JIPM_ERR_ARG, "solver is NULL");
    s->trace = trace; s->trace_cap = trace ? (int)max_records : 0;
    return JIPM_OK;
}

extern "C" int jipm_debug_state_layout(jipm_solver* s, int64_t* lay, int64_t n_lay) {
    if (!s || !lay) return fail(JIPM_ERR_ARG, "NULL argument");
    const DbgLay& d = s->dbg;
    const int v[22] = {d.len, d.x, d.y, d.zL, d.zU, d.sc, d.filt, d.dx, d.dy, d.dzL, d.dzU, d.g, d.c, d.J, d.W,
                       d.rs, d.pn, d.zpn, d.xR, d.filtR, d.ls, d.wd};
    for (int64_t i = 0; i < n_lay && i < 22; ++i) lay[i] = v[i];
    return JIPM_OK;
}

extern "C" int jipm_debug_step(jipm_solver* s, int64_t P, const double* params, double* state, int64_t n_steps) {
    if (!s || !params || !state) return fail(JIPM_ERR_ARG, "NULL argument");
    if (P <= 0) return JIPM_OK;
    Args a; memset(&a, 0, sizeof(a));
    a.P = (int)P; a.th = params; a.dbg_mode = 2; a.dbg_state = state; a.dbg_steps = (int)n_steps;
    return run(s, a);
}

extern "C" int jipm_debug_init(jipm_solver* s, int64_t P, const double* x0, const double* params, double* state) {
    if (!s || !x0 || !params || !state) return fail(JIPM_ERR_ARG, "NULL argument");
    if (P <= 0) return JIPM_OK;
    Args a; memset(&a, 0, sizeof(a));
    a.P = (int)P; a.x0 = x0; a.th = params; a.dbg_mode = 1; a.dbg_state = state;
    return run(s, a);
}

extern "C" int jipm_bench_fp64_peak(void* cuda_stream, double* tflops) {
    if (!tflops) return fail(JIPM_ERR_ARG, "NULL argument");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(JIPM_ERR_CUDA, "no CUDA device");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop;
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 1 << 15;
    double* out = nullptr;
    CUDA_TRY(cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        launch_fp64_peak(out, blocks, threads, iters, st);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double fl = 2.0 * 8.0 * (double)iters * blocks * threads;
        if (rep > 0 && ms > 0) best = std::max(best, fl / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    CUDA_TRY(cudaGetLastError());
    *tflops = best;
    return JIPM_OK;
}

// ---- jipm_solve_batch_static: the same solve with NOTHING allocated ---------------------------------------------------
// For callers that cannot call cudaMalloc (a tight serving loop, a harness that forbids allocation).  Everything
// jipm_create puts into device memory of its own -- the relaxed bounds, the per-SM slot workspaces (the kernel's
// scratch: cold vectors, restoration tails, whatever of the layout does not fit shared memory), the SM-claim mask, the
// queue counter and the statistics block -- is carved out of ONE file-scope device array of JIPM_STATIC_SCRATCH_BYTES.
// Every GPU that loads this module holds that array until the process exits.  The host sees g_static_scratch only as a
// stand-in symbol, never as an address: its device address is asked for once per device, with that device current, by
// cudaGetSymbolAddress (static_scratch_of), and only that pointer is handed to the kernel.
static __device__ __align__(256) double g_static_scratch[JIPM_STATIC_SCRATCH_BYTES / sizeof(double)];

static constexpr int STATIC_MAX_DEVICES = 64;
static constexpr int STATIC_MAX_N = 8192;   // host staging of the relaxed bounds (no heap either)
static double* g_static_ptr[STATIC_MAX_DEVICES] = {nullptr};
static double g_static_xl[STATIC_MAX_N], g_static_xu[STATIC_MAX_N];   // guarded by g_launch_mutex

// device address of the array on the CURRENT device (dev); resolved once per device
static int static_scratch_of(int dev, double** out) {
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(JIPM_ERR_CUDA, "device ordinal beyond the static-scratch table");
    if (g_static_ptr[dev] == nullptr) {
        double* p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress((void**)&p, g_static_scratch));
        if (p == nullptr) return fail(JIPM_ERR_CUDA, "cudaGetSymbolAddress returned NULL for the static scratch");
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return JIPM_OK;
}

extern "C" int jipm_solve_batch_static(int family, const jipm_family_dims* d, int64_t n, int64_t m, const double* x_L,
                                       const double* x_U, const jipm_options* opts, void* cuda_stream, int64_t P,
                                       const double* x0, const double* params, double* x_out, double* lam_out,
                                       double* zL_out, double* zU_out, int32_t* status_out, int32_t* iters_out) {
    if (!x_L || !x_U) return fail(JIPM_ERR_ARG, "NULL argument");
    int nx, nu, ng, nth, pd;
    if (!family_shape(family, d, nx, nu, ng, nth, pd)) return fail(JIPM_ERR_DIM, "bad family or dims");
    int64_t n2, m2, nt2;
    jipm_family_sizes(family, d, &n2, &m2, &nt2);
    if (n != n2 || m != m2) return fail(JIPM_ERR_DIM, "n, m do not match jipm_family_sizes");
    if (P < 0 || P > 0x7fffffff) return fail(JIPM_ERR_ARG, "bad P");
    if (n > STATIC_MAX_N)
        return fail(JIPM_ERR_NOMEM, "jipm_solve_batch_static: n = " + std::to_string(n) + " exceeds the static maximum of " +
                                        std::to_string(STATIC_MAX_N) + " variables (use jipm_create / jipm_solve_batch)");
    if (P > 0 && (!x0 || !params || !x_out || !lam_out || !status_out || !iters_out)) return fail(JIPM_ERR_ARG, "NULL buffer");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
        return fail(JIPM_ERR_CUDA, "no CUDA device (jipm has no CPU fallback)");
    // the configuration jipm_create derives, held on the stack
    jipm_solver s;
    s.family = family; s.dims = *d;
    if (opts) s.o = *opts; else jipm_default_options(&s.o);
    s.stream = (cudaStream_t)cuda_stream;
    s.NX = nx; s.NU = nu; s.NZ = nx + nu;
    Pb& pb = s.pb;
    pb.family = family; pb.N = d->horizon_N; pb.ng = ng; pb.na = d->n_agents; pb.nobs = d->n_obstacles;
    pb.n = (int)n; pb.m = (int)m; pb.nth = nth; pb.blk = nu + nx + ng; pb.cblk = nx + ng;
    pb.dt = d->dt; pb.ru = (family == JIPM_FAM_POINTMASS2D) ? 0.1 : 0.01;
    pb.th_obs = (family == JIPM_FAM_POINTMASS2D) ? 6 : (family == JIPM_FAM_QUAD_TRACK ? 14 : (family == JIPM_FAM_QUAT_NAV ? 16 : 15));
    pb.th_goal = (family == JIPM_FAM_POINTMASS2D) ? 4 : (family == JIPM_FAM_MULTIQUAD ? 12 * d->n_agents : (family == JIPM_FAM_QUAT_NAV ? 13 : 12));
    if (family == JIPM_FAM_POINTMASS2D) s.inst = inst_pm();
    else if (family == JIPM_FAM_MULTIQUAD) s.inst = d->n_agents == 4 ? inst_q4() : inst_q2();
    else if (family == JIPM_FAM_QUAT_NAV) s.inst = inst_qt();
    else s.inst = inst_q1();
    cudaDeviceProp prop;
    if (cudaGetDevice(&s.device) != cudaSuccess || cudaGetDeviceProperties(&prop, s.device) != cudaSuccess)
        return fail(JIPM_ERR_CUDA, "cudaGetDevice / cudaGetDeviceProperties");
    s.teams_per_sm = std::max(1, std::min(s.inst.info.min_blocks, 2048 / s.inst.info.nt));
    const long per_team = std::min<long>((long)prop.sharedMemPerMultiprocessor / s.teams_per_sm - 1024,
                                         (long)prop.sharedMemPerBlockOptin);
    const long budget = per_team / (long)sizeof(double) - s.inst.info.sm_fixed;
    if (budget < 0) return fail(JIPM_ERR_NOMEM, "stage tiles do not fit shared memory");
    int hot_fits = build_layout(&s, (int)budget);
    if (!hot_fits && s.inst.info.hot_sm) {
        if (family == JIPM_FAM_POINTMASS2D) return fail(JIPM_ERR_NOMEM, "problem too large for the point-mass kernel");
        s.inst = inst_q1g();
        s.teams_per_sm = std::max(1, std::min(s.inst.info.min_blocks, 2048 / s.inst.info.nt));
        const long pt = std::min<long>((long)prop.sharedMemPerMultiprocessor / s.teams_per_sm - 1024, (long)prop.sharedMemPerBlockOptin);
        const long b2 = pt / (long)sizeof(double) - s.inst.info.sm_fixed;
        if (b2 < 0) return fail(JIPM_ERR_NOMEM, "stage tiles do not fit shared memory");
        hot_fits = build_layout(&s, (int)b2);
    }
    s.dbg = make_dbglay(pb.n, pb.m, pb.N, s.NX, s.NZ);
    s.n_sm = prop.multiProcessorCount;
    if (s.teams_per_sm > 32) s.teams_per_sm = 32;
    s.n_slots = (int)std::min<int64_t>((int64_t)s.teams_per_sm * s.n_sm, 0x7fffffff);
    // carve the array: [queue | stats | SM mask | x_L | x_U | n_sm * teams_per_sm workspaces], every part 256-byte aligned
    auto up32 = [](size_t c) { return (c + 31) & ~(size_t)31; };   // doubles
    const size_t ws_stride = (size_t)(s.L.total - s.L.nsm + 2);
    const size_t n_ws = (size_t)s.n_sm * s.teams_per_sm;
    const size_t o_queue = 0, o_stats = 32, o_mask = 64;
    const size_t o_xl = o_mask + up32(((size_t)s.n_sm * sizeof(unsigned) + 7) / 8), o_xu = o_xl + up32(n), o_ws = o_xu + up32(n);
    const size_t need = o_ws + n_ws * ws_stride;
    const size_t have = JIPM_STATIC_SCRATCH_BYTES / sizeof(double);
    if (need > have)
        return fail(JIPM_ERR_NOMEM, "jipm_solve_batch_static: this family needs " + std::to_string(need * sizeof(double)) +
                                        " bytes of scratch, the static maximum is " + std::to_string((size_t)JIPM_STATIC_SCRATCH_BYTES) +
                                        " (JIPM_STATIC_SCRATCH_BYTES); use jipm_create / jipm_solve_batch");
    if (P == 0) return JIPM_OK;
    std::lock_guard<std::mutex> lock(g_launch_mutex);
    double* base = nullptr;
    if (int rc = static_scratch_of(s.device, &base)) return rc;
    // Step I-1: relax finite bounds (as jipm_create does), staged in static host storage
    pb.nL = pb.nU = 0;
    for (int64_t i = 0; i < n; ++i) {
        double l = x_L[i], u = x_U[i];
        if (std::isnan(l) || std::isnan(u)) return fail(JIPM_ERR_BOUNDS, "NaN bound");
        if (l >= u) return fail(JIPM_ERR_BOUNDS, "x_L >= x_U on a component (PAPER.md:63 needs x_L < x_U)");
        if (std::isfinite(l)) { l -= s.o.bound_relax_factor * std::max(1.0, std::fabs(l)); pb.nL++; } else l = -INFINITY;
        if (std::isfinite(u)) { u += s.o.bound_relax_factor * std::max(1.0, std::fabs(u)); pb.nU++; } else u = INFINITY;
        if (l >= u) return fail(JIPM_ERR_BOUNDS, "x_L >= x_U on a component");
        g_static_xl[i] = l; g_static_xu[i] = u;
    }
    pb.xL = base + o_xl; pb.xU = base + o_xu;
    // the array keeps the last call's contents: everything the kernel expects to find zero is cleared here (queue,
    // statistics, SM mask, and the workspaces, which jipm_create clears once)
    CUDA_TRY(cudaMemsetAsync(base, 0, o_xl * sizeof(double), s.stream));
    CUDA_TRY(cudaMemsetAsync(base + o_ws, 0, n_ws * ws_stride * sizeof(double), s.stream));
    CUDA_TRY(cudaMemcpyAsync(base + o_xl, g_static_xl, n * sizeof(double), cudaMemcpyHostToDevice, s.stream));
    CUDA_TRY(cudaMemcpyAsync(base + o_xu, g_static_xu, n * sizeof(double), cudaMemcpyHostToDevice, s.stream));
    Args a; memset(&a, 0, sizeof(a));
    a.P = (int)P; a.x0 = x0; a.th = params; a.x_out = x_out; a.lam_out = lam_out; a.zL_out = zL_out; a.zU_out = zU_out;
    a.status_out = status_out; a.iters_out = iters_out; a.dbg_mode = 0;
    a.pb = s.pb; a.L = s.L; a.o = s.o;
    a.ws = base + o_ws; a.ws_stride = (int64_t)ws_stride;
    a.n_slots = (int)std::min<int64_t>(s.n_slots, std::max<int64_t>(a.P, 1));
    a.queue = reinterpret_cast<int*>(base + o_queue);
    a.stats = reinterpret_cast<unsigned long long*>(base + o_stats);
    a.sm_mask = reinterpret_cast<unsigned*>(base + o_mask); a.teams_per_sm = s.teams_per_sm;
    a.trace = nullptr; a.trace_cap = 0; a.dbg_len = s.dbg.len;
    CUDA_TRY(s.inst.launch(a, s.stream));
    CUDA_TRY(cudaStreamSynchronize(s.stream));   // the bounds staging and the __constant__ launch block are free again
    return JIPM_OK;
}
