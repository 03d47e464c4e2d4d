// common.cuh -- shared structs and warp helpers of the jipm CUDA path (sm_100a, fp64).
//
// Execution model: ONE TEAM OF NT THREADS OWNS ONE PROBLEM SLOT.  A team runs the whole
// interior-point iteration of PAPER.md:77-150 for its problem, synchronising only inside the team (warp sync or
// a named barrier), and pops the next problem id from a global queue when its problem reaches a final status
// (iteration-level batching).  All decisions are team-uniform predicates.
#pragma once
#include <cstdint>
#include <cmath>
#include <cuda_runtime.h>
#include "../../include/jipm.h"

namespace jipm {

constexpr unsigned FULL = 0xffffffffu;
constexpr int MAX_FILTER = 256;
constexpr double EPS_MACH = 2.220446049250313e-16;

// problem description, passed by value to the kernel
struct Pb {
    int family, N, ng, na, nobs;
    int n, m, nth;
    int blk, cblk;       // nu+nx+ng, nx+ng
    int nL, nU;          // number of finite lower / upper bounds
    int th_obs, th_goal; // offsets inside theta
    double dt, ru;
    const double* xL;    // DEVICE [n], relaxed, -inf = none
    const double* xU;    // DEVICE [n], relaxed, +inf = none
};

// offsets (in doubles) into the per-slot workspace
struct Lay {
    int x, y, zL, zU, g, c, gv, dgv, cnd, tgt, J, W, Sig, Hd, Dc, T, Kf, Gf, Psi, pv, qv, sv, wv, tv, bl, bu, imap, cmap;
    int b1, b2, b3, b4, dx, dy, dzL, dzU, r1, r2, r3, r4, e1, e2, e3, e4;
    int sx, sy, szL, szU, xt, ct, csoc, bs2, rr, rk, filt, total;
    int pv0, npad, tail0, tpad;  // primal-sized vectors: contiguous block of npad-strided heads, 2m-tails (restoration) apart
    int nsm;  // the first nsm doubles of the layout are shared-memory resident (per team), the rest global
    int xR, DR2, filtR, rc2;  // restoration mode: reference point, scaling D_R^2, its own filter, condensed rhs
    // watchdog (Table I row 3): entry iterate and its search direction
    int wx, wzL, wzU, wdx, wdzL, wdzU, wy, wdy;
    int ab1, ab3, ab4;   // right-hand side of the affine-scaling step (adaptive barrier parameter, Table I row 7)
};

// per-launch arguments
struct Args {
    Pb pb;
    Lay L;
    jipm_options o;
    double* ws;          // [slots * L.total]
    int64_t ws_stride;
    int n_slots;
    int P;
    const double* x0;    // [P x n]
    const double* th;    // [P x nth]
    double* x_out; double* lam_out; double* zL_out; double* zU_out;
    int32_t* status_out; int32_t* iters_out;
    int* queue;          // [1] next problem id
    // R CTAs may be launched but only teams_per_sm per SM are ever co-resident (the shared memory a CTA asks for is the
    // SM's divided by teams_per_sm): the global scratch holds n_sm * teams_per_sm workspaces and a CTA claims one of its
    // SM's workspaces when it starts (a bit of sm_mask[%smid]) and releases it when it ends.
    unsigned* sm_mask;   // [n_sm], zero at launch
    int teams_per_sm;
    unsigned long long* stats; // [16]
    double* trace; int trace_cap;
    // debug
    int dbg_mode;        // 0 solve, 1 init only, 2 load state + step
    double* dbg_state; int dbg_len; int dbg_steps;
};

// debug state layout (doubles) -- mirrored by jipm_debug_state_layout
struct DbgLay { int len, x, y, zL, zU, sc, filt, dx, dy, dzL, dzU, g, c, J, W, rs, pn, zpn, xR, filtR, ls, wd; };

constexpr int RKW = 42;  // doubles of quadrotor phase-1 output per (stage, RK point); see dyn.cuh

__host__ __device__ inline DbgLay make_dbglay(int n, int m, int N, int NX, int NZ) {
    DbgLay d;
    int o = 0;
    d.x = o; o += n; d.y = o; o += m; d.zL = o; o += n; d.zU = o; o += n;
    d.sc = o; o += 8; d.filt = o; o += 2 * MAX_FILTER;
    d.dx = o; o += n; d.dy = o; o += m; d.dzL = o; o += n; d.dzU = o; o += n;
    d.g = o; o += n; d.c = o; o += m;
    d.J = o; o += N * NX * NZ; d.W = o; o += N * NZ * NZ + NX * NX;
    // restoration mode (Step R): scalars, (p, n), (z_p, z_n), reference point x_R, the restoration filter
    d.rs = o; o += 16; d.pn = o; o += 2 * m; d.zpn = o; o += 2 * m; d.xR = o; o += n; d.filtR = o; o += 2 * MAX_FILTER;
    // line-search memory (Table I rows 3-5, 7): 24 scalars; the watchdog's entry iterate and direction: six vectors of
    // n + 2m (x, zL, zU, dx, dzL, dzU), then y, dy
    d.ls = o; o += 24; d.wd = o; o += 6 * (n + 2 * m) + 2 * m;
    d.len = o;
    return d;
}

#ifdef __CUDACC__
// Launch arguments live in constant memory (one copy per translation unit / family instantiation, uploaded by the
// launcher on the solver's stream): every pb->, L->, o->, A-> below compiles to a c[3][offset] operand instead of a
// load through a pointer to the kernel parameters.
static __constant__ Args g_A;
extern __shared__ double jipm_smem[];  // the CTA's dynamic shared memory: fixed tiles, then the hot part of the layout
struct PbProxy { __device__ __forceinline__ const Pb* operator->() const { return &g_A.pb; } };
struct LayProxy { __device__ __forceinline__ const Lay* operator->() const { return &g_A.L; } };
struct OptProxy { __device__ __forceinline__ const jipm_options* operator->() const { return &g_A.o; } };
struct ArgsProxy { __device__ __forceinline__ const Args* operator->() const { return &g_A; } };

// A primal-sized vector: entries [0, n) at a (shared memory or scratch), the restoration tail [n, n + 2m) -- the
// p and n variables of Step R -- in the global scratch at t (pre-shifted by -n so that t[i] is entry i).
struct Vec {
    double* a; double* t; int n;
    __device__ __forceinline__ double& operator[](int i) const { return i < n ? a[i] : t[i]; }
    __device__ __forceinline__ operator double*() const { return a; }  // the head: what the base problem's code sees
};

// A TEAM of NT threads (NT = 32, 64, 128 or 256; whole warps) owns one problem slot.  All decisions of the
// interior-point iteration are team-uniform predicates: every thread of the team holds the same scalar state,
// obtained from the reductions below, which return bit-identical values to every thread.
template <int NT>
struct Team {
    static constexpr int NW = NT / 32;
    int tid;      // 0 .. NT-1
    int flip;     // which half of the reduction scratch the next reduction uses
    double* red;  // shared memory, 2 * NW doubles

    __device__ __forceinline__ void sync() const {
        if constexpr (NT == 32) __syncwarp();
        else __syncthreads();  // one team per CTA
    }
    template <class Op>
    __device__ __forceinline__ double reduce(double v, Op op) {
#pragma unroll
        for (int o = 16; o; o >>= 1) v = op(v, __shfl_xor_sync(FULL, v, o));
        if constexpr (NT == 32) return v;
        double* r = red + flip * NW;
        if ((tid & 31) == 0) r[tid >> 5] = v;
        sync();
        double a = r[0];
#pragma unroll
        for (int w = 1; w < NW; ++w) a = op(a, r[w]);
        flip ^= 1;  // the next reduction writes the other half: one barrier per reduction is enough
        return a;
    }
    __device__ __forceinline__ double sum(double v) { return reduce(v, [](double a, double b) { return a + b; }); }
    __device__ __forceinline__ double max(double v) { return reduce(v, [](double a, double b) { return fmax(a, b); }); }
    __device__ __forceinline__ double min(double v) { return reduce(v, [](double a, double b) { return fmin(a, b); }); }
    __device__ __forceinline__ int any(int v) { return reduce(v ? 1.0 : 0.0, [](double a, double b) { return fmax(a, b); }) > 0.0; }
    // broadcast an int from thread 0
    __device__ __forceinline__ int bcast0(int v) { return (int)reduce(tid == 0 ? (double)v : -1.0e300, [](double a, double b) { return fmax(a, b); }); }
};
#endif

}  // namespace jipm
