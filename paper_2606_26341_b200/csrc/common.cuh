// common.cuh -- shared structs and warp helpers of the jipm CUDA path (sm_100a, fp64).
//
// Execution model: ONE WARP OWNS ONE PROBLEM SLOT.  A warp runs the whole
// interior-point iteration of PAPER.md:77-150 for its problem, synchronising only with __syncwarp(), and
// pops the next problem id from a global queue when its problem reaches a final status (iteration-level
// batching).  All decisions are warp-uniform predicates.
#pragma once
#include <cstdint>
#include <cmath>
#include <cuda_runtime.h>
#include "../../include/jipm.h"

namespace jipm {

constexpr unsigned FULL = 0xffffffffu;
constexpr int MAX_FILTER = 128;
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

// offsets (in doubles) into the per-warp workspace
struct Lay {
    int x, y, zL, zU, g, c, gv, tgt, J, W, Sig, Hd, Dc, T, Xf, Lf, wv, tv;
    int b1, b2, b3, b4, dx, dy, dzL, dzU, r1, r2, r3, r4, e1, e2, e3, e4;
    int sx, sy, szL, szU, xt, ct, csoc, bs2, rr, rk, filt, total;
    int xR, DR2, filtR, rc2;  // restoration mode: reference point, scaling D_R^2, its own filter, condensed rhs
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
    unsigned long long* stats; // [8]
    double* trace; int trace_cap;
    // debug
    int dbg_mode;        // 0 solve, 1 init only, 2 load state + step
    double* dbg_state; int dbg_len; int dbg_steps;
};

// debug state layout (doubles) -- mirrored by jipm_debug_state_layout
struct DbgLay { int len, x, y, zL, zU, sc, filt, dx, dy, dzL, dzU, g, c, J, W; };

constexpr int RKW = 42;  // doubles of quadrotor phase-1 output per (stage, RK point); see dyn.cuh

__host__ __device__ inline DbgLay make_dbglay(int n, int m, int N, int NX, int NZ) {
    DbgLay d;
    int o = 0;
    d.x = o; o += n; d.y = o; o += m; d.zL = o; o += n; d.zU = o; o += n;
    d.sc = o; o += 8; d.filt = o; o += 2 * MAX_FILTER;
    d.dx = o; o += n; d.dy = o; o += m; d.dzL = o; o += n; d.dzU = o; o += n;
    d.g = o; o += n; d.c = o; o += m;
    d.J = o; o += N * NX * NZ; d.W = o; o += N * NZ * NZ + NX * NX;
    d.len = o;
    return d;
}

#ifdef __CUDACC__
__device__ __forceinline__ double wsum(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
    return v;
}
__device__ __forceinline__ double wmax(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fmax(v, __shfl_xor_sync(FULL, v, o));
    return v;
}
__device__ __forceinline__ double wmin(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fmin(v, __shfl_xor_sync(FULL, v, o));
    return v;
}
__device__ __forceinline__ int wor(int v) { return __any_sync(FULL, v); }
__device__ __forceinline__ bool finite_d(double v) { return isfinite(v); }
#endif

}  // namespace jipm
