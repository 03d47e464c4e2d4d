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
//
// What the factor stores per stage k (so that a solve is two sweeps of ONE nx-by-nx product per stage plus
// stage-parallel work):
//   T_k   = (I + P_k D_k)^{-1} P_k                       nx x nx, k = 0..N
//   Kf_k  = Rt_k^{-1} M_ux            (feedback)         nu x nx
//   G_k   = Rt_k^{-1}                                    nu x nu
//   Psi_k = (I - D_{k+1} T_{k+1}) (A_k - B_k Kf_k)       nx x nx   (closed-loop transition)
// All loops are element-parallel over the team (thread <-> tile element), one barrier per dependent phase.
#pragma once
#include "core.cuh"

#ifndef JIPM_USE_DMMA
#define JIPM_USE_DMMA 1   // FP64 tensor-core path of the multi-agent stage products (measured: DESIGN.md section 6)
#endif

namespace jipm {

template <class C>
struct Kkt {
    static constexpr int NX = C::NX, NU = C::NU, NZ = C::NZ, PD = C::PD, AX = C::AX, AU = C::AU, NA = C::NA, NT = C::NT, LDJ = C::LDJ;
    static constexpr bool USE_DMMA = JIPM_USE_DMMA != 0;
    using X = Ctx<C>;
    // J_k = [A B] is block diagonal over the agents (AX x (AX | AU) blocks): every product with J runs over one
    // agent's rows / columns only.  agent of column j of z = (x, u):
    __device__ static __forceinline__ int col_agent(int j) {
        if constexpr (NA == 1) return 0;
        else return j < NX ? j / AX : (j - NX) / AU;
    }
    __device__ static __forceinline__ int row_agent(int i) {
        if constexpr (NA == 1) return 0;
        else return i / AX;
    }
    __device__ static __forceinline__ int ctl_agent(int p) {
        if constexpr (NA == 1) return 0;
        else return p / AU;
    }

    // Tile loop with a compile-time trip count: thread `lane` visits the elements lane, lane + NT, ... of an NE-element
    // tile.  Fully unrolled, so that the independent dependent-chains of a thread's elements interleave (a team of 128
    // or 64 threads owns 2 - 4 elements of a 16 x 16 tile; run one after the other they would double the phase's latency).
    template <int NE, class F>
    __device__ static __forceinline__ void tile_for(int lane, F f) {
#pragma unroll
        for (int r = 0; r < (NE + NT - 1) / NT; ++r) {
            const int e = lane + r * NT;
            if (NE % NT == 0 || e < NE) f(e);
        }
    }

    // FP64 tensor-core MMA (sm_80+ "DMMA", legacy warp-level path: tcgen05 has no f64 kind): D(8x8) += A(8x4) B(4x8).
    // Lane l holds A[l/4][l%4], B[l%4][l/4] and D[l/4][2(l%4)], D[l/4][2(l%4)+1].  Used only for the multi-agent
    // family, whose stage products are 48 x 12 x 16 / 16 x 12 x 64 contractions per agent.
    __device__ static __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
    }
    // index in z = (x, u) of entry c (0 .. AX+AU-1) of agent a's own (x_a, u_a)
    __device__ static __forceinline__ int zmap(int a, int c) { return c < AX ? AX * a + c : NX + AU * a + (c - AX); }

    // dot product with 4 independent partial sums (dependent-chain latency / 4), compile-time length and strides: fully unrolled, immediate offsets
    template <int LEN, int SA, int SB>
    __device__ static __forceinline__ double dotc(const double* a, const double* b) {
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
        for (int l = 0; l + 3 < LEN; l += 4) {
            s0 = fma(a[l * SA], b[l * SB], s0);
            s1 = fma(a[(l + 1) * SA], b[(l + 1) * SB], s1);
            s2 = fma(a[(l + 2) * SA], b[(l + 2) * SB], s2);
            s3 = fma(a[(l + 3) * SA], b[(l + 3) * SB], s3);
        }
#pragma unroll
        for (int l = LEN & ~3; l < LEN; ++l) s0 = fma(a[l * SA], b[l * SB], s0);
        return (s0 + s1) + (s2 + s3);
    }

    // reciprocal of a pivot: hardware approximation (relative error 2^-23) and one cubic Newton step,
    // x0 (1 + e + e^2) with e = 1 - d x0, error e^3 = 2^-69: within one ulp, in 4 dependent instructions instead of
    // the ~12 of the IEEE division (the G reciprocals of a pivot group are a dependent chain on the critical path of
    // every stage).  Pivots lie within 1e-40 .. 1e40 (delta_w_max), far inside the range of the approximation.
    __device__ static __forceinline__ double rcp(double d) {
        double x;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
        const double e = fma(-d, x, 1.0);
        return fma(x, fma(e, e, e), x);
    }

    // G consecutive Gauss-Jordan pivots p0 .. p0+G-1 on the n x n tile src (row stride LD, NE = n * LD elements) in ONE
    // phase: every element of dst is computed from src alone (no races, one barrier per G pivots), by the thread that
    // owns it, with exactly the operations the G sequential pivot steps would apply to it -- bit-identical to the
    // one-pivot-per-barrier form, in particular as stable (forming the inverse of the G x G pivot block explicitly
    // is not: its determinant cancels when the block is dominated by a rank-one term, e.g. Sigma of one active
    // obstacle constraint seen through B).  Per element (a, b) this is Gaussian elimination of the bordered matrix
    //      [ A    B_b  ]      A = src[Pi, Pi],  B_b = src[Pi, b],  C_a = src[a, Pi],  D = src[a, b]
    //      [ C_a  D    ]
    // down to its Schur complement D - C_a A^{-1} B_b; the rows / columns inside Pi use C_a = -e_a^T, B_b = e_b,
    // D = 0, which reproduces the Gauss-Jordan entries (scaled pivot row, negated scaled pivot column, reciprocal
    // pivot) with exact operations.  The elimination of A (pivots, scaled rows, multipliers) is the same for every
    // element and done once per thread; the pivot signs carry the inertia test.  An exactly-zero pivot is counted in
    // nzero and replaced by 1 (the factorisation is rejected anyway).
    template <int G, int LD, int NE>
    __device__ static __forceinline__ void gjk(const X& c, const double* src, double* dst, int p0, int& bad, int& nzero) {
        double A[G][G], id[G];
#pragma unroll
        for (int i = 0; i < G; ++i)
#pragma unroll
            for (int l = 0; l < G; ++l) A[i][l] = src[(p0 + i) * LD + p0 + l];
        // after step i: id[i] = 1 / pivot, A[i][l] (l > i) = scaled pivot row, A[j][i] (j > i) = multiplier
#pragma unroll
        for (int i = 0; i < G; ++i) {
            double d = A[i][i];
            if (!(d > 0.0)) { bad++; if (d == 0.0) { nzero++; d = 1.0; } }
            id[i] = rcp(d);
#pragma unroll
            for (int l = i + 1; l < G; ++l) A[i][l] *= id[i];
#pragma unroll
            for (int j = i + 1; j < G; ++j)
#pragma unroll
                for (int l = i + 1; l < G; ++l) A[j][l] -= A[j][i] * A[i][l];
        }
        tile_for<NE>(c.lane, [&](int e) {
            const int a = e / LD, b = e % LD;
            const int ia = a - p0, ib = b - p0;
            const bool ain = ia >= 0 && ia < G, bin = ib >= 0 && ib < G;
            double Bv[G], Cv[G];
#pragma unroll
            for (int i = 0; i < G; ++i) {
                Bv[i] = bin ? (ib == i ? 1.0 : 0.0) : src[(p0 + i) * LD + b];
                Cv[i] = ain ? (ia == i ? -1.0 : 0.0) : src[a * LD + p0 + i];
            }
            double D = (ain || bin) ? 0.0 : src[e];
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const double rb = Bv[i] * id[i];
#pragma unroll
                for (int j = i + 1; j < G; ++j) Bv[j] -= A[j][i] * rb;
#pragma unroll
                for (int l = i + 1; l < G; ++l) Cv[l] -= Cv[i] * A[i][l];
                D -= Cv[i] * rb;
            }
            dst[e] = D;
        });
    }
    // pivots p0 .. p0+n-1 in groups of four (then two, then one); src / dst are swapped after every phase
    template <int LD, int NE, int NP>
    __device__ static __forceinline__ void gj_range(const X& c, double*& src, double*& dst, int p0, int& bad, int& nzero) {
#pragma unroll 1
        for (int p = 0; p + 4 <= NP; p += 4) {
            gjk<4, LD, NE>(c, src, dst, p0 + p, bad, nzero);
            c.tm.sync();
            double* t = src; src = dst; dst = t;
        }
        if constexpr ((NP & 3) >= 2) {
            gjk<2, LD, NE>(c, src, dst, p0 + (NP & ~3), bad, nzero);
            c.tm.sync();
            double* t = src; src = dst; dst = t;
        }
        if constexpr (NP & 1) {
            gjk<1, LD, NE>(c, src, dst, p0 + NP - 1, bad, nzero);
            c.tm.sync();
            double* t = src; src = dst; dst = t;
        }
    }

    // T = (I + P D)^{-1} P (D != 0): the tile wk (2 NX^2) holds I + P D in its first half
    // (written by the caller, barrier passed).  I + P D = E^{-1} (I + E P E) E with E = sqrt(D): the same leading
    // minors, hence the same unpivoted pivots as the symmetric I + E P E whose inertia the test needs.  Gauss-Jordan
    // inversion ping-pong between the halves of wk, four pivots per barrier (gjk); `first` runs inside the first phase (work
    // of the caller that only needs the same barrier).  Then T = sym(inv P) with both (i,q) and (q,i) products in
    // the same thread (no separate symmetrisation phase); P symmetric at Pm with row stride LDP.  Writes sT and Tg.
    template <int LDP, class F>
    __device__ static __forceinline__ void transform_T(const X& c, double* wk, const double* Pm, double* sT, double* Tg,
                                                       int& bad, int& nzero, F first) {
        double* src = wk;
        double* dst = wk + NX * NX;
        first();
        gj_range<NX, NX * NX, NX>(c, src, dst, 0, bad, nzero);
        tile_for<NX * NX>(c.lane, [&](int e) {
            const int i = e / NX, q = e % NX;
            const double v = 0.5 * (dotc<NX, 1, LDP>(src + i * NX, Pm + q) + dotc<NX, 1, LDP>(src + q * NX, Pm + i));
            sT[e] = v; Tg[e] = v;
        });
        c.tm.sync();
    }

    // Factor.  Reads W, J, Sig, Dc, gv from the workspace; writes T, Kf, Gf, Psi, dgv.  Returns the number of pivots
    // with the wrong sign (0 <=> inertia (n, m, 0)); nzero counts exactly-zero pivots.  any_dc: some Dc entry != 0.
    // Per stage (regular mode, one barrier per item): T J | M = Q + J^T (T J) + condensed slacks | the nu Gauss-Jordan
    // pivots on the control block, four per barrier (gjk), ping-pong between two tiles (afterwards the tile holds P_k,
    // Kf_k, G_k at once) | Phi, stores.  With D != 0: the Phi phase also symmetrises P_k and writes I + P_k D_k, Psi runs
    // inside the first pivot phase of transform_T.
    __device__ static __noinline__ int factor(const X& c, int& nzero, bool any_dc, bool useW) {
        const PbProxy pb;
        const int N = pb->N, lane = c.lane, ng = pb->ng;
        double* sT = c.smt(C::SM_T);     // NX x NX   current T_{k+1} / P_k
        double* sJc = c.smt(C::SM_J);    // NX x LDJ  copy of J_k when J is not shared-memory resident
        double* tA = c.smt(C::SM_M);     // NZ x NZ   stage tile (>= 2 NX^2: scratch of transform_T)
        double* tB = c.smt(C::SM_M2);    // NZ x NZ   second tile of the Gauss-Jordan ping-pong
        double* sTJ = c.smt(C::SM_TJ);   // NX x NZ   T J, later Phi (NX x NX)
        const double* Sig = c.v(c.L->Sig);
        const double* Dc = c.vh(c.L->Dc);
        const double* gvv = c.vh(c.L->gv);
        double* dgv = c.vh(c.L->dgv);
        const bool j_in_sm = c.L->J < c.L->nsm;
        int bad = 0;
        nzero = 0;
        // weights of the condensed (slack, multiplier) pairs and their position-block sums G^T Dg G for every stage,
        // once per factorisation and stage-parallel (the solves reuse the weights)
        constexpr int NPOS = NA * PD;
        double* cnd = c.vh(c.L->cnd);
        for (int it = lane; it < N * ng; it += NT) {
            const int k = it / ng + 1, j = it % ng;
            dgv[it] = 1.0 / (1.0 / Sig[c.is(k) + j] + Dc[c.icg(k) + j]);
        }
        c.tm.sync();
        if (ng > 0) {
            for (int it = lane; it < N * NPOS * NPOS; it += NT) {
                const int k = it / (NPOS * NPOS) + 1, e = it % (NPOS * NPOS), r = e / NPOS, q = e % NPOS;
                cnd[it] = cond_entry(c, gvv, dgv, k, AX * (r / PD) + r % PD, AX * (q / PD) + q % PD);
            }
            c.tm.sync();
        }
        // terminal block: P_N = W_N + Sigma + condensed slacks
        {
            const double* WN = c.Wk(N);
            double* TN = c.vh(c.L->T) + N * NX * NX;
            double* Pn = any_dc ? tB : sT;
            for (int e = lane; e < NX * NX; e += NT) {
                const int r = e / NX, q = e % NX;
                double v = (useW ? WN[e] : 0.0) + (r == q ? Sig[c.ix(N) + r] : 0.0);
                if (ng > 0 && r % AX < PD && q % AX < PD) v += cnd[(N - 1) * NPOS * NPOS + (PD * (r / AX) + r % AX) * NPOS + PD * (q / AX) + q % AX];
                Pn[e] = v;
                if (any_dc) tA[e] = v * Dc[c.icd(N) + q] + (r == q ? 1.0 : 0.0);
                else TN[e] = v;
            }
            c.tm.sync();
            if (any_dc) transform_T<NX>(c, tA, tB, sT, TN, bad, nzero, [] {});
        }
        for (int k = N - 1; k >= 0; --k) {
            long long tq = clock64();
            const double* sJ = c.Jk(k);
            if (!j_in_sm) {
                for (int e = lane; e < NX * LDJ; e += NT) sJc[e] = sJ[e];
                sJ = sJc;
                c.tm.sync();
            }
            // TJ = T_{k+1} J_k
            if constexpr (NA > 1 && USE_DMMA) {
                // per agent a: TJ[:, z_a] = T[:, x_a] (NX x AX) * J_a (AX x (AX+AU)) on the FP64 tensor cores
                constexpr int AZ = AX + AU, MT = NX / 8, NTL = AZ / 8;
                static_assert(AX % 4 == 0 && NX % 8 == 0 && AZ % 8 == 0, "DMMA tiling");
                const int wl = lane & 31, g = wl >> 2, t = wl & 3;
                for (int tile = lane >> 5; tile < NA * MT * NTL; tile += NT / 32) {
                    const int a = tile / (MT * NTL), rem = tile % (MT * NTL), mt = rem / NTL, nt = rem % NTL;
                    double d0 = 0.0, d1 = 0.0;
                    const int cB = zmap(a, 8 * nt + g);
#pragma unroll
                    for (int ks = 0; ks < AX / 4; ++ks)
                        dmma884(d0, d1, sT[(8 * mt + g) * NX + AX * a + 4 * ks + t], sJ[(AX * a + 4 * ks + t) * LDJ + cB]);
                    sTJ[(8 * mt + g) * NZ + zmap(a, 8 * nt + 2 * t)] = d0;
                    sTJ[(8 * mt + g) * NZ + zmap(a, 8 * nt + 2 * t + 1)] = d1;
                }
            } else {
            tile_for<NX * NZ>(lane, [&](int e) {
                const int l = e / NZ, j = e % NZ;
                const int aj = col_agent(j);
                sTJ[e] = dotc<AX, 1, LDJ>(sT + l * NX + AX * aj, sJ + AX * aj * LDJ + j);
            });
            }
            c.tm.sync();
            { const long long t2 = clock64(); c.tick(8, t2 - tq); tq = t2; }
            // M = Q_k + J^T (T J) + condensed slacks
            const double* Wg = c.Wk(k);
            auto m_extra = [&](double m, int a, int j) {  // what M gets besides J^T (T J): W, Sigma, the condensed slacks
                if (useW) m += Wg[a * NZ + j];
                if (a == j) m += Sig[c.zidx(k, j)];
                if (k >= 1 && ng > 0 && a < NX && j < NX && a % AX < PD && j % AX < PD)
                    m += cnd[(k - 1) * NPOS * NPOS + (PD * (a / AX) + a % AX) * NPOS + PD * (j / AX) + j % AX];
                return m;
            };
            if constexpr (NA > 1 && USE_DMMA) {
                // per agent aa: M[z_aa, :] = J_aa^T ((AX+AU) x AX) * TJ[x_aa, :] (AX x NZ)
                constexpr int AZ = AX + AU, MTm = AZ / 8, NTn = NZ / 8;
                const int wl = lane & 31, g = wl >> 2, t = wl & 3;
                for (int tile = lane >> 5; tile < NA * MTm * NTn; tile += NT / 32) {
                    const int aa = tile / (MTm * NTn), rem = tile % (MTm * NTn), mt = rem / NTn, nt = rem % NTn;
                    double d0 = 0.0, d1 = 0.0;
                    const int rA = zmap(aa, 8 * mt + g);
#pragma unroll
                    for (int ks = 0; ks < AX / 4; ++ks)
                        dmma884(d0, d1, sJ[(AX * aa + 4 * ks + t) * LDJ + rA], sTJ[(AX * aa + 4 * ks + t) * NZ + 8 * nt + g]);
                    const int j0 = 8 * nt + 2 * t;
                    tA[rA * NZ + j0] = m_extra(d0, rA, j0);
                    tA[rA * NZ + j0 + 1] = m_extra(d1, rA, j0 + 1);
                }
            } else {
            tile_for<NZ * NZ>(lane, [&](int e) {
                const int a = e / NZ, j = e % NZ;
                const int aa = col_agent(a);
                tA[e] = m_extra(dotc<AX, LDJ, NZ>(sJ + AX * aa * LDJ + a, sTJ + AX * aa * NZ + j), a, j);
            });
            }
            c.tm.sync();
            { const long long t2 = clock64(); c.tick(9, t2 - tq); tq = t2; }
            // Gauss-Jordan pivots on the controls NX .. NZ-1, four per barrier: every element from the previous tile
            double* src = tA; double* dst = tB;
            gj_range<NZ, NZ * NZ, NU>(c, src, dst, NX, bad, nzero);
            { const long long t2 = clock64(); c.tick(10, t2 - tq); tq = t2; }
            // src: [[P_k, -Kf^T], [Kf, G]].  Phi = A - B Kf; stores
            double* Kg = c.vh(c.L->Kf) + k * NU * NX;
            double* Gg = c.vh(c.L->Gf) + k * NU * NU;
            double* Pg = c.vh(c.L->Psi) + k * NX * NX;
            double* Tg = c.vh(c.L->T) + k * NX * NX;
            const int r1 = c.icd(k);
            tile_for<NX * NX>(lane, [&](int e) {
                const int i = e / NX, a = e % NX;
                const int ai = row_agent(i);
                const double phi = sJ[i * LDJ + a] - dotc<AU, 1, NZ>(sJ + i * LDJ + NX + AU * ai, src + (NX + AU * ai) * NZ + a);
                if (any_dc) {
                    sTJ[e] = phi;
                    // P_k symmetrised in place (the thread of (i, a), i <= a, owns both entries) and I + P_k D_k
                    if (i <= a) {
                        const double tn = 0.5 * (src[i * NZ + a] + src[a * NZ + i]);
                        src[i * NZ + a] = tn; src[a * NZ + i] = tn;
                        dst[i * NX + a] = tn * Dc[r1 + a] + (i == a ? 1.0 : 0.0);
                        dst[a * NX + i] = tn * Dc[r1 + i] + (i == a ? 1.0 : 0.0);
                    }
                } else {
                    Pg[e] = phi;
                    const double tn = 0.5 * (src[i * NZ + a] + src[a * NZ + i]);
                    sT[e] = tn; Tg[e] = tn;
                }
            });
            for (int e = lane; e < NU * NX; e += NT) Kg[e] = src[(NX + e / NX) * NZ + e % NX];
            for (int e = lane; e < NU * NU; e += NT) Gg[e] = src[(NX + e / NU) * NZ + NX + e % NU];
            c.tm.sync();
            { const long long t2 = clock64(); c.tick(11, t2 - tq); tq = t2; }
            if (any_dc) {
                // Psi = (I - D_{k+1} T_{k+1}) Phi inside the first pivot phase, then P_k -> T_k = (I + P_k D_k)^{-1} P_k
                const int r0 = c.icd(k + 1);
                transform_T<NZ>(c, dst, src, sT, Tg, bad, nzero, [&] {
                    tile_for<NX * NX>(lane, [&](int e) {
                        const int i = e / NX, a = e % NX;
                        Pg[e] = sTJ[e] - Dc[r0 + i] * dotc<NX, 1, NX>(sT + i * NX, sTJ + a);
                    });
                });
                c.tick(12, clock64() - tq);
            }
        }
        return bad;
    }

    // entry (r, q) of sum_j Dg_j G_j^T G_j of stage k (k >= 1) in the x-block (0 outside the position entries)
    __device__ static __forceinline__ double cond_entry(const X& c, const double* gvv, const double* dgv, int k, int r, int q) {
        const int a = r / AX, i = r % AX, b = q / AX, i2 = q % AX;
        if (i >= PD || i2 >= PD) return 0.0;
        const PbProxy pb;
        const int ng = pb->ng;
        const double* gv = gvv + (k - 1) * ng * PD;
        const double* dg = dgv + (k - 1) * ng;
        double s = 0.0;
        if (pb->family == JIPM_FAM_MULTIQUAD) {
            for (int j = 0; j < ng; ++j) {
                int pa, pb2; c.pair_ab(j, pa, pb2);
                const double sa = (pa == a) ? 1.0 : (pb2 == a ? -1.0 : 0.0);
                const double sb = (pa == b) ? 1.0 : (pb2 == b ? -1.0 : 0.0);
                if (sa != 0.0 && sb != 0.0) s += sa * sb * dg[j] * gv[j * PD + i] * gv[j * PD + i2];
            }
        } else {
            if (a != 0 || b != 0) return 0.0;
            for (int j = 0; j < ng; ++j) s += dg[j] * gv[j * PD + i] * gv[j * PD + i2];
        }
        return s;
    }

    // condensed right-hand side contribution to x_k position entry (agent a, coordinate i), k >= 1:
    //   sum_j G_j^T Dg_j (rc_g,j + rp_s,j / sig_j)
    __device__ static double cond_rhs(const X& c, const double* rp, const double* rc, int k, int a, int i) {
        const PbProxy pb;
        const int ng = pb->ng;
        const double* gv = c.vh(c.L->gv) + (k - 1) * ng * PD;
        const double* dg = c.vh(c.L->dgv) + (k - 1) * ng;
        const double* Sig = c.v(c.L->Sig) + c.is(k);
        double s = 0.0;
        for (int j = 0; j < ng; ++j) {
            double sgn = 1.0;
            if (pb->family == JIPM_FAM_MULTIQUAD) {
                int pa, pb2; c.pair_ab(j, pa, pb2);
                sgn = (pa == a) ? 1.0 : (pb2 == a ? -1.0 : 0.0);
                if (sgn == 0.0) continue;
            }
            s += sgn * gv[j * PD + i] * dg[j] * (rc[c.icg(k) + j] + rp[c.is(k) + j] / Sig[j]);
        }
        return s;
    }

    // Solve with the current factor: [dx; dy] = K^{-1} [rp; rc].
    //   phase 0 (stage-parallel)  cr_k = rp_x,k + condensed rhs;  w_k = T_{k+1} rc_{k+1};
    //                             h_k = rp_u,k - B_k^T w_k;  q_k = cr_k - A_k^T w_k - Kf_k^T h_k
    //   phase 1 (sequential)      p_N = cr_N;  p_k = q_k + Psi_k^T p_{k+1}
    //   phase 2 (stage-parallel)  sw_k = w_k - p_{k+1} + T_{k+1} (D_{k+1} p_{k+1});  uo_k = G_k (rp_u,k - B_k^T sw_k);
    //                             e_k = (I - D T)(B_k uo_k) - D sw_k + rc_{k+1};  x_0 from the initial-condition rows
    //   phase 3 (sequential)      x_{k+1} = Psi_k x_k + e_k
    //   phase 4 (stage-parallel)  u_k = uo_k - Kf_k x_k;  nu_k = sw_k + T_{k+1} (A x_k + B u_k);  dy = -nu;  slacks
    __device__ static __noinline__ void solve(const X& c, const double* rp, const double* rc, double* dx, double* dy,
                                              bool any_dc) {
        const PbProxy pb;
        const int N = pb->N, lane = c.lane;
        const double* Dc = c.vh(c.L->Dc);
        const double* Tf = c.vh(c.L->T);
        const double* Kf = c.vh(c.L->Kf);
        const double* Gf = c.vh(c.L->Gf);
        const double* Psi = c.vh(c.L->Psi);
        double* pv = c.vh(c.L->pv);    // (N+1) x NX : cr_k, then p_k, then x_k
        double* wv = c.vh(c.L->wv);    // N x NX     : w_k, then sw_k
        double* qv = c.vh(c.L->qv);    // N x NX     : q_k, then e_k
        double* hv = c.vh(c.L->tv);    // N x NU     : h_k, then uo_k, then u_k
        double* sv = c.vh(c.L->sv);    // N x NX     : scratch (st_k, B uo_k, A x_k + B u_k)
        // ---- phase 0a ----
#pragma unroll 2
        for (int e = lane; e < (N + 1) * NX; e += NT) {
            const int k = e / NX, i = e % NX;
            double v = rp[c.ix(k) + i];
            const int ag = i / AX, ii = i % AX;
            if (k >= 1 && ii < PD && pb->ng > 0) v += cond_rhs(c, rp, rc, k, ag, ii);
            pv[e] = v;
        }
#pragma unroll 2
        for (int e = lane; e < N * NX; e += NT) {
            const int k = e / NX, i = e % NX;
            wv[e] = dotc<NX, NX, 1>(Tf + (k + 1) * NX * NX + i, rc + c.icd(k + 1));  // T symmetric
        }
        c.tm.sync();
        // ---- phase 0b: h_k ----
#pragma unroll 2
        for (int e = lane; e < N * NU; e += NT) {
            const int k = e / NU, p = e % NU;
            const int ap = ctl_agent(p);
            hv[e] = rp[c.iu(k) + p] - dotc<AX, LDJ, 1>(c.Jk(k) + AX * ap * LDJ + NX + p, wv + k * NX + AX * ap);
        }
        c.tm.sync();
        // ---- phase 0c: q_k ----
#pragma unroll 2
        for (int e = lane; e < N * NX; e += NT) {
            const int k = e / NX, i = e % NX;
            const int ai = row_agent(i);
            qv[e] = pv[e] - dotc<AX, LDJ, 1>(c.Jk(k) + AX * ai * LDJ + i, wv + k * NX + AX * ai) - dotc<NU, NX, 1>(Kf + k * NU * NX + i, hv + k * NU);
        }
        c.tm.sync();
        // ---- phase 1: backward sweep (threads i < NX; whole-team barrier only if NX spans several warps) ----
        for (int k = N - 1; k >= 0; --k) {
            if (lane < NX) pv[k * NX + lane] = qv[k * NX + lane] + dotc<NX, NX, 1>(Psi + k * NX * NX + lane, pv + (k + 1) * NX);
            if (NX <= 32) __syncwarp(); else c.tm.sync();
        }
        c.tm.sync();
        // ---- phase 2 ----
        if (any_dc) {
            for (int e = lane; e < N * NX; e += NT) {
                const int k = e / NX, i = e % NX, r0 = c.icd(k + 1);
                double s = 0.0;
                const double* Tn = Tf + (k + 1) * NX * NX;
                for (int l = 0; l < NX; ++l) s += Tn[l * NX + i] * (Dc[r0 + l] * pv[(k + 1) * NX + l]);
                wv[e] += s - pv[(k + 1) * NX + i];
            }
        } else {
            for (int e = lane; e < N * NX; e += NT) wv[e] -= pv[e + NX];
        }
        c.tm.sync();
#pragma unroll 2
        for (int e = lane; e < N * NU; e += NT) {
            const int k = e / NU, p = e % NU;
            const int ap = ctl_agent(p);
            sv[e] = rp[c.iu(k) + p] - dotc<AX, LDJ, 1>(c.Jk(k) + AX * ap * LDJ + NX + p, wv + k * NX + AX * ap);  // st_k
        }
        c.tm.sync();
#pragma unroll 2
        for (int e = lane; e < N * NU; e += NT) {
            const int k = e / NU, p = e % NU;
            hv[e] = dotc<NU, 1, 1>(Gf + k * NU * NU + p * NU, sv + k * NU);  // uo_k = G st_k
        }
        c.tm.sync();
#pragma unroll 2
        for (int e = lane; e < N * NX; e += NT) {
            const int k = e / NX, i = e % NX;
            const int ai = row_agent(i);
            sv[e] = dotc<AU, 1, 1>(c.Jk(k) + i * LDJ + NX + AU * ai, hv + k * NU + AU * ai);  // B uo_k   (st_k is dead)
        }
        c.tm.sync();
#pragma unroll 2
        for (int e = lane; e < N * NX; e += NT) {
            const int k = e / NX, i = e % NX, r0 = c.icd(k + 1);
            double v = sv[e] + rc[r0 + i];
            if (any_dc) v -= Dc[r0 + i] * (dotc<NX, NX, 1>(Tf + (k + 1) * NX * NX + i, sv + k * NX) + wv[e]);
            qv[e] = v;  // e_k
        }
        // stage 0: nu_0 = T_0 (rc_0 + D_0 p_0) - p_0, x_0 = rc_0 - D_0 nu_0
        double x0 = 0.0;
        if (lane < NX) {
            double s = -pv[lane];
            for (int l = 0; l < NX; ++l) s += Tf[l * NX + lane] * (rc[l] + Dc[l] * pv[l]);
            x0 = rc[lane] - Dc[lane] * s;
            dx[lane] = x0; dy[lane] = -s;
        }
        c.tm.sync();
        // ---- phase 3: forward sweep, x_k kept in pv (p_k is dead once sw_k, x_0 are formed) ----
        if (lane < NX) pv[lane] = x0;
        if (NX <= 32) __syncwarp(); else c.tm.sync();
        for (int k = 0; k < N; ++k) {
            if (lane < NX) {
                const double xn = qv[k * NX + lane] + dotc<NX, 1, 1>(Psi + k * NX * NX + lane * NX, pv + k * NX);
                pv[(k + 1) * NX + lane] = xn;
            }
            if (NX <= 32) __syncwarp(); else c.tm.sync();
        }
        c.tm.sync();
        // ---- phase 4 ----
        for (int e = lane; e < N * NX; e += NT) dx[c.ix(e / NX + 1) + e % NX] = pv[e + NX];
#pragma unroll 2
        for (int e = lane; e < N * NU; e += NT) {
            const int k = e / NU, p = e % NU;
            const double u = hv[e] - dotc<NX, 1, 1>(Kf + k * NU * NX + p * NX, pv + k * NX);
            hv[e] = u; dx[c.iu(k) + p] = u;
        }
        c.tm.sync();
#pragma unroll 2
        for (int e = lane; e < N * NX; e += NT) {
            const int k = e / NX, i = e % NX;
            const int ai = row_agent(i);
            sv[e] = dotc<AX, 1, 1>(c.Jk(k) + i * LDJ + AX * ai, pv + k * NX + AX * ai) +
                    dotc<AU, 1, 1>(c.Jk(k) + i * LDJ + NX + AU * ai, hv + k * NU + AU * ai);
        }
        c.tm.sync();
#pragma unroll 2
        for (int e = lane; e < N * NX; e += NT) {
            const int k = e / NX, i = e % NX;
            const double nu = wv[e] + dotc<NX, NX, 1>(Tf + (k + 1) * NX * NX + i, sv + k * NX);
            dy[c.icd(k + 1) + i] = -nu;
        }
        // ---- slack / inequality-multiplier recovery ----
        const double* gv = c.vh(c.L->gv);
        for (int it = lane; it < N * pb->ng; it += NT) {
            const int k = it / pb->ng + 1, j = it % pb->ng;
            const double sig = c.v(c.L->Sig)[c.is(k) + j];
            const double rps = rp[c.is(k) + j];
            const double dyg = c.vh(c.L->dgv)[it] * (c.G_dot(gv, dx, k, j) - rc[c.icg(k) + j] - rps / sig);
            dy[c.icg(k) + j] = dyg;
            dx[c.is(k) + j] = (rps + dyg) / sig;
        }
        c.tm.sync();
    }
};

}  // namespace jipm
