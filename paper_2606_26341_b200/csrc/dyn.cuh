// dyn.cuh -- hand-written dynamics device functions per problem family (BASELINE.json configs):
// value F(x,u), Jacobian dF/d(x,u) and the adjoint-contracted Hessian lam^T d2F/d(x,u)^2 that the
// Lagrangian Hessian W and the constraint Jacobian A of PAPER.md:90 need.
//
// Quadrotor: 12 states (p, ZYX Euler phi/theta/psi, world velocity v, body rates w),
// 4 rotor thrusts, classical RK4 with zero-order hold.  Derivatives are ANALYTIC and chained through the
// four RK4 stages:
//     xi_1 = x, xi_{i+1} = x + a_{i+1} h k_i, k_i = f(xi_i,u), x+ = x + sum_i b_i k_i
//     dk_i/dz   = Df(xi_i) Y_i,              Y_{i+1} = [I 0] + a_{i+1} h dk_i/dz
//     lam^T d2x+/dz2 = sum_i Y_i^T (mu_i^T D2f(xi_i)) Y_i,   mu_4 = b_4 lam, mu_{i-1} = b_{i-1} lam + a_i h Df_x(xi_i)^T mu_i
// D2f only involves q = (phi,theta,psi,wp,wq,wr,T): a 7x7 contracted Hessian per RK stage.
// Phase 1 (lane <-> stage) evaluates the stage points, Df entries and the 7x7 Hessians; phase 2
// (half-warp <-> stage, lane <-> column of z=(x,u)) propagates the 16 columns.
#pragma once
#include "common.cuh"
#include "dyn_quat_gen.cuh"

namespace jipm {

constexpr double Q_G = 9.81, Q_MASS = 1.0, Q_ARM = 0.2, Q_JX = 0.01, Q_JY = 0.01, Q_JZ = 0.02, Q_KTAU = 0.02;

struct PointmassDyn {
    static constexpr int AX = 4, AU = 2, PD = 2, AZ = 6;
    static constexpr int RK_SCRATCH = 0;
    // exact zero-order hold of the double integrator
    __device__ static void F(const double* x, const double* u, double h, double* out) {
        out[0] = x[0] + h * x[2] + 0.5 * h * h * u[0];
        out[1] = x[1] + h * x[3] + 0.5 * h * h * u[1];
        out[2] = x[2] + h * u[0];
        out[3] = x[3] + h * u[1];
    }
};

// The paper's own vehicle: 13 states (p, quaternion, body velocity, body rates), four rotor speeds.
// ode / Jacobian-vector / transposed-Jacobian-vector / contracted-Hessian-vector products are generated from the model
// equations by gen_quat_dyn.py (dyn_quat_gen.cuh); derivs.cuh chains them through the four RK4 points.
struct QuatDyn {
    static constexpr int AX = 13, AU = 4, PD = 3, AZ = 17;
    static constexpr int RK_SCRATCH = 4 * RKW;
    __device__ static void F(const double* x, const double* u, double h, double* out) {
        double k1[13], k2[13], k3[13], k4[13], xi[13];
        quat_ode(x, u, k1);
#pragma unroll
        for (int i = 0; i < 13; ++i) xi[i] = x[i] + (0.5 * h) * k1[i];
        quat_ode(xi, u, k2);
#pragma unroll
        for (int i = 0; i < 13; ++i) xi[i] = x[i] + (0.5 * h) * k2[i];
        quat_ode(xi, u, k3);
#pragma unroll
        for (int i = 0; i < 13; ++i) xi[i] = x[i] + h * k3[i];
        quat_ode(xi, u, k4);
#pragma unroll
        for (int i = 0; i < 13; ++i) out[i] = x[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
    }
};

struct QuadBasics {
    double sph, cph, sth, cth, sps, cps, wp, wq, wr, a;
};

struct QuadDyn {
    static constexpr int AX = 12, AU = 4, PD = 3, AZ = 16;
    static constexpr int RK_SCRATCH = 4 * RKW;  // per (stage, agent)

    // continuous dynamics xdot = f(x,u); also returns the quantities the derivatives reuse
    __device__ static void ode(const double* x, const double* u, double* d, QuadBasics& b) {
        double sph, cph, sth, cth, sps, cps;
        sincos(x[3], &sph, &cph);
        sincos(x[4], &sth, &cth);
        sincos(x[5], &sps, &cps);
        const double wp = x[9], wq = x[10], wr = x[11];
        const double T = u[0] + u[1] + u[2] + u[3];
        const double tan_th = sth / cth;
        const double qr = wq * sph + wr * cph;
        d[0] = x[6]; d[1] = x[7]; d[2] = x[8];
        d[3] = wp + qr * tan_th;
        d[4] = wq * cph - wr * sph;
        d[5] = qr / cth;
        const double a = T * (1.0 / Q_MASS);
        d[6] = a * (cps * sth * cph + sps * sph);
        d[7] = a * (sps * sth * cph - cps * sph);
        d[8] = a * (cth * cph) - Q_G;
        const double tx = Q_ARM * (u[1] - u[3]);
        const double ty = Q_ARM * (u[2] - u[0]);
        const double tz = Q_KTAU * (u[0] - u[1] + u[2] - u[3]);
        d[9] = (tx - (Q_JZ - Q_JY) * wq * wr) * (1.0 / Q_JX);
        d[10] = (ty - (Q_JX - Q_JZ) * wr * wp) * (1.0 / Q_JY);
        d[11] = (tz - (Q_JY - Q_JX) * wp * wq) * (1.0 / Q_JZ);
        b.sph = sph; b.cph = cph; b.sth = sth; b.cth = cth; b.sps = sps; b.cps = cps;
        b.wp = wp; b.wq = wq; b.wr = wr; b.a = a;
    }

    __device__ static void F(const double* x, const double* u, double h, double* out) {
        double k1[12], k2[12], k3[12], k4[12], xi[12];
        QuadBasics b;
        ode(x, u, k1, b);
#pragma unroll
        for (int i = 0; i < 12; ++i) xi[i] = x[i] + (0.5 * h) * k1[i];
        ode(xi, u, k2, b);
#pragma unroll
        for (int i = 0; i < 12; ++i) xi[i] = x[i] + (0.5 * h) * k2[i];
        ode(xi, u, k3, b);
#pragma unroll
        for (int i = 0; i < 12; ++i) xi[i] = x[i] + h * k3[i];
        ode(xi, u, k4, b);
#pragma unroll
        for (int i = 0; i < 12; ++i) out[i] = x[i] + (h / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
    }

    // first-derivative entries of f at one RK point (layout in the header comment of derivs_phase1)
    __device__ static void dentries(const QuadBasics& b, double* D) {
        const double sec = 1.0 / b.cth, tan_th = b.sth * sec, sec2 = sec * sec;
        const double qr = b.wq * b.sph + b.wr * b.cph, qs = b.wq * b.cph - b.wr * b.sph;
        D[0] = qs * tan_th; D[1] = qr * sec2; D[2] = b.sph * tan_th; D[3] = b.cph * tan_th;
        D[4] = -qr; D[5] = b.cph; D[6] = -b.sph;
        D[7] = qs * sec; D[8] = qr * b.sth * sec2; D[9] = b.sph * sec; D[10] = b.cph * sec;
        const double a = b.a;
        // a * dr/dphi, a * dr/dtheta, a * dr/dpsi, r/m with r = R(phi,theta,psi) e3
        D[11] = a * (-b.cps * b.sth * b.sph + b.sps * b.cph);
        D[12] = a * (-b.sps * b.sth * b.sph - b.cps * b.cph);
        D[13] = a * (-b.cth * b.sph);
        D[14] = a * (b.cps * b.cth * b.cph);
        D[15] = a * (b.sps * b.cth * b.cph);
        D[16] = a * (-b.sth * b.cph);
        const double rx = b.cps * b.sth * b.cph + b.sps * b.sph, ry = b.sps * b.sth * b.cph - b.cps * b.sph;
        D[17] = a * (-ry); D[18] = a * rx; D[19] = 0.0;
        D[20] = rx * (1.0 / Q_MASS); D[21] = ry * (1.0 / Q_MASS); D[22] = b.cth * b.cph * (1.0 / Q_MASS);
        D[23] = b.wp; D[24] = b.wq; D[25] = b.wr;
    }
};

constexpr double QC1 = (Q_JZ - Q_JY) / Q_JX, QC2 = (Q_JX - Q_JZ) / Q_JY, QC3 = (Q_JY - Q_JX) / Q_JZ;

// out = Df_x(xi)^T mu  (12-vector) from the D entries
__device__ __forceinline__ void quad_dfxT(const double* D, const double* mu, double* out) {
    out[0] = out[1] = out[2] = 0.0;
    out[3] = D[0] * mu[3] + D[4] * mu[4] + D[7] * mu[5] + D[11] * mu[6] + D[12] * mu[7] + D[13] * mu[8];
    out[4] = D[1] * mu[3] + D[8] * mu[5] + D[14] * mu[6] + D[15] * mu[7] + D[16] * mu[8];
    out[5] = D[17] * mu[6] + D[18] * mu[7] + D[19] * mu[8];
    out[6] = mu[0]; out[7] = mu[1]; out[8] = mu[2];
    const double wp = D[23], wq = D[24], wr = D[25];
    out[9] = mu[3] - QC2 * wr * mu[10] - QC3 * wq * mu[11];
    out[10] = D[2] * mu[3] + D[5] * mu[4] + D[9] * mu[5] - QC1 * wr * mu[9] - QC3 * wp * mu[11];
    out[11] = D[3] * mu[3] + D[6] * mu[4] + D[10] * mu[5] - QC1 * wq * mu[9] - QC2 * wp * mu[10];
}

// H = sum_j mu_j D2 f_j over q = (phi,theta,psi,wp,wq,wr,T); 16 structural non-zeros, order:
// pp pt ps tt ts ss | p-wq p-wr t-wq t-wr | pT tT sT | wpwq wpwr wqwr      (p=phi, t=theta, s=psi)
__device__ __forceinline__ void quad_hentries(const QuadBasics& b, const double* mu, double* H) {
    const double sec = 1.0 / b.cth, tan_th = b.sth * sec, sec2 = sec * sec;
    const double qr = b.wq * b.sph + b.wr * b.cph, qs = b.wq * b.cph - b.wr * b.sph;
    const double m3 = mu[3], m4 = mu[4], m5 = mu[5];
    const double a = b.a, mx = mu[6], my = mu[7], mz = mu[8];
    const double sph = b.sph, cph = b.cph, sth = b.sth, cth = b.cth, sps = b.sps, cps = b.cps;
    const double rx = cps * sth * cph + sps * sph, ry = sps * sth * cph - cps * sph, rz = cth * cph;
    // angle-angle
    double pp = m3 * (-qr * tan_th) + m4 * (-qs) + m5 * (-qr * sec);
    double pt = m3 * (qs * sec2) + m5 * (qs * sth * sec2);
    double tt = m3 * (2.0 * qr * sec2 * tan_th) + m5 * (qr * (sec + 2.0 * sth * sth * sec2 * sec));
    // thrust direction second derivatives
    const double rpp_x = -rx, rpp_y = -ry, rpp_z = -rz;
    const double rpt_x = -cps * cth * sph, rpt_y = -sps * cth * sph, rpt_z = sth * sph;
    const double rps_x = sps * sth * sph + cps * cph, rps_y = -cps * sth * sph + sps * cph;
    const double rtt_x = -cps * sth * cph, rtt_y = -sps * sth * cph, rtt_z = -cth * cph;
    const double rts_x = -sps * cth * cph, rts_y = cps * cth * cph;
    const double rss_x = -rx, rss_y = -ry;
    pp += a * (mx * rpp_x + my * rpp_y + mz * rpp_z);
    pt += a * (mx * rpt_x + my * rpt_y + mz * rpt_z);
    double ps = a * (mx * rps_x + my * rps_y);
    tt += a * (mx * rtt_x + my * rtt_y + mz * rtt_z);
    double ts = a * (mx * rts_x + my * rts_y);
    double ss = a * (mx * rss_x + my * rss_y);
    H[0] = pp; H[1] = pt; H[2] = ps; H[3] = tt; H[4] = ts; H[5] = ss;
    // angle-rate
    H[6] = m3 * (cph * tan_th) + m4 * (-sph) + m5 * (cph * sec);    // phi-wq
    H[7] = m3 * (-sph * tan_th) + m4 * (-cph) + m5 * (-sph * sec);  // phi-wr
    H[8] = m3 * (sph * sec2) + m5 * (sph * sth * sec2);             // theta-wq
    H[9] = m3 * (cph * sec2) + m5 * (cph * sth * sec2);             // theta-wr
    // angle-thrust: (1/m) mu_v . dr/dangle
    const double im = 1.0 / Q_MASS;
    H[10] = im * (mx * (-cps * sth * sph + sps * cph) + my * (-sps * sth * sph - cps * cph) + mz * (-cth * sph));
    H[11] = im * (mx * (cps * cth * cph) + my * (sps * cth * cph) + mz * (-sth * cph));
    H[12] = im * (mx * (-ry) + my * rx);
    // rate-rate
    H[13] = -QC3 * mu[11]; H[14] = -QC2 * mu[10]; H[15] = -QC1 * mu[9];
}

// t = Hq v for the 7-vector v = (phi,theta,psi,wp,wq,wr,T)
__device__ __forceinline__ void quad_hmul(const double* H, const double* v, double* t) {
    t[0] = H[0] * v[0] + H[1] * v[1] + H[2] * v[2] + H[6] * v[4] + H[7] * v[5] + H[10] * v[6];
    t[1] = H[1] * v[0] + H[3] * v[1] + H[4] * v[2] + H[8] * v[4] + H[9] * v[5] + H[11] * v[6];
    t[2] = H[2] * v[0] + H[4] * v[1] + H[5] * v[2] + H[12] * v[6];
    t[3] = H[13] * v[4] + H[14] * v[5];
    t[4] = H[6] * v[0] + H[8] * v[1] + H[13] * v[3] + H[15] * v[5];
    t[5] = H[7] * v[0] + H[9] * v[1] + H[14] * v[3] + H[15] * v[4];
    t[6] = H[10] * v[0] + H[11] * v[1] + H[12] * v[2];
}

// column of dk/dz = Df(xi) [Yx; e_u] for one column; Yx = d xi / d z_j (12), uj = d u / d z_j (4)
__device__ __forceinline__ void quad_dfcol(const double* D, const double* Y, const double* uj, double* K) {
    K[0] = Y[6]; K[1] = Y[7]; K[2] = Y[8];
    K[3] = D[0] * Y[3] + D[1] * Y[4] + Y[9] + D[2] * Y[10] + D[3] * Y[11];
    K[4] = D[4] * Y[3] + D[5] * Y[10] + D[6] * Y[11];
    K[5] = D[7] * Y[3] + D[8] * Y[4] + D[9] * Y[10] + D[10] * Y[11];
    const double Tj = uj[0] + uj[1] + uj[2] + uj[3];
    K[6] = D[11] * Y[3] + D[14] * Y[4] + D[17] * Y[5] + D[20] * Tj;
    K[7] = D[12] * Y[3] + D[15] * Y[4] + D[18] * Y[5] + D[21] * Tj;
    K[8] = D[13] * Y[3] + D[16] * Y[4] + D[19] * Y[5] + D[22] * Tj;
    const double wp = D[23], wq = D[24], wr = D[25];
    K[9] = -QC1 * (wr * Y[10] + wq * Y[11]) + (Q_ARM / Q_JX) * (uj[1] - uj[3]);
    K[10] = -QC2 * (wr * Y[9] + wp * Y[11]) + (Q_ARM / Q_JY) * (uj[2] - uj[0]);
    K[11] = -QC3 * (wq * Y[9] + wp * Y[10]) + (Q_KTAU / Q_JZ) * (uj[0] - uj[1] + uj[2] - uj[3]);
}

}  // namespace jipm
