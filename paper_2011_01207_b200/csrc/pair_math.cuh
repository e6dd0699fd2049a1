// pair_math.cuh -- per-pair arithmetic of the real-space AMOEBA polarization kernels.
//
// The paper prints no interaction formula (refs only); these functions
// implement DESIGN.md section 2 (= SURVEY 8(c)):
//   Ewald   bn_0 = erfc(bR)/R,  bn_k = [(2k-1) bn_{k-1} + (2b^2)^k/(b sqrt(pi)) exp(-b^2R^2)]/R^2
//   Thole   x = a R^3/sqrt(alpha_i alpha_j) = R^3 w_i w_j, w = (a/alpha)^(1/2)
//           1-lam3 = e^-x, 1-lam5 = (1+x)e^-x, 1-lam7 = (1+x+0.6x^2)e^-x
//   (F1)    G_k = bn_k - (1 - lam_{2k+1}) rr_k        (unmasked pairs; masked pairs: correction pass)
//   (F2)    E_i += [q_j G1 + G2 (d_j.R) + (G3/3)(R.Q_j R)] R - G1 d_j - (2/3) G2 (Q_j R)
//   (T1,T2) m1 = G1, m2 = G2 ;  (T mu)_i += -m1 mu_j + m2 (mu_j.R) R
// with R = r_i - r_j.  Written so that R^(2k+1) G_k is formed first (one common e^{-z^2} factor),
// then scaled by R^-(2k+1):  R^3 bn1 = e^{-z^2}[erfcx(z) + c z],  R^5 bn2 = e^{-z^2}[3(..) + 2c z^3],
// R^7 bn3 = e^{-z^2}[15(..) + 10 c z^3 + 4 c z^5],  z = bR, c = 2/sqrt(pi).
//
// MIXED (float): erfcx by the degree-7 polynomial of erfcx_coeffs.h in u = 1/(1+0.35z)
// (MUFU.RCP), exponentials by ex2.approx, 1/R by MUFU.RSQ: 4 MUFU + ~45 FMA-pipe ops per pair.
// FP64 (double): erfcx by a degree-16 polynomial in the same u, exponentials by exp_neg (below);
// libm only in the FP64 correction pass over the few same-group pairs.
#pragma once

#include <cuda_runtime.h>

#include "erfcx_coeffs.h"
#include "erfcx_coeffs64.h"

namespace tkhp {

template <typename real>
struct PairConsts {
    real beta;      // Ewald coefficient
    real c1;        // 2/sqrt(pi)
    real c23;       // (2/3) c1
    real rc2;       // cutoff^2
    real box;       // box edge (PPI kernels)
    real inv_box;
    // products formed once on the host for the packed FP32 kernels (atom_pairs.cu)
    real pb;        // P beta (P = TKHP_ERFCX_P): u = 1 / (1 + pb R)
    real nb2l;      // -beta^2 log2 e:          e^{-z^2} = ex2(nb2l R^2)
    real c1b;       // (2/sqrt pi) beta:        c z = c1b R
    real k3;        // (4/(3 sqrt pi)) beta^3:  (2c/3) z^3 = k3 R^3
    int fixed;      // TKHP_FIXED (FP32 kernels only): int64 fixed-point accumulators (common.cuh acc_add)
    int far_rows;   // ATOM lists: the first class of rows holds pairs whose Thole damping has died out (THOLE = false)
};

template <typename real> struct Vec4;
template <> struct Vec4<float> { using type = float4; };
template <> struct Vec4<double> { using type = double4; };

__device__ __forceinline__ float fast_rcp(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float fast_ex2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float fast_rsqrt(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// erfc(z) exp(z^2), 0 <= z <= 6, relative error ~4e-7 in FP32
__device__ __forceinline__ float erfcx_f32(float z) {
    constexpr float c[TKHP_ERFCX_DEG + 1] = TKHP_ERFCX_COEFFS;
    const float u = fast_rcp(fmaf(TKHP_ERFCX_P, z, 1.0f));
    float p = c[TKHP_ERFCX_DEG];
#pragma unroll
    for (int k = TKHP_ERFCX_DEG - 1; k >= 0; --k) p = fmaf(p, u, c[k]);
    return p;
}

// ---- MIXED: G_1..G_NK for W unmasked pairs at once ------------------------------------------
// Written stage by stage over W independent pairs so that the scheduler can interleave W
// dependency chains (the Horner chain alone is 8 dependent FFMAs); W = 2 in the cluster kernels.
// Scaled forms: R^3 G1 = ez g1 - et;  R^5 G2 / 3 = ez (g1 + (2c/3) z^3) - (1+x) et;
// R^7 G3 / 15 = ez (g1 + (2c/3) z^3 + (4c/15) z^5) - (1 + x + 0.6 x^2) et.
// THOLE = false (FAR rows of the ATOM lists): x = R^3 w_i w_j is so large that e^-x is below the
// resolution of the sums; the Thole exponential and its polynomial are skipped (lambda = 1).
template <int NK, int W, bool THOLE = true>
__device__ __forceinline__ void radial_f32_w(const float (&r2)[W], const float (&ww)[W],
                                             const PairConsts<float> &k, float (&G)[W][NK]) {
    constexpr float c[TKHP_ERFCX_DEG + 1] = TKHP_ERFCX_COEFFS;
    constexpr float NLOG2E = -1.4426950408889634f;
    float rinv[W], r[W], z[W], u[W], p[W], z2[W], ez[W], t[W], x[W], et[W], g1[W], rinv2[W], rinv3[W];
#pragma unroll
    for (int i = 0; i < W; ++i) rinv[i] = fast_rsqrt(r2[i]);
#pragma unroll
    for (int i = 0; i < W; ++i) r[i] = r2[i] * rinv[i];
#pragma unroll
    for (int i = 0; i < W; ++i) z[i] = k.beta * r[i];
#pragma unroll
    for (int i = 0; i < W; ++i) u[i] = fast_rcp(fmaf(TKHP_ERFCX_P, z[i], 1.0f));
#pragma unroll
    for (int i = 0; i < W; ++i) { z2[i] = z[i] * z[i]; t[i] = r2[i] * r[i]; }
#pragma unroll
    for (int i = 0; i < W; ++i) { ez[i] = fast_ex2(z2[i] * NLOG2E); x[i] = THOLE ? t[i] * ww[i] : 0.f; }
#pragma unroll
    for (int i = 0; i < W; ++i) { et[i] = THOLE ? fast_ex2(x[i] * NLOG2E) : 0.f; p[i] = c[TKHP_ERFCX_DEG]; }
#pragma unroll
    for (int d = TKHP_ERFCX_DEG - 1; d >= 0; --d) {
#pragma unroll
        for (int i = 0; i < W; ++i) p[i] = fmaf(p[i], u[i], c[d]);
    }
#pragma unroll
    for (int i = 0; i < W; ++i) {
        g1[i] = fmaf(k.c1, z[i], p[i]);                 // erfcx(z) + c z
        rinv2[i] = rinv[i] * rinv[i];
        rinv3[i] = rinv2[i] * rinv[i];
        G[i][0] = fmaf(ez[i], g1[i], -et[i]) * rinv3[i];
    }
    if (NK >= 2) {
#pragma unroll
        for (int i = 0; i < W; ++i) {
            const float t5 = (k.c23 * z[i]) * z2[i];    // (2c/3) z^3
            const float h2 = g1[i] + t5;
            const float xet = x[i] * et[i];
            const float xe = xet + et[i];               // (1+x) e^-x
            const float r5 = (3.0f * rinv2[i]) * rinv3[i];
            G[i][1] = fmaf(ez[i], h2, -xe) * r5;
            if (NK >= 3) {
                const float h3 = fmaf(0.4f * t5, z2[i], h2);
                const float xe7 = fmaf(0.6f * x[i], xet, xe);   // (1 + x + 0.6 x^2) e^-x
                G[i][2] = fmaf(ez[i], h3, -xe7) * ((5.0f * rinv2[i]) * r5);
            }
        }
    }
}

template <int NK>
__device__ __forceinline__ void radial_f32(float r2, float ww, const PairConsts<float> &k, float *G) {
    const float r2a[1] = {r2}, wwa[1] = {ww};
    float Ga[1][NK];
    radial_f32_w<NK, 1>(r2a, wwa, k, Ga);
#pragma unroll
    for (int i = 0; i < NK; ++i) G[i] = Ga[0][i];
}

// ---- FP64: G_1..G_NK for an unmasked pair --------------------------------------------------
// libm's erfc() and exp() cost about 250 FP64-pipe instructions per pair; the same scaled form as the
// FP32 path needs about 90: erfcx(z) by the degree-16 polynomial of erfcx_coeffs64.h in
// u = 1/(1 + 0.35 z) (5e-15 relative, 0 <= z <= 6) and e^{-y} by exp_neg below (2e-15).
//
// e^{y} for y <= 0: y log2(e) = n + f, |f| <= 1/2, 2^f = e^{f ln 2} by its Taylor polynomial of degree
// 11 (6e-15), scaled by 2^n through the exponent field; 0 below the normal range.
__device__ __forceinline__ double exp_neg(double y) {
    constexpr double L2E_HI = 1.4426950408889634, L2E_LO = 2.0355273740931033e-17;
    const double tq = y * L2E_HI;
    if (tq < -1020.0) return 0.0;
    const double n = rint(tq);
    const double f = fma(y, L2E_HI, -n) + y * L2E_LO;
    constexpr double c[12] = {1.0, 0.6931471805599453, 0.2402265069591007, 0.05550410866482158,
                              0.009618129107628477, 0.0013333558146428443, 1.5403530393381608e-4,
                              1.5252733804059841e-5, 1.3215486790144307e-6, 1.0178086009239699e-7,
                              7.054911620801123e-9, 4.445538271870811e-10};
    double p = c[11];
#pragma unroll
    for (int k = 10; k >= 0; --k) p = fma(p, f, c[k]);
    const int hi = __double2hiint(p) + ((int)n << 20);
    return __hiloint2double(hi, __double2loint(p));
}

template <int NK, bool THOLE = true>
__device__ __forceinline__ void radial_f64(double r2, double ww, const PairConsts<double> &k, double *G) {
    constexpr double c[TKHP_ERFCX64_DEG + 1] = TKHP_ERFCX64_COEFFS;
    const double rinv = rsqrt(r2);
    const double r = r2 * rinv;
    const double rinv2 = rinv * rinv;
    const double z = k.beta * r;
    const double z2 = z * z;
    const double ez = exp_neg(-z2);
    // R^(2k+1) bn_k = ez [(2k-1)!! (erfcx(z) + c z) + ...]  (pair_math header)
    const double u = 1.0 / fma(TKHP_ERFCX64_P, z, 1.0);
    double p = c[TKHP_ERFCX64_DEG];
#pragma unroll
    for (int d = TKHP_ERFCX64_DEG - 1; d >= 0; --d) p = fma(p, u, c[d]);
    const double cz = k.c1 * z;
    const double B1 = ez * (p + cz);                       // erfc(z) + c z e^{-z^2}
    const double x = THOLE ? (r2 * r) * ww : 0.0;
    const double et = THOLE ? exp_neg(-x) : 0.0;
    const double rinv3 = rinv2 * rinv;
    G[0] = (B1 - et) * rinv3;
    if (NK >= 2) {
        const double B2 = 3.0 * B1 + 2.0 * cz * z2 * ez;
        const double rinv5 = rinv3 * rinv2;
        G[1] = (B2 - 3.0 * (1.0 + x) * et) * rinv5;
        if (NK >= 3) {
            const double B3 = 5.0 * B2 + 4.0 * cz * z2 * z2 * ez;
            G[2] = (B3 - 15.0 * (1.0 + x + 0.6 * x * x) * et) * (rinv5 * rinv2);
        }
    }
}

template <int NK>
__device__ __forceinline__ void radial(float r2, float ww, const PairConsts<float> &k, float *G) {
    radial_f32<NK>(r2, ww, k, G);
}
template <int NK, int W, bool THOLE = true>
__device__ __forceinline__ void radial_w(const float (&r2)[W], const float (&ww)[W], const PairConsts<float> &k,
                                         float (&G)[W][NK]) {
    radial_f32_w<NK, W, THOLE>(r2, ww, k, G);
}
template <int NK, int W, bool THOLE = true>
__device__ __forceinline__ void radial_w(const double (&r2)[W], const double (&ww)[W], const PairConsts<double> &k,
                                         double (&G)[W][NK]) {
#pragma unroll
    for (int i = 0; i < W; ++i) radial_f64<NK, THOLE>(r2[i], ww[i], k, G[i]);
}
template <int NK>
__device__ __forceinline__ void radial(double r2, double ww, const PairConsts<double> &k, double *G) {
    radial_f64<NK>(r2, ww, k, G);
}

// ---- masked pair (same polarization group), FP64 only: G_k = bn_k - rr_k --------------------
// Cancellation-prone (10x..1400x at R ~ 1 A, SURVEY hard part 3): always evaluated in FP64 in the
// correction pass ("correct_scaling" second kernel of the paper).
__device__ __forceinline__ void radial_masked_f64(double r2, double beta, double *G) {
    const double r = sqrt(r2);
    const double rinv = 1.0 / r;
    const double rinv2 = rinv * rinv;
    const double z = beta * r;
    const double z2 = z * z;
    const double ez = exp(-z2);
    const double cz = (beta > 0.0 ? 1.1283791670955125739 : 0.0) * z;   // 2/sqrt(pi) z
    // B_k - (2k-1)!! with erfc(z) - 1 = -erf(z): no cancellation against the bare Coulomb term
    const double B1m = -erf(z) + cz * ez;
    const double B2m = 3.0 * B1m + 2.0 * cz * z2 * ez;
    const double B3m = 5.0 * B2m + 4.0 * cz * z2 * z2 * ez;
    const double rinv3 = rinv2 * rinv, rinv5 = rinv3 * rinv2;
    G[0] = B1m * rinv3;
    G[1] = B2m * rinv5;
    G[2] = B3m * rinv5 * rinv2;
}

// ---- (T1,T2) one direction: out += -m1 mu + m2 (mu.R) R ------------------------------------
template <typename real>
__device__ __forceinline__ void tmu_apply(real m1, real m2, real Rx, real Ry, real Rz, real mx, real my,
                                          real mz, real &ox, real &oy, real &oz) {
    const real c = m2 * (mx * Rx + my * Ry + mz * Rz);
    const real n1 = -m1;
    ox = fma(c, Rx, fma(n1, mx, ox));
    oy = fma(c, Ry, fma(n1, my, oy));
    oz = fma(c, Rz, fma(n1, mz, oz));
}

// ---- (F2) field at the point R away from a multipole (q, d, Q); sign = +1: R = r_i - r_j ----
// For the mirrored direction (field at j from i's multipoles) pass (-Rx,-Ry,-Rz).
template <typename real>
__device__ __forceinline__ void field_apply(const real *G, real Rx, real Ry, real Rz, real q, real dx, real dy,
                                            real dz, real qxx, real qxy, real qxz, real qyy, real qyz,
                                            real qzz, real &ex, real &ey, real &ez) {
    const real dR = dx * Rx + dy * Ry + dz * Rz;
    const real tx = qxx * Rx + qxy * Ry + qxz * Rz;
    const real ty = qxy * Rx + qyy * Ry + qyz * Rz;
    const real tz = qxz * Rx + qyz * Ry + qzz * Rz;
    const real RTR = Rx * tx + Ry * ty + Rz * tz;
    const real rad = q * G[0] + G[1] * dR + (G[2] * (real)(1.0 / 3.0)) * RTR;
    const real g23 = G[1] * (real)(-2.0 / 3.0);
    const real n1 = -G[0];
    ex = fma(rad, Rx, fma(n1, dx, fma(g23, tx, ex)));
    ey = fma(rad, Ry, fma(n1, dy, fma(g23, ty, ey)));
    ez = fma(rad, Rz, fma(n1, dz, fma(g23, tz, ez)));
}

}  // namespace tkhp
