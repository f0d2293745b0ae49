// Device building blocks of the reverse-mode derivative shared by adjoint.cu (one simulation, O(N^2) grid
// kernel) and ensemble_adjoint.cu (one CTA per simulation).  Formulas: header of adjoint.cu.
#pragma once

#include "odisseo_common.cuh"
#include "ext_potential.cuh"

namespace odisseo {

constexpr int VJP_THREADS = 256;
constexpr int VJP_COMPS = 6;       // gx, gy, gz, mass term, eps term, G term

__device__ __forceinline__ void inv_powers(float s, float& f, float& g)
{
    const float y = rsqrt_approx(s);
    const float y2 = y * y;
    f = y2 * y;
    g = -3.0f * f * y2;
}
__device__ __forceinline__ void inv_powers(double s, double& f, double& g)
{
    const double y0 = rsqrt_approx_f64(s);
    const double e = fma(-s, y0 * y0, 1.0);
    const double y = y0 * fma(e, fma(0.375, e, 0.5), 1.0);       // s^-1/2 to fp64 rounding
    const double y2 = y * y;
    f = y2 * y;
    g = -3.0 * f * y2;
}

// One source j against one target i: accumulates (J^T c)_i / G (ax, ay, az), -dL/dm_i / G (am) and, when EG,
// dL/deps / (eps G) (ae) and dL/dG of the pair part (ag).
//   EQM (all masses equal): u = m (c_j - c_i), so the mass leaves the loop and ax, ay, az accumulate
//       (J^T c)_i / (G m); 28 instead of 35 FP32-pipe instructions per pair (no eps / G terms).
//   EG = false drops the eps and G terms (6 instructions): neither is in the paper's Theta.
template <typename T, bool EQM, bool EG>
__device__ __forceinline__ void vjp_pair_term(const T px, const T py, const T pz, const T pm, const T cjx, const T cjy,
                                              const T cjz, const T xi, const T yi, const T zi, const T mi, const T cxi,
                                              const T cyi, const T czi, const T eps2, T& ax, T& ay, T& az, T& am, T& ae,
                                              T& ag)
{
    const T dx = px - xi, dy = py - yi, dz = pz - zi;
    const T s = fma(dz, dz, fma(dy, dy, fma(dx, dx, eps2)));
    T f, g;
    inv_powers(s, f, g);
    const T pj = fma(dz, cjz, fma(dy, cjy, dx * cjx));              // d . c_j
    // u = m_i c_j - m_j c_i written as m_i (c_j - c_i) + (m_i - m_j) c_i: the difference of cotangents is
    // taken first (exact for close values), and the self term is exactly 0
    T ux = cjx - cxi, uy = cjy - cyi, uz = cjz - czi;
    if (!EQM) {
        const T dm = mi - pm;
        ux = fma(dm, cxi, mi * ux);
        uy = fma(dm, cyi, mi * uy);
        uz = fma(dm, czi, mi * uz);
    }
    const T gdu = g * fma(dz, uz, fma(dy, uy, dx * ux));            // g (d . u)
    ax = fma(f, ux, fma(gdu, dx, ax));
    ay = fma(f, uy, fma(gdu, dy, ay));
    az = fma(f, uz, fma(gdu, dz, az));
    am = fma(f, pj, am);
    if (EG) {
        const T qi = fma(dz, czi, fma(dy, cyi, dx * cxi));          // d . c_i
        const T mq = pm * qi;                                       // m_j (d . c_i)
        ae = fma(g, mq, ae);
        ag = fma(f, mq, ag);
    }
}

// The equal-mass, no-eps/G term on packed fp32 pairs: TWO sources (j, j+1) against one target whose coordinates and
// cotangent are duplicated in both halves.  27 FFMA2/FADD2/FMUL2 + 2 MUFU per two pairs; the halves of the
// accumulators are the even-j and odd-j partial sums.  Same formulas as vjp_pair_term<float, true, false>.
__device__ __forceinline__ void vjp_pair_term_x2(const f32x2 px, const f32x2 py, const f32x2 pz, const f32x2 cjx, const f32x2 cjy,
                                                 const f32x2 cjz, const f32x2 xi, const f32x2 yi, const f32x2 zi,
                                                 const f32x2 cxi, const f32x2 cyi, const f32x2 czi, const f32x2 e2,
                                                 const f32x2 minus3, f32x2& ax, f32x2& ay, f32x2& az, f32x2& am)
{
    const f32x2 dx = sub2(px, xi), dy = sub2(py, yi), dz = sub2(pz, zi);
    const f32x2 s = fma2(dz, dz, fma2(dy, dy, fma2(dx, dx, e2)));
    float sl, sh;
    unpk(s, sl, sh);
    const f32x2 y = pk(rsqrt_approx(sl), rsqrt_approx(sh));
    const f32x2 y2 = mul2(y, y);
    const f32x2 f = mul2(y2, y);
    const f32x2 g = mul2(mul2(f, y2), minus3);
    const f32x2 pj = fma2(dz, cjz, fma2(dy, cjy, mul2(dx, cjx)));          // d . c_j
    const f32x2 ux = sub2(cjx, cxi), uy = sub2(cjy, cyi), uz = sub2(cjz, czi);
    const f32x2 gdu = mul2(g, fma2(dz, uz, fma2(dy, uy, mul2(dx, ux))));     // g (d . u)
    ax = fma2(f, ux, fma2(gdu, dx, ax));
    ay = fma2(f, uy, fma2(gdu, dy, ay));
    az = fma2(f, uz, fma2(gdu, dz, az));
    am = fma2(f, pj, am);
}

// Fixed-shape sum over the block (xor-shuffle tree, then warp sums in order); valid in thread 0.
__device__ __forceinline__ double vjp_block_sum(double v, double* warp_scratch)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) warp_scratch[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < VJP_THREADS / 32; ++w) s += warp_scratch[w];
    return s;
}

// Cotangent c pulled back through a_NFW + a_MN at x, in fp64: h = (da/dx)^T c, and the terms of the
// parameter sums t[0..7] = d(c.a)/d(M_s, r_s, M_d, a, b, G, M_b, r_c).
__device__ __forceinline__ void ext_vjp(const PotParams<double>& pot, const double G, const double x, const double y,
                                        const double z, const double cx, const double cy, const double cz,
                                        double (&h)[3], double (&t)[8])
{
    h[0] = h[1] = h[2] = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) t[k] = 0.0;
    const double invG = G != 0.0 ? 1.0 / G : 0.0;
    if (pot.GMs != 0.0) {
        const double r2 = fma(x, x, fma(y, y, z * z));
        if (r2 > 0.0) {
            const double r = sqrt(r2), ir = 1.0 / r, ir3 = ir * ir * ir;
            const double cc = r * pot.inv_rs, opc = 1.0 + cc;
            const double mu = nfw_menc(cc);
            const double dmu_dr = pot.inv_rs * cc / (opc * opc);
            const double F = mu * ir3;
            const double dF_over_r = (dmu_dr * ir3 - 3.0 * mu * ir3 * ir) * ir;
            const double xc = fma(x, cx, fma(y, cy, z * cz));
            const double k1 = -pot.GMs * F, k2 = -pot.GMs * dF_over_r * xc;
            h[0] = fma(k1, cx, k2 * x); h[1] = fma(k1, cy, k2 * y); h[2] = fma(k1, cz, k2 * z);
            const double ca = k1 * xc;                                   // c . a_NFW
            t[0] += ca * (G * (1.0 / pot.GMs));                          // / M_s
            t[5] += ca * invG;
            const double dmu_drs = -cc * cc * pot.inv_rs / (opc * opc);
            t[1] += -pot.GMs * dmu_drs * ir3 * xc;
        }
    }
    if (pot.GMd != 0.0) {
        const double b = sqrt(pot.b2);
        const double B = sqrt(fma(z, z, pot.b2)), iB = 1.0 / B;
        const double s = pot.a + B;
        const double D2 = fma(x, x, fma(y, y, s * s));
        const double iD = 1.0 / sqrt(D2), iD3 = iD * iD * iD, iD5 = iD3 * iD * iD;
        const double kz = s * iB;                                        // a_z numerator is z kz
        const double wz = z * kz;
        const double dzk_dz = kz - pot.a * z * z * iB * iB * iB;         // d(z kz)/dz
        const double cw = fma(cx, x, fma(cy, y, cz * wz));
        const double q = -3.0 * cw * iD5;
        h[0] += -pot.GMd * fma(q, x, cx * iD3);
        h[1] += -pot.GMd * fma(q, y, cy * iD3);
        h[2] += -pot.GMd * fma(q, wz, cz * dzk_dz * iD3);
        const double ca = -pot.GMd * cw * iD3;                           // c . a_MN
        t[2] += ca * (G * (1.0 / pot.GMd));
        t[5] += ca * invG;
        t[3] += -pot.GMd * fma(q, s, cz * z * iB * iD3);
        t[4] += -pot.GMd * fma(q, s * b * iB, cz * z * (-pot.a * b * iB * iB * iB) * iD3);
    }
    if (pot.GMb != 0.0) {
        // a = -G M_b F(r) x,  F = P(s, tt)/r^3,  tt = (r/r_c)^2,  dP/dtt = tt^(s-1) e^-tt / Gamma(s)
        const double r2 = fma(x, x, fma(y, y, z * z));
        if (r2 > 0.0) {
            const double r = sqrt(r2), ir = 1.0 / r, ir3 = ir * ir * ir;
            const double tt = r2 * pot.inv_rc * pot.inv_rc;
            double dP;
            const double P = gamma_p(pot.bs, tt, pot.lgam_s, &dP);
            const double F = P * ir3;
            const double dF_over_r = (dP * 2.0 * pot.inv_rc * pot.inv_rc * ir3 * r - 3.0 * P * ir3 * ir) * ir;
            const double xc = fma(x, cx, fma(y, cy, z * cz));
            const double k1 = -pot.GMb * F, k2 = -pot.GMb * dF_over_r * xc;
            h[0] += fma(k1, cx, k2 * x); h[1] += fma(k1, cy, k2 * y); h[2] += fma(k1, cz, k2 * z);
            const double ca = k1 * xc;                                   // c . a_bulge
            t[6] += ca * (G * (1.0 / pot.GMb));                          // / M_b
            t[5] += ca * invG;
            t[7] += -pot.GMb * (dP * (-2.0 * tt * pot.inv_rc)) * ir3 * xc;   // dP/dr_c = dP/dtt (-2 tt / r_c)
        }
    }
}

}  // namespace odisseo
