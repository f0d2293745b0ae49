// External Milky-Way acceleration a_NFW + a_MN (+ the bulge of MWPotential2014, L45) (PAPER.md:L9 Abstract, L45 section 2.2.1, L63 section 2.2.2;
// SURVEY.md 8a row a2), shared by the integrator kernel (integrate.cu) and the ensemble kernel
// (ensemble.cu).  Accurate sqrt / divide / log1p: these translation units are built without fast-math.
#pragma once

#include "odisseo_common.cuh"

namespace odisseo {

__device__ __forceinline__ float rsqrt_acc(float x) { return 1.0f / sqrtf(x); }
__device__ __forceinline__ double rsqrt_acc(double x) { return 1.0 / sqrt(x); }
__device__ __forceinline__ float sqrt_acc(float x) { return sqrtf(x); }
__device__ __forceinline__ double sqrt_acc(double x) { return sqrt(x); }
__device__ __forceinline__ float log1p_acc(float x) { return log1pf(x); }
__device__ __forceinline__ double log1p_acc(double x) { return log1p(x); }

// NFW enclosed-mass function m(c) = ln(1+c) - c/(1+c).  For small c the two terms cancel
// (m ~ c^2/2), so below c = 0.1 use the alternating series sum_{k>=2} (-1)^k (k-1)/k c^k
// (reading R12); the truncation c^(K+1) is < 1 ulp for the K used.
template <typename T> __device__ __forceinline__ T nfw_menc(T c)
{
    if (c < (T)0.1) {
        constexpr int K = sizeof(T) == 4 ? 9 : 18;
        T s = (T)0;
#pragma unroll
        for (int k = K; k >= 2; --k) {
            const T coef = (T)((k & 1) ? -1.0 : 1.0) * (T)(k - 1) / (T)k;
            s = fma(s, c, coef);
        }
        return s * c * c;
    }
    return log1p_acc(c) - c / ((T)1 + c);
}

__device__ __forceinline__ float exp_acc(float x) { return expf(x); }
__device__ __forceinline__ double exp_acc(double x) { return exp(x); }
__device__ __forceinline__ float log_acc(float x) { return logf(x); }
__device__ __forceinline__ double log_acc(double x) { return log(x); }

// Regularised lower incomplete gamma function P(s, t), 0 < s < 2 (bulge enclosed mass, reading R21):
//   t < s + 1 : Kummer series  P = t^s e^-t / Gamma(s+1) * sum_k t^k / ((s+1)...(s+k))   (all terms positive)
//   t >= s + 1: Legendre continued fraction of Q = 1 - P by the modified Lentz recurrence
//   t > TMAX  : 1 - P < 1 ulp: P = 1.
// lgam_s = ln Gamma(s) comes from the host.  Also returns dP/dt = t^(s-1) e^-t / Gamma(s) when asked.
template <typename T>
__device__ __forceinline__ T gamma_p(const T s, const T t, const T lgam_s, T* dP_dt = nullptr)
{
    constexpr T TMAX = sizeof(T) == 4 ? (T)20 : (T)40;
    constexpr T EPS = sizeof(T) == 4 ? (T)6e-8 : (T)1e-16;
    constexpr int ITMAX = sizeof(T) == 4 ? 40 : 120;
    if (!(t > (T)0)) { if (dP_dt) *dP_dt = (T)0; return (T)0; }
    if (t > (T)700) { if (dP_dt) *dP_dt = (T)0; return (T)1; }
    const T pre = exp_acc(s * log_acc(t) - t - lgam_s);              // t^s e^-t / Gamma(s)
    if (dP_dt) *dP_dt = pre / t;
    if (t > TMAX) return (T)1;
    if (t < s + (T)1) {
        T term = (T)1 / s, sum = term;                                // sum_k t^k / (s (s+1) ... (s+k))
        for (int k = 1; k < ITMAX; ++k) {
            term *= t / (s + (T)k);
            sum += term;
            if (term < EPS * sum) break;
        }
        const T p = pre * sum;
        return p < (T)1 ? p : (T)1;
    }
    // Q = pre / (t + 1 - s - 1 (1 - s) / (t + 3 - s - 2 (2 - s) / (t + 5 - s - ...)))
    constexpr T TINY = sizeof(T) == 4 ? (T)1e-30 : (T)1e-300;
    T b = t + (T)1 - s, c = (T)1 / TINY, d = (T)1 / b, h = d;
    for (int k = 1; k < ITMAX; ++k) {
        const T an = -(T)k * ((T)k - s);
        b += (T)2;
        d = an * d + b;
        d = (d < TINY && d > -TINY) ? TINY : d;
        c = b + an / c;
        c = (c < TINY && c > -TINY) ? TINY : c;
        d = (T)1 / d;
        const T del = d * c;
        h *= del;
        if ((del > (T)1 ? del - (T)1 : (T)1 - del) < EPS) break;
    }
    const T p = (T)1 - pre * h;
    return p > (T)0 ? p : (T)0;
}

template <typename T>
__device__ __forceinline__ void ext_accel(const PotParams<T>& pot, T x, T y, T z, T& ax, T& ay, T& az)
{
    ax = ay = az = (T)0;
    if (pot.GMs != (T)0) {
        const T r2 = fma(x, x, fma(y, y, z * z));
        if (r2 > (T)0) {
            const T rinv = rsqrt_acc(r2);
            const T c = (r2 * rinv) * pot.inv_rs;
            const T f = -pot.GMs * nfw_menc(c) * (rinv * rinv * rinv);
            ax = f * x; ay = f * y; az = f * z;
        }
    }
    if (pot.GMd != (T)0) {
        const T B = sqrt_acc(fma(z, z, pot.b2));
        const T sB = pot.a + B;
        const T D2 = fma(x, x, fma(y, y, sB * sB));
        const T dinv = rsqrt_acc(D2);
        const T f = -pot.GMd * (dinv * dinv * dinv);
        ax = fma(f, x, ax);
        ay = fma(f, y, ay);
        az = fma(f * z, sB / B, az);
    }
    if (pot.GMb != (T)0) {
        const T r2 = fma(x, x, fma(y, y, z * z));
        if (r2 > (T)0) {                                     // direction undefined at the centre: 0 (as NFW, R12)
            const T rinv = rsqrt_acc(r2);
            const T f = -pot.GMb * gamma_p(pot.bs, r2 * pot.inv_rc * pot.inv_rc, pot.lgam_s) * (rinv * rinv * rinv);
            ax = fma(f, x, ax);
            ay = fma(f, y, ay);
            az = fma(f, z, az);
        }
    }
}

}  // namespace odisseo
