// External Milky-Way acceleration a_NFW + a_MN (PAPER.md:L9 Abstract, L45 section 2.2.1, L63 section 2.2.2;
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
}

}  // namespace odisseo
