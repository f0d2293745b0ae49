// The per-particle body of one KDK step, shared by the O(N) step kernel (integrate.cu) and the persistent whole-loop
// kernel (fused_step.cuh) so that both execute the same instruction sequence (their results are bit-identical):
//
//   a_pair = G [m] * sum of the S rows of the particle's i-block, increasing s   [REDUCE] -> acc
//   a      = a_pair + a_ext(x)
//   v     += a dt/2                    [STEP_CLOSE: second half kick of the step that just ended]
//   snapshot {x, v, a_pair}            [tape of the reverse mode]
//   v     += a dt/2 ; x += v dt        [STEP_OPEN: first half kick + drift of the next step] -> staged record
//
// The two half kicks are two separate FMAs, so a step split across two calls is bit-identical to the fused one
// (PAPER.md:L47 Velocity-Verlet; chaining contract in include/odisseo.h).
#pragma once

#include "odisseo_common.cuh"
#include "ext_potential.cuh"

namespace odisseo {

template <typename T> struct Vec4;
template <> struct Vec4<float> { typedef float4 type; };
template <> struct Vec4<double> { typedef double4 type; };

// Staged source record writers: plain {x, y, z, m} in both precisions (fp32 16 B, fp64 32 B).  The packed fp32 loops
// take the source coordinate as a scalar operand broadcast to both halves (SASS FADD2 R, Rj.F32, -Ri.F32x2), so nothing
// is pre-duplicated.  Records [n, n_pad) are massless padding parked far away (odisseo_common.cuh PAD_POS_*).
__device__ __forceinline__ void stage_record(void* jsrc, int64_t i, float x, float y, float z, float m)
{
    reinterpret_cast<float4*>(jsrc)[i] = make_float4(x, y, z, m);
}
__device__ __forceinline__ void stage_record(void* jsrc, int64_t i, double x, double y, double z, double m)
{
    reinterpret_cast<double4*>(jsrc)[i] = make_double4(x, y, z, m);
}

__device__ __forceinline__ float pad_pos(float) { return PAD_POS_F32; }
__device__ __forceinline__ double pad_pos(double) { return PAD_POS_F64; }

// Particle i of the count particles that posm, vel, acc address (global index lo + i); i >= count pads the staged tail
// when this call owns it.  Returns "this particle's mass differs from the first one's" (equal-mass flags).
template <typename T, bool REDUCE>
__device__ __forceinline__ int step_particle(typename Vec4<T>::type* __restrict__ posm, typename Vec4<T>::type* __restrict__ vel,
                                             typename Vec4<T>::type* __restrict__ acc, void* __restrict__ jsrc,
                                             const double* __restrict__ partials, const PairPlan& plan, const T G,
                                             const PotParams<T>& pot, const T dt, const int flags,
                                             typename Vec4<T>::type* __restrict__ snapshot, const int64_t lo, const int64_t count,
                                             const int64_t i)
{
    typedef typename Vec4<T>::type V4;
    const bool staging = (flags & (STEP_OPEN | STEP_PACK_ONLY)) != 0;
    const bool flagging = staging && !(flags & STEP_SLICE);
    const bool records = !(flags & STEP_NO_STAGE);                      // the pair kernel reads posm itself otherwise (plan.direct)
    int mass_differs = 0;
    if (i < count) {
        const T mass0 = reinterpret_cast<const T*>(posm)[3];            // masses are never modified
        V4 p = posm[i];
        if (flags & STEP_PACK_ONLY) {
            if (records) stage_record(jsrc, lo + i, p.x, p.y, p.z, p.w);
        } else {
            T apx, apy, apz;
            if (REDUCE) {
                // fixed order: the S rows of this i-block in increasing s, then the factors left out of the rows
                const double gm = (double)G * plan_row_mass<T>(jsrc, plan, plan.direct ? (const void*)posm : (const void*)jsrc);   // loads in flight with the rows'
                double sum[3];
                reduce_unit_rows<3>(partials, plan, i, sum);
                const double sx = sum[0], sy = sum[1], sz = sum[2];
                apx = (T)(gm * sx);
                apy = (T)(gm * sy);
                apz = (T)(gm * sz);
                V4 a; a.x = apx; a.y = apy; a.z = apz; a.w = (T)0;
                acc[i] = a;
            } else {
                const V4 a = acc[i];
                apx = a.x; apy = a.y; apz = a.z;
            }
            if (flags & (STEP_CLOSE | STEP_OPEN | STEP_SNAPSHOT)) {
                T ex, ey, ez;
                ext_accel<T>(pot, p.x, p.y, p.z, ex, ey, ez);
                const T tx = apx + ex, ty = apy + ey, tz = apz + ez;
                const T h = (T)0.5 * dt;
                V4 v = vel[i];
                if (flags & STEP_CLOSE) {
                    v.x = fma(tx, h, v.x); v.y = fma(ty, h, v.y); v.z = fma(tz, h, v.z);
                }
                if (snapshot) {
                    // tape of the reverse-mode derivative (odisseo_leapfrog_kdk_tape_*): the synchronised state
                    // {x_k, v_k, pair-only a_k} between the closing kick of step k - 1 and the opening kick of step k
                    V4 vs = v; vs.w = (T)0;
                    V4 as; as.x = apx; as.y = apy; as.z = apz; as.w = (T)0;
                    snapshot[i] = p;
                    snapshot[plan.n + i] = vs;
                    snapshot[2 * plan.n + i] = as;
                }
                if (flags & STEP_OPEN) {
                    v.x = fma(tx, h, v.x); v.y = fma(ty, h, v.y); v.z = fma(tz, h, v.z);
                    p.x = fma(v.x, dt, p.x); p.y = fma(v.y, dt, p.y); p.z = fma(v.z, dt, p.z);
                    if (i == 0) {
                        // every thread of the launch reads the mass word of record 0 (mass0 above, plan_row_mass): its
                        // owner stores the position words only, so that word is never written while others read it
                        T* const p0 = reinterpret_cast<T*>(posm);
                        p0[0] = p.x; p0[1] = p.y; p0[2] = p.z;
                    } else {
                        posm[i] = p;
                    }
                    if (records) stage_record(jsrc, lo + i, p.x, p.y, p.z, p.w);
                }
                v.w = (T)0;
                vel[i] = v;
            }
        }
        if (flagging) mass_differs = !(p.w == mass0);               // NaN counts as different
    } else if (staging && records && lo + count == plan.n && lo + i < plan_npad(plan)) {
        const T far = pad_pos((T)0);                                    // whoever holds the last particle pads the tail
        stage_record(jsrc, lo + i, far, far, far, (T)0);
    }
    return mass_differs;
}

}  // namespace odisseo
