// Batched small-N ensembles: many independent simulations of n <= 2,048 particles,
// each advanced nsteps KDK steps by ONE CTA with the whole time loop inside one kernel.
//
// This is the workload the paper's inference actually runs: a 10^4-point grid search plus bootstrap
// resamples, every point an N = 1,000, 1,000-step simulation with its own potential masses, progenitor
// mass and integration time (Fig. 2, L47, L53 section 2.2.1).  One simulation per launch is
// launch-bound there (~12 us per step at N = 1,024 against 0.4 us of arithmetic); here a simulation's
// state never leaves the SM:
//   * positions, velocities and masses of a thread's targets live in registers as packed f32x2 pairs
//     (thread t owns particles (2p+h)*256 + t);
//   * after every drift each thread re-stages its own particles into the CTA's shared-memory source
//     array as plain {x, y, z, m} records (the layout of pair_f32.cu: one LDS.128 per source, the coordinate a
//     scalar broadcast operand of the packed instructions), so the inner loop is the same 3 FADD2 + 6 FFMA2 +
//     3 FMUL2 + 2 MUFU.RSQ per two interactions (2 FMUL2 for equal masses, detected per simulation);
//   * two __syncthreads per step (sources staged / sources consumed), no global traffic in the loop;
//   * two-level fp32 summation: 512-source tiles, tile sums added in tile order (n <= 2,048, so the
//     single-accumulator stagnation of SURVEY.md section 0 cannot occur).
// Per-simulation parameters (G, eps, dt, NFW, MN) come from a device array written by the C ABI.
#include "odisseo_common.cuh"
#include "ext_potential.cuh"

namespace odisseo {

namespace {

constexpr int ENS_THREADS = 256;
constexpr int ENS_TILE = 512;

// One pass of a thread's NPAIR target pairs over sources [j0, j0 + ENS_TILE) of the staged array.
template <int NPAIR, bool EQM>
__device__ __forceinline__ void ens_tile(const float4* __restrict__ src, const int j0, const f32x2 e2,
                                         const f32x2 (&xi)[NPAIR], const f32x2 (&yi)[NPAIR], const f32x2 (&zi)[NPAIR],
                                         f32x2 (&ax)[NPAIR], f32x2 (&ay)[NPAIR], f32x2 (&az)[NPAIR])
{
#pragma unroll 8
    for (int j = j0; j < j0 + ENS_TILE; ++j) {
        // one LDS.128 per source {x, y, z, m}; the splats are scalar broadcast operands of the packed ops (pair_f32.cu)
        const float4 q = src[j];
        const f32x2 qx = pk(q.x, q.x), qy = pk(q.y, q.y), qz = pk(q.z, q.z), qm = pk(q.w, q.w);
#pragma unroll
        for (int p = 0; p < NPAIR; ++p) {
            const f32x2 dx = sub2(qx, xi[p]);
            const f32x2 dy = sub2(qy, yi[p]);
            const f32x2 dz = sub2(qz, zi[p]);
            f32x2 r2 = fma2(dx, dx, e2);
            r2 = fma2(dy, dy, r2);
            r2 = fma2(dz, dz, r2);
            float r2l, r2h;
            unpk(r2, r2l, r2h);
            const f32x2 ri = pk(rsqrt_approx(r2l), rsqrt_approx(r2h));
            const f32x2 ri2 = mul2(ri, ri);
            const f32x2 w = mul2(ri2, EQM ? ri : mul2(qm, ri));
            ax[p] = fma2(w, dx, ax[p]);
            ay[p] = fma2(w, dy, ay[p]);
            az[p] = fma2(w, dz, az[p]);
        }
    }
}

// a_pair of the thread's targets from the staged sources: G * (m0 *) sum over tiles, tile order.
template <int NPAIR, bool EQM>
__device__ __forceinline__ void ens_pair(const float4* __restrict__ src, const int n_pad, const float eps2,
                                         const float scale, const f32x2 (&xi)[NPAIR], const f32x2 (&yi)[NPAIR],
                                         const f32x2 (&zi)[NPAIR], f32x2 (&gx)[NPAIR], f32x2 (&gy)[NPAIR],
                                         f32x2 (&gz)[NPAIR])
{
    const f32x2 e2 = pk(eps2, eps2);
    const f32x2 nz = pk(-0.0f, -0.0f);
    f32x2 tx[NPAIR], ty[NPAIR], tz[NPAIR];
#pragma unroll
    for (int p = 0; p < NPAIR; ++p) tx[p] = ty[p] = tz[p] = 0ull;
    for (int j0 = 0; j0 < n_pad; j0 += ENS_TILE) {
        f32x2 ax[NPAIR], ay[NPAIR], az[NPAIR];
#pragma unroll
        for (int p = 0; p < NPAIR; ++p) ax[p] = ay[p] = az[p] = 0ull;
        ens_tile<NPAIR, EQM>(src, j0, e2, xi, yi, zi, ax, ay, az);
#pragma unroll
        for (int p = 0; p < NPAIR; ++p) {
            tx[p] = add2(tx[p], ax[p]);
            ty[p] = add2(ty[p], ay[p]);
            tz[p] = add2(tz[p], az[p]);
        }
    }
    const f32x2 s2 = pk(scale, scale);
#pragma unroll
    for (int p = 0; p < NPAIR; ++p) {
        gx[p] = fma2(tx[p], s2, nz);
        gy[p] = fma2(ty[p], s2, nz);
        gz[p] = fma2(tz[p], s2, nz);
    }
}

// THREADS x 2 NPAIR target slots per simulation.
template <int NPAIR, int THREADS>
__global__ void __launch_bounds__(THREADS, NPAIR <= 2 ? 2 : 1)
ensemble_kdk_kernel(float4* __restrict__ posm, float4* __restrict__ vel, const EnsembleParams* __restrict__ params,
                    const int shared_params, const int n, const int64_t nsteps, float4* __restrict__ tape)
{
    extern __shared__ __align__(16) unsigned char ens_smem[];
    float4* const stage4 = reinterpret_cast<float4*>(ens_smem);
    const float4* const src = reinterpret_cast<const float4*>(ens_smem);
    constexpr int n_pad = 2 * NPAIR * THREADS;
    const int tid = threadIdx.x;
    const int64_t sim = blockIdx.x;
    const EnsembleParams prm = params[shared_params ? 0 : sim];
    float4* const P = posm + sim * n;
    float4* const V = vel + sim * n;

    // ---- load the thread's targets; slots beyond n are massless records parked far away ----------
    f32x2 xi[NPAIR], yi[NPAIR], zi[NPAIR], mi[NPAIR], vx[NPAIR], vy[NPAIR], vz[NPAIR];
    const float mass0 = P[0].w;
    int differs = 0;
#pragma unroll
    for (int p = 0; p < NPAIR; ++p) {
        float4 q[2], w[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int i = (2 * p + h) * THREADS + tid;
            if (i < n) {
                q[h] = P[i];
                w[h] = V[i];
                differs |= !(q[h].w == mass0);
            } else {
                q[h] = make_float4(PAD_POS_F32, PAD_POS_F32, PAD_POS_F32, 0.0f);
                w[h] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            }
        }
        const f32x2 nz = pk(-0.0f, -0.0f);             // native 64-bit pairs (see pair_f32.cu)
        xi[p] = add2(pk(q[0].x, q[1].x), nz);
        yi[p] = add2(pk(q[0].y, q[1].y), nz);
        zi[p] = add2(pk(q[0].z, q[1].z), nz);
        mi[p] = pk(q[0].w, q[1].w);
        vx[p] = pk(w[0].x, w[1].x);
        vy[p] = pk(w[0].y, w[1].y);
        vz[p] = pk(w[0].z, w[1].z);
    }
    const bool eqm = __syncthreads_or(differs) == 0;

    // total acceleration of the thread's targets at the current positions
    f32x2 gx[NPAIR], gy[NPAIR], gz[NPAIR];
    auto accel = [&]() {
#pragma unroll
        for (int p = 0; p < NPAIR; ++p) {
            float x0, x1, y0, y1, z0, z1, m0, m1;
            unpk(xi[p], x0, x1); unpk(yi[p], y0, y1); unpk(zi[p], z0, z1); unpk(mi[p], m0, m1);
            const int i0 = (2 * p) * THREADS + tid, i1 = i0 + THREADS;
            stage4[i0] = make_float4(x0, y0, z0, m0);
            stage4[i1] = make_float4(x1, y1, z1, m1);
        }
        __syncthreads();                                   // sources staged
        if (n == 1) {
            // a single particle feels only the external potential (its softened self term is exactly 0): the orbit
            // mode of the paper's pipeline (backward integration of the centre of mass, PAPER.md:L43 step 2; orbit
            // fitting, L57) skips the pair loop
#pragma unroll
            for (int p = 0; p < NPAIR; ++p) gx[p] = gy[p] = gz[p] = 0ull;
        } else if (eqm) ens_pair<NPAIR, true>(src, n_pad, prm.eps2, prm.G * mass0, xi, yi, zi, gx, gy, gz);
        else            ens_pair<NPAIR, false>(src, n_pad, prm.eps2, prm.G, xi, yi, zi, gx, gy, gz);
        __syncthreads();                                   // sources consumed: the next drift may overwrite them
        if (prm.pot.GMs != 0.0f || prm.pot.GMd != 0.0f) {
#pragma unroll
            for (int p = 0; p < NPAIR; ++p) {
                float x0, x1, y0, y1, z0, z1, a0, a1, b0, b1, c0, c1;
                unpk(xi[p], x0, x1); unpk(yi[p], y0, y1); unpk(zi[p], z0, z1);
                unpk(gx[p], a0, a1); unpk(gy[p], b0, b1); unpk(gz[p], c0, c1);
                float ex, ey, ez;
                if ((2 * p) * THREADS + tid < n) {
                    ext_accel<float>(prm.pot, x0, y0, z0, ex, ey, ez);
                    a0 += ex; b0 += ey; c0 += ez;
                }
                if ((2 * p + 1) * THREADS + tid < n) {
                    ext_accel<float>(prm.pot, x1, y1, z1, ex, ey, ez);
                    a1 += ex; b1 += ey; c1 += ez;
                }
                gx[p] = pk(a0, a1); gy[p] = pk(b0, b1); gz[p] = pk(c0, c1);
            }
        }
    };

    // optional tape for the reverse-mode derivative (ensemble_adjoint.cu): snapshot k of this simulation =
    // {posm, vel, TOTAL acceleration} at the synchronised time t0 + k dt, (nsteps + 1) x 3 x n records
    float4* const T0 = tape ? tape + (size_t)sim * (size_t)(nsteps + 1) * 3 * n : nullptr;
    auto record = [&](const int64_t k) {
        if (!T0) return;
        float4* const S = T0 + (size_t)k * 3 * n;
#pragma unroll
        for (int p = 0; p < NPAIR; ++p) {
            float x[2], y[2], z[2], m[2], a[2], b[2], c[2], ga[2], gb[2], gc[2];
            unpk(xi[p], x[0], x[1]); unpk(yi[p], y[0], y[1]); unpk(zi[p], z[0], z[1]); unpk(mi[p], m[0], m[1]);
            unpk(vx[p], a[0], a[1]); unpk(vy[p], b[0], b[1]); unpk(vz[p], c[0], c[1]);
            unpk(gx[p], ga[0], ga[1]); unpk(gy[p], gb[0], gb[1]); unpk(gz[p], gc[0], gc[1]);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int i = (2 * p + h) * THREADS + tid;
                if (i < n) {
                    S[i] = make_float4(x[h], y[h], z[h], m[h]);
                    S[n + i] = make_float4(a[h], b[h], c[h], 0.0f);
                    S[2 * n + i] = make_float4(ga[h], gb[h], gc[h], 0.0f);
                }
            }
        }
    };

    // ---- KDK: a <- a(x); repeat { v += a dt/2; x += v dt; a <- a(x); v += a dt/2 } ----
    const float hdt = 0.5f * prm.dt;
    const f32x2 h2 = pk(hdt, hdt), d2 = pk(prm.dt, prm.dt);
    accel();
    record(0);
    for (int64_t s = 0; s < nsteps; ++s) {
#pragma unroll
        for (int p = 0; p < NPAIR; ++p) {
            vx[p] = fma2(gx[p], h2, vx[p]); vy[p] = fma2(gy[p], h2, vy[p]); vz[p] = fma2(gz[p], h2, vz[p]);
            xi[p] = fma2(vx[p], d2, xi[p]); yi[p] = fma2(vy[p], d2, yi[p]); zi[p] = fma2(vz[p], d2, zi[p]);
        }
        accel();
#pragma unroll
        for (int p = 0; p < NPAIR; ++p) {
            vx[p] = fma2(gx[p], h2, vx[p]); vy[p] = fma2(gy[p], h2, vy[p]); vz[p] = fma2(gz[p], h2, vz[p]);
        }
        record(s + 1);
    }

#pragma unroll
    for (int p = 0; p < NPAIR; ++p) {
        float x[2], y[2], z[2], m[2], a[2], b[2], c[2];
        unpk(xi[p], x[0], x[1]); unpk(yi[p], y[0], y[1]); unpk(zi[p], z[0], z[1]); unpk(mi[p], m[0], m[1]);
        unpk(vx[p], a[0], a[1]); unpk(vy[p], b[0], b[1]); unpk(vz[p], c[0], c[1]);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int i = (2 * p + h) * THREADS + tid;
            if (i < n) {
                P[i] = make_float4(x[h], y[h], z[h], m[h]);
                V[i] = make_float4(a[h], b[h], c[h], 0.0f);
            }
        }
    }
}

template <int NPAIR, int THREADS>
cudaError_t launch_ens(float* posm, float* vel, const EnsembleParams* params, int shared_params, int n, int64_t nsim,
                       int64_t nsteps, float* tape, cudaStream_t stream)
{
    static_assert((2 * NPAIR * THREADS) % ENS_TILE == 0, "whole source tiles");
    const size_t smem = (size_t)2 * NPAIR * THREADS * 16;
    cudaError_t e = cudaFuncSetAttribute(ensemble_kdk_kernel<NPAIR, THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    ensemble_kdk_kernel<NPAIR, THREADS><<<(unsigned)nsim, THREADS, smem, stream>>>(
        reinterpret_cast<float4*>(posm), reinterpret_cast<float4*>(vel), params, shared_params, n, nsteps,
        reinterpret_cast<float4*>(tape));
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_ensemble_f32(float* posm, float* vel, const EnsembleParams* params, int shared_params, int n,
                                int64_t nsim, int64_t nsteps, float* tape, cudaStream_t stream)
{
    // (128 threads x 8 targets, the pair kernel's register tile, measured no faster: 2.45-2.49 against 2.51 M simulation-steps/s)
    if (n <= 1 * ENS_TILE) return launch_ens<1, 256>(posm, vel, params, shared_params, n, nsim, nsteps, tape, stream);
    if (n <= 2 * ENS_TILE) return launch_ens<2, 256>(posm, vel, params, shared_params, n, nsim, nsteps, tape, stream);
    if (n <= 3 * ENS_TILE) return launch_ens<3, 256>(posm, vel, params, shared_params, n, nsim, nsteps, tape, stream);
    return launch_ens<4, 256>(posm, vel, params, shared_params, n, nsim, nsteps, tape, stream);
}

}  // namespace odisseo
