// Reverse-mode derivative of the batched small-N ensembles (SURVEY.md 8f NEXT-2 + NEXT-3): the gradient of a
// loss of the final state of EVERY simulation of a batch with respect to its own initial conditions, masses,
// potential parameters, G, eps and dt, one CTA per simulation, the whole backward time loop in one kernel.
// This is the shape of the paper's gradient-descent stage: 10 gradient steps for each of 1,000 bootstrap
// resamples, every one an N = 1,000, 1,000-step simulation differentiated with respect to
// Theta = (t_end, M_Plummer, M_NFW, M_MN) (Fig. 2 steps 5-6, L47, L53).
//
// The forward ensemble kernel (ensemble.cu) records {posm, vel, total acceleration} per step; this kernel walks
// the tape backwards with the recursion of adjoint.cu's header.  Per step a thread reloads its NQ particles'
// snapshot, forms the cotangent w_k Lv, stages {x, m} and {c} of its particles into shared memory, runs the
// O(n^2) pair pull-back over all staged sources (vjp_pair_term, two-level fp32 sums in 512-source tiles),
// adds the fp64 external-potential pull-back, and updates Lx, Lv, the mass gradients and its share of the
// parameter sums in registers; one fixed-shape block sum per parameter at the very end.  Two __syncthreads per step.
#include "adjoint_terms.cuh"

namespace odisseo {

namespace {

constexpr int EVJP_TILE = 512;

template <int NQ, bool EG>
__global__ void __launch_bounds__(VJP_THREADS, NQ <= 2 ? 2 : 1)
ensemble_vjp_kernel(const float4* __restrict__ tape, const EnsembleParams64* __restrict__ params, const int shared_params,
                    const int n, const int64_t nsteps, float4* __restrict__ lx, float4* __restrict__ lv,
                    double* __restrict__ gm_out, double* __restrict__ gparams, const int accumulate)
{
    extern __shared__ __align__(16) unsigned char evjp_smem[];
    constexpr int n_pad = NQ * VJP_THREADS;
    float4* const sp = reinterpret_cast<float4*>(evjp_smem);            // {x, y, z, m}
    float4* const sc = sp + n_pad;                                      // {cx, cy, cz, 0}
    float* const soa = reinterpret_cast<float*>(sc + n_pad);            // x[], y[], z[], cx[], cy[], cz[] (packed loop)
    __shared__ double warp_scratch[VJP_THREADS / 32];
    const int tid = threadIdx.x;
    const int64_t sim = blockIdx.x;
    const EnsembleParams64 prm = params[shared_params ? 0 : sim];
    const float4* const T0 = tape + (size_t)sim * (size_t)(nsteps + 1) * 3 * n;
    float4* const LX = lx + sim * n;
    float4* const LV = lv + sim * n;
    const float dt = (float)prm.dt, eps2 = (float)(prm.eps * prm.eps);
    const float hdt = 0.5f * dt;

    float Lx[NQ][3], Lv[NQ][3], an[NQ][3];                              // an = a_{k+1} of the previous iteration
    double gm[NQ], gp[VJP_NOUT];
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int i = q * VJP_THREADS + tid;
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
        if (i < n) { a = LX[i]; b = LV[i]; }
        Lx[q][0] = a.x; Lx[q][1] = a.y; Lx[q][2] = a.z;
        Lv[q][0] = b.x; Lv[q][1] = b.y; Lv[q][2] = b.z;
        an[q][0] = an[q][1] = an[q][2] = 0.f;
        gm[q] = 0.0;
    }
#pragma unroll
    for (int k = 0; k < VJP_NOUT; ++k) gp[k] = 0.0;

    // equal masses (checked once on snapshot 0; masses never change): the mass leaves the pair loop
    int differs = 0;
    const float mass0 = T0[0].w;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int i = q * VJP_THREADS + tid;
        if (i < n) differs |= !(T0[i].w == mass0);
    }
    const bool eqm = __syncthreads_or(differs) == 0;

    for (int64_t k = nsteps; k >= 0 && nsteps > 0; --k) {
        const float4* const S = T0 + (size_t)k * 3 * n;
        const bool first = k == nsteps;
        const float w = (first || k == 0) ? hdt : dt;
        float xs[NQ][4], cs[NQ][3];
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const int i = q * VJP_THREADS + tid;
            // slots beyond n: massless, zero cotangent, parked so far away that f and g underflow to exactly 0
            // (the equal-mass loop does not multiply by m_j)
            float4 p = make_float4(PAD_POS_F32, PAD_POS_F32, PAD_POS_F32, 0.f), v = make_float4(0.f, 0.f, 0.f, 0.f), a = v;
            if (i < n) { p = __ldcs(S + i); v = __ldcs(S + n + i); a = __ldcs(S + 2 * n + i); }
            if (!first) {
                // dL/ddt terms and Lv_k = Lv_{k+1} + dt Lx_{k+1}   (vh_k = v_k + dt/2 a_k as in the forward kernel)
                const float vhx = fmaf(a.x, hdt, v.x), vhy = fmaf(a.y, hdt, v.y), vhz = fmaf(a.z, hdt, v.z);
                double d = (double)Lx[q][0] * vhx + (double)Lx[q][1] * vhy + (double)Lx[q][2] * vhz
                         + 0.5 * ((double)Lv[q][0] * an[q][0] + (double)Lv[q][1] * an[q][1] + (double)Lv[q][2] * an[q][2]);
                Lv[q][0] = fmaf(dt, Lx[q][0], Lv[q][0]); Lv[q][1] = fmaf(dt, Lx[q][1], Lv[q][1]); Lv[q][2] = fmaf(dt, Lx[q][2], Lv[q][2]);
                d += 0.5 * ((double)Lv[q][0] * a.x + (double)Lv[q][1] * a.y + (double)Lv[q][2] * a.z);
                gp[7] += d;
            }
            an[q][0] = a.x; an[q][1] = a.y; an[q][2] = a.z;
            xs[q][0] = p.x; xs[q][1] = p.y; xs[q][2] = p.z; xs[q][3] = p.w;
            cs[q][0] = w * Lv[q][0]; cs[q][1] = w * Lv[q][1]; cs[q][2] = w * Lv[q][2];
            if (eqm && !EG) {                                          // structure of arrays: LDS.64 = two sources
                soa[i] = p.x; soa[n_pad + i] = p.y; soa[2 * n_pad + i] = p.z;
                soa[3 * n_pad + i] = cs[q][0]; soa[4 * n_pad + i] = cs[q][1]; soa[5 * n_pad + i] = cs[q][2];
            } else {
                sp[i] = p;
                sc[i] = make_float4(cs[q][0], cs[q][1], cs[q][2], 0.f);
            }
        }
        __syncthreads();                                               // sources staged
        float o[NQ][VJP_COMPS];                                        // n <= 2,048: two-level fp32 sums suffice
#pragma unroll
        for (int q = 0; q < NQ; ++q)
#pragma unroll
            for (int c = 0; c < VJP_COMPS; ++c) o[q][c] = 0.f;
        for (int j0 = 0; j0 < n_pad && n > 1; j0 += EVJP_TILE) {          // n == 1: no pairs (orbit mode)
            float t[NQ][VJP_COMPS];
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int c = 0; c < VJP_COMPS; ++c) t[q][c] = 0.f;
            const int j1 = j0 + EVJP_TILE < n_pad ? j0 + EVJP_TILE : n_pad;
            if (eqm && !EG) {
                // packed loop: two sources per instruction, the target duplicated in both halves
                const f32x2 e2 = pk(eps2, eps2), m3 = pk(-3.0f, -3.0f);
                f32x2 X[NQ], Y[NQ], Z[NQ], CX[NQ], CY[NQ], CZ[NQ], a2[NQ][4];
#pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    X[q] = pk(xs[q][0], xs[q][0]); Y[q] = pk(xs[q][1], xs[q][1]); Z[q] = pk(xs[q][2], xs[q][2]);
                    CX[q] = pk(cs[q][0], cs[q][0]); CY[q] = pk(cs[q][1], cs[q][1]); CZ[q] = pk(cs[q][2], cs[q][2]);
                    a2[q][0] = a2[q][1] = a2[q][2] = a2[q][3] = 0ull;
                }
                const f32x2* const s2 = reinterpret_cast<const f32x2*>(soa);
                constexpr int H = n_pad / 2;                            // f32x2 elements per array
#pragma unroll 2
                for (int j = j0 / 2; j < j1 / 2; ++j) {
                    const f32x2 px = s2[j], py = s2[H + j], pz = s2[2 * H + j];
                    const f32x2 qx = s2[3 * H + j], qy = s2[4 * H + j], qz = s2[5 * H + j];
#pragma unroll
                    for (int q = 0; q < NQ; ++q)
                        vjp_pair_term_x2(px, py, pz, qx, qy, qz, X[q], Y[q], Z[q], CX[q], CY[q], CZ[q], e2, m3, a2[q][0], a2[q][1],
                                         a2[q][2], a2[q][3]);
                }
#pragma unroll
                for (int q = 0; q < NQ; ++q)
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        float lo, hi;
                        unpk(a2[q][c], lo, hi);
                        t[q][c] = lo + hi;
                    }
            } else {
#pragma unroll 4
                for (int j = j0; j < j1; ++j) {
                    const float4 p = sp[j], c = sc[j];
#pragma unroll
                    for (int q = 0; q < NQ; ++q)
                        vjp_pair_term<float, false, EG>(p.x, p.y, p.z, p.w, c.x, c.y, c.z, xs[q][0], xs[q][1], xs[q][2], xs[q][3],
                                                        cs[q][0], cs[q][1], cs[q][2], eps2, t[q][0], t[q][1], t[q][2], t[q][3],
                                                        t[q][4], t[q][5]);
                }
            }
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int c = 0; c < VJP_COMPS; ++c) o[q][c] += t[q][c];
        }
        __syncthreads();                                               // sources consumed
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            if (q * VJP_THREADS + tid < n) {
                double h[3], t6[8];
                ext_vjp(prm.pot, prm.G, (double)xs[q][0], (double)xs[q][1], (double)xs[q][2], (double)cs[q][0], (double)cs[q][1],
                        (double)cs[q][2], h, t6);
                const double gscale = (eqm && !EG) ? prm.G * (double)mass0 : prm.G;   // the equal-mass loop left m out
                Lx[q][0] = (float)((double)Lx[q][0] + fma(gscale, (double)o[q][0], h[0]));
                Lx[q][1] = (float)((double)Lx[q][1] + fma(gscale, (double)o[q][1], h[1]));
                Lx[q][2] = (float)((double)Lx[q][2] + fma(gscale, (double)o[q][2], h[2]));
                gm[q] += -prm.G * (double)o[q][3];
#pragma unroll
                for (int c = 0; c < 5; ++c) gp[c] += t6[c];
                gp[8] += t6[6];
                gp[9] += t6[7];
                if (EG) {
                    gp[5] += t6[5] + (double)o[q][5];
                    gp[6] += prm.eps * prm.G * (double)o[q][4];
                }
            }
        }
    }

#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int i = q * VJP_THREADS + tid;
        if (i < n) {
            LX[i] = make_float4(Lx[q][0], Lx[q][1], Lx[q][2], 0.f);
            LV[i] = make_float4(Lv[q][0], Lv[q][1], Lv[q][2], 0.f);
            gm_out[sim * n + i] = accumulate ? gm_out[sim * n + i] + gm[q] : gm[q];
        }
    }
#pragma unroll
    for (int k = 0; k < VJP_NOUT; ++k) {
        const double tot = vjp_block_sum(gp[k], warp_scratch);
        if (tid == 0) gparams[sim * VJP_NOUT + k] = accumulate ? gparams[sim * VJP_NOUT + k] + tot : tot;
    }
}

template <int NQ, bool EG>
cudaError_t launch_evjp(const float* tape, const EnsembleParams64* params, int shared_params, int n, int64_t nsim,
                        int64_t nsteps, float* lx, float* lv, double* gm, double* gparams, int accumulate, cudaStream_t stream)
{
    const size_t smem = (size_t)NQ * VJP_THREADS * (32 + 24);
    cudaError_t e = cudaFuncSetAttribute(ensemble_vjp_kernel<NQ, EG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    ensemble_vjp_kernel<NQ, EG><<<(unsigned)nsim, VJP_THREADS, smem, stream>>>(
        reinterpret_cast<const float4*>(tape), params, shared_params, n, nsteps, reinterpret_cast<float4*>(lx),
        reinterpret_cast<float4*>(lv), gm, gparams, accumulate);
    return cudaGetLastError();
}

}  // namespace

template <bool EG>
static cudaError_t dispatch_evjp(const float* tape, const EnsembleParams64* params, int shared_params, int n, int64_t nsim,
                                 int64_t nsteps, float* lx, float* lv, double* gm, double* gparams, int accumulate, cudaStream_t stream)
{
    switch ((n + VJP_THREADS - 1) / VJP_THREADS) {
        case 1: return launch_evjp<1, EG>(tape, params, shared_params, n, nsim, nsteps, lx, lv, gm, gparams, accumulate, stream);
        case 2: return launch_evjp<2, EG>(tape, params, shared_params, n, nsim, nsteps, lx, lv, gm, gparams, accumulate, stream);
        case 3: return launch_evjp<3, EG>(tape, params, shared_params, n, nsim, nsteps, lx, lv, gm, gparams, accumulate, stream);
        case 4: return launch_evjp<4, EG>(tape, params, shared_params, n, nsim, nsteps, lx, lv, gm, gparams, accumulate, stream);
        case 5: return launch_evjp<5, EG>(tape, params, shared_params, n, nsim, nsteps, lx, lv, gm, gparams, accumulate, stream);
        case 6: return launch_evjp<6, EG>(tape, params, shared_params, n, nsim, nsteps, lx, lv, gm, gparams, accumulate, stream);
        case 7: return launch_evjp<7, EG>(tape, params, shared_params, n, nsim, nsteps, lx, lv, gm, gparams, accumulate, stream);
        default: return launch_evjp<8, EG>(tape, params, shared_params, n, nsim, nsteps, lx, lv, gm, gparams, accumulate, stream);
    }
}

cudaError_t launch_ensemble_vjp_f32(const float* tape, const EnsembleParams64* params, int shared_params, int n,
                                    int64_t nsim, int64_t nsteps, int with_eps_G, float* lx, float* lv, double* gm,
                                    double* gparams, int accumulate, cudaStream_t stream)
{
    if (with_eps_G) return dispatch_evjp<true>(tape, params, shared_params, n, nsim, nsteps, lx, lv, gm, gparams, accumulate, stream);
    return dispatch_evjp<false>(tape, params, shared_params, n, nsim, nsteps, lx, lv, gm, gparams, accumulate, stream);
}

}  // namespace odisseo
