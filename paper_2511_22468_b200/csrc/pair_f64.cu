// fp64 all-pairs Plummer-softened acceleration (section 1).
//
// Same persistent stream-K / TMA-ring structure as pair_f32.cu; sources are plain
// {x, y, z, m} double records (32 B) copied into a zero-mass-padded staging array.
// (r2)^-3/2 comes from the double-precision seed y0 = rsqrt.approx.ftz.f64(r2) (MUFU.RSQ64H on the
// high word: relative error ~2^-22, low word zero, no F2F conversions) and ONE correction of the
// cube:  t = y0^2,  e = 1 - r2 t,  (r2)^-3/2 = y0^3 (1-e)^-3/2 = y0^3 (1 + e (3/2 + 15/8 e)) + O(e^3),
// remainder (35/16) e^3 ~ 2e-19: 7 FP64 ops for m (r2)^-3/2 instead of ~20 with the library rsqrt().
// 16 FP64-pipe ops + 1 MUFU per interaction (3 DADD, 9 DFMA, 4 DMUL).  A DFMA holds a scheduler's
// dispatch port 2 cycles and every other instruction 1, so F2F or integer conversions around an fp32
// seed cost as much as the arithmetic they feed.
// Sums are kept in fp64 registers for the whole segment (no tile flush needed).
#include "odisseo_common.cuh"

namespace odisseo {

namespace {

constexpr int STAGES = 4;

// Consumer side for one CTA.  EQM = all masses equal (flags from the staging kernel): the mass
// factor leaves the inner loop (15 instead of 16 FP64 ops) and multiplies the sums once per segment.
// POT = accumulate the softened potential sum_j m_j (r2)^-1/2 (x-plane of the partial rows only)
// instead of the acceleration: the O(N^2) part of odisseo_diagnostics_* (diagnostics.cu).
template <int IPT, int CWARPS, int JUNROLL, bool EQM, bool POT>
__device__ __forceinline__ void consume_tiles(const double4* __restrict__ posm, const double4* __restrict__ jsrc,
                                              double* __restrict__ partials,
                                              const PairPlan& plan, const double eps2, unsigned char* smem_raw,
                                              uint64_t* full_bar, uint64_t* empty_bar, const int64_t c,
                                              const int64_t u0, const int64_t u1, const uint32_t tile_bytes)
{
    constexpr int CTHREADS = CWARPS * 32;
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const double m0 = EQM ? jsrc[0].w : 1.0;                 // mass of staged record 0
    double xi[IPT], yi[IPT], zi[IPT], ax[IPT], ay[IPT], az[IPT];
    int32_t b = (int32_t)(u0 / plan.J);
    int32_t t = (int32_t)(u0 - (int64_t)b * plan.J);
    bool seg_start = true;
    int s = 0;
    uint32_t ph = 0;

    for (int64_t u = u0; u < u1; ++u) {
        if (seg_start) {
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                int64_t i = (int64_t)b * plan.IB + (int64_t)k * CTHREADS + tid;
                i = i < plan.nt ? i : plan.nt - 1;
                const double4 p = posm[i];
                xi[k] = p.x; yi[k] = p.y; zi[k] = p.z;
                ax[k] = ay[k] = az[k] = 0.0;
            }
            seg_start = false;
        }

        mbar_wait(&full_bar[s], ph);
        const double4* __restrict__ tile = reinterpret_cast<const double4*>(smem_raw + (size_t)s * tile_bytes);
#pragma unroll JUNROLL
        for (int j = 0; j < plan.T; ++j) {
            const double4 q = tile[j];
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                const double dx = q.x - xi[k];
                const double dy = q.y - yi[k];
                const double dz = q.z - zi[k];
                double r2 = fma(dx, dx, eps2);
                r2 = fma(dy, dy, r2);
                r2 = fma(dz, dz, r2);
                const double y0 = rsqrt_approx_f64(r2);
                const double t = y0 * y0;
                const double e = fma(-r2, t, 1.0);
                if (POT) {
                    // (r2)^-1/2 = y0 (1-e)^-1/2 = y0 (1 + e (1/2 + 3/8 e)) + O(e^3)
                    const double y = y0 * fma(e, fma(0.375, e, 0.5), 1.0);
                    ax[k] = EQM ? ax[k] + y : fma(q.w, y, ax[k]);
                } else {
                    const double c = fma(e, fma(1.875, e, 1.5), 1.0);
                    const double w = EQM ? (t * y0) * c : ((t * y0) * q.w) * c;
                    ax[k] = fma(w, dx, ax[k]);
                    ay[k] = fma(w, dy, ay[k]);
                    az[k] = fma(w, dz, az[k]);
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[s]);
        if (++s == STAGES) { s = 0; ph ^= 1u; }

        const bool seg_end = (t == plan.J - 1) || (u == u1 - 1);
        if (seg_end) {
            double* row = partials + (size_t)(c + b) * 3 * plan.IB;
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                const int r = k * CTHREADS + tid;
                row[r] = m0 * ax[k];
                if (!POT) {
                    row[plan.IB + r] = m0 * ay[k];
                    row[2 * plan.IB + r] = m0 * az[k];
                }
            }
            seg_start = true;
        }
        if (++t == plan.J) { t = 0; ++b; }
    }
}

template <int IPT, int CWARPS, int MINB, int JUNROLL, bool POT>
__global__ void __launch_bounds__((CWARPS + 1) * 32, MINB)
pair_f64_kernel(const double4* __restrict__ posm, const double4* __restrict__ jsrc, double* __restrict__ partials,
                const PairPlan plan, const double eps2)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[STAGES];
    __shared__ __align__(8) uint64_t empty_bar[STAGES];

    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    const int lane = tid & 31;
    const int64_t c = blockIdx.x;
    const int64_t u0 = plan_start(plan, c);
    const int64_t u1 = plan_start(plan, c + 1);
    // Let the next kernel become resident early only when this one is short (a few tiles per CTA): its
    // CTAs then hide their launch latency behind our tail.  Behind a long evaluation, early dependents would
    // sit on the SMs for milliseconds (measured -0.3 % at N = 262,144); there the implicit trigger at exit is used.
    if (u1 - u0 <= 16) pdl_launch_dependents();
    if (u0 >= u1) return;

    const uint32_t tile_bytes = (uint32_t)plan.T * 32u;
    if (tid == CWARPS * 32) {                               // the producer lane owns init and the first loads
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], CWARPS);
        }
        mbar_fence_init();
    }
    pdl_wait();                                             // the staging kernel's records and flags are complete
    // the first STAGES tiles need no hand-over: issue them before anything else so that their latency
    // overlaps the flag reduction and the target loads
    const int prefetch = (int)((u1 - u0) < STAGES ? (u1 - u0) : STAGES);
    if (tid == CWARPS * 32) {
        int32_t t = (int32_t)(u0 % plan.J);
        for (int s = 0; s < prefetch; ++s) {
            mbar_arrive_expect_tx(&full_bar[s], tile_bytes);
            tma_load_1d(smem_raw + (size_t)s * tile_bytes,
                        reinterpret_cast<const unsigned char*>(jsrc) + (size_t)t * tile_bytes, tile_bytes, &full_bar[s]);
            if (++t == plan.J) t = 0;
        }
    }
    int differs = 0;
    {
        const int* __restrict__ mflags = plan_flags(jsrc, plan);
        const int nflags = plan_nflags(plan);
        for (int k = tid; k < nflags; k += (CWARPS + 1) * 32) differs |= __ldg(mflags + k);
    }
    const bool eqm = __syncthreads_or(differs) == 0;        // also publishes the mbarrier inits

    if (warp == CWARPS) {
        if (lane == 0) {
            int s = prefetch % STAGES;
            uint32_t ph = prefetch == STAGES ? 1u : 0u;
            int32_t t = (int32_t)((u0 + prefetch) % plan.J);
            for (int64_t u = u0 + prefetch; u < u1; ++u) {
                mbar_wait_backoff(&empty_bar[s], ph ^ 1u);
                mbar_arrive_expect_tx(&full_bar[s], tile_bytes);
                tma_load_1d(smem_raw + (size_t)s * tile_bytes,
                            reinterpret_cast<const unsigned char*>(jsrc) + (size_t)t * tile_bytes, tile_bytes,
                            &full_bar[s]);
                if (++t == plan.J) t = 0;
                if (++s == STAGES) { s = 0; ph ^= 1u; }
            }
        }
        return;
    }

    if (eqm)
        consume_tiles<IPT, CWARPS, JUNROLL, true, POT>(posm, jsrc, partials, plan, eps2, smem_raw, full_bar, empty_bar, c, u0, u1, tile_bytes);
    else
        consume_tiles<IPT, CWARPS, JUNROLL, false, POT>(posm, jsrc, partials, plan, eps2, smem_raw, full_bar, empty_bar, c, u0, u1, tile_bytes);
}

template <int IPT, int CWARPS, int MINB, int JUNROLL, bool POT>
cudaError_t launch_variant(const PairPlan& plan, const double* posm, const void* jsrc, double* partials, double eps,
                           cudaStream_t stream)
{
    const size_t smem = (size_t)STAGES * plan.T * 32;
    return launch_pdl(pair_f64_kernel<IPT, CWARPS, MINB, JUNROLL, POT>, dim3(plan.P), dim3((CWARPS + 1) * 32), smem, stream,
                      reinterpret_cast<const double4*>(posm), reinterpret_cast<const double4*>(jsrc), partials, plan, eps * eps);
}

}  // namespace

cudaError_t configure_pair_f64()
{
    const int smem = STAGES * 256 * 32;
    cudaError_t e = cudaFuncSetAttribute(pair_f64_kernel<4, 8, 1, 4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(pair_f64_kernel<2, 2, 8, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(pair_f64_kernel<4, 8, 1, 4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(pair_f64_kernel<2, 2, 8, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
}

cudaError_t launch_pair_f64(const PairPlan& plan, const double* posm, const void* jsrc, double* partials, double eps,
                            cudaStream_t stream)
{
    if (plan.variant == 0) return launch_variant<4, 8, 1, 4, false>(plan, posm, jsrc, partials, eps, stream);
    return launch_variant<2, 2, 8, 2, false>(plan, posm, jsrc, partials, eps, stream);
}

// Softened potential sums phi'_i = sum_j m_j (r_ij^2 + eps^2)^-1/2 (self term included) into the x-plane of
// the partial rows; targets are read from the staged double records themselves.
cudaError_t launch_potential_f64(const PairPlan& plan, const void* jsrc, double* partials, double eps,
                                 cudaStream_t stream)
{
    const double* targets = static_cast<const double*>(jsrc);
    if (plan.variant == 0) return launch_variant<4, 8, 1, 4, true>(plan, targets, jsrc, partials, eps, stream);
    return launch_variant<2, 2, 8, 2, true>(plan, targets, jsrc, partials, eps, stream);
}

}  // namespace odisseo
