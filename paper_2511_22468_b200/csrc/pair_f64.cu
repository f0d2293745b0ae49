// fp64 all-pairs Plummer-softened acceleration (section 1).
//
// Same persistent stream-K / TMA-ring structure as pair_f32.cu; sources are plain
// {x, y, z, m} double records (32 B) copied into a zero-mass-padded staging array.
// r^-1 = (r2)^-1/2 is an fp32 MUFU.RSQ seed (relative error ~2^-22 plus the fp32 rounding of
// r2) refined by ONE third-order step  y' = y + y e (1/2 + 3/8 e),  e = 1 - r2 y^2,
// whose remainder (5/16) e^3 ~ 1e-21 is far below fp64 rounding: 5 FP64 ops instead of the
// ~20 of the library rsqrt().  The seed needs r2 inside the fp32 normal range; api.cu rejects
// eps^2 outside [1e-30, 1e30] and larger r2 saturates to a zero contribution.
// Sums are kept in fp64 registers for the whole segment (no tile flush needed).
#include "odisseo_common.cuh"

namespace odisseo {

namespace {

constexpr int STAGES = 4;

template <int IPT, int CWARPS, int MINB>
__global__ void __launch_bounds__((CWARPS + 1) * 32, MINB)
pair_f64_kernel(const double4* __restrict__ posm, const double4* __restrict__ jsrc, double* __restrict__ partials,
                const PairPlan plan, const double eps2)
{
    constexpr int CTHREADS = CWARPS * 32;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[STAGES];
    __shared__ __align__(8) uint64_t empty_bar[STAGES];

    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    const int lane = tid & 31;
    const int64_t c = blockIdx.x;
    const int64_t u0 = plan_start(plan, c);
    const int64_t u1 = plan_start(plan, c + 1);
    if (u0 >= u1) return;

    const uint32_t tile_bytes = (uint32_t)plan.T * 32u;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], CWARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp == CWARPS) {
        if (lane == 0) {
            int s = 0;
            uint32_t ph = 0;
            int32_t t = (int32_t)(u0 % plan.J);
            for (int64_t u = u0; u < u1; ++u) {
                mbar_wait(&empty_bar[s], ph ^ 1u);
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
                i = i < plan.n ? i : plan.n - 1;
                const double4 p = posm[i];
                xi[k] = p.x; yi[k] = p.y; zi[k] = p.z;
                ax[k] = ay[k] = az[k] = 0.0;
            }
            seg_start = false;
        }

        mbar_wait(&full_bar[s], ph);
        const double4* __restrict__ tile = reinterpret_cast<const double4*>(smem_raw + (size_t)s * tile_bytes);
#pragma unroll 2
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
                const double y0 = (double)rsqrt_approx((float)r2);
                const double e = fma(-r2 * y0, y0, 1.0);
                const double y = fma(y0 * e, fma(0.375, e, 0.5), y0);
                const double w = (y * y) * (q.w * y);
                ax[k] = fma(w, dx, ax[k]);
                ay[k] = fma(w, dy, ay[k]);
                az[k] = fma(w, dz, az[k]);
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
                row[r] = ax[k];
                row[plan.IB + r] = ay[k];
                row[2 * plan.IB + r] = az[k];
            }
            seg_start = true;
        }
        if (++t == plan.J) { t = 0; ++b; }
    }
}

template <int IPT, int CWARPS, int MINB>
cudaError_t launch_variant(const PairPlan& plan, const double* posm, const void* jsrc, double* partials, double eps,
                           cudaStream_t stream)
{
    const size_t smem = (size_t)STAGES * plan.T * 32;
    pair_f64_kernel<IPT, CWARPS, MINB><<<plan.P, (CWARPS + 1) * 32, smem, stream>>>(
        reinterpret_cast<const double4*>(posm), reinterpret_cast<const double4*>(jsrc), partials, plan, eps * eps);
    return cudaGetLastError();
}

}  // namespace

cudaError_t configure_pair_f64()
{
    cudaError_t e = cudaFuncSetAttribute(pair_f64_kernel<4, 8, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         STAGES * 256 * 32);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(pair_f64_kernel<2, 2, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                STAGES * 256 * 32);
}

cudaError_t launch_pair_f64(const PairPlan& plan, const double* posm, const void* jsrc, double* partials, double eps,
                            cudaStream_t stream)
{
    if (plan.variant == 0) return launch_variant<4, 8, 2>(plan, posm, jsrc, partials, eps, stream);
    return launch_variant<2, 2, 8>(plan, posm, jsrc, partials, eps, stream);
}

}  // namespace odisseo
