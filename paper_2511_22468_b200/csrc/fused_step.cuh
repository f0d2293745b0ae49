// Whole-loop persistent kernel for small and mid N (SURVEY.md 8a row a5 "decisive for configs 0-1"): at N <= 16,384 a
// KDK step is a few microseconds to ~100 us of arithmetic, and two launches per step (even graph-replayed, with
// programmatic dependent launch) cost ~8.5 us.  Here ONE cooperative launch runs all nsteps steps: the same CTAs
// alternate between the pair phase (the stream kernel's producer / consumer code on the same unit plan) and the integrate
// phase (the step kernel's per-particle body over a grid-stride loop), separated by a grid-wide barrier -- one atomic
// arrive per CTA on a counter in the workspace and a spin on it; the cooperative launch guarantees that every CTA is
// resident.  Both phases execute the very code of the two-kernel path (consume_units, step_particle) on the same plan,
// so the results are bit-identical to it (tests).  Staged records are written with ordinary stores and read by TMA
// in the next phase: writers issue fence.proxy.async before the barrier.
#pragma once

#include <type_traits>

#include "pair_stream.cuh"
#include "step_body.cuh"

namespace odisseo {

constexpr int64_t FUSED_MAX_N = 16384;

template <typename T> struct FusedArgs {
    typename Vec4<T>::type *posm, *vel, *acc;
    T G, dt;
    PotParams<T> pot;
    int64_t nsteps;
    int acc_valid;
    unsigned* barrier;      // 256-byte grid-barrier block, zeroed by the host before the launch
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }

// Grid barrier.  bar[0] counts arrivals and only grows during a launch; the CTA whose arrival completes generation g
// publishes g in bar[32] (another 128-byte line), and everybody else spins on that read-only line, so the spinning
// loads do not queue behind the arrival atomics.
__device__ __forceinline__ void grid_barrier(unsigned* bar, unsigned& generation)
{
    ++generation;
    fence_proxy_async_global();                     // this thread's staged records, for the TMA reads of the next phase
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned arrived = atomicAdd(bar, 1u) + 1u;
        if (arrived == generation * gridDim.x) {
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(bar + 32), "r"(generation) : "memory");
        } else {
            while (ld_acquire_u32(bar + 32) < generation) { }
        }
        __threadfence();
    }
    __syncthreads();
}

template <class C, typename T>
__global__ void __launch_bounds__((C::CWARPS + 1) * 32, C::MINB)
fused_kdk_kernel(const typename C::Params prm, unsigned char* __restrict__ jsrc, double* __restrict__ rows, const PairPlan plan,
                 const FusedArgs<T> fa)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[STAGES];
    __shared__ __align__(8) uint64_t empty_bar[STAGES];
    constexpr int CWARPS = C::CWARPS;
    constexpr int NTHREADS = (CWARPS + 1) * 32;
    typedef typename Vec4<T>::type V4;

    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    const int lane = tid & 31;
    const int64_t c = blockIdx.x;
    const int64_t u0 = plan_start(plan, c);
    const int64_t u1 = plan_start(plan, c + 1);
    const uint32_t stage_bytes = (uint32_t)plan.T * C::REC;
    const int64_t gtid = c * NTHREADS + tid, gsize = (int64_t)gridDim.x * NTHREADS;
    const int64_t nwork = plan.n + (plan_npad(plan) - plan.n);          // particles + staged padding
    unsigned generation = 0;

    if (tid == CWARPS * 32) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], CWARPS);
        }
        mbar_fence_init();
    }

    // ---- phase 0: equal-mass flags of every 256-particle group (masses never change), initial staging --------------
    int* const mflags = const_cast<int*>(plan_flags(jsrc, plan));
    const int nflags = plan_nflags(plan);
    const T mass0 = reinterpret_cast<const T*>(fa.posm)[3];
    for (int g = (int)c; g < nflags; g += (int)gridDim.x) {
        int differs = 0;
        for (int64_t i = (int64_t)g * STEP_THREADS + tid; i < (int64_t)(g + 1) * STEP_THREADS && i < plan.n; i += NTHREADS)
            differs |= !(fa.posm[i].w == mass0);                       // NaN counts as different
        const int any = __syncthreads_or(differs);
        if (tid == 0) mflags[g] = any;
    }
    auto integrate = [&](auto reduce_tag, const int flags) {
        constexpr bool REDUCE = decltype(reduce_tag)::value;
        for (int64_t i = gtid; i < nwork; i += gsize)
            (void)step_particle<T, REDUCE>(fa.posm, fa.vel, fa.acc, jsrc, rows, plan, fa.G, fa.pot, fa.dt, flags | STEP_SLICE,
                                           (V4*)nullptr, 0, plan.n, i);
    };
    typedef std::integral_constant<bool, true> True;
    typedef std::integral_constant<bool, false> False;
    if (!fa.acc_valid) integrate(False{}, STEP_PACK_ONLY);
    grid_barrier(fa.barrier, generation);                               // also publishes the mbarrier inits in the CTA

    int differs = 0;
    for (int k = tid; k < nflags; k += NTHREADS) differs |= __ldcg(mflags + k);
    const bool eqm = __syncthreads_or(differs) == 0;
    if (c == 0 && tid == 0) *const_cast<int*>(plan_eqm_word(jsrc, plan)) = eqm ? 1 : 0;

    // ---- the two phases ----------------------------------------------------------------------------------------------
    int ps = 0, cs = 0;                                                 // ring positions of the producer and of the consumers
    uint32_t pph = 0, cph = 0;
    auto pair_phase = [&]() {
        if (warp == CWARPS) {
            if (lane == 0) {
                // wait(empty, parity ^ 1) passes at once on a fresh barrier, so the same loop serves the first tiles too
                for (TileWalk pw(plan, u0, u1); pw.valid(); pw.next()) {
                    mbar_wait_backoff(&empty_bar[ps], pph ^ 1u);
                    const uint32_t bytes = (uint32_t)pw.len() * C::REC;
                    mbar_arrive_expect_tx(&full_bar[ps], bytes);
                    tma_load_1d(smem_raw + (size_t)ps * stage_bytes, jsrc + (size_t)pw.j * C::REC, bytes, &full_bar[ps]);
                    if (++ps == STAGES) { ps = 0; pph ^= 1u; }
                }
            }
        } else if (eqm) {
            consume_units<C, true>(prm, rows, plan, smem_raw, full_bar, empty_bar, u0, u1, cs, cph);
        } else {
            consume_units<C, false>(prm, rows, plan, smem_raw, full_bar, empty_bar, u0, u1, cs, cph);
        }
    };

    // ---- the KDK loop of odisseo_leapfrog_kdk_* (api.cu leapfrog_impl), nsteps >= 1 ------------------------------------
    if (fa.acc_valid) {
        integrate(False{}, STEP_OPEN);
    } else {
        pair_phase();
        grid_barrier(fa.barrier, generation);
        integrate(True{}, STEP_OPEN);
    }
    grid_barrier(fa.barrier, generation);
    for (int64_t k = 1; k < fa.nsteps; ++k) {
        pair_phase();
        grid_barrier(fa.barrier, generation);
        integrate(True{}, STEP_CLOSE | STEP_OPEN);
        grid_barrier(fa.barrier, generation);
    }
    pair_phase();
    grid_barrier(fa.barrier, generation);
    integrate(True{}, STEP_CLOSE);
}

template <class C, typename T> cudaError_t configure_fused(int max_tile, int num_sms, int* max_ctas)
{
    const int smem = (int)((size_t)STAGES * max_tile * C::REC + C::outer_bytes());
    cudaError_t e = cudaFuncSetAttribute(fused_kdk_kernel<C, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fused_kdk_kernel<C, T>, (C::CWARPS + 1) * 32, (size_t)smem);
    if (e != cudaSuccess) return e;
    *max_ctas = per_sm * num_sms;
    return cudaSuccess;
}

template <class C, typename T>
cudaError_t launch_fused(const PairPlan& plan, const typename C::Params& prm, void* jsrc, double* rows, const FusedArgs<T>& fa,
                         cudaStream_t stream)
{
    typename C::Params p = prm;
    unsigned char* j = static_cast<unsigned char*>(jsrc);
    PairPlan pl = plan;
    FusedArgs<T> f = fa;
    void* args[] = {&p, &j, &rows, &pl, &f};
    return cudaLaunchCooperativeKernel(reinterpret_cast<void*>(fused_kdk_kernel<C, T>), dim3(plan.P), dim3((C::CWARPS + 1) * 32), args,
                                       stream_smem_bytes<C>(plan), stream);
}

}  // namespace odisseo
