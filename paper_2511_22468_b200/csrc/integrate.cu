// O(N) kernels of the hot path: fixed-order reduction of the pair partial sums, external
// NFW + Miyamoto-Nagai acceleration, kick / drift, and (re)staging of the source array the
// pair kernels read by TMA.  One fused launch per KDK step:
//
//   a_pair = G * sum_{rows of this i-block, increasing j} partial      [STEP_FROM_PARTIALS] -> acc
//   a      = a_pair + a_NFW(x) + a_MN(x)
//   v     += a dt/2          [STEP_CLOSE: second half kick of the step that just ended]
//   v     += a dt/2 ; x += v dt   [STEP_OPEN: first half kick + drift of the next step]
//   stage x for the next pair evaluation -- only in the staged forms (cross, sharded, cooperative); on the default
//   path the pair kernel's TMA reads posm itself and this kernel writes posm, vel, acc and the equal-mass flags only
//
// The two half kicks are two separate FMAs, so a step split across two calls is bit-identical to
// the fused one (PAPER.md:L47 Velocity-Verlet; chaining contract in include/odisseo.h).
// Memory-bound: one 16 B (32 B) record load per array, coalesced 128-bit accesses.
#include "step_body.cuh"

namespace odisseo {

namespace {

// REDUCE = the launch starts from the pair kernel's partial rows (flags & STEP_FROM_PARTIALS); a
// compile-time switch so that the plain kick/drift instantiation does not carry the reduce batch in
// registers (occupancy is what hides HBM latency here).
template <typename T, bool REDUCE>
__global__ void __launch_bounds__(STEP_THREADS, REDUCE ? 2 : (sizeof(T) == 4 ? 6 : 3))
step_kernel(typename Vec4<T>::type* __restrict__ posm, typename Vec4<T>::type* __restrict__ vel,
            typename Vec4<T>::type* __restrict__ acc, void* __restrict__ jsrc, const double* __restrict__ partials,
            const PairPlan plan, const T G, const PotParams<T> pot, const T dt, const int flags,
            typename Vec4<T>::type* __restrict__ snapshot, const int64_t lo, const int64_t count)
{
    // posm, vel, acc address the particles [lo, lo + count) of the plan's n (the whole set: lo = 0, count = n; a
    // rank's slice in the sharded form, STEP_SLICE); staged records are written at their global index.
    typedef typename Vec4<T>::type V4;
    pdl_launch_dependents();
    pdl_wait();                                      // the pair kernel's rows (or the caller's state) are complete
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool staging = (flags & (STEP_OPEN | STEP_PACK_ONLY)) != 0;
    const bool flagging = staging && !(flags & STEP_SLICE);             // masses never change: a slice keeps the flags
    int* const block_flag = const_cast<int*>(plan_flags(jsrc, plan)) + blockIdx.x;
    if (flagging) {                                  // uniform branch: flags is a kernel argument
        if (threadIdx.x == 0) *block_flag = 0;
        __syncthreads();                             // before any load is in flight: costs nothing
    }
    const int mass_differs = step_particle<T, REDUCE>(posm, vel, acc, jsrc, partials, plan, G, pot, dt, flags, snapshot, lo, count, i);
    if (flagging) {
        // same-value plain stores after the block's own zeroing: no atomics, no closing barrier
        const unsigned any = __ballot_sync(0xffffffffu, mass_differs);
        if (any != 0u && (threadIdx.x & 31) == 0) *block_flag = 1;
    }
}

// Fixed-order row reduce alone (cross call: the targets are not the staged sources): acc_i = G * sum of rows.
template <typename T>
__global__ void __launch_bounds__(STEP_THREADS)
reduce_rows_kernel(const double* __restrict__ partials, const void* __restrict__ jsrc, const void* __restrict__ records,
                   const PairPlan plan, const T G, typename Vec4<T>::type* __restrict__ acc)
{
    pdl_wait();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= plan.nt) return;
    const double gm = (double)G * plan_row_mass<T>(jsrc, plan, records);
    double sum[3];
    reduce_unit_rows<3>(partials, plan, i, sum);
    typename Vec4<T>::type a;
    a.x = (T)(gm * sum[0]); a.y = (T)(gm * sum[1]); a.z = (T)(gm * sum[2]); a.w = (T)0;
    acc[i] = a;
}

template <typename T>
__global__ void __launch_bounds__(256)
ext_kernel(const typename Vec4<T>::type* __restrict__ posm, typename Vec4<T>::type* __restrict__ acc, const int64_t n,
           const PotParams<T> pot, const int accumulate)
{
    typedef typename Vec4<T>::type V4;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const V4 p = posm[i];
    T ex, ey, ez;
    ext_accel<T>(pot, p.x, p.y, p.z, ex, ey, ez);
    V4 a;
    if (accumulate) {
        a = acc[i];
        a.x += ex; a.y += ey; a.z += ez;
    } else {
        a.x = ex; a.y = ey; a.z = ez; a.w = (T)0;
    }
    acc[i] = a;
}

__global__ void __launch_bounds__(256)
soa_pack_kernel(const float* __restrict__ x, const float* __restrict__ y, const float* __restrict__ z,
                const float* __restrict__ m, float4* __restrict__ posm, const int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) posm[i] = make_float4(x[i], y[i], z[i], m[i]);
}

__global__ void __launch_bounds__(256)
soa_unpack_kernel(const float4* __restrict__ acc, float* __restrict__ ax, float* __restrict__ ay,
                  float* __restrict__ az, const int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const float4 a = acc[i];
        ax[i] = a.x; ay[i] = a.y; az[i] = a.z;
    }
}

inline unsigned grid_for(int64_t n) { return (unsigned)((n + 255) / 256); }

}  // namespace

cudaError_t launch_step_f32(const PairPlan& plan, float* posm, float* vel, float* acc, void* jsrc,
                            const double* partials, float G, const PotParams<float>& pot, float dt, int flags,
                            float* snapshot, int64_t lo, int64_t count, cudaStream_t stream)
{
    const dim3 grid(grid_for(count + (plan_npad(plan) - plan.n))), block(STEP_THREADS);
    typedef float4 V4;
    if (flags & STEP_FROM_PARTIALS)
        return launch_pdl(step_kernel<float, true>, grid, block, 0, stream, reinterpret_cast<V4*>(posm), reinterpret_cast<V4*>(vel),
                          reinterpret_cast<V4*>(acc), jsrc, partials, plan, G, pot, dt, flags, reinterpret_cast<V4*>(snapshot), lo, count);
    return launch_pdl(step_kernel<float, false>, grid, block, 0, stream, reinterpret_cast<V4*>(posm), reinterpret_cast<V4*>(vel),
                      reinterpret_cast<V4*>(acc), jsrc, partials, plan, G, pot, dt, flags, reinterpret_cast<V4*>(snapshot), lo, count);
}

cudaError_t launch_step_f64(const PairPlan& plan, double* posm, double* vel, double* acc, void* jsrc,
                            const double* partials, double G, const PotParams<double>& pot, double dt, int flags,
                            double* snapshot, int64_t lo, int64_t count, cudaStream_t stream)
{
    const dim3 grid(grid_for(count + (plan_npad(plan) - plan.n))), block(STEP_THREADS);
    typedef double4 V4;
    if (flags & STEP_FROM_PARTIALS)
        return launch_pdl(step_kernel<double, true>, grid, block, 0, stream, reinterpret_cast<V4*>(posm), reinterpret_cast<V4*>(vel),
                          reinterpret_cast<V4*>(acc), jsrc, partials, plan, G, pot, dt, flags, reinterpret_cast<V4*>(snapshot), lo, count);
    return launch_pdl(step_kernel<double, false>, grid, block, 0, stream, reinterpret_cast<V4*>(posm), reinterpret_cast<V4*>(vel),
                      reinterpret_cast<V4*>(acc), jsrc, partials, plan, G, pot, dt, flags, reinterpret_cast<V4*>(snapshot), lo, count);
}

cudaError_t launch_reduce_rows_f32(const PairPlan& plan, const double* partials, const void* jsrc, const void* records, float G,
                                   float* acc, cudaStream_t stream)
{
    return launch_pdl(reduce_rows_kernel<float>, dim3(grid_for(plan.nt)), dim3(STEP_THREADS), 0, stream, partials, jsrc, records, plan, G,
                      reinterpret_cast<float4*>(acc));
}
cudaError_t launch_reduce_rows_f64(const PairPlan& plan, const double* partials, const void* jsrc, const void* records, double G,
                                   double* acc, cudaStream_t stream)
{
    return launch_pdl(reduce_rows_kernel<double>, dim3(grid_for(plan.nt)), dim3(STEP_THREADS), 0, stream, partials, jsrc, records, plan, G,
                      reinterpret_cast<double4*>(acc));
}

cudaError_t launch_ext_f32(const float* posm, float* acc, int64_t n, const PotParams<float>& pot, int accumulate,
                           cudaStream_t stream)
{
    ext_kernel<float><<<grid_for(n), 256, 0, stream>>>(reinterpret_cast<const float4*>(posm),
                                                       reinterpret_cast<float4*>(acc), n, pot, accumulate);
    return cudaGetLastError();
}

cudaError_t launch_ext_f64(const double* posm, double* acc, int64_t n, const PotParams<double>& pot, int accumulate,
                           cudaStream_t stream)
{
    ext_kernel<double><<<grid_for(n), 256, 0, stream>>>(reinterpret_cast<const double4*>(posm),
                                                        reinterpret_cast<double4*>(acc), n, pot, accumulate);
    return cudaGetLastError();
}

cudaError_t launch_soa_pack_f32(const float* x, const float* y, const float* z, const float* m, float* posm,
                                int64_t n, cudaStream_t stream)
{
    soa_pack_kernel<<<grid_for(n), 256, 0, stream>>>(x, y, z, m, reinterpret_cast<float4*>(posm), n);
    return cudaGetLastError();
}

cudaError_t launch_soa_unpack_f32(const float* acc, float* ax, float* ay, float* az, int64_t n, cudaStream_t stream)
{
    soa_unpack_kernel<<<grid_for(n), 256, 0, stream>>>(reinterpret_cast<const float4*>(acc), ax, ay, az, n);
    return cudaGetLastError();
}

}  // namespace odisseo
