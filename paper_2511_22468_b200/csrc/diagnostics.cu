// Conservation diagnostics of a particle state: kinetic energy, softened
// pair potential energy W = -1/2 G sum_i sum_{j != i} m_i m_j (r_ij^2 + eps^2)^-1/2, external potential
// energy sum_i m_i (Phi_NFW + Phi_MN)(x_i), linear and angular momentum, centre of mass, total mass.
// The integrator the paper uses is symplectic and time-reversible ("second-order
// Velocity-Verlet"), so these are what a user monitors; they are evaluated in fp64 whatever the precision
// of the state (an fp32 energy cannot resolve the 1e-6 .. 1e-9 drifts of interest).
//
//   stage   : promote {x,y,z,m} to double records (+ massless far-away padding, + equal-mass flags)
//   O(N^2)  : pair_f64.cu in POT mode -> partial rows of phi'_i = sum_j m_j (r_ij^2 + eps^2)^-1/2
//   terms   : fixed-order row sum, self term m_i / eps removed, per-particle terms, block sums
//   final   : one block adds the block sums in index order -> 16 doubles
// Every reduction has a fixed order: results are bit-reproducible run to run.
#include "odisseo_common.cuh"
#include "ext_potential.cuh"

namespace odisseo {

namespace {

template <typename T> struct DVec4;
template <> struct DVec4<float> { typedef float4 type; };
template <> struct DVec4<double> { typedef double4 type; };

template <typename T>
__global__ void __launch_bounds__(STEP_THREADS)
diag_stage_kernel(const typename DVec4<T>::type* __restrict__ posm, double4* __restrict__ jsrc, const PairPlan plan)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int* const block_flag = const_cast<int*>(plan_flags(jsrc, plan)) + blockIdx.x;
    if (threadIdx.x == 0) *block_flag = 0;
    __syncthreads();
    int differs = 0;
    if (i < plan.n) {
        const typename DVec4<T>::type p = posm[i];
        jsrc[i] = make_double4((double)p.x, (double)p.y, (double)p.z, (double)p.w);
        differs = !(p.w == reinterpret_cast<const T*>(posm)[3]);
    } else if (i < plan_npad(plan)) {
        jsrc[i] = make_double4(PAD_POS_F64, PAD_POS_F64, PAD_POS_F64, 0.0);
    }
    const unsigned any = __ballot_sync(0xffffffffu, differs);
    if (any != 0u && (threadIdx.x & 31) == 0) *block_flag = 1;
}

// External potential Phi_NFW + Phi_MN in double (include/odisseo.h; readings R10-R12).
__device__ __forceinline__ double ext_potential(const PotParams<double>& pot, double x, double y, double z)
{
    double phi = 0.0;
    if (pot.GMs != 0.0) {
        const double r = sqrt(fma(x, x, fma(y, y, z * z)));
        phi += r > 0.0 ? -pot.GMs * log1p(r * pot.inv_rs) / r : -pot.GMs * pot.inv_rs;   // ln(1+c)/c -> 1
    }
    if (pot.GMd != 0.0) {
        const double sB = pot.a + sqrt(fma(z, z, pot.b2));
        phi += -pot.GMd / sqrt(fma(x, x, fma(y, y, sB * sB)));
    }
    if (pot.GMb != 0.0) {
        // Phi = -G M_b [ P(s, t)/r + Gamma(s - 1/2, t) / (r_c Gamma(s)) ],  Gamma(a, t) = Gamma(a) (1 - P(a, t))
        const double r = sqrt(fma(x, x, fma(y, y, z * z)));
        const double t = (r * pot.inv_rc) * (r * pot.inv_rc);
        const double outer = pot.phi_outer * (1.0 - gamma_p(pot.bs_half, t, pot.lgam_s_half));
        phi += -pot.GMb * ((r > 0.0 ? gamma_p(pot.bs, t, pot.lgam_s) / r : 0.0) + outer);
    }
    return phi;
}

// Fixed-shape sum over the block: xor-shuffle tree inside a warp, then warp 0 adds the warp sums in order.
__device__ __forceinline__ double block_sum(double v, double* warp_scratch)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();                                   // scratch free from the previous value
    if (lane == 0) warp_scratch[warp] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < STEP_THREADS / 32; ++w) s += warp_scratch[w];
    return s;                                          // valid in thread 0
}

template <typename T>
__global__ void __launch_bounds__(STEP_THREADS)
diag_terms_kernel(const typename DVec4<T>::type* __restrict__ posm, const typename DVec4<T>::type* __restrict__ vel,
                  const double* __restrict__ partials, const void* __restrict__ jsrc, const PairPlan plan, const double G,
                  const double eps, const PotParams<double> pot, double* __restrict__ block_sums, double* __restrict__ phi_out)
{
    __shared__ double warp_scratch[STEP_THREADS / 32];
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double val[DIAG_VALUES];
#pragma unroll
    for (int k = 0; k < DIAG_VALUES; ++k) val[k] = 0.0;
    if (i < plan.n) {
        const typename DVec4<T>::type p = posm[i];
        const typename DVec4<T>::type w = vel[i];
        const double x = p.x, y = p.y, z = p.z, m = p.w, vx = w.x, vy = w.y, vz = w.z;
        double rows[1];
        reduce_unit_rows<1>(partials, plan, i, rows);                    // increasing j, fixed grouping
        const double sum = plan_row_mass<double>(jsrc, plan, jsrc) * rows[0];
        const double phi = -G * (sum - m / eps);       // the kernel's self term is m_i (0 + eps^2)^-1/2
        if (phi_out) phi_out[i] = phi;
        val[0] = 0.5 * m * fma(vx, vx, fma(vy, vy, vz * vz));
        val[1] = 0.5 * m * phi;
        val[2] = m * ext_potential(pot, x, y, z);
        val[3] = m * vx; val[4] = m * vy; val[5] = m * vz;
        val[6] = m * (y * vz - z * vy); val[7] = m * (z * vx - x * vz); val[8] = m * (x * vy - y * vx);
        val[9] = m * x; val[10] = m * y; val[11] = m * z;
        val[12] = m;
    }
#pragma unroll
    for (int k = 0; k < 13; ++k) {
        const double s = block_sum(val[k], warp_scratch);
        if (threadIdx.x == 0) block_sums[(size_t)blockIdx.x * DIAG_VALUES + k] = s;
    }
}

__global__ void __launch_bounds__(STEP_THREADS)
diag_final_kernel(const double* __restrict__ block_sums, const int nblocks, double* __restrict__ out)
{
    __shared__ double warp_scratch[STEP_THREADS / 32];
    double tot[13];
#pragma unroll
    for (int k = 0; k < 13; ++k) {
        double v = 0.0;
        for (int b = threadIdx.x; b < nblocks; b += STEP_THREADS) v += block_sums[(size_t)b * DIAG_VALUES + k];
        tot[k] = block_sum(v, warp_scratch);
    }
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < 13; ++k) out[k] = tot[k];
        const double M = tot[12];
        for (int k = 9; k < 12; ++k) out[k] = M != 0.0 ? tot[k] / M : 0.0;       // centre of mass
        out[13] = tot[0] + tot[1] + tot[2];                                        // total energy
        out[14] = 0.0; out[15] = 0.0;
    }
}

inline unsigned grid_for(int64_t n) { return (unsigned)((n + STEP_THREADS - 1) / STEP_THREADS); }

}  // namespace

cudaError_t launch_diag_stage_f32(const PairPlan& plan, const float* posm, void* jsrc, cudaStream_t stream)
{
    diag_stage_kernel<float><<<grid_for(plan_npad(plan)), STEP_THREADS, 0, stream>>>(
        reinterpret_cast<const float4*>(posm), static_cast<double4*>(jsrc), plan);
    return cudaGetLastError();
}
cudaError_t launch_diag_stage_f64(const PairPlan& plan, const double* posm, void* jsrc, cudaStream_t stream)
{
    diag_stage_kernel<double><<<grid_for(plan_npad(plan)), STEP_THREADS, 0, stream>>>(
        reinterpret_cast<const double4*>(posm), static_cast<double4*>(jsrc), plan);
    return cudaGetLastError();
}
cudaError_t launch_diag_terms_f32(const PairPlan& plan, const float* posm, const float* vel, const double* partials,
                                  const void* jsrc, double G, double eps, const PotParams<double>& pot, double* block_sums,
                                  double* phi_out, cudaStream_t stream)
{
    diag_terms_kernel<float><<<grid_for(plan.n), STEP_THREADS, 0, stream>>>(
        reinterpret_cast<const float4*>(posm), reinterpret_cast<const float4*>(vel), partials, jsrc, plan, G, eps, pot,
        block_sums, phi_out);
    return cudaGetLastError();
}
cudaError_t launch_diag_terms_f64(const PairPlan& plan, const double* posm, const double* vel, const double* partials,
                                  const void* jsrc, double G, double eps, const PotParams<double>& pot, double* block_sums,
                                  double* phi_out, cudaStream_t stream)
{
    diag_terms_kernel<double><<<grid_for(plan.n), STEP_THREADS, 0, stream>>>(
        reinterpret_cast<const double4*>(posm), reinterpret_cast<const double4*>(vel), partials, jsrc, plan, G, eps, pot,
        block_sums, phi_out);
    return cudaGetLastError();
}
cudaError_t launch_diag_final(const double* block_sums, int nblocks, double* out, cudaStream_t stream)
{
    diag_final_kernel<<<1, STEP_THREADS, 0, stream>>>(block_sums, nblocks, out);
    return cudaGetLastError();
}

}  // namespace odisseo
