// fp64 all-pairs Plummer-softened acceleration (section 1).
//
// Same persistent-grid / TMA-ring skeleton as pair_f32.cu (pair_stream.cuh); sources are plain
// {x, y, z, m} double records (32 B) copied into a zero-mass-padded staging array.
// (r2)^-3/2 comes from the double-precision seed y0 = rsqrt.approx.ftz.f64(r2) (MUFU.RSQ64H on the
// high word: relative error ~2^-22, low word zero, no F2F conversions) and ONE correction of the
// cube:  t = y0^2,  e = 1 - r2 t,  (r2)^-3/2 = y0^3 (1-e)^-3/2 = y0^3 (1 + e (3/2 + 15/8 e)) + O(e^3),
// remainder (35/16) e^3 ~ 2e-19: 7 FP64 ops for m (r2)^-3/2 instead of ~20 with the library rsqrt().
// 16 FP64-pipe ops + 1 MUFU per interaction (3 DADD, 9 DFMA, 4 DMUL).  A DFMA holds a scheduler's
// dispatch port 2 cycles and every other instruction 1, so F2F or integer conversions around an fp32
// seed cost as much as the arithmetic they feed.
// Summation: fp64 inside a tile, tile sums added in tile order inside a unit, one row per unit -- the
// same fixed grouping as the fp32 kernel.
#include <stdio.h>

#include <string>

#include "fused_step.cuh"
#include "cluster_kdk.cuh"
#include "ll_kdk.cuh"

namespace odisseo {

namespace {

// POT = accumulate the softened potential sum_j m_j (r2)^-1/2 (x-plane of the rows only) instead of the
// acceleration: the O(N^2) part of odisseo_diagnostics_* (diagnostics.cu).
template <int IPT, int CWARPS_, int MINB_, int JUNROLL, bool POT>
struct PairF64 {
    static constexpr int CWARPS = CWARPS_, MINB = MINB_, REC = 32, COMPS = 3;
    static constexpr int CTHREADS = CWARPS * 32;
    struct Params { const double4* posm; double eps2; };
    static size_t outer_bytes() { return (size_t)3 * IPT * CTHREADS * sizeof(double); }

    // EQM = all masses equal (flags from the staging kernel): the mass factor leaves the inner loop
    // (15 instead of 16 FP64 ops); the reduce step multiplies by the mass once.
    template <bool EQM>
    struct State {
        const double4* __restrict__ posm;
        const int64_t nt;
        const int32_t IB;
        const double eps2;
        double* __restrict__ osum;                 // osum[3k + comp][tid]
        double xi[IPT], yi[IPT], zi[IPT], ax[IPT], ay[IPT], az[IPT];

        __device__ __forceinline__ State(const Params& prm, const PairPlan& plan, unsigned char* outer)
            : posm(prm.posm), nt(plan.nt), IB(plan.IB), eps2(prm.eps2), osum(reinterpret_cast<double*>(outer) + threadIdx.x)
        {
        }
        __device__ __forceinline__ void load_targets(const int32_t b)
        {
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                int64_t i = (int64_t)b * IB + (int64_t)k * CTHREADS + threadIdx.x;
                i = i < nt ? i : nt - 1;
                // coherent (L2) loads: posm is rewritten between pair phases inside the whole-loop kernels
                const double2 pxy = __ldcg(reinterpret_cast<const double2*>(posm + i));
                const double pz = __ldcg(reinterpret_cast<const double*>(posm + i) + 2);
                xi[k] = pxy.x; yi[k] = pxy.y; zi[k] = pz;
                ax[k] = ay[k] = az[k] = 0.0;
            }
        }
        __device__ __forceinline__ void zero_outer()
        {
#pragma unroll
            for (int k = 0; k < 3 * IPT; ++k) osum[k * CTHREADS] = 0.0;
        }
        __device__ __forceinline__ void tile(const unsigned char* tile_raw, const int len)
        {
            const double4* __restrict__ t = reinterpret_cast<const double4*>(tile_raw);
#pragma unroll JUNROLL
            for (int j = 0; j < len; ++j) {
                const double4 q = t[j];
#pragma unroll
                for (int k = 0; k < IPT; ++k) {
                    const double dx = q.x - xi[k];
                    const double dy = q.y - yi[k];
                    const double dz = q.z - zi[k];
                    double r2 = fma(dx, dx, eps2);
                    r2 = fma(dy, dy, r2);
                    r2 = fma(dz, dz, r2);
                    const double y0 = rsqrt_approx_f64(r2);
                    const double y2 = y0 * y0;
                    const double e = fma(-r2, y2, 1.0);
                    if (POT) {
                        // (r2)^-1/2 = y0 (1-e)^-1/2 = y0 (1 + e (1/2 + 3/8 e)) + O(e^3)
                        const double y = y0 * fma(e, fma(0.375, e, 0.5), 1.0);
                        ax[k] = EQM ? ax[k] + y : fma(q.w, y, ax[k]);
                    } else {
                        const double c = fma(e, fma(1.875, e, 1.5), 1.0);
                        const double w = EQM ? (y2 * y0) * c : ((y2 * y0) * q.w) * c;
                        ax[k] = fma(w, dx, ax[k]);
                        ay[k] = fma(w, dy, ay[k]);
                        az[k] = fma(w, dz, az[k]);
                    }
                }
            }
        }
        __device__ __forceinline__ void flush_tile()
        {
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                osum[(3 * k + 0) * CTHREADS] += ax[k];
                if (!POT) {
                    osum[(3 * k + 1) * CTHREADS] += ay[k];
                    osum[(3 * k + 2) * CTHREADS] += az[k];
                }
                ax[k] = ay[k] = az[k] = 0.0;
            }
        }
        // cluster kernel (cluster_kdk.cuh): two targets handed over as records; tile sums added into six doubles
        __device__ __forceinline__ void set_target_pair(const double4 p0, const double4 p1)
        {
            static_assert(IPT >= 2, "two targets per thread");
            xi[0] = p0.x; yi[0] = p0.y; zi[0] = p0.z;
            xi[1] = p1.x; yi[1] = p1.y; zi[1] = p1.z;
            ax[0] = ay[0] = az[0] = ax[1] = ay[1] = az[1] = 0.0;
        }
        __device__ __forceinline__ void take_sums(double (&s)[6])
        {
            s[0] += ax[0]; s[1] += ay[0]; s[2] += az[0];
            s[3] += ax[1]; s[4] += ay[1]; s[5] += az[1];
            ax[0] = ay[0] = az[0] = ax[1] = ay[1] = az[1] = 0.0;
        }
        __device__ __forceinline__ void write_row(double* __restrict__ row)
        {
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                const int r = k * CTHREADS + threadIdx.x;
                row[r] = osum[(3 * k + 0) * CTHREADS];
                if (!POT) {
                    row[IB + r] = osum[(3 * k + 1) * CTHREADS];
                    row[2 * IB + r] = osum[(3 * k + 2) * CTHREADS];
                }
            }
        }
    };
};

typedef PairF64<4, 8, 1, 4, false> LargeF64;
typedef PairF64<2, 2, 8, 2, false> SmallF64;
typedef PairF64<4, 8, 1, 4, true> LargePot;
typedef PairF64<2, 2, 8, 2, true> SmallPot;
typedef PairF64<2, 2, 4, 2, false> SmallF64Fused;

typedef PairF64<2, 2, 1, 2, false> ClusterF64;   // the same loop inside the cluster kernel (cluster_kdk.cuh)
typedef PairF64<2, 2, 1, 4, false> LLF64;        // ... and inside the flag-in-data kernel (ll_kdk.cuh)

int g_fused_max_ctas64[2] = {0, 0};
int g_cluster_size64 = 0;
int g_ll_max_ctas64 = 0;
constexpr bool LL_TAPE_CODE_DOUBLE = false;     // see LL_TAPE_CODE_FLOAT in pair_f32.cu (measured: 6.8 against 8.7 us per step)

}  // namespace

cudaError_t configure_pair_f64(int num_sms)
{
    cudaError_t e = configure_stream<LargeF64>(256);
    if (e == cudaSuccess) e = configure_stream<SmallF64>(256);
    if (e == cudaSuccess) e = configure_stream<LargePot>(256);
    if (e == cudaSuccess) e = configure_stream<SmallPot>(256);
    if (e == cudaSuccess) e = configure_fused<LargeF64, double>(256, num_sms, &g_fused_max_ctas64[0]);
    if (e == cudaSuccess) e = configure_fused<SmallF64Fused, double>(256, num_sms, &g_fused_max_ctas64[1]);
    if (e == cudaSuccess) e = configure_cluster<ClusterF64, double>(&g_cluster_size64);
    if (e == cudaSuccess) e = configure_ll<LLF64, double>(num_sms, &g_ll_max_ctas64);
    return e;
}

int fused_max_ctas_f64(int variant) { return g_fused_max_ctas64[variant ? 1 : 0]; }

cudaError_t launch_fused_f64(const PairPlan& plan, double* posm, double* vel, double* acc, void* jsrc, double* partials, double G,
                             double eps, double dt, const PotParams<double>& pot, int64_t nsteps, int acc_valid, unsigned* barrier,
                             cudaStream_t stream)
{
    FusedArgs<double> fa;
    fa.posm = reinterpret_cast<double4*>(posm); fa.vel = reinterpret_cast<double4*>(vel); fa.acc = reinterpret_cast<double4*>(acc);
    fa.G = G; fa.dt = dt; fa.pot = pot; fa.nsteps = nsteps; fa.acc_valid = acc_valid; fa.barrier = barrier;
    if (plan.variant == 0) {
        const LargeF64::Params prm{reinterpret_cast<const double4*>(posm), eps * eps};
        return launch_fused<LargeF64, double>(plan, prm, jsrc, partials, fa, stream);
    }
    const SmallF64Fused::Params prm{reinterpret_cast<const double4*>(posm), eps * eps};
    return launch_fused<SmallF64Fused, double>(plan, prm, jsrc, partials, fa, stream);
}

bool cluster_fits_f64(const PairPlan& plan)
{
    int32_t tpc;
    return g_cluster_size64 > 0 && plan.n <= CLUSTER_MAX_N && cluster_geometry<double>(plan, g_cluster_size64, &tpc) != 0;
}

cudaError_t launch_cluster_f64(const PairPlan& plan, double* posm, double* vel, double* acc, double G, double eps, double dt,
                               const PotParams<double>& pot, int64_t nsteps, int acc_valid, cudaStream_t stream)
{
    ClusterArgs<double> ca;
    ca.posm = reinterpret_cast<double4*>(posm); ca.vel = reinterpret_cast<double4*>(vel); ca.acc = reinterpret_cast<double4*>(acc);
    ca.G = G; ca.eps2 = eps * eps; ca.dt = dt; ca.pot = pot; ca.nsteps = nsteps; ca.acc_valid = acc_valid;
    ca.n = (int32_t)plan.n; ca.n8 = (int32_t)plan.n8; ca.S = plan.S; ca.Ttile = plan.T;
    const size_t smem = cluster_geometry<double>(plan, g_cluster_size64, &ca.tpc);
    return launch_cluster<ClusterF64, double>(ca, g_cluster_size64, smem, stream);
}

size_t ll_fits_f64(const PairPlan& plan)
{
    int32_t tpc, ctas;
    size_t xbytes = 0;
    return ll_geometry<double>(plan, g_ll_max_ctas64, &tpc, &ctas, &xbytes) != 0 ? xbytes : 0;
}

cudaError_t launch_ll_f64(const PairPlan& plan, double* posm, double* vel, double* acc, double G, double eps, double dt,
                          const PotParams<double>& pot, int64_t nsteps, int acc_valid, void* xbuf, double* tape, cudaStream_t stream)
{
    LLArgs<double> ca;
    ca.posm = reinterpret_cast<double4*>(posm); ca.vel = reinterpret_cast<double4*>(vel); ca.acc = reinterpret_cast<double4*>(acc);
    ca.G = G; ca.eps2 = eps * eps; ca.dt = dt; ca.pot = pot; ca.nsteps = nsteps; ca.acc_valid = acc_valid;
    ca.n = (int32_t)plan.n; ca.n8 = (int32_t)plan.n8; ca.S = plan.S; ca.Ttile = plan.T;
    ca.xbuf = static_cast<unsigned long long*>(xbuf);
    ca.tape = reinterpret_cast<double4*>(tape);
    int32_t ctas;
    size_t xbytes;
    const size_t smem = ll_geometry<double>(plan, g_ll_max_ctas64, &ca.tpc, &ctas, &xbytes);
    cudaError_t e = cudaMemsetAsync(xbuf, 0, xbytes, stream);          // tags start at 1
    if (e != cudaSuccess) return e;
    return launch_ll<LLF64, double>(ca, ctas, smem, LL_TAPE_CODE_DOUBLE, stream);
}

template <int A, int B, int C, int D, bool POT>
static std::string stream_kernel_name(const PairF64<A, B, C, D, POT>*)
{
    char buf[96];
    snprintf(buf, sizeof buf, "stream_kernel<PairF64<%d,%d,%d,%d,%d>>", A, B, C, D, (int)POT);
    return buf;
}
const char* pair_kernel_name_f64(int variant)
{
    static const std::string names[2] = {stream_kernel_name(static_cast<const LargeF64*>(nullptr)),
                                         stream_kernel_name(static_cast<const SmallF64*>(nullptr))};
    return names[variant ? 1 : 0].c_str();
}

cudaError_t launch_pair_f64(const PairPlan& plan, const double* posm, const void* jsrc, const void* src, double* partials, double eps,
                            cudaStream_t stream)
{
    const LargeF64::Params prm{reinterpret_cast<const double4*>(posm), eps * eps};
    if (plan.variant == 0) return launch_stream<LargeF64>(plan, prm, jsrc, src, partials, stream);
    return launch_stream<SmallF64>(plan, SmallF64::Params{prm.posm, prm.eps2}, jsrc, src, partials, stream);
}

// Softened potential sums phi'_i = sum_j m_j (r_ij^2 + eps^2)^-1/2 (self term included) into the x-plane of
// the rows; targets are read from the staged double records themselves.
cudaError_t launch_potential_f64(const PairPlan& plan, const void* jsrc, double* partials, double eps,
                                 cudaStream_t stream)
{
    const double4* targets = static_cast<const double4*>(jsrc);
    if (plan.variant == 0) return launch_stream<LargePot>(plan, LargePot::Params{targets, eps * eps}, jsrc, jsrc, partials, stream);
    return launch_stream<SmallPot>(plan, SmallPot::Params{targets, eps * eps}, jsrc, jsrc, partials, stream);
}

}  // namespace odisseo
