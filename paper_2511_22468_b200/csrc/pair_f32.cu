// fp32 all-pairs Plummer-softened acceleration (section 1; SURVEY.md 8a rows a1, a1').
//
//   row(b, s)_i = sum_{j in chunk s} m_j (x_j - x_i) (|x_j - x_i|^2 + eps^2)^{-3/2}      (G applied in the reduce step)
//
// Design (B200-first, not the paper's XLA broadcast):
//   * persistent grid, one 9-warp CTA per SM (8 compute warps + 1 producer warp, ~160 registers per
//     thread so that ptxas interleaves a thread's four interaction chains), contiguous equal ranges of
//     (i-block x source-chunk) units per CTA, source tiles through a TMA ring (pair_stream.cuh)
//     -> every SM busy for any N, no wave-quantisation tail;
//   * each compute thread keeps 2*NPAIR targets in registers as packed f32x2 pairs; sources are plain
//     {x,y,z,m} records (16 B) -- on the default path the particles' OWN records, read by TMA with no
//     staged copy (plan.direct) -- so that one LDS.128 broadcast yields a source, whose coordinates enter
//     the packed instructions as scalar operands broadcast to both halves; the body is
//     3 FADD2 + 6 FFMA2 + 3 FMUL2 + 2 MUFU.RSQ per TWO interactions (half the issue slots of the scalar
//     form, no register-pair MOVs);
//   * two-level summation: fp32 inside one tile (<= 512 terms), promoted to fp64 between tiles
//     (a single running fp32 sum fails the 1e-5 tolerance at N >= 2^18); one row of
//     fp64 sums per unit, rows added in unit order by the reduce step (fixed grouping, function of n only);
//   * the self term contributes exactly 0 because eps > 0; the direct path has no padding (the last tile
//     ends at n and tile() takes any length -- keep its remainder handling); the staged forms (cross, sharded,
//     cooperative) pad with massless records parked at 3e18, where the inverse cube underflows to exactly 0 (ftz);
//   * equal masses (the paper's Plummer progenitors, PAPER.md:L43 step 3) are detected on the device by
//     the step / staging kernel (one flag per 256 particles); the mass factor then leaves the inner loop: 3 FADD2 + 6 FFMA2 + 2 FMUL2, and the
//     reduce step multiplies by the mass once;
//   * programmatic dependent launch: barrier init and plan arithmetic overlap the predecessor's tail.
#include <stdio.h>

#include <string>

#include "fused_step.cuh"
#include "cluster_kdk.cuh"
#include "ll_kdk.cuh"

namespace odisseo {

namespace {

// JUNROLL / JUNROLL_G: unroll of the j loop on the equal-mass / general-mass path (the general body holds one more
// packed value per source).  Measured at N = 262,144: equal-mass loop 24.43 ms at 8, 24.21 at 16 and 32; the general loop is
// within 1 % for 2 ... 16 (25.9-26.2 ms; 25.8 when the equal-mass loop is unrolled 8: the two paths share one register budget).
template <int NPAIR, int CWARPS_, int MINB_, int JUNROLL, int JUNROLL_G = JUNROLL>
struct PairF32 {
    static constexpr int CWARPS = CWARPS_, MINB = MINB_, REC = 16, COMPS = 3;
    static constexpr int CTHREADS = CWARPS * 32;
    struct Params { const float4* posm; float eps2; };
    static size_t outer_bytes() { return (size_t)6 * NPAIR * CTHREADS * sizeof(double); }

    // EQM = all masses equal (detected on the device by the staging kernel): the per-source mass factor
    // leaves the inner loop (11 instead of 12 packed FP32 ops per two interactions).
    template <bool EQM>
    struct State {
        const float4* __restrict__ posm;
        const int64_t nt;
        const int32_t IB;
        const f32x2 e2;
        // fp64 outer sums live in shared memory (48 registers otherwise): osum[k][tid], k = 3*(2p+h)+comp
        double* __restrict__ osum;
        f32x2 xi[NPAIR], yi[NPAIR], zi[NPAIR];
        f32x2 ax[NPAIR], ay[NPAIR], az[NPAIR];

        __device__ __forceinline__ State(const Params& prm, const PairPlan& plan, unsigned char* outer)
            : posm(prm.posm), nt(plan.nt), IB(plan.IB), e2(pk(prm.eps2, prm.eps2)),
              osum(reinterpret_cast<double*>(outer) + threadIdx.x)
        {
        }
        __device__ __forceinline__ void load_targets(const int32_t b)
        {
            const int64_t base = (int64_t)b * IB + threadIdx.x;
#pragma unroll
            for (int p = 0; p < NPAIR; ++p) {
                int64_t i0 = base + (int64_t)(2 * p) * CTHREADS;
                int64_t i1 = i0 + CTHREADS;
                i0 = i0 < nt ? i0 : nt - 1;               // clamped rows are computed and never read back
                i1 = i1 < nt ? i1 : nt - 1;
                // coherent (L2) loads: this consumer also runs inside the whole-loop kernels (fused_step.cuh), where
                // posm is rewritten between pair phases of ONE launch; a non-coherent ld.global.nc would be undefined there
                const float4 p0 = __ldcg(posm + i0);
                const float4 p1 = __ldcg(posm + i1);
                // x + (-0) == x exactly; routing the pack through FADD2 makes the pair a native 64-bit
                // register value, so ptxas does not re-assemble it with MOVs inside the j loop
                const f32x2 nz = pk(-0.0f, -0.0f);
                xi[p] = add2(pk(p0.x, p1.x), nz);
                yi[p] = add2(pk(p0.y, p1.y), nz);
                zi[p] = add2(pk(p0.z, p1.z), nz);
                ax[p] = ay[p] = az[p] = 0ull;
            }
        }
        __device__ __forceinline__ void zero_outer()
        {
#pragma unroll
            for (int k = 0; k < 6 * NPAIR; ++k) osum[k * CTHREADS] = 0.0;
        }
        __device__ __forceinline__ void tile(const unsigned char* tile_raw, const int len)
        {
            const float4* __restrict__ t = reinterpret_cast<const float4*>(tile_raw);
#pragma unroll (EQM ? JUNROLL : JUNROLL_G)
            for (int j = 0; j < len; ++j) {
                // one LDS.128 per source; the splats below cost nothing: ptxas feeds the scalar register to the packed
                // instruction as a broadcast operand (FADD2 R, Rj.F32, -Ri.F32x2) -- no MOV, no pre-duplicated staging
                const float4 q = t[j];
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
        // second summation level: promote the tile sums to fp64
        __device__ __forceinline__ void flush_tile()
        {
#pragma unroll
            for (int p = 0; p < NPAIR; ++p) {
                float lo, hi;
                unpk(ax[p], lo, hi); osum[(6 * p + 0) * CTHREADS] += (double)lo; osum[(6 * p + 3) * CTHREADS] += (double)hi;
                unpk(ay[p], lo, hi); osum[(6 * p + 1) * CTHREADS] += (double)lo; osum[(6 * p + 4) * CTHREADS] += (double)hi;
                unpk(az[p], lo, hi); osum[(6 * p + 2) * CTHREADS] += (double)lo; osum[(6 * p + 5) * CTHREADS] += (double)hi;
                ax[p] = ay[p] = az[p] = 0ull;
            }
        }
        // cluster kernel (cluster_kdk.cuh): two targets handed over as records; tile sums promoted into six doubles
        __device__ __forceinline__ void set_target_pair(const float4 p0, const float4 p1)
        {
            static_assert(NPAIR >= 1, "one packed pair");
            const f32x2 nz = pk(-0.0f, -0.0f);
            xi[0] = add2(pk(p0.x, p1.x), nz);
            yi[0] = add2(pk(p0.y, p1.y), nz);
            zi[0] = add2(pk(p0.z, p1.z), nz);
            ax[0] = ay[0] = az[0] = 0ull;
        }
        __device__ __forceinline__ void take_sums(double (&s)[6])
        {
            float lo, hi;
            unpk(ax[0], lo, hi); s[0] += (double)lo; s[3] += (double)hi;
            unpk(ay[0], lo, hi); s[1] += (double)lo; s[4] += (double)hi;
            unpk(az[0], lo, hi); s[2] += (double)lo; s[5] += (double)hi;
            ax[0] = ay[0] = az[0] = 0ull;
        }
        __device__ __forceinline__ void write_row(double* __restrict__ row)
        {
#pragma unroll
            for (int k = 0; k < 2 * NPAIR; ++k) {
                const int r = k * CTHREADS + threadIdx.x;
                row[r] = osum[(3 * k + 0) * CTHREADS];
                row[IB + r] = osum[(3 * k + 1) * CTHREADS];
                row[2 * IB + r] = osum[(3 * k + 2) * CTHREADS];
            }
        }
    };
};

typedef PairF32<4, 8, 1, 16, 8> LargeF32;  // 2,048 targets per CTA, one CTA per SM
typedef PairF32<1, 2, 8, 4> SmallF32;    // 128 targets per CTA, up to 8 CTAs per SM (n <= 4,096)
typedef PairF32<1, 2, 4, 4> SmallF32Fused;   // the same loop inside the whole-loop kernel, which also holds the reduce batch

typedef PairF32<1, 2, 1, 4> ClusterF32;      // the same loop, two targets per lane, inside the cluster kernel (cluster_kdk.cuh)
typedef PairF32<1, 2, 1, 8> LLF32;           // ... and inside the flag-in-data kernel (ll_kdk.cuh): one warp deep, so unrolled further

int g_fused_max_ctas[2] = {0, 0};        // co-resident CTAs of the whole-loop kernel, [variant]
int g_cluster_size = 0;                  // CTAs per cluster the device schedules for the cluster kernel (0 = none)
int g_ll_max_ctas = 0;                   // co-resident CTAs of the flag-in-data whole-loop kernel (ll_kdk.cuh)
// Which instantiation serves calls WITHOUT a tape.  The step of that kernel is a latency chain, and the two instantiations,
// which differ by a few predicated stores in the owner threads, schedule differently: measured at N = 1,024 the one with
// the tape code runs 3.1 us per step in fp32 (4.5 without) and 8.7 in fp64 (6.8 without).  Measured choice, per precision.
constexpr bool LL_TAPE_CODE_FLOAT = true;

}  // namespace

cudaError_t configure_pair_f32(int num_sms)
{
    cudaError_t e = configure_stream<LargeF32>(512);
    if (e == cudaSuccess) e = configure_stream<SmallF32>(256);
    if (e == cudaSuccess) e = configure_fused<LargeF32, float>(512, num_sms, &g_fused_max_ctas[0]);
    if (e == cudaSuccess) e = configure_fused<SmallF32Fused, float>(256, num_sms, &g_fused_max_ctas[1]);
    if (e == cudaSuccess) e = configure_cluster<ClusterF32, float>(&g_cluster_size);
    if (e == cudaSuccess) e = configure_ll<LLF32, float>(num_sms, &g_ll_max_ctas);
    return e;
}

// Whole-loop kernel (fused_step.cuh): all nsteps KDK steps of odisseo_leapfrog_kdk_f32 in one cooperative launch.
int fused_max_ctas_f32(int variant) { return g_fused_max_ctas[variant ? 1 : 0]; }

cudaError_t launch_fused_f32(const PairPlan& plan, float* posm, float* vel, float* acc, void* jsrc, double* partials, float G, float eps,
                             float dt, const PotParams<float>& pot, int64_t nsteps, int acc_valid, unsigned* barrier, cudaStream_t stream)
{
    FusedArgs<float> fa;
    fa.posm = reinterpret_cast<float4*>(posm); fa.vel = reinterpret_cast<float4*>(vel); fa.acc = reinterpret_cast<float4*>(acc);
    fa.G = G; fa.dt = dt; fa.pot = pot; fa.nsteps = nsteps; fa.acc_valid = acc_valid; fa.barrier = barrier;
    if (plan.variant == 0) {
        const LargeF32::Params prm{reinterpret_cast<const float4*>(posm), eps * eps};
        return launch_fused<LargeF32, float>(plan, prm, jsrc, partials, fa, stream);
    }
    const SmallF32Fused::Params prm{reinterpret_cast<const float4*>(posm), eps * eps};
    return launch_fused<SmallF32Fused, float>(plan, prm, jsrc, partials, fa, stream);
}

// Cluster kernel (cluster_kdk.cuh): does this call fit the shared memory of one cluster?
bool cluster_fits_f32(const PairPlan& plan)
{
    int32_t tpc;
    return g_cluster_size > 0 && plan.n <= CLUSTER_MAX_N && cluster_geometry<float>(plan, g_cluster_size, &tpc) != 0;
}

cudaError_t launch_cluster_f32(const PairPlan& plan, float* posm, float* vel, float* acc, float G, float eps, float dt,
                               const PotParams<float>& pot, int64_t nsteps, int acc_valid, cudaStream_t stream)
{
    ClusterArgs<float> ca;
    ca.posm = reinterpret_cast<float4*>(posm); ca.vel = reinterpret_cast<float4*>(vel); ca.acc = reinterpret_cast<float4*>(acc);
    ca.G = G; ca.eps2 = eps * eps; ca.dt = dt; ca.pot = pot; ca.nsteps = nsteps; ca.acc_valid = acc_valid;
    ca.n = (int32_t)plan.n; ca.n8 = (int32_t)plan.n8; ca.S = plan.S; ca.Ttile = plan.T;
    const size_t smem = cluster_geometry<float>(plan, g_cluster_size, &ca.tpc);
    return launch_cluster<ClusterF32, float>(ca, g_cluster_size, smem, stream);
}

// Flag-in-data whole-loop kernel (ll_kdk.cuh): bytes of the exchange buffer the call needs, 0 = the call does not fit.
size_t ll_fits_f32(const PairPlan& plan)
{
    int32_t tpc, ctas;
    size_t xbytes = 0;
    return ll_geometry<float>(plan, g_ll_max_ctas, &tpc, &ctas, &xbytes) != 0 ? xbytes : 0;
}

cudaError_t launch_ll_f32(const PairPlan& plan, float* posm, float* vel, float* acc, float G, float eps, float dt,
                          const PotParams<float>& pot, int64_t nsteps, int acc_valid, void* xbuf, float* tape, cudaStream_t stream)
{
    LLArgs<float> ca;
    ca.posm = reinterpret_cast<float4*>(posm); ca.vel = reinterpret_cast<float4*>(vel); ca.acc = reinterpret_cast<float4*>(acc);
    ca.G = G; ca.eps2 = eps * eps; ca.dt = dt; ca.pot = pot; ca.nsteps = nsteps; ca.acc_valid = acc_valid;
    ca.n = (int32_t)plan.n; ca.n8 = (int32_t)plan.n8; ca.S = plan.S; ca.Ttile = plan.T;
    ca.xbuf = static_cast<unsigned long long*>(xbuf);
    ca.tape = reinterpret_cast<float4*>(tape);
    int32_t ctas;
    size_t xbytes;
    const size_t smem = ll_geometry<float>(plan, g_ll_max_ctas, &ca.tpc, &ctas, &xbytes);
    cudaError_t e = cudaMemsetAsync(xbuf, 0, xbytes, stream);          // tags start at 1
    if (e != cudaSuccess) return e;
    return launch_ll<LLF32, float>(ca, ctas, smem, LL_TAPE_CODE_FLOAT, stream);
}

// The instantiation launch_pair_f32 selects, spelled from the template arguments themselves (odisseo_pair_kernel_name).
template <int A, int B, int C, int D, int E>
static std::string stream_kernel_name(const PairF32<A, B, C, D, E>*)
{
    char buf[96];
    snprintf(buf, sizeof buf, "stream_kernel<PairF32<%d,%d,%d,%d,%d>>", A, B, C, D, E);
    return buf;
}
const char* pair_kernel_name_f32(int variant)
{
    static const std::string names[2] = {stream_kernel_name(static_cast<const LargeF32*>(nullptr)),
                                         stream_kernel_name(static_cast<const SmallF32*>(nullptr))};
    return names[variant ? 1 : 0].c_str();
}

cudaError_t launch_pair_f32(const PairPlan& plan, const float* posm, const void* jsrc, const void* src, double* partials, float eps,
                            cudaStream_t stream)
{
    if (plan.variant == 0) {
        const LargeF32::Params prm{reinterpret_cast<const float4*>(posm), eps * eps};
        return launch_stream<LargeF32>(plan, prm, jsrc, src, partials, stream);
    }
    const SmallF32::Params prm{reinterpret_cast<const float4*>(posm), eps * eps};
    return launch_stream<SmallF32>(plan, prm, jsrc, src, partials, stream);
}

}  // namespace odisseo
