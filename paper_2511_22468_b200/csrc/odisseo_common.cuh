// Shared device/host definitions of the ODISSEO B200 library: the launch plan (stream-K
// decomposition of the (i-block x j-tile) interaction space), PTX wrappers for mbarrier /
// 1-D TMA bulk copies / packed fp32 arithmetic.  sm_100a only.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/odisseo.h"

namespace odisseo {

// ---------------------------------------------------------------------------------------
// Launch plan.  The nt x n interaction matrix (nt = n except for the cross
// call) is cut into nb = ceil(nt / IB) i-blocks (IB targets held in registers by one CTA) times
// S source chunks.  The chunk boundaries are a function of n alone: with n8 = ceil(n / 8) source
// octets, chunk s holds the records [8 floor(s n8 / S), 8 floor((s+1) n8 / S)), and a chunk is
// walked in tiles of at most T records (one TMA copy each).  The U = nb * S units are numbered
// u = b * S + s and dealt to P persistent CTAs in contiguous, equal (+-1) ranges: CTA c owns
// [start(c), start(c+1)), start(c) = floor(c*U/P).  Every unit writes its own row of partial sums
// (row index = u), and the reduce step adds the S rows of an i-block in increasing s: the value
// a target receives is  G m0 sum_s ( sum_{tiles of chunk s} fp32 tile sum ),  a fixed grouping
// that depends on n only -- not on the number of targets, CTAs or ranks (SURVEY.md 8f NEXT-1:
// "same fixed reduction order per i"), with no atomics: bit-reproducible.
// S is chosen on the host by a cost model of the busiest CTA (source_split, api.cu): at n = 2^18 on 148 SMs
// S = 15, U = 128 * 15 = 1,920 units, 12 or 13 per CTA.
// ---------------------------------------------------------------------------------------
struct PairPlan {
    int64_t n;        // source particles (staged, chunked along j)
    int64_t nt;       // target particles (held in registers, blocked along i); == n except for the cross call
    int64_t n8;       // source octets = ceil(n / 8); the staged array holds 8 * n8 records
    int64_t U;        // work units = nb * S = rows of the partial buffer
    int32_t IB;       // targets per i-block = ipt * cthreads
    int32_t T;        // most source records per tile (a function of n)
    int32_t S;        // source chunks (a function of n and the SM count)
    int32_t nb;       // i-blocks
    int32_t P;        // persistent CTAs (grid size)
    int32_t ipt;      // i-bodies per thread
    int32_t cthreads; // compute threads per CTA (one extra producer warp is added at launch)
    int32_t variant;  // 0 = large (8 compute warps), 1 = small (2 compute warps)
    int32_t rec_bytes;// bytes per staged source record
    int32_t comps;    // planes of IB doubles per row (3: x, y, z sums)
    int32_t direct;   // 1: the sources are read from the caller's posm array itself (n records, no padding): the last tile ends at n
};

__host__ __device__ __forceinline__ int64_t plan_start(const PairPlan& p, int64_t c) {
    return (c * p.U) / p.P;
}
// CTA that owns unit u: the largest c with start(c) <= u.
__host__ __device__ __forceinline__ int32_t plan_owner(const PairPlan& p, int64_t u) {
    int64_t c = ((u + 1) * p.P + p.U - 1) / p.U - 1;
    return (int32_t)(c < p.P - 1 ? c : p.P - 1);
}
// First record of source chunk s (s = S gives the end of the staged array).
__host__ __device__ __forceinline__ int64_t plan_chunk_lo(const PairPlan& p, int64_t s) {
    return 8 * ((s * p.n8) / p.S);
}
__host__ __device__ __forceinline__ int64_t plan_npad(const PairPlan& p) { return 8 * p.n8; }
// Equal-mass detection: the kernel that stages the sources also writes one
// int per block of STEP_THREADS particles, non-zero when some mass in the block differs from
// posm[0].m.  The flags sit behind the staged records; the pair kernels OR them at start-up and CTA 0
// records the decision in the word behind the flags (1 = the rows were summed without the mass factor:
// the reduce step multiplies by the mass of staged record 0).
constexpr int STEP_THREADS = 256;
__host__ __device__ __forceinline__ int32_t plan_nflags(const PairPlan& p) {
    return (int32_t)((plan_npad(p) + STEP_THREADS - 1) / STEP_THREADS);
}
// Workspace layout of the staged sources: [flags + decision word, rounded to 256 B][records].  `jsrc` always points
// at the first RECORD; the flags sit in front of it, so that the record array can be longer than 8 * n8 records:
// STAGED_SLACK extra records leave room for an in-place all-gather of equal, 8-aligned slices of up to 128 ranks
// (sharded form).  The kernels never read a record past 8 * n8.
constexpr int64_t STAGED_SLACK = 1024;
__host__ __device__ __forceinline__ size_t plan_flag_bytes(const PairPlan& p) {
    // [256 B grid-barrier block: arrival counter | release flag, 128 B apart][flags, decision word], rounded to 256 B
    return 256 + ((((size_t)plan_nflags(p) + 1) * sizeof(int) + 255) & ~(size_t)255);
}
__host__ __device__ __forceinline__ size_t plan_jsrc_bytes(const PairPlan& p) {
    const size_t b = plan_flag_bytes(p) + (size_t)(plan_npad(p) + STAGED_SLACK) * p.rec_bytes;
    return (b + 255) & ~(size_t)255;
}
__host__ __device__ __forceinline__ void* plan_records(void* ws, const PairPlan& p) {
    return static_cast<unsigned char*>(ws) + plan_flag_bytes(p);
}
__host__ __device__ __forceinline__ const int* plan_flags(const void* jsrc, const PairPlan& p) {
    return reinterpret_cast<const int*>(static_cast<const unsigned char*>(jsrc) - plan_flag_bytes(p) + 256);
}
__host__ __device__ __forceinline__ const int* plan_eqm_word(const void* jsrc, const PairPlan& p) {
    return plan_flags(jsrc, p) + plan_nflags(p);
}
// 256-byte block of the whole-loop kernel's grid barrier (fused_step.cuh), zeroed by the host before each launch:
// word 0 = arrival counter, word 32 (another 128-byte line) = release flag.
__host__ __device__ __forceinline__ unsigned* plan_barrier_block(void* jsrc, const PairPlan& p) {
    return reinterpret_cast<unsigned*>(static_cast<unsigned char*>(jsrc) - plan_flag_bytes(p));
}
// Padding records of the staged source array: zero mass, parked so far away that the softened
// inverse cube underflows to exactly 0 (ftz) -- they contribute 0 with or without the mass factor.
constexpr float PAD_POS_F32 = 3.0e18f;
constexpr double PAD_POS_F64 = 1.0e150;
// The area of the unit rows also serves the flag-in-data whole-loop kernels (ll_kdk.cuh), which need no rows but two
// buffers of tagged exchange words: at most 2 x 6 x 8 bytes per particle (fp64), for n up to LL_MAX_N.
constexpr int LL_MAX_N = 6144;                    // upper bound of odisseo_set_ll_max_n; shared memory bounds it further
__host__ __device__ __forceinline__ size_t plan_partial_bytes(const PairPlan& p) {
    const size_t rows = (size_t)p.U * p.comps * p.IB * sizeof(double);
    const size_t exchange = p.n <= LL_MAX_N ? (size_t)(p.n + 1) * 96 : 0;
    return rows > exchange ? rows : exchange;
}

#if defined(__CUDACC__)
// Reduce step: the S rows of target i's i-block added in increasing s (fixed order), NCOMP planes.
// Rows are fetched REDUCE_BATCH at a time so the L2 latencies of a batch overlap (a plain loop serialises
// one ~1 us round trip per row); absent rows add +0.0, which leaves the sum unchanged.
template <int NCOMP>
__device__ __forceinline__ void reduce_unit_rows(const double* __restrict__ partials, const PairPlan& plan, const int64_t i,
                                                 double (&sum)[NCOMP])
{
    constexpr int REDUCE_BATCH = 8;
    const int32_t b = (int32_t)(i / plan.IB);
    const int32_t r = (int32_t)(i - (int64_t)b * plan.IB);
    const size_t stride = (size_t)plan.comps * plan.IB;
    const double* base = partials + (size_t)b * plan.S * stride + r;
#pragma unroll
    for (int k = 0; k < NCOMP; ++k) sum[k] = 0.0;
    for (int32_t s = 0; s < plan.S; s += REDUCE_BATCH) {
        double v[REDUCE_BATCH][NCOMP];
#pragma unroll
        for (int q = 0; q < REDUCE_BATCH; ++q) {
            const bool live = s + q < plan.S;
            const double* row = base + (size_t)(s + (live ? q : 0)) * stride;
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) v[q][k] = live ? __ldcg(row + (size_t)k * plan.IB) : 0.0;
        }
#pragma unroll
        for (int q = 0; q < REDUCE_BATCH; ++q)
#pragma unroll
            for (int k = 0; k < NCOMP; ++k) sum[k] += v[q][k];
    }
}
// Factor the pair kernel left out of the rows: the common mass when it took the equal-mass loop, else 1.
// records: the array the pair kernel read its sources from (the staged array, or posm itself when plan.direct).
template <typename T>
__device__ __forceinline__ double plan_row_mass(const void* __restrict__ jsrc, const PairPlan& plan, const void* __restrict__ records)
{
    // both loads are issued unconditionally (no dependent round trip: at small N the reduce is latency-bound)
    const int eqm = __ldcg(plan_eqm_word(jsrc, plan));
    // mass of source record 0 ({x, y, z, m} in both precisions)
    const double m0 = sizeof(T) == 4 ? (double)__ldcg(static_cast<const float*>(records) + 3) : __ldcg(static_cast<const double*>(records) + 3);
    return eqm != 0 ? m0 : 1.0;
}
#endif

PairPlan make_plan(int64_t n, int is_f64, int num_sms);
PairPlan make_cross_plan(int64_t nt, int64_t n, int is_f64, int num_sms);   // nt targets against n sources

// External potential with the host-side pre-combined products (reading R4).
template <typename T> struct PotParams {
    T GMs, inv_rs;   // NFW: G*M_s, 1/r_s   (GMs == 0 disables)
    T GMd, a, b2;    // MN:  G*M, a, b^2    (GMd == 0 disables)
    // bulge (GMb == 0 disables): G*M_b, 1/r_c, s = (3 - alpha)/2, ln Gamma(s), and for the potential
    // s - 1/2, ln Gamma(s - 1/2) and Gamma(s - 1/2) / (r_c Gamma(s))
    T GMb, inv_rc, bs, lgam_s, bs_half, lgam_s_half, phi_outer;
};
constexpr int VJP_NOUT = 10;      // gradient slots: M_s, r_s, M_d, a, b, G, eps, dt, M_b, r_c

// Per-simulation parameters of the ensemble kernel (ensemble.cu), device layout, 32 bytes.
struct EnsembleParams {
    float G, eps2, dt;
    PotParams<float> pot;
};
// The same in double for the O(N) parts of the ensemble pull-back (ensemble_adjoint.cu), 64 bytes.
struct EnsembleParams64 {
    double G, eps, dt;
    PotParams<double> pot;
};
constexpr int ENSEMBLE_MAX_N = 2048;

// Step-kernel flags.
enum : int {
    STEP_FROM_PARTIALS = 1,   // a_pair = G * fixed-order sum of partial rows (else read acc)
    STEP_CLOSE = 2,           // closing half kick  v += a dt/2  (end of a step)
    STEP_OPEN = 4,            // opening half kick + drift: v += a dt/2; x += v dt (start of next step)
    STEP_PACK_ONLY = 8,       // only (re)write the staged source array from posm
    STEP_SNAPSHOT = 16,       // no kick: only store the tape snapshot {x, v, pair-only a} (nsteps == 0 with a tape)
    STEP_SLICE = 32,          // the arrays address a slice [lo, lo + count) of the plan's particles (sharded form)
    STEP_NO_STAGE = 64        // write the equal-mass flags but no staged records: the pair kernel reads posm itself (plan.direct)
};

// ---------------------------------------------------------------------------------------
// PTX wrappers
// ---------------------------------------------------------------------------------------
#if defined(__CUDACC__)
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// The producer lane's wait: it has a whole tile time (microseconds) of slack, so it backs off between polls instead
// of competing with the two compute warps of its scheduler for issue slots (the plain loop retired ~7 % of the
// kernel's warp instructions, all on one of the four schedulers).
__device__ __forceinline__ void mbar_wait_backoff(uint64_t* bar, uint32_t parity) {
    uint32_t done = 0;
    while (true) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (done) break;
        __nanosleep(256);
    }
}
// 1-D TMA bulk copy global -> shared, completion signalled on an mbarrier.  dst, src and
// bytes must be multiples of 16.  SASS: UBLKCP.
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// Packed fp32 pairs in 64-bit registers (FFMA2 / FADD2 / FMUL2 on sm_100a).
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpk(f32x2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("sub.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("add.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 r;
    asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
// Programmatic dependent launch (sm_90+): a kernel launched with launch_pdl() may become resident while
// its predecessor in the stream is still running; pdl_wait() blocks until the predecessor has completed
// and its writes are visible, so everything before it (barrier init, plan arithmetic) overlaps the
// predecessor's tail and the launch latency.  pdl_launch_dependents() lets the NEXT kernel start that
// early; it is issued first thing, which is safe because the dependent's pdl_wait() still waits for full
// completion.  Both are no-ops when the kernel was launched without the attribute.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Double-precision reciprocal-square-root seed (MUFU.RSQ64H): ~22 good bits, low word zero.
__device__ __forceinline__ double rsqrt_approx_f64(double x) {
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    return r;
}
#endif  // __CUDACC__

#if defined(__CUDACC__)
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
#endif

// launchers (defined in pair_f32.cu / pair_f64.cu / integrate.cu)
cudaError_t launch_pair_f32(const PairPlan& plan, const float* posm, const void* jsrc, const void* src, double* partials,
                            float eps, cudaStream_t stream);
cudaError_t launch_pair_f64(const PairPlan& plan, const double* posm, const void* jsrc, const void* src, double* partials,
                            double eps, cudaStream_t stream);
cudaError_t launch_step_f32(const PairPlan& plan, float* posm, float* vel, float* acc, void* jsrc,
                            const double* partials, float G, const PotParams<float>& pot, float dt, int flags,
                            float* snapshot, int64_t lo, int64_t count, cudaStream_t stream);
cudaError_t launch_step_f64(const PairPlan& plan, double* posm, double* vel, double* acc, void* jsrc,
                            const double* partials, double G, const PotParams<double>& pot, double dt, int flags,
                            double* snapshot, int64_t lo, int64_t count, cudaStream_t stream);
cudaError_t launch_ext_f32(const float* posm, float* acc, int64_t n, const PotParams<float>& pot, int accumulate,
                           cudaStream_t stream);
cudaError_t launch_ext_f64(const double* posm, double* acc, int64_t n, const PotParams<double>& pot, int accumulate,
                           cudaStream_t stream);
cudaError_t launch_soa_pack_f32(const float* x, const float* y, const float* z, const float* m, float* posm,
                                int64_t n, cudaStream_t stream);
cudaError_t launch_soa_unpack_f32(const float* acc, float* ax, float* ay, float* az, int64_t n, cudaStream_t stream);
cudaError_t launch_reduce_rows_f32(const PairPlan& plan, const double* partials, const void* jsrc, const void* records, float G,
                                   float* acc, cudaStream_t stream);
cudaError_t launch_reduce_rows_f64(const PairPlan& plan, const double* partials, const void* jsrc, const void* records, double G,
                                   double* acc, cudaStream_t stream);
cudaError_t launch_potential_f64(const PairPlan& plan, const void* jsrc, double* partials, double eps,
                                 cudaStream_t stream);
// diagnostics.cu: stage (promote to double) / per-particle terms + block sums / final fixed-order sum
constexpr int DIAG_VALUES = 16;
cudaError_t launch_diag_stage_f32(const PairPlan& plan, const float* posm, void* jsrc, cudaStream_t stream);
cudaError_t launch_diag_stage_f64(const PairPlan& plan, const double* posm, void* jsrc, cudaStream_t stream);
cudaError_t launch_diag_terms_f32(const PairPlan& plan, const float* posm, const float* vel, const double* partials,
                                  const void* jsrc, double G, double eps, const PotParams<double>& pot, double* block_sums,
                                  double* phi_out, cudaStream_t stream);
cudaError_t launch_diag_terms_f64(const PairPlan& plan, const double* posm, const double* vel, const double* partials,
                                  const void* jsrc, double G, double eps, const PotParams<double>& pot, double* block_sums,
                                  double* phi_out, cudaStream_t stream);
cudaError_t launch_diag_final(const double* block_sums, int nblocks, double* out, cudaStream_t stream);
// adjoint.cu
void vjp_geometry(int is_f64, int* ipt, int* cthreads, int* tile, int* minb);
PairPlan make_vjp_plan(int64_t n, int is_f64, int num_sms);          // api.cu
size_t vjp_workspace_bytes(const PairPlan& plan, int is_f64);
cudaError_t launch_accel_vjp_f32(const PairPlan& plan, const float* posm, const float* cot, double G, double eps,
                                 const PotParams<double>& pot, float* gx, double* gm, double* gparams, int with_eps_G, void* ws,
                                 cudaStream_t stream);
cudaError_t launch_accel_vjp_f64(const PairPlan& plan, const double* posm, const double* cot, double G, double eps,
                                 const PotParams<double>& pot, double* gx, double* gm, double* gparams, int with_eps_G, void* ws,
                                 cudaStream_t stream);
cudaError_t launch_leapfrog_vjp_f32(const PairPlan& plan, const float* tape, int64_t nsteps, double G, double eps, float dt,
                                    const PotParams<double>& pot64, const PotParams<float>& pot, int with_eps_G, float* lx, float* lv,
                                    double* gm, double* gparams, void* ws, int64_t* launches, cudaStream_t stream);
cudaError_t launch_leapfrog_vjp_f64(const PairPlan& plan, const double* tape, int64_t nsteps, double G, double eps, double dt,
                                    const PotParams<double>& pot64, const PotParams<double>& pot, int with_eps_G, double* lx, double* lv,
                                    double* gm, double* gparams, void* ws, int64_t* launches, cudaStream_t stream);
cudaError_t configure_vjp();
cudaError_t launch_ensemble_f32(float* posm, float* vel, const EnsembleParams* params, int shared_params, int n,
                                int64_t nsim, int64_t nsteps, float* tape, cudaStream_t stream);
cudaError_t launch_ensemble_vjp_f32(const float* tape, const EnsembleParams64* params, int shared_params, int n,
                                    int64_t nsim, int64_t nsteps, int with_eps_G, float* lx, float* lv, double* gm,
                                    double* gparams, int accumulate, cudaStream_t stream);
// mmd.cu
size_t mmd_workspace_bytes(int64_t n, int64_t m, int64_t nsim);
cudaError_t launch_mmd_f32(const float* xpos, const float* xvel, int64_t n, const float* ypos, const float* yvel, int64_t m,
                           int shared_y, const double inv_sigma[6], int64_t nsim, const double* grad_scale, double* mmd2,
                           float* gpos, float* gvel, void* ws, cudaStream_t stream);
size_t mmd_static_scratch_bytes();
cudaError_t launch_mmd_f32_static(const float* xpos, const float* xvel, int64_t n, const float* ypos, const float* yvel,
                                  int64_t m, int shared_y, const double inv_sigma[6], int64_t nsim, const double* grad_scale,
                                  double* mmd2, float* gpos, float* gvel, cudaStream_t stream);
const char* pair_kernel_name_f32(int variant);
const char* pair_kernel_name_f64(int variant);
cudaError_t configure_pair_f32(int num_sms);
cudaError_t configure_pair_f64(int num_sms);
// whole-loop kernels (fused_step.cuh)
int fused_max_ctas_f32(int variant);
int fused_max_ctas_f64(int variant);
cudaError_t launch_fused_f32(const PairPlan& plan, float* posm, float* vel, float* acc, void* jsrc, double* partials, float G, float eps,
                             float dt, const PotParams<float>& pot, int64_t nsteps, int acc_valid, unsigned* barrier, cudaStream_t stream);
cudaError_t launch_fused_f64(const PairPlan& plan, double* posm, double* vel, double* acc, void* jsrc, double* partials, double G,
                             double eps, double dt, const PotParams<double>& pot, int64_t nsteps, int acc_valid, unsigned* barrier,
                             cudaStream_t stream);

// cluster kernels (cluster_kdk.cuh): the whole KDK loop of a small simulation on one thread-block cluster
constexpr int CLUSTER_MAX_N = 4096;               // upper bound of the knob; shared memory bounds it further
bool cluster_fits_f32(const PairPlan& plan);
bool cluster_fits_f64(const PairPlan& plan);
cudaError_t launch_cluster_f32(const PairPlan& plan, float* posm, float* vel, float* acc, float G, float eps, float dt,
                               const PotParams<float>& pot, int64_t nsteps, int acc_valid, cudaStream_t stream);
cudaError_t launch_cluster_f64(const PairPlan& plan, double* posm, double* vel, double* acc, double G, double eps, double dt,
                               const PotParams<double>& pot, int64_t nsteps, int acc_valid, cudaStream_t stream);
// flag-in-data whole-loop kernels (ll_kdk.cuh): owner-computes on all SMs, one L2 round trip per step
size_t ll_fits_f32(const PairPlan& plan);         // bytes of exchange buffer needed, 0 = the call does not fit
size_t ll_fits_f64(const PairPlan& plan);
cudaError_t launch_ll_f32(const PairPlan& plan, float* posm, float* vel, float* acc, float G, float eps, float dt,
                          const PotParams<float>& pot, int64_t nsteps, int acc_valid, void* xbuf, float* tape, cudaStream_t stream);
cudaError_t launch_ll_f64(const PairPlan& plan, double* posm, double* vel, double* acc, double G, double eps, double dt,
                          const PotParams<double>& pot, int64_t nsteps, int acc_valid, void* xbuf, double* tape, cudaStream_t stream);

}  // namespace odisseo
