// Pipe-rate micro-benchmarks (SURVEY.md section 7 step 0, section 8d "verify with step-0
// micro-benchmarks"): instrumentation, not part of the hot path.  One persistent grid of
// ctas_per_sm * SMs CTAs runs `iters` iterations of a register-only instruction stream and is timed
// with CUDA events on the launching stream; bench.py turns the counts into operations per clock per
// SM and prints them beside the nominal peaks (roofline.peak_measured).
//
// Every arithmetic instruction is inline PTX so that the SASS stream is the one named in the table
// (FFMA / FFMA2 / FADD2 / FMUL2 / MUFU.RSQ / DFMA / LDS.128); chains are independent of each other
// and each chain depends on itself, so the loop measures throughput once enough warps are resident.
// The "mix" kinds interleave the pair kernel's instruction mix (11 or 12 packed FP32 ops + 2 MUFU.RSQ
// + 1/2 LDS.128 per two interactions) without its data flow: they measure what
// the issue/dispatch logic allows for that mix, i.e. the reachable bound of the pair kernel.
#include "odisseo_common.cuh"

namespace odisseo {
namespace {

enum UbenchKind : int {
    UB_FFMA = 0,          // scalar FFMA, 3 distinct source registers
    UB_FFMA2_3SRC,        // packed FFMA2 d = a_k * b_k + d_k : 3 distinct 64-bit sources
    UB_FFMA2_SHARED,      // packed FFMA2 d = a_k * b + d_k   : one source shared by all chains (operand reuse)
    UB_FFMA2_SQUARE,      // packed FFMA2 d = a_k * a_k + d_k : 2 distinct 64-bit sources
    UB_FADD2,             // packed FADD2
    UB_FMUL2,             // packed FMUL2
    UB_MUFU_RSQ,          // MUFU.RSQ
    UB_DFMA,              // DFMA
    UB_MIX_FIRST          // interleaved mixes, one per row of kMixes
};

// Interleaved mixes: per loop iteration NP packed FP32 ops (6 FFMA2 with a shared multiplier, 3 FADD2, the
// rest FMUL2 -- the pair body's own proportions), NM MUFU.RSQ, NA integer ALU-pipe ops, NS scalar FFMA and
// NL broadcast LDS.128 per TWO iterations whose words are operands of the following packed ops.
struct MixSpec { const char* name; int NP, NM, NA, NS, NL; };
constexpr MixSpec kMixes[] = {
    {"mix_11p", 11, 0, 0, 0, 0},
    {"mix_11p_1mufu", 11, 1, 0, 0, 0},
    {"mix_11p_2mufu", 11, 2, 0, 0, 0},                 // equal-mass pair body without its loads
    {"mix_11p_4mufu", 11, 4, 0, 0, 0},
    {"mix_12p_2mufu", 12, 2, 0, 0, 0},                 // general-mass pair body without its loads
    {"mix_11p_2alu", 11, 0, 2, 0, 0},
    {"mix_11p_2ffma", 11, 0, 0, 2, 0},
    {"mix_11p_1lds_per2", 11, 0, 0, 0, 1},
    {"mix_11p_2mufu_1lds_per2", 11, 2, 0, 0, 1},       // equal-mass pair body (3/8 + overhead ~ 1/2 LDS per iteration)
    {"mix_12p_2mufu_1lds_per2", 12, 2, 0, 0, 1},       // general-mass pair body
    {"mix_11p_2mufu_2lds_per2", 11, 2, 0, 0, 2},
    {"mix_22ffma_2mufu", 0, 2, 0, 22, 0},              // the unpacked (scalar) form of the equal-mass body
};
constexpr int NMIX = (int)(sizeof(kMixes) / sizeof(kMixes[0]));
constexpr int UB_KINDS = UB_MIX_FIRST + NMIX;

const char* const kPureNames[UB_MIX_FIRST] = {"ffma", "ffma2_3src", "ffma2_shared", "ffma2_square", "fadd2", "fmul2",
                                              "mufu_rsq", "dfma"};

// per iteration and thread: {FP32-pipe lane operations, MUFU results, FP64 operations, shared loads}
struct UbenchCounts { double fp32, mufu, fp64, lds; };
__host__ UbenchCounts counts_of(int kind)
{
    switch (kind) {
        case UB_FFMA: return {12, 0, 0, 0};
        case UB_FFMA2_3SRC: case UB_FFMA2_SHARED: case UB_FFMA2_SQUARE: case UB_FADD2: case UB_FMUL2: return {24, 0, 0, 0};
        case UB_MUFU_RSQ: return {0, 8, 0, 0};
        case UB_DFMA: return {0, 0, 8, 0};
    }
    const MixSpec& m = kMixes[kind - UB_MIX_FIRST];
    return {2.0 * m.NP + m.NS, (double)m.NM, 0, 0.5 * m.NL};
}

__device__ __forceinline__ float ffma(float a, float b, float c)
{
    float r;
    asm("fma.rn.ftz.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}
__device__ __forceinline__ double dfma(double a, double b, double c)
{
    double r;
    asm("fma.rn.f64 %0, %1, %2, %3;" : "=d"(r) : "d"(a), "d"(b), "d"(c));
    return r;
}
template <int KIND>
__global__ void __launch_bounds__(1024) ubench_kernel(float* __restrict__ out, const int64_t iters, const float seed)
{
    __shared__ __align__(16) float tile[1024];
    const int tid = threadIdx.x;
    tile[tid & 1023] = seed;
    __syncthreads();
    float sink = 0.f;

    if constexpr (KIND == UB_FFMA) {
        float a[12], b[12], d[12];
#pragma unroll
        for (int k = 0; k < 12; ++k) { a[k] = seed + k; b[k] = 1.0f / (seed + k + tid); d[k] = (float)tid; }
        for (int64_t it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < 12; ++k) d[k] = ffma(a[k], b[k], d[k]);
        }
#pragma unroll
        for (int k = 0; k < 12; ++k) sink += d[k];
    } else if constexpr (KIND == UB_FFMA2_3SRC || KIND == UB_FFMA2_SHARED || KIND == UB_FFMA2_SQUARE || KIND == UB_FADD2 ||
                         KIND == UB_FMUL2) {
        f32x2 a[12], b[12], d[12];
        const f32x2 nz = pk(-0.0f, -0.0f);
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            a[k] = add2(pk(seed + k, seed - k), nz);
            b[k] = add2(pk(1.0f / (seed + k + tid), 1.0f / (seed + 2 * k + tid)), nz);
            d[k] = add2(pk((float)tid, (float)k), nz);
        }
        const f32x2 one = add2(pk(seed, seed), nz);
        for (int64_t it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < 12; ++k) {
                if constexpr (KIND == UB_FFMA2_3SRC) d[k] = fma2(a[k], b[k], d[k]);
                if constexpr (KIND == UB_FFMA2_SHARED) d[k] = fma2(one, a[k], d[k]);
                if constexpr (KIND == UB_FFMA2_SQUARE) d[k] = fma2(a[k], a[k], d[k]);
                if constexpr (KIND == UB_FADD2) d[k] = add2(d[k], a[k]);
                if constexpr (KIND == UB_FMUL2) d[k] = mul2(d[k], one);
            }
        }
#pragma unroll
        for (int k = 0; k < 12; ++k) { float lo, hi; unpk(d[k], lo, hi); sink += lo + hi; }
    } else if constexpr (KIND == UB_MUFU_RSQ) {
        float r[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) r[k] = seed + k + tid;
        for (int64_t it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < 8; ++k) r[k] = rsqrt_approx(r[k]);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) sink += r[k];
    } else if constexpr (KIND == UB_DFMA) {
        double a[8], d[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) { a[k] = 1.0 / (seed + k + tid); d[k] = tid; }
        const double b = seed;
        for (int64_t it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < 8; ++k) d[k] = dfma(a[k], b, d[k]);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) sink += (float)d[k];
    } else {
        constexpr MixSpec M = kMixes[KIND - UB_MIX_FIRST];
        constexpr int NP = M.NP, NM = M.NM, NA = M.NA, NS = M.NS, NL = M.NL;
        constexpr int NPA = NP > 0 ? NP : 1, NSA = NS > 0 ? NS : 1;
        f32x2 a[NPA], d[NPA];
        float sa[NSA], sd[NSA];
        const f32x2 nz = pk(-0.0f, -0.0f);
#pragma unroll
        for (int k = 0; k < NPA; ++k) {
            a[k] = add2(pk(1.0f / (seed + k + tid), 1.0f / (seed + 2 * k + tid)), nz);
            d[k] = add2(pk((float)tid, (float)k), nz);
        }
#pragma unroll
        for (int k = 0; k < NSA; ++k) { sa[k] = 1.0f / (seed + 3 * k + tid); sd[k] = (float)(tid + k); }
        f32x2 one = add2(pk(seed, seed), nz);
        f32x2 addend = a[NPA > 6 ? 6 : 0];
        float sw = seed;
        const ulonglong2* __restrict__ rec = reinterpret_cast<const ulonglong2*>(tile);
        float r[4] = {seed + tid, seed + 2 * tid, seed + 3 * tid, seed + 4 * tid};
        uint32_t q[2] = {(uint32_t)tid, (uint32_t)(tid * 3)};
        for (int64_t it = 0; it < iters; it += 2) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (NL >= 1 && h == 0) { const ulonglong2 v = rec[(it >> 1) & 63]; one = v.x; addend = v.y; }
                if (NL >= 2 && h == 1) { const ulonglong2 v = rec[64 + ((it >> 1) & 63)]; one = v.x; addend = v.y; }
                constexpr int SLOTS = NP > NS ? NP : NS;
#pragma unroll
                for (int k = 0; k < SLOTS; ++k) {
                    if (k < NP) {
                        if (k < 6) d[k] = fma2(one, a[k], d[k]);
                        else if (k < 9) d[k] = add2(d[k], k == 6 ? addend : a[k]);
                        else d[k] = mul2(d[k], one);
                    }
                    if (NP == 0 && k < NS) sd[k] = ffma(sw, sa[k], sd[k]);
                    if (NP > 0 && k < NS) sd[k] = ffma(sw, sa[k], sd[k]);
                    // the other pipes' instructions are spread evenly over the iteration
                    if (NM >= 1 && k == (SLOTS * 1) / 5) r[0] = rsqrt_approx(r[0]);
                    if (NM >= 2 && k == (SLOTS * 3) / 5) r[1] = rsqrt_approx(r[1]);
                    if (NM >= 3 && k == (SLOTS * 2) / 5) r[2] = rsqrt_approx(r[2]);
                    if (NM >= 4 && k == (SLOTS * 4) / 5) r[3] = rsqrt_approx(r[3]);
                    if (NA >= 1 && k == (SLOTS * 1) / 5) asm volatile("xor.b32 %0, %0, %1;" : "+r"(q[0]) : "r"(q[1]));
                    if (NA >= 2 && k == (SLOTS * 3) / 5) asm volatile("xor.b32 %0, %0, %1;" : "+r"(q[1]) : "r"(q[0]));
                }
            }
        }
#pragma unroll
        for (int k = 0; k < NPA; ++k) { float lo, hi; unpk(d[k], lo, hi); sink += lo + hi; }
#pragma unroll
        for (int k = 0; k < NSA; ++k) sink += sd[k];
        sink += r[0] + r[1] + r[2] + r[3] + __uint_as_float(q[0] ^ q[1]);
    }
    if (sink == 123.456f) out[0] = sink;      // keeps the chains alive; practically never true
}

template <int KIND>
cudaError_t launch_kind(int grid, int threads, float* out, int64_t iters, cudaStream_t s)
{
    ubench_kernel<KIND><<<grid, threads, 0, s>>>(out, iters, 1.0f);
    return cudaGetLastError();
}

template <int K>
cudaError_t launch_from(int kind, int grid, int threads, float* out, int64_t iters, cudaStream_t s)
{
    if constexpr (K >= UB_KINDS) {
        return cudaErrorInvalidValue;
    } else {
        if (kind == K) return launch_kind<K>(grid, threads, out, iters, s);
        return launch_from<K + 1>(kind, grid, threads, out, iters, s);
    }
}

cudaError_t launch_ubench(int kind, int grid, int threads, float* out, int64_t iters, cudaStream_t s)
{
    return launch_from<0>(kind, grid, threads, out, iters, s);
}

}  // namespace
}  // namespace odisseo

using namespace odisseo;

extern "C" {

int odisseo_ubench_kinds(void) { return (int)UB_KINDS; }

const char* odisseo_ubench_name(int kind)
{
    if (kind < 0 || kind >= UB_KINDS) return nullptr;
    return kind < UB_MIX_FIRST ? kPureNames[kind] : kMixes[kind - UB_MIX_FIRST].name;
}

odisseo_status odisseo_ubench_run(int kind, int ctas_per_sm, int threads, int64_t iters, double h_out[6], void* stream)
{
    if (!h_out) return ODISSEO_ERR_NULL;
    if (kind < 0 || kind >= (int)UB_KINDS || ctas_per_sm < 1 || ctas_per_sm > 32 || threads < 32 || threads > 1024 ||
        (threads & 31) || iters < 2 || (iters & 1))
        return ODISSEO_ERR_ARG;
    int dev = 0, sms = 0, major = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return ODISSEO_ERR_CUDA; }
    if (major != 10) return ODISSEO_ERR_ARCH;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    float* d_out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    e = cudaMalloc(&d_out, 256);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    float best = 0.f;
    const int grid = sms * ctas_per_sm;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {     // rep 0 is the warm-up
        e = cudaEventRecord(e0, s);
        if (e == cudaSuccess) e = launch_ubench(kind, grid, threads, d_out, iters, s);
        if (e == cudaSuccess) e = cudaEventRecord(e1, s);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && (best == 0.f || ms < best)) best = ms;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (d_out) cudaFree(d_out);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return ODISSEO_ERR_CUDA; }
    const UbenchCounts c = counts_of(kind);
    const double total = (double)grid * threads * (double)iters;
    h_out[0] = (double)best;
    h_out[1] = c.fp32 * total;
    h_out[2] = c.mufu * total;
    h_out[3] = c.fp64 * total;
    h_out[4] = c.lds * total;
    h_out[5] = (double)sms;
    return ODISSEO_OK;
}

}  // extern "C"
