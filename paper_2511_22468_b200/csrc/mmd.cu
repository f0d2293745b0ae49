// Maximum Mean Discrepancy between simulated and observed 6-D point clouds and its gradient with respect to the
// simulated cloud (Fig. 2 step 4 "compared to the observed stream using the Maximum Mean Discrepancy
// (MMD), and the gradient of the loss is computed"; L39 "full 6D phase-space information"; L47).
// The paper prints neither kernel nor estimator; reading R20: Gaussian kernel with one scale per
// coordinate, biased V-statistic,
//
//   k(u, v)     = exp(-1/2 sum_d ((u_d - v_d)/sigma_d)^2),  d = x, y, z, vx, vy, vz
//   MMD^2(X, Y) = 1/n^2 sum_ii' k(x_i, x_i') + 1/m^2 sum_jj' k(y_j, y_j') - 2/(n m) sum_ij k(x_i, y_j)
//   dMMD^2/dx_i = -2/(n^2 sigma^2) sum_i' k(x_i, x_i') (x_i - x_i') + 2/(n m sigma^2) sum_j k(x_i, y_j) (x_i - y_j)
//
// Batched like the ensemble kernels (the paper's grid search and gradient steps run thousands of N = 1,000 simulations
// against one observed stream, L47): grid = (target blocks, simulations).  All-pairs tiling as in the pair kernels:
// a thread keeps the six scaled coordinates u = x s_d, s_d = sqrt(log2(e)/2)/sigma_d, of TWO targets in registers as packed
// f32x2 pairs, so that two evaluations k = ex2(-|u - u'|^2) cost 6 FADD2 + 6 FFMA2 + 2 MUFU.EX2; source tiles of 256 points
// are staged scaled in shared memory ({x,y,z,vx},{vy,vz}: two broadcast loads per source, each coordinate a scalar
// broadcast operand of the packed instructions); sums are fp32 inside a tile and fp64 across tiles; per-block sums are added
// in block order by a second kernel (fixed order, no atomics: bit-reproducible).  The gradient lands in the layout of
// the pull-back's cotangents (float4 {d/dx, d/dy, d/dz, 0}), so loss -> gradient never leaves the device.
#include <mutex>

#include "odisseo_common.cuh"

namespace odisseo {

namespace {

constexpr int MMD_THREADS = 256;
constexpr int MMD_TILE = 256;
constexpr int MMD_PER_BLOCK = 2 * MMD_THREADS;      // two target slots per thread

struct MmdScales { float s[6]; float back[6]; };    // u = x s_d;  back_d = 4 s_d ln 2 (below)

__device__ __forceinline__ float ex2_approx(float x)
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

__device__ __forceinline__ double mmd_block_sum(double v, double* warp_scratch)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) warp_scratch[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < MMD_THREADS / 32; ++w) s += warp_scratch[w];
    return s;
}

// One pass of the block's targets over a source cloud.  A thread holds TWO targets as packed f32x2 pairs (slots t and
// t + 256 of the block's 512); a source arrives as {x,y,z,vx},{vy,vz} (LDS.128 + LDS.64 broadcasts) and each coordinate
// enters the packed instructions as a scalar operand broadcast to both halves (pair_f32.cu): per source and thread
// 7 FADD2 + 12 FFMA2 + 2 MUFU.EX2 for two kernel evaluations with their gradient terms.  Returns sum_j k per target and,
// when GRAD, adds sum_j k (u_src - u_tgt)_d into acc0 / acc1.
template <bool GRAD>
__device__ __forceinline__ void mmd_pass(const float4* __restrict__ spos, const float4* __restrict__ svel, const int ns,
                                         const MmdScales& sc, const f32x2 (&u)[6], float4* tileA, float2* tileB, double (&acc0)[6],
                                         double (&acc1)[6], double& total0, double& total1)
{
    total0 = total1 = 0.0;
    for (int j0 = 0; j0 < ns; j0 += MMD_TILE) {
        __syncthreads();                                     // the previous tile is consumed
        const int j = j0 + threadIdx.x;
        if (threadIdx.x < MMD_TILE) {
            float4 p = make_float4(0.f, 0.f, 0.f, 0.f), v = p;
            if (j < ns) { p = spos[j]; v = svel[j]; }
            tileA[threadIdx.x] = make_float4(p.x * sc.s[0], p.y * sc.s[1], p.z * sc.s[2], v.x * sc.s[3]);
            tileB[threadIdx.x] = make_float2(v.y * sc.s[4], v.z * sc.s[5]);
        }
        __syncthreads();
        const int len = ns - j0 < MMD_TILE ? ns - j0 : MMD_TILE;
        f32x2 ksum = 0ull, g[6] = {0ull, 0ull, 0ull, 0ull, 0ull, 0ull};
#pragma unroll 4
        for (int t = 0; t < len; ++t) {
            const float4 A = tileA[t];
            const float2 Bv = tileB[t];
            const float s6[6] = {A.x, A.y, A.z, A.w, Bv.x, Bv.y};
            f32x2 d[6], q = 0ull;
#pragma unroll
            for (int c = 0; c < 6; ++c) { d[c] = sub2(pk(s6[c], s6[c]), u[c]); q = fma2(d[c], d[c], q); }
            float ql, qh;
            unpk(q, ql, qh);
            const f32x2 k = pk(ex2_approx(-ql), ex2_approx(-qh));
            ksum = add2(ksum, k);
            if (GRAD) {
#pragma unroll
                for (int c = 0; c < 6; ++c) g[c] = fma2(k, d[c], g[c]);
            }
        }
        float lo, hi;
        unpk(ksum, lo, hi);
        total0 += (double)lo;                                // second summation level, as in the pair kernels
        total1 += (double)hi;
        if (GRAD) {
#pragma unroll
            for (int c = 0; c < 6; ++c) { unpk(g[c], lo, hi); acc0[c] += (double)lo; acc1[c] += (double)hi; }
        }
    }
}

// grid = (ceil(max(n, m) / 512), nsim).  Thread t of block b handles simulated points i0 = b*512 + t and i1 = i0 + 256
// (xx and xy sums, gradient) and the observed points with the same indices (yy sum).
// block_sums[sim][block][3] = {sum k_xx, sum k_xy, sum k_yy}  (with a shared observed cloud sum k_yy is formed by sim 0 only).
template <bool GRAD>
__global__ void __launch_bounds__(MMD_THREADS)
mmd_kernel(const float4* __restrict__ xpos, const float4* __restrict__ xvel, const int n, const float4* __restrict__ ypos,
           const float4* __restrict__ yvel, const int m, const int shared_y, const MmdScales sc,
           const double* __restrict__ grad_scale, float4* __restrict__ gpos, float4* __restrict__ gvel,
           double* __restrict__ block_sums)
{
    __shared__ float4 tileA[MMD_TILE];
    __shared__ float2 tileB[MMD_TILE];
    __shared__ double warp_scratch[MMD_THREADS / 32];
    const int64_t sim = blockIdx.y;
    const float4* const XP = xpos + sim * n;
    const float4* const XV = xvel + sim * n;
    const float4* const YP = ypos + (shared_y ? 0 : sim * m);
    const float4* const YV = yvel + (shared_y ? 0 : sim * m);
    const int base = blockIdx.x * MMD_PER_BLOCK;
    const int i0 = base + threadIdx.x, i1 = i0 + MMD_THREADS;
    const f32x2 nz = pk(-0.0f, -0.0f);

    // scaled coordinates of two points of a cloud as packed pairs (slots beyond the cloud: zeros, their sums are dropped)
    auto load_pair = [&](const float4* P, const float4* V, const int cnt, f32x2 (&u)[6]) {
        float a[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, b[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (i0 < cnt) {
            const float4 p = P[i0], v = V[i0];
            a[0] = p.x * sc.s[0]; a[1] = p.y * sc.s[1]; a[2] = p.z * sc.s[2]; a[3] = v.x * sc.s[3]; a[4] = v.y * sc.s[4]; a[5] = v.z * sc.s[5];
        }
        if (i1 < cnt) {
            const float4 p = P[i1], v = V[i1];
            b[0] = p.x * sc.s[0]; b[1] = p.y * sc.s[1]; b[2] = p.z * sc.s[2]; b[3] = v.x * sc.s[3]; b[4] = v.y * sc.s[4]; b[5] = v.z * sc.s[5];
        }
#pragma unroll
        for (int c = 0; c < 6; ++c) u[c] = add2(pk(a[c], b[c]), nz);
    };

    // ---- simulated points against X and against Y ---------------------------------------------------------------
    double sxx = 0.0, sxy = 0.0, syy = 0.0;
    if (base < n) {                                           // block-uniform: the barriers inside are safe
        f32x2 u[6];
        load_pair(XP, XV, n, u);
        double axx0[6] = {0, 0, 0, 0, 0, 0}, axx1[6] = {0, 0, 0, 0, 0, 0}, axy0[6] = {0, 0, 0, 0, 0, 0}, axy1[6] = {0, 0, 0, 0, 0, 0};
        double xx0, xx1, xy0, xy1;
        mmd_pass<GRAD>(XP, XV, n, sc, u, tileA, tileB, axx0, axx1, xx0, xx1);
        mmd_pass<GRAD>(YP, YV, m, sc, u, tileA, tileB, axy0, axy1, xy0, xy1);
        sxx = (i0 < n ? xx0 : 0.0) + (i1 < n ? xx1 : 0.0);
        sxy = (i0 < n ? xy0 : 0.0) + (i1 < n ? xy1 : 0.0);
        if (GRAD) {
            // with k = ex2(-|u - u'|^2): dk/dx_d = -2 ln2 s_d k (u - u')_d, and the symmetric double sum doubles the xx
            // term: dMMD^2/dx_{i,d} = 4 ln2 s_d [ sum_i' k (u_i' - u_i)_d / n^2 - sum_j k (u_j - u_i)_d / (n m) ];
            // the accumulators hold exactly those two sums
            const double gs = grad_scale ? grad_scale[sim] : 1.0;
            const double cxx = gs / ((double)n * n), cxy = -gs / ((double)n * m);
            if (i0 < n) {
                float o[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) o[c] = (float)((cxx * axx0[c] + cxy * axy0[c]) * (double)sc.back[c]);
                gpos[sim * n + i0] = make_float4(o[0], o[1], o[2], 0.f);
                gvel[sim * n + i0] = make_float4(o[3], o[4], o[5], 0.f);
            }
            if (i1 < n) {
                float o[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) o[c] = (float)((cxx * axx1[c] + cxy * axy1[c]) * (double)sc.back[c]);
                gpos[sim * n + i1] = make_float4(o[0], o[1], o[2], 0.f);
                gvel[sim * n + i1] = make_float4(o[3], o[4], o[5], 0.f);
            }
        }
    }
    // ---- observed points against Y (value only) -------------------------------------------------------------------
    // One observed cloud shared by every simulation (the paper's case: thousands of simulated streams against one observed
    // stream): sum k_yy is the same number for all of them, so only simulation 0 forms it and
    // mmd_final_kernel reads it from there -- a third of the kernel's pair work otherwise.
    if (base < m && (!shared_y || sim == 0)) {
        f32x2 w[6];
        load_pair(YP, YV, m, w);
        double unused0[6] = {0, 0, 0, 0, 0, 0}, unused1[6] = {0, 0, 0, 0, 0, 0}, yy0, yy1;
        mmd_pass<false>(YP, YV, m, sc, w, tileA, tileB, unused0, unused1, yy0, yy1);
        syy = (i0 < m ? yy0 : 0.0) + (i1 < m ? yy1 : 0.0);
    }
    const double bxx = mmd_block_sum(sxx, warp_scratch);
    const double bxy = mmd_block_sum(sxy, warp_scratch);
    const double byy = mmd_block_sum(syy, warp_scratch);
    if (threadIdx.x == 0) {
        double* o = block_sums + ((size_t)sim * gridDim.x + blockIdx.x) * 3;
        o[0] = bxx; o[1] = bxy; o[2] = byy;
    }
}

// mmd2[sim] = sum_blocks xx / n^2 + sum_blocks yy / m^2 - 2 sum_blocks xy / (n m), blocks in order.
__global__ void __launch_bounds__(32)
mmd_final_kernel(const double* __restrict__ block_sums, const int nblocks, const int64_t nsim, const int n, const int m,
                 const int shared_y, double* __restrict__ out)
{
    const int64_t sim = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (sim >= nsim) return;
    double xx = 0.0, xy = 0.0, yy = 0.0;
    for (int b = 0; b < nblocks; ++b) {
        const double* o = block_sums + ((size_t)sim * nblocks + b) * 3;
        xx += o[0]; xy += o[1];
        yy += shared_y ? block_sums[(size_t)b * 3 + 2] : o[2];      // shared observed cloud: simulation 0 holds sum k_yy
    }
    out[sim] = xx / ((double)n * n) + yy / ((double)m * m) - 2.0 * xy / ((double)n * m);
}

}  // namespace

size_t mmd_workspace_bytes(int64_t n, int64_t m, int64_t nsim)
{
    const int64_t big = n > m ? n : m;
    const size_t blocks = (size_t)((big + MMD_PER_BLOCK - 1) / MMD_PER_BLOCK);
    return ((size_t)nsim * blocks * 3 * sizeof(double) + 255) & ~(size_t)255;
}

cudaError_t launch_mmd_f32(const float* xpos, const float* xvel, int64_t n, const float* ypos, const float* yvel, int64_t m,
                           int shared_y, const double inv_sigma[6], int64_t nsim, const double* grad_scale, double* mmd2,
                           float* gpos, float* gvel, void* ws, cudaStream_t stream)
{
    MmdScales sc;
    for (int c = 0; c < 6; ++c) {
        const double s = inv_sigma[c] * 0.84932180028801904272;      // sqrt(log2(e) / 2)
        sc.s[c] = (float)s;
        sc.back[c] = (float)(4.0 * s * 0.69314718055994530942);      // 4 ln2 s_d
    }
    const int64_t big = n > m ? n : m;
    const dim3 grid((unsigned)((big + MMD_PER_BLOCK - 1) / MMD_PER_BLOCK), (unsigned)nsim);
    double* block_sums = static_cast<double*>(ws);
    const float4* xp = reinterpret_cast<const float4*>(xpos);
    const float4* xv = reinterpret_cast<const float4*>(xvel);
    const float4* yp = reinterpret_cast<const float4*>(ypos);
    const float4* yv = reinterpret_cast<const float4*>(yvel);
    if (gpos)
        mmd_kernel<true><<<grid, MMD_THREADS, 0, stream>>>(xp, xv, (int)n, yp, yv, (int)m, shared_y, sc, grad_scale,
                                                           reinterpret_cast<float4*>(gpos), reinterpret_cast<float4*>(gvel), block_sums);
    else
        mmd_kernel<false><<<grid, MMD_THREADS, 0, stream>>>(xp, xv, (int)n, yp, yv, (int)m, shared_y, sc, nullptr, nullptr, nullptr,
                                                            block_sums);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    mmd_final_kernel<<<(unsigned)((nsim + 31) / 32), 32, 0, stream>>>(block_sums, (int)grid.x, nsim, (int)n, (int)m, shared_y, mmd2);
    return cudaGetLastError();
}

// ---- MMD^2 with the library's own scratch (odisseo_mmd2_static_f32) ------------------------------------------------------
// The per-block sums of mmd_kernel normally live in a workspace the caller allocates.  Some callers have no way to do
// that: a loss evaluated from inside a host program whose own memory pool already holds the whole HBM (an ML
// framework that reserves the device at start-up is the usual case for this library's users), or from a code region
// whose rules forbid cudaMalloc because it stalls every stream of the device.  For them the same two kernels run on
// this array instead.  It is part of the library image: every GPU that loads the library holds these bytes until the
// process exits, which is why the size is kept small; problems that need more are refused, not truncated.
constexpr size_t MMD_STATIC_BYTES = (size_t)1 << 20;
static __device__ __align__(256) unsigned char g_mmd_static_scratch[MMD_STATIC_BYTES];

namespace {

// In host code the name g_mmd_static_scratch is only the handle the runtime looks the array up by -- it is NOT the
// address the GPU sees, and must never be handed to a kernel.  The device address is asked for once per device, with
// that device current, and remembered here.
constexpr int MMD_STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;
void* g_static_ptr[MMD_STATIC_MAX_DEVICES] = {};

cudaError_t mmd_static_scratch(void** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);                     // the device the caller made current owns the launch
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MMD_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (g_static_ptr[dev] == nullptr) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_mmd_static_scratch);  // this device's copy of the array
        if (e != cudaSuccess) return e;
        if (p == nullptr) return cudaErrorInvalidSymbol;
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return cudaSuccess;
}

}  // namespace

size_t mmd_static_scratch_bytes() { return MMD_STATIC_BYTES; }

// Same launches as launch_mmd_f32 on the array above; the caller has checked mmd_workspace_bytes(n, m, nsim) against
// mmd_static_scratch_bytes().  Nothing in the array has to start at zero: every block of mmd_kernel stores its three
// sums before mmd_final_kernel (same stream, later) reads exactly those, so what an earlier call left behind is
// never read.  No cudaMalloc / cudaFree here or below.
cudaError_t launch_mmd_f32_static(const float* xpos, const float* xvel, int64_t n, const float* ypos, const float* yvel,
                                  int64_t m, int shared_y, const double inv_sigma[6], int64_t nsim, const double* grad_scale,
                                  double* mmd2, float* gpos, float* gvel, cudaStream_t stream)
{
    void* scratch = nullptr;
    const cudaError_t e = mmd_static_scratch(&scratch);
    if (e != cudaSuccess) return e;
    return launch_mmd_f32(xpos, xvel, n, ypos, yvel, m, shared_y, inv_sigma, nsim, grad_scale, mmd2, gpos, gvel, scratch, stream);
}

}  // namespace odisseo
