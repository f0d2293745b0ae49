// Whole-loop kernel for small N on ONE thread-block cluster (SURVEY.md 8a row a5 "decisive for configs 0-1"; the paper's
// inference runs single N = 1,000 simulations of 1,000 steps).  At N ~ 1,000 a KDK step is ~0.4 us of
// arithmetic on 148 SMs, but every step needs all new positions everywhere: through global memory that is a chain of
// ~8 L2 round trips (8-10 us per step, per-step launches or grid barrier alike).  Here the whole simulation lives in the
// shared memory of a cluster of up to 16 CTAs (16 SMs of one GPC):
//
//   * every CTA holds ALL staged source records in its own shared memory and owns a contiguous slice of the targets;
//   * pair phase: warp items (64 owned targets x source chunk s): two targets per lane, the chunk's records read as
//     shared-memory broadcasts, the Consumer's very inner loop (State::tile of pair_f32.cu / pair_f64.cu);
//   * reduce + integrate: the owner thread of a particle adds its S chunk sums in increasing s (fp64), applies G [m],
//     the external acceleration and the kicks / drift (the arithmetic of step_body.cuh), and PUSHES the new record into
//     the shared memory of every CTA of the cluster with asynchronous distributed-shared-memory stores whose bytes are
//     counted on an mbarrier of the destination CTA (st.async ... mbarrier::complete_tx::bytes);
//   * a CTA starts the next step when its own "inbox" barrier has counted the n records of this step: no cluster-wide
//     barrier, no grid barrier, no launch edge inside the loop; positions, velocities and accelerations never leave
//     the SMs.  Two record buffers and two inbox barriers alternate, which is enough: a CTA pushes step k + 1 only
//     after it has received every push of step k, and a CTA pushes step k only after it has read buffer k.
// Measured (B200, us per KDK step, this kernel / per-step launches): fp32 N = 256 2.5 / 5.2, 512 4.1 / 6.2, 1,024 6.1 / 7.7;
// fp64 256 6.1 / 7.4, 512 7.8 / 8.3, 1,024 13.8 / 10.8.  It runs on 16 of the 148 SMs, so above N ~ 1,000 the pair phase
// (N^2 / 16 per SM; two thirds of a step at N = 1,024) costs more than the latency it saves; the rest of a step is the
// owners' row reduce, kicks + drift + 16 pushes, and the wait for the other CTAs' records
// (profiles/r02_cluster_kdk_ncu_full.txt).  The
// flag-in-data kernel (ll_kdk.cuh: all SMs, one L2 round trip per step) is tried first; this form serves when that
// cooperative grid cannot be placed.
//
// Summation order: chunk and tile boundaries are the launch plan's (functions of n alone), tile sums in the Consumer's
// precision, promoted to fp64 per tile, chunk sums added in increasing s, factor G [m] applied once in fp64 -- the
// canonical grouping of odisseo_common.cuh, so the results are BIT-IDENTICAL to the {pair, step} launch sequence and to
// the cooperative whole-loop kernel (tests).
#pragma once

#include "odisseo_common.cuh"
#include "step_body.cuh"

namespace odisseo {

constexpr int CLUSTER_WARPS = 24;                 // 768 threads per CTA, one CTA per SM
constexpr int CLUSTER_THREADS = CLUSTER_WARPS * 32;
constexpr int CLUSTER_GROUP = 64;                 // targets per warp item (two per lane)
constexpr int CLUSTER_SMEM_MAX = 226 * 1024;      // dynamic shared memory per CTA (the kernel also holds two static barriers)

template <typename T> struct ClusterArgs {
    typename Vec4<T>::type *posm, *vel, *acc;
    T G, eps2, dt;
    PotParams<T> pot;
    int64_t nsteps;
    int32_t acc_valid;
    int32_t n, n8, S, Ttile;                      // the plan's source split (chunks of octets, tile length)
    int32_t tpc;                                  // targets owned per CTA (multiple of CLUSTER_GROUP)
};

// Shared-memory carve (bytes), identical on the host and on the device.
//   cur[2] = 8 n8 staged records {x, y, z, m} each (pushed as they are; fp32 16 B, fp64 32 B per record)
//   part   = (tpc / 64) S items x 3 planes x 64 doubles;  svel, sacc = tpc records each
template <typename T> struct ClusterSmem {
    size_t cur, part, svel, sacc, total;
    __host__ __device__ ClusterSmem(int32_t n, int32_t n8, int32_t S, int32_t tpc)
    {
        const size_t npad = (size_t)8 * n8;
        size_t off = 0;
        cur = off; off += 2 * npad * 4 * sizeof(T);
        off = (off + 127) & ~(size_t)127;
        part = off; off += (size_t)(tpc / CLUSTER_GROUP) * S * 3 * CLUSTER_GROUP * sizeof(double);
        svel = off; off += (size_t)tpc * 4 * sizeof(T);
        sacc = off; off += (size_t)tpc * 4 * sizeof(T);
        total = off;
        (void)n;
    }
};

// ---- cluster primitives (PTX) ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t cluster_nctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t cluster_map(uint32_t smem_addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
// Asynchronous store of one record into the shared memory of a CTA of the cluster; its bytes are counted on an
// mbarrier of the DESTINATION CTA (st.async ... mbarrier::complete_tx::bytes): the receiver waits on its own barrier,
// no cluster-wide barrier and no proxy fence are involved.  addr and mbar are shared::cluster addresses (cluster_map).
__device__ __forceinline__ void st_async_record(uint32_t addr, const float4 v, uint32_t mbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];" ::"r"(addr), "f"(v.x),
                 "f"(v.y), "f"(v.z), "f"(v.w), "r"(mbar)
                 : "memory");
}
__device__ __forceinline__ void st_async_record(uint32_t addr, const double4 v, uint32_t mbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(addr), "d"(v.x), "d"(v.y),
                 "r"(mbar)
                 : "memory");
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(addr + 16), "d"(v.z),
                 "d"(v.w), "r"(mbar)
                 : "memory");
}
// release: this thread's shared::cluster stores are visible to every CTA that passes the matching wait
__device__ __forceinline__ void cluster_barrier()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// C: a pair Consumer with two targets per thread (PairF32<1, ...> / PairF64<2, ...>); its State<EQM> supplies
// set_target_pair(), tile() and take_sums().
template <class C, typename T, bool EQM>
__device__ __forceinline__ void cluster_kdk_loop(const ClusterArgs<T>& ca, unsigned char* smem, const uint32_t rank, const uint32_t nranks,
                                                 const double m0, uint64_t* inbox)
{
    typedef typename Vec4<T>::type V4;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int32_t n = ca.n, S = ca.S;
    const ClusterSmem<T> L(n, ca.n8, S, ca.tpc);
    const size_t npad = (size_t)8 * ca.n8;
    double* const part = reinterpret_cast<double*>(smem + L.part);
    V4* const svel = reinterpret_cast<V4*>(smem + L.svel);
    V4* const sacc = reinterpret_cast<V4*>(smem + L.sacc);
    // the staged {x, y, z, m} records of buffer b: what the pair loop reads and what the owners push
    auto records = [&](int b) -> V4* { return reinterpret_cast<V4*>(smem + L.cur) + (size_t)b * npad; };
    auto staged = [&](int b) -> const unsigned char* { return reinterpret_cast<const unsigned char*>(records(b)); };

    const int32_t lo = (int32_t)rank * ca.tpc;                       // this CTA owns the particles [lo, lo + owned)
    const int32_t owned = lo >= n ? 0 : (n - lo < ca.tpc ? n - lo : ca.tpc);
    const int32_t ngroups = (owned + CLUSTER_GROUP - 1) / CLUSTER_GROUP;
    const int32_t nitems = ngroups * S;
    const bool owner = tid < owned;
    const int32_t me = lo + tid;
    const double gm = (double)ca.G * (EQM ? m0 : 1.0);               // plan_row_mass(): the factor left out of the sums
    const T h = (T)0.5 * ca.dt;
    int cb = 0;
    uint32_t inbox_phase[2] = {0u, 0u};
    const uint32_t incoming = (uint32_t)n * (uint32_t)sizeof(V4);                // bytes pushed into this CTA per step

    PairPlan fake;                                                   // State's constructor reads nt and IB only
    fake.nt = n; fake.IB = CLUSTER_GROUP;
    const typename C::Params prm{nullptr, ca.eps2};

    // chunk sums of the owned targets: item = (group of 64 targets, chunk s) per warp, two targets per lane
    auto pair_phase = [&]() {
        typename C::template State<EQM> st(prm, fake, nullptr);
        const V4* rec = records(cb);
        const unsigned char* src = staged(cb);
        for (int32_t item = warp; item < nitems; item += CLUSTER_WARPS) {
            const int32_t g = item / S, s = item - g * S;
            int32_t i0 = lo + g * CLUSTER_GROUP + lane, i1 = i0 + 32;
            i0 = i0 < n ? i0 : n - 1;                                // clamped lanes are computed and never read back
            i1 = i1 < n ? i1 : n - 1;
            st.set_target_pair(rec[i0], rec[i1]);
            const int64_t j1 = 8 * (((int64_t)(s + 1) * ca.n8) / S);
            double sum[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
            for (int64_t j = 8 * (((int64_t)s * ca.n8) / S); j < j1; j += ca.Ttile) {
                const int64_t left = j1 - j;
                st.tile(src + (size_t)j * sizeof(V4), (int)(left < ca.Ttile ? left : ca.Ttile));
                st.take_sums(sum);                                   // second level: tile sums promoted to fp64
            }
            double* out = part + (size_t)item * 3 * CLUSTER_GROUP + lane;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                out[k * CLUSTER_GROUP] = sum[k];
                out[k * CLUSTER_GROUP + 32] = sum[3 + k];
            }
        }
        __syncthreads();
    };
    // the per-particle body of step_body.cuh on the owner thread; OPEN pushes the moved record to every CTA
    auto integrate = [&](const bool reduce, const bool close, const bool open) {
        if (owner) {
            V4 p = records(cb)[me];
            V4 a;
            if (reduce) {
                const double* row = part + (size_t)(tid / CLUSTER_GROUP) * S * 3 * CLUSTER_GROUP + (tid % CLUSTER_GROUP);
                double sx = 0.0, sy = 0.0, sz = 0.0;
                constexpr int BATCH = 8;                             // loads of a batch in flight together, adds in order
                for (int32_t s0 = 0; s0 < S; s0 += BATCH) {          // fixed order: increasing s (absent rows add +0.0)
                    double v[BATCH][3];
#pragma unroll
                    for (int q = 0; q < BATCH; ++q) {
                        const bool live = s0 + q < S;                // clamped, unconditional loads: no branch per row
                        const double* r = row + (size_t)3 * (live ? s0 + q : s0) * CLUSTER_GROUP;
#pragma unroll
                        for (int k = 0; k < 3; ++k) {
                            const double x = r[k * CLUSTER_GROUP];
                            v[q][k] = live ? x : 0.0;
                        }
                    }
#pragma unroll
                    for (int q = 0; q < BATCH; ++q) { sx += v[q][0]; sy += v[q][1]; sz += v[q][2]; }
                }
                a.x = (T)(gm * sx); a.y = (T)(gm * sy); a.z = (T)(gm * sz); a.w = (T)0;
                sacc[tid] = a;
            } else {
                a = sacc[tid];
            }
            if (close || open) {
                T ex, ey, ez;
                ext_accel<T>(ca.pot, p.x, p.y, p.z, ex, ey, ez);
                const T tx = a.x + ex, ty = a.y + ey, tz = a.z + ez;
                V4 v = svel[tid];
                if (close) { v.x = fma(tx, h, v.x); v.y = fma(ty, h, v.y); v.z = fma(tz, h, v.z); }
                if (open) {
                    v.x = fma(tx, h, v.x); v.y = fma(ty, h, v.y); v.z = fma(tz, h, v.z);
                    p.x = fma(v.x, ca.dt, p.x); p.y = fma(v.y, ca.dt, p.y); p.z = fma(v.z, ca.dt, p.z);
                    // Push the moved record into buffer cb ^ 1 of EVERY CTA (this one included), its bytes counted on the
                    // destination's inbox barrier of that buffer.  No cluster barrier: a CTA pushes step k + 1 only after
                    // it has received every CTA's push of step k, and a CTA pushes step k only after it has finished
                    // reading the buffer that the pushes of step k + 1 overwrite.
                    const uint32_t slot = smem_u32(records(cb ^ 1) + me), box = smem_u32(&inbox[cb ^ 1]);
                    for (uint32_t r = 0; r < nranks; ++r) {
                        uint32_t dst = rank + r;
                        dst = dst >= nranks ? dst - nranks : dst;
                        st_async_record(cluster_map(slot, dst), p, cluster_map(box, dst));
                    }
                }
                v.w = (T)0;
                svel[tid] = v;
            }
        }
        if (open) {
            const int nb = cb ^ 1;
            mbar_wait(&inbox[nb], inbox_phase[nb]);                  // every other CTA's records of this step have landed
            inbox_phase[nb] ^= 1u;
            if (tid == 0) mbar_arrive_expect_tx(&inbox[nb], incoming);   // arm the next use of this buffer (two steps on)
            cb = nb;
            __syncthreads();
        }
    };

    if (owner) {
        svel[tid] = ca.vel[me];
        if (ca.acc_valid) sacc[tid] = ca.acc[me];
    }
    if (tid == 0) {                                                  // arm both inboxes for their first use
        mbar_arrive_expect_tx(&inbox[0], incoming);
        mbar_arrive_expect_tx(&inbox[1], incoming);
    }
    __syncthreads();                                                 // buffer 0 was filled from global memory by the caller
    // ---- the KDK loop of odisseo_leapfrog_kdk_* (api.cu leapfrog_impl), nsteps >= 1 ------------------------------------
    if (!ca.acc_valid) pair_phase();
    integrate(!ca.acc_valid, false, true);
    for (int64_t k = 1; k < ca.nsteps; ++k) {
        pair_phase();
        integrate(true, true, true);
    }
    pair_phase();
    integrate(true, true, false);
    if (owner) {
        ca.posm[me] = records(cb)[me];
        ca.vel[me] = svel[tid];
        ca.acc[me] = sacc[tid];
    }
}

template <class C, typename T>
__global__ void __launch_bounds__(CLUSTER_THREADS, 1)
cluster_kdk_kernel(const ClusterArgs<T> ca)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t inbox[2];                       // bytes pushed into record buffer 0 / 1 by the other CTAs
    typedef typename Vec4<T>::type V4;
    const int tid = threadIdx.x;
    const uint32_t rank = cluster_ctarank(), nranks = cluster_nctarank();
    if (tid == 0) {
        mbar_init(&inbox[0], 1);
        mbar_init(&inbox[1], 1);
        mbar_fence_init();
    }
    const ClusterSmem<T> L(ca.n, ca.n8, ca.S, ca.tpc);
    const size_t npad = (size_t)8 * ca.n8;

    // every CTA reads all n records from global memory into buffer 0, pads the staged tails (both buffers) and
    // decides "all masses equal" for itself (the same answer everywhere)
    const T mass0 = reinterpret_cast<const T*>(ca.posm)[3];
    int differs = 0;
    V4* rec0 = reinterpret_cast<V4*>(smem_raw + L.cur);
    for (int32_t j = tid; j < ca.n; j += CLUSTER_THREADS) {
        const V4 p = ca.posm[j];
        differs |= !(p.w == mass0);                                  // NaN counts as different
        rec0[j] = p;
    }
    const T far = pad_pos((T)0);
    for (size_t j = (size_t)ca.n + tid; j < npad; j += CLUSTER_THREADS) {
        V4 pad; pad.x = far; pad.y = far; pad.z = far; pad.w = (T)0;
        rec0[j] = rec0[npad + j] = pad;
    }
    const bool eqm = __syncthreads_or(differs) == 0;
    cluster_barrier();                         // every CTA is running and its inbox barriers are initialised: pushes may start
    if (eqm)
        cluster_kdk_loop<C, T, true>(ca, smem_raw, rank, nranks, (double)mass0, inbox);
    else
        cluster_kdk_loop<C, T, false>(ca, smem_raw, rank, nranks, (double)mass0, inbox);
    cluster_barrier();                         // no CTA leaves while a copy out of its shared memory may be in flight
}

// Host side: the largest cluster this device schedules for the kernel (16, else 8; 0 = unavailable).
template <class C, typename T> cudaError_t configure_cluster(int* cluster_size)
{
    *cluster_size = 0;
    auto kernel = cluster_kdk_kernel<C, T>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, CLUSTER_SMEM_MAX);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e != cudaSuccess) return e;
    for (int cs = 16; cs >= 8; cs /= 2) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(cs);
        cfg.blockDim = dim3(CLUSTER_THREADS);
        cfg.dynamicSmemBytes = CLUSTER_SMEM_MAX;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = cs; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        int nclusters = 0;
        e = cudaOccupancyMaxActiveClusters(&nclusters, kernel, &cfg);
        if (e == cudaSuccess && nclusters >= 1) { *cluster_size = cs; return cudaSuccess; }
        (void)cudaGetLastError();
    }
    return cudaSuccess;
}

// Targets per CTA and shared-memory need of a call on n particles with a cluster of cs CTAs; 0 bytes = does not fit.
template <typename T> size_t cluster_geometry(const PairPlan& plan, int cs, int32_t* tpc)
{
    const int64_t per = (plan.n + cs - 1) / cs;
    *tpc = (int32_t)(((per + CLUSTER_GROUP - 1) / CLUSTER_GROUP) * CLUSTER_GROUP);
    if (*tpc > CLUSTER_THREADS) return 0;                            // one owner thread per particle
    const ClusterSmem<T> L((int32_t)plan.n, (int32_t)plan.n8, plan.S, *tpc);
    return L.total <= (size_t)CLUSTER_SMEM_MAX ? L.total : 0;
}

template <class C, typename T>
cudaError_t launch_cluster(const ClusterArgs<T>& ca, int cs, size_t smem, cudaStream_t stream)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cs);
    cfg.blockDim = dim3(CLUSTER_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cs; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, cluster_kdk_kernel<C, T>, ca);
}

}  // namespace odisseo
