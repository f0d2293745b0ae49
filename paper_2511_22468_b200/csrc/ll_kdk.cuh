// Whole-loop kernel for small N on ALL SMs with a flag-in-data exchange (SURVEY.md 8a row a5 "decisive for configs
// 0-1"; the paper's inference runs single N = 1,000 simulations of 1,000 steps).
//
// At N ~ 1,000-4,000 a KDK step is 0.4-7 us of arithmetic, and what the per-step launches and the cooperative kernel
// (fused_step.cuh) pay on top is a chain of ~8 dependent L2 / TMA round trips per step: rows of partial sums written by
// one CTA and reduced by another, staged records written by the integrator and fetched by TMA, two launch edges or two
// grid barriers.  This kernel cuts the chain to ONE round trip per step:
//
//   * owner computes: CTA c owns a few targets (8 at N = 1,024 on 128 CTAs) and keeps ALL staged source records in its
//     own shared memory, so every chunk sum of its targets is computed, reduced (fixed order) and integrated inside the
//     CTA -- no partial rows through L2, no second kernel;
//   * pair phase: one LANE per (pair of owned targets, source chunk s): a lane walks its chunk's records in order with
//     the very inner loop of pair_f32.cu / pair_f64.cu (State::tile).  Lanes of a warp read different chunks, so chunk s
//     is stored skewed by 16 s bytes: the 8 lanes of a quarter-warp hit 8 different 16-byte bank groups;
//   * exchange: the only thing a step must publish is the moved position of every particle.  The owner writes each
//     coordinate as ONE 64-bit word {value bits, step tag} into a global array (NCCL's "LL" idea: the flag travels in
//     the same 8-byte store as the data, so no fence and no separate flag is needed); every CTA polls the n records with
//     64-bit volatile loads until the tags equal the step it waits for and refreshes its shared-memory copy.  Two
//     buffers alternate: a CTA writes step k + 2 only after it has read every record of step k + 1, which their owners
//     wrote after reading every record of step k.  No grid barrier, no launch edge, no atomics inside the loop.
//
// The CTAs wait for one another, so they must be co-resident: the kernel is launched cooperatively (the launch fails
// instead of hanging when it does not fit).  Summation order: the launch plan's chunks and tiles (functions of n alone),
// tile sums in the Consumer's precision promoted to fp64 per tile, chunk sums added in increasing s, G [m] applied once
// in fp64 -- the canonical grouping of odisseo_common.cuh: BIT-IDENTICAL to the other launch forms (tests).
#pragma once

#include "odisseo_common.cuh"
#include "step_body.cuh"

namespace odisseo {

#ifndef ODISSEO_LL_WARPS
#define ODISSEO_LL_WARPS 16
#endif
constexpr int LL_WARPS = ODISSEO_LL_WARPS;        // threads per CTA / 32, one CTA per SM
constexpr int LL_THREADS = LL_WARPS * 32;
constexpr int LL_SMEM_MAX = 226 * 1024;
#ifndef ODISSEO_LL_LANES
#define ODISSEO_LL_LANES 128
#endif
constexpr int LL_LANES = ODISSEO_LL_LANES;        // lanes of pair-phase work a CTA takes before the grid grows

template <typename T> struct LLArgs {
    typename Vec4<T>::type *posm, *vel, *acc;
    T G, eps2, dt;
    PotParams<T> pot;
    int64_t nsteps;
    int32_t acc_valid;
    int32_t n, n8, S, Ttile;                      // the plan's source split (chunks of octets, tile length)
    int32_t tpc;                                  // targets owned per CTA (even)
    unsigned long long* xbuf;                     // [2][n rounded up to even][LLWords<T>] tagged words, zeroed by the host before the launch
    typename Vec4<T>::type* tape;                 // reverse mode's tape of nsteps + 1 snapshots {x_k, v_k, pair-only a_k}, or null
};

template <typename T> struct LLWords { static constexpr int value = sizeof(T) == 4 ? 3 : 6; };
template <typename T> struct LLSkew { static constexpr int value = sizeof(T) == 4 ? 16 : 32; };   // bytes per chunk index

// Shared-memory carve (bytes), identical on the host and on the device.
template <typename T> struct LLSmem {
    size_t cur, chunk, part, svel, sacc, total;
    __host__ __device__ LLSmem(int32_t n8, int32_t S, int32_t tpc)
    {
        size_t off = 0;
        cur = off; off += (size_t)8 * n8 * 4 * sizeof(T) + (size_t)LLSkew<T>::value * S;
        chunk = off; off += (size_t)8 * n8 * sizeof(uint16_t);          // chunk index of every staged record
        off = (off + 127) & ~(size_t)127;
        part = off; off += (size_t)(tpc / 2) * S * 6 * sizeof(double);
        svel = off; off += (size_t)tpc * 4 * sizeof(T);
        sacc = off; off += (size_t)tpc * 4 * sizeof(T);
        total = off;
    }
};

__device__ __forceinline__ unsigned long long ll_ld(const unsigned long long* p)
{
    unsigned long long v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void ll_st(unsigned long long* p, unsigned long long v)
{
    asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// chunk that holds source record j: the largest s with 8 floor(s n8 / S) <= j
__device__ __forceinline__ int32_t ll_chunk_of(int32_t j, int32_t n8, int32_t S)
{
    const int32_t oct = j >> 3;
    const int32_t s = (int32_t)((((int64_t)oct + 1) * S + n8 - 1) / n8) - 1;
    return s < S - 1 ? s : S - 1;
}
// staged record j of chunk s in the skewed array ({x, y, z, m}; fp32 16 B, fp64 32 B per record)
__device__ __forceinline__ float4 ll_record(const unsigned char* cur, int32_t j, int32_t s, float)
{
    return *reinterpret_cast<const float4*>(cur + (size_t)16 * j + (size_t)16 * s);
}
__device__ __forceinline__ double4 ll_record(const unsigned char* cur, int32_t j, int32_t s, double)
{
    const double2* w = reinterpret_cast<const double2*>(cur + (size_t)32 * j + (size_t)32 * s);
    const double2 A = w[0], B = w[1];
    return make_double4(A.x, A.y, B.x, B.y);
}
__device__ __forceinline__ float4 ll_record_at(const unsigned char* rec, float) { return *reinterpret_cast<const float4*>(rec); }
__device__ __forceinline__ double4 ll_record_at(const unsigned char* rec, double)
{
    const double2* w = reinterpret_cast<const double2*>(rec);
    const double2 A = w[0], B = w[1];
    return make_double4(A.x, A.y, B.x, B.y);
}
// (re)write the position of staged record j; the mass word stays
__device__ __forceinline__ void ll_put_position(unsigned char* cur, int32_t j, int32_t s, float x, float y, float z)
{
    float* w = reinterpret_cast<float*>(cur + (size_t)16 * j + (size_t)16 * s);
    *reinterpret_cast<float2*>(w) = make_float2(x, y);
    w[2] = z;
}
__device__ __forceinline__ void ll_put_position(unsigned char* cur, int32_t j, int32_t s, double x, double y, double z)
{
    double* w = reinterpret_cast<double*>(cur + (size_t)32 * j + (size_t)32 * s);
    *reinterpret_cast<double2*>(w) = make_double2(x, y);
    w[2] = z;
}
__device__ __forceinline__ void ll_put_mass(unsigned char* cur, int32_t j, int32_t s, float m)
{
    reinterpret_cast<float*>(cur + (size_t)16 * j + (size_t)16 * s)[3] = m;
}
__device__ __forceinline__ void ll_put_mass(unsigned char* cur, int32_t j, int32_t s, double m)
{
    reinterpret_cast<double*>(cur + (size_t)32 * j + (size_t)32 * s)[3] = m;
}

// Tagged exchange words: {tag : 32 | payload : 32}.  fp32: one word per coordinate; fp64: two (low, high half).
__device__ __forceinline__ void ll_publish(unsigned long long* rec, uint32_t tag, float x, float y, float z)
{
    const unsigned long long t = (unsigned long long)tag << 32;
    ll_st(rec + 0, t | __float_as_uint(x));
    ll_st(rec + 1, t | __float_as_uint(y));
    ll_st(rec + 2, t | __float_as_uint(z));
}
__device__ __forceinline__ void ll_publish(unsigned long long* rec, uint32_t tag, double x, double y, double z)
{
    const unsigned long long t = (unsigned long long)tag << 32;
    const double c[3] = {x, y, z};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const unsigned long long b = (unsigned long long)__double_as_longlong(c[k]);
        ll_st(rec + 2 * k, t | (b & 0xffffffffull));
        ll_st(rec + 2 * k + 1, t | (b >> 32));
    }
}
// spin until every word of the record carries `tag`
__device__ __forceinline__ void ll_fetch(const unsigned long long* rec, uint32_t tag, float& x, float& y, float& z)
{
    unsigned long long w0, w1, w2;
    do {
        w0 = ll_ld(rec + 0); w1 = ll_ld(rec + 1); w2 = ll_ld(rec + 2);
    } while ((uint32_t)(w0 >> 32) != tag || (uint32_t)(w1 >> 32) != tag || (uint32_t)(w2 >> 32) != tag);
    x = __uint_as_float((uint32_t)w0); y = __uint_as_float((uint32_t)w1); z = __uint_as_float((uint32_t)w2);
}
__device__ __forceinline__ void ll_fetch(const unsigned long long* rec, uint32_t tag, double& x, double& y, double& z)
{
    unsigned long long w[6];
    bool ok;
    do {
        ok = true;
#pragma unroll
        for (int k = 0; k < 6; ++k) w[k] = ll_ld(rec + k);
#pragma unroll
        for (int k = 0; k < 6; ++k) ok = ok && (uint32_t)(w[k] >> 32) == tag;
    } while (!ok);
    x = __longlong_as_double((long long)((w[0] & 0xffffffffull) | (w[1] << 32)));
    y = __longlong_as_double((long long)((w[2] & 0xffffffffull) | (w[3] << 32)));
    z = __longlong_as_double((long long)((w[4] & 0xffffffffull) | (w[5] << 32)));
}

__device__ __forceinline__ void ll_ld16(const unsigned long long* p, unsigned long long& a, unsigned long long& b)
{
    asm volatile("ld.volatile.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}
// Two consecutive records (2 W words, 16-byte aligned) polled with 16-byte loads: half the requests at the L2 lines
// that every CTA polls.  Each 8-byte word still validates itself by its own tag, so it does not matter whether the
// hardware performs a 16-byte access as one transaction.  second = false: only the first record exists.
template <typename T>
__device__ __forceinline__ void ll_fetch_pair(const unsigned long long* rec, const bool second, uint32_t tag, T& x, T& y, T& z, T& x2,
                                              T& y2, T& z2)
{
    constexpr int W = LLWords<T>::value;
    unsigned long long w[2 * W];
    bool ok;
    do {
#pragma unroll
        for (int k = 0; k < W; ++k) ll_ld16(rec + 2 * k, w[2 * k], w[2 * k + 1]);
        ok = true;
#pragma unroll
        for (int k = 0; k < 2 * W; ++k) ok = ok && ((uint32_t)(w[k] >> 32) == tag || (k >= W && !second));
    } while (!ok);
    if (sizeof(T) == 4) {
        x = (T)__uint_as_float((uint32_t)w[0]); y = (T)__uint_as_float((uint32_t)w[1]); z = (T)__uint_as_float((uint32_t)w[2]);
        x2 = (T)__uint_as_float((uint32_t)w[W]); y2 = (T)__uint_as_float((uint32_t)w[W + 1]); z2 = (T)__uint_as_float((uint32_t)w[W + 2]);
    } else {
        x = (T)__longlong_as_double((long long)((w[0] & 0xffffffffull) | (w[1] << 32)));
        y = (T)__longlong_as_double((long long)((w[2] & 0xffffffffull) | (w[3] << 32)));
        z = (T)__longlong_as_double((long long)((w[4 % (2 * W)] & 0xffffffffull) | (w[5 % (2 * W)] << 32)));
        x2 = (T)__longlong_as_double((long long)((w[W] & 0xffffffffull) | (w[W + 1] << 32)));
        y2 = (T)__longlong_as_double((long long)((w[(W + 2) % (2 * W)] & 0xffffffffull) | (w[(W + 3) % (2 * W)] << 32)));
        z2 = (T)__longlong_as_double((long long)((w[(W + 4) % (2 * W)] & 0xffffffffull) | (w[(W + 5) % (2 * W)] << 32)));
    }
}

// C: a pair Consumer with two targets per thread (PairF32<1, ...> / PairF64<2, ...>); its State<EQM> supplies
// set_target_pair(), tile() and take_sums().
template <class C, typename T, bool EQM, bool TAPE>
__device__ __forceinline__ void ll_kdk_loop(const LLArgs<T>& ca, unsigned char* smem, const double m0)
{
    typedef typename Vec4<T>::type V4;
    constexpr int WORDS = LLWords<T>::value;
    constexpr int SKEW = LLSkew<T>::value;
    constexpr int REC = 4 * (int)sizeof(T);                          // bytes per staged record {x, y, z, m}
    const int tid = threadIdx.x;
    const int32_t n = ca.n, n8 = ca.n8, S = ca.S;
    const LLSmem<T> L(n8, S, ca.tpc);
    unsigned char* const cur = smem + L.cur;
    const uint16_t* const chunk_of = reinterpret_cast<const uint16_t*>(smem + L.chunk);
    double* const part = reinterpret_cast<double*>(smem + L.part);
    V4* const svel = reinterpret_cast<V4*>(smem + L.svel);
    V4* const sacc = reinterpret_cast<V4*>(smem + L.sacc);

    const int32_t lo = (int32_t)blockIdx.x * ca.tpc;                 // this CTA owns the particles [lo, lo + owned)
    const int32_t owned = lo >= n ? 0 : (n - lo < ca.tpc ? n - lo : ca.tpc);
    const bool owner = tid < owned;
    const int32_t me = lo + tid;
    const int32_t my_chunk = owner ? chunk_of[me] : 0;
    const double gm = (double)ca.G * (EQM ? m0 : 1.0);               // plan_row_mass(): the factor left out of the sums
    const T h = (T)0.5 * ca.dt;
    uint32_t pushes = 0;                                             // tag of the latest exchange
    const size_t nbuf = ((size_t)n + 1) & ~(size_t)1;                // records per exchange buffer (16-byte aligned buffers)

    PairPlan fake;                                                   // State's constructor reads nt and IB only
    fake.nt = n; fake.IB = 2;
    const typename C::Params prm{nullptr, ca.eps2};

#ifdef ODISSEO_LL_TIMING
    long long tq[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tmark = clock64();
#define LL_MARK(k) do { const long long now_ = clock64(); tq[k] += now_ - tmark; tmark = now_; } while (0)
#else
#define LL_MARK(k) do { } while (0)
#endif
    // Lane geometry of the pair phase (fixed for the launch).  The owned pairs sit in groups of G = 2^k >= pairs lanes
    // (at most 32); a warp item is 32 / G consecutive chunks x G pairs: the lanes of a group walk the same chunk (one
    // broadcast address), different groups walk different chunks (kept off each other's banks by the skew).
    const int32_t npairs = (owned + 1) / 2;
    int32_t G = 1;
    while (G < npairs && G < 32) G <<= 1;
    const int32_t cpw = 32 / G;                                      // chunks per warp item
    const int32_t nsw = (S + cpw - 1) / cpw;                         // warp items along the chunks
    const int32_t nwitems = npairs == 0 ? 0 : ((npairs + G - 1) / G) * nsw;
    const int32_t lane_g = (tid & 31) / G, lane_q = (tid & 31) % G;
    // What a lane does in warp item wi: nothing here changes from step to step, so the first item of every warp (the
    // only one unless the CTA owns many targets) is worked out once, before the time loop -- the index arithmetic
    // (three integer divisions) would otherwise sit on the critical path of every step of a one-warp-deep pair phase.
    struct LaneItem { int32_t t0, t1, src, len, out; };              // byte offsets in cur, records, doubles in part; len < 0: idle
    auto lane_item = [&](const int32_t wi) {
        LaneItem it;
        it.len = -1; it.t0 = it.t1 = it.src = it.out = 0;
        if (wi >= nwitems) return it;
        const int32_t pg = wi / nsw, sw = wi - pg * nsw;
        const int32_t sc = sw * cpw + lane_g, p = pg * G + lane_q;
        if (sc >= S || p >= npairs) return it;
        int32_t i0 = lo + 2 * p, i1 = i0 + 1;
        i1 = i1 < n ? i1 : n - 1;                                    // an odd tail pairs the last target with itself
        it.t0 = REC * i0 + SKEW * (int32_t)chunk_of[i0];
        it.t1 = REC * i1 + SKEW * (int32_t)chunk_of[i1];
        const int32_t j0 = 8 * (int32_t)(((uint32_t)sc * (uint32_t)n8) / (uint32_t)S);
        const int32_t j1 = 8 * (int32_t)(((uint32_t)(sc + 1) * (uint32_t)n8) / (uint32_t)S);
        it.src = REC * j0 + SKEW * sc;
        it.len = j1 - j0;
        it.out = (p * S + sc) * 6;
        return it;
    };
    const LaneItem first_item = lane_item(tid >> 5);
    // chunk sums of the owned targets: one lane per (pair of targets, chunk s)
    auto pair_phase = [&]() {
        LL_MARK(7);
        typename C::template State<EQM> st(prm, fake, nullptr);
        LaneItem it = first_item;
        for (int32_t wi = tid >> 5; wi < nwitems; wi += LL_WARPS) {
            if (it.len >= 0) {
                st.set_target_pair(ll_record_at(cur + it.t0, T()), ll_record_at(cur + it.t1, T()));
                double sum[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
                for (int32_t j = 0; j < it.len; j += ca.Ttile) {
                    const int32_t left = it.len - j;
                    st.tile(cur + it.src + (size_t)REC * j, left < ca.Ttile ? left : ca.Ttile);
                    st.take_sums(sum);                               // second level: tile sums promoted to fp64
                }
                double* out = part + it.out;
#pragma unroll
                for (int k = 0; k < 6; ++k) out[k] = sum[k];
            }
            if (wi + LL_WARPS < nwitems) it = lane_item(wi + LL_WARPS);
        }
        LL_MARK(0);
        __syncthreads();
        LL_MARK(1);
    };
    // the per-particle body of step_body.cuh on the owner thread; OPEN publishes the moved position and refreshes
    // every CTA's copy of all n positions
    auto integrate = [&](const bool reduce, const bool close, const bool open) {
        if (owner) {
            V4 p = ll_record(cur, me, my_chunk, T());
            V4 a;
            if (reduce) {
                const double* row = part + (size_t)(tid >> 1) * S * 6 + 3 * (tid & 1);
                double sx = 0.0, sy = 0.0, sz = 0.0;
                constexpr int BATCH = 8;                             // loads of a batch in flight together, adds in order
                for (int32_t s0 = 0; s0 < S; s0 += BATCH) {          // fixed order: increasing s (absent rows add +0.0)
                    double v[BATCH][3];
#pragma unroll
                    for (int q = 0; q < BATCH; ++q) {
                        const bool live = s0 + q < S;                // clamped, unconditional loads: no branch per row
                        const double* r = row + (size_t)6 * (live ? s0 + q : s0);
#pragma unroll
                        for (int k = 0; k < 3; ++k) {
                            const double x = r[k];
                            v[q][k] = live ? x : 0.0;
                        }
                    }
#pragma unroll
                    for (int q = 0; q < BATCH; ++q) { sx += v[q][0]; sy += v[q][1]; sz += v[q][2]; }
                }
                a.x = (T)(gm * sx); a.y = (T)(gm * sy); a.z = (T)(gm * sz); a.w = (T)0;
                sacc[tid] = a;
                LL_MARK(2);
            } else {
                a = sacc[tid];
            }
            if (close || open) {
                T ex, ey, ez;
                ext_accel<T>(ca.pot, p.x, p.y, p.z, ex, ey, ez);
                const T tx = a.x + ex, ty = a.y + ey, tz = a.z + ez;
                V4 v = svel[tid];
                if (close) { v.x = fma(tx, h, v.x); v.y = fma(ty, h, v.y); v.z = fma(tz, h, v.z); }
                if (TAPE && ca.tape) {
                    // the synchronised state between the closing kick of step k - 1 and the opening kick of step k
                    // (step_body.cuh's snapshot); k = pushes: one snapshot per integrate call
                    V4* snap = ca.tape + (size_t)pushes * 3 * n;
                    V4 vs = v; vs.w = (T)0;
                    snap[me] = p;
                    snap[n + me] = vs;
                    snap[2 * (size_t)n + me] = a;
                }
                if (open) {
                    v.x = fma(tx, h, v.x); v.y = fma(ty, h, v.y); v.z = fma(tz, h, v.z);
                    p.x = fma(v.x, ca.dt, p.x); p.y = fma(v.y, ca.dt, p.y); p.z = fma(v.z, ca.dt, p.z);
                    ll_publish(ca.xbuf + ((size_t)((pushes + 1) & 1u) * nbuf + me) * WORDS, pushes + 1, p.x, p.y, p.z);
                }
                v.w = (T)0;
                svel[tid] = v;
            }
        }
        LL_MARK(3);
        if (open) {
            ++pushes;
            __syncthreads();                                         // the owners have read their old records
            LL_MARK(4);
            const unsigned long long* buf = ca.xbuf + (size_t)(pushes & 1u) * nbuf * WORDS;
            for (int32_t j = 2 * tid; j < n; j += 2 * LL_THREADS) {   // two consecutive records per thread
                const bool second = j + 1 < n;
                T x, y, z, x2, y2, z2;
                ll_fetch_pair(buf + (size_t)j * WORDS, second, pushes, x, y, z, x2, y2, z2);
                ll_put_position(cur, j, chunk_of[j], x, y, z);
                if (second) ll_put_position(cur, j + 1, chunk_of[j + 1], x2, y2, z2);
            }
            LL_MARK(5);
            __syncthreads();
            LL_MARK(6);
        }
    };

    if (owner) {
        svel[tid] = ca.vel[me];
        if (ca.acc_valid) sacc[tid] = ca.acc[me];
    }
    __syncthreads();
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
        ca.posm[me] = ll_record(cur, me, my_chunk, T());
        ca.vel[me] = svel[tid];
        ca.acc[me] = sacc[tid];
    }
#ifdef ODISSEO_LL_TIMING
    __syncthreads();
    if (blockIdx.x == 0 && tid == 0)
        for (int k = 0; k < 8; ++k) reinterpret_cast<T*>(ca.acc + k)[3] = (T)((double)tq[k] / (double)ca.nsteps);
#endif
}

// TAPE: the instantiation that can store the reverse mode's snapshots (it also runs with a null tape).
template <class C, typename T, bool TAPE>
__global__ void __launch_bounds__(LL_THREADS, 1)
ll_kdk_kernel(const LLArgs<T> ca)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    typedef typename Vec4<T>::type V4;
    const int tid = threadIdx.x;
    const LLSmem<T> L(ca.n8, ca.S, ca.tpc);
    unsigned char* const cur = smem_raw + L.cur;
    const int32_t npad = 8 * ca.n8;

    // every CTA stages all n records (skewed by chunk), pads the tail and decides "all masses equal" for itself
    const T mass0 = reinterpret_cast<const T*>(ca.posm)[3];
    int differs = 0;
    uint16_t* const chunk_tab = reinterpret_cast<uint16_t*>(smem_raw + L.chunk);
    for (int32_t j = tid; j < npad; j += LL_THREADS) {
        const int32_t s = ll_chunk_of(j, ca.n8, ca.S);
        chunk_tab[j] = (uint16_t)s;
        if (j < ca.n) {
            const V4 p = ca.posm[j];
            differs |= !(p.w == mass0);                              // NaN counts as different
            ll_put_position(cur, j, s, p.x, p.y, p.z);
            ll_put_mass(cur, j, s, p.w);
        } else {
            const T far = pad_pos((T)0);                             // massless padding parked far away
            ll_put_position(cur, j, s, far, far, far);
            ll_put_mass(cur, j, s, (T)0);
        }
    }
    const bool eqm = __syncthreads_or(differs) == 0;
    if (eqm)
        ll_kdk_loop<C, T, true, TAPE>(ca, smem_raw, (double)mass0);
    else
        ll_kdk_loop<C, T, false, TAPE>(ca, smem_raw, (double)mass0);
}

// Host side.  Co-resident CTAs of the kernel on this device (cooperative launch bound).
template <class C, typename T> cudaError_t configure_ll(int num_sms, int* max_ctas)
{
    *max_ctas = 0;
    cudaError_t e = cudaFuncSetAttribute(ll_kdk_kernel<C, T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, LL_SMEM_MAX);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(ll_kdk_kernel<C, T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, LL_SMEM_MAX);
    if (e != cudaSuccess) return e;
    int per_sm = 0, per_sm2 = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ll_kdk_kernel<C, T, true>, LL_THREADS, (size_t)LL_SMEM_MAX);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm2, ll_kdk_kernel<C, T, false>, LL_THREADS, (size_t)LL_SMEM_MAX);
    if (e != cudaSuccess) return e;
    *max_ctas = (per_sm < per_sm2 ? per_sm : per_sm2) * num_sms;
    return cudaSuccess;
}

// Targets per CTA, CTA count, shared-memory and exchange-buffer need of a call; smem 0 = does not fit.
template <typename T> size_t ll_geometry(const PairPlan& plan, int max_ctas, int32_t* tpc, int32_t* ctas, size_t* xbuf_bytes)
{
    if (max_ctas < 1) return 0;
    // Few CTAs are better than many as long as a CTA's pair phase stays one warp per scheduler deep (its length is the
    // chunk length either way): every CTA polls every record, and the polls of all CTAs queue at the same L2 lines.
    const int64_t pairs = (plan.n + 1) / 2;
    int64_t per_cta = (pairs + max_ctas - 1) / max_ctas;             // what the co-resident grid forces
    int64_t comfy = 1;                                               // largest power of two of pairs whose (pair, chunk)
    while (2 * comfy * plan.S <= LL_LANES) comfy *= 2;               // lanes fit LL_LANES lanes (groups are powers of two)
    if (per_cta < comfy) per_cta = comfy;
    *tpc = (int32_t)(2 * per_cta);
    *ctas = (int32_t)((plan.n + *tpc - 1) / *tpc);
    *xbuf_bytes = (size_t)2 * (((size_t)plan.n + 1) & ~(size_t)1) * LLWords<T>::value * sizeof(unsigned long long);
    if (*tpc > LL_THREADS) return 0;                                 // one owner thread per particle
    const LLSmem<T> L((int32_t)plan.n8, plan.S, *tpc);
    return L.total <= (size_t)LL_SMEM_MAX ? L.total : 0;
}

// tape_code: launch the instantiation that carries the snapshot stores (required when ca.tape is set).
template <class C, typename T>
cudaError_t launch_ll(const LLArgs<T>& ca, int ctas, size_t smem, bool tape_code, cudaStream_t stream)
{
    LLArgs<T> a = ca;
    void* args[] = {&a};
    void* kernel = tape_code || ca.tape ? reinterpret_cast<void*>(ll_kdk_kernel<C, T, true>) : reinterpret_cast<void*>(ll_kdk_kernel<C, T, false>);
    return cudaLaunchCooperativeKernel(kernel, dim3(ctas), dim3(LL_THREADS), args, smem, stream);
}

}  // namespace odisseo
