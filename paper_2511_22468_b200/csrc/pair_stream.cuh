// Skeleton shared by the all-pairs kernels (pair_f32.cu, pair_f64.cu, adjoint.cu): a persistent grid,
// one CTA per SM (or several small ones), each walking a contiguous range of (i-block, source chunk)
// units of the launch plan (odisseo_common.cuh).  A dedicated producer warp streams the CTA's tile
// sequence with 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx, SASS UBLKCP) into a
// STAGES-deep shared-memory ring; consumers release a stage with one mbarrier arrive per warp -- no
// __syncthreads in the main loop.  The kernel is specialised by a Consumer type:
//
//   struct Consumer {
//       static constexpr int CWARPS, MINB, REC (bytes per staged record), COMPS (planes per row);
//       struct Params;                                  // kernel argument (targets, scalars)
//       static size_t outer_bytes();                    // shared memory behind the ring
//       template <bool EQM> struct State {              // per-thread registers
//           State(const Params&, const PairPlan&, unsigned char* outer_smem);
//           void load_targets(int32_t b);               // i-block b -> registers
//           void zero_outer();                          // start of a unit
//           void tile(const unsigned char* tile, int len);   // len source records, ANY length >= 1 (direct path: the last tile ends at n)
//           void flush_tile();                          // second summation level: tile sums -> fp64
//           void write_row(double* row);                // end of a unit
//       };
//   };
//
// Summation order (SURVEY.md 8a row a1'): inside a tile in the consumer's precision, tile sums added in
// fp64 in tile order inside a unit, one row per unit; rows are added by the reduce step in unit order.
// Every boundary is a function of n alone (odisseo_common.cuh), so the result does not depend on the
// number of CTAs, targets or ranks.
#pragma once

#include "odisseo_common.cuh"

namespace odisseo {

constexpr int STAGES = 4;

// The tile sequence of one CTA: units [u0, u1); unit u = chunk s = u % S of i-block b = u / S; the chunk's
// records [lo, hi) are cut into tiles of at most T records.  Producer and consumers run the same walk.
struct TileWalk {
    int64_t u, u1, j, hi, n8, nlim;
    int32_t T, S, b, s;
    __device__ __forceinline__ void set_unit()
    {
        b = (int32_t)(u / S);
        s = (int32_t)(u - (int64_t)b * S);
        j = 8 * (((int64_t)s * n8) / S);
        hi = 8 * (((int64_t)(s + 1) * n8) / S);
        hi = hi < nlim ? hi : nlim;                       // sources read from posm itself end at n, not at the padding
    }
    __device__ __forceinline__ TileWalk(const PairPlan& p, int64_t u0_, int64_t u1_)
        : u(u0_), u1(u1_), j(0), hi(0), n8(p.n8), nlim(p.direct ? p.n : 8 * p.n8), T(p.T), S(p.S), b(0), s(0)
    {
        if (u < u1) set_unit();
    }
    __device__ __forceinline__ bool valid() const { return u < u1; }
    __device__ __forceinline__ int32_t len() const { const int64_t r = hi - j; return (int32_t)(r < T ? r : T); }
    __device__ __forceinline__ bool last_of_unit() const { return j + T >= hi; }
    __device__ __forceinline__ void next()
    {
        j += T;
        if (j >= hi) {
            ++u;
            if (u < u1) set_unit();
        }
    }
};

template <class C, bool EQM>
__device__ __forceinline__ void consume_units(const typename C::Params& prm, double* __restrict__ rows, const PairPlan& plan,
                                              unsigned char* smem_raw, uint64_t* full_bar, uint64_t* empty_bar,
                                              const int64_t u0, const int64_t u1, int& s, uint32_t& ph)
{
    // s, ph: the ring position, kept by the caller so that a persistent kernel can walk its units again and again
    const uint32_t stage_bytes = (uint32_t)plan.T * C::REC;
    typename C::template State<EQM> st(prm, plan, smem_raw + (size_t)STAGES * stage_bytes);
    const int lane = threadIdx.x & 31;
    TileWalk w(plan, u0, u1);
    int32_t b_cur = -1;
    bool fresh = true;
    while (w.valid()) {
        if (w.b != b_cur) { st.load_targets(w.b); b_cur = w.b; }
        if (fresh) { st.zero_outer(); fresh = false; }
        mbar_wait(&full_bar[s], ph);
        st.tile(smem_raw + (size_t)s * stage_bytes, w.len());
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[s]);
        if (++s == STAGES) { s = 0; ph ^= 1u; }
        st.flush_tile();
        if (w.last_of_unit()) {
            st.write_row(rows + (size_t)w.u * C::COMPS * plan.IB);
            fresh = true;
        }
        w.next();
    }
}

template <class C>
__global__ void __launch_bounds__((C::CWARPS + 1) * 32, C::MINB)
stream_kernel(const typename C::Params prm, const unsigned char* __restrict__ jsrc, const unsigned char* __restrict__ src,
              double* __restrict__ rows, const PairPlan plan)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[STAGES];
    __shared__ __align__(8) uint64_t empty_bar[STAGES];
    constexpr int CWARPS = C::CWARPS;

    const int tid = threadIdx.x;
    const int warp = tid >> 5;
    const int lane = tid & 31;
    const int64_t c = blockIdx.x;
    const int64_t u0 = plan_start(plan, c);
    const int64_t u1 = plan_start(plan, c + 1);
    // Let the next kernel become resident early only when this one is short (a few tiles per CTA): its
    // CTAs then hide their launch latency behind our tail.  Behind a long evaluation, early dependents would
    // sit on the SMs for milliseconds (measured -0.3 % at N = 262,144); there the implicit trigger at exit is used.
    if ((u1 - u0) * (plan_chunk_lo(plan, 1) + plan.T) <= 16 * (int64_t)plan.T) pdl_launch_dependents();
    if (u0 >= u1) return;

    const uint32_t stage_bytes = (uint32_t)plan.T * C::REC;
    if (tid == CWARPS * 32) {                               // the producer lane owns init and the first loads
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], CWARPS);
        }
        mbar_fence_init();
    }
    pdl_wait();                                             // the staging kernel's records and flags are complete
    // the first STAGES tiles need no hand-over: issue them before anything else so that their latency
    // overlaps the flag reduction and the target loads
    TileWalk pw(plan, u0, u1);
    int prefetch = 0;
    if (tid == CWARPS * 32) {
        for (; prefetch < STAGES && pw.valid(); ++prefetch) {
            const uint32_t bytes = (uint32_t)pw.len() * C::REC;
            mbar_arrive_expect_tx(&full_bar[prefetch], bytes);
            tma_load_1d(smem_raw + (size_t)prefetch * stage_bytes, src + (size_t)pw.j * C::REC, bytes, &full_bar[prefetch]);
            pw.next();
        }
    }
    // equal-mass flags written by the staging kernel (odisseo_common.cuh): one uniform decision per grid
    int differs = 0;
    {
        const int* __restrict__ mflags = plan_flags(jsrc, plan);
        const int nflags = plan_nflags(plan);
        for (int k = tid; k < nflags; k += (CWARPS + 1) * 32) differs |= __ldg(mflags + k);
    }
    const bool eqm = __syncthreads_or(differs) == 0;        // also publishes the mbarrier inits
    if (c == 0 && tid == 0) *const_cast<int*>(plan_eqm_word(jsrc, plan)) = eqm ? 1 : 0;   // for the reduce step

    if (warp == CWARPS) {
        // ---- producer warp: one elected lane streams the rest of the CTA's tile sequence --------------
        if (lane == 0) {
            int s = prefetch % STAGES;
            uint32_t ph = prefetch == STAGES ? 1u : 0u;
            for (; pw.valid(); pw.next()) {
                mbar_wait_backoff(&empty_bar[s], ph ^ 1u);
                const uint32_t bytes = (uint32_t)pw.len() * C::REC;
                mbar_arrive_expect_tx(&full_bar[s], bytes);
                tma_load_1d(smem_raw + (size_t)s * stage_bytes, src + (size_t)pw.j * C::REC, bytes, &full_bar[s]);
                if (++s == STAGES) { s = 0; ph ^= 1u; }
            }
        }
        return;
    }

    int cs = 0;
    uint32_t cph = 0;
    if (eqm)
        consume_units<C, true>(prm, rows, plan, smem_raw, full_bar, empty_bar, u0, u1, cs, cph);
    else
        consume_units<C, false>(prm, rows, plan, smem_raw, full_bar, empty_bar, u0, u1, cs, cph);
}

template <class C> size_t stream_smem_bytes(const PairPlan& plan) { return (size_t)STAGES * plan.T * C::REC + C::outer_bytes(); }

template <class C> cudaError_t configure_stream(int max_tile)
{
    return cudaFuncSetAttribute(stream_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)((size_t)STAGES * max_tile * C::REC + C::outer_bytes()));
}

template <class C>
// jsrc: the workspace's staged array (the flags sit in front of it); src: the records the tiles are copied from (jsrc, or
// the caller's posm array when plan.direct).
cudaError_t launch_stream(const PairPlan& plan, const typename C::Params& prm, const void* jsrc, const void* src, double* rows,
                          cudaStream_t stream)
{
    return launch_pdl(stream_kernel<C>, dim3(plan.P), dim3((C::CWARPS + 1) * 32), stream_smem_bytes<C>(plan), stream, prm,
                      static_cast<const unsigned char*>(jsrc), static_cast<const unsigned char*>(src), rows, plan);
}

}  // namespace odisseo
