// Reverse-mode derivative of the hot path.  The paper's simulator is "end-to-end
// differentiable" with respect to initial conditions, integration time, particle masses and potential
// parameters (section 1, L21 section 2; used in L43 Fig. 2 step 5 and L63) through JAX autodiff; here
// the vector-Jacobian products are written out by hand:
//
//   pair   a_i = G sum_j m_j d f,  d = x_j - x_i,  s = |d|^2 + eps^2,  f = s^-3/2,  g = -3 s^-5/2
//          (J^T c)_i = G sum_j (f u + g d (d.u)),   u = m_i c_j - m_j c_i
//          dL/dm_i   = -G sum_j f (d.c_j)           dL/deps = eps G sum_i sum_j m_j g (d.c_i)
//          dL/dG     = sum_i c_i . a_pair,i / G
//   ext    Hessians and parameter derivatives of the NFW and Miyamoto-Nagai accelerations
//   kdk    Lv_N = lam_v, Lx_N = lam_x + J(x_N)^T (dt/2 Lv_N);
//          Lv_k = Lv_{k+1} + dt Lx_{k+1};  Lx_k = Lx_{k+1} + J(x_k)^T (w_k Lv_k),  w_k = dt (0<k<N), dt/2 (k=0)
//          dL/ddt = sum_k [ Lx_{k+1}.vh_k + (Lv_k.a_k + Lv_{k+1}.a_{k+1}) / 2 ]
//
// The O(N^2) pass runs on the forward kernels' skeleton (pair_stream.cuh): persistent grid, contiguous unit
// ranges, {position, cotangent} source records through the TMA ring, one row of fp64 sums per unit, rows added
// in fixed order by vjp_finish_kernel (bit-reproducible, no atomics).  fp32: every loop form (equal or general
// masses, with or without the eps / G terms) runs on packed f32x2 pairs, two targets per instruction, sources
// staged as plain {x,y,z,m},{cx,cy,cz,0} records (two LDS.128 per source, scalar broadcast operands): 26 packed ops + 2 MUFU
// per two pairs in the equal-mass form.  fp64: the scalar term of adjoint_terms.cuh.  Per-tile sums in the state's precision, promoted
// to fp64 between tiles.  The O(N) parts (external potential, parameter sums) are evaluated in fp64 whatever the
// state precision.
#include "adjoint_terms.cuh"
#include "pair_stream.cuh"

namespace odisseo {

namespace {

template <typename T> struct AVec4;
template <> struct AVec4<float> { typedef float4 type; };
template <> struct AVec4<double> { typedef double4 type; };

// ---- fp32 consumer: 2*NPAIR targets per thread as packed pairs -------------------------------------------------
template <int NPAIR, bool EG, int CWARPS_, int MINB_, int JUNROLL>
struct VjpF32 {
    static constexpr int CWARPS = CWARPS_, MINB = MINB_, REC = 32, COMPS = EG ? 6 : 4;
    static constexpr int CTHREADS = CWARPS * 32;
    struct Params { const float4* posm; const float4* cot; float eps2; };
    static size_t outer_bytes() { return (size_t)2 * NPAIR * COMPS * CTHREADS * sizeof(double); }

    // EQM (all masses equal, flags from the staging kernel): u = c_j - c_i, the common mass multiplies the x, y, z
    // (and eps, G) sums in vjp_finish_kernel.
    template <bool EQM>
    struct State {
        const float4* __restrict__ posm;
        const float4* __restrict__ cot;
        const int64_t nt;
        const int32_t IB;
        const f32x2 e2, m3;
        double* __restrict__ osum;                 // osum[(2p + h) * COMPS + comp][tid]
        f32x2 xi[NPAIR], yi[NPAIR], zi[NPAIR], cxi[NPAIR], cyi[NPAIR], czi[NPAIR], mi[NPAIR];
        f32x2 acc[NPAIR][COMPS];

        __device__ __forceinline__ State(const Params& prm, const PairPlan& plan, unsigned char* outer)
            : posm(prm.posm), cot(prm.cot), nt(plan.nt), IB(plan.IB), e2(pk(prm.eps2, prm.eps2)), m3(pk(-3.0f, -3.0f)),
              osum(reinterpret_cast<double*>(outer) + threadIdx.x)
        {
        }
        __device__ __forceinline__ void load_targets(const int32_t b)
        {
            const int64_t base = (int64_t)b * IB + threadIdx.x;
            const f32x2 nz = pk(-0.0f, -0.0f);       // pack through FADD2: native 64-bit register pairs (pair_f32.cu)
#pragma unroll
            for (int p = 0; p < NPAIR; ++p) {
                int64_t i0 = base + (int64_t)(2 * p) * CTHREADS;
                int64_t i1 = i0 + CTHREADS;
                i0 = i0 < nt ? i0 : nt - 1;               // clamped rows are computed and never read back
                i1 = i1 < nt ? i1 : nt - 1;
                const float4 p0 = __ldg(posm + i0), p1 = __ldg(posm + i1);
                const float4 c0 = __ldg(cot + i0), c1 = __ldg(cot + i1);
                xi[p] = add2(pk(p0.x, p1.x), nz); yi[p] = add2(pk(p0.y, p1.y), nz); zi[p] = add2(pk(p0.z, p1.z), nz);
                cxi[p] = add2(pk(c0.x, c1.x), nz); cyi[p] = add2(pk(c0.y, c1.y), nz); czi[p] = add2(pk(c0.z, c1.z), nz);
                mi[p] = add2(pk(p0.w, p1.w), nz);
#pragma unroll
                for (int k = 0; k < COMPS; ++k) acc[p][k] = 0ull;
            }
        }
        __device__ __forceinline__ void zero_outer()
        {
#pragma unroll
            for (int k = 0; k < 2 * NPAIR * COMPS; ++k) osum[k * CTHREADS] = 0.0;
        }
        __device__ __forceinline__ void tile(const unsigned char* tile_raw, const int len)
        {
            const float4* __restrict__ t = reinterpret_cast<const float4*>(tile_raw);
#pragma unroll JUNROLL
            for (int j = 0; j < len; ++j) {
                // two LDS.128 per source: {x, y, z, m}, {cx, cy, cz, 0}; the splats are scalar broadcast operands of the
                // packed instructions (pair_f32.cu), nothing is pre-duplicated
                const float4 q = t[2 * j], c = t[2 * j + 1];
                struct { f32x2 x, y; } A, B, C;
                A.x = pk(q.x, q.x); A.y = pk(q.y, q.y); B.x = pk(q.z, q.z);
                B.y = pk(c.x, c.x); C.x = pk(c.y, c.y); C.y = pk(c.z, c.z);
                f32x2 mj = 0ull;
                if (!EQM) mj = pk(q.w, q.w);
#pragma unroll
                for (int p = 0; p < NPAIR; ++p) {
                    const f32x2 dx = sub2(A.x, xi[p]), dy = sub2(A.y, yi[p]), dz = sub2(B.x, zi[p]);
                    const f32x2 s = fma2(dz, dz, fma2(dy, dy, fma2(dx, dx, e2)));
                    float sl, sh;
                    unpk(s, sl, sh);
                    const f32x2 y = pk(rsqrt_approx(sl), rsqrt_approx(sh));
                    const f32x2 y2 = mul2(y, y);
                    const f32x2 f = mul2(y2, y);                                         // s^-3/2
                    const f32x2 pj = fma2(dz, C.y, fma2(dy, C.x, mul2(dx, B.y)));          // d . c_j
                    // u = m_i c_j - m_j c_i written as m_i (c_j - c_i) + (m_i - m_j) c_i: the difference of
                    // cotangents is taken first (exact for close values), and the self term is exactly 0
                    f32x2 ux = sub2(B.y, cxi[p]), uy = sub2(C.x, cyi[p]), uz = sub2(C.y, czi[p]);
                    if (!EQM) {
                        const f32x2 dm = sub2(mi[p], mj);
                        ux = fma2(dm, cxi[p], mul2(mi[p], ux));
                        uy = fma2(dm, cyi[p], mul2(mi[p], uy));
                        uz = fma2(dm, czi[p], mul2(mi[p], uz));
                    }
                    const f32x2 du = fma2(dz, uz, fma2(dy, uy, mul2(dx, ux)));            // d . u
                    const f32x2 k3 = mul2(mul2(y2, du), m3);                             // -3 s^-1 (d . u) = g (d . u) / f
                    acc[p][0] = fma2(f, fma2(k3, dx, ux), acc[p][0]);                     // f u + g d (d . u)
                    acc[p][1] = fma2(f, fma2(k3, dy, uy), acc[p][1]);
                    acc[p][2] = fma2(f, fma2(k3, dz, uz), acc[p][2]);
                    acc[p][3] = fma2(f, pj, acc[p][3]);
                    if (EG) {
                        const f32x2 qi = fma2(dz, czi[p], fma2(dy, cyi[p], mul2(dx, cxi[p])));   // d . c_i
                        const f32x2 mq = EQM ? qi : mul2(mj, qi);                                // m_j (d . c_i)
                        const f32x2 g = mul2(mul2(f, y2), m3);                                   // -3 s^-5/2
                        acc[p][4] = fma2(g, mq, acc[p][4]);
                        acc[p][5] = fma2(f, mq, acc[p][5]);
                    }
                }
            }
        }
        __device__ __forceinline__ void flush_tile()
        {
#pragma unroll
            for (int p = 0; p < NPAIR; ++p)
#pragma unroll
                for (int k = 0; k < COMPS; ++k) {
                    float lo, hi;
                    unpk(acc[p][k], lo, hi);
                    osum[((2 * p) * COMPS + k) * CTHREADS] += (double)lo;
                    osum[((2 * p + 1) * COMPS + k) * CTHREADS] += (double)hi;
                    acc[p][k] = 0ull;
                }
        }
        __device__ __forceinline__ void write_row(double* __restrict__ row)
        {
#pragma unroll
            for (int q = 0; q < 2 * NPAIR; ++q) {
                const int r = q * CTHREADS + threadIdx.x;
#pragma unroll
                for (int k = 0; k < COMPS; ++k) row[(size_t)k * IB + r] = osum[(q * COMPS + k) * CTHREADS];
            }
        }
    };
};

// ---- fp64 consumer: IPT targets per thread, the scalar term of adjoint_terms.cuh --------------------------------
template <int IPT, bool EG>
struct VjpF64 {
    static constexpr int CWARPS = 8, MINB = 1, REC = 64, COMPS = EG ? 6 : 4;
    static constexpr int CTHREADS = CWARPS * 32;
    struct Params { const double4* posm; const double4* cot; double eps2; };
    static size_t outer_bytes() { return (size_t)IPT * COMPS * CTHREADS * sizeof(double); }

    template <bool EQM>
    struct State {
        const double4* __restrict__ posm;
        const double4* __restrict__ cot;
        const int64_t nt;
        const int32_t IB;
        const double eps2;
        double* __restrict__ osum;                 // osum[k * COMPS + comp][tid]
        double xi[IPT], yi[IPT], zi[IPT], mi[IPT], cxi[IPT], cyi[IPT], czi[IPT];
        double acc[IPT][6];

        __device__ __forceinline__ State(const Params& prm, const PairPlan& plan, unsigned char* outer)
            : posm(prm.posm), cot(prm.cot), nt(plan.nt), IB(plan.IB), eps2(prm.eps2), osum(reinterpret_cast<double*>(outer) + threadIdx.x)
        {
        }
        __device__ __forceinline__ void load_targets(const int32_t b)
        {
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                int64_t i = (int64_t)b * IB + (int64_t)k * CTHREADS + threadIdx.x;
                i = i < nt ? i : nt - 1;
                const double4 p = posm[i], c = cot[i];
                xi[k] = p.x; yi[k] = p.y; zi[k] = p.z; mi[k] = p.w;
                cxi[k] = c.x; cyi[k] = c.y; czi[k] = c.z;
#pragma unroll
                for (int q = 0; q < 6; ++q) acc[k][q] = 0.0;
            }
        }
        __device__ __forceinline__ void zero_outer()
        {
#pragma unroll
            for (int k = 0; k < IPT * COMPS; ++k) osum[k * CTHREADS] = 0.0;
        }
        __device__ __forceinline__ void tile(const unsigned char* tile_raw, const int len)
        {
            const double4* __restrict__ t = reinterpret_cast<const double4*>(tile_raw);
#pragma unroll 2
            for (int j = 0; j < len; ++j) {
                const double4 p = t[2 * j], c = t[2 * j + 1];
#pragma unroll
                for (int k = 0; k < IPT; ++k)
                    vjp_pair_term<double, EQM, EG>(p.x, p.y, p.z, p.w, c.x, c.y, c.z, xi[k], yi[k], zi[k], mi[k], cxi[k], cyi[k],
                                                   czi[k], eps2, acc[k][0], acc[k][1], acc[k][2], acc[k][3], acc[k][4], acc[k][5]);
            }
        }
        __device__ __forceinline__ void flush_tile()
        {
#pragma unroll
            for (int k = 0; k < IPT; ++k)
#pragma unroll
                for (int q = 0; q < COMPS; ++q) {
                    osum[(k * COMPS + q) * CTHREADS] += acc[k][q];
                    acc[k][q] = 0.0;
                }
        }
        __device__ __forceinline__ void write_row(double* __restrict__ row)
        {
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                const int r = k * CTHREADS + threadIdx.x;
#pragma unroll
                for (int q = 0; q < COMPS; ++q) row[(size_t)q * IB + r] = osum[(k * COMPS + q) * CTHREADS];
            }
        }
    };
};

// 6 targets per thread as 3 packed pairs, 8 compute warps, one CTA per SM, j loop unrolled 4: the best of the
// measured geometries (2-4 pairs x 8/12/16 warps x 1-2 CTAs: 1,080-1,180 G-pairs/s at N = 262,144).
constexpr int VJP_NPAIR = 3, VJP_CW = 8, VJP_MINB = 1, VJP_JU = 8;
constexpr int VJP_IPT64 = 2, VJP_T32 = 256, VJP_T64 = 128;

// Staged source record of the pull-back: {x, y, z, m}, {cx, cy, cz, 0} (fp32 32 B, fp64 64 B); padding records massless,
// parked far away, zero cotangent.
__device__ __forceinline__ void vjp_stage_record(void* jsrc, int64_t i, float x, float y, float z, float m, float cx, float cy, float cz)
{
    float4* out = reinterpret_cast<float4*>(jsrc) + 2 * i;
    out[0] = make_float4(x, y, z, m);
    out[1] = make_float4(cx, cy, cz, 0.f);
}
__device__ __forceinline__ void vjp_stage_record(void* jsrc, int64_t i, double x, double y, double z, double m, double cx, double cy,
                                                 double cz)
{
    double4* out = reinterpret_cast<double4*>(jsrc) + 2 * i;
    out[0] = make_double4(x, y, z, m);
    out[1] = make_double4(cx, cy, cz, 0.0);
}
__device__ __forceinline__ float vjp_pad_pos(float) { return PAD_POS_F32; }
__device__ __forceinline__ double vjp_pad_pos(double) { return PAD_POS_F64; }

// Stages record i (or its padding) and returns "this mass differs from posm[0].m"; block flags as in integrate.cu.
template <typename T>
__device__ __forceinline__ void vjp_stage_and_flag(void* __restrict__ jsrc, const PairPlan& plan, const int64_t i,
                                                   const typename AVec4<T>::type* __restrict__ posm, const T cx, const T cy, const T cz)
{
    int* const block_flag = const_cast<int*>(plan_flags(jsrc, plan)) + blockIdx.x;
    if (threadIdx.x == 0) *block_flag = 0;
    __syncthreads();
    int differs = 0;
    if (i < plan.n) {
        const typename AVec4<T>::type p = posm[i];
        vjp_stage_record(jsrc, i, p.x, p.y, p.z, p.w, cx, cy, cz);
        differs = !(p.w == posm[0].w);
    } else if (i < plan_npad(plan)) {
        const T far = vjp_pad_pos((T)0);
        vjp_stage_record(jsrc, i, far, far, far, (T)0, (T)0, (T)0, (T)0);
    }
    const unsigned any = __ballot_sync(0xffffffffu, differs);
    if (any != 0u && (threadIdx.x & 31) == 0) *block_flag = 1;
}

template <typename T>
__global__ void __launch_bounds__(VJP_THREADS)
vjp_stage_kernel(const typename AVec4<T>::type* __restrict__ posm, const typename AVec4<T>::type* __restrict__ cot,
                 void* __restrict__ jsrc, const PairPlan plan)
{
    pdl_launch_dependents();
    pdl_wait();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    T cx = (T)0, cy = (T)0, cz = (T)0;
    if (i < plan.n) { const typename AVec4<T>::type c = cot[i]; cx = c.x; cy = c.y; cz = c.z; }
    vjp_stage_and_flag<T>(jsrc, plan, i, posm, cx, cy, cz);
}

// Arguments of the backward KDK step that vjp_finish_kernel<.., PRE = true> fuses behind the row reduce.
template <typename T> struct VjpPreArgs {
    const typename AVec4<T>::type *posm_k, *vel_k, *accp_k, *posm_k1, *accp_k1;   // tape snapshots k and k + 1
    typename AVec4<T>::type *lv, *cot;
    PotParams<T> pot;
    T dt, w;
    int first;
};

// One backward KDK step before its pull-back (header of this file): with (x_k, v_k, a_k) and a_{k+1} from the tape,
//   dt term = Lx.vh_k + Lv.a_{k+1}/2 ;  Lv += dt Lx ;  dt term += Lv.a_k/2 ;  cot = w Lv.
// first != 0 (k = N): only cot = w Lv.  a = a_pair + a_ext(x) is rebuilt exactly as the forward kernel does.
// Also stages {x_k, cot} for the O(N^2) pull-back that follows (records, padding, equal-mass flags).  Returns the
// particle's dt term.  X = Lx_{k+1} of this particle.
template <typename T>
__device__ __forceinline__ double vjp_pre_step(const VjpPreArgs<T>& a, const PairPlan& plan, void* __restrict__ jsrc, const int64_t i,
                                               const typename AVec4<T>::type X)
{
    typedef typename AVec4<T>::type V4;
    double dterm = 0.0;
    V4 c; c.x = c.y = c.z = c.w = (T)0;
    if (i < plan.n) {
        V4 L = a.lv[i];
        if (!a.first) {
            const V4 p = a.posm_k[i], v = a.vel_k[i], ap = a.accp_k[i], p1 = a.posm_k1[i], ap1 = a.accp_k1[i];
            T ex, ey, ez;
            ext_accel<T>(a.pot, p.x, p.y, p.z, ex, ey, ez);
            const T ax = ap.x + ex, ay = ap.y + ey, az = ap.z + ez;
            ext_accel<T>(a.pot, p1.x, p1.y, p1.z, ex, ey, ez);
            const T bx = ap1.x + ex, by = ap1.y + ey, bz = ap1.z + ez;
            const T h = (T)0.5 * a.dt;
            const T vhx = fma(ax, h, v.x), vhy = fma(ay, h, v.y), vhz = fma(az, h, v.z);
            dterm = (double)X.x * vhx + (double)X.y * vhy + (double)X.z * vhz
                  + 0.5 * ((double)L.x * bx + (double)L.y * by + (double)L.z * bz);
            L.x = fma(a.dt, X.x, L.x); L.y = fma(a.dt, X.y, L.y); L.z = fma(a.dt, X.z, L.z);
            dterm += 0.5 * ((double)L.x * ax + (double)L.y * ay + (double)L.z * az);
            L.w = (T)0;
            a.lv[i] = L;
        }
        c.x = a.w * L.x; c.y = a.w * L.y; c.z = a.w * L.z;
        a.cot[i] = c;
    }
    vjp_stage_and_flag<T>(jsrc, plan, i, a.posm_k, c.x, c.y, c.z);
    return dterm;
}

// Row reduce (fixed unit order) + external part + accumulation:  gx_out (+)= G [m] rows + h,  gm_out (+)= -G row,
// block_sums[block][0..6] (+)= this block's terms of d/d(M_s, r_s, M_d, a, b, G, eps); slot 7 (+)= its dt terms;
// slots 8, 9 (+)= d/d(M_b, r_c).
// REDUCE = false skips the reduce (the step k = N, before any pull-back); PRE = true appends the backward KDK step
// of snapshot k - 1 for the same particle (everything it needs is this particle's own Lx, Lv): one O(N) launch per
// backward step instead of three.  Block sums accumulate over the steps of a backward pass in fixed step order;
// vjp_final_kernel adds the blocks once at the end.
template <typename T, bool EG, bool REDUCE, bool PRE>
__global__ void __launch_bounds__(VJP_THREADS)
vjp_finish_kernel(const typename AVec4<T>::type* __restrict__ posm, const typename AVec4<T>::type* __restrict__ cot,
                  const double* __restrict__ partials, void* __restrict__ jsrc, const PairPlan plan,
                  const double G, const double eps, const PotParams<double> pot,
                  typename AVec4<T>::type* __restrict__ gx_out, double* __restrict__ gm_out, const int accumulate,
                  double* __restrict__ block_sums, const VjpPreArgs<T> pre)
{
    typedef typename AVec4<T>::type V4;
    constexpr int COMPS = EG ? 6 : 4;
    __shared__ double warp_scratch[VJP_THREADS / 32];
    pdl_launch_dependents();
    pdl_wait();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double term[VJP_NOUT];
#pragma unroll
    for (int k = 0; k < VJP_NOUT; ++k) term[k] = 0.0;
    V4 o; o.x = o.y = o.z = o.w = (T)0;
    if (REDUCE && i < plan.n) {
        double r[COMPS];
        reduce_unit_rows<COMPS>(partials, plan, i, r);
        // the equal-mass loop left the common mass out of the x, y, z (and eps, G) sums
        const double mu = __ldcg(plan_eqm_word(jsrc, plan)) != 0 ? (double)posm[0].w : 1.0;
        const V4 p = posm[i], c = cot[i];
        double h[3], t[8];
        ext_vjp(pot, G, (double)p.x, (double)p.y, (double)p.z, (double)c.x, (double)c.y, (double)c.z, h, t);
        const double Gm = G * mu;
        double gx = fma(Gm, r[0], h[0]), gy = fma(Gm, r[1], h[1]), gz = fma(Gm, r[2], h[2]);
        double gm = -G * r[3];
        if (accumulate) {
            const V4 old = gx_out[i];
            gx += (double)old.x; gy += (double)old.y; gz += (double)old.z;
            gm += gm_out[i];
        }
        o.x = (T)gx; o.y = (T)gy; o.z = (T)gz;
        gx_out[i] = o;
        gm_out[i] = gm;
#pragma unroll
        for (int k = 0; k < 5; ++k) term[k] = t[k];
        term[8] = t[6];
        term[9] = t[7];
        if (EG) {
            term[5] = t[5] + mu * r[COMPS - 1];                         // d/dG: external + pair (sum_j m_j f d.c_i)
            term[6] = eps * Gm * r[COMPS - 2];
        }
    } else if (PRE && i < plan.n) {
        o = gx_out[i];
    }
    if (PRE) {
        __syncthreads();                                                // every read of the old staged flags / eqm word is done
        term[7] = vjp_pre_step<T>(pre, plan, jsrc, i, o);
    }
    if ((int64_t)blockIdx.x * blockDim.x < plan.n) {
#pragma unroll
        for (int k = 0; k < VJP_NOUT; ++k) {
            const double sum = vjp_block_sum(term[k], warp_scratch);
            if (threadIdx.x == 0) {
                double* slot = block_sums + (size_t)blockIdx.x * VJP_NOUT + k;
                *slot = accumulate ? *slot + sum : sum;
            }
        }
    }
}

// out[0..9] (+)= sum over blocks, in block order, of block_sums.
__global__ void __launch_bounds__(VJP_THREADS)
vjp_final_kernel(const double* __restrict__ block_sums, const int nblocks, double* __restrict__ out, const int accumulate)
{
    __shared__ double warp_scratch[VJP_THREADS / 32];
    pdl_wait();
    for (int k = 0; k < VJP_NOUT; ++k) {
        double v = 0.0;
        for (int b = threadIdx.x; b < nblocks; b += VJP_THREADS) v += block_sums[(size_t)b * VJP_NOUT + k];
        const double tot = vjp_block_sum(v, warp_scratch);
        if (threadIdx.x == 0) out[k] = accumulate ? out[k] + tot : tot;
    }
}

inline unsigned vjp_grid(int64_t n) { return (unsigned)((n + VJP_THREADS - 1) / VJP_THREADS); }

template <typename T> struct VjpKernels;
template <> struct VjpKernels<float> {
    typedef VjpF32<VJP_NPAIR, false, VJP_CW, VJP_MINB, VJP_JU> Plain;
    typedef VjpF32<VJP_NPAIR, true, VJP_CW, VJP_MINB, VJP_JU> WithEG;
};
template <> struct VjpKernels<double> {
    typedef VjpF64<VJP_IPT64, false> Plain;
    typedef VjpF64<VJP_IPT64, true> WithEG;
};

}  // namespace

cudaError_t configure_vjp()
{
    cudaError_t e = configure_stream<VjpKernels<float>::Plain>(VJP_T32);
    if (e == cudaSuccess) e = configure_stream<VjpKernels<float>::WithEG>(VJP_T32);
    if (e == cudaSuccess) e = configure_stream<VjpKernels<double>::Plain>(VJP_T64);
    if (e == cudaSuccess) e = configure_stream<VjpKernels<double>::WithEG>(VJP_T64);
    return e;
}

// Geometry of the pull-back kernels for make_vjp_plan (api.cu): {targets per thread, compute threads, tile records}.
void vjp_geometry(int is_f64, int* ipt, int* cthreads, int* tile, int* minb)
{
    *ipt = is_f64 ? VJP_IPT64 : 2 * VJP_NPAIR;
    *cthreads = is_f64 ? 256 : VJP_CW * 32;
    *tile = is_f64 ? VJP_T64 : VJP_T32;
    *minb = is_f64 ? 1 : VJP_MINB;
}

// Workspace of the pull-back: [staged records + flags][unit rows, 6 planes][block sums (VJP_NOUT = 10 per block)][cotangents].
static size_t vjp_rows_bytes(const PairPlan& plan) { return ((size_t)plan.U * 6 * plan.IB * sizeof(double) + 255) & ~(size_t)255; }
static size_t vjp_blocks_bytes(const PairPlan& plan)
{
    return ((size_t)((plan_npad(plan) + VJP_THREADS - 1) / VJP_THREADS) * VJP_NOUT * sizeof(double) + 255) & ~(size_t)255;
}

size_t vjp_workspace_bytes(const PairPlan& plan, int is_f64)
{
    return plan_jsrc_bytes(plan) + vjp_rows_bytes(plan) + vjp_blocks_bytes(plan) +
           (((size_t)plan.n * 4 * (is_f64 ? 8 : 4) + 255) & ~(size_t)255);
}

struct VjpCarve { void* jsrc; double* rows; double* block_sums; void* cot; };
static VjpCarve vjp_carve_all(void* ws, const PairPlan& plan)
{
    unsigned char* base = static_cast<unsigned char*>(ws);
    VjpCarve c;
    c.jsrc = plan_records(base, plan);
    c.rows = reinterpret_cast<double*>(base + plan_jsrc_bytes(plan));
    c.block_sums = reinterpret_cast<double*>(base + plan_jsrc_bytes(plan) + vjp_rows_bytes(plan));
    c.cot = base + plan_jsrc_bytes(plan) + vjp_rows_bytes(plan) + vjp_blocks_bytes(plan);
    return c;
}

template <typename T, bool EG, bool REDUCE, bool PRE>
static cudaError_t finish_launch(const PairPlan& plan, const VjpCarve& cv, const T* posm, double G, double eps,
                                 const PotParams<double>& pot, T* gx, double* gm, int accumulate, const VjpPreArgs<T>& pre,
                                 cudaStream_t stream)
{
    typedef typename AVec4<T>::type V4;
    const unsigned blocks = vjp_grid(PRE ? plan_npad(plan) : plan.n);
    return launch_pdl(vjp_finish_kernel<T, EG, REDUCE, PRE>, dim3(blocks), dim3(VJP_THREADS), 0, stream,
                      reinterpret_cast<const V4*>(posm), reinterpret_cast<const V4*>(cv.cot), (const double*)cv.rows, cv.jsrc, plan, G,
                      eps, pot, reinterpret_cast<V4*>(gx), gm, accumulate, cv.block_sums, pre);
}

template <typename T>
static cudaError_t pair_vjp_launch(const PairPlan& plan, const VjpCarve& cv, const T* posm, const T* cot, double eps, int with_eps_G,
                                   cudaStream_t stream)
{
    typedef typename AVec4<T>::type V4;
    typedef typename VjpKernels<T>::Plain Plain;
    typedef typename VjpKernels<T>::WithEG WithEG;
    const V4* p4 = reinterpret_cast<const V4*>(posm);
    const V4* c4 = reinterpret_cast<const V4*>(cot);
    if (with_eps_G) {
        const typename WithEG::Params prm{p4, c4, (T)(eps * eps)};
        return launch_stream<WithEG>(plan, prm, cv.jsrc, cv.jsrc, cv.rows, stream);
    }
    const typename Plain::Params prm{p4, c4, (T)(eps * eps)};
    return launch_stream<Plain>(plan, prm, cv.jsrc, cv.jsrc, cv.rows, stream);
}

// Cotangent cot pulled back through a = a_pair + a_ext at posm (odisseo_accel_vjp_*): stage, O(N^2) pass, finish, final.
template <typename T>
static cudaError_t accel_vjp_launch(const PairPlan& base_plan, const T* posm, const T* cot, double G, double eps,
                                    const PotParams<double>& pot, T* gx, double* gm, double* gparams, int with_eps_G, void* ws,
                                    cudaStream_t stream)
{
    typedef typename AVec4<T>::type V4;
    PairPlan plan = base_plan;
    plan.comps = with_eps_G ? 6 : 4;
    VjpCarve cv = vjp_carve_all(ws, plan);
    cudaError_t e = launch_pdl(vjp_stage_kernel<T>, dim3(vjp_grid(plan_npad(plan))), dim3(VJP_THREADS), 0, stream,
                               reinterpret_cast<const V4*>(posm), reinterpret_cast<const V4*>(cot), cv.jsrc, plan);
    if (e != cudaSuccess) return e;
    e = pair_vjp_launch<T>(plan, cv, posm, cot, eps, with_eps_G, stream);
    if (e != cudaSuccess) return e;
    cv.cot = const_cast<T*>(cot);                           // the finish kernel reads the caller's cotangents
    VjpPreArgs<T> none;
    memset(&none, 0, sizeof(none));
    e = with_eps_G ? finish_launch<T, true, true, false>(plan, cv, posm, G, eps, pot, gx, gm, 0, none, stream)
                   : finish_launch<T, false, true, false>(plan, cv, posm, G, eps, pot, gx, gm, 0, none, stream);
    if (e != cudaSuccess) return e;
    return launch_pdl(vjp_final_kernel, dim3(1), dim3(VJP_THREADS), 0, stream, (const double*)cv.block_sums, (int)vjp_grid(plan.n),
                      gparams, 0);
}

cudaError_t launch_accel_vjp_f32(const PairPlan& plan, const float* posm, const float* cot, double G, double eps,
                                 const PotParams<double>& pot, float* gx, double* gm, double* gparams, int with_eps_G, void* ws,
                                 cudaStream_t stream)
{ return accel_vjp_launch<float>(plan, posm, cot, G, eps, pot, gx, gm, gparams, with_eps_G, ws, stream); }
cudaError_t launch_accel_vjp_f64(const PairPlan& plan, const double* posm, const double* cot, double G, double eps,
                                 const PotParams<double>& pot, double* gx, double* gm, double* gparams, int with_eps_G, void* ws,
                                 cudaStream_t stream)
{ return accel_vjp_launch<double>(plan, posm, cot, G, eps, pot, gx, gm, gparams, with_eps_G, ws, stream); }

// Backward pass through nsteps KDK steps recorded on `tape` (odisseo_leapfrog_kdk_vjp_*): per snapshot k = N .. 0 one
// O(N^2) pull-back and ONE O(N) kernel (row reduce of k fused with the backward KDK step and staging of k - 1);
// the parameter sums are added over blocks once at the end.  lx, lv: in = dL/d(final state), out = dL/d(initial state).
template <typename T>
static cudaError_t leapfrog_vjp_launch(const PairPlan& base_plan, const T* tape, int64_t nsteps, double G, double eps, T dt,
                                       const PotParams<double>& pot64, const PotParams<T>& pot, int with_eps_G, T* lx, T* lv,
                                       double* gm, double* gparams, void* ws, int64_t* launches, cudaStream_t stream)
{
    typedef typename AVec4<T>::type V4;
    PairPlan plan = base_plan;
    plan.comps = with_eps_G ? 6 : 4;
    const VjpCarve cv = vjp_carve_all(ws, plan);
    const size_t arr = (size_t)plan.n * 4, snap = 3 * arr;
    const T half = (T)0.5 * dt;
    auto pre_args = [&](int64_t k, int first) {
        const T* tk = tape + (size_t)k * snap;
        const T* tk1 = first ? nullptr : tk + snap;
        VjpPreArgs<T> a;
        a.posm_k = reinterpret_cast<const V4*>(tk);
        a.vel_k = reinterpret_cast<const V4*>(tk + arr);
        a.accp_k = reinterpret_cast<const V4*>(tk + 2 * arr);
        a.posm_k1 = reinterpret_cast<const V4*>(tk1);
        a.accp_k1 = reinterpret_cast<const V4*>(tk1 ? tk1 + 2 * arr : nullptr);
        a.lv = reinterpret_cast<V4*>(lv);
        a.cot = reinterpret_cast<V4*>(cv.cot);
        a.pot = pot;
        a.dt = dt;
        a.w = (first || k == 0) ? half : dt;
        a.first = first;
        return a;
    };
    // k = N: cot = dt/2 Lv_N, stage x_N; also zeroes the block sums (accumulate = 0)
    cudaError_t e = with_eps_G
        ? finish_launch<T, true, false, true>(plan, cv, tape + (size_t)nsteps * snap, G, eps, pot64, lx, gm, 0, pre_args(nsteps, 1), stream)
        : finish_launch<T, false, false, true>(plan, cv, tape + (size_t)nsteps * snap, G, eps, pot64, lx, gm, 0, pre_args(nsteps, 1), stream);
    if (e != cudaSuccess) return e;
    *launches += 1;
    for (int64_t k = nsteps; k >= 0; --k) {
        const T* tk = tape + (size_t)k * snap;
        e = pair_vjp_launch<T>(plan, cv, tk, static_cast<const T*>(cv.cot), eps, with_eps_G, stream);
        if (e != cudaSuccess) return e;
        if (k > 0) {
            const VjpPreArgs<T> a = pre_args(k - 1, 0);
            e = with_eps_G ? finish_launch<T, true, true, true>(plan, cv, tk, G, eps, pot64, lx, gm, 1, a, stream)
                           : finish_launch<T, false, true, true>(plan, cv, tk, G, eps, pot64, lx, gm, 1, a, stream);
        } else {
            VjpPreArgs<T> none;
            memset(&none, 0, sizeof(none));
            e = with_eps_G ? finish_launch<T, true, true, false>(plan, cv, tk, G, eps, pot64, lx, gm, 1, none, stream)
                           : finish_launch<T, false, true, false>(plan, cv, tk, G, eps, pot64, lx, gm, 1, none, stream);
        }
        if (e != cudaSuccess) return e;
        *launches += 2;
    }
    *launches += 1;
    return launch_pdl(vjp_final_kernel, dim3(1), dim3(VJP_THREADS), 0, stream, (const double*)cv.block_sums, (int)vjp_grid(plan.n),
                      gparams, 0);
}

cudaError_t launch_leapfrog_vjp_f32(const PairPlan& plan, const float* tape, int64_t nsteps, double G, double eps, float dt,
                                    const PotParams<double>& pot64, const PotParams<float>& pot, int with_eps_G, float* lx, float* lv,
                                    double* gm, double* gparams, void* ws, int64_t* launches, cudaStream_t stream)
{ return leapfrog_vjp_launch<float>(plan, tape, nsteps, G, eps, dt, pot64, pot, with_eps_G, lx, lv, gm, gparams, ws, launches, stream); }
cudaError_t launch_leapfrog_vjp_f64(const PairPlan& plan, const double* tape, int64_t nsteps, double G, double eps, double dt,
                                    const PotParams<double>& pot64, const PotParams<double>& pot, int with_eps_G, double* lx, double* lv,
                                    double* gm, double* gparams, void* ws, int64_t* launches, cudaStream_t stream)
{ return leapfrog_vjp_launch<double>(plan, tape, nsteps, G, eps, dt, pot64, pot, with_eps_G, lx, lv, gm, gparams, ws, launches, stream); }

}  // namespace odisseo
