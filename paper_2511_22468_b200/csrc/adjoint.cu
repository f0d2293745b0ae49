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
// The O(N^2) pass is a plain shared-memory tiled kernel (35 flops per pair, about 2.7x the forward pass):
// grid = (target blocks, source splits); per-tile sums in the state's precision, promoted to fp64 between
// tiles; split rows and every block sum are combined in a fixed order (bit-reproducible, no atomics).
// The O(N) parts (external potential, parameter sums) are evaluated in fp64 whatever the state precision.
#include "adjoint_terms.cuh"

namespace odisseo {

namespace {

constexpr int VJP_TILE = 128;

template <typename T> struct AVec4;
template <> struct AVec4<float> { typedef float4 type; };
template <> struct AVec4<double> { typedef double4 type; };

// partial rows: partials[((split * VJP_COMPS + comp) * n_rows) + i], comp = gx, gy, gz, mass term, eps term, G term
template <typename T, int IPT, bool EG>
__global__ void __launch_bounds__(VJP_THREADS)
pair_vjp_kernel(const typename AVec4<T>::type* __restrict__ posm, const typename AVec4<T>::type* __restrict__ cot,
                const int64_t n, const int64_t n_rows, const int64_t chunk, const T eps2, double* __restrict__ partials)
{
    typedef typename AVec4<T>::type V4;
    __shared__ V4 sp[VJP_TILE];
    __shared__ V4 sc[VJP_TILE];
    __shared__ __align__(8) float soa[sizeof(T) == 4 ? 6 * VJP_TILE : 2];   // x[], y[], z[], cx[], cy[], cz[] (packed fp32 loop)
    const int tid = threadIdx.x;
    const int64_t i_base = (int64_t)blockIdx.x * (VJP_THREADS * IPT) + tid;
    const int64_t j_begin = (int64_t)blockIdx.y * chunk;
    const int64_t j_end = j_begin + chunk < n ? j_begin + chunk : n;

    T xi[IPT], yi[IPT], zi[IPT], mi[IPT], cxi[IPT], cyi[IPT], czi[IPT];
    double ox[IPT], oy[IPT], oz[IPT], om[IPT], oe[IPT], og[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        int64_t i = i_base + (int64_t)k * VJP_THREADS;
        i = i < n ? i : n - 1;                              // clamped rows are computed and never read back
        const V4 p = posm[i], c = cot[i];
        xi[k] = p.x; yi[k] = p.y; zi[k] = p.z; mi[k] = p.w;
        cxi[k] = c.x; cyi[k] = c.y; czi[k] = c.z;
        ox[k] = oy[k] = oz[k] = om[k] = oe[k] = og[k] = 0.0;
    }
    // Equal masses are recognised tile by tile: when every target of this block and every source of the tile
    // carry the same mass mu, u = mu (c_j - c_i) and the mass leaves the loop (vjp_pair_term EQM: 28 instead of
    // 35 instructions); the tile sum is scaled by mu when it is promoted.  A block-uniform decision per tile.
    const T mu = posm[(int64_t)blockIdx.x * (VJP_THREADS * IPT) < n ? (int64_t)blockIdx.x * (VJP_THREADS * IPT) : n - 1].w;
    int mine_equal = 1;
#pragma unroll
    for (int k = 0; k < IPT; ++k) mine_equal &= (mi[k] == mu);
    const bool targets_equal = !EG && __syncthreads_and(mine_equal) != 0;

    for (int64_t j0 = j_begin; j0 < j_end; j0 += VJP_TILE) {
        __syncthreads();                                    // previous tile consumed
        int src_equal = 1;
        if (tid < VJP_TILE) {
            const int64_t j = j0 + tid;
            V4 p, c;
            if (j < j_end) { p = posm[j]; c = cot[j]; }
            else { p.x = p.y = p.z = p.w = (T)0; c.x = c.y = c.z = c.w = (T)0; }   // m = 0, c = 0: contributes 0
            sp[tid] = p;
            sc[tid] = c;
            if constexpr (sizeof(T) == 4) {
                soa[tid] = p.x; soa[VJP_TILE + tid] = p.y; soa[2 * VJP_TILE + tid] = p.z;
                soa[3 * VJP_TILE + tid] = c.x; soa[4 * VJP_TILE + tid] = c.y; soa[5 * VJP_TILE + tid] = c.z;
            }
            src_equal = (p.w == mu);                        // padding (m = 0) makes the tile general
        }
        const bool eqm = __syncthreads_and(src_equal) != 0 && targets_equal;      // also: tile staged
        T ax[IPT], ay[IPT], az[IPT], am[IPT], ae[IPT], ag[IPT];
#pragma unroll
        for (int k = 0; k < IPT; ++k) ax[k] = ay[k] = az[k] = am[k] = ae[k] = ag[k] = (T)0;
        if (eqm) {
            if constexpr (sizeof(T) == 4) {
                // packed fp32 loop: two sources per instruction, the target duplicated in both halves
                const f32x2 e2 = pk(eps2, eps2), m3 = pk(-3.0f, -3.0f);
                f32x2 X[IPT], Y[IPT], Z[IPT], CX[IPT], CY[IPT], CZ[IPT], a2[IPT][4];
#pragma unroll
                for (int k = 0; k < IPT; ++k) {
                    X[k] = pk(xi[k], xi[k]); Y[k] = pk(yi[k], yi[k]); Z[k] = pk(zi[k], zi[k]);
                    CX[k] = pk(cxi[k], cxi[k]); CY[k] = pk(cyi[k], cyi[k]); CZ[k] = pk(czi[k], czi[k]);
                    a2[k][0] = a2[k][1] = a2[k][2] = a2[k][3] = 0ull;
                }
                const f32x2* const s2 = reinterpret_cast<const f32x2*>(soa);
                constexpr int H = VJP_TILE / 2;
#pragma unroll 2
                for (int j = 0; j < H; ++j) {
                    const f32x2 px = s2[j], py = s2[H + j], pz = s2[2 * H + j];
                    const f32x2 qx = s2[3 * H + j], qy = s2[4 * H + j], qz = s2[5 * H + j];
#pragma unroll
                    for (int k = 0; k < IPT; ++k)
                        vjp_pair_term_x2(px, py, pz, qx, qy, qz, X[k], Y[k], Z[k], CX[k], CY[k], CZ[k], e2, m3, a2[k][0], a2[k][1],
                                         a2[k][2], a2[k][3]);
                }
#pragma unroll
                for (int k = 0; k < IPT; ++k) {
                    float lo, hi;
                    unpk(a2[k][0], lo, hi); ax[k] = lo + hi;
                    unpk(a2[k][1], lo, hi); ay[k] = lo + hi;
                    unpk(a2[k][2], lo, hi); az[k] = lo + hi;
                    unpk(a2[k][3], lo, hi); am[k] = lo + hi;
                }
            } else {
#pragma unroll 4
                for (int j = 0; j < VJP_TILE; ++j) {
                    const V4 p = sp[j], c = sc[j];
#pragma unroll
                    for (int k = 0; k < IPT; ++k)
                        vjp_pair_term<T, true, false>(p.x, p.y, p.z, p.w, c.x, c.y, c.z, xi[k], yi[k], zi[k], mi[k], cxi[k], cyi[k],
                                                      czi[k], eps2, ax[k], ay[k], az[k], am[k], ae[k], ag[k]);
                }
            }
        } else {
#pragma unroll 4
            for (int j = 0; j < VJP_TILE; ++j) {
                const V4 p = sp[j], c = sc[j];
#pragma unroll
                for (int k = 0; k < IPT; ++k)
                    vjp_pair_term<T, false, EG>(p.x, p.y, p.z, p.w, c.x, c.y, c.z, xi[k], yi[k], zi[k], mi[k], cxi[k], cyi[k],
                                                czi[k], eps2, ax[k], ay[k], az[k], am[k], ae[k], ag[k]);
            }
        }
        const double scale = eqm ? (double)mu : 1.0;
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            ox[k] = fma(scale, (double)ax[k], ox[k]); oy[k] = fma(scale, (double)ay[k], oy[k]); oz[k] = fma(scale, (double)az[k], oz[k]);
            om[k] += (double)am[k]; oe[k] += (double)ae[k]; og[k] += (double)ag[k];
        }
    }
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int64_t i = i_base + (int64_t)k * VJP_THREADS;
        if (i < n) {
            double* row = partials + (size_t)blockIdx.y * VJP_COMPS * n_rows + i;
            row[0] = ox[k]; row[n_rows] = oy[k]; row[2 * n_rows] = oz[k]; row[3 * n_rows] = om[k]; row[4 * n_rows] = oe[k]; row[5 * n_rows] = og[k];
        }
    }
}

// Row reduce (fixed split order) + external part + accumulation:  gx_out (+)= G rows + h,  gm_out (+)= -G row,
// block_sums[block][0..7] = this block's terms of d/d(M_s, r_s, M_d, a, b, G, eps) (slot 7 left 0).
template <typename T>
__global__ void __launch_bounds__(VJP_THREADS)
vjp_finish_kernel(const typename AVec4<T>::type* __restrict__ posm, const typename AVec4<T>::type* __restrict__ cot,
                  const double* __restrict__ partials, const int64_t n, const int64_t n_rows, const int nsplit,
                  const double G, const double eps, const PotParams<double> pot,
                  typename AVec4<T>::type* __restrict__ gx_out, double* __restrict__ gm_out, const int accumulate,
                  const int with_eps_G, double* __restrict__ block_sums)
{
    typedef typename AVec4<T>::type V4;
    __shared__ double warp_scratch[VJP_THREADS / 32];
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double term[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) term[k] = 0.0;
    if (i < n) {
        double r[VJP_COMPS];
#pragma unroll
        for (int k = 0; k < VJP_COMPS; ++k) r[k] = 0.0;
        for (int sidx = 0; sidx < nsplit; ++sidx) {                     // increasing j
            const double* row = partials + (size_t)sidx * VJP_COMPS * n_rows + i;
#pragma unroll
            for (int k = 0; k < VJP_COMPS; ++k) r[k] += __ldcg(row + (size_t)k * n_rows);
        }
        const V4 p = posm[i], c = cot[i];
        double h[3], t[6];
        ext_vjp(pot, G, (double)p.x, (double)p.y, (double)p.z, (double)c.x, (double)c.y, (double)c.z, h, t);
        double gx = fma(G, r[0], h[0]), gy = fma(G, r[1], h[1]), gz = fma(G, r[2], h[2]);
        double gm = -G * r[3];
        if (accumulate) {
            const V4 old = gx_out[i];
            gx += (double)old.x; gy += (double)old.y; gz += (double)old.z;
            gm += gm_out[i];
        }
        V4 o; o.x = (T)gx; o.y = (T)gy; o.z = (T)gz; o.w = (T)0;
        gx_out[i] = o;
        gm_out[i] = gm;
#pragma unroll
        for (int k = 0; k < 5; ++k) term[k] = t[k];
        if (with_eps_G) {
            term[5] = t[5] + r[5];                                      // d/dG: external + pair (sum_j m_j f d.c_i)
            term[6] = eps * G * r[4];
        }
    }
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        const double sum = vjp_block_sum(term[k], warp_scratch);
        if (threadIdx.x == 0) block_sums[(size_t)blockIdx.x * 8 + k] = sum;
    }
    if (threadIdx.x == 0) block_sums[(size_t)blockIdx.x * 8 + 7] = 0.0;
}

// out[0..7] (+)= sum over blocks, in block order, of block_sums (and of dt_sums into slot 7 when given).
__global__ void __launch_bounds__(VJP_THREADS)
vjp_final_kernel(const double* __restrict__ block_sums, const double* __restrict__ dt_sums, const int nblocks,
                 double* __restrict__ out, const int accumulate)
{
    __shared__ double warp_scratch[VJP_THREADS / 32];
    for (int k = 0; k < 8; ++k) {
        double v = 0.0;
        if (block_sums)
            for (int b = threadIdx.x; b < nblocks; b += VJP_THREADS) v += block_sums[(size_t)b * 8 + k];
        if (k == 7 && dt_sums)
            for (int b = threadIdx.x; b < nblocks; b += VJP_THREADS) v += dt_sums[b];
        const double tot = vjp_block_sum(v, warp_scratch);
        if (threadIdx.x == 0) out[k] = accumulate ? out[k] + tot : tot;
    }
}

// One backward KDK step before its pull-back (header of this file): with (x_k, v_k, a_k) and a_{k+1} from the tape,
//   dt term = Lx.vh_k + Lv.a_{k+1}/2 ;  Lv += dt Lx ;  dt term += Lv.a_k/2 ;  cot = w Lv.
// first != 0 (k = N): only cot = w Lv.  a = a_pair + a_ext(x) is rebuilt exactly as the forward kernel does.
template <typename T>
__global__ void __launch_bounds__(VJP_THREADS)
vjp_pre_kernel(const typename AVec4<T>::type* __restrict__ posm_k, const typename AVec4<T>::type* __restrict__ vel_k,
               const typename AVec4<T>::type* __restrict__ accp_k, const typename AVec4<T>::type* __restrict__ posm_k1,
               const typename AVec4<T>::type* __restrict__ accp_k1, const int64_t n, const PotParams<T> pot, const T dt,
               const T w, const int first, const typename AVec4<T>::type* __restrict__ lx,
               typename AVec4<T>::type* __restrict__ lv, typename AVec4<T>::type* __restrict__ cot,
               double* __restrict__ dt_sums)
{
    typedef typename AVec4<T>::type V4;
    __shared__ double warp_scratch[VJP_THREADS / 32];
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double dterm = 0.0;
    if (i < n) {
        V4 L = lv[i];
        if (!first) {
            const V4 X = lx[i];
            const V4 p = posm_k[i], v = vel_k[i], ap = accp_k[i], p1 = posm_k1[i], ap1 = accp_k1[i];
            T ex, ey, ez;
            ext_accel<T>(pot, p.x, p.y, p.z, ex, ey, ez);
            const T ax = ap.x + ex, ay = ap.y + ey, az = ap.z + ez;
            ext_accel<T>(pot, p1.x, p1.y, p1.z, ex, ey, ez);
            const T bx = ap1.x + ex, by = ap1.y + ey, bz = ap1.z + ez;
            const T h = (T)0.5 * dt;
            const T vhx = fma(ax, h, v.x), vhy = fma(ay, h, v.y), vhz = fma(az, h, v.z);
            dterm = (double)X.x * vhx + (double)X.y * vhy + (double)X.z * vhz
                  + 0.5 * ((double)L.x * bx + (double)L.y * by + (double)L.z * bz);
            L.x = fma(dt, X.x, L.x); L.y = fma(dt, X.y, L.y); L.z = fma(dt, X.z, L.z);
            dterm += 0.5 * ((double)L.x * ax + (double)L.y * ay + (double)L.z * az);
            L.w = (T)0;
            lv[i] = L;
        }
        V4 c; c.x = w * L.x; c.y = w * L.y; c.z = w * L.z; c.w = (T)0;
        cot[i] = c;
    }
    const double sum = vjp_block_sum(dterm, warp_scratch);
    if (threadIdx.x == 0) dt_sums[blockIdx.x] = sum;
}

inline unsigned vjp_grid(int64_t n) { return (unsigned)((n + VJP_THREADS - 1) / VJP_THREADS); }

}  // namespace

// Launch geometry of the O(N^2) pull-back for n particles: source splits and rows (host arithmetic).
void vjp_plan(int64_t n, int num_sms, int* nsplit, int64_t* chunk)
{
    const int64_t iblocks = (n + VJP_THREADS * 2 - 1) / (VJP_THREADS * 2);
    int64_t s = (2 * (int64_t)num_sms + iblocks - 1) / iblocks;
    const int64_t max_s = (n + VJP_TILE - 1) / VJP_TILE;
    if (s > max_s) s = max_s;
    if (s > 64) s = 64;
    if (s < 1) s = 1;
    int64_t c = (n + s - 1) / s;
    c = (c + VJP_TILE - 1) / VJP_TILE * VJP_TILE;
    *chunk = c;
    *nsplit = (int)((n + c - 1) / c);
}

size_t vjp_workspace_bytes(int64_t n, int is_f64, int num_sms)
{
    int nsplit; int64_t chunk;
    vjp_plan(n, num_sms, &nsplit, &chunk);
    const size_t blocks = (size_t)((n + VJP_THREADS - 1) / VJP_THREADS);
    size_t b = (size_t)nsplit * VJP_COMPS * n * sizeof(double);       // partial rows
    b = (b + 255) & ~(size_t)255;
    b += (blocks * 9 * sizeof(double) + 255) & ~(size_t)255;           // block sums (8) + dt sums (1)
    b += ((size_t)n * 4 * (is_f64 ? 8 : 4) + 255) & ~(size_t)255;      // cotangent array of the KDK pull-back
    return b;
}

template <typename T>
static cudaError_t accel_vjp_launch(const T* posm, const T* cot, int64_t n, double G, double eps,
                                    const PotParams<double>& pot, T* gx, double* gm, double* gparams, const double* dt_sums,
                                    int accumulate, int with_eps_G, void* ws, int num_sms, cudaStream_t stream)
{
    typedef typename AVec4<T>::type V4;
    int nsplit; int64_t chunk;
    vjp_plan(n, num_sms, &nsplit, &chunk);
    double* partials = static_cast<double*>(ws);
    size_t off = ((size_t)nsplit * VJP_COMPS * n * sizeof(double) + 255) & ~(size_t)255;
    double* block_sums = reinterpret_cast<double*>(static_cast<unsigned char*>(ws) + off);
    const unsigned blocks = vjp_grid(n);
    dim3 grid((unsigned)((n + VJP_THREADS * 2 - 1) / (VJP_THREADS * 2)), (unsigned)nsplit);
    if (with_eps_G)
        pair_vjp_kernel<T, 2, true><<<grid, VJP_THREADS, 0, stream>>>(reinterpret_cast<const V4*>(posm), reinterpret_cast<const V4*>(cot),
                                                                      n, n, chunk, (T)(eps * eps), partials);
    else
        pair_vjp_kernel<T, 2, false><<<grid, VJP_THREADS, 0, stream>>>(reinterpret_cast<const V4*>(posm), reinterpret_cast<const V4*>(cot),
                                                                       n, n, chunk, (T)(eps * eps), partials);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    vjp_finish_kernel<T><<<blocks, VJP_THREADS, 0, stream>>>(reinterpret_cast<const V4*>(posm), reinterpret_cast<const V4*>(cot),
                                                             partials, n, n, nsplit, G, eps, pot, reinterpret_cast<V4*>(gx), gm,
                                                             accumulate, with_eps_G, block_sums);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    vjp_final_kernel<<<1, VJP_THREADS, 0, stream>>>(block_sums, dt_sums, (int)blocks, gparams, accumulate);
    return cudaGetLastError();
}

cudaError_t launch_accel_vjp_f32(const float* posm, const float* cot, int64_t n, double G, double eps, const PotParams<double>& pot,
                                 float* gx, double* gm, double* gparams, const double* dt_sums, int accumulate, int with_eps_G,
                                 void* ws, int num_sms, cudaStream_t stream)
{ return accel_vjp_launch<float>(posm, cot, n, G, eps, pot, gx, gm, gparams, dt_sums, accumulate, with_eps_G, ws, num_sms, stream); }
cudaError_t launch_accel_vjp_f64(const double* posm, const double* cot, int64_t n, double G, double eps, const PotParams<double>& pot,
                                 double* gx, double* gm, double* gparams, const double* dt_sums, int accumulate, int with_eps_G,
                                 void* ws, int num_sms, cudaStream_t stream)
{ return accel_vjp_launch<double>(posm, cot, n, G, eps, pot, gx, gm, gparams, dt_sums, accumulate, with_eps_G, ws, num_sms, stream); }

// dt sums and cotangent array live behind the block sums in the workspace (vjp_workspace_bytes).
void vjp_carve(void* ws, int64_t n, int num_sms, double** dt_sums, void** cot)
{
    int nsplit; int64_t chunk;
    vjp_plan(n, num_sms, &nsplit, &chunk);
    const size_t blocks = (size_t)((n + VJP_THREADS - 1) / VJP_THREADS);
    size_t off = ((size_t)nsplit * VJP_COMPS * n * sizeof(double) + 255) & ~(size_t)255;
    *dt_sums = reinterpret_cast<double*>(static_cast<unsigned char*>(ws) + off) + blocks * 8;
    off += (blocks * 9 * sizeof(double) + 255) & ~(size_t)255;
    *cot = static_cast<unsigned char*>(ws) + off;
}

template <typename T>
static cudaError_t vjp_pre_launch(const T* tape_k, const T* tape_k1, int64_t n, const PotParams<T>& pot, T dt, T w, int first,
                                  const T* lx, T* lv, T* cot, double* dt_sums, cudaStream_t stream)
{
    typedef typename AVec4<T>::type V4;
    const size_t arr = (size_t)n * 4;
    vjp_pre_kernel<T><<<vjp_grid(n), VJP_THREADS, 0, stream>>>(
        reinterpret_cast<const V4*>(tape_k), reinterpret_cast<const V4*>(tape_k + arr), reinterpret_cast<const V4*>(tape_k + 2 * arr),
        reinterpret_cast<const V4*>(tape_k1), reinterpret_cast<const V4*>(tape_k1 ? tape_k1 + 2 * arr : nullptr), n, pot, dt, w,
        first, reinterpret_cast<const V4*>(lx), reinterpret_cast<V4*>(lv), reinterpret_cast<V4*>(cot), dt_sums);
    return cudaGetLastError();
}
cudaError_t launch_vjp_pre_f32(const float* tape_k, const float* tape_k1, int64_t n, const PotParams<float>& pot, float dt, float w,
                               int first, const float* lx, float* lv, float* cot, double* dt_sums, cudaStream_t stream)
{ return vjp_pre_launch<float>(tape_k, tape_k1, n, pot, dt, w, first, lx, lv, cot, dt_sums, stream); }
cudaError_t launch_vjp_pre_f64(const double* tape_k, const double* tape_k1, int64_t n, const PotParams<double>& pot, double dt,
                               double w, int first, const double* lx, double* lv, double* cot, double* dt_sums, cudaStream_t stream)
{ return vjp_pre_launch<double>(tape_k, tape_k1, n, pot, dt, w, first, lx, lv, cot, dt_sums, stream); }

}  // namespace odisseo
