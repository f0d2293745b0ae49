// C ABI of the ODISSEO B200 library (include/odisseo.h): argument validation, launch plan,
// workspace carving, per-step launch sequence and its CUDA-graph capture.
#include <math.h>
#include <string.h>

#include <atomic>
#include <mutex>
#include <vector>

#include "odisseo_common.cuh"

namespace odisseo {

// ------------------------------- launch plan ------------------------------------------
PairPlan make_plan(int64_t n, int is_f64, int num_sms) { return make_cross_plan(n, n, is_f64, num_sms); }

// Geometry of one kernel variant: i-bodies per thread, compute threads, resident CTAs per SM.
struct VariantGeom { int ipt, cthreads, minb; };
static VariantGeom variant_geom(int variant, int is_f64)
{
    // fp32: one 8-warp CTA per SM with ~160 registers per thread lets ptxas interleave the four
    // packed interaction chains of a thread (2 warps per scheduler x ILP 4 beats 4.5 warps x ILP 1:
    // 68.9 % vs 60.2 % of FP32 peak at N = 262,144)
    if (variant == 0) return VariantGeom{is_f64 ? 4 : 8, 256, 1};
    return VariantGeom{2, 64, 8};
}

// Tile length and chunk count: functions of the SOURCE count (and the SM count) alone, so that a slice of
// the targets evaluated anywhere adds the same numbers in the same grouping.
// T: the longest tile the variant n would get on its own stages.  S: the busiest CTA walks
// ceil(nb S / P) units of (chunk records + per-tile and per-row overheads, in records' worth of time); take
// the S that minimises that product for the single-device evaluation nt = n; chunks hold >= 32 sources.
static int32_t source_split(int64_t n, int32_t T, int64_t targets_per_cta, int64_t Pmax)
{
    const int64_t n8 = (n + 7) / 8;
    const int64_t nb = (n + targets_per_cta - 1) / targets_per_cta;
    int64_t smax = n8 / 4;
    if (smax < 1) smax = 1;
    if (smax > 512) smax = 512;
    int64_t best = -1;
    int32_t S = 1;
    for (int64_t s = 1; s <= smax; ++s) {
        const int64_t chunk = 8 * ((n8 + s - 1) / s);
        const int64_t tiles = (chunk + T - 1) / T;
        const int64_t U = nb * s;
        const int64_t ctas = U < Pmax ? U : Pmax;
        const int64_t cost = ((U + ctas - 1) / ctas) * (chunk + 16 * tiles + 32) + 2 * s;
        if (best < 0 || cost < best) { best = cost; S = (int32_t)s; }
    }
    return S;
}

PairPlan make_cross_plan(int64_t nt, int64_t n, int is_f64, int num_sms)
{
    PairPlan p;
    memset(&p, 0, sizeof(p));
    p.n = n;
    p.nt = nt;
    p.n8 = (n + 7) / 8;
    {
        // T: the longest tile the variant n would get on its own stages (the small variant's hold 256 records)
        const VariantGeom gn = variant_geom(n <= 4096 ? 1 : 0, is_f64);
        p.T = (n > 4096 && !is_f64) ? 512 : 256;
        p.S = source_split(n, p.T, (int64_t)gn.ipt * gn.cthreads, (int64_t)num_sms * gn.minb);
    }
    p.variant = (nt <= 4096 && n <= 4096) ? 1 : 0;
    const VariantGeom g = variant_geom(p.variant, is_f64);
    p.ipt = g.ipt;
    p.cthreads = g.cthreads;
    p.rec_bytes = is_f64 ? 32 : 16;                       // staged records are plain {x, y, z, m}
    p.comps = 3;
    p.IB = p.ipt * p.cthreads;
    p.nb = (int32_t)((nt + p.IB - 1) / p.IB);
    p.U = (int64_t)p.nb * p.S;
    int64_t P = (int64_t)num_sms * g.minb;
    if (P > p.U) P = p.U;
    if (P < 1) P = 1;
    p.P = (int32_t)P;
    return p;
}

// Plan of the O(N^2) pull-back kernels (adjoint.cu): targets = sources = the n particles, one CTA per SM.
PairPlan make_vjp_plan(int64_t n, int is_f64, int num_sms)
{
    PairPlan p;
    memset(&p, 0, sizeof(p));
    int ipt, cthreads, tile, minb;
    vjp_geometry(is_f64, &ipt, &cthreads, &tile, &minb);
    p.n = p.nt = n;
    p.n8 = (n + 7) / 8;
    p.T = tile;
    p.ipt = ipt;
    p.cthreads = cthreads;
    p.IB = ipt * cthreads;
    p.S = source_split(n, p.T, p.IB, (int64_t)num_sms * minb);
    p.variant = 0;
    p.rec_bytes = is_f64 ? 64 : 32;                       // {x, y, z, m}, {cx, cy, cz, 0}
    p.comps = 6;
    p.nb = (int32_t)((n + p.IB - 1) / p.IB);
    p.U = (int64_t)p.nb * p.S;
    int64_t P = (int64_t)num_sms * minb;
    if (P > p.U) P = p.U;
    if (P < 1) P = 1;
    p.P = (int32_t)P;
    return p;
}

namespace {

// Largest n the whole-loop kernel (fused_step.cuh) serves, per precision {fp32, fp64}; odisseo_set_fused_max_n sets
// both (0 = never).  Measured on B200, us per KDK step, whole-loop kernel / per-step launches (graph + programmatic
// dependent launch):   fp32  N = 1,024 10.2 / 8.3   2,048 12.5 / 12.6   4,096 23.8 / 20.2   16,384 112.7 / 108.9
//                      fp64  N = 1,024 12.6 / 12.0  2,048 16.3 / 19.8   4,096 31.5 / 36.1   16,384 285 / 261
// Two grid barriers per step (arrive atomic + release flag, ~2.5 us each with the fences around them) cost as much as
// the two launch edges they replace, so the whole-loop form only pays where the per-step kernels are slowest to start:
// fp64 up to 4,096.  fp32 keeps the per-step launches by default.
// Below n ~ 1,280 the per-step launches are faster again in fp64 (10.8 against 12.0 us at N = 1,024), hence a lower bound.
constexpr int64_t FUSED_DEFAULT_MAX_N[2] = {0, 4096}, FUSED_DEFAULT_MIN_N[2] = {0, 1280};
std::atomic<int64_t> g_fused_max_n[2] = {{FUSED_DEFAULT_MAX_N[0]}, {FUSED_DEFAULT_MAX_N[1]}};
std::atomic<int64_t> g_fused_min_n[2] = {{FUSED_DEFAULT_MIN_N[0]}, {FUSED_DEFAULT_MIN_N[1]}};

// Largest n the cluster kernel (cluster_kdk.cuh) serves, per precision {fp32, fp64}: the whole simulation in the shared
// memory of one cluster of 16 CTAs, one hardware cluster barrier per step.  It uses 16 of the 148 SMs, so it wins while a
// step on all SMs is latency-bound; odisseo_set_cluster_max_n changes the bounds (measurements at CLUSTER_DEFAULT_MAX_N).
// Largest n the flag-in-data whole-loop kernel (ll_kdk.cuh) serves, per precision {fp32, fp64}: owner-computes on all SMs,
// the moved positions exchanged as {value, step tag} words through L2 -- one round trip per step.  Tried first.
constexpr int64_t LL_DEFAULT_MAX_N[2] = {4096, 2048};
std::atomic<int64_t> g_ll_max_n[2] = {{LL_DEFAULT_MAX_N[0]}, {LL_DEFAULT_MAX_N[1]}};
constexpr int64_t CLUSTER_DEFAULT_MAX_N[2] = {1024, 512};
std::atomic<int64_t> g_cluster_max_n[2] = {{CLUSTER_DEFAULT_MAX_N[0]}, {CLUSTER_DEFAULT_MAX_N[1]}};

thread_local int g_last_cuda_error = 0;

// ---- instrumentation (include/odisseo.h "Instrumentation") --------------------------------
std::atomic<int64_t> g_launches{0};
struct Profile {
    std::atomic<bool> active{false};     // read without the lock on the launch path
    std::vector<cudaEvent_t> ev;     // pairs (start, stop) around pair-kernel launches
    size_t used = 0;                 // events used so far
    int64_t dropped = 0;             // launches seen after the pool ran out
};
Profile g_prof;
constexpr size_t PROFILE_MAX_LAUNCHES = 4096;

odisseo_status cuda_fail(cudaError_t e)
{
    g_last_cuda_error = (int)e;
    (void)cudaGetLastError();
    return ODISSEO_ERR_CUDA;
}

struct DeviceInfo { int device; int sms; int major; int minor; bool configured; };
std::mutex g_mutex;
std::vector<DeviceInfo> g_devices;

odisseo_status device_info(DeviceInfo& out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    std::lock_guard<std::mutex> lock(g_mutex);
    for (const DeviceInfo& d : g_devices)
        if (d.device == dev) { out = d; return (d.major == 10 && d.minor == 0) ? ODISSEO_OK : ODISSEO_ERR_ARCH; }
    DeviceInfo d{dev, 0, 0, 0, false};
    e = cudaDeviceGetAttribute(&d.major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaDeviceGetAttribute(&d.minor, cudaDevAttrComputeCapabilityMinor, dev);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_fail(e);
    // the library holds sm_100a code only (architecture-specific, no PTX fallback): any other part, 10.x included, is ERR_ARCH
    if (d.major != 10 || d.minor != 0) { g_devices.push_back(d); out = d; return ODISSEO_ERR_ARCH; }
    e = configure_pair_f32(d.sms);
    if (e != cudaSuccess) return cuda_fail(e);
    e = configure_pair_f64(d.sms);
    if (e != cudaSuccess) return cuda_fail(e);
    e = configure_vjp();
    if (e != cudaSuccess) return cuda_fail(e);
    d.configured = true;
    g_devices.push_back(d);
    out = d;
    return ODISSEO_OK;
}

inline bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) != 0; }
inline bool overlap(const void* a, size_t na, const void* b, size_t nb)
{
    const uintptr_t x = reinterpret_cast<uintptr_t>(a), y = reinterpret_cast<uintptr_t>(b);
    return x < y + nb && y < x + na;
}

// eps > 0 (reading R2) and inside the range where the unbranched self term stays finite in the precision of
// the call: the forward kernels form eps^-3 (fp32: eps >= 1e-12; fp64 seeds its rsqrt in fp32 range: eps^2 >= 1e-30), the
// pull-back kernels form 3 eps^-5 (fp32: eps >= 1e-7), so that inf * 0 = NaN cannot arise from an accepted eps.
template <typename T> odisseo_status check_pair_scalars(T G, T eps, bool pullback = false)
{
    if (!isfinite((double)G) || !isfinite((double)eps) || !(eps > (T)0)) return ODISSEO_ERR_ARG;
    const double e = (double)eps;
    if (e * e < 1e-30 || e * e > 1e30) return ODISSEO_ERR_ARG;
    if (sizeof(T) == 4 && e < (pullback ? 1e-7 : 1e-12)) return ODISSEO_ERR_ARG;
    return ODISSEO_OK;
}

template <typename T> odisseo_status make_pot(T G, const odisseo_potential* pot, PotParams<T>& out)
{
    memset(&out, 0, sizeof(out));
    if (!pot) return ODISSEO_OK;
    if (pot->nfw.M_s > 0.0) {
        if (!(pot->nfw.r_s > 0.0) || !isfinite(pot->nfw.M_s) || !isfinite(pot->nfw.r_s)) return ODISSEO_ERR_ARG;
        out.GMs = (T)((double)G * pot->nfw.M_s);
        out.inv_rs = (T)(1.0 / pot->nfw.r_s);
    }
    if (pot->mn.M > 0.0) {
        if (!(pot->mn.b > 0.0) || !(pot->mn.a >= 0.0) || !isfinite(pot->mn.M) || !isfinite(pot->mn.a) ||
            !isfinite(pot->mn.b))
            return ODISSEO_ERR_ARG;
        out.GMd = (T)((double)G * pot->mn.M);
        out.a = (T)pot->mn.a;
        out.b2 = (T)(pot->mn.b * pot->mn.b);
    }
    if (pot->bulge.M_b > 0.0) {
        const odisseo_bulge& b = pot->bulge;
        if (!(b.r_c > 0.0) || !(b.alpha >= 0.0) || !(b.alpha < 2.0) || !isfinite(b.M_b) || !isfinite(b.r_c)) return ODISSEO_ERR_ARG;
        const double s = 0.5 * (3.0 - b.alpha);
        out.GMb = (T)((double)G * b.M_b);
        out.inv_rc = (T)(1.0 / b.r_c);
        out.bs = (T)s;
        out.lgam_s = (T)lgamma(s);
        out.bs_half = (T)(s - 0.5);
        out.lgam_s_half = (T)lgamma(s - 0.5);
        out.phi_outer = (T)(tgamma(s - 0.5) / (b.r_c * tgamma(s)));
    }
    return ODISSEO_OK;
}

// ---- typed launch shims ----------------------------------------------------------------
// j: the workspace's staged array (flags in front of it); the tiles are copied from the targets' own array x when the plan
// says so (plan.direct: no staged copy exists), else from j.
inline cudaError_t launch_pair_raw(const PairPlan& p, const float* x, const void* j, double* part, float eps, cudaStream_t s)
{ return launch_pair_f32(p, x, j, p.direct ? (const void*)x : j, part, eps, s); }
inline cudaError_t launch_pair_raw(const PairPlan& p, const double* x, const void* j, double* part, double eps, cudaStream_t s)
{ return launch_pair_f64(p, x, j, p.direct ? (const void*)x : j, part, eps, s); }
// Pair-kernel launch; while a profile is open (and the stream is not capturing) it is bracketed
// by a pair of CUDA events on the launching stream.
template <typename T>
cudaError_t launch_pair(const PairPlan& p, const T* x, const void* j, double* part, T eps, cudaStream_t s, bool capturing = false)
{
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (!g_prof.active || capturing) return launch_pair_raw(p, x, j, part, eps, s);
    std::lock_guard<std::mutex> lock(g_mutex);
    if (g_prof.used + 2 > g_prof.ev.size()) {
        ++g_prof.dropped;
        return launch_pair_raw(p, x, j, part, eps, s);
    }
    cudaError_t e = cudaEventRecord(g_prof.ev[g_prof.used], s);
    if (e != cudaSuccess) return e;
    e = launch_pair_raw(p, x, j, part, eps, s);
    if (e != cudaSuccess) return e;
    e = cudaEventRecord(g_prof.ev[g_prof.used + 1], s);
    g_prof.used += 2;
    return e;
}
inline cudaError_t launch_step(const PairPlan& p, float* x, float* v, float* a, void* j, const double* part, float G,
                               const PotParams<float>& pot, float dt, int flags, cudaStream_t s, float* snap = nullptr,
                               int64_t lo = 0, int64_t count = -1)
{ g_launches.fetch_add(1, std::memory_order_relaxed); return launch_step_f32(p, x, v, a, j, part, G, pot, dt, flags, snap, lo, count < 0 ? p.n : count, s); }
inline cudaError_t launch_step(const PairPlan& p, double* x, double* v, double* a, void* j, const double* part, double G,
                               const PotParams<double>& pot, double dt, int flags, cudaStream_t s, double* snap = nullptr,
                               int64_t lo = 0, int64_t count = -1)
{ g_launches.fetch_add(1, std::memory_order_relaxed); return launch_step_f64(p, x, v, a, j, part, G, pot, dt, flags, snap, lo, count < 0 ? p.n : count, s); }

inline cudaError_t launch_fused(const PairPlan& p, float* x, float* v, float* a, void* j, double* part, float G, float eps, float dt,
                                const PotParams<float>& pot, int64_t nsteps, int acc_valid, unsigned* bar, cudaStream_t s)
{ return launch_fused_f32(p, x, v, a, j, part, G, eps, dt, pot, nsteps, acc_valid, bar, s); }
inline cudaError_t launch_fused(const PairPlan& p, double* x, double* v, double* a, void* j, double* part, double G, double eps, double dt,
                                const PotParams<double>& pot, int64_t nsteps, int acc_valid, unsigned* bar, cudaStream_t s)
{ return launch_fused_f64(p, x, v, a, j, part, G, eps, dt, pot, nsteps, acc_valid, bar, s); }
inline size_t ll_fits(float, const PairPlan& p) { return ll_fits_f32(p); }
inline size_t ll_fits(double, const PairPlan& p) { return ll_fits_f64(p); }
inline cudaError_t launch_ll(const PairPlan& p, float* x, float* v, float* a, float G, float eps, float dt, const PotParams<float>& pot,
                             int64_t nsteps, int acc_valid, void* xbuf, float* tape, cudaStream_t s)
{ return launch_ll_f32(p, x, v, a, G, eps, dt, pot, nsteps, acc_valid, xbuf, tape, s); }
inline cudaError_t launch_ll(const PairPlan& p, double* x, double* v, double* a, double G, double eps, double dt, const PotParams<double>& pot,
                             int64_t nsteps, int acc_valid, void* xbuf, double* tape, cudaStream_t s)
{ return launch_ll_f64(p, x, v, a, G, eps, dt, pot, nsteps, acc_valid, xbuf, tape, s); }
inline bool cluster_fits(float, const PairPlan& p) { return cluster_fits_f32(p); }
inline bool cluster_fits(double, const PairPlan& p) { return cluster_fits_f64(p); }
inline cudaError_t launch_cluster(const PairPlan& p, float* x, float* v, float* a, float G, float eps, float dt, const PotParams<float>& pot,
                                  int64_t nsteps, int acc_valid, cudaStream_t s)
{ return launch_cluster_f32(p, x, v, a, G, eps, dt, pot, nsteps, acc_valid, s); }
inline cudaError_t launch_cluster(const PairPlan& p, double* x, double* v, double* a, double G, double eps, double dt, const PotParams<double>& pot,
                                  int64_t nsteps, int acc_valid, cudaStream_t s)
{ return launch_cluster_f64(p, x, v, a, G, eps, dt, pot, nsteps, acc_valid, s); }
inline int fused_max_ctas(float, int variant) { return fused_max_ctas_f32(variant); }
inline int fused_max_ctas(double, int variant) { return fused_max_ctas_f64(variant); }

inline cudaError_t launch_ext(const float* x, float* a, int64_t n, const PotParams<float>& pot, int accumulate, cudaStream_t s)
{ g_launches.fetch_add(1, std::memory_order_relaxed); return launch_ext_f32(x, a, n, pot, accumulate, s); }
inline cudaError_t launch_ext(const double* x, double* a, int64_t n, const PotParams<double>& pot, int accumulate, cudaStream_t s)
{ g_launches.fetch_add(1, std::memory_order_relaxed); return launch_ext_f64(x, a, n, pot, accumulate, s); }

struct Carve { void* jsrc; double* partials; };

odisseo_status carve(const PairPlan& plan, void* ws, size_t ws_bytes, Carve& out)
{
    if (!ws) return ODISSEO_ERR_NULL;
    if (misaligned(ws, 256)) return ODISSEO_ERR_ALIGN;
    const size_t need = plan_jsrc_bytes(plan) + plan_partial_bytes(plan);
    if (ws_bytes < need) return ODISSEO_ERR_WORKSPACE;
    out.jsrc = plan_records(ws, plan);
    out.partials = reinterpret_cast<double*>(static_cast<unsigned char*>(ws) + plan_jsrc_bytes(plan));
    return ODISSEO_OK;
}

template <typename T>
odisseo_status pair_accel_impl(const T* posm, T* acc, int64_t n, T G, T eps, void* ws, size_t ws_bytes, void* stream)
{
    if (n < 0) return ODISSEO_ERR_ARG;
    if (n == 0) return ODISSEO_OK;
    if (!posm || !acc) return ODISSEO_ERR_NULL;
    const size_t rec = 4 * sizeof(T);
    if (misaligned(posm, rec) || misaligned(acc, rec)) return ODISSEO_ERR_ALIGN;
    if (overlap(posm, n * rec, acc, n * rec)) return ODISSEO_ERR_ARG;
    odisseo_status st = check_pair_scalars<T>(G, eps);
    if (st != ODISSEO_OK) return st;
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    PairPlan plan = make_plan(n, sizeof(T) == 8, dev.sms);
    plan.direct = 1;                               // the sources are the targets' own records: no staged copy, only the flags
    Carve cv;
    st = carve(plan, ws, ws_bytes, cv);
    if (st != ODISSEO_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    PotParams<T> nopot;
    memset(&nopot, 0, sizeof(nopot));
    cudaError_t e = launch_step(plan, const_cast<T*>(posm), (T*)nullptr, acc, cv.jsrc, cv.partials, G, nopot, (T)0,
                                STEP_PACK_ONLY | STEP_NO_STAGE, s);
    if (e != cudaSuccess) return cuda_fail(e);
    e = launch_pair(plan, posm, cv.jsrc, cv.partials, eps, s);
    if (e != cudaSuccess) return cuda_fail(e);
    e = launch_step(plan, const_cast<T*>(posm), (T*)nullptr, acc, cv.jsrc, cv.partials, G, nopot, (T)0,
                    STEP_FROM_PARTIALS, s);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

inline cudaError_t launch_reduce_rows(const PairPlan& p, const double* part, const void* j, float G, float* a, cudaStream_t s)
{ g_launches.fetch_add(1, std::memory_order_relaxed); return launch_reduce_rows_f32(p, part, j, j, G, a, s); }
inline cudaError_t launch_reduce_rows(const PairPlan& p, const double* part, const void* j, double G, double* a, cudaStream_t s)
{ g_launches.fetch_add(1, std::memory_order_relaxed); return launch_reduce_rows_f64(p, part, j, j, G, a, s); }

// Acceleration at nt target positions due to n sources (targets need not be sources; their masses are ignored).
template <typename T>
odisseo_status pair_cross_impl(const T* targets, int64_t nt, const T* sources, int64_t n, T* acc, T G, T eps, void* ws,
                               size_t ws_bytes, void* stream)
{
    if (n < 0 || nt < 0) return ODISSEO_ERR_ARG;
    if (nt == 0) return ODISSEO_OK;
    if (!targets || !acc || (n > 0 && !sources)) return ODISSEO_ERR_NULL;
    const size_t rec = 4 * sizeof(T);
    if (misaligned(targets, rec) || misaligned(acc, rec) || (n > 0 && misaligned(sources, rec))) return ODISSEO_ERR_ALIGN;
    if (overlap(targets, nt * rec, acc, nt * rec) || (n > 0 && overlap(sources, n * rec, acc, nt * rec))) return ODISSEO_ERR_ARG;
    odisseo_status st = check_pair_scalars<T>(G, eps);
    if (st != ODISSEO_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (n == 0) {
        cudaError_t e0 = cudaMemsetAsync(acc, 0, (size_t)nt * rec, s);
        return e0 == cudaSuccess ? ODISSEO_OK : cuda_fail(e0);
    }
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    const PairPlan plan = make_cross_plan(nt, n, sizeof(T) == 8, dev.sms);
    Carve cv;
    st = carve(plan, ws, ws_bytes, cv);
    if (st != ODISSEO_OK) return st;
    PotParams<T> nopot;
    memset(&nopot, 0, sizeof(nopot));
    cudaError_t e = launch_step(plan, const_cast<T*>(sources), (T*)nullptr, (T*)nullptr, cv.jsrc, cv.partials, G, nopot, (T)0,
                                STEP_PACK_ONLY, s);
    if (e != cudaSuccess) return cuda_fail(e);
    e = launch_pair(plan, targets, cv.jsrc, cv.partials, eps, s);
    if (e != cudaSuccess) return cuda_fail(e);
    e = launch_reduce_rows(plan, cv.partials, cv.jsrc, G, acc, s);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

// ---- sharded form: the three calls of one rank's KDK step on a slice ----------------
// The staged source array in the workspace is kept across calls: stage_sources writes all of it (records, padding,
// equal-mass flags), kick_drift_slice re-stages the records of the slice it moves, the caller's exchange fills in the
// other ranks' records (an in-place all-gather of the record array), pair_accel_staged evaluates targets against it.
template <typename T>
odisseo_status stage_sources_impl(const T* posm, int64_t n, void* ws, size_t ws_bytes, void* stream)
{
    if (n < 0) return ODISSEO_ERR_ARG;
    if (n == 0) return ODISSEO_OK;
    if (!posm || !ws) return ODISSEO_ERR_NULL;
    if (misaligned(posm, 4 * sizeof(T)) || misaligned(ws, 256)) return ODISSEO_ERR_ALIGN;
    DeviceInfo dev;
    odisseo_status st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    const PairPlan plan = make_plan(n, sizeof(T) == 8, dev.sms);
    if (ws_bytes < plan_jsrc_bytes(plan)) return ODISSEO_ERR_WORKSPACE;
    PotParams<T> nopot;
    memset(&nopot, 0, sizeof(nopot));
    cudaError_t e = launch_step(plan, const_cast<T*>(posm), (T*)nullptr, (T*)nullptr, plan_records(ws, plan), nullptr, (T)0, nopot,
                                (T)0, STEP_PACK_ONLY, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? ODISSEO_OK : cuda_fail(e);
}

template <typename T>
odisseo_status pair_staged_impl(const T* targets, int64_t nt, int64_t n, T* acc, T G, T eps, void* ws, size_t ws_bytes,
                                void* stream)
{
    if (n < 0 || nt < 0) return ODISSEO_ERR_ARG;
    if (nt == 0) return ODISSEO_OK;
    if (!targets || !acc || !ws) return ODISSEO_ERR_NULL;
    const size_t rec = 4 * sizeof(T);
    if (misaligned(targets, rec) || misaligned(acc, rec)) return ODISSEO_ERR_ALIGN;
    if (overlap(targets, nt * rec, acc, nt * rec)) return ODISSEO_ERR_ARG;
    odisseo_status st = check_pair_scalars<T>(G, eps);
    if (st != ODISSEO_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (n == 0) {
        cudaError_t e0 = cudaMemsetAsync(acc, 0, (size_t)nt * rec, s);
        return e0 == cudaSuccess ? ODISSEO_OK : cuda_fail(e0);
    }
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    const PairPlan plan = make_cross_plan(nt, n, sizeof(T) == 8, dev.sms);
    Carve cv;
    st = carve(plan, ws, ws_bytes, cv);
    if (st != ODISSEO_OK) return st;
    cudaError_t e = launch_pair(plan, targets, cv.jsrc, cv.partials, eps, s);
    if (e != cudaSuccess) return cuda_fail(e);
    e = launch_reduce_rows(plan, cv.partials, cv.jsrc, G, acc, s);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

template <typename T>
odisseo_status kick_drift_slice_impl(T* posm, T* vel, const T* acc, int64_t n, int64_t lo, int64_t count, T G, T dt,
                                     const odisseo_potential* pot, int mode, void* ws, size_t ws_bytes, void* stream)
{
    if (n < 0 || lo < 0 || count < 0 || lo + count > n || mode < 1 || mode > 3) return ODISSEO_ERR_ARG;
    if (!ws) return ODISSEO_ERR_NULL;
    if (misaligned(ws, 256)) return ODISSEO_ERR_ALIGN;
    if (n == 0) return ODISSEO_OK;
    const size_t rec = 4 * sizeof(T);
    if (count > 0) {
        if (!posm || !vel || !acc) return ODISSEO_ERR_NULL;
        if (misaligned(posm, rec) || misaligned(vel, rec) || misaligned(acc, rec)) return ODISSEO_ERR_ALIGN;
        if (overlap(posm, count * rec, acc, count * rec) || overlap(posm, count * rec, vel, count * rec) ||
            overlap(vel, count * rec, acc, count * rec))
            return ODISSEO_ERR_ARG;
    }
    if (!isfinite((double)G) || !isfinite((double)dt)) return ODISSEO_ERR_ARG;
    PotParams<T> pp;
    odisseo_status st = make_pot<T>(G, pot, pp);
    if (st != ODISSEO_OK) return st;
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    const PairPlan plan = make_plan(n, sizeof(T) == 8, dev.sms);
    if (ws_bytes < plan_jsrc_bytes(plan)) return ODISSEO_ERR_WORKSPACE;
    if (count == 0 && lo != n) return ODISSEO_OK;          // an empty slice that does not own the padding
    const int flags = ((mode & 1) ? STEP_CLOSE : 0) | ((mode & 2) ? STEP_OPEN : 0) | STEP_SLICE;
    cudaError_t e = launch_step(plan, posm, vel, const_cast<T*>(acc), plan_records(ws, plan), nullptr, G, pp, dt, flags,
                                static_cast<cudaStream_t>(stream), nullptr, lo, count);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

template <typename T>
odisseo_status ext_accel_impl(const T* posm, T* acc, int64_t n, T G, const odisseo_potential* pot, int accumulate,
                              void* stream)
{
    if (n < 0) return ODISSEO_ERR_ARG;
    if (n == 0) return ODISSEO_OK;
    if (!posm || !acc) return ODISSEO_ERR_NULL;
    const size_t rec = 4 * sizeof(T);
    if (misaligned(posm, rec) || misaligned(acc, rec)) return ODISSEO_ERR_ALIGN;
    if (overlap(posm, n * rec, acc, n * rec)) return ODISSEO_ERR_ARG;
    if (!isfinite((double)G)) return ODISSEO_ERR_ARG;
    PotParams<T> pp;
    odisseo_status st = make_pot<T>(G, pot, pp);
    if (st != ODISSEO_OK) return st;
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaError_t e = launch_ext(posm, acc, n, pp, accumulate, s);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

// ---- CUDA-graph cache for the per-step launch sequence -----------------------------------
struct GraphKey {
    int is_f64;
    const void *posm, *vel, *acc, *ws;
    int64_t n;
    double G, eps, dt;
    odisseo_potential pot;
    int has_pot;
    int block;   // steps per graph
    int device;
    bool operator==(const GraphKey& o) const { return memcmp(this, &o, sizeof(GraphKey)) == 0; }
};
struct GraphEntry { GraphKey key; cudaGraphExec_t exec; uint64_t stamp; };
std::vector<GraphEntry> g_graphs;
std::mutex g_graph_mutex;
uint64_t g_stamp = 0;
constexpr size_t GRAPH_CACHE = 8;

template <typename T>
odisseo_status leapfrog_impl(T* posm, T* vel, T* acc, int acc_valid, int64_t n, T G, T eps, T dt, int64_t nsteps,
                             const odisseo_potential* pot, void* ws, size_t ws_bytes, void* stream, T* tape = nullptr)
{
    if (n < 0 || nsteps < 0) return ODISSEO_ERR_ARG;
    if (n == 0) return ODISSEO_OK;
    if (!posm || !vel || !acc) return ODISSEO_ERR_NULL;
    const size_t rec = 4 * sizeof(T);
    if (misaligned(posm, rec) || misaligned(vel, rec) || misaligned(acc, rec)) return ODISSEO_ERR_ALIGN;
    if (overlap(posm, n * rec, acc, n * rec) || overlap(posm, n * rec, vel, n * rec) ||
        overlap(vel, n * rec, acc, n * rec))
        return ODISSEO_ERR_ARG;
    odisseo_status st = check_pair_scalars<T>(G, eps);
    if (st != ODISSEO_OK) return st;
    if (!isfinite((double)dt)) return ODISSEO_ERR_ARG;
    PotParams<T> pp;
    st = make_pot<T>(G, pot, pp);
    if (st != ODISSEO_OK) return st;
    if (nsteps == 0 && acc_valid) return ODISSEO_OK;
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    const PairPlan plan = make_plan(n, sizeof(T) == 8, dev.sms);
    Carve cv;
    st = carve(plan, ws, ws_bytes, cv);
    if (st != ODISSEO_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaError_t e;

#define ODISSEO_TRY(call) do { e = (call); if (e != cudaSuccess) return cuda_fail(e); } while (0)
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (s != nullptr) ODISSEO_TRY(cudaStreamIsCapturing(s, &cap));
    // Small N: the whole call on ONE thread-block cluster (cluster_kdk.cuh): state in distributed shared memory, one
    // cluster barrier per step, the canonical summation order -- bit-identical to the sequences below.
    const bool one_launch_ok = nsteps >= 1 && !tape && cap == cudaStreamCaptureStatusNone && !g_prof.active;
    // Small N, first choice: the whole call as ONE cooperative launch of the owner-computes kernel (ll_kdk.cuh): every CTA
    // holds all sources in shared memory and integrates its own few targets; the moved positions travel as {value, step
    // tag} words through the (otherwise unused) partial-row area of the workspace -- one L2 round trip per step.
    // (it also writes the reverse mode's tape: the owner threads store the snapshots)
    if ((one_launch_ok || (tape && nsteps >= 1 && cap == cudaStreamCaptureStatusNone && !g_prof.active)) &&
        n <= g_ll_max_n[sizeof(T) == 8].load(std::memory_order_relaxed) && nsteps < (int64_t)0x7fffffff) {
        const size_t xbytes = ll_fits(T(), plan);
        if (xbytes != 0 && xbytes <= plan_partial_bytes(plan)) {
            if (launch_ll(plan, posm, vel, acc, G, eps, dt, pp, nsteps, acc_valid, cv.partials, tape, s) == cudaSuccess) {
                g_launches.fetch_add(1, std::memory_order_relaxed);
                return ODISSEO_OK;
            }
            (void)cudaGetLastError();          // the device cannot hold the grid right now: the forms below do not need that
        }
    }
    if (one_launch_ok && n <= g_cluster_max_n[sizeof(T) == 8].load(std::memory_order_relaxed) && cluster_fits(T(), plan)) {
        // a device that cannot place the cluster right now (partitioned or shared GPU) takes the sequences below
        if (launch_cluster(plan, posm, vel, acc, G, eps, dt, pp, nsteps, acc_valid, s) == cudaSuccess) {
            g_launches.fetch_add(1, std::memory_order_relaxed);
            return ODISSEO_OK;
        }
        (void)cudaGetLastError();
    }
    // Small and mid N: the whole call in ONE cooperative launch (fused_step.cuh) -- same plan, same code per phase, hence
    // bit-identical to the two-kernel sequence below.  Not inside a caller's capture, with a tape, or while a profile
    // is open (its event pairs bracket pair-kernel launches).
    if (one_launch_ok && n <= g_fused_max_n[sizeof(T) == 8].load(std::memory_order_relaxed) &&
        n >= g_fused_min_n[sizeof(T) == 8].load(std::memory_order_relaxed)) {
        PairPlan fplan = plan;
        const int cap_ctas = fused_max_ctas(T(), plan.variant);
        if (cap_ctas >= 1) {
            if (fplan.P > cap_ctas) fplan.P = cap_ctas;          // P only deals the units out: the sums do not depend on it
            unsigned* bar = plan_barrier_block(cv.jsrc, plan);
            ODISSEO_TRY(cudaMemsetAsync(bar, 0, 256, s));
            g_launches.fetch_add(1, std::memory_order_relaxed);
            ODISSEO_TRY(launch_fused(fplan, posm, vel, acc, cv.jsrc, cv.partials, G, eps, dt, pp, nsteps, acc_valid, bar, s));
            return ODISSEO_OK;
        }
    }
    // tape != nullptr (odisseo_leapfrog_kdk_tape_*): every step kernel also stores the synchronised snapshot
    // {x_k, v_k, pair-only a_k} it holds in registers at the moment between two steps -- no copies, no extra launch
    // The per-step launches keep no staged copy of the sources: the pair kernel's TMA reads the particles' own records
    // (plan.direct), and the step kernel writes posm, vel, acc and the equal-mass flags only (80 bytes per particle in fp32).
    PairPlan dplan = plan;
    dplan.direct = 1;
    const int NS = STEP_NO_STAGE;
    const size_t snap = (size_t)n * 12;
    int first = 0;
    if (!acc_valid) {
        ODISSEO_TRY(launch_step(dplan, posm, vel, acc, cv.jsrc, cv.partials, G, pp, dt, STEP_PACK_ONLY | NS, s));
        ODISSEO_TRY(launch_pair(dplan, (const T*)posm, cv.jsrc, cv.partials, eps, s));
        first = STEP_FROM_PARTIALS;
    }
    if (nsteps == 0) {
        ODISSEO_TRY(launch_step(dplan, posm, vel, acc, cv.jsrc, cv.partials, G, pp, dt, first | (tape ? STEP_SNAPSHOT : 0) | NS, s, tape));
        return ODISSEO_OK;
    }
    ODISSEO_TRY(launch_step(dplan, posm, vel, acc, cv.jsrc, cv.partials, G, pp, dt, first | STEP_OPEN | NS, s, tape));

    int64_t mid = nsteps - 1;     // full steps: pair + (close, open)
    // no graph on the legacy stream, inside a caller's capture, or while a profile is open
    // (event pairs around the pair kernels cannot be read back from graph nodes)
    const bool use_graph = (s != nullptr) && cap == cudaStreamCaptureStatusNone && mid >= 2 && !g_prof.active && !tape;
    if (use_graph) {
        const int block = (int)(mid < 16 ? mid : 16);
        GraphKey key;
        memset(&key, 0, sizeof(key));
        key.is_f64 = sizeof(T) == 8; key.posm = posm; key.vel = vel; key.acc = acc; key.ws = ws; key.n = n;
        key.G = (double)G; key.eps = (double)eps; key.dt = (double)dt; key.has_pot = pot != nullptr;
        if (pot) key.pot = *pot;
        key.block = block; key.device = dev.device;
        // The cache is shared by every host thread: an executable is looked up, created, evicted AND launched under
        // g_graph_mutex, so no thread can destroy an executable another one is about to launch.
        std::lock_guard<std::mutex> graph_lock(g_graph_mutex);
        cudaGraphExec_t exec = nullptr;
        for (GraphEntry& ge : g_graphs)
            if (ge.key == key) { exec = ge.exec; ge.stamp = ++g_stamp; break; }
        if (!exec) {
            cudaGraph_t graph = nullptr;
            ODISSEO_TRY(cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal));
            const int64_t counted = g_launches.load();   // captured launches run at replay, not now
            cudaError_t ce = cudaSuccess;
            for (int k = 0; k < block && ce == cudaSuccess; ++k) {
                ce = launch_pair(dplan, (const T*)posm, cv.jsrc, cv.partials, eps, s, true);
                if (ce == cudaSuccess)
                    ce = launch_step(dplan, posm, vel, acc, cv.jsrc, cv.partials, G, pp, dt,
                                     STEP_FROM_PARTIALS | STEP_CLOSE | STEP_OPEN | NS, s);
            }
            e = cudaStreamEndCapture(s, &graph);
            g_launches.store(counted);
            if (ce != cudaSuccess) { if (graph) cudaGraphDestroy(graph); return cuda_fail(ce); }
            if (e != cudaSuccess) return cuda_fail(e);
            e = cudaGraphInstantiate(&exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) return cuda_fail(e);
            if (g_graphs.size() >= GRAPH_CACHE) {
                size_t victim = 0;
                for (size_t k = 1; k < g_graphs.size(); ++k)
                    if (g_graphs[k].stamp < g_graphs[victim].stamp) victim = k;
                cudaGraphExecDestroy(g_graphs[victim].exec);
                g_graphs.erase(g_graphs.begin() + victim);
            }
            g_graphs.push_back(GraphEntry{key, exec, ++g_stamp});
        }
        while (mid >= block) {
            ODISSEO_TRY(cudaGraphLaunch(exec, s));
            g_launches.fetch_add(2 * block, std::memory_order_relaxed);
            mid -= block;
        }
    }
    for (; mid > 0; --mid) {
        ODISSEO_TRY(launch_pair(dplan, (const T*)posm, cv.jsrc, cv.partials, eps, s));
        ODISSEO_TRY(launch_step(dplan, posm, vel, acc, cv.jsrc, cv.partials, G, pp, dt,
                                STEP_FROM_PARTIALS | STEP_CLOSE | STEP_OPEN | NS, s, tape ? tape + (size_t)(nsteps - mid) * snap : nullptr));
    }
    ODISSEO_TRY(launch_pair(dplan, (const T*)posm, cv.jsrc, cv.partials, eps, s));
    ODISSEO_TRY(launch_step(dplan, posm, vel, acc, cv.jsrc, cv.partials, G, pp, dt, STEP_FROM_PARTIALS | STEP_CLOSE | NS, s,
                            tape ? tape + (size_t)nsteps * snap : nullptr));
    return ODISSEO_OK;
}

template <typename T>
odisseo_status kick_drift_impl(T* posm, T* vel, const T* acc, int64_t n, T G, T dt, const odisseo_potential* pot,
                               int mode, void* ws, size_t ws_bytes, void* stream)
{
    if (n < 0 || mode < 1 || mode > 3) return ODISSEO_ERR_ARG;
    if (n == 0) return ODISSEO_OK;
    if (!posm || !vel || !acc) return ODISSEO_ERR_NULL;
    const size_t rec = 4 * sizeof(T);
    if (misaligned(posm, rec) || misaligned(vel, rec) || misaligned(acc, rec)) return ODISSEO_ERR_ALIGN;
    if (overlap(posm, n * rec, acc, n * rec) || overlap(posm, n * rec, vel, n * rec) ||
        overlap(vel, n * rec, acc, n * rec))
        return ODISSEO_ERR_ARG;
    if (!isfinite((double)G) || !isfinite((double)dt)) return ODISSEO_ERR_ARG;
    PotParams<T> pp;
    odisseo_status st = make_pot<T>(G, pot, pp);
    if (st != ODISSEO_OK) return st;
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    const PairPlan plan = make_plan(n, sizeof(T) == 8, dev.sms);
    Carve cv;
    st = carve(plan, ws, ws_bytes, cv);
    if (st != ODISSEO_OK) return st;
    // no staged copy: odisseo_pair_accel_* reads the particles' own records (the equal-mass flags are still refreshed)
    const int flags = ((mode & 1) ? STEP_CLOSE : 0) | ((mode & 2) ? STEP_OPEN : 0) | STEP_NO_STAGE;
    cudaError_t e = launch_step(plan, posm, vel, const_cast<T*>(acc), cv.jsrc, cv.partials, G, pp, dt, flags,
                                static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

inline cudaError_t launch_diag_stage(const PairPlan& p, const float* x, void* j, cudaStream_t s) { return launch_diag_stage_f32(p, x, j, s); }
inline cudaError_t launch_diag_stage(const PairPlan& p, const double* x, void* j, cudaStream_t s) { return launch_diag_stage_f64(p, x, j, s); }
inline cudaError_t launch_diag_terms(const PairPlan& p, const float* x, const float* v, const double* part, const void* j, double G,
                                     double eps, const PotParams<double>& pot, double* bs, double* phi, cudaStream_t s)
{ return launch_diag_terms_f32(p, x, v, part, j, G, eps, pot, bs, phi, s); }
inline cudaError_t launch_diag_terms(const PairPlan& p, const double* x, const double* v, const double* part, const void* j, double G,
                                     double eps, const PotParams<double>& pot, double* bs, double* phi, cudaStream_t s)
{ return launch_diag_terms_f64(p, x, v, part, j, G, eps, pot, bs, phi, s); }

inline size_t diag_block_sum_bytes(int64_t n)
{ return ((size_t)((n + STEP_THREADS - 1) / STEP_THREADS) * DIAG_VALUES * sizeof(double) + 255) & ~(size_t)255; }

template <typename T>
odisseo_status diagnostics_impl(const T* posm, const T* vel, int64_t n, T G, T eps, const odisseo_potential* pot,
                                double* out, double* phi, void* ws, size_t ws_bytes, void* stream)
{
    if (n < 0) return ODISSEO_ERR_ARG;
    if (!out) return ODISSEO_ERR_NULL;
    if (misaligned(out, 8) || (phi && misaligned(phi, 8))) return ODISSEO_ERR_ALIGN;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaError_t e;
    if (n == 0) {
        e = cudaMemsetAsync(out, 0, DIAG_VALUES * sizeof(double), s);
        return e == cudaSuccess ? ODISSEO_OK : cuda_fail(e);
    }
    if (!posm || !vel) return ODISSEO_ERR_NULL;
    const size_t rec = 4 * sizeof(T);
    if (misaligned(posm, rec) || misaligned(vel, rec)) return ODISSEO_ERR_ALIGN;
    odisseo_status st = check_pair_scalars<T>(G, eps);
    if (st != ODISSEO_OK) return st;
    PotParams<double> pp;
    st = make_pot<double>((double)G, pot, pp);
    if (st != ODISSEO_OK) return st;
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    const PairPlan plan = make_plan(n, 1, dev.sms);        // the O(N^2) pass is always the fp64 kernel
    if (!ws) return ODISSEO_ERR_NULL;
    if (misaligned(ws, 256)) return ODISSEO_ERR_ALIGN;
    const size_t bs_bytes = diag_block_sum_bytes(n);
    if (ws_bytes < bs_bytes) return ODISSEO_ERR_WORKSPACE;
    Carve cv;
    st = carve(plan, static_cast<unsigned char*>(ws) + bs_bytes, ws_bytes - bs_bytes, cv);
    if (st != ODISSEO_OK) return st;
    double* block_sums = static_cast<double*>(ws);
    g_launches.fetch_add(4, std::memory_order_relaxed);
    e = launch_diag_stage(plan, posm, cv.jsrc, s);
    if (e != cudaSuccess) return cuda_fail(e);
    e = launch_potential_f64(plan, cv.jsrc, cv.partials, (double)eps, s);
    if (e != cudaSuccess) return cuda_fail(e);
    e = launch_diag_terms(plan, posm, vel, cv.partials, cv.jsrc, (double)G, (double)eps, pp, block_sums, phi, s);
    if (e != cudaSuccess) return cuda_fail(e);
    e = launch_diag_final(block_sums, (int)((n + STEP_THREADS - 1) / STEP_THREADS), out, s);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

inline cudaError_t launch_accel_vjp(const PairPlan& p, const float* x, const float* c, double G, double eps, const PotParams<double>& pot,
                                    float* gx, double* gm, double* gp, int eg, void* ws, cudaStream_t s)
{ return launch_accel_vjp_f32(p, x, c, G, eps, pot, gx, gm, gp, eg, ws, s); }
inline cudaError_t launch_accel_vjp(const PairPlan& p, const double* x, const double* c, double G, double eps, const PotParams<double>& pot,
                                    double* gx, double* gm, double* gp, int eg, void* ws, cudaStream_t s)
{ return launch_accel_vjp_f64(p, x, c, G, eps, pot, gx, gm, gp, eg, ws, s); }
inline cudaError_t launch_leapfrog_vjp(const PairPlan& p, const float* tape, int64_t nsteps, double G, double eps, float dt,
                                       const PotParams<double>& pd, const PotParams<float>& pt, int eg, float* lx, float* lv, double* gm,
                                       double* gp, void* ws, int64_t* nl, cudaStream_t s)
{ return launch_leapfrog_vjp_f32(p, tape, nsteps, G, eps, dt, pd, pt, eg, lx, lv, gm, gp, ws, nl, s); }
inline cudaError_t launch_leapfrog_vjp(const PairPlan& p, const double* tape, int64_t nsteps, double G, double eps, double dt,
                                       const PotParams<double>& pd, const PotParams<double>& pt, int eg, double* lx, double* lv, double* gm,
                                       double* gp, void* ws, int64_t* nl, cudaStream_t s)
{ return launch_leapfrog_vjp_f64(p, tape, nsteps, G, eps, dt, pd, pt, eg, lx, lv, gm, gp, ws, nl, s); }

template <typename T>
odisseo_status accel_vjp_impl(const T* posm, const T* cot, int64_t n, T G, T eps, const odisseo_potential* pot, int with_eps_G,
                              T* gx, double* gm, double* gparams, void* ws, size_t ws_bytes, void* stream)
{
    if (n < 0) return ODISSEO_ERR_ARG;
    if (!gparams) return ODISSEO_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (n == 0) {
        cudaError_t e0 = cudaMemsetAsync(gparams, 0, VJP_NOUT * sizeof(double), s);
        return e0 == cudaSuccess ? ODISSEO_OK : cuda_fail(e0);
    }
    if (!posm || !cot || !gx || !gm || !ws) return ODISSEO_ERR_NULL;
    const size_t rec = 4 * sizeof(T);
    if (misaligned(posm, rec) || misaligned(cot, rec) || misaligned(gx, rec) || misaligned(gm, 8) || misaligned(gparams, 8) ||
        misaligned(ws, 256))
        return ODISSEO_ERR_ALIGN;
    if (overlap(posm, n * rec, gx, n * rec) || overlap(cot, n * rec, gx, n * rec)) return ODISSEO_ERR_ARG;
    odisseo_status st = check_pair_scalars<T>(G, eps, true);
    if (st != ODISSEO_OK) return st;
    PotParams<double> pp;
    st = make_pot<double>((double)G, pot, pp);
    if (st != ODISSEO_OK) return st;
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    const PairPlan plan = make_vjp_plan(n, sizeof(T) == 8, dev.sms);
    if (ws_bytes < vjp_workspace_bytes(plan, sizeof(T) == 8)) return ODISSEO_ERR_WORKSPACE;
    g_launches.fetch_add(4, std::memory_order_relaxed);
    cudaError_t e = launch_accel_vjp(plan, posm, cot, (double)G, (double)eps, pp, gx, gm, gparams, with_eps_G != 0, ws, s);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

template <typename T>
odisseo_status leapfrog_tape_impl(T* posm, T* vel, T* acc, int64_t n, T G, T eps, T dt, int64_t nsteps,
                                  const odisseo_potential* pot, T* tape, size_t tape_bytes, void* ws, size_t ws_bytes,
                                  void* stream)
{
    if (n < 0 || nsteps < 0) return ODISSEO_ERR_ARG;
    if (n == 0) return ODISSEO_OK;
    if (!tape) return ODISSEO_ERR_NULL;
    const size_t arr = (size_t)n * 4 * sizeof(T);
    if (misaligned(tape, 4 * sizeof(T))) return ODISSEO_ERR_ALIGN;
    if (tape_bytes < (size_t)(nsteps + 1) * 3 * arr) return ODISSEO_ERR_WORKSPACE;
    return leapfrog_impl<T>(posm, vel, acc, 0, n, G, eps, dt, nsteps, pot, ws, ws_bytes, stream, tape);
}

template <typename T>
odisseo_status leapfrog_vjp_impl(const T* tape, int64_t n, T G, T eps, T dt, int64_t nsteps, const odisseo_potential* pot,
                                 int with_eps_G, T* lx, T* lv, double* gm, double* gparams, void* ws, size_t ws_bytes, void* stream)
{
    if (n < 0 || nsteps < 0) return ODISSEO_ERR_ARG;
    if (!gparams) return ODISSEO_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaError_t e = cudaMemsetAsync(gparams, 0, VJP_NOUT * sizeof(double), s);
    if (e != cudaSuccess) return cuda_fail(e);
    if (n == 0) return ODISSEO_OK;
    if (!tape || !lx || !lv || !gm || !ws) return ODISSEO_ERR_NULL;
    const size_t rec = 4 * sizeof(T);
    if (misaligned(tape, rec) || misaligned(lx, rec) || misaligned(lv, rec) || misaligned(gm, 8) || misaligned(gparams, 8) ||
        misaligned(ws, 256))
        return ODISSEO_ERR_ALIGN;
    if (overlap(lx, n * rec, lv, n * rec)) return ODISSEO_ERR_ARG;
    odisseo_status st = check_pair_scalars<T>(G, eps, true);
    if (st != ODISSEO_OK) return st;
    if (!isfinite((double)dt)) return ODISSEO_ERR_ARG;
    PotParams<double> pd;
    st = make_pot<double>((double)G, pot, pd);
    if (st != ODISSEO_OK) return st;
    PotParams<T> pt;
    st = make_pot<T>(G, pot, pt);
    if (st != ODISSEO_OK) return st;
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    const PairPlan plan = make_vjp_plan(n, sizeof(T) == 8, dev.sms);
    if (ws_bytes < vjp_workspace_bytes(plan, sizeof(T) == 8)) return ODISSEO_ERR_WORKSPACE;
    e = cudaMemsetAsync(gm, 0, (size_t)n * sizeof(double), s);
    if (e != cudaSuccess) return cuda_fail(e);
    if (nsteps == 0) return ODISSEO_OK;                    // the final state is the initial state
    int64_t launches = 0;
    e = launch_leapfrog_vjp(plan, tape, nsteps, (double)G, (double)eps, dt, pd, pt, with_eps_G != 0, lx, lv, gm, gparams, ws, &launches, s);
    g_launches.fetch_add(launches, std::memory_order_relaxed);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

template <typename T>
odisseo_status leapfrog_host_impl(T* h_posm, T* h_vel, T* h_acc, int acc_valid, int64_t n, T G, T eps, T dt, int64_t nsteps,
                                  const odisseo_potential* pot, void* ws, size_t ws_bytes, void* stream)
{
    if (n < 0 || nsteps < 0) return ODISSEO_ERR_ARG;
    if (n == 0) return ODISSEO_OK;
    if (!h_posm || !h_vel || !ws || (acc_valid && !h_acc)) return ODISSEO_ERR_NULL;
    if (misaligned(ws, 256)) return ODISSEO_ERR_ALIGN;
    const size_t arr = ((size_t)n * 4 * sizeof(T) + 255) & ~(size_t)255;
    if (ws_bytes < 3 * arr) return ODISSEO_ERR_WORKSPACE;
    unsigned char* base = static_cast<unsigned char*>(ws);
    T* d_posm = reinterpret_cast<T*>(base);
    T* d_vel = reinterpret_cast<T*>(base + arr);
    T* d_acc = reinterpret_cast<T*>(base + 2 * arr);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaError_t e;
    ODISSEO_TRY(cudaMemcpyAsync(d_posm, h_posm, (size_t)n * 4 * sizeof(T), cudaMemcpyHostToDevice, s));
    ODISSEO_TRY(cudaMemcpyAsync(d_vel, h_vel, (size_t)n * 4 * sizeof(T), cudaMemcpyHostToDevice, s));
    if (acc_valid) ODISSEO_TRY(cudaMemcpyAsync(d_acc, h_acc, (size_t)n * 4 * sizeof(T), cudaMemcpyHostToDevice, s));
    odisseo_status st = leapfrog_impl<T>(d_posm, d_vel, d_acc, acc_valid, n, G, eps, dt, nsteps, pot, base + 3 * arr,
                                         ws_bytes - 3 * arr, stream);
    if (st != ODISSEO_OK) return st;
    ODISSEO_TRY(cudaMemcpyAsync(h_posm, d_posm, (size_t)n * 4 * sizeof(T), cudaMemcpyDeviceToHost, s));
    ODISSEO_TRY(cudaMemcpyAsync(h_vel, d_vel, (size_t)n * 4 * sizeof(T), cudaMemcpyDeviceToHost, s));
    if (h_acc) ODISSEO_TRY(cudaMemcpyAsync(h_acc, d_acc, (size_t)n * 4 * sizeof(T), cudaMemcpyDeviceToHost, s));
    return ODISSEO_OK;
}
#undef ODISSEO_TRY

}  // namespace
}  // namespace odisseo

using namespace odisseo;

extern "C" {

const char* odisseo_version(void) { return "odisseo-b200 0.1 (sm_100a)"; }

const char* odisseo_status_string(odisseo_status s)
{
    switch (s) {
        case ODISSEO_OK: return "ok";
        case ODISSEO_ERR_NULL: return "null pointer";
        case ODISSEO_ERR_ALIGN: return "misaligned pointer";
        case ODISSEO_ERR_ARG: return "invalid argument";
        case ODISSEO_ERR_WORKSPACE: return "workspace too small";
        case ODISSEO_ERR_ARCH: return "device is not compute capability 10.0 (B200, sm_100a)";
        case ODISSEO_ERR_CUDA: return "CUDA error (see odisseo_last_cuda_error)";
        case ODISSEO_ERR_STATIC_LIMIT:
            return "problem too large for the library's built-in scratch array (odisseo_mmd2_static_scratch_bytes); "
                   "use the call that takes a workspace";
    }
    return "unknown status";
}

int odisseo_last_cuda_error(void) { return g_last_cuda_error; }

int64_t odisseo_launch_count(void) { return g_launches.load(); }

const char* odisseo_pair_kernel_name(int64_t n, int is_f64)
{
    if (n <= 0) return "";
    const int variant = make_cross_plan(n, n, is_f64 != 0, 148).variant;       // the variant is a function of n alone
    return is_f64 ? pair_kernel_name_f64(variant) : pair_kernel_name_f32(variant);
}

int64_t odisseo_set_fused_max_n(int64_t n)
{
    if (n > 16384) n = 16384;
    for (int k = 0; k < 2; ++k) g_fused_min_n[k].store(n < 0 ? FUSED_DEFAULT_MIN_N[k] : 0);
    g_fused_max_n[0].store(n < 0 ? FUSED_DEFAULT_MAX_N[0] : n);
    return g_fused_max_n[1].exchange(n < 0 ? FUSED_DEFAULT_MAX_N[1] : n);
}

int64_t odisseo_set_ll_max_n(int64_t n)
{
    if (n > LL_MAX_N) n = LL_MAX_N;
    g_ll_max_n[1].store(n < 0 ? LL_DEFAULT_MAX_N[1] : n);
    return g_ll_max_n[0].exchange(n < 0 ? LL_DEFAULT_MAX_N[0] : n);
}

int64_t odisseo_set_cluster_max_n(int64_t n)
{
    if (n > CLUSTER_MAX_N) n = CLUSTER_MAX_N;
    g_cluster_max_n[1].store(n < 0 ? CLUSTER_DEFAULT_MAX_N[1] : n);
    return g_cluster_max_n[0].exchange(n < 0 ? CLUSTER_DEFAULT_MAX_N[0] : n);
}

odisseo_status odisseo_shutdown(void)
{
    {
        std::lock_guard<std::mutex> graph_lock(g_graph_mutex);
        for (GraphEntry& ge : g_graphs) cudaGraphExecDestroy(ge.exec);
        g_graphs.clear();
    }
    std::lock_guard<std::mutex> lock(g_mutex);
    if (g_prof.active.load()) return ODISSEO_ERR_ARG;     // a profile is open: close it first
    for (cudaEvent_t ev : g_prof.ev) cudaEventDestroy(ev);
    g_prof.ev.clear();
    g_prof.used = 0;
    (void)cudaGetLastError();
    return ODISSEO_OK;
}

odisseo_status odisseo_profile_begin(void)
{
    DeviceInfo dev;
    odisseo_status st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    std::lock_guard<std::mutex> lock(g_mutex);
    while (g_prof.ev.size() < 2 * PROFILE_MAX_LAUNCHES) {
        cudaEvent_t ev;
        cudaError_t e = cudaEventCreate(&ev);
        if (e != cudaSuccess) return cuda_fail(e);
        g_prof.ev.push_back(ev);
    }
    g_prof.used = 0;
    g_prof.dropped = 0;
    g_prof.active = true;
    return ODISSEO_OK;
}

odisseo_status odisseo_profile_end(double* h_ms_total, int64_t* h_launches, int64_t* h_dropped)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_prof.active) return ODISSEO_ERR_ARG;
    g_prof.active = false;
    double total = 0.0;
    for (size_t k = 0; k + 1 < g_prof.used; k += 2) {
        cudaError_t e = cudaEventSynchronize(g_prof.ev[k + 1]);
        if (e != cudaSuccess) return cuda_fail(e);
        float ms = 0.f;
        e = cudaEventElapsedTime(&ms, g_prof.ev[k], g_prof.ev[k + 1]);
        if (e != cudaSuccess) return cuda_fail(e);
        total += (double)ms;
    }
    if (h_ms_total) *h_ms_total = total;
    if (h_launches) *h_launches = (int64_t)(g_prof.used / 2);
    if (h_dropped) *h_dropped = g_prof.dropped;
    return ODISSEO_OK;
}

odisseo_status odisseo_profile_times(double* h_ms, int64_t capacity, int64_t* h_count)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    if (g_prof.active) return ODISSEO_ERR_ARG;            // read the durations after odisseo_profile_end
    if (capacity < 0 || (capacity > 0 && !h_ms)) return ODISSEO_ERR_ARG;
    const int64_t n = (int64_t)(g_prof.used / 2);
    if (h_count) *h_count = n;
    for (int64_t k = 0; k < n && k < capacity; ++k) {
        float ms = 0.f;
        cudaError_t e = cudaEventElapsedTime(&ms, g_prof.ev[2 * k], g_prof.ev[2 * k + 1]);
        if (e != cudaSuccess) return cuda_fail(e);
        h_ms[k] = (double)ms;
    }
    return ODISSEO_OK;
}

size_t odisseo_workspace_bytes(int64_t n, int is_f64) { return odisseo_cross_workspace_bytes(n, n, is_f64); }

size_t odisseo_cross_workspace_bytes(int64_t nt, int64_t n, int is_f64)
{
    if (n <= 0 || nt <= 0) return 0;
    size_t best = 0;
    int lo = 64, hi = 192;                                // bound over devices with 64 to 192 SMs ...
    {
        int dev = -1, sms = 0;                            // ... or exactly the current device when there is one
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
            sms > 0)
            lo = hi = sms;
        else
            (void)cudaGetLastError();
    }
    for (int sms = lo; sms <= hi; ++sms) {
        const PairPlan p = make_cross_plan(nt, n, is_f64, sms);
        const size_t b = plan_jsrc_bytes(p) + plan_partial_bytes(p);
        if (b > best) best = b;
    }
    return best;
}

odisseo_status odisseo_pair_accel_cross_f32(const float* d_targets, int64_t nt, const float* d_sources, int64_t n,
                                            float* d_acc, float G, float eps, void* d_workspace, size_t workspace_bytes,
                                            void* stream)
{ return pair_cross_impl<float>(d_targets, nt, d_sources, n, d_acc, G, eps, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_pair_accel_cross_f64(const double* d_targets, int64_t nt, const double* d_sources, int64_t n,
                                            double* d_acc, double G, double eps, void* d_workspace, size_t workspace_bytes,
                                            void* stream)
{ return pair_cross_impl<double>(d_targets, nt, d_sources, n, d_acc, G, eps, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_describe_cross_plan_for(int64_t nt, int64_t n, int is_f64, int num_sms, int64_t out[8])
{
    if (!out) return ODISSEO_ERR_NULL;
    if (n <= 0 || nt <= 0 || num_sms <= 0) return ODISSEO_ERR_ARG;
    const PairPlan p = make_cross_plan(nt, n, is_f64, num_sms);
    out[0] = p.ipt; out[1] = p.cthreads + 32; out[2] = p.T; out[3] = p.P;
    out[4] = p.nb; out[5] = p.S; out[6] = p.U; out[7] = 2;
    return ODISSEO_OK;
}

odisseo_status odisseo_describe_plan_for(int64_t n, int is_f64, int num_sms, int64_t out[8])
{ return odisseo_describe_cross_plan_for(n, n, is_f64, num_sms, out); }

odisseo_status odisseo_describe_plan(int64_t n, int is_f64, int64_t out[8])
{
    if (!out) return ODISSEO_ERR_NULL;
    DeviceInfo dev;
    odisseo_status st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    return odisseo_describe_plan_for(n, is_f64, dev.sms, out);
}

// Host-side check of the unit bookkeeping for tests: for unit u the owning CTA and the source records of its
// chunk, and for CTA c its [start, end) unit range, exactly as the kernels compute them.
odisseo_status odisseo_plan_probe(int64_t nt, int64_t n, int is_f64, int num_sms, int64_t u, int64_t c, int64_t out[5])
{
    if (!out) return ODISSEO_ERR_NULL;
    if (n <= 0 || nt <= 0 || num_sms <= 0) return ODISSEO_ERR_ARG;
    const PairPlan p = make_cross_plan(nt, n, is_f64, num_sms);
    if (u < 0 || u >= p.U || c < 0 || c >= p.P) return ODISSEO_ERR_ARG;
    out[0] = plan_owner(p, u);
    out[1] = plan_start(p, c);
    out[2] = plan_start(p, c + 1);
    out[3] = plan_chunk_lo(p, u % p.S);
    out[4] = plan_chunk_lo(p, u % p.S + 1);
    return ODISSEO_OK;
}

odisseo_status odisseo_pair_accel_f32(const float* d_posm, float* d_acc, int64_t n, float G, float eps,
                                      void* d_workspace, size_t workspace_bytes, void* stream)
{ return pair_accel_impl<float>(d_posm, d_acc, n, G, eps, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_pair_accel_f64(const double* d_posm, double* d_acc, int64_t n, double G, double eps,
                                      void* d_workspace, size_t workspace_bytes, void* stream)
{ return pair_accel_impl<double>(d_posm, d_acc, n, G, eps, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_pair_accel_soa_f32(const float* d_x, const float* d_y, const float* d_z, const float* d_m,
                                          float* d_ax, float* d_ay, float* d_az, int64_t n, float G, float eps,
                                          void* d_workspace, size_t workspace_bytes, void* stream)
{
    if (n < 0) return ODISSEO_ERR_ARG;
    if (n == 0) return ODISSEO_OK;
    if (!d_x || !d_y || !d_z || !d_m || !d_ax || !d_ay || !d_az || !d_workspace) return ODISSEO_ERR_NULL;
    if (misaligned(d_x, 4) || misaligned(d_y, 4) || misaligned(d_z, 4) || misaligned(d_m, 4) || misaligned(d_ax, 4) ||
        misaligned(d_ay, 4) || misaligned(d_az, 4))
        return ODISSEO_ERR_ALIGN;
    if (misaligned(d_workspace, 256)) return ODISSEO_ERR_ALIGN;
    const size_t arr = ((size_t)n * 16 + 255) & ~(size_t)255;
    if (workspace_bytes < 2 * arr) return ODISSEO_ERR_WORKSPACE;
    odisseo_status st = check_pair_scalars<float>(G, eps);
    if (st != ODISSEO_OK) return st;
    DeviceInfo dev;
    st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    unsigned char* base = static_cast<unsigned char*>(d_workspace);
    float* posm = reinterpret_cast<float*>(base);
    float* acc = reinterpret_cast<float*>(base + arr);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    g_launches.fetch_add(2, std::memory_order_relaxed);
    cudaError_t e = launch_soa_pack_f32(d_x, d_y, d_z, d_m, posm, n, s);
    if (e != cudaSuccess) return cuda_fail(e);
    st = pair_accel_impl<float>(posm, acc, n, G, eps, base + 2 * arr, workspace_bytes - 2 * arr, stream);
    if (st != ODISSEO_OK) return st;
    e = launch_soa_unpack_f32(acc, d_ax, d_ay, d_az, n, s);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

odisseo_status odisseo_ext_accel_f32(const float* d_posm, float* d_acc, int64_t n, float G,
                                     const odisseo_potential* pot, int accumulate, void* stream)
{ return ext_accel_impl<float>(d_posm, d_acc, n, G, pot, accumulate, stream); }

odisseo_status odisseo_ext_accel_f64(const double* d_posm, double* d_acc, int64_t n, double G,
                                     const odisseo_potential* pot, int accumulate, void* stream)
{ return ext_accel_impl<double>(d_posm, d_acc, n, G, pot, accumulate, stream); }

odisseo_status odisseo_leapfrog_kdk_f32(float* d_posm, float* d_vel, float* d_acc, int acc_valid, int64_t n, float G,
                                        float eps, float dt, int64_t nsteps, const odisseo_potential* pot,
                                        void* d_workspace, size_t workspace_bytes, void* stream)
{ return leapfrog_impl<float>(d_posm, d_vel, d_acc, acc_valid, n, G, eps, dt, nsteps, pot, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_leapfrog_kdk_f64(double* d_posm, double* d_vel, double* d_acc, int acc_valid, int64_t n,
                                        double G, double eps, double dt, int64_t nsteps, const odisseo_potential* pot,
                                        void* d_workspace, size_t workspace_bytes, void* stream)
{ return leapfrog_impl<double>(d_posm, d_vel, d_acc, acc_valid, n, G, eps, dt, nsteps, pot, d_workspace, workspace_bytes, stream); }

size_t odisseo_vjp_workspace_bytes(int64_t n, int is_f64)
{
    if (n <= 0) return 0;
    int lo = 64, hi = 192;                                // as odisseo_workspace_bytes: the current device, else a bound
    {
        int dev = -1, sms = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
            sms > 0)
            lo = hi = sms;
        else
            (void)cudaGetLastError();
    }
    size_t b = 0;
    for (int sms = lo; sms <= hi; ++sms) {
        const size_t c = vjp_workspace_bytes(make_vjp_plan(n, is_f64, sms), is_f64);
        if (c > b) b = c;
    }
    return b;
}

size_t odisseo_tape_bytes(int64_t n, int64_t nsteps, int is_f64)
{
    if (n <= 0 || nsteps < 0) return 0;
    return (size_t)(nsteps + 1) * 3 * (size_t)n * 4 * (is_f64 ? 8 : 4);
}

odisseo_status odisseo_accel_vjp_f32(const float* d_posm, const float* d_cot, int64_t n, float G, float eps,
                                     const odisseo_potential* pot, int with_eps_G, float* d_gx, double* d_gm, double* d_gparams,
                                     void* d_workspace, size_t workspace_bytes, void* stream)
{ return accel_vjp_impl<float>(d_posm, d_cot, n, G, eps, pot, with_eps_G, d_gx, d_gm, d_gparams, d_workspace, workspace_bytes, stream); }
odisseo_status odisseo_accel_vjp_f64(const double* d_posm, const double* d_cot, int64_t n, double G, double eps,
                                     const odisseo_potential* pot, int with_eps_G, double* d_gx, double* d_gm, double* d_gparams,
                                     void* d_workspace, size_t workspace_bytes, void* stream)
{ return accel_vjp_impl<double>(d_posm, d_cot, n, G, eps, pot, with_eps_G, d_gx, d_gm, d_gparams, d_workspace, workspace_bytes, stream); }
odisseo_status odisseo_leapfrog_kdk_tape_f32(float* d_posm, float* d_vel, float* d_acc, int64_t n, float G, float eps, float dt,
                                             int64_t nsteps, const odisseo_potential* pot, float* d_tape, size_t tape_bytes,
                                             void* d_workspace, size_t workspace_bytes, void* stream)
{ return leapfrog_tape_impl<float>(d_posm, d_vel, d_acc, n, G, eps, dt, nsteps, pot, d_tape, tape_bytes, d_workspace, workspace_bytes, stream); }
odisseo_status odisseo_leapfrog_kdk_tape_f64(double* d_posm, double* d_vel, double* d_acc, int64_t n, double G, double eps, double dt,
                                             int64_t nsteps, const odisseo_potential* pot, double* d_tape, size_t tape_bytes,
                                             void* d_workspace, size_t workspace_bytes, void* stream)
{ return leapfrog_tape_impl<double>(d_posm, d_vel, d_acc, n, G, eps, dt, nsteps, pot, d_tape, tape_bytes, d_workspace, workspace_bytes, stream); }
odisseo_status odisseo_leapfrog_kdk_vjp_f32(const float* d_tape, int64_t n, float G, float eps, float dt, int64_t nsteps,
                                            const odisseo_potential* pot, int with_eps_G, float* d_lx, float* d_lv, double* d_gm,
                                            double* d_gparams, void* d_workspace, size_t workspace_bytes, void* stream)
{ return leapfrog_vjp_impl<float>(d_tape, n, G, eps, dt, nsteps, pot, with_eps_G, d_lx, d_lv, d_gm, d_gparams, d_workspace, workspace_bytes, stream); }
odisseo_status odisseo_leapfrog_kdk_vjp_f64(const double* d_tape, int64_t n, double G, double eps, double dt, int64_t nsteps,
                                            const odisseo_potential* pot, int with_eps_G, double* d_lx, double* d_lv, double* d_gm,
                                            double* d_gparams, void* d_workspace, size_t workspace_bytes, void* stream)
{ return leapfrog_vjp_impl<double>(d_tape, n, G, eps, dt, nsteps, pot, with_eps_G, d_lx, d_lv, d_gm, d_gparams, d_workspace, workspace_bytes, stream); }

size_t odisseo_diagnostics_workspace_bytes(int64_t n)
{
    if (n <= 0) return 0;
    return diag_block_sum_bytes(n) + odisseo_workspace_bytes(n, 1);
}

odisseo_status odisseo_diagnostics_f32(const float* d_posm, const float* d_vel, int64_t n, float G, float eps,
                                       const odisseo_potential* pot, double* d_out, double* d_phi, void* d_workspace,
                                       size_t workspace_bytes, void* stream)
{ return diagnostics_impl<float>(d_posm, d_vel, n, G, eps, pot, d_out, d_phi, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_diagnostics_f64(const double* d_posm, const double* d_vel, int64_t n, double G, double eps,
                                       const odisseo_potential* pot, double* d_out, double* d_phi, void* d_workspace,
                                       size_t workspace_bytes, void* stream)
{ return diagnostics_impl<double>(d_posm, d_vel, n, G, eps, pot, d_out, d_phi, d_workspace, workspace_bytes, stream); }

size_t odisseo_ensemble_workspace_bytes(int64_t nsim)
{
    if (nsim <= 0) return 0;
    return (((size_t)nsim * (sizeof(EnsembleParams) + sizeof(EnsembleParams64))) + 511) & ~(size_t)255;
}

size_t odisseo_ensemble_tape_bytes(int64_t n, int64_t nsim, int64_t nsteps)
{
    if (n <= 0 || nsim <= 0 || nsteps < 0) return 0;
    return (size_t)nsim * (size_t)(nsteps + 1) * 3 * (size_t)n * 16;
}

namespace {

// Validates the host records and uploads them: float records at ws, double records behind them.
odisseo_status ensemble_upload_params(const odisseo_sim_params* h_params, int64_t nparams, void* ws, size_t ws_bytes,
                                      cudaStream_t s, const EnsembleParams** d32, const EnsembleParams64** d64,
                                      bool pullback = false)
{
    const size_t off64 = (((size_t)nparams * sizeof(EnsembleParams)) + 255) & ~(size_t)255;
    if (ws_bytes < off64 + (size_t)nparams * sizeof(EnsembleParams64)) return ODISSEO_ERR_WORKSPACE;
    std::vector<EnsembleParams> p32((size_t)nparams);
    std::vector<EnsembleParams64> p64((size_t)nparams);
    for (int64_t k = 0; k < nparams; ++k) {
        const odisseo_sim_params& hp = h_params[k];
        const float G = (float)hp.G, eps = (float)hp.eps, dt = (float)hp.dt;
        odisseo_status st = check_pair_scalars<float>(G, eps, pullback);
        if (st != ODISSEO_OK) return st;
        if (!isfinite((double)dt)) return ODISSEO_ERR_ARG;
        EnsembleParams& d = p32[(size_t)k];
        st = make_pot<float>(G, &hp.pot, d.pot);
        if (st != ODISSEO_OK) return st;
        d.G = G; d.eps2 = eps * eps; d.dt = dt;
        EnsembleParams64& q = p64[(size_t)k];            // the fp32-rounded scalars, as the forward kernel used them
        st = make_pot<double>((double)G, &hp.pot, q.pot);
        if (st != ODISSEO_OK) return st;
        q.G = (double)G; q.eps = (double)eps; q.dt = (double)dt;
    }
    unsigned char* base = static_cast<unsigned char*>(ws);
    // pageable sources: the runtime stages them before returning, so the vectors may die with this frame
    cudaError_t e = cudaMemcpyAsync(base, p32.data(), (size_t)nparams * sizeof(EnsembleParams), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(base + off64, p64.data(), (size_t)nparams * sizeof(EnsembleParams64), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(e);
    *d32 = reinterpret_cast<const EnsembleParams*>(base);
    *d64 = reinterpret_cast<const EnsembleParams64*>(base + off64);
    return ODISSEO_OK;
}

odisseo_status ensemble_forward(float* d_posm, float* d_vel, int64_t n, int64_t nsim, const odisseo_sim_params* h_params,
                                int64_t nparams, int64_t nsteps, float* d_tape, size_t tape_bytes, bool want_tape,
                                void* d_workspace, size_t workspace_bytes, void* stream)
{
    if (n < 0 || nsim < 0 || nsteps < 0 || n > ENSEMBLE_MAX_N || nsim > 0x7fffffff) return ODISSEO_ERR_ARG;
    if (n == 0 || nsim == 0) return ODISSEO_OK;
    if (!d_posm || !d_vel || !h_params || !d_workspace || (want_tape && !d_tape)) return ODISSEO_ERR_NULL;
    if (misaligned(d_posm, 16) || misaligned(d_vel, 16) || misaligned(d_workspace, 256) || (want_tape && misaligned(d_tape, 16)))
        return ODISSEO_ERR_ALIGN;
    const size_t bytes = (size_t)nsim * n * 16;
    if (overlap(d_posm, bytes, d_vel, bytes)) return ODISSEO_ERR_ARG;
    if (nparams != 1 && nparams != nsim) return ODISSEO_ERR_ARG;
    if (want_tape && tape_bytes < odisseo_ensemble_tape_bytes(n, nsim, nsteps)) return ODISSEO_ERR_WORKSPACE;
    DeviceInfo dev;
    odisseo_status st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const EnsembleParams* d32;
    const EnsembleParams64* d64;
    st = ensemble_upload_params(h_params, nparams, d_workspace, workspace_bytes, s, &d32, &d64);
    if (st != ODISSEO_OK) return st;
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = launch_ensemble_f32(d_posm, d_vel, d32, nparams == 1 ? 1 : 0, (int)n, nsim, nsteps,
                                        want_tape ? d_tape : nullptr, s);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

}  // namespace

odisseo_status odisseo_ensemble_leapfrog_kdk_f32(float* d_posm, float* d_vel, int64_t n, int64_t nsim,
                                                 const odisseo_sim_params* h_params, int64_t nparams, int64_t nsteps,
                                                 void* d_workspace, size_t workspace_bytes, void* stream)
{ return ensemble_forward(d_posm, d_vel, n, nsim, h_params, nparams, nsteps, nullptr, 0, false, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_ensemble_leapfrog_kdk_tape_f32(float* d_posm, float* d_vel, int64_t n, int64_t nsim,
                                                      const odisseo_sim_params* h_params, int64_t nparams, int64_t nsteps,
                                                      float* d_tape, size_t tape_bytes, void* d_workspace,
                                                      size_t workspace_bytes, void* stream)
{ return ensemble_forward(d_posm, d_vel, n, nsim, h_params, nparams, nsteps, d_tape, tape_bytes, true, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_ensemble_leapfrog_kdk_vjp_f32(const float* d_tape, int64_t n, int64_t nsim,
                                                     const odisseo_sim_params* h_params, int64_t nparams, int64_t nsteps,
                                                     int with_eps_G, int accumulate, float* d_lx, float* d_lv, double* d_gm,
                                                     double* d_gparams, void* d_workspace, size_t workspace_bytes, void* stream)
{
    if (n < 0 || nsim < 0 || nsteps < 0 || n > ENSEMBLE_MAX_N || nsim > 0x7fffffff) return ODISSEO_ERR_ARG;
    if (n == 0 || nsim == 0) return ODISSEO_OK;
    if (!d_tape || !d_lx || !d_lv || !d_gm || !d_gparams || !h_params || !d_workspace) return ODISSEO_ERR_NULL;
    if (misaligned(d_tape, 16) || misaligned(d_lx, 16) || misaligned(d_lv, 16) || misaligned(d_gm, 8) ||
        misaligned(d_gparams, 8) || misaligned(d_workspace, 256))
        return ODISSEO_ERR_ALIGN;
    const size_t bytes = (size_t)nsim * n * 16;
    if (overlap(d_lx, bytes, d_lv, bytes)) return ODISSEO_ERR_ARG;
    if (nparams != 1 && nparams != nsim) return ODISSEO_ERR_ARG;
    DeviceInfo dev;
    odisseo_status st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const EnsembleParams* d32;
    const EnsembleParams64* d64;
    st = ensemble_upload_params(h_params, nparams, d_workspace, workspace_bytes, s, &d32, &d64, true);
    if (st != ODISSEO_OK) return st;
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = launch_ensemble_vjp_f32(d_tape, d64, nparams == 1 ? 1 : 0, (int)n, nsim, nsteps, with_eps_G != 0, d_lx, d_lv, d_gm,
                                            d_gparams, accumulate != 0, s);
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

odisseo_status odisseo_kick_drift_f32(float* d_posm, float* d_vel, const float* d_acc, int64_t n, float G, float dt,
                                      const odisseo_potential* pot, int mode, void* d_workspace,
                                      size_t workspace_bytes, void* stream)
{ return kick_drift_impl<float>(d_posm, d_vel, d_acc, n, G, dt, pot, mode, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_kick_drift_f64(double* d_posm, double* d_vel, const double* d_acc, int64_t n, double G, double dt,
                                      const odisseo_potential* pot, int mode, void* d_workspace,
                                      size_t workspace_bytes, void* stream)
{ return kick_drift_impl<double>(d_posm, d_vel, d_acc, n, G, dt, pot, mode, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_leapfrog_kdk_host_f32(float* h_posm, float* h_vel, float* h_acc, int acc_valid, int64_t n, float G, float eps,
                                             float dt, int64_t nsteps, const odisseo_potential* pot,
                                             void* d_workspace, size_t workspace_bytes, void* stream)
{ return leapfrog_host_impl<float>(h_posm, h_vel, h_acc, acc_valid, n, G, eps, dt, nsteps, pot, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_leapfrog_kdk_host_f64(double* h_posm, double* h_vel, double* h_acc, int acc_valid, int64_t n, double G,
                                             double eps, double dt, int64_t nsteps, const odisseo_potential* pot,
                                             void* d_workspace, size_t workspace_bytes, void* stream)
{ return leapfrog_host_impl<double>(h_posm, h_vel, h_acc, acc_valid, n, G, eps, dt, nsteps, pot, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_staged_sources_layout(int64_t n, int is_f64, int64_t out[3])
{
    if (!out) return ODISSEO_ERR_NULL;
    if (n <= 0) return ODISSEO_ERR_ARG;
    const PairPlan p = make_plan(n, is_f64, 148);          // the layout depends on n only
    out[0] = (int64_t)plan_flag_bytes(p);
    out[1] = p.rec_bytes;
    out[2] = plan_npad(p) + STAGED_SLACK;
    return ODISSEO_OK;
}

odisseo_status odisseo_stage_sources_f32(const float* d_posm, int64_t n, void* d_workspace, size_t workspace_bytes, void* stream)
{ return stage_sources_impl<float>(d_posm, n, d_workspace, workspace_bytes, stream); }
odisseo_status odisseo_stage_sources_f64(const double* d_posm, int64_t n, void* d_workspace, size_t workspace_bytes, void* stream)
{ return stage_sources_impl<double>(d_posm, n, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_pair_accel_staged_f32(const float* d_targets, int64_t nt, int64_t n, float* d_acc, float G, float eps,
                                             void* d_workspace, size_t workspace_bytes, void* stream)
{ return pair_staged_impl<float>(d_targets, nt, n, d_acc, G, eps, d_workspace, workspace_bytes, stream); }
odisseo_status odisseo_pair_accel_staged_f64(const double* d_targets, int64_t nt, int64_t n, double* d_acc, double G, double eps,
                                             void* d_workspace, size_t workspace_bytes, void* stream)
{ return pair_staged_impl<double>(d_targets, nt, n, d_acc, G, eps, d_workspace, workspace_bytes, stream); }

odisseo_status odisseo_kick_drift_slice_f32(float* d_posm, float* d_vel, const float* d_acc, int64_t n, int64_t lo, int64_t count,
                                            float G, float dt, const odisseo_potential* pot, int mode, void* d_workspace,
                                            size_t workspace_bytes, void* stream)
{ return kick_drift_slice_impl<float>(d_posm, d_vel, d_acc, n, lo, count, G, dt, pot, mode, d_workspace, workspace_bytes, stream); }
odisseo_status odisseo_kick_drift_slice_f64(double* d_posm, double* d_vel, const double* d_acc, int64_t n, int64_t lo, int64_t count,
                                            double G, double dt, const odisseo_potential* pot, int mode, void* d_workspace,
                                            size_t workspace_bytes, void* stream)
{ return kick_drift_slice_impl<double>(d_posm, d_vel, d_acc, n, lo, count, G, dt, pot, mode, d_workspace, workspace_bytes, stream); }

size_t odisseo_mmd_workspace_bytes(int64_t n, int64_t m, int64_t nsim)
{
    if (n <= 0 || m <= 0 || nsim <= 0) return 0;
    return mmd_workspace_bytes(n, m, nsim);
}

odisseo_status odisseo_mmd2_f32(const float* d_xpos, const float* d_xvel, int64_t n, const float* d_ypos, const float* d_yvel,
                                int64_t m, int64_t nsim, int shared_y, const double* h_sigma, const double* d_grad_scale,
                                double* d_mmd2, float* d_gpos, float* d_gvel, void* d_workspace, size_t workspace_bytes,
                                void* stream)
{
    if (n < 0 || m < 0 || nsim < 0 || n > 0x7fffffff || m > 0x7fffffff || nsim > 65535) return ODISSEO_ERR_ARG;
    if (nsim == 0) return ODISSEO_OK;
    if (n == 0 || m == 0) return ODISSEO_ERR_ARG;          // the estimator divides by n and m
    if (!d_xpos || !d_xvel || !d_ypos || !d_yvel || !h_sigma || !d_mmd2 || !d_workspace) return ODISSEO_ERR_NULL;
    if ((d_gpos == nullptr) != (d_gvel == nullptr)) return ODISSEO_ERR_NULL;
    if (misaligned(d_xpos, 16) || misaligned(d_xvel, 16) || misaligned(d_ypos, 16) || misaligned(d_yvel, 16) ||
        misaligned(d_mmd2, 8) || misaligned(d_workspace, 256) || (d_gpos && (misaligned(d_gpos, 16) || misaligned(d_gvel, 16))) ||
        (d_grad_scale && misaligned(d_grad_scale, 8)))
        return ODISSEO_ERR_ALIGN;
    double inv[6];
    for (int c = 0; c < 6; ++c) {
        if (!(h_sigma[c] > 0.0) || !isfinite(h_sigma[c])) return ODISSEO_ERR_ARG;
        inv[c] = 1.0 / h_sigma[c];
    }
    if (workspace_bytes < mmd_workspace_bytes(n, m, nsim)) return ODISSEO_ERR_WORKSPACE;
    DeviceInfo dev;
    odisseo_status st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    g_launches.fetch_add(2, std::memory_order_relaxed);
    cudaError_t e = launch_mmd_f32(d_xpos, d_xvel, n, d_ypos, d_yvel, m, shared_y != 0, inv, nsim, d_grad_scale, d_mmd2, d_gpos,
                                   d_gvel, d_workspace, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return cuda_fail(e);
    return ODISSEO_OK;
}

size_t odisseo_mmd2_static_scratch_bytes(void) { return mmd_static_scratch_bytes(); }

// odisseo_mmd2_f32 without a workspace argument (include/odisseo.h): for callers that cannot cudaMalloc one.  The
// checks are those of odisseo_mmd2_f32; the size test is against the built-in array instead of the caller's bytes.
odisseo_status odisseo_mmd2_static_f32(const float* d_xpos, const float* d_xvel, int64_t n, const float* d_ypos,
                                       const float* d_yvel, int64_t m, int64_t nsim, int shared_y, const double* h_sigma,
                                       const double* d_grad_scale, double* d_mmd2, float* d_gpos, float* d_gvel, void* stream)
{
    if (n < 0 || m < 0 || nsim < 0 || n > 0x7fffffff || m > 0x7fffffff || nsim > 65535) return ODISSEO_ERR_ARG;
    if (nsim == 0) return ODISSEO_OK;
    if (n == 0 || m == 0) return ODISSEO_ERR_ARG;
    if (!d_xpos || !d_xvel || !d_ypos || !d_yvel || !h_sigma || !d_mmd2) return ODISSEO_ERR_NULL;
    if ((d_gpos == nullptr) != (d_gvel == nullptr)) return ODISSEO_ERR_NULL;
    if (misaligned(d_xpos, 16) || misaligned(d_xvel, 16) || misaligned(d_ypos, 16) || misaligned(d_yvel, 16) ||
        misaligned(d_mmd2, 8) || (d_gpos && (misaligned(d_gpos, 16) || misaligned(d_gvel, 16))) ||
        (d_grad_scale && misaligned(d_grad_scale, 8)))
        return ODISSEO_ERR_ALIGN;
    double inv[6];
    for (int c = 0; c < 6; ++c) {
        if (!(h_sigma[c] > 0.0) || !isfinite(h_sigma[c])) return ODISSEO_ERR_ARG;
        inv[c] = 1.0 / h_sigma[c];
    }
    if (mmd_workspace_bytes(n, m, nsim) > mmd_static_scratch_bytes()) return ODISSEO_ERR_STATIC_LIMIT;
    DeviceInfo dev;
    odisseo_status st = device_info(dev);
    if (st != ODISSEO_OK) return st;
    cudaError_t e = launch_mmd_f32_static(d_xpos, d_xvel, n, d_ypos, d_yvel, m, shared_y != 0, inv, nsim, d_grad_scale, d_mmd2,
                                          d_gpos, d_gvel, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return cuda_fail(e);
    g_launches.fetch_add(2, std::memory_order_relaxed);
    return ODISSEO_OK;
}

}  // extern "C"
