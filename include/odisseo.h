/*
 * odisseo.h -- C ABI of the B200-native hot path of ODISSEO's direct N-body solver
 * (arxiv 2511.22468).  PAPER.md = the paper's text; citations are PAPER.md line + section.
 *
 * What the library computes
 *   pair   a_i = G * sum_j m_j (x_j - x_i) / (|x_j - x_i|^2 + eps^2)^{3/2}
 *          "direct pairwise force computations with softening, without a tree or
 *          fast-multipole algorithm ... exact forces (up to the softening scale)"
 *          (section 1; formula: BASELINE.json north_star).
 *   ext    a_NFW(x) = -G M_s [ln(1+r/r_s) - (r/r_s)/(1+r/r_s)] x / r^3
 *          a_MN(x)  = -G M (x, y, z (a+B)/B) / D^3,  B = sqrt(z^2+b^2), D^2 = x^2+y^2+(a+B)^2
 *          NFW halo + Miyamoto-Nagai disk (PAPER.md:L9 Abstract; L45 section 2.2.1; L63 section 2.2.2).
 *   kdk    a <- a(x); repeat nsteps: v += a dt/2; x += v dt; a <- a(x); v += a dt/2
 *          "second-order Velocity-Verlet integrator with ... fixed time steps".
 *
 * Conventions (all entry points)
 *   - Every pointer named d_* is a DEVICE pointer, h_* a HOST pointer.  The caller owns
 *     every buffer; the library allocates no device memory (scratch comes in as
 *     `d_workspace`; a plan owns only its CUDA graph objects).
 *   - Particle records are 4 scalars: posm = {x, y, z, m}; vel = {vx, vy, vz, pad};
 *     acc = {ax, ay, az, pad}.  fp32 records are 16 bytes and must be 16-byte aligned,
 *     fp64 records are 32 bytes and must be 32-byte aligned.  posm[i].m is read-only and
 *     is preserved by the integrator.  Pad lanes of outputs are written as 0.
 *   - Calls are asynchronous on `stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream).  No hidden synchronisation, no host-side reads of results.
 *   - posm and acc (and vel) must not alias or overlap: ODISSEO_ERR_ARG.
 *   - Errors are return codes, never exceptions or aborts: NULL pointer -> ERR_NULL,
 *     misaligned pointer -> ERR_ALIGN, n < 0, nsteps < 0, eps <= 0 (the kernels include the
 *     self term, which is exactly 0 only when eps > 0) or eps so small that the self term
 *     overflows in the precision of the call (eps^-3 in the forward calls: fp32 needs
 *     eps >= 1e-12, fp64 eps^2 >= 1e-30; 3 eps^-5 in the fp32 reverse-mode and ensemble-gradient
 *     calls: eps >= 1e-7), eps^2 > 1e30, non-finite scalar, enabled MN term with b <= 0,
 *     enabled NFW term with r_s <= 0, enabled bulge with r_c <= 0 or alpha outside [0, 2)
 *     -> ERR_ARG, workspace too small -> ERR_WORKSPACE, device is not compute capability
 *     10.0 (the library holds sm_100a code only, no PTX fallback) -> ERR_ARCH, CUDA failure ->
 *     ERR_CUDA (code in odisseo_last_cuda_error()).  n == 0 or nsteps == 0 is an OK no-op
 *     (nsteps == 0 with acc_valid == 0 still evaluates acc).  Inputs are not screened for
 *     NaN/Inf particles; they propagate.  The masses live on the device, so the eps bound above cannot
 *     know them: the fp32 loop for UNEQUAL masses forms m_j eps^-3 in the self term, and the accepted region
 *     is  max_j |m_j| * eps^-3 < 3.4e38 (FLT_MAX);  beyond it that product is inf, inf * 0 = NaN, and every
 *     acceleration of the call is NaN (tests/test_gpu_parity.py pins both sides of the edge).  Equal masses
 *     are applied in fp64 after the sum and have no such bound; fp64 calls need |m_j| eps^-3 < 1.8e308.
 *   - There is no CPU fallback: without a B200 every compute call fails with ERR_ARCH/ERR_CUDA.
 *   - Results are bit-reproducible run to run for fixed (n, device SM count): partial sums
 *     are combined in a fixed order, never with atomics.
 */
#ifndef ODISSEO_H
#define ODISSEO_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    ODISSEO_OK = 0,
    ODISSEO_ERR_NULL = 1,
    ODISSEO_ERR_ALIGN = 2,
    ODISSEO_ERR_ARG = 3,
    ODISSEO_ERR_WORKSPACE = 4,
    ODISSEO_ERR_ARCH = 5,
    ODISSEO_ERR_CUDA = 6,
    ODISSEO_ERR_STATIC_LIMIT = 7   /* the problem needs more scratch than odisseo_mmd2_static_scratch_bytes() */
} odisseo_status;

/* NFW: Phi = -G M_s ln(1 + r/r_s) / r, i.e. M_s = 4 pi rho_0 r_s^3 (reading R10).
 * M_s <= 0 disables the term.  At r = 0 the acceleration is defined as 0. */
typedef struct { double M_s, r_s; } odisseo_nfw;
/* Miyamoto-Nagai: Phi = -G M / sqrt(R^2 + (a + sqrt(z^2 + b^2))^2).  M <= 0 disables; b > 0. */
typedef struct { double M, a, b; } odisseo_mn;
/* Bulge of galpy's MWPotential2014 (reading R21): spherical power law with exponential cut-off,
 * rho = A r^-alpha exp(-(r/r_c)^2), total mass M_b = 2 pi A r_c^(3-alpha) Gamma((3-alpha)/2);  a = -G M_b P(s, t) x / r^3 with
 * s = (3-alpha)/2, t = (r/r_c)^2 and P the regularised lower incomplete gamma function.  M_b <= 0 disables; 0 <= alpha < 2,
 * r_c > 0 required when enabled (MWPotential2014: alpha = 1.8, r_c = 1.9 kpc, M_b = 4.5e9 Msun).  a(0) := 0. */
typedef struct { double M_b, alpha, r_c; } odisseo_bulge;
/* A NULL odisseo_potential pointer means "no external potential" (config 0). HOST struct. */
typedef struct { odisseo_nfw nfw; odisseo_mn mn; odisseo_bulge bulge; } odisseo_potential;

/* Library version string, e.g. "odisseo-b200 0.1 (sm_100a)". Never NULL. */
const char *odisseo_version(void);
const char *odisseo_status_string(odisseo_status s);
/* cudaError_t value of the most recent ODISSEO_ERR_CUDA on this thread (0 if none). */
int odisseo_last_cuda_error(void);

/* odisseo_leapfrog_kdk_* can run a whole call as ONE cooperative launch: a persistent kernel with the time loop inside
 * and a grid barrier between the pair and the integrate phase, bit-identical to the per-step launch sequence.  By
 * default only fp64 calls on 1,280 <= n <= 4,096 take it (measured: the two barriers per step cost what the launch edges
 * cost; see csrc/api.cu).  This sets the largest n served that way for both precisions, with no lower bound (clamped
 * to 16384; 0 = always launch per step; negative = restore the defaults) and returns the previous fp64 value: a
 * tuning and test knob, process-wide. */
int64_t odisseo_set_fused_max_n(int64_t n);

/* Small simulations (the inference runs N = 1,000 particles for 1,000 steps) take a third form of
 * odisseo_leapfrog_kdk_*: ONE launch of one thread-block cluster (16 CTAs) that keeps every position in the shared
 * memory of each CTA, exchanges the moved records through distributed shared memory and synchronises with one
 * hardware cluster barrier per step; same summation order, bit-identical to the other two forms.  Default bounds:
 * n <= 1,024 (fp32) / 512 (fp64).  This sets the largest n served that way for both precisions (clamped to 4,096;
 * the shared memory of a CTA bounds it further; 0 = never; negative = restore the defaults) and returns the previous
 * fp32 value: a tuning and test knob, process-wide.  Not used with a tape, inside a stream capture or while a
 * profile is open. */
int64_t odisseo_set_cluster_max_n(int64_t n);

/* The form tried first for small simulations: ONE cooperative launch on all SMs in which every CTA keeps all source
 * records in shared memory and owns a few targets (pair sums, fixed-order reduce, kicks and drift stay inside the CTA),
 * and the moved positions are exchanged through global memory as 64-bit words {value bits, step tag} that every CTA
 * polls (the flag travels with the data: no grid barrier, no fence, one L2 round trip per step).  Same summation
 * order, bit-identical to the other forms.  Default bounds: n <= 4,096 (fp32) / 2,048 (fp64).  This sets the largest n
 * served that way for both precisions (clamped to 6,144; the shared memory of a CTA bounds it further; 0 = never;
 * negative = restore the defaults) and returns the previous fp32 value: a tuning and test knob, process-wide.  It
 * also serves odisseo_leapfrog_kdk_tape_* (the owner threads store the snapshots).  Not used inside a stream capture
 * or while a profile is open; when the device cannot hold the grid the call falls back to the other forms. */
int64_t odisseo_set_ll_max_n(int64_t n);

/* Releases what the library keeps between calls: the cached CUDA-graph executables of odisseo_leapfrog_kdk_* and the
 * CUDA events of odisseo_profile_*.  Call with no library work in flight on other host threads; every entry point may
 * be used again afterwards (the caches refill).  ERR_ARG while a profile is open.  The library's other globals are a
 * launch counter and per-device attribute records; calls from several host threads are safe (the graph cache is
 * looked up, filled, evicted and launched under one lock). */
odisseo_status odisseo_shutdown(void);

/* Upper bound, in bytes, of the device scratch any pair/leapfrog call on n particles
 * needs (room for staged source records -- used by the cross, sharded and cooperative forms only; the default path
 * reads the particles' own records -- + one row of fixed-order partial sums per work unit; for n <= 6,144 the row area
 * is at least 96 (n + 1) bytes, the exchange words of the small-n whole-loop kernel).
 * is_f64 != 0 for the fp64 calls.  Returns 0 for n <= 0.  With a current CUDA device the
 * bound is the one for that device's SM count; without one (no GPU) it is the maximum over
 * devices with 64..192 SMs.  Host arithmetic only. */
size_t odisseo_workspace_bytes(int64_t n, int is_f64);

/* Pair acceleration, fp32.
 *   d_posm [n][4] float in, d_acc [n][4] float out = G * sum_j ... (pad lane 0).
 * Sum over ALL j including j == i (exactly 0 for eps > 0).  Per-tile fp32 partial sums are
 * promoted to fp64 and combined in fixed order, then scaled by G and rounded once. */
odisseo_status odisseo_pair_accel_f32(const float *d_posm, float *d_acc, int64_t n,
                                      float G, float eps,
                                      void *d_workspace, size_t workspace_bytes, void *stream);

/* Same in fp64: d_posm [n][4] double (32-byte aligned), d_acc [n][4] double. */
odisseo_status odisseo_pair_accel_f64(const double *d_posm, double *d_acc, int64_t n,
                                      double G, double eps,
                                      void *d_workspace, size_t workspace_bytes, void *stream);

/* Cross form (SURVEY.md 8b "optional subset call", 8e, 8f NEXT-1): acceleration AT nt target positions DUE TO n
 * sources,  d_acc[i] = G sum_j m_j (x_j - t_i) / (|x_j - t_i|^2 + eps^2)^{3/2}.  Targets need not be sources
 * (tracer particles, a seeded subset, one rank's slice of a sharded run: targets = my slice, sources = all
 * particles); the mass lane of d_targets is ignored; a target that coincides with a source gets exactly 0 from it.
 * Same kernels, same fixed-order sums.  Workspace: odisseo_cross_workspace_bytes(nt, n, is_f64). */
size_t odisseo_cross_workspace_bytes(int64_t nt, int64_t n, int is_f64);
odisseo_status odisseo_pair_accel_cross_f32(const float *d_targets, int64_t nt, const float *d_sources, int64_t n,
                                            float *d_acc, float G, float eps,
                                            void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_pair_accel_cross_f64(const double *d_targets, int64_t nt, const double *d_sources, int64_t n,
                                            double *d_acc, double G, double eps,
                                            void *d_workspace, size_t workspace_bytes, void *stream);

/* Sharded form: one simulation spread over R ranks by TARGET slices (section 2.1, Fig. 1 -- the paper's
 * only performance experiment).  Rank r owns the particles [lo_r, lo_r + count_r), holds
 * the staged source records of ALL n particles in its workspace, and per KDK step calls
 *     odisseo_kick_drift_slice_*   (moves its slice, re-stages the slice's records at their global index)
 *     <exchange>                   (in-place all-gather of the record array, by the caller: NCCL / torch.distributed)
 *     odisseo_pair_accel_staged_*  (its targets against the staged sources; no re-packing of the n sources)
 * after one odisseo_stage_sources_* (records, padding and the equal-mass flags, which never change: masses are
 * constant).  The summation order of a target depends on n only (chunk and tile boundaries are functions of n),
 * so every rank count -- 1 included -- gives results BIT-IDENTICAL to odisseo_leapfrog_kdk_* on one GPU.
 *   odisseo_staged_sources_layout: out = {byte offset of record 0 in the workspace, bytes per record, records the
 *     array has room for (8 ceil(n/8) + 1,024: room for equal 8-aligned slices of up to 128 ranks)}.  Host arithmetic.
 *     Records are plain {x,y,z,m} in both precisions: 16 bytes (fp32) / 32 bytes (fp64).
 *   odisseo_stage_sources_*: d_posm [n][4].  Workspace >= odisseo_cross_workspace_bytes(nt, n, is_f64).
 *   odisseo_pair_accel_staged_*: d_targets [nt][4] (positions; lane 3 ignored), d_acc [nt][4] out (pair-only).
 *   odisseo_kick_drift_slice_*: d_posm, d_vel, d_acc address the slice's count records (d_posm may point into the
 *     array of all particles); mode as odisseo_kick_drift_*.  The rank whose slice ends at n also writes the padding
 *     records; an empty slice with lo == n still does.  lo + count > n -> ERR_ARG. */
odisseo_status odisseo_staged_sources_layout(int64_t n, int is_f64, int64_t out[3]);
odisseo_status odisseo_stage_sources_f32(const float *d_posm, int64_t n, void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_stage_sources_f64(const double *d_posm, int64_t n, void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_pair_accel_staged_f32(const float *d_targets, int64_t nt, int64_t n, float *d_acc, float G, float eps,
                                             void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_pair_accel_staged_f64(const double *d_targets, int64_t nt, int64_t n, double *d_acc, double G, double eps,
                                             void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_kick_drift_slice_f32(float *d_posm, float *d_vel, const float *d_acc, int64_t n, int64_t lo, int64_t count,
                                            float G, float dt, const odisseo_potential *pot, int mode, void *d_workspace,
                                            size_t workspace_bytes, void *stream);
odisseo_status odisseo_kick_drift_slice_f64(double *d_posm, double *d_vel, const double *d_acc, int64_t n, int64_t lo, int64_t count,
                                            double G, double dt, const odisseo_potential *pot, int mode, void *d_workspace,
                                            size_t workspace_bytes, void *stream);

/* Structure-of-arrays face of the fp32 pair call: seven length-n float arrays (4-byte
 * aligned).  Packs into the workspace, runs the same kernel, unpacks.  Workspace must be
 * odisseo_workspace_bytes(n, 0) + 32 * n + 512 bytes, 256-byte aligned. */
odisseo_status odisseo_pair_accel_soa_f32(const float *d_x, const float *d_y, const float *d_z,
                                          const float *d_m, float *d_ax, float *d_ay, float *d_az,
                                          int64_t n, float G, float eps,
                                          void *d_workspace, size_t workspace_bytes, void *stream);

/* External acceleration a_NFW + a_MN.
 * accumulate == 0: d_acc = a_ext (pad 0); accumulate != 0: d_acc.xyz += a_ext.
 * pot == NULL or both terms disabled: zeros / unchanged.  `pot` is read on the host during
 * the call (G*M_s, G*M, 1/r_s are combined in double there, then rounded once). */
odisseo_status odisseo_ext_accel_f32(const float *d_posm, float *d_acc, int64_t n, float G,
                                     const odisseo_potential *pot, int accumulate, void *stream);
odisseo_status odisseo_ext_accel_f64(const double *d_posm, double *d_acc, int64_t n, double G,
                                     const odisseo_potential *pot, int accumulate, void *stream);

/* nsteps kick-drift-kick steps in place.
 *   d_posm, d_vel in/out; d_acc in/out holds the PAIR-ONLY acceleration a_pair(x):
 *   acc_valid != 0 promises d_acc == a_pair(d_posm) on entry (as left by a previous call),
 *   which skips the initial evaluation; on exit d_acc == a_pair(x_final), x and v are
 *   synchronised at t0 + nsteps*dt.  Chained calls are bit-identical to one long call.
 * The external acceleration is recomputed from x inside the kick kernels.  dt may be
 * negative or zero (backward integration, PAPER.md:L43 step 2).  One pair evaluation per
 * step (+1 at the start unless acc_valid).  The per-step launch sequence is captured
 * once in a CUDA graph and replayed. */
odisseo_status odisseo_leapfrog_kdk_f32(float *d_posm, float *d_vel, float *d_acc, int acc_valid,
                                        int64_t n, float G, float eps, float dt, int64_t nsteps,
                                        const odisseo_potential *pot,
                                        void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_leapfrog_kdk_f64(double *d_posm, double *d_vel, double *d_acc, int acc_valid,
                                        int64_t n, double G, double eps, double dt, int64_t nsteps,
                                        const odisseo_potential *pot,
                                        void *d_workspace, size_t workspace_bytes, void *stream);

/* The O(N) integrator kernel on its own (SURVEY.md 8a rows a2 + a3): given the
 * pair-only acceleration in d_acc (input, unchanged), with a = d_acc + a_NFW(x) + a_MN(x):
 *   mode & 1: closing half kick          v += a dt/2
 *   mode & 2: opening half kick + drift  v += a dt/2 ; x += v dt   (a evaluated BEFORE the drift).
 * Nothing is staged: odisseo_pair_accel_* and the leapfrog read the particles' own {x,y,z,m} records (the
 * workspace only receives the equal-mass flags), so the launch moves the 80 algorithmic bytes per particle in fp32.
 * mode 3 = the kernel a full leapfrog step launches between two pair evaluations.  This is the launch
 * bench.py times for the integrator's HBM roofline; it is also the building block for callers that
 * obtain pair accelerations elsewhere.  Workspace as for odisseo_pair_accel_*.  mode outside 1..3 ->
 * ERR_ARG. */
odisseo_status odisseo_kick_drift_f32(float *d_posm, float *d_vel, const float *d_acc, int64_t n, float G,
                                      float dt, const odisseo_potential *pot, int mode,
                                      void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_kick_drift_f64(double *d_posm, double *d_vel, const double *d_acc, int64_t n, double G,
                                      double dt, const odisseo_potential *pot, int mode,
                                      void *d_workspace, size_t workspace_bytes, void *stream);

/* Host-buffer face of the leapfrog (end-to-end path): copies h_posm, h_vel [n][4] (and, when
 * acc_valid != 0, h_acc, which must then be non-NULL and hold a_pair(h_posm) as left by a
 * previous call) to the device, runs nsteps KDK steps, copies posm, vel and (if h_acc != NULL)
 * the pair-only acceleration back.  All copies are cudaMemcpyAsync on `stream`; host buffers should be
 * pinned for true asynchrony and must stay valid until the stream is synchronised.
 * d_workspace must hold odisseo_workspace_bytes(n, is_f64) + 3 state arrays
 * (3 * n * 16 bytes fp32, 3 * n * 32 bytes fp64) + 768 bytes, 256-byte aligned. */
odisseo_status odisseo_leapfrog_kdk_host_f32(float *h_posm, float *h_vel, float *h_acc, int acc_valid,
                                             int64_t n, float G, float eps, float dt, int64_t nsteps,
                                             const odisseo_potential *pot,
                                             void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_leapfrog_kdk_host_f64(double *h_posm, double *h_vel, double *h_acc, int acc_valid,
                                             int64_t n, double G, double eps, double dt, int64_t nsteps,
                                             const odisseo_potential *pot,
                                             void *d_workspace, size_t workspace_bytes, void *stream);

/* Conservation diagnostics: everything is evaluated in fp64 from the
 * given state, whatever its precision, with fixed-order reductions (bit-reproducible).
 *   d_out [16] double, DEVICE:  [0] kinetic energy 1/2 sum m v^2
 *                               [1] pair potential energy -1/2 G sum_i sum_{j!=i} m_i m_j (r_ij^2+eps^2)^-1/2
 *                               [2] external potential energy sum m_i (Phi_NFW + Phi_MN)(x_i)  (0 if pot NULL)
 *                               [3..5] linear momentum  [6..8] angular momentum about the origin
 *                               [9..11] centre of mass  [12] total mass  [13] = [0]+[1]+[2]  [14..15] 0
 *   d_phi  optional DEVICE array of n doubles: per-particle pair potential phi_i (W = 1/2 sum m_i phi_i); may be NULL.
 *   d_workspace  odisseo_diagnostics_workspace_bytes(n) bytes, 256-byte aligned.
 * One O(N^2) fp64 pass (the fp64 pair kernel in potential mode) plus three O(N) kernels.  The pass sums
 * the self term m_i / eps with the others and removes it afterwards, so [1] carries a rounding of a few
 * ulp of the self energy 1/2 G sum m_i^2 / eps (invisible unless n is tiny). */
size_t odisseo_diagnostics_workspace_bytes(int64_t n);
odisseo_status odisseo_diagnostics_f32(const float *d_posm, const float *d_vel, int64_t n, float G, float eps,
                                       const odisseo_potential *pot, double *d_out, double *d_phi,
                                       void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_diagnostics_f64(const double *d_posm, const double *d_vel, int64_t n, double G, double eps,
                                       const odisseo_potential *pot, double *d_out, double *d_phi,
                                       void *d_workspace, size_t workspace_bytes, void *stream);

/* Reverse-mode derivative.  The paper's simulator is "end-to-end differentiable" with
 * respect to initial conditions, integration time, particle masses and potential parameters (PAPER.md:L15,
 * L21; used for Theta = (t_end, M_Plummer, M_NFW, M_MN) in L43 and for (M_vir, r_s, M, a, b) in L63).
 *
 * odisseo_accel_vjp_*: cotangent d_cot [n][4] (lanes x, y, z; pad ignored) pulled back through
 *   a(x) = a_pair(x; m, G, eps) + a_NFW(x) + a_MN(x):
 *     d_gx [n][4]      (da/dx)^T c                      (pad lane 0)
 *     d_gm [n] double  d(c.a)/dm_i
 *     d_gparams [10] double, DEVICE: d(c.a)/d(M_s, r_s, M_d, a, b, G, eps), slot 7 = 0, slots 8, 9 = d/d(M_b, r_c)
 * odisseo_leapfrog_kdk_tape_*: odisseo_leapfrog_kdk_* (acc_valid = 0) that also records the nsteps + 1
 *   snapshots {posm, vel, pair-only acc} k = 0..nsteps into d_tape (odisseo_tape_bytes(n, nsteps, is_f64)
 *   bytes: snapshot k at byte offset k * 3 * n * record size).  Final state bit-identical to the plain call.
 * odisseo_leapfrog_kdk_vjp_*: given the tape and the cotangents of the final state, d_lx = dL/dx_N and
 *   d_lv = dL/dv_N ([n][4], in/out), returns in place dL/dx_0 and dL/dv_0, and
 *     d_gm [n] double  dL/dm_i        d_gparams [10] double: dL/d(M_s, r_s, M_d, a, b, G, eps, dt, M_b, r_c)
 *   (dt at fixed nsteps, i.e. t_end / nsteps; M_s, r_s, M_d, a, b as in odisseo_potential, disabled terms give 0).
 * with_eps_G == 0 leaves the G and eps slots 0 and skips their terms in the O(N^2) loop (neither is in the
 * paper's parameter vectors; ~15 % of the pull-back's instructions).
 * O(N^2) pull-back per recorded step (29-41 instructions per pair), fixed-order sums (bit-reproducible), O(N)
 * parts in fp64.  Workspace: odisseo_vjp_workspace_bytes(n, is_f64), 256-byte aligned. */
size_t odisseo_vjp_workspace_bytes(int64_t n, int is_f64);
size_t odisseo_tape_bytes(int64_t n, int64_t nsteps, int is_f64);
odisseo_status odisseo_accel_vjp_f32(const float *d_posm, const float *d_cot, int64_t n, float G, float eps,
                                     const odisseo_potential *pot, int with_eps_G, float *d_gx, double *d_gm,
                                     double *d_gparams,
                                     void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_accel_vjp_f64(const double *d_posm, const double *d_cot, int64_t n, double G, double eps,
                                     const odisseo_potential *pot, int with_eps_G, double *d_gx, double *d_gm,
                                     double *d_gparams,
                                     void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_leapfrog_kdk_tape_f32(float *d_posm, float *d_vel, float *d_acc, int64_t n, float G, float eps,
                                             float dt, int64_t nsteps, const odisseo_potential *pot,
                                             float *d_tape, size_t tape_bytes,
                                             void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_leapfrog_kdk_tape_f64(double *d_posm, double *d_vel, double *d_acc, int64_t n, double G, double eps,
                                             double dt, int64_t nsteps, const odisseo_potential *pot,
                                             double *d_tape, size_t tape_bytes,
                                             void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_leapfrog_kdk_vjp_f32(const float *d_tape, int64_t n, float G, float eps, float dt, int64_t nsteps,
                                            const odisseo_potential *pot, int with_eps_G, float *d_lx, float *d_lv, double *d_gm,
                                            double *d_gparams, void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_leapfrog_kdk_vjp_f64(const double *d_tape, int64_t n, double G, double eps, double dt, int64_t nsteps,
                                            const odisseo_potential *pot, int with_eps_G, double *d_lx, double *d_lv, double *d_gm,
                                            double *d_gparams, void *d_workspace, size_t workspace_bytes, void *stream);

/* Batched small-N ensembles (the paper's inference workload: 10^4 grid points and
 * bootstrap resamples, each an N = 1,000, 1,000-step simulation with its own potential masses,
 * progenitor mass and integration time, Fig. 2, L47, L53).  nsim independent simulations
 * of n particles each (1 <= n <= 2,048) are advanced nsteps KDK steps by one kernel launch, one CTA per
 * simulation, state resident on the SM for the whole time loop.
 *   d_posm, d_vel  [nsim][n][4] float, in/out (device, 16-byte aligned); masses preserved, vel pad lane 0.
 *   h_params       HOST array of nparams records; nparams == 1: all simulations share it, else
 *                  nparams must equal nsim.  eps > 0 per record; pot terms with mass <= 0 are disabled.
 *   d_workspace    odisseo_ensemble_workspace_bytes(nsim) bytes, 256-byte aligned (device copies of the
 *                  parameter records; h_params may be reused as soon as the call returns).
 * Each simulation computes exactly what odisseo_leapfrog_kdk_f32 computes (acc_valid = 0), with fp32
 * two-level summation in 512-source tiles; results agree with it to rounding, not bit for bit. */
typedef struct { double G, eps, dt; odisseo_potential pot; } odisseo_sim_params;
size_t odisseo_ensemble_workspace_bytes(int64_t nsim);
odisseo_status odisseo_ensemble_leapfrog_kdk_f32(float *d_posm, float *d_vel, int64_t n, int64_t nsim,
                                                 const odisseo_sim_params *h_params, int64_t nparams,
                                                 int64_t nsteps, void *d_workspace, size_t workspace_bytes,
                                                 void *stream);

/* Reverse-mode derivative of the ensembles (the paper's gradient-descent stage: 10 gradient steps for each of
 * 1,000 bootstrap resamples of an N = 1,000, 1,000-step simulation, PAPER.md:L43 steps 5-6, L47, L53).
 *   odisseo_ensemble_leapfrog_kdk_tape_f32: the ensemble call that also records, per simulation and per step
 *     k = 0..nsteps, {posm, vel, TOTAL acceleration} ([nsim][nsteps+1][3][n][4] float,
 *     odisseo_ensemble_tape_bytes(n, nsim, nsteps) bytes).  Final state identical to the plain call.
 *   odisseo_ensemble_leapfrog_kdk_vjp_f32: d_lx, d_lv [nsim][n][4] hold dL/dx_N, dL/dv_N of every simulation on
 *     entry and dL/dx_0, dL/dv_0 on exit; d_gm [nsim][n] double = dL/dm_i; d_gparams [nsim][10] double =
 *     dL/d(M_s, r_s, M_d, a, b, G, eps, dt, M_b, r_c) of each simulation.  h_params as in the forward call (the same
 *     records).  accumulate != 0: d_gm and d_gparams are added to instead of overwritten (a backward pass cut
 *     into segments, the later segment first: no gradient arithmetic is left to the caller).
 *     One CTA per simulation, the whole backward time loop in one kernel. */
size_t odisseo_ensemble_tape_bytes(int64_t n, int64_t nsim, int64_t nsteps);
odisseo_status odisseo_ensemble_leapfrog_kdk_tape_f32(float *d_posm, float *d_vel, int64_t n, int64_t nsim,
                                                      const odisseo_sim_params *h_params, int64_t nparams,
                                                      int64_t nsteps, float *d_tape, size_t tape_bytes,
                                                      void *d_workspace, size_t workspace_bytes, void *stream);
odisseo_status odisseo_ensemble_leapfrog_kdk_vjp_f32(const float *d_tape, int64_t n, int64_t nsim,
                                                     const odisseo_sim_params *h_params, int64_t nparams,
                                                     int64_t nsteps, int with_eps_G, int accumulate, float *d_lx, float *d_lv,
                                                     double *d_gm, double *d_gparams, void *d_workspace,
                                                     size_t workspace_bytes, void *stream);

/* Maximum Mean Discrepancy loss between simulated and observed streams, and its gradient (Fig. 2 step 4:
 * "The resulting simulated stream is compared to the observed stream using the Maximum Mean Discrepancy (MMD), and the
 * gradient of the loss is computed"; L39 "full 6D phase-space information"; L47).  The paper prints
 * neither kernel nor estimator (reading R20): Gaussian kernel, one scale per coordinate, biased V-statistic,
 *   k(u, v) = exp(-1/2 sum_d ((u_d - v_d) / sigma_d)^2),  d = x, y, z, vx, vy, vz,
 *   MMD^2 = 1/n^2 sum_ii' k(x_i, x_i') + 1/m^2 sum_jj' k(y_j, y_j') - 2/(n m) sum_ij k(x_i, y_j).
 * Batched like the ensemble calls: d_xpos, d_xvel [nsim][n][4] float (the final state of odisseo_ensemble_leapfrog_kdk_f32;
 * lane 3 ignored) are the simulated clouds, d_ypos, d_yvel the observed one(s): [m][4] shared by every simulation
 * (shared_y != 0) or [nsim][m][4].  h_sigma: 6 HOST doubles > 0 (ERR_ARG otherwise).  d_mmd2 [nsim] double out.
 * d_gpos, d_gvel (both or neither; [nsim][n][4] float out, lane 3 = 0): d_grad_scale[sim] * dMMD^2/d(position, velocity)
 * of every simulated point -- the layout of d_lx, d_lv of odisseo_ensemble_leapfrog_kdk_vjp_f32, so loss -> gradient ->
 * pull-back stays on the device; d_grad_scale [nsim] double or NULL (= 1).  n, m >= 1 (ERR_ARG for an empty cloud),
 * nsim <= 65,535; nsim == 0 -> OK no-op.  Sums: fp32 inside 256-point tiles, fp64 across tiles and blocks in fixed
 * order (bit-reproducible).  Workspace: odisseo_mmd_workspace_bytes(n, m, nsim), 256-byte aligned. */
size_t odisseo_mmd_workspace_bytes(int64_t n, int64_t m, int64_t nsim);
odisseo_status odisseo_mmd2_f32(const float *d_xpos, const float *d_xvel, int64_t n, const float *d_ypos, const float *d_yvel,
                                int64_t m, int64_t nsim, int shared_y, const double *h_sigma, const double *d_grad_scale,
                                double *d_mmd2, float *d_gpos, float *d_gvel, void *d_workspace, size_t workspace_bytes,
                                void *stream);

/* odisseo_mmd2_f32 for callers that cannot allocate device memory (same operation and passages: Fig. 2
 * step 4, L47; reading R20).  odisseo_mmd2_f32 needs a workspace for its per-block sums, and somebody has to
 * cudaMalloc it.  Two kinds of caller cannot: code living inside a host program whose own memory pool took the whole
 * HBM at start-up (a loss called from a JAX or PyTorch process is the usual case here, and a cudaMalloc next to such a
 * pool can simply fail), and code in a region where allocation is ruled out because cudaMalloc / cudaFree stall every
 * stream of the device (an optimisation loop that must not hiccup, a plug-in whose host forbids it).  This entry
 * point takes inputs and outputs only and calls no cudaMalloc, cudaFree or allocating library routine: the block sums
 * go to a fixed array of odisseo_mmd2_static_scratch_bytes() = 1 MiB that is part of the library image (every GPU
 * that loads the library holds it until the process exits).
 *   Arguments, layouts, validation, results: exactly those of odisseo_mmd2_f32 without d_workspace / workspace_bytes;
 *     the same two kernels run, so the outputs are bit-identical to odisseo_mmd2_f32's.
 *   Limit: odisseo_mmd_workspace_bytes(n, m, nsim) = 24 * nsim * ceil(max(n, m) / 512) bytes (rounded up to 256)
 *     must not exceed odisseo_mmd2_static_scratch_bytes(); otherwise ODISSEO_ERR_STATIC_LIMIT and nothing is
 *     launched (2,960 clouds of 1,000 points need 139 KiB; 43,690 cloud-blocks fit).  Use odisseo_mmd2_f32 beyond it.
 *   First call on each device: looks up the array's device address (with that device current) and keeps it; make
 *     this first call before any stream capture begins.  Later calls only launch.
 *   Sharing: every call on a device uses the same array.  Nothing in it has to be cleared -- each call overwrites the
 *     sums it later reads -- but two calls that overlap on the GPU (different streams, or threads, without an
 *     ordering between them) race on it and corrupt each other's d_mmd2.  Calls on one stream are safe. */
size_t odisseo_mmd2_static_scratch_bytes(void);
odisseo_status odisseo_mmd2_static_f32(const float *d_xpos, const float *d_xvel, int64_t n, const float *d_ypos,
                                       const float *d_yvel, int64_t m, int64_t nsim, int shared_y, const double *h_sigma,
                                       const double *d_grad_scale, double *d_mmd2, float *d_gpos, float *d_gvel, void *stream);

/* Instrumentation (bench.py's gpu_launches and roofline legs).
 *   odisseo_launch_count: kernels this library has launched in this process so far (a CUDA
 *     graph replay counts its kernel nodes).  Host counter, no GPU work.
 *   odisseo_profile_begin / _end: between the two calls every pair-kernel launch (the O(N^2)
 *     kernel only, not the O(N) kernels around it) is bracketed by a pair of CUDA events on
 *     the stream it is launched on, and the leapfrog calls replay no graph (graph nodes
 *     cannot be timed individually).  _end waits for the recorded launches and returns the
 *     sum of their durations in milliseconds, how many were timed, and how many were not
 *     because the pool of 4,096 event pairs ran out.  One profile at a time per process;
 *     _end without _begin -> ERR_ARG.  Output pointers are HOST pointers and may be NULL.
 *   odisseo_profile_times: after _end, the individual durations (ms) of the launches it timed, in launch order:
 *     fills h_ms[0 .. min(count, capacity)) and *h_count = count (bench.py's min / median / mean +- std,
 *     SURVEY.md 8d timing protocol).  While a profile is open -> ERR_ARG. */
int64_t odisseo_launch_count(void);
/* Name of the O(N^2) kernel instantiation odisseo_pair_accel_f32 / _f64 (and the per-step leapfrog) launch for n
 * particles, as profilers print it without namespaces, e.g. "stream_kernel<PairF32<4,8,1,16,8>>" -- spelled from the
 * template arguments in the library, so bench.py's roofline.kernel and the summaries under profiles/ cannot go
 * stale.  Static string, never NULL ("" for n <= 0). */
const char *odisseo_pair_kernel_name(int64_t n, int is_f64);
odisseo_status odisseo_profile_begin(void);
odisseo_status odisseo_profile_end(double *h_ms_total, int64_t *h_launches, int64_t *h_dropped);
odisseo_status odisseo_profile_times(double *h_ms, int64_t capacity, int64_t *h_count);

/* Pipe-rate micro-benchmarks ("verify with step-0
 * micro-benchmarks"): the measured FP32 / FP64 / MUFU rates the roofline fractions are quoted
 * against, next to the nominal ones.  Instrumentation, not part of the hot path.
 *   odisseo_ubench_kinds: number of kinds; odisseo_ubench_name(kind): static string, NULL if out of
 *     range ("ffma", "ffma2_3src", "ffma2_shared", "ffma2_square", "fadd2", "fmul2", "mufu_rsq",
 *     "dfma", and interleaved mixes with the pair kernel's instruction proportions).
 *   odisseo_ubench_run: launches kind on ctas_per_sm * SMs CTAs of `threads` threads (multiple of 32,
 *     <= 1024), `iters` (even, >= 2) loop iterations per thread, one warm-up launch + 3 timed with
 *     CUDA events on `stream`; SYNCHRONISES the stream and allocates 256 B of device memory for
 *     the duration of the call.  h_out (HOST, 6 doubles) = {best time in ms, FP32-pipe lane
 *     operations executed (a packed instruction counts 2 per thread), MUFU results, FP64
 *     operations, shared-memory loads (per thread), SM count}.
 *   Errors: ERR_NULL, ERR_ARG (range), ERR_ARCH, ERR_CUDA. */
int odisseo_ubench_kinds(void);
const char *odisseo_ubench_name(int kind);
odisseo_status odisseo_ubench_run(int kind, int ctas_per_sm, int threads, int64_t iters, double h_out[6], void *stream);

/* Description of the launch plan the library would use for n particles on the current
 * device (host arithmetic + one device-attribute query): fills out[0..7] with
 * {i_bodies_per_thread, threads_per_cta, max_tile_records, persistent_ctas, i_blocks,
 *  source_chunks, partial_rows, kernels_per_step}.  For tests, bench.py and DESIGN.md. */
odisseo_status odisseo_describe_plan(int64_t n, int is_f64, int64_t out[8]);
/* Same for a hypothetical device with num_sms SMs: pure host arithmetic, needs no GPU. */
odisseo_status odisseo_describe_plan_for(int64_t n, int is_f64, int num_sms, int64_t out[8]);
/* Same for nt targets against n sources (the cross call): max_tile_records and source_chunks depend on
 * n and num_sms only, never on nt (the same fixed reduction order per target). */
odisseo_status odisseo_describe_cross_plan_for(int64_t nt, int64_t n, int is_f64, int num_sms, int64_t out[8]);
/* Unit bookkeeping exactly as the kernels compute it (SURVEY.md 8a row a1'), for host tests: units number
 * the (i-block, source chunk) pairs u = b * source_chunks + s;
 * out = {CTA that owns unit u, first unit of CTA c, one past the last unit of CTA c,
 *        first source record of u's chunk, one past its last source record}.  Pure host arithmetic. */
odisseo_status odisseo_plan_probe(int64_t nt, int64_t n, int is_f64, int num_sms, int64_t u, int64_t c, int64_t out[5]);

#ifdef __cplusplus
}
#endif
#endif /* ODISSEO_H */
