/*
 * odisseo_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct fp64 CPU statement of what the ODISSEO hot
 * path computes.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.
 * It shares no code, header, table or helper with the CUDA library under
 * paper_2511_22468_b200/csrc/, and neither includes the other.
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md):
 *   - "direct pairwise force computations with softening, without a tree or
 *     fast-multipole algorithm ... exact forces (up to the softening scale)"
 *     (section 1)  -> oracle_pair_accel is the plain double sum.
 *   - external Milky-Way potential = NFW halo + Miyamoto-Nagai disk
 *     (PAPER.md:L9 Abstract; L45 section 2.2.1; L63 section 2.2.2).
 *   - "second-order Velocity-Verlet integrator with ... fixed time steps"
 *     (section 2.2.1)  -> oracle_leapfrog_kdk.
 * The paper prints no formula; the formulas are the ones BASELINE.json
 * north_star states (Plummer softening) and the textbook NFW / MN forms
 * (readings R1, R10, R11).
 *
 * Because direct summation reaches the plain definition exactly (up to
 * rounding order), the oracle IS that definition: double loop, sqrt and
 * divide, no rsqrt tricks, no tiling, no reordering.  Each target's sum is
 * accumulated in long double (80-bit on x86-64 gcc) in source-index order so
 * the oracle's own rounding (~1e-19 S) sits far below the 1e-12 fp64 parity
 * tolerance.  OpenMP parallelises over targets only, so results do not depend
 * on the thread count.
 *
 * Parity pins (tests/test_oracle_*.py): 3-4-5 hand example, mpmath brute
 * force, Newton's third law, translation/permutation invariance, MN(a=0,b=eps)
 * == softened point mass, finite differences of the potentials, Poisson
 * equation, NFW circular speed, two-body circular and Kepler orbits, leapfrog
 * order / energy / reversibility / L_z, Plummer W = -3 pi G M^2 / (32 a); bulge:
 * enclosed mass against 40-digit quadrature of rho, Poisson, finite differences,
 * point-mass and power-law limits, scipy's incomplete gamma (tests/test_oracle_bulge.py).
 * No function here is "parity unpinned".
 *
 * Layouts: posm = n records of 4 doubles {x, y, z, m}; vel, acc = n records of
 * 3 doubles.  All pointers are host pointers owned by the caller.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { double M_s, r_s; } oracle_nfw;    /* M_s <= 0 disables the term */
typedef struct { double M, a, b; } oracle_mn;      /* M   <= 0 disables the term */
typedef struct { double M_b, alpha, r_c; } oracle_bulge;   /* M_b <= 0 disables the term */
typedef struct { oracle_nfw nfw; oracle_mn mn; oracle_bulge bulge; } oracle_potential;

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * Pair acceleration, north_star / PAPER.md:L15-17:
 *   a_i = G * sum_{j != i} m_j (x_j - x_i) / (|x_j - x_i|^2 + eps^2)^{3/2}
 *   S_i = G * sum_{j != i} m_j |x_j - x_i| / (|x_j - x_i|^2 + eps^2)^{3/2}
 * S_i = sum_j |a_ij| is the denominator of north_star's error ratio.
 * The self term is skipped explicitly (so eps = 0 is legal here).  A distinct
 * particle at the same position with eps = 0 would divide by zero; with
 * eps > 0 it contributes exactly 0 (reading R3).
 * targets == NULL: targets are 0..nt-1 (nt must equal n for "all").
 * acc: nt x 3, S: nt (may be NULL).
 */
void oracle_pair_accel(int64_t n, const double *posm, double G, double eps,
                       int64_t nt, const int64_t *targets,
                       double *acc, double *S)
{
    const double eps2 = eps * eps;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < nt; ++t) {
        const int64_t i = targets ? targets[t] : t;
        const double xi = posm[4 * i + 0];
        const double yi = posm[4 * i + 1];
        const double zi = posm[4 * i + 2];
        long double sx = 0.0L, sy = 0.0L, sz = 0.0L, sn = 0.0L;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            const double dx = posm[4 * j + 0] - xi;
            const double dy = posm[4 * j + 1] - yi;
            const double dz = posm[4 * j + 2] - zi;
            const double d2 = dx * dx + dy * dy + dz * dz;
            const double r2 = d2 + eps2;
            const double w = posm[4 * j + 3] / (r2 * sqrt(r2));
            sx += (long double)(w * dx);
            sy += (long double)(w * dy);
            sz += (long double)(w * dz);
            sn += (long double)(w * sqrt(d2));
        }
        acc[3 * t + 0] = (double)((long double)G * sx);
        acc[3 * t + 1] = (double)((long double)G * sy);
        acc[3 * t + 2] = (double)((long double)G * sz);
        if (S) S[t] = (double)((long double)G * sn);
    }
}

/*
 * Softened pair potential energy (diagnostic):
 *   W = -1/2 G sum_i sum_{j != i} m_i m_j / sqrt(r_ij^2 + eps^2)
 */
double oracle_pair_potential_energy(int64_t n, const double *posm, double G, double eps)
{
    const double eps2 = eps * eps;
    long double total = 0.0L;
#pragma omp parallel
    {
        long double part = 0.0L;
#pragma omp for schedule(dynamic, 16)
        for (int64_t i = 0; i < n; ++i) {
            long double s = 0.0L;
            for (int64_t j = 0; j < n; ++j) {
                if (j == i) continue;
                const double dx = posm[4 * j + 0] - posm[4 * i + 0];
                const double dy = posm[4 * j + 1] - posm[4 * i + 1];
                const double dz = posm[4 * j + 2] - posm[4 * i + 2];
                s += (long double)(posm[4 * j + 3] / sqrt(dx * dx + dy * dy + dz * dz + eps2));
            }
            part += (long double)posm[4 * i + 3] * s;
        }
#pragma omp critical
        total += part;
    }
    return (double)(-0.5L * (long double)G * total);
}

/*
 * NFW halo (reading R10):
 *   Phi(r) = -G M_s ln(1 + r/r_s) / r
 *   a(x)   = -G M_s [ln(1 + r/r_s) - (r/r_s)/(1 + r/r_s)] x / r^3
 * i.e. enclosed mass M(<r) = M_s [ln(1+c) - c/(1+c)], c = r/r_s.
 * At r = 0 the direction is undefined: acceleration := 0 (reading R12),
 * Phi(0) = limit = -G M_s / r_s.
 */
static double nfw_phi(double G, const oracle_nfw *p, double x, double y, double z)
{
    const double r = sqrt(x * x + y * y + z * z);
    if (r == 0.0) return -G * p->M_s / p->r_s;
    return -G * p->M_s * log1p(r / p->r_s) / r;
}

static void nfw_acc(double G, const oracle_nfw *p, double x, double y, double z, double a[3])
{
    const double r = sqrt(x * x + y * y + z * z);
    if (r == 0.0) { a[0] = a[1] = a[2] = 0.0; return; }
    const double c = r / p->r_s;
    const double menc = log1p(c) - c / (1.0 + c);
    const double f = -G * p->M_s * menc / (r * r * r);
    a[0] = f * x; a[1] = f * y; a[2] = f * z;
}

/*
 * Miyamoto-Nagai disk ("MN mass, scale height b, length a"):
 *   Phi(R, z) = -G M / sqrt(R^2 + (a + B)^2),  B = sqrt(z^2 + b^2), R^2 = x^2 + y^2
 *   a(x) = -G M (x, y, z (a + B)/B) / D^3,     D = sqrt(R^2 + (a + B)^2)
 */
static double mn_phi(double G, const oracle_mn *p, double x, double y, double z)
{
    const double B = sqrt(z * z + p->b * p->b);
    const double s = p->a + B;
    return -G * p->M / sqrt(x * x + y * y + s * s);
}

static void mn_acc(double G, const oracle_mn *p, double x, double y, double z, double a[3])
{
    const double B = sqrt(z * z + p->b * p->b);
    const double s = p->a + B;
    const double D2 = x * x + y * y + s * s;
    const double f = -G * p->M / (D2 * sqrt(D2));
    a[0] = f * x; a[1] = f * y; a[2] = f * z * (s / B);
}

/*
 * Bulge of galpy's MWPotential2014 ("we adopt the MWPotential2014 model from galpy"; DESIGN.md reading
 * R21): a spherical power law with an exponential cut-off,
 *   rho(r) = A r^-alpha exp(-(r/r_c)^2),   total mass M_b = 2 pi A r_c^(3-alpha) Gamma(s),  s = (3 - alpha)/2,
 *   M(<r)  = M_b P(s, t),  t = (r/r_c)^2,  P = regularised lower incomplete gamma function,
 *   a(x)   = -G M(<r) x / r^3,
 *   Phi(r) = -G M(<r)/r - 4 pi G int_r^inf rho r' dr' = -G M_b [ P(s, t)/r + Gamma(s - 1/2, t) / (r_c Gamma(s)) ]
 * (alpha < 2 so that Phi(0) = -G M_b Gamma(s - 1/2)/(r_c Gamma(s)) is finite; MWPotential2014: alpha = 1.8, r_c = 1.9 kpc).
 * P(s, t) is evaluated by its all-positive Kummer series  t^s e^-t / Gamma(s+1) * sum_k t^k / ((s+1)...(s+k)),
 * which converges for every t (no cancellation; up to ~t + 60 terms); for t > 60, 1 - P < 1e-26: P = 1 to rounding.
 */
static double gamma_p(double s, double t)
{
    if (t <= 0.0) return 0.0;
    if (t > 60.0) return 1.0;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 4000; ++k) {
        term *= t / (s + k);
        sum += term;
        if (term < 1e-18 * sum) break;
    }
    const double p = exp(s * log(t) - t - lgamma(s + 1.0)) * sum;
    return p < 1.0 ? p : 1.0;
}

static double bulge_phi(double G, const oracle_bulge *p, double x, double y, double z)
{
    const double s = 0.5 * (3.0 - p->alpha);
    const double r = sqrt(x * x + y * y + z * z);
    const double t = (r / p->r_c) * (r / p->r_c);
    const double outer = tgamma(s - 0.5) * (1.0 - gamma_p(s - 0.5, t)) / (p->r_c * tgamma(s));
    if (r == 0.0) return -G * p->M_b * outer;
    return -G * p->M_b * (gamma_p(s, t) / r + outer);
}

static void bulge_acc(double G, const oracle_bulge *p, double x, double y, double z, double a[3])
{
    const double s = 0.5 * (3.0 - p->alpha);
    const double r = sqrt(x * x + y * y + z * z);
    if (r == 0.0) { a[0] = a[1] = a[2] = 0.0; return; }
    const double t = (r / p->r_c) * (r / p->r_c);
    const double f = -G * p->M_b * gamma_p(s, t) / (r * r * r);
    a[0] = f * x; a[1] = f * y; a[2] = f * z;
}

/* External acceleration a_NFW + a_MN + a_bulge per particle; pot == NULL -> zeros. acc: n x 3. */
void oracle_ext_accel(int64_t n, const double *posm, double G,
                      const oracle_potential *pot, double *acc)
{
    for (int64_t i = 0; i < n; ++i) {
        double a[3] = {0, 0, 0}, t[3];
        if (pot && pot->nfw.M_s > 0.0) {
            nfw_acc(G, &pot->nfw, posm[4 * i], posm[4 * i + 1], posm[4 * i + 2], t);
            a[0] += t[0]; a[1] += t[1]; a[2] += t[2];
        }
        if (pot && pot->mn.M > 0.0) {
            mn_acc(G, &pot->mn, posm[4 * i], posm[4 * i + 1], posm[4 * i + 2], t);
            a[0] += t[0]; a[1] += t[1]; a[2] += t[2];
        }
        if (pot && pot->bulge.M_b > 0.0) {
            bulge_acc(G, &pot->bulge, posm[4 * i], posm[4 * i + 1], posm[4 * i + 2], t);
            a[0] += t[0]; a[1] += t[1]; a[2] += t[2];
        }
        acc[3 * i] = a[0]; acc[3 * i + 1] = a[1]; acc[3 * i + 2] = a[2];
    }
}

/* External potential Phi_NFW + Phi_MN + Phi_bulge per particle (per unit mass). phi: n. */
void oracle_ext_potential(int64_t n, const double *posm, double G,
                          const oracle_potential *pot, double *phi)
{
    for (int64_t i = 0; i < n; ++i) {
        double p = 0.0;
        if (pot && pot->nfw.M_s > 0.0)
            p += nfw_phi(G, &pot->nfw, posm[4 * i], posm[4 * i + 1], posm[4 * i + 2]);
        if (pot && pot->mn.M > 0.0)
            p += mn_phi(G, &pot->mn, posm[4 * i], posm[4 * i + 1], posm[4 * i + 2]);
        if (pot && pot->bulge.M_b > 0.0)
            p += bulge_phi(G, &pot->bulge, posm[4 * i], posm[4 * i + 1], posm[4 * i + 2]);
        phi[i] = p;
    }
}

/* Total acceleration a_pair + a_ext for every particle. acc: n x 3. */
void oracle_total_accel(int64_t n, const double *posm, double G, double eps,
                        const oracle_potential *pot, double *acc)
{
    double *ext = (double *)malloc(sizeof(double) * 3 * (size_t)(n > 0 ? n : 1));
    oracle_pair_accel(n, posm, G, eps, n, NULL, acc, NULL);
    oracle_ext_accel(n, posm, G, pot, ext);
    for (int64_t k = 0; k < 3 * n; ++k) acc[k] += ext[k];
    free(ext);
}

/*
 * Kick-drift-kick leapfrog == Velocity-Verlet (reading R7):
 *   a <- acc(x)
 *   repeat nsteps:  v += a dt/2;  x += v dt;  a <- acc(x);  v += a dt/2
 * One acceleration evaluation per step plus one at the start.  dt < 0 and
 * dt = 0 are legal (backward integration, PAPER.md:L43 step 2; reading R8).
 * posm (n x 4) and vel (n x 3) are updated in place; masses are untouched.
 * acc_out (n x 3, may be NULL) receives the TOTAL acceleration at the final x.
 */
void oracle_leapfrog_kdk(int64_t n, double *posm, double *vel, double G, double eps,
                         double dt, int64_t nsteps, const oracle_potential *pot,
                         double *acc_out)
{
    double *a = (double *)malloc(sizeof(double) * 3 * (size_t)(n > 0 ? n : 1));
    const double h = 0.5 * dt;
    oracle_total_accel(n, posm, G, eps, pot, a);
    for (int64_t s = 0; s < nsteps; ++s) {
        for (int64_t i = 0; i < n; ++i)
            for (int k = 0; k < 3; ++k) vel[3 * i + k] += a[3 * i + k] * h;
        for (int64_t i = 0; i < n; ++i)
            for (int k = 0; k < 3; ++k) posm[4 * i + k] += vel[3 * i + k] * dt;
        oracle_total_accel(n, posm, G, eps, pot, a);
        for (int64_t i = 0; i < n; ++i)
            for (int k = 0; k < 3; ++k) vel[3 * i + k] += a[3 * i + k] * h;
    }
    if (acc_out) memcpy(acc_out, a, sizeof(double) * 3 * (size_t)n);
    free(a);
}
