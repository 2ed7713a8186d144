/*
 * plic_oracle.c -- fp64 CPU oracle for the PLIC plane-cube problem.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this
 * file.  It shares no code, header, table or constant with the CUDA path under
 * paper_2006_12838_b200/csrc/ and neither includes the other.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, arxiv 2006.12838):
 *
 *   forward  V0(d0, n) = Vol{ x in [-1/2,1/2]^3 : n.x <= d0 }
 *            written out as the paper's closed form: eq. (2)-(4) mirror+sort
 *            (PAPER.md:40-46), eq. (7) d = S/2 - |d0|, eq. (11)
 *            five-case volume, eq. (6) upper half by symmetry
 *            (PAPER.md:54).
 *
 *   inverse  d0(V0, n) = the unique d0 in [-S/2, S/2] (eq. (1))
 *            with V0(d0, n) = V0.  The analytic methods of the paper reach
 *            exactly this value, so the oracle is the plain definition:
 *            bisection of the forward map on [-S/2, S/2] down to an interval
 *            narrower than 1e-13.  It does NOT follow any of the paper's four
 *            inverse methods.
 *
 * Arithmetic: fp64 throughout.  Inputs are the fp32 values the CUDA path sees,
 * promoted exactly.  No blocking, fusion or reordering beyond what eq. (11)
 * states.
 *
 * Readings of the paper taken here (each also listed in DESIGN.md):
 *   R1  eq. (4) n2 := |nx|+|ny|+|nz|-n1-n3 is, in exact arithmetic, the median
 *       of the three magnitudes; the oracle takes the median itself so that
 *       n1 <= n2 <= n3 holds exactly.
 *   R2  eq. (11) case (5) is printed "min(n1+n2,n3) <= d <= n3".  When
 *       n3 < n1+n2 that is the single point d = n3, where the case-(5)
 *       expression is NOT the volume (e.g. n1=n2=n3, d=n3: case (3) gives 1/6,
 *       case (5) gives 0).  The text calls case (5) "the
 *       remaining free sector ... mutually excluded by the other four cases",
 *       i.e. n1+n2 <= d (<= S/2 <= n3).  That reading is used; V(d) is then
 *       continuous at every case boundary.
 *   R3  case (5) is tested first and case (2) uses the n1-free expansion
 *       d^3-(d-n1)^3 = n1 (3d^2 - 3 d n1 + n1^2), so n1 = 0 and n1 = n2 = 0
 *       never reach a division by zero (caption of Listing 1).
 *   R4  the truncated volume is on the side n.x <= d0, so V0 = 1 <=> d0 = +S/2
 *       (eq. (1), (6), (8)).
 *   R5  sign(0): at d0 = 0 eq. (6) gives V0 = 1/2 for either sign because
 *       V = 1/2 there.
 *   R6  outside the paper's domain: V0 <= 0 -> d0 = -S/2, V0 >= 1 -> +S/2
 *       (the ends of the interval of eq. (1)); n = (0,0,0) -> d0 = 0 and
 *       V0(d0) = 0, 1/2, 1 for d0 <, =, > 0; NaN in -> NaN out.
 *
 * Pins (tests/test_oracle_pins.py): closed forms of cases (1), (2), (5)
 * (eq. (25)), 1D and 2D special cases (eq. (28), (30)), symmetry and
 * monotonicity, endpoints, permutation / sign
 * invariance (eq. (2)-(4)), the textbook inclusion-exclusion formula for the
 * volume of a half-space cut of a box, brute-force sub-cell counting, worked
 * examples with rational values (tests/golden/worked_examples.txt).  No
 * function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* eq. (2)-(4): mirror into positive, sort ascending (R1). */
static void mirror_sort(double nx, double ny, double nz,
                        double *n1, double *n2, double *n3)
{
    double a = fabs(nx), b = fabs(ny), c = fabs(nz), t;
    if (a > b) { t = a; a = b; b = t; }
    if (b > c) { t = b; b = c; c = t; }
    if (a > b) { t = a; a = b; b = t; }
    *n1 = a; *n2 = b; *n3 = c;
}

/* Which of the five intersection cases of eq. (11) the reduced offset d falls in. */
static int case_of(double d, double n1, double n2, double n3)
{
    (void)n3;
    if (d >= n1 + n2) return 5;   /* R2, R3: tested first */
    if (d < n1)       return 1;
    if (d <= n2)      return 2;
    if (d <= n3)      return 3;   /* here d < n1+n2, so d <= min(n1+n2, n3) */
    return 4;
}

/* eq. (11): reduced volume V in [0, 1/2] from reduced offset d in [0, S/2]. */
static double reduced_volume(double d, double n1, double n2, double n3)
{
    double P6 = 6.0 * n1 * n2 * n3;
    double d3 = d * d * d;
    double e1, e2, e3;
    switch (case_of(d, n1, n2, n3)) {
    case 5:  return (d - 0.5 * (n1 + n2)) / n3;
    case 1:  return d3 / P6;
    case 2:  return (3.0 * d * d - 3.0 * d * n1 + n1 * n1) / (6.0 * n2 * n3);   /* R3 */
    case 3:  e1 = d - n1; e2 = d - n2;
             return (d3 - e1 * e1 * e1 - e2 * e2 * e2) / P6;
    default: e1 = d - n1; e2 = d - n2; e3 = d - n3;
             return (d3 - e1 * e1 * e1 - e2 * e2 * e2 - e3 * e3 * e3) / P6;
    }
}

/* Forward map V0(d0, n): eq. (2)-(4), (7), (11), (6). */
double oracle_plic_volume(double d0, double nx, double ny, double nz)
{
    double n1, n2, n3, S, d, V;
    if (isnan(d0) || isnan(nx) || isnan(ny) || isnan(nz)) return NAN;
    mirror_sort(nx, ny, nz, &n1, &n2, &n3);
    if (n3 == 0.0) return d0 < 0.0 ? 0.0 : (d0 > 0.0 ? 1.0 : 0.5);   /* R6 */
    S = n1 + n2 + n3;
    d = 0.5 * S - fabs(d0);                      /* eq. (7) */
    if (d < 0.0) d = 0.0;                        /* plane misses the cube */
    V = reduced_volume(d, n1, n2, n3);
    return d0 > 0.0 ? 1.0 - V : V;               /* eq. (6), R5 */
}

/* Intersection case (1..5) of the plane (d0, n); 0 for the zero normal. */
int oracle_plic_case(double d0, double nx, double ny, double nz)
{
    double n1, n2, n3, d;
    mirror_sort(nx, ny, nz, &n1, &n2, &n3);
    if (n3 == 0.0) return 0;
    d = 0.5 * (n1 + n2 + n3) - fabs(d0);
    if (d < 0.0) d = 0.0;
    return case_of(d, n1, n2, n3);
}

/* Inverse d0(V0, n): bisection of the forward map on [-S/2, S/2] (eq. (1)). */
double oracle_plic_solve(double V0, double nx, double ny, double nz)
{
    double n1, n2, n3, S, lo, hi, mid;
    if (isnan(V0) || isnan(nx) || isnan(ny) || isnan(nz)) return NAN;
    mirror_sort(nx, ny, nz, &n1, &n2, &n3);
    if (n3 == 0.0) return 0.0;                   /* R6 */
    S = n1 + n2 + n3;
    if (V0 <= 0.0) return -0.5 * S;              /* R6 */
    if (V0 >= 1.0) return  0.5 * S;
    lo = -0.5 * S; hi = 0.5 * S;
    while (hi - lo > 1e-13) {
        mid = 0.5 * (lo + hi);
        if (mid <= lo || mid >= hi) break;       /* fp64 fixed point */
        if (oracle_plic_volume(mid, nx, ny, nz) < V0) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

/* Batched forms over N independent cells; `threads` <= 0 means all cores. */
void oracle_plic_volume_batch(const double *d0, const double *nx, const double *ny,
                              const double *nz, double *V0, int64_t N, int threads)
{
    int64_t i;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#else
    (void)threads;
#endif
#pragma omp parallel for schedule(static)
    for (i = 0; i < N; ++i) V0[i] = oracle_plic_volume(d0[i], nx[i], ny[i], nz[i]);
}

void oracle_plic_solve_batch(const double *V0, const double *nx, const double *ny,
                             const double *nz, double *d0, int64_t N, int threads)
{
    int64_t i;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#else
    (void)threads;
#endif
#pragma omp parallel for schedule(dynamic, 4096)
    for (i = 0; i < N; ++i) d0[i] = oracle_plic_solve(V0[i], nx[i], ny[i], nz[i]);
}

void oracle_plic_case_batch(const double *d0, const double *nx, const double *ny,
                            const double *nz, int32_t *kase, int64_t N, int threads)
{
    int64_t i;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#else
    (void)threads;
#endif
#pragma omp parallel for schedule(static)
    for (i = 0; i < N; ++i) kase[i] = oracle_plic_case(d0[i], nx[i], ny[i], nz[i]);
}

/* Same entry points reading the fp32 arrays the CUDA path reads (promoted exactly). */
void oracle_plic_solve_batch_f32(const float *V0, const float *nx, const float *ny,
                                 const float *nz, double *d0, int64_t N, int threads)
{
    int64_t i;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#else
    (void)threads;
#endif
#pragma omp parallel for schedule(dynamic, 4096)
    for (i = 0; i < N; ++i)
        d0[i] = oracle_plic_solve((double)V0[i], (double)nx[i], (double)ny[i], (double)nz[i]);
}

void oracle_plic_volume_batch_f32(const float *d0, const float *nx, const float *ny,
                                  const float *nz, double *V0, int64_t N, int threads)
{
    int64_t i;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#else
    (void)threads;
#endif
#pragma omp parallel for schedule(static)
    for (i = 0; i < N; ++i)
        V0[i] = oracle_plic_volume((double)d0[i], (double)nx[i], (double)ny[i], (double)nz[i]);
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
