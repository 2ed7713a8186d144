/*
 * stratified.c -- the case-stratified workload of BASELINE.json configs[2] -- TEST / BENCH
 * INFRASTRUCTURE, part of the oracle library (it needs the oracle's case classifier and forward
 * map, so it cannot live in gen/, which holds none of the method's arithmetic).  Nothing under
 * paper_2006_12838_b200/ uses it.
 *
 * Recipe (BASELINE.json: "normal uniform on sphere, d0 ~ U[-S/2, +S/2]
 * rejection-sampled so each of the 5 intersection cases is 20% of cells, V0 computed by the
 * oracle's forward map"): cell i targets the intersection case k = (i mod 5) + 1 of eq. (11)
 * (PAPER.md:84).  Draws (n = g/|g| with g ~ N(0, I3), rounded to fp32; d0 = (U - 1/2) S with
 * S = |nx|+|ny|+|nz| of the fp32 normal, rounded to fp32) are repeated until
 * oracle_plic_case(d0, n) == k; then V0 = fp32(oracle_plic_volume(d0, n)).  Acceptance per
 * draw is about 26 / 33 / 18 / 4 / 18 % for cases 1..5.
 *
 * Random numbers: counter based, so cell i depends on (seed, i) only -- not on N, the thread
 * count or the rank.  u(seed, i, j) = splitmix64 finaliser of a key derived from (seed, i) plus
 * j golden-ratio increments, mapped to (0, 1); attempt a of cell i uses j = 5a .. 5a+4: two
 * Box-Muller pairs (three Gaussians used) and one uniform for d0.
 */
#include <math.h>
#include <stdint.h>

#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_plic_case(double d0, double nx, double ny, double nz);
double oracle_plic_volume(double d0, double nx, double ny, double nz);

static uint64_t mix64(uint64_t z)
{
    z += 0x9e3779b97f4a7c15ULL;
    z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ULL;
    z = (z ^ (z >> 27)) * 0x94d049bb133111ebULL;
    return z ^ (z >> 31);
}

static double unit_open(uint64_t key, uint64_t j)
{
    uint64_t r = mix64(key + j * 0x9e3779b97f4a7c15ULL);
    return ((double)(r >> 11) + 0.5) * (1.0 / 9007199254740992.0);     /* (0, 1) */
}

/* cells [start, start + count) of the stream `seed`; returns the largest number of draws one
 * cell needed (diagnostic), or -1 if a cell exhausted max_draws (its case label is then 0). */
int64_t oracle_stratified_cells(uint64_t seed, int64_t start, int64_t count, float *V0, float *nx,
                                float *ny, float *nz, int8_t *kase, int threads)
{
    const double two_pi = 6.283185307179586476925286766559;
    const int max_draws = 100000;
    int64_t worst = 0, c;
    int failed = 0;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#else
    (void)threads;
#endif
#pragma omp parallel for schedule(dynamic, 4096) reduction(max : worst) reduction(| : failed)
    for (c = 0; c < count; ++c) {
        const int64_t i = start + c;
        const int target = (int)(i % 5) + 1;
        const uint64_t key = mix64(mix64(seed) ^ (uint64_t)i);
        int a, found = 0;
        for (a = 0; a < max_draws && !found; ++a) {
            const uint64_t j = 5u * (uint64_t)a;
            const double r1 = sqrt(-2.0 * log(unit_open(key, j))), t1 = two_pi * unit_open(key, j + 1);
            const double r2 = sqrt(-2.0 * log(unit_open(key, j + 2))), t2 = two_pi * unit_open(key, j + 3);
            const double g0 = r1 * cos(t1), g1 = r1 * sin(t1), g2 = r2 * cos(t2);
            const double len = sqrt(g0 * g0 + g1 * g1 + g2 * g2);
            float fx, fy, fz, fd;
            double S;
            if (!(len > 0.0)) continue;
            fx = (float)(g0 / len); fy = (float)(g1 / len); fz = (float)(g2 / len);
            S = fabs((double)fx) + fabs((double)fy) + fabs((double)fz);
            fd = (float)((unit_open(key, j + 4) - 0.5) * S);
            if (oracle_plic_case((double)fd, (double)fx, (double)fy, (double)fz) == target) {
                nx[c] = fx; ny[c] = fy; nz[c] = fz;
                V0[c] = (float)oracle_plic_volume((double)fd, (double)fx, (double)fy, (double)fz);
                kase[c] = (int8_t)target;
                found = 1;
            }
        }
        if (!found) { nx[c] = 0.0f; ny[c] = 0.0f; nz[c] = 1.0f; V0[c] = 0.5f; kase[c] = 0; failed = 1; }
        if (a > worst) worst = a;
    }
    return failed ? -1 : worst;
}
