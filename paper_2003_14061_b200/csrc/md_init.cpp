// Host-side initial states for md_create: cubic grid + random velocities, following the
// recipe of DESIGN.md "Input recipe" (the same recipe md_workloads/ implements in numpy; tests compare them).
#include <cmath>
#include <cstdint>
#include <vector>

#include "md_init.h"

namespace {

inline uint64_t mix64(uint64_t seed, uint64_t ctr)
{
    uint64_t z = seed * 0xD1342543DE82EF95ull + (ctr + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

inline double u01(uint64_t seed, uint64_t ctr) { return ((double)(mix64(seed, ctr) >> 11) + 0.5) * 0x1.0p-53; }

int64_t icbrt(int64_t n)
{
    int64_t c = (int64_t)std::llround(std::cbrt((double)n));
    for (int64_t k = c - 1; k <= c + 1; k++)
        if (k > 0 && k * k * k == n) return k;
    return 0;
}

}  // namespace

int md_init_pick_lattice(int64_t n)
{
    if (icbrt(n)) return 1;                       // SC
    if (n % 4 == 0 && icbrt(n / 4)) return 2;     // FCC
    return 0;
}

bool md_init_lattice(int kind, int64_t n, double box, double *xyz)
{
    if (kind == 1) {
        const int64_t ne = icbrt(n);
        if (!ne) return false;
        const double a = box / (double)ne;
        for (int64_t i = 0; i < n; i++) {
            const int64_t ix = i % ne, iy = (i / ne) % ne, iz = i / (ne * ne);
            xyz[3 * i] = ((double)ix + 0.5) * a;
            xyz[3 * i + 1] = ((double)iy + 0.5) * a;
            xyz[3 * i + 2] = ((double)iz + 0.5) * a;
        }
        return true;
    }
    if (kind == 2) {
        if (n % 4) return false;
        const int64_t nc = icbrt(n / 4);
        if (!nc) return false;
        const double a = box / (double)nc;
        static const double basis[4][3] = {{0, 0, 0}, {0.5, 0.5, 0}, {0.5, 0, 0.5}, {0, 0.5, 0.5}};
        for (int64_t i = 0; i < n; i++) {
            const int64_t b = i % 4, cell = i / 4;
            const int64_t cx = cell % nc, cy = (cell / nc) % nc, cz = cell / (nc * nc);
            xyz[3 * i] = ((double)cx + basis[b][0] + 0.25) * a;
            xyz[3 * i + 1] = ((double)cy + basis[b][1] + 0.25) * a;
            xyz[3 * i + 2] = ((double)cz + basis[b][2] + 0.25) * a;
        }
        return true;
    }
    return false;
}

void md_init_velocities(int64_t n, double temperature, uint64_t seed, double *v)
{
    const double two_pi = 2.0 * 3.14159265358979323846;
    const double st = std::sqrt(temperature);
    double mean[3] = {0, 0, 0};
    for (int64_t c = 0; c < 3 * n; c++) {
        const double u1 = u01(seed, 2ull * (uint64_t)c), u2 = u01(seed, 2ull * (uint64_t)c + 1ull);
        v[c] = std::sqrt(-2.0 * std::log(u1)) * std::cos(two_pi * u2) * st;
    }
    // pairwise-free but well-conditioned mean: long double accumulation
    long double m[3] = {0, 0, 0};
    for (int64_t i = 0; i < n; i++)
        for (int k = 0; k < 3; k++) m[k] += v[3 * i + k];
    for (int k = 0; k < 3; k++) mean[k] = (double)(m[k] / (long double)n);
    long double s2 = 0;
    for (int64_t i = 0; i < n; i++)
        for (int k = 0; k < 3; k++) {
            v[3 * i + k] -= mean[k];
            s2 += (long double)v[3 * i + k] * v[3 * i + k];
        }
    if (s2 > 0 && n > 1) {
        const double scale = std::sqrt(3.0 * (double)(n - 1) * temperature / (double)s2);
        for (int64_t c = 0; c < 3 * n; c++) v[c] *= scale;
    }
}
