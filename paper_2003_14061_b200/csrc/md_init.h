#pragma once
#include <cstdint>

// kind: 1 = simple cubic, 2 = FCC.  Returns 0 when n fits neither.
int md_init_pick_lattice(int64_t n);
bool md_init_lattice(int kind, int64_t n, double box, double *xyz);
void md_init_velocities(int64_t n, double temperature, uint64_t seed, double *v);
