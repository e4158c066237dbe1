/*
 * md_oracle_sp.c -- CPU ORACLE for the SINGLE-PRECISION variant of the MD hot path.
 * TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs, never by the product.  Shares no code with paper_2003_14061_b200/ nor with
 * md_oracle.c (the fp64 oracle), against which tests/test_oracle_sp_pins.py pins it.
 *
 * What it follows (P:<n> = /root/reference/PAPER.md line n):
 *   - the paper's own precision: "single precision" results throughout Table 1, state
 *     held as float4 arrays r, v, a.  Here: coordinates, velocities, forces and all pair arithmetic
 *     are IEEE binary32; every per-atom and global SUM OF ENERGIES (u_i, w_i, KE, momentum) is accumulated
 *     in binary64 (reading R18).
 *   - the same model and step order as md_oracle.c (neighbor set by definition; F1 without
 *     Newton-3; two-half-kick leapfrog with wrap; rebuild when the accumulated
 *     dt * max|v| exceeds delta/2), each operation rounded to binary32 in the order written here
 *     (compile with -ffp-contract=off: a*b+c rounds twice unless written fmaf()).
 *   - where binary32 decides an integer (j in the neighbor set of i; a pair inside r_c) the decision is
 *     r2 < bound with r2 = fmaf(dz,dz, fmaf(dy,dy, dx*dx)), d = minimum image of fl(a - b), bound =
 *     (float)(double r)^2: the CUDA path takes it on the same bits (R18).
 *
 * Boundary arrays are double (the product's C ABI is); they are rounded to binary32 on entry.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double ke, pe_pair, pe_bond, virial, px, py, pz, vmax;
    int64_t step, n_rebuilds;
    int32_t max_neighbors, max_cell_occupancy;
    double mean_neighbors;
} orcs_energy;

typedef struct orcs_sys {
    int64_t N;
    double L, rc, dr, dt;       /* as given */
    float Lf, halff, rc2f, rn2f, ucf, dtf, hdtf;
    float *r, *v, *f;           /* N x 3 */
    double *u, *w;              /* per-atom sums of the binary32 pair terms, accumulated in binary64 */
    int64_t *nb_start;
    int32_t *nb;
    int64_t nb_cap;
    int64_t n_bonds;
    int32_t *bonds;
    float fene_kf, fene_R02f;
    double pe_bond, vir_bond;
    int bond_broken;
    int32_t *partner;           /* 2 x N, from the bond list */
    int has_angles;
    float ang_kf, ang_c0f;
    double pe_angle;
    int has_dihedrals;
    float dih_kf, dih_c0f;
    double pe_dihedral;
    double disp_acc;
    int64_t step, n_rebuilds;
    int32_t max_cell_occ;
    int force_brute;
} orcs_sys;

static inline float minimgf(float d, float L, float half)
{
    if (d > half) d -= L;
    else if (d < -half) d += L;
    return d;
}

static inline float dist2f(const float *a, const float *b, float L, float half, float d[3])
{
    d[0] = minimgf(a[0] - b[0], L, half);
    d[1] = minimgf(a[1] - b[1], L, half);
    d[2] = minimgf(a[2] - b[2], L, half);
    return fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
}

static inline float wrap1f(float x, float L)
{
    if (x >= L) x -= L;
    else if (x < 0.0f) { x += L; if (x >= L) x = 0.0f; }
    return x;
}

void orcs_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orcs_get_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

orcs_sys *orcs_create(int64_t N, double L, double rc, double dr, double dt)
{
    if (N <= 0 || L <= 0 || rc <= 0 || dr < 0 || dt <= 0) return NULL;
    orcs_sys *s = (orcs_sys *)calloc(1, sizeof(orcs_sys));
    s->N = N; s->L = L; s->rc = rc; s->dr = dr; s->dt = dt;
    s->Lf = (float)L;
    s->halff = 0.5f * s->Lf;
    s->rc2f = (float)(rc * rc);
    s->rn2f = (float)((rc + dr) * (rc + dr));
    {   /* energy shift u(r_c), evaluated in binary64 and rounded once */
        double sc = 1.0 / (rc * rc), sc3 = sc * sc * sc;
        s->ucf = (float)(4.0 * sc3 * (sc3 - 1.0));
    }
    s->dtf = (float)dt;
    s->hdtf = (float)(0.5 * dt);
    s->r = (float *)calloc(3 * N, sizeof(float));
    s->v = (float *)calloc(3 * N, sizeof(float));
    s->f = (float *)calloc(3 * N, sizeof(float));
    s->u = (double *)calloc(N, sizeof(double));
    s->w = (double *)calloc(N, sizeof(double));
    s->nb_start = (int64_t *)calloc(N + 1, sizeof(int64_t));
    return s;
}

void orcs_destroy(orcs_sys *s)
{
    if (!s) return;
    free(s->r); free(s->v); free(s->f); free(s->u); free(s->w);
    free(s->nb_start); free(s->nb); free(s->bonds); free(s->partner);
    free(s);
}

void orcs_force_brute_search(orcs_sys *s, int on) { s->force_brute = on; }

/* neighbor sets by definition, O(N^2) */
static void build_brute(orcs_sys *s)
{
    const int64_t N = s->N;
    const float L = s->Lf, half = s->halff, rn2 = s->rn2f;
    int64_t *cnt = s->nb_start;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; i++) {
        int64_t c = 0; float d[3];
        for (int64_t j = 0; j < N; j++)
            if (j != i && dist2f(s->r + 3 * i, s->r + 3 * j, L, half, d) < rn2) c++;
        cnt[i + 1] = c;
    }
    cnt[0] = 0;
    for (int64_t i = 0; i < N; i++) cnt[i + 1] += cnt[i];
    if (cnt[N] > s->nb_cap) { free(s->nb); s->nb_cap = cnt[N] + cnt[N] / 8 + 16; s->nb = (int32_t *)malloc(s->nb_cap * sizeof(int32_t)); }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; i++) {
        int64_t p = cnt[i]; float d[3];
        for (int64_t j = 0; j < N; j++)
            if (j != i && dist2f(s->r + 3 * i, s->r + 3 * j, L, half, d) < rn2) s->nb[p++] = (int32_t)j;
    }
    s->max_cell_occ = 0;
}

/* Textbook linked-cell search producing the same sets as build_brute (tests verify that).  The cell of an atom is
 * found in binary64 from its binary32 coordinate, and cells are kept wider than r_n by 1e-5 relative, more than
 * the rounding error of a binary32 r2 (~2e-7), so no accepted pair lies outside the 27-cell stencil. */
static void build_cells(orcs_sys *s)
{
    const int64_t N = s->N;
    const float L = s->Lf, half = s->halff, rn2 = s->rn2f;
    const double Ld = (double)s->Lf, rn = s->rc + s->dr;
    int nc = (int)floor(Ld / rn);
    if (nc >= 1 && Ld / nc - rn < 1e-5 * rn) nc -= 1;
    if (nc < 3 || s->force_brute) { build_brute(s); return; }
    const int64_t NC = (int64_t)nc * nc * nc;
    int32_t *head = (int32_t *)malloc(NC * sizeof(int32_t));
    int32_t *next = (int32_t *)malloc(N * sizeof(int32_t));
    int32_t *occ = (int32_t *)calloc(NC, sizeof(int32_t));
    for (int64_t c = 0; c < NC; c++) head[c] = -1;
    const double inv = nc / Ld;
    for (int64_t i = N - 1; i >= 0; i--) {
        int c[3];
        for (int k = 0; k < 3; k++) {
            int q = (int)floor((double)s->r[3 * i + k] * inv);
            if (q < 0) q = 0;
            if (q >= nc) q = nc - 1;
            c[k] = q;
        }
        int64_t cell = c[0] + (int64_t)nc * (c[1] + (int64_t)nc * c[2]);
        next[i] = head[cell]; head[cell] = (int32_t)i; occ[cell]++;
    }
    int32_t mo = 0;
    for (int64_t c = 0; c < NC; c++) if (occ[c] > mo) mo = occ[c];
    s->max_cell_occ = mo;
    free(occ);

    int64_t *cnt = s->nb_start;
    for (int pass = 0; pass < 2; pass++) {
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < N; i++) {
            int c[3]; float d[3];
            for (int k = 0; k < 3; k++) {
                int q = (int)floor((double)s->r[3 * i + k] * inv);
                if (q < 0) q = 0;
                if (q >= nc) q = nc - 1;
                c[k] = q;
            }
            int64_t p = pass ? cnt[i] : 0;
            for (int dz = -1; dz <= 1; dz++)
                for (int dy = -1; dy <= 1; dy++)
                    for (int dx = -1; dx <= 1; dx++) {
                        int x = (c[0] + dx + nc) % nc, y = (c[1] + dy + nc) % nc, z = (c[2] + dz + nc) % nc;
                        int64_t cell = x + (int64_t)nc * (y + (int64_t)nc * z);
                        for (int32_t j = head[cell]; j >= 0; j = next[j]) {
                            if (j == i) continue;
                            if (dist2f(s->r + 3 * i, s->r + 3 * j, L, half, d) < rn2) {
                                if (pass) s->nb[p] = j;
                                p++;
                            }
                        }
                    }
            if (!pass) cnt[i + 1] = p;
        }
        if (!pass) {
            cnt[0] = 0;
            for (int64_t i = 0; i < N; i++) cnt[i + 1] += cnt[i];
            if (cnt[N] > s->nb_cap) { free(s->nb); s->nb_cap = cnt[N] + cnt[N] / 8 + 16; s->nb = (int32_t *)malloc(s->nb_cap * sizeof(int32_t)); }
        }
    }
    free(head); free(next);
}

/* F1 in binary32; u_i, w_i summed in binary64 */
static void compute_forces(orcs_sys *s)
{
    const int64_t N = s->N;
    const float L = s->Lf, half = s->halff, rc2 = s->rc2f, uc = s->ucf;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; i++) {
        float fx = 0, fy = 0, fz = 0, d[3];
        double ui = 0, wi = 0;
        for (int64_t p = s->nb_start[i]; p < s->nb_start[i + 1]; p++) {
            int64_t j = s->nb[p];
            float r2 = dist2f(s->r + 3 * i, s->r + 3 * j, L, half, d);
            if (r2 < rc2) {
                float sv = 1.0f / r2, s3 = sv * sv * sv;
                float fc = 48.0f * s3 * (s3 - 0.5f) * sv;
                fx += fc * d[0]; fy += fc * d[1]; fz += fc * d[2];
                ui += (double)(4.0f * s3 * (s3 - 1.0f) - uc);
                wi += (double)(fc * r2);
            }
        }
        s->f[3 * i] = fx; s->f[3 * i + 1] = fy; s->f[3 * i + 2] = fz;
        s->u[i] = ui; s->w[i] = wi;
    }
    s->pe_bond = 0; s->vir_bond = 0;
    if (s->n_bonds) {   /* FENE (R12) in binary32, energies summed in binary64 */
        const float k = s->fene_kf, R02 = s->fene_R02f;
        double pe = 0, vr = 0; float d[3];
        for (int64_t b = 0; b < s->n_bonds; b++) {
            int64_t i = s->bonds[2 * b], j = s->bonds[2 * b + 1];
            float r2 = dist2f(s->r + 3 * i, s->r + 3 * j, L, half, d);
            if (!(r2 < R02)) { s->bond_broken = 1; continue; }
            float x = 1.0f - r2 / R02;
            float fc = -k / x;
            for (int q = 0; q < 3; q++) { s->f[3 * i + q] += fc * d[q]; s->f[3 * j + q] -= fc * d[q]; }
            pe += (double)(-0.5f * k * R02 * logf(x));
            vr += (double)(fc * r2);
        }
        s->pe_bond = pe; s->vir_bond = vr;
    }
    /* bond angles (R19) in binary32: the fp64 oracle's formulas, every operation rounded to binary32 */
    s->pe_angle = 0;
    if (s->has_angles) {
        const float k = s->ang_kf, c0 = s->ang_c0f;
        double pe = 0;
        for (int64_t b = 0; b < N; b++) {
            int64_t a = s->partner[b], c = s->partner[N + b];
            if (a < 0 || c < 0) continue;
            float d1[3], d2[3];
            float n1 = dist2f(s->r + 3 * a, s->r + 3 * b, L, half, d1);
            float n2 = dist2f(s->r + 3 * c, s->r + 3 * b, L, half, d2);
            float dot = d1[0] * d2[0] + d1[1] * d2[1] + d1[2] * d2[2];
            float inv12 = 1.0f / sqrtf(n1 * n2);
            float cs = dot * inv12;
            float g = -k * (cs - c0);
            for (int q = 0; q < 3; q++) {
                float fa = g * (d2[q] * inv12 - cs * d1[q] / n1);
                float fc = g * (d1[q] * inv12 - cs * d2[q] / n2);
                s->f[3 * a + q] += fa; s->f[3 * c + q] += fc; s->f[3 * b + q] -= fa + fc;
            }
            pe += (double)(0.5f * k * (cs - c0) * (cs - c0));
        }
        s->pe_angle = pe;
    }
    /* dihedrals (R19) in binary32: the fp64 oracle's formulas, every operation rounded to binary32 */
    s->pe_dihedral = 0;
    if (s->has_dihedrals) {
        const float k = s->dih_kf, c0 = s->dih_c0f;
        double pe = 0;
        for (int64_t q = 0; q < s->n_bonds; q++) {
            int64_t b = s->bonds[2 * q], c = s->bonds[2 * q + 1];
            int64_t a = s->partner[b] == c ? s->partner[N + b] : s->partner[b];
            int64_t d = s->partner[c] == b ? s->partner[N + c] : s->partner[c];
            if (a < 0 || d < 0) continue;
            float b1[3], b2[3], b3[3], A[3], B[3], gA[3], gB[3], g1[3], g2[3], g3[3], t1[3], t2[3];
            dist2f(s->r + 3 * b, s->r + 3 * a, L, half, b1);
            dist2f(s->r + 3 * c, s->r + 3 * b, L, half, b2);
            dist2f(s->r + 3 * d, s->r + 3 * c, L, half, b3);
#define CROSS(o, u, v) do { o[0] = u[1] * v[2] - u[2] * v[1]; o[1] = u[2] * v[0] - u[0] * v[2]; o[2] = u[0] * v[1] - u[1] * v[0]; } while (0)
            CROSS(A, b1, b2); CROSS(B, b2, b3);
            float nA = A[0] * A[0] + A[1] * A[1] + A[2] * A[2], nB = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
            float invAB = 1.0f / sqrtf(nA * nB);
            float cs = (A[0] * B[0] + A[1] * B[1] + A[2] * B[2]) * invAB;
            for (int m = 0; m < 3; m++) { gA[m] = B[m] * invAB - cs * A[m] / nA; gB[m] = A[m] * invAB - cs * B[m] / nB; }
            CROSS(g1, b2, gA); CROSS(t1, gA, b1); CROSS(t2, b3, gB); CROSS(g3, gB, b2);
            for (int m = 0; m < 3; m++) g2[m] = t1[m] + t2[m];
#undef CROSS
            float g = -k * (cs - c0);
            for (int m = 0; m < 3; m++) {
                s->f[3 * a + m] += g * (-g1[m]);
                s->f[3 * b + m] += g * (g1[m] - g2[m]);
                s->f[3 * c + m] += g * (g2[m] - g3[m]);
                s->f[3 * d + m] += g * g3[m];
            }
            pe += (double)(0.5f * k * (cs - c0) * (cs - c0));
        }
        s->pe_dihedral = pe;
    }
}

static void rebuild(orcs_sys *s)
{
    build_cells(s);
    s->disp_acc = 0.0;
    s->n_rebuilds++;
}

void orcs_set_state(orcs_sys *s, const double *xyz, const double *vxyz)
{
    for (int64_t i = 0; i < 3 * s->N; i++) s->r[i] = wrap1f((float)xyz[i], s->Lf);
    if (vxyz) for (int64_t i = 0; i < 3 * s->N; i++) s->v[i] = (float)vxyz[i];
    s->step = 0; s->n_rebuilds = 0; s->bond_broken = 0;
    rebuild(s);
    s->n_rebuilds = 0;
    compute_forces(s);
}

int orcs_set_bonds(orcs_sys *s, int64_t nb, const int32_t *ij, double k, double R0)
{
    free(s->bonds);
    s->bonds = (int32_t *)malloc(2 * nb * sizeof(int32_t));
    memcpy(s->bonds, ij, 2 * nb * sizeof(int32_t));
    s->n_bonds = nb; s->fene_kf = (float)k; s->fene_R02f = (float)(R0 * R0);
    free(s->partner);
    s->partner = (int32_t *)malloc(2 * s->N * sizeof(int32_t));
    for (int64_t i = 0; i < 2 * s->N; i++) s->partner[i] = -1;
    for (int64_t b = 0; b < nb; b++)
        for (int side = 0; side < 2; side++) {
            int32_t a = ij[2 * b + side], c = ij[2 * b + 1 - side];
            if (s->partner[a] < 0) s->partner[a] = c;
            else if (s->partner[s->N + a] < 0) s->partner[s->N + a] = c;
            else return -6;
        }
    compute_forces(s);
    return s->bond_broken ? -3 : 0;
}

int orcs_set_dihedrals(orcs_sys *s, double k, double cos0)
{
    if (!s->partner) return -1;
    s->has_dihedrals = 1; s->dih_kf = (float)k; s->dih_c0f = (float)cos0;
    compute_forces(s);
    return 0;
}

int orcs_set_angles(orcs_sys *s, double k, double cos0)
{
    if (!s->partner) return -1;
    s->has_angles = 1; s->ang_kf = (float)k; s->ang_c0f = (float)cos0;
    compute_forces(s);
    return 0;
}

void orcs_rebuild_neighbors(orcs_sys *s) { rebuild(s); s->n_rebuilds--; compute_forces(s); }

/* half kick, drift, wrap, rebuild test, forces, half kick -- the step of md_oracle.c in binary32;
 * the displacement accumulator and its threshold stay binary64 (scalars) */
int orcs_step(orcs_sys *s, int64_t n)
{
    const int64_t N = s->N;
    const float dt = s->dtf, hdt = s->hdtf, L = s->Lf;
    for (int64_t it = 0; it < n; it++) {
        float vmax2 = 0.0f;
        for (int64_t i = 0; i < N; i++) {
            float vv[3];
            for (int k = 0; k < 3; k++) {
                float vk = s->v[3 * i + k] + hdt * s->f[3 * i + k];
                s->v[3 * i + k] = vk;
                s->r[3 * i + k] = wrap1f(s->r[3 * i + k] + dt * vk, L);
                vv[k] = vk;
            }
            float v2 = vv[0] * vv[0] + vv[1] * vv[1] + vv[2] * vv[2];
            if (v2 > vmax2) vmax2 = v2;
        }
        s->disp_acc += s->dt * sqrt((double)vmax2);
        if (s->disp_acc > 0.5 * s->dr) rebuild(s);
        compute_forces(s);
        for (int64_t i = 0; i < 3 * N; i++) s->v[i] = s->v[i] + hdt * s->f[i];
        s->step++;
        if (s->bond_broken) return -3;
    }
    return 0;
}

/* totals, accumulated in binary64 from the binary32 state */
void orcs_energies(orcs_sys *s, orcs_energy *e)
{
    const int64_t N = s->N;
    double ke = 0, px = 0, py = 0, pz = 0, pe = 0, vir = 0, vmax2 = 0;
    for (int64_t i = 0; i < N; i++) {
        const double vx = s->v[3 * i], vy = s->v[3 * i + 1], vz = s->v[3 * i + 2];
        const double v2 = vx * vx + vy * vy + vz * vz;
        ke += v2; px += vx; py += vy; pz += vz;
        if (v2 > vmax2) vmax2 = v2;
        pe += s->u[i]; vir += s->w[i];
    }
    e->ke = 0.5 * ke;
    e->pe_pair = 0.5 * pe;
    e->pe_bond = s->pe_bond + s->pe_angle + s->pe_dihedral;
    e->virial = 0.5 * vir + s->vir_bond;
    e->px = px; e->py = py; e->pz = pz;
    e->vmax = sqrt(vmax2);
    e->step = s->step; e->n_rebuilds = s->n_rebuilds;
    int64_t mx = 0;
    for (int64_t i = 0; i < N; i++) { int64_t c = s->nb_start[i + 1] - s->nb_start[i]; if (c > mx) mx = c; }
    e->max_neighbors = (int32_t)mx;
    e->max_cell_occupancy = s->max_cell_occ;
    e->mean_neighbors = (double)s->nb_start[N] / (double)N;
}

static void out3(const float *a, int64_t n, double *o) { for (int64_t i = 0; i < 3 * n; i++) o[i] = (double)a[i]; }
void orcs_get_positions(orcs_sys *s, double *xyz) { out3(s->r, s->N, xyz); }
void orcs_get_velocities(orcs_sys *s, double *xyz) { out3(s->v, s->N, xyz); }
void orcs_get_forces(orcs_sys *s, double *xyz) { out3(s->f, s->N, xyz); }
void orcs_get_atom_energies(orcs_sys *s, double *u, double *w)
{
    if (u) memcpy(u, s->u, s->N * sizeof(double));
    if (w) memcpy(w, s->w, s->N * sizeof(double));
}
void orcs_set_velocities(orcs_sys *s, const double *vxyz) { for (int64_t i = 0; i < 3 * s->N; i++) s->v[i] = (float)vxyz[i]; }
int64_t orcs_neighbor_total(orcs_sys *s) { return s->nb_start[s->N]; }
void orcs_get_neighbors(orcs_sys *s, int32_t *counts, int32_t *list)
{
    for (int64_t i = 0; i < s->N; i++) counts[i] = (int32_t)(s->nb_start[i + 1] - s->nb_start[i]);
    if (list) memcpy(list, s->nb, s->nb_start[s->N] * sizeof(int32_t));
}
