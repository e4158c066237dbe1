/*
 * md_oracle.c -- CPU ORACLE for the short-range MD hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct fp64 implementation of what the CUDA path in
 * paper_2003_14061_b200/ computes.  It shares no code with that path and is
 * imported only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs.  The product never routes through it.
 *
 * What it follows (P:<n> = /root/reference/PAPER.md line n; S8c = SURVEY.md 8(c)):
 *   - neighbor set of atom i = the plain definition { j != i : |minimg(r_i - r_j)|^2 < (r_c + delta)^2 }.
 *     The paper's neighbor matrix W (step N5) tabulates exactly this set ("shell thickness"
 *     delta); the cell/layer machinery (N1-N4) is only a faster way to reach
 *     it, so the oracle is the definition: O(N^2) brute force, plus a textbook linked-cell search
 *     for larger N that the tests verify against the brute force.
 *   - forces (F1): for every listed neighbor within interaction range accumulate f_i and u_i;
 *     pairs are visited twice, Newton's third law is not used.  PAPER.md has no equations
 *     (it defers to refs [1],[2]); the potential is the textbook Lennard-Jones form truncated at r_c
 *     and energy-shifted (readings R1, R2).
 *   - total interaction energy = half the sum of u_i ("actually 2U", step F2).
 *   - integration: two-half-kick leapfrog / velocity Verlet with periodic wrap (
 *     DESIGN.md reading R3).
 *   - rebuild rule: decided from the maximal atom velocity: accumulate dt * max|v| and
 *     rebuild when it exceeds delta/2 (reading R8).
 *   - bonds (polymer chains): FENE bond force between chain neighbours (R12).
 *   - bond angles ("bond-angle torque"): PAPER.md gives no form; the textbook
 *     cosine-harmonic U = k/2 (cos(theta) - cos(theta0))^2 at every atom with two bonded partners
 *     (reading R19), forces by the chain rule on cos(theta) = d1.d2 / (|d1||d2|).
 *   - dihedral terms ("optional dihedral"): U = k/2 (cos(phi) - cos(phi0))^2 for every four consecutive
 *     beads, cos(phi) = A.B/(|A||B|), A = b1 x b2, B = b2 x b3 (R19); forces by the chain rule through A, B.
 *
 * Parity pins for every function here live in tests/test_oracle_pins.py (brute force on tiny
 * inputs, closed forms on the SC/FCC lattices, two-atom values, conservation laws, reversibility,
 * dt^2 scaling, symmetries).  Unpinned by the paper: the absolute energy-drift bound (R17) and the
 * chain initial state -- see DESIGN.md.
 *
 * Plain C11.  Per-atom loops carry an OpenMP pragma so the oracle can be timed on all host cores;
 * the pragma does not change any per-atom arithmetic (full list, no shared accumulators).
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
} orc_energy;

typedef struct orc_sys {
    int64_t N;
    double L, rc, dr, dt;
    double rc2, rn2, uc;
    double *r, *v, *f;      /* N x 3 */
    double *u, *w;          /* per-atom pair energy u_i and virial w_i (both double counted) */
    /* neighbor list: CSR, full (each pair twice) */
    int64_t *nb_start;      /* N+1 */
    int32_t *nb;            /* nb_start[N] */
    int64_t nb_cap;
    /* bonds */
    int64_t n_bonds;
    int32_t *bonds;         /* 2 x n_bonds */
    double fene_k, fene_R0;
    double pe_bond, vir_bond;
    int bond_broken;
    /* bond angles: partner table built from the bond list (-1 = none), potential constants */
    int32_t *partner;       /* 2 x N */
    int has_angles;
    double ang_k, ang_c0, pe_angle;
    int has_dihedrals;
    double dih_k, dih_c0, pe_dihedral;
    /* bookkeeping */
    double disp_acc;
    int64_t step, n_rebuilds;
    int32_t max_cell_occ;
    int force_brute;        /* 1: always use the O(N^2) neighbor search */
} orc_sys;

/* ---- minimum image, P:163 ("periodic boundaries"), S8c O3 ------------------------------- */
static inline double minimg(double d, double L, double half)
{
    if (d > half) d -= L;
    else if (d < -half) d += L;
    return d;
}

/* squared distance with a fixed, IEEE-exact operation order (reading R5) */
static inline double dist2(const double *a, const double *b, double L, double half, double d[3])
{
    d[0] = minimg(a[0] - b[0], L, half);
    d[1] = minimg(a[1] - b[1], L, half);
    d[2] = minimg(a[2] - b[2], L, half);
    return fma(d[2], d[2], fma(d[1], d[1], d[0] * d[0]));
}

void orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_get_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- stand-alone definitions (used as pins and for sampled checks at full size) ---------- */

/* all-pairs truncated-shifted LJ, S8c O4.  f: N x 3, u,w: N (double counted per atom). */
void orc_brute_forces(int64_t N, double L, const double *r, double rc, double *f, double *u, double *w)
{
    const double half = 0.5 * L, rc2 = rc * rc;
    const double sc = 1.0 / rc2, sc3 = sc * sc * sc, uc = 4.0 * sc3 * (sc3 - 1.0);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; i++) {
        double fx = 0, fy = 0, fz = 0, ui = 0, wi = 0, d[3];
        for (int64_t j = 0; j < N; j++) {
            if (j == i) continue;
            double r2 = dist2(r + 3 * i, r + 3 * j, L, half, d);
            if (r2 < rc2) {
                double s = 1.0 / r2, s3 = s * s * s;
                double fc = 48.0 * s3 * (s3 - 0.5) * s;
                fx += fc * d[0]; fy += fc * d[1]; fz += fc * d[2];
                ui += 4.0 * s3 * (s3 - 1.0) - uc;
                wi += fc * r2;
            }
        }
        f[3 * i] = fx; f[3 * i + 1] = fy; f[3 * i + 2] = fz;
        if (u) u[i] = ui;
        if (w) w[i] = wi;
    }
}

/* the same sum for a sample of atoms only: O(N) per sampled atom */
void orc_brute_forces_sample(int64_t N, double L, const double *r, double rc, int64_t ns,
                             const int64_t *idx, double *f, double *u, double *w)
{
    const double half = 0.5 * L, rc2 = rc * rc;
    const double sc = 1.0 / rc2, sc3 = sc * sc * sc, uc = 4.0 * sc3 * (sc3 - 1.0);
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < ns; k++) {
        int64_t i = idx[k];
        double fx = 0, fy = 0, fz = 0, ui = 0, wi = 0, d[3];
        for (int64_t j = 0; j < N; j++) {
            if (j == i) continue;
            double r2 = dist2(r + 3 * i, r + 3 * j, L, half, d);
            if (r2 < rc2) {
                double s = 1.0 / r2, s3 = s * s * s;
                double fc = 48.0 * s3 * (s3 - 0.5) * s;
                fx += fc * d[0]; fy += fc * d[1]; fz += fc * d[2];
                ui += 4.0 * s3 * (s3 - 1.0) - uc;
                wi += fc * r2;
            }
        }
        f[3 * k] = fx; f[3 * k + 1] = fy; f[3 * k + 2] = fz;
        if (u) u[k] = ui;
        if (w) w[k] = wi;
    }
}

/* neighbor set by definition for a sample of atoms.  out: ns x cap (ascending j, -1 padded),
 * counts: ns.  Returns the largest count (may exceed cap: then rows are truncated). */
int32_t orc_brute_neighbors_sample(int64_t N, double L, const double *r, double rn, int64_t ns,
                                   const int64_t *idx, int32_t cap, int32_t *counts, int32_t *out)
{
    const double half = 0.5 * L, rn2 = rn * rn;
    int32_t mx = 0;
#pragma omp parallel for schedule(static) reduction(max : mx)
    for (int64_t k = 0; k < ns; k++) {
        int64_t i = idx[k];
        int32_t c = 0;
        double d[3];
        for (int64_t j = 0; j < N; j++) {
            if (j == i) continue;
            if (dist2(r + 3 * i, r + 3 * j, L, half, d) < rn2) {
                if (c < cap) out[k * cap + c] = (int32_t)j;
                c++;
            }
        }
        for (int32_t m = c; m < cap; m++) out[k * cap + m] = -1;
        counts[k] = c;
        if (c > mx) mx = c;
    }
    return mx;
}

/* ---- system ------------------------------------------------------------------------------- */

orc_sys *orc_create(int64_t N, double L, double rc, double dr, double dt)
{
    if (N <= 0 || L <= 0 || rc <= 0 || dr < 0 || dt <= 0) return NULL;
    orc_sys *s = (orc_sys *)calloc(1, sizeof(orc_sys));
    s->N = N; s->L = L; s->rc = rc; s->dr = dr; s->dt = dt;
    s->rc2 = rc * rc;
    double rn = rc + dr;
    s->rn2 = rn * rn;
    double sc = 1.0 / s->rc2, sc3 = sc * sc * sc;
    s->uc = 4.0 * sc3 * (sc3 - 1.0);
    s->r = (double *)calloc(3 * N, sizeof(double));
    s->v = (double *)calloc(3 * N, sizeof(double));
    s->f = (double *)calloc(3 * N, sizeof(double));
    s->u = (double *)calloc(N, sizeof(double));
    s->w = (double *)calloc(N, sizeof(double));
    s->nb_start = (int64_t *)calloc(N + 1, sizeof(int64_t));
    return s;
}

void orc_destroy(orc_sys *s)
{
    if (!s) return;
    free(s->r); free(s->v); free(s->f); free(s->u); free(s->w);
    free(s->nb_start); free(s->nb); free(s->bonds); free(s->partner);
    free(s);
}

void orc_force_brute_search(orc_sys *s, int on) { s->force_brute = on; }

/* neighbor sets by definition, O(N^2) */
static void build_brute(orc_sys *s)
{
    const int64_t N = s->N;
    const double L = s->L, half = 0.5 * L, rn2 = s->rn2;
    int64_t *cnt = s->nb_start;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; i++) {
        int64_t c = 0; double d[3];
        for (int64_t j = 0; j < N; j++)
            if (j != i && dist2(s->r + 3 * i, s->r + 3 * j, L, half, d) < rn2) c++;
        cnt[i + 1] = c;
    }
    cnt[0] = 0;
    for (int64_t i = 0; i < N; i++) cnt[i + 1] += cnt[i];
    if (cnt[N] > s->nb_cap) { free(s->nb); s->nb_cap = cnt[N] + cnt[N] / 8 + 16; s->nb = (int32_t *)malloc(s->nb_cap * sizeof(int32_t)); }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; i++) {
        int64_t p = cnt[i]; double d[3];
        for (int64_t j = 0; j < N; j++)
            if (j != i && dist2(s->r + 3 * i, s->r + 3 * j, L, half, d) < rn2) s->nb[p++] = (int32_t)j;
    }
    s->max_cell_occ = 0;
}

/* textbook linked-cell search (cells of width >= r_n, 27-cell periodic stencil, P:49-53 N1/N5).
 * Produces the same sets as build_brute; tests verify that. */
static void build_cells(orc_sys *s)
{
    const int64_t N = s->N;
    const double L = s->L, half = 0.5 * L, rn2 = s->rn2, rn = s->rc + s->dr;
    int nc = (int)floor(L / rn);
    if (nc < 3 || s->force_brute) { build_brute(s); return; }
    const double w = L / nc;
    if (w - rn < 1e-9 * rn) { nc -= 1; if (nc < 3) { build_brute(s); return; } }
    const int64_t NC = (int64_t)nc * nc * nc;
    int32_t *head = (int32_t *)malloc(NC * sizeof(int32_t));
    int32_t *next = (int32_t *)malloc(N * sizeof(int32_t));
    int32_t *occ = (int32_t *)calloc(NC, sizeof(int32_t));
    for (int64_t c = 0; c < NC; c++) head[c] = -1;
    const double inv = nc / L;
    for (int64_t i = N - 1; i >= 0; i--) {   /* reverse so each cell's chain is ascending in i */
        int c[3];
        for (int k = 0; k < 3; k++) {
            int q = (int)floor(s->r[3 * i + k] * inv);
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
            int c[3]; double d[3];
            for (int k = 0; k < 3; k++) {
                int q = (int)floor(s->r[3 * i + k] * inv);
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
                            if (dist2(s->r + 3 * i, s->r + 3 * j, L, half, d) < rn2) {
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

/* F1: per atom, over its listed neighbors, those within interaction range. */
static void compute_forces(orc_sys *s)
{
    const int64_t N = s->N;
    const double L = s->L, half = 0.5 * L, rc2 = s->rc2, uc = s->uc;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; i++) {
        double fx = 0, fy = 0, fz = 0, ui = 0, wi = 0, d[3];
        for (int64_t p = s->nb_start[i]; p < s->nb_start[i + 1]; p++) {
            int64_t j = s->nb[p];
            double r2 = dist2(s->r + 3 * i, s->r + 3 * j, L, half, d);
            if (r2 < rc2) {
                double sv = 1.0 / r2, s3 = sv * sv * sv;
                double fc = 48.0 * s3 * (s3 - 0.5) * sv;
                fx += fc * d[0]; fy += fc * d[1]; fz += fc * d[2];
                ui += 4.0 * s3 * (s3 - 1.0) - uc;
                wi += fc * r2;
            }
        }
        s->f[3 * i] = fx; s->f[3 * i + 1] = fy; s->f[3 * i + 2] = fz;
        s->u[i] = ui; s->w[i] = wi;
    }
    /* bonds (S8c O5): serial, each bond once, both ends updated */
    s->pe_bond = 0; s->vir_bond = 0;
    if (s->n_bonds) {
        const double k = s->fene_k, R02 = s->fene_R0 * s->fene_R0;
        double pe = 0, pc = 0, vr = 0, vc = 0, d[3];
        for (int64_t b = 0; b < s->n_bonds; b++) {
            int64_t i = s->bonds[2 * b], j = s->bonds[2 * b + 1];
            double r2 = dist2(s->r + 3 * i, s->r + 3 * j, L, half, d);
            if (!(r2 < R02)) { s->bond_broken = 1; continue; }
            double fc = -k / (1.0 - r2 / R02);
            for (int q = 0; q < 3; q++) { s->f[3 * i + q] += fc * d[q]; s->f[3 * j + q] -= fc * d[q]; }
            double e = -0.5 * k * R02 * log(1.0 - r2 / R02), t;
            /* Neumaier sums */
            t = pe + e; pc += (fabs(pe) >= fabs(e)) ? (pe - t) + e : (e - t) + pe; pe = t;
            double x = fc * r2;
            t = vr + x; vc += (fabs(vr) >= fabs(x)) ? (vr - t) + x : (x - t) + vr; vr = t;
        }
        s->pe_bond = pe + pc; s->vir_bond = vr + vc;
    }
    /* bond angles (R19): vertex b with partners a, c; d1 = r_a - r_b, d2 = r_c - r_b (minimum image);
     * c = d1.d2 / (|d1||d2|); U = k/2 (c - c0)^2; f_a = -dU/dc dc/dr_a, dc/dr_a = d2/(|d1||d2|) - c d1/|d1|^2;
     * f_c likewise with 1 <-> 2; f_b = -(f_a + f_c).  cos(theta) is scale invariant: no virial contribution. */
    s->pe_angle = 0;
    if (s->has_angles) {
        double pe = 0;
        for (int64_t b = 0; b < N; b++) {
            int64_t a = s->partner[b], c = s->partner[N + b];
            if (a < 0 || c < 0) continue;
            double d1[3], d2[3];
            double n1 = dist2(s->r + 3 * a, s->r + 3 * b, L, half, d1);
            double n2 = dist2(s->r + 3 * c, s->r + 3 * b, L, half, d2);
            double dot = d1[0] * d2[0] + d1[1] * d2[1] + d1[2] * d2[2];
            double inv12 = 1.0 / sqrt(n1 * n2);
            double cs = dot * inv12;
            double g = -s->ang_k * (cs - s->ang_c0);          /* -dU/dc */
            for (int q = 0; q < 3; q++) {
                double fa = g * (d2[q] * inv12 - cs * d1[q] / n1);
                double fc = g * (d1[q] * inv12 - cs * d2[q] / n2);
                s->f[3 * a + q] += fa; s->f[3 * c + q] += fc; s->f[3 * b + q] -= fa + fc;
            }
            pe += 0.5 * s->ang_k * (cs - s->ang_c0) * (cs - s->ang_c0);
        }
        s->pe_angle = pe;
    }
    /* dihedrals (R19): one per bond (b, c) whose ends both continue: a - b - c - d.
     * b1 = r_b - r_a, b2 = r_c - r_b, b3 = r_d - r_c (minimum image); A = b1 x b2, B = b2 x b3; c = A.B/(|A||B|).
     * gA = dc/dA = B/(|A||B|) - c A/|A|^2, gB likewise; dc/db1 = b2 x gA, dc/db2 = gA x b1 + b3 x gB, dc/db3 = gB x b2;
     * dc/dr_a = -dc/db1, dc/dr_b = dc/db1 - dc/db2, dc/dr_c = dc/db2 - dc/db3, dc/dr_d = dc/db3;  f = -k (c - c0) dc/dr. */
    s->pe_dihedral = 0;
    if (s->has_dihedrals) {
        double pe = 0;
        for (int64_t q = 0; q < s->n_bonds; q++) {
            int64_t b = s->bonds[2 * q], c = s->bonds[2 * q + 1];
            int64_t a = s->partner[b] == c ? s->partner[N + b] : s->partner[b];
            int64_t d = s->partner[c] == b ? s->partner[N + c] : s->partner[c];
            if (a < 0 || d < 0) continue;
            double b1[3], b2[3], b3[3], A[3], B[3], gA[3], gB[3], g1[3], g2[3], g3[3], t1[3], t2[3];
            dist2(s->r + 3 * b, s->r + 3 * a, L, half, b1);
            dist2(s->r + 3 * c, s->r + 3 * b, L, half, b2);
            dist2(s->r + 3 * d, s->r + 3 * c, L, half, b3);
#define CROSS(o, u, v) do { o[0] = u[1] * v[2] - u[2] * v[1]; o[1] = u[2] * v[0] - u[0] * v[2]; o[2] = u[0] * v[1] - u[1] * v[0]; } while (0)
            CROSS(A, b1, b2); CROSS(B, b2, b3);
            double nA = A[0] * A[0] + A[1] * A[1] + A[2] * A[2], nB = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
            double invAB = 1.0 / sqrt(nA * nB);
            double cs = (A[0] * B[0] + A[1] * B[1] + A[2] * B[2]) * invAB;
            for (int k = 0; k < 3; k++) { gA[k] = B[k] * invAB - cs * A[k] / nA; gB[k] = A[k] * invAB - cs * B[k] / nB; }
            CROSS(g1, b2, gA);                       /* dc/db1 */
            CROSS(t1, gA, b1); CROSS(t2, b3, gB);    /* dc/db2 = t1 + t2 */
            CROSS(g3, gB, b2);                       /* dc/db3 */
            for (int k = 0; k < 3; k++) g2[k] = t1[k] + t2[k];
#undef CROSS
            double g = -s->dih_k * (cs - s->dih_c0);
            for (int k = 0; k < 3; k++) {
                s->f[3 * a + k] += g * (-g1[k]);
                s->f[3 * b + k] += g * (g1[k] - g2[k]);
                s->f[3 * c + k] += g * (g2[k] - g3[k]);
                s->f[3 * d + k] += g * g3[k];
            }
            pe += 0.5 * s->dih_k * (cs - s->dih_c0) * (cs - s->dih_c0);
        }
        s->pe_dihedral = pe;
    }
}

static void rebuild(orc_sys *s)
{
    build_cells(s);
    s->disp_acc = 0.0;
    s->n_rebuilds++;
}

/* load a state (xyz, vxyz: N x 3), build the neighbor sets and evaluate forces */
void orc_set_state(orc_sys *s, const double *xyz, const double *vxyz)
{
    memcpy(s->r, xyz, 3 * s->N * sizeof(double));
    if (vxyz) memcpy(s->v, vxyz, 3 * s->N * sizeof(double));
    s->step = 0; s->n_rebuilds = 0; s->bond_broken = 0;
    rebuild(s);
    s->n_rebuilds = 0;
    compute_forces(s);
}

int orc_set_bonds(orc_sys *s, int64_t nb, const int32_t *ij, double k, double R0)
{
    free(s->bonds);
    s->bonds = (int32_t *)malloc(2 * nb * sizeof(int32_t));
    memcpy(s->bonds, ij, 2 * nb * sizeof(int32_t));
    s->n_bonds = nb; s->fene_k = k; s->fene_R0 = R0;
    /* partner table (at most 2 per atom: linear chains) */
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

/* dihedral terms for every four consecutive bonded atoms; call after orc_set_bonds */
int orc_set_dihedrals(orc_sys *s, double k, double cos0)
{
    if (!s->partner) return -1;
    s->has_dihedrals = 1; s->dih_k = k; s->dih_c0 = cos0;
    compute_forces(s);
    return 0;
}

/* bond-angle terms at every atom with two bonded partners; call after orc_set_bonds */
int orc_set_angles(orc_sys *s, double k, double cos0)
{
    if (!s->partner) return -1;
    s->has_angles = 1; s->ang_k = k; s->ang_c0 = cos0;
    compute_forces(s);
    return 0;
}

void orc_rebuild_neighbors(orc_sys *s) { rebuild(s); s->n_rebuilds--; compute_forces(s); }

static inline double wrap1(double x, double L)
{
    if (x >= L) x -= L;
    else if (x < 0.0) { x += L; if (x >= L) x = 0.0; }
    return x;
}

/* S8c O6/O7: half kick, drift, wrap, rebuild test, forces, half kick */
int orc_step(orc_sys *s, int64_t n)
{
    const int64_t N = s->N;
    const double dt = s->dt, hdt = 0.5 * s->dt, L = s->L;
    for (int64_t it = 0; it < n; it++) {
        double vmax2 = 0.0;
        for (int64_t i = 0; i < N; i++) {
            double v2 = 0.0;
            for (int k = 0; k < 3; k++) {
                double vk = s->v[3 * i + k] + hdt * s->f[3 * i + k];
                s->v[3 * i + k] = vk;
                s->r[3 * i + k] = wrap1(s->r[3 * i + k] + dt * vk, L);
                v2 += vk * vk;
            }
            if (v2 > vmax2) vmax2 = v2;
        }
        s->disp_acc += dt * sqrt(vmax2);
        if (s->disp_acc > 0.5 * s->dr) rebuild(s);
        compute_forces(s);
        for (int64_t i = 0; i < 3 * N; i++) s->v[i] += hdt * s->f[i];
        s->step++;
        if (s->bond_broken) return -3;
    }
    return 0;
}

static double nsum(const double *x, int64_t n, int64_t stride)
{
    double sum = 0.0, c = 0.0;
    for (int64_t i = 0; i < n; i++) {
        double xi = x[i * stride], t = sum + xi;
        c += (fabs(sum) >= fabs(xi)) ? (sum - t) + xi : (xi - t) + sum;
        sum = t;
    }
    return sum + c;
}

/* S8c O8: totals */
void orc_energies(orc_sys *s, orc_energy *e)
{
    const int64_t N = s->N;
    double *v2 = (double *)malloc(N * sizeof(double));
    double vmax2 = 0.0;
    for (int64_t i = 0; i < N; i++) {
        const double *v = s->v + 3 * i;
        v2[i] = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
        if (v2[i] > vmax2) vmax2 = v2[i];
    }
    e->ke = 0.5 * nsum(v2, N, 1);
    free(v2);
    e->pe_pair = 0.5 * nsum(s->u, N, 1);
    e->pe_bond = s->pe_bond + s->pe_angle + s->pe_dihedral;      /* bonded energy: FENE + angle + dihedral terms */
    e->virial = 0.5 * nsum(s->w, N, 1) + s->vir_bond;
    e->px = nsum(s->v, N, 3); e->py = nsum(s->v + 1, N, 3); e->pz = nsum(s->v + 2, N, 3);
    e->vmax = sqrt(vmax2);
    e->step = s->step; e->n_rebuilds = s->n_rebuilds;
    int64_t mx = 0;
    for (int64_t i = 0; i < N; i++) { int64_t c = s->nb_start[i + 1] - s->nb_start[i]; if (c > mx) mx = c; }
    e->max_neighbors = (int32_t)mx;
    e->max_cell_occupancy = s->max_cell_occ;
    e->mean_neighbors = (double)s->nb_start[N] / (double)N;
}

void orc_get_positions(orc_sys *s, double *xyz) { memcpy(xyz, s->r, 3 * s->N * sizeof(double)); }
void orc_get_velocities(orc_sys *s, double *xyz) { memcpy(xyz, s->v, 3 * s->N * sizeof(double)); }
void orc_get_forces(orc_sys *s, double *xyz) { memcpy(xyz, s->f, 3 * s->N * sizeof(double)); }
void orc_get_atom_energies(orc_sys *s, double *u, double *w)
{
    if (u) memcpy(u, s->u, s->N * sizeof(double));
    if (w) memcpy(w, s->w, s->N * sizeof(double));
}
void orc_set_velocities(orc_sys *s, const double *vxyz) { memcpy(s->v, vxyz, 3 * s->N * sizeof(double)); }

int64_t orc_neighbor_total(orc_sys *s) { return s->nb_start[s->N]; }

/* counts: N; list: nb_total entries, CSR order (row i = neighbors of atom i) */
void orc_get_neighbors(orc_sys *s, int32_t *counts, int32_t *list)
{
    for (int64_t i = 0; i < s->N; i++) counts[i] = (int32_t)(s->nb_start[i + 1] - s->nb_start[i]);
    if (list) memcpy(list, s->nb, s->nb_start[s->N] * sizeof(int32_t));
}
