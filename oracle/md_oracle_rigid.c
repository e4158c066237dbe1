/*
 * md_oracle_rigid.c -- CPU ORACLE for rigid molecules on the short-range MD path.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow fp64 C; shares no code with paper_2003_14061_b200/ and is imported only by tests/.
 *
 * What it follows (P:<n> = /root/reference/PAPER.md line n; reading R20):
 *   P:183-185, sec. 4.3(1): "Modeling molecules based on rigid bodies with multiple interaction sites follows directly
 *   from the basic method ... e.g., four SP spheres in a rigid tetrahedral configuration ... Spatial orientation can be
 *   described ... as quaternions or (as used here) rotation matrices [1].  Integration of the rotational equations of
 *   motion employs a generalization of the symplectic leapfrog technique."  The paper prints no equations and ref. [1]
 *   is not in the container, so the model is written from textbook forms (R20):
 *     - a molecule = n_s unit-mass sites at fixed body-frame positions b_k (centre of mass at the origin, axes = the
 *       principal axes: the inertia tensor sum_k (|b_k|^2 1 - b_k b_k^T) is diagonal, moments I_1..3 > 0);
 *     - state per molecule: centre of mass R, its velocity V, rotation matrix A (body -> space: site k sits at
 *       R + A b_k) and the angular momentum pi in the BODY frame;
 *     - sites of DIFFERENT molecules interact through the truncated, energy-shifted Lennard-Jones potential of the
 *       atomic path (R1, R2); molecule force F = sum_k f_k, torque (space frame) T = sum_k (A b_k) x f_k;
 *     - integration: two half kicks around a drift, as for atoms (R3), with the free rotation over dt done by the
 *       symplectic splitting of the free rigid rotor into rotations about the body axes,
 *           Rx(dt/2) Ry(dt/2) Rz(dt) Ry(dt/2) Rx(dt/2),
 *       each a rotation of (pi, A) by the angle h pi_k / I_k about body axis k (Dullweber, Leimkuhler, McLachlan 1997;
 *       Leimkuhler & Reich, "Simulating Hamiltonian Dynamics", ch. 8) -- a rotation-matrix generalisation of leapfrog:
 *       explicit, time-reversible, conserves |A pi| exactly;
 *     - neighbor set of site i = { sites j of OTHER molecules with |minimg(r_i - r_j)|^2 < (r_c + delta)^2 } (the
 *       definition; found by brute force), rebuilt by the rule of R8 with a rigorous bound on the largest site speed:
 *       |V| + |pi| / I_min * max_k |b_k|  (|pi| is conserved by the free rotation), taken after the first half kick.
 *
 * Pins: tests/test_oracle_rigid_pins.py (force / torque = minus the gradient of an independent numpy energy, zero net
 * force, a torque-free asymmetric top conserves angular momentum and -- to O(dt^2) -- energy, A stays orthonormal,
 * reversibility, dt^2 scaling of the energy error, the symmetric top's precession rate).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double ke_trans, ke_rot, pe, virial, px, py, pz, vbound;
    double lx, ly, lz;          /* total angular momentum about the origin is not conserved under periodic wrap; this is sum_m A pi */
    int64_t step, n_rebuilds;
    int32_t max_neighbors;
    double mean_neighbors;
} orr_energy;

typedef struct orr_sys {
    int64_t nm;
    int ns;
    double L, rc, dr, dt, rc2, rn2, uc;
    double *b;                  /* ns x 3 */
    double I[3], M, bmax, Imin;
    double *R, *V, *A, *pi;     /* nm x 3, nm x 3, nm x 9 (row-major), nm x 3 */
    double *site, *fs, *u, *w;  /* per site: wrapped position (x3), force (x3), pair energy, pair virial (double counted) */
    double *F, *T;              /* per molecule: force, torque in the space frame */
    int64_t *nb_start;
    int32_t *nb;
    int64_t nb_cap;
    double disp_acc;
    int64_t step, n_rebuilds;
} orr_sys;

static double minimg(double d, double L, double half)
{
    if (d > half) d -= L;
    else if (d < -half) d += L;
    return d;
}

static double wrap(double x, double L)
{
    x -= L * floor(x / L);
    if (x >= L) x = 0.0;
    if (x < 0.0) x = 0.0;
    return x;
}

/* site k of molecule m: R + A b_k, wrapped into the box */
static void place_sites(orr_sys *s)
{
    for (int64_t m = 0; m < s->nm; m++) {
        const double *A = s->A + 9 * m, *R = s->R + 3 * m;
        for (int k = 0; k < s->ns; k++) {
            const double *b = s->b + 3 * k;
            double *x = s->site + 3 * (m * s->ns + k);
            for (int c = 0; c < 3; c++) x[c] = wrap(R[c] + (A[3 * c] * b[0] + A[3 * c + 1] * b[1] + A[3 * c + 2] * b[2]), s->L);
        }
    }
}

static void build_list(orr_sys *s)
{
    const int64_t N = s->nm * s->ns;
    const double L = s->L, half = 0.5 * L;
    int64_t *cnt = s->nb_start;
    for (int pass = 0; pass < 2; pass++) {
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < N; i++) {
            int64_t n = 0, p = pass ? s->nb_start[i] : 0;
            for (int64_t j = 0; j < N; j++) {
                if (j / s->ns == i / s->ns) continue;       /* sites of one molecule do not interact */
                const double dx = minimg(s->site[3 * i] - s->site[3 * j], L, half), dy = minimg(s->site[3 * i + 1] - s->site[3 * j + 1], L, half),
                             dz = minimg(s->site[3 * i + 2] - s->site[3 * j + 2], L, half);
                if (fma(dz, dz, fma(dy, dy, dx * dx)) < s->rn2) {
                    if (pass) s->nb[p++] = (int32_t)j;
                    n++;
                }
            }
            if (!pass) cnt[i + 1] = n;
        }
        if (!pass) {
            cnt[0] = 0;
            for (int64_t i = 0; i < N; i++) cnt[i + 1] += cnt[i];
            if (cnt[N] > s->nb_cap) {
                free(s->nb);
                s->nb_cap = cnt[N] + cnt[N] / 4 + 16;
                s->nb = (int32_t *)malloc(sizeof(int32_t) * (size_t)s->nb_cap);
            }
        }
    }
}

static void forces(orr_sys *s)
{
    const int64_t N = s->nm * s->ns;
    const double L = s->L, half = 0.5 * L;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; i++) {
        double fx = 0, fy = 0, fz = 0, u = 0, w = 0;
        for (int64_t q = s->nb_start[i]; q < s->nb_start[i + 1]; q++) {
            const int64_t j = s->nb[q];
            const double dx = minimg(s->site[3 * i] - s->site[3 * j], L, half), dy = minimg(s->site[3 * i + 1] - s->site[3 * j + 1], L, half),
                         dz = minimg(s->site[3 * i + 2] - s->site[3 * j + 2], L, half);
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            if (r2 < s->rc2) {
                const double si = 1.0 / r2, s3 = si * si * si;
                const double fc = 48.0 * s3 * (s3 - 0.5) * si;
                fx += fc * dx; fy += fc * dy; fz += fc * dz;
                u += 4.0 * s3 * (s3 - 1.0) - s->uc;
                w += fc * r2;
            }
        }
        s->fs[3 * i] = fx; s->fs[3 * i + 1] = fy; s->fs[3 * i + 2] = fz;
        s->u[i] = u; s->w[i] = w;
    }
    for (int64_t m = 0; m < s->nm; m++) {
        const double *A = s->A + 9 * m;
        double F[3] = {0, 0, 0}, T[3] = {0, 0, 0};
        for (int k = 0; k < s->ns; k++) {
            const double *b = s->b + 3 * k, *f = s->fs + 3 * (m * s->ns + k);
            double a[3];                                   /* lever arm A b_k */
            for (int c = 0; c < 3; c++) a[c] = A[3 * c] * b[0] + A[3 * c + 1] * b[1] + A[3 * c + 2] * b[2];
            for (int c = 0; c < 3; c++) F[c] += f[c];
            T[0] += a[1] * f[2] - a[2] * f[1];
            T[1] += a[2] * f[0] - a[0] * f[2];
            T[2] += a[0] * f[1] - a[1] * f[0];
        }
        memcpy(s->F + 3 * m, F, sizeof(F));
        memcpy(s->T + 3 * m, T, sizeof(T));
    }
}

/* V += h F / M;  pi += h A^T T */
static void kick(orr_sys *s, double h)
{
    for (int64_t m = 0; m < s->nm; m++) {
        const double *A = s->A + 9 * m, *T = s->T + 3 * m;
        for (int c = 0; c < 3; c++) s->V[3 * m + c] += h * s->F[3 * m + c] / s->M;
        for (int c = 0; c < 3; c++) s->pi[3 * m + c] += h * (A[c] * T[0] + A[3 + c] * T[1] + A[6 + c] * T[2]);
    }
}

/* free rotation about body axis k for time h: angle phi = h pi_k / I_k;  pi <- R_k(-phi) pi,  A <- A R_k(phi).
 * With (k, a, c) cyclic: pi_a' = cos pi_a + sin pi_c, pi_c' = -sin pi_a + cos pi_c; columns A_a' = cos A_a + sin A_c, A_c' = -sin A_a + cos A_c. */
static void rotate_axis(orr_sys *s, int64_t m, int k, double h)
{
    double *pi = s->pi + 3 * m, *A = s->A + 9 * m;
    const int a = (k + 1) % 3, c = (k + 2) % 3;
    const double phi = h * pi[k] / s->I[k], cs = cos(phi), sn = sin(phi);
    const double pa = pi[a], pc = pi[c];
    pi[a] = cs * pa + sn * pc;
    pi[c] = -sn * pa + cs * pc;
    for (int r = 0; r < 3; r++) {
        const double Aa = A[3 * r + a], Ac = A[3 * r + c];
        A[3 * r + a] = cs * Aa + sn * Ac;
        A[3 * r + c] = -sn * Aa + cs * Ac;
    }
}

static double speed_bound(const orr_sys *s, int64_t m)
{
    const double *V = s->V + 3 * m, *pi = s->pi + 3 * m;
    return sqrt(V[0] * V[0] + V[1] * V[1] + V[2] * V[2]) + sqrt(pi[0] * pi[0] + pi[1] * pi[1] + pi[2] * pi[2]) / s->Imin * s->bmax;
}

orr_sys *orr_create(int64_t nm, int ns, const double *body, double L, double rc, double dr, double dt)
{
    if (nm < 1 || ns < 1) return NULL;
    orr_sys *s = (orr_sys *)calloc(1, sizeof(orr_sys));
    s->nm = nm; s->ns = ns; s->L = L; s->rc = rc; s->dr = dr; s->dt = dt;
    s->rc2 = rc * rc; s->rn2 = (rc + dr) * (rc + dr);
    { const double sc = 1.0 / s->rc2, sc3 = sc * sc * sc; s->uc = 4.0 * sc3 * (sc3 - 1.0); }
    s->b = (double *)malloc(sizeof(double) * 3 * ns);
    memcpy(s->b, body, sizeof(double) * 3 * ns);
    double I[3][3] = {{0}}, com[3] = {0, 0, 0};
    s->M = (double)ns;
    s->bmax = 0.0;
    for (int k = 0; k < ns; k++) {
        const double *b = body + 3 * k, b2 = b[0] * b[0] + b[1] * b[1] + b[2] * b[2];
        for (int c = 0; c < 3; c++) com[c] += b[c];
        if (sqrt(b2) > s->bmax) s->bmax = sqrt(b2);
        for (int r = 0; r < 3; r++)
            for (int c = 0; c < 3; c++) I[r][c] += (r == c ? b2 : 0.0) - b[r] * b[c];
    }
    const double tol = 1e-12 * (I[0][0] + I[1][1] + I[2][2] + 1.0);
    int bad = fabs(com[0]) + fabs(com[1]) + fabs(com[2]) > 1e-12 * ns * (s->bmax + 1.0);
    for (int r = 0; r < 3; r++)
        for (int c = 0; c < 3; c++)
            if (r != c && fabs(I[r][c]) > tol) bad = 1;
    s->Imin = 1e300;
    for (int c = 0; c < 3; c++) { s->I[c] = I[c][c]; if (!(I[c][c] > 0)) bad = 1; if (I[c][c] < s->Imin) s->Imin = I[c][c]; }
    if (bad) { free(s->b); free(s); return NULL; }      /* not the principal frame about the centre of mass, or collinear sites */
    const int64_t N = nm * ns;
    s->R = (double *)calloc(3 * nm, sizeof(double)); s->V = (double *)calloc(3 * nm, sizeof(double));
    s->A = (double *)calloc(9 * nm, sizeof(double)); s->pi = (double *)calloc(3 * nm, sizeof(double));
    s->F = (double *)calloc(3 * nm, sizeof(double)); s->T = (double *)calloc(3 * nm, sizeof(double));
    s->site = (double *)calloc(3 * N, sizeof(double)); s->fs = (double *)calloc(3 * N, sizeof(double));
    s->u = (double *)calloc(N, sizeof(double)); s->w = (double *)calloc(N, sizeof(double));
    s->nb_start = (int64_t *)calloc(N + 1, sizeof(int64_t));
    s->nb_cap = 64 * N;
    s->nb = (int32_t *)malloc(sizeof(int32_t) * (size_t)s->nb_cap);
    return s;
}

void orr_destroy(orr_sys *s)
{
    if (!s) return;
    free(s->b); free(s->R); free(s->V); free(s->A); free(s->pi); free(s->F); free(s->T);
    free(s->site); free(s->fs); free(s->u); free(s->w); free(s->nb_start); free(s->nb);
    free(s);
}

void orr_set_state(orr_sys *s, const double *R, const double *A, const double *V, const double *pi)
{
    memcpy(s->R, R, sizeof(double) * 3 * s->nm); memcpy(s->A, A, sizeof(double) * 9 * s->nm);
    memcpy(s->V, V, sizeof(double) * 3 * s->nm); memcpy(s->pi, pi, sizeof(double) * 3 * s->nm);
    place_sites(s);
    build_list(s);
    forces(s);
    s->disp_acc = 0.0; s->step = 0; s->n_rebuilds = 0;
}

int orr_step(orr_sys *s, int64_t n)
{
    const double dt = s->dt, h = 0.5 * dt;
    for (int64_t it = 0; it < n; it++) {
        kick(s, h);
        double vb = 0.0;
        for (int64_t m = 0; m < s->nm; m++) { const double b = speed_bound(s, m); if (b > vb) vb = b; }
        for (int64_t m = 0; m < s->nm; m++) {
            rotate_axis(s, m, 0, h); rotate_axis(s, m, 1, h); rotate_axis(s, m, 2, dt); rotate_axis(s, m, 1, h); rotate_axis(s, m, 0, h);
            for (int c = 0; c < 3; c++) s->R[3 * m + c] += dt * s->V[3 * m + c];
        }
        place_sites(s);
        s->disp_acc += dt * vb;
        if (s->disp_acc > 0.5 * s->dr) { build_list(s); s->disp_acc = 0.0; s->n_rebuilds++; }
        forces(s);
        kick(s, h);
        s->step++;
        for (int64_t m = 0; m < 3 * s->nm; m++) if (!isfinite(s->R[m]) || !isfinite(s->V[m])) return -4;
    }
    return 0;
}

void orr_energies(orr_sys *s, orr_energy *e)
{
    memset(e, 0, sizeof(*e));
    const int64_t N = s->nm * s->ns;
    long double kt = 0, kr = 0, pe = 0, vir = 0, p[3] = {0, 0, 0}, l[3] = {0, 0, 0};
    double vb = 0;
    for (int64_t m = 0; m < s->nm; m++) {
        const double *V = s->V + 3 * m, *pi = s->pi + 3 * m, *A = s->A + 9 * m;
        kt += 0.5L * s->M * (V[0] * V[0] + V[1] * V[1] + V[2] * V[2]);
        kr += 0.5L * (pi[0] * pi[0] / s->I[0] + pi[1] * pi[1] / s->I[1] + pi[2] * pi[2] / s->I[2]);
        for (int c = 0; c < 3; c++) { p[c] += s->M * V[c]; l[c] += A[3 * c] * pi[0] + A[3 * c + 1] * pi[1] + A[3 * c + 2] * pi[2]; }
        const double b = speed_bound(s, m);
        if (b > vb) vb = b;
    }
    int64_t mx = 0;
    for (int64_t i = 0; i < N; i++) {
        pe += 0.5L * s->u[i]; vir += 0.5L * s->w[i];
        const int64_t c = s->nb_start[i + 1] - s->nb_start[i];
        if (c > mx) mx = c;
    }
    e->ke_trans = (double)kt; e->ke_rot = (double)kr; e->pe = (double)pe; e->virial = (double)vir;
    e->px = (double)p[0]; e->py = (double)p[1]; e->pz = (double)p[2];
    e->lx = (double)l[0]; e->ly = (double)l[1]; e->lz = (double)l[2];
    e->vbound = vb; e->step = s->step; e->n_rebuilds = s->n_rebuilds;
    e->max_neighbors = (int32_t)mx; e->mean_neighbors = (double)s->nb_start[N] / (double)N;
}

void orr_get_state(orr_sys *s, double *R, double *A, double *V, double *pi)
{
    memcpy(R, s->R, sizeof(double) * 3 * s->nm); memcpy(A, s->A, sizeof(double) * 9 * s->nm);
    memcpy(V, s->V, sizeof(double) * 3 * s->nm); memcpy(pi, s->pi, sizeof(double) * 3 * s->nm);
}
void orr_get_sites(orr_sys *s, double *xyz) { memcpy(xyz, s->site, sizeof(double) * 3 * s->nm * s->ns); }
void orr_get_site_forces(orr_sys *s, double *xyz) { memcpy(xyz, s->fs, sizeof(double) * 3 * s->nm * s->ns); }
void orr_get_force_torque(orr_sys *s, double *F, double *T)
{
    memcpy(F, s->F, sizeof(double) * 3 * s->nm); memcpy(T, s->T, sizeof(double) * 3 * s->nm);
}
void orr_get_inertia(orr_sys *s, double *I3) { memcpy(I3, s->I, sizeof(double) * 3); }
int64_t orr_neighbor_total(orr_sys *s) { return s->nb_start[s->nm * s->ns]; }
void orr_get_neighbors(orr_sys *s, int32_t *counts, int32_t *flat)
{
    const int64_t N = s->nm * s->ns;
    for (int64_t i = 0; i < N; i++) counts[i] = (int32_t)(s->nb_start[i + 1] - s->nb_start[i]);
    memcpy(flat, s->nb, sizeof(int32_t) * (size_t)s->nb_start[N]);
}
