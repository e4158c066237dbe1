// Push-off of an overlapping chain start (BASELINE.json configs[4]: "chains grown as seeded random walks then pushed
// apart"; PAPER.md:187 polymer chains).  INITIALISATION ONLY: it runs once, before the timed and
// parity-checked path, and its result is handed on as data.
//
// The same MD as the hot path, softened: the pair force is capped -- for r < r_cap the magnitude of the truncated LJ
// force is frozen at its value at r_cap, direction kept -- with r_cap ramped down from ~1.0 to ~0.8; the FENE force is
// clamped short of its pole; no atom moves more than a fixed distance per step; and the velocities are rescaled to the
// target temperature every step, which removes the energy the overlaps release.  It reuses the hot path's integrator
// order (half kick, drift, rebuild decision + rebuild chain, forces, half kick: md_api.cu) and its cell / neighbor-matrix
// kernels unchanged; only the kernels below are its own.  Global-index W, fp64.
#include "md_device.cuh"

namespace {

struct PoArgs {
    double rcap2;       // r_cap^2
    double vlim2;       // (largest displacement per step / dt)^2
    double ke_target;   // 3/2 (N - 1) T
    int first;          // first step: no rescale (the kinetic-energy sum does not exist yet)
};

__device__ __forceinline__ double mi_disp2(const MdDev &P, const pos_t &a, const pos_t &b, double &dx, double &dy, double &dz)
{
    dx = minimg(a.x - b.x, P.L, P.half_L); dy = minimg(a.y - b.y, P.L, P.half_L); dz = minimg(a.z - b.z, P.L, P.half_L);
    return dz * dz + dy * dy + dx * dx;
}

// v <- scale v + dt/2 f, limited; r += dt v; per-block max v^2 for the rebuild decision
__global__ void __launch_bounds__(256) k_po_kick_drift(const __grid_constant__ MdDev P, const PoArgs A)
{
    __shared__ double sm[32];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    const double ke = __ldcg(&P.ctrl->red[RED_KE]);
    const double scale = (A.first || !(ke > 0.0)) ? 1.0 : sqrt(A.ke_target / ke);
    double v2 = 0.0;
    if (i < P.N) {
        pos_t *pp = P.pos[pc] + i;
        double *vx = P.vel[vc] + i, *vy = vx + P.N_pad, *vz = vy + P.N_pad;
        const double *fx = P.frc + i, *fy = fx + P.N_pad, *fz = fy + P.N_pad;
        const pos_t r = ld_pos_rw(pp);
        double ax = scale * *vx + P.hdt * *fx, ay = scale * *vy + P.hdt * *fy, az = scale * *vz + P.hdt * *fz;
        v2 = ax * ax + ay * ay + az * az;
        if (v2 > A.vlim2) { const double c = sqrt(A.vlim2 / v2); ax *= c; ay *= c; az *= c; v2 = A.vlim2; }
        *vx = ax; *vy = ay; *vz = az;
        const double x = r.x + P.dt * ax, y = r.y + P.dt * ay, z = r.z + P.dt * az;
        st_pos(pp, x, y, z);
        if (!isfinite(v2 + x + y + z)) { set_err(P, MD_ERR_NONFINITE); v2 = 0.0; }
    }
    const double bm = block_max(v2, sm);
    if (threadIdx.x == 0) publish_vmax2(P, blockIdx.x, bm);
}

// capped pair force over column i of W + clamped FENE bonds -> f
__global__ void __launch_bounds__(256) k_po_force(const __grid_constant__ MdDev P, const PoArgs A)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const pos_t *__restrict__ pos = P.pos[__ldcg(&P.ctrl->p_dst)];
    const pos_t ri = ld_pos(pos + i);
    const int m = P.nnb[i];
    const int *__restrict__ w = P.W + (size_t)i * P.w_col;
    double fx = 0.0, fy = 0.0, fz = 0.0;
    for (int k = 0; k < m; k++) {
        const unsigned en = (unsigned)w[(size_t)k * P.w_row];
        const pos_t rj = ld_pos(pos + (en & W_INDEX_MASK));
        double dx, dy, dz;
        const double r2 = disp2(ri, rj, en >> W_FLAG_SHIFT, P.L, dx, dy, dz);
        if (r2 < P.rc2) {
            // inside the cap the force keeps the magnitude it has at r_cap: fc(r_cap) r_cap / r along d
            const bool capped = r2 < A.rcap2;
            const double q = capped ? A.rcap2 : r2;
            const double s = 1.0 / q, s3 = s * s * s;
            double fc = 48.0 * s3 * (s3 - 0.5) * s;
            if (capped) fc *= sqrt(A.rcap2 / fmax(r2, 1e-24));
            fx += fc * dx; fy += fc * dy; fz += fc * dz;
        }
    }
    if (P.has_bonds) {
#pragma unroll
        for (int k = 0; k < 2; k++) {
            const int j = P.bond_dev[(size_t)k * P.N_pad + i];
            if (j < 0) continue;
            const pos_t rj = ld_pos(pos + j);
            const double dx = minimg(ri.x - rj.x, P.L, P.half_L), dy = minimg(ri.y - rj.y, P.L, P.half_L),
                         dz = minimg(ri.z - rj.z, P.L, P.half_L);
            const double r2 = dz * dz + dy * dy + dx * dx;
            const double x = fmax(1.0 - r2 / P.fene_R02, 0.02);      // clamped short of the pole at r = R0
            const double fc = -P.fene_k / x;
            fx += fc * dx; fy += fc * dy; fz += fc * dz;
        }
    }
    const size_t np = (size_t)P.N_pad;
    double *f = P.frc + i;
    f[0] = fx; f[np] = fy; f[2 * np] = fz;
}

// v += dt/2 f; per-block sum of v^2 / 2
__global__ void __launch_bounds__(256) k_po_kick(const __grid_constant__ MdDev P)
{
    __shared__ double sm[8];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int vc = __ldcg(&P.ctrl->v_dst);
    double ke = 0.0;
    if (i < P.N) {
        double *v = P.vel[vc] + i;
        const double *f = P.frc + i;
        const size_t np = (size_t)P.N_pad;
        const double vx = v[0] + P.hdt * f[0], vy = v[np] + P.hdt * f[np], vz = v[2 * np] + P.hdt * f[2 * np];
        v[0] = vx; v[np] = vy; v[2 * np] = vz;
        ke = 0.5 * (vx * vx + vy * vy + vz * vz);
    }
    ke = warp_sum(ke);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = ke;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; w++) t += sm[w];
        P.partials[blockIdx.x] = t;
    }
}

// one block: kinetic energy = sum of the per-block partials, fixed order
__global__ void __launch_bounds__(1024) k_po_reduce(const __grid_constant__ MdDev P, int nblk)
{
    __shared__ double sm[32];
    double t = 0.0;
    for (int b = threadIdx.x; b < nblk; b += 1024) t += P.partials[b];
    t = warp_sum(t);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = t;
    __syncthreads();
    if (threadIdx.x < 32) {
        t = warp_sum(sm[threadIdx.x]);
        if (threadIdx.x == 0) P.ctrl->red[RED_KE] = t;
    }
}

// the two stopping criteria: smallest distance of a listed pair that is not bonded, longest bond.  Squared lengths are
// non-negative doubles, so their bit patterns order like the numbers and integer atomics can take the min / max.
__global__ void __launch_bounds__(256) k_po_check(const __grid_constant__ MdDev P, unsigned long long *out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double mn = 1e300, mx = 0.0;
    if (i < P.N) {
        const pos_t *__restrict__ pos = P.pos[__ldcg(&P.ctrl->p_dst)];
        const pos_t ri = ld_pos(pos + i);
        const int b0 = P.has_bonds ? P.bond_dev[i] : -1, b1 = P.has_bonds ? P.bond_dev[(size_t)P.N_pad + i] : -1;
        const int m = P.nnb[i];
        const int *__restrict__ w = P.W + (size_t)i * P.w_col;
        for (int k = 0; k < m; k++) {
            const unsigned en = (unsigned)w[(size_t)k * P.w_row];
            const int j = (int)(en & W_INDEX_MASK);
            double dx, dy, dz;
            const double r2 = disp2(ri, ld_pos(pos + j), en >> W_FLAG_SHIFT, P.L, dx, dy, dz);
            if (j != b0 && j != b1) mn = fmin(mn, r2);
        }
        // bonds straight from the bond table (a bond longer than r_n is not in W)
        if (b0 >= 0) { double dx, dy, dz; mx = fmax(mx, mi_disp2(P, ri, ld_pos(pos + b0), dx, dy, dz)); }
        if (b1 >= 0) { double dx, dy, dz; mx = fmax(mx, mi_disp2(P, ri, ld_pos(pos + b1), dx, dy, dz)); }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        mn = fmin(mn, __shfl_xor_sync(FULL_MASK, mn, o));
        mx = fmax(mx, __shfl_xor_sync(FULL_MASK, mx, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMin(out, (unsigned long long)__double_as_longlong(mn));
        atomicMax(out + 1, (unsigned long long)__double_as_longlong(mx));
    }
}

__global__ void k_po_check_init(unsigned long long *out)
{
    out[0] = (unsigned long long)__double_as_longlong(1e300);
    out[1] = 0ull;
}

inline int cdiv(long long a, int b) { return (int)((a + b - 1) / b); }

}  // namespace

void mdk_po_kick_drift(const MdDev &P, double rcap2, double vlim2, double ke_target, int first, cudaStream_t st)
{
    const PoArgs A = {rcap2, vlim2, ke_target, first};
    k_po_kick_drift<<<cdiv(P.N, 256), 256, 0, st>>>(P, A);
}

void mdk_po_force(const MdDev &P, double rcap2, cudaStream_t st)
{
    const PoArgs A = {rcap2, 0.0, 0.0, 0};
    k_po_force<<<cdiv(P.N, 256), 256, 0, st>>>(P, A);
}

void mdk_po_kick(const MdDev &P, cudaStream_t st)
{
    const int nblk = cdiv(P.N, 256);
    k_po_kick<<<nblk, 256, 0, st>>>(P);
    k_po_reduce<<<1, 1024, 0, st>>>(P, nblk);
}

// out: two 64-bit words on the device (min non-bonded r^2, max bond r^2 as bit patterns)
void mdk_po_check(const MdDev &P, unsigned long long *out, cudaStream_t st)
{
    k_po_check_init<<<1, 1, 0, st>>>(out);
    k_po_check<<<cdiv(P.N, 256), 256, 0, st>>>(P, out);
}
