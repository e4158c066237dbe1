// Rigid molecules on the short-range MD path (sec. 4.3(1); R20): "molecules based on rigid
// bodies with multiple interaction sites ... rotation matrices ... a generalization of the symplectic leapfrog ... the
// additional matrix computations during integration and force/torque evaluation are readily adapted for the GPU, with
// neighbor processing and forces still dominating the work."
//
// The interaction SITES are the atoms of the hot path: they are binned, sorted into cell order, listed in W (sites of one
// molecule excluded: md_kernels.cu k_build<.., true>) and their pair forces evaluated by the kernels of md_kernels.cu
// unchanged.  What is new is per MOLECULE, one thread each:
//   k_rigid_kick_drift   F = sum f_k, T = sum (A b_k) x f_k;  V += dt/2 F/M, pi += dt/2 A^T T;  bound on the largest site
//                        speed for the rebuild rule;  free rotation by the splitting Rx(dt/2) Ry(dt/2) Rz(dt) Ry(dt/2)
//                        Rx(dt/2) of (pi, A);  R += dt V;  new site positions R + A b_k (+ the site's image offset)
//   k_rigid_kick         second half kick with the new forces; site velocities V + A (omega x b_k) for the energy kernel
//                        (sum_k 1/2 |v_k|^2 is the molecule's translational + rotational kinetic energy exactly)
//   k_rigid_offsets      after the sites were re-sorted and wrapped into the box one by one (k_reorder): the multiple of L
//                        each stored site differs by from R + A b_k, kept until the next rebuild so that the coordinates
//                        stay continuous between rebuilds (the image flags frozen into W need that, R9)
// Molecule arrays are in original order (molecule m = sites m n_s .. m n_s + n_s - 1 by original id) and never permuted;
// P.inv maps a site's original id to its current slot.  fp64, global-index W, split steps.
#include <algorithm>

#include "md_device.cuh"

namespace {

struct Mol {
    double R[3], V[3], A[9], pi[3];
};

__device__ __forceinline__ void mol_load(const MdDev &P, int m, Mol &M)
{
#pragma unroll
    for (int c = 0; c < 3; c++) { M.R[c] = P.rb_R[3 * (size_t)m + c]; M.V[c] = P.rb_V[3 * (size_t)m + c]; M.pi[c] = P.rb_pi[3 * (size_t)m + c]; }
#pragma unroll
    for (int c = 0; c < 9; c++) M.A[c] = P.rb_A[9 * (size_t)m + c];
}

// F = sum_k f_k and the torque in the BODY frame, A^T sum_k (A b_k) x f_k, from the site forces of molecule m
__device__ __forceinline__ void mol_force_torque(const MdDev &P, int m, const Mol &M, double F[3], double Tb[3])
{
    const size_t np = (size_t)P.N_pad;
    double T[3] = {0.0, 0.0, 0.0};
    F[0] = F[1] = F[2] = 0.0;
    for (int k = 0; k < P.rb_ns; k++) {
        const int n = P.inv[m * P.rb_ns + k];
        const double fx = P.frc[n], fy = P.frc[np + n], fz = P.frc[2 * np + n];
        const double bx = P.rb_body[3 * k], by = P.rb_body[3 * k + 1], bz = P.rb_body[3 * k + 2];
        const double ax = M.A[0] * bx + M.A[1] * by + M.A[2] * bz, ay = M.A[3] * bx + M.A[4] * by + M.A[5] * bz,
                     az = M.A[6] * bx + M.A[7] * by + M.A[8] * bz;
        F[0] += fx; F[1] += fy; F[2] += fz;
        T[0] += ay * fz - az * fy; T[1] += az * fx - ax * fz; T[2] += ax * fy - ay * fx;
    }
#pragma unroll
    for (int c = 0; c < 3; c++) Tb[c] = M.A[c] * T[0] + M.A[3 + c] * T[1] + M.A[6 + c] * T[2];
}

// free rotation about body axis K for time h: angle h pi_K / I_K; (pi_a, pi_c) and the columns (A_a, A_c) turn together
template <int K>
__device__ __forceinline__ void rotate_axis(const MdDev &P, Mol &M, double h)
{
    constexpr int a = (K + 1) % 3, c = (K + 2) % 3;
    double sn, cs;
    sincos(h * M.pi[K] / P.rb_I[K], &sn, &cs);
    const double pa = M.pi[a], pc = M.pi[c];
    M.pi[a] = cs * pa + sn * pc;
    M.pi[c] = -sn * pa + cs * pc;
#pragma unroll
    for (int r = 0; r < 3; r++) {
        const double Aa = M.A[3 * r + a], Ac = M.A[3 * r + c];
        M.A[3 * r + a] = cs * Aa + sn * Ac;
        M.A[3 * r + c] = -sn * Aa + cs * Ac;
    }
}

__global__ void __launch_bounds__(128) k_rigid_kick_drift(const __grid_constant__ MdDev P)
{
    __shared__ double sm[32];
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    double s2 = 0.0;
    if (m < P.rb_nm) {
        Mol M;
        mol_load(P, m, M);
        double F[3], Tb[3];
        mol_force_torque(P, m, M, F, Tb);
#pragma unroll
        for (int c = 0; c < 3; c++) { M.V[c] += P.hdt * F[c] / P.rb_M; M.pi[c] += P.hdt * Tb[c]; }
        // rigorous bound on the speed of any site during the step: |V| + |pi| / I_min * max |b_k|  (|pi| is conserved by the rotation)
        const double s = sqrt(M.V[0] * M.V[0] + M.V[1] * M.V[1] + M.V[2] * M.V[2]) +
                         sqrt(M.pi[0] * M.pi[0] + M.pi[1] * M.pi[1] + M.pi[2] * M.pi[2]) / P.rb_Imin * P.rb_bmax;
        s2 = s * s;
        rotate_axis<0>(P, M, P.hdt); rotate_axis<1>(P, M, P.hdt); rotate_axis<2>(P, M, P.dt); rotate_axis<1>(P, M, P.hdt); rotate_axis<0>(P, M, P.hdt);
#pragma unroll
        for (int c = 0; c < 3; c++) M.R[c] += P.dt * M.V[c];
#pragma unroll
        for (int c = 0; c < 3; c++) { P.rb_R[3 * (size_t)m + c] = M.R[c]; P.rb_V[3 * (size_t)m + c] = M.V[c]; P.rb_pi[3 * (size_t)m + c] = M.pi[c]; }
#pragma unroll
        for (int c = 0; c < 9; c++) P.rb_A[9 * (size_t)m + c] = M.A[c];
        pos_t *pos = P.pos[__ldcg(&P.ctrl->p_dst)];
        for (int k = 0; k < P.rb_ns; k++) {
            const int id = m * P.rb_ns + k, n = P.inv[id];
            const double bx = P.rb_body[3 * k], by = P.rb_body[3 * k + 1], bz = P.rb_body[3 * k + 2];
            const double x = (M.R[0] + (M.A[0] * bx + M.A[1] * by + M.A[2] * bz)) + P.rb_off[3 * (size_t)id];
            const double y = (M.R[1] + (M.A[3] * bx + M.A[4] * by + M.A[5] * bz)) + P.rb_off[3 * (size_t)id + 1];
            const double z = (M.R[2] + (M.A[6] * bx + M.A[7] * by + M.A[8] * bz)) + P.rb_off[3 * (size_t)id + 2];
            st_pos(pos + n, x, y, z);
            if (!isfinite(x + y + z)) { set_err(P, MD_ERR_NONFINITE); s2 = 0.0; }
        }
    }
    const double bm = block_max(s2, sm);
    if (threadIdx.x == 0) publish_vmax2(P, blockIdx.x, bm);
}

__global__ void __launch_bounds__(128) k_rigid_kick(const __grid_constant__ MdDev P)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= P.rb_nm) return;
    Mol M;
    mol_load(P, m, M);
    double F[3], Tb[3];
    mol_force_torque(P, m, M, F, Tb);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        M.V[c] += P.hdt * F[c] / P.rb_M; M.pi[c] += P.hdt * Tb[c];
        P.rb_V[3 * (size_t)m + c] = M.V[c]; P.rb_pi[3 * (size_t)m + c] = M.pi[c];
    }
    // site velocities at the synchronised instant: V + A (omega x b_k), omega = I^-1 pi in the body frame
    const double wx = M.pi[0] / P.rb_I[0], wy = M.pi[1] / P.rb_I[1], wz = M.pi[2] / P.rb_I[2];
    double *vel = P.vel[__ldcg(&P.ctrl->v_dst)];
    const size_t np = (size_t)P.N_pad;
    for (int k = 0; k < P.rb_ns; k++) {
        const int n = P.inv[m * P.rb_ns + k];
        const double bx = P.rb_body[3 * k], by = P.rb_body[3 * k + 1], bz = P.rb_body[3 * k + 2];
        const double ux = wy * bz - wz * by, uy = wz * bx - wx * bz, uz = wx * by - wy * bx;
        vel[n] = M.V[0] + (M.A[0] * ux + M.A[1] * uy + M.A[2] * uz);
        vel[np + n] = M.V[1] + (M.A[3] * ux + M.A[4] * uy + M.A[5] * uz);
        vel[2 * np + n] = M.V[2] + (M.A[6] * ux + M.A[7] * uy + M.A[8] * uz);
    }
}

// one thread per site slot: image offset of the stored (wrapped) coordinate against R + A b_k
__global__ void __launch_bounds__(256) k_rigid_offsets(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    const pos_t *pos = P.pos[__ldcg(&P.ctrl->p_dst)];
    const int *__restrict__ idv = P.id[__ldcg(&P.ctrl->v_dst)];
    for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < P.N; n += gridDim.x * blockDim.x) {
        const int id = idv[n], m = id / P.rb_ns, k = id - m * P.rb_ns;
        const double *A = P.rb_A + 9 * (size_t)m, *R = P.rb_R + 3 * (size_t)m;
        const double bx = P.rb_body[3 * k], by = P.rb_body[3 * k + 1], bz = P.rb_body[3 * k + 2];
        const pos_t r = ld_pos_rw(pos + n);
        P.rb_off[3 * (size_t)id] = P.L * rint((r.x - (R[0] + (A[0] * bx + A[1] * by + A[2] * bz))) / P.L);
        P.rb_off[3 * (size_t)id + 1] = P.L * rint((r.y - (R[1] + (A[3] * bx + A[4] * by + A[5] * bz))) / P.L);
        P.rb_off[3 * (size_t)id + 2] = P.L * rint((r.z - (R[2] + (A[6] * bx + A[7] * by + A[8] * bz))) / P.L);
    }
}

inline int cdiv(long long a, int b) { return (int)((a + b - 1) / b); }

}  // namespace

void mdk_rigid_kick_drift(const MdDev &P, cudaStream_t st) { k_rigid_kick_drift<<<cdiv(P.rb_nm, 128), 128, 0, st>>>(P); }
void mdk_rigid_kick(const MdDev &P, cudaStream_t st) { k_rigid_kick<<<cdiv(P.rb_nm, 128), 128, 0, st>>>(P); }
void mdk_rigid_offsets(const MdDev &P, cudaStream_t st) { k_rigid_offsets<<<std::min(cdiv(P.N, 256), P.sm_count * 8), 256, 0, st>>>(P); }
