// Single-precision variant of the MD hot path (md_params.precision = MD_PREC_F32).
// The paper's own numbers are single precision (Table 1; "0.3x" for double) with the
// state held as float4 arrays r, v, a.  Here: positions, velocities and forces are float4 records
// (16 bytes: two per L2 sector), all pair arithmetic is binary32, and every sum of energies (u_i, w_i, KE, momentum)
// is accumulated in binary64 (reading R18).  The integer machinery (occupancy scan, placement, bond
// remap) and the rebuild decision are the kernels of md_kernels.cu; only the kernels that touch coordinates are here.
//
// Where binary32 decides an integer -- j in the neighbor set of i, a pair inside r_c -- the decision is taken on
//   d = fl(a - b), one conditional +-L (rounded once), r2 = fmaf(dz,dz, fmaf(dy,dy, fl(dx*dx)))  <  (float)(r*r)
// exactly as stated in DESIGN.md R18, so neighbor sets are compared bit-exactly with the oracle.
// No code is shared with oracle/.
#include <algorithm>

#include <cooperative_groups.h>

#include "md_device.cuh"
#include "md_rebuild.cuh"

namespace {

__device__ __forceinline__ float wrap1f(float x, float L)
{
    if (x >= L) x -= L;
    else if (x < 0.0f) { x += L; if (x >= L) x = 0.0f; }
    return x;
}

__device__ __forceinline__ float4 ld4(const float4 *p) { return __ldg(p); }

constexpr int SP_PAD = 4;      // columns of W are padded to a multiple of this many rows with self entries (k_sp_build)

// the displacement of md_device.cuh:disp2 in binary32 (image flags frozen into the W entry)
__device__ __forceinline__ float disp2f(const float4 &a, const float4 &b, unsigned fl, float L, float &dx, float &dy, float &dz)
{
    dx = __fsub_rn(a.x, b.x);
    dy = __fsub_rn(a.y, b.y);
    dz = __fsub_rn(a.z, b.z);
    if (fl) {
        if (fl & 1u) dx = __fsub_rn(dx, copysignf(L, dx));
        if (fl & 2u) dy = __fsub_rn(dy, copysignf(L, dy));
        if (fl & 4u) dz = __fsub_rn(dz, copysignf(L, dz));
    }
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

__device__ __forceinline__ float minimgf(float d, float L, float half)
{
    return d > half ? __fsub_rn(d, L) : (d < -half ? __fadd_rn(d, L) : d);
}

// ------------------------------------------------------------------------------------------------
// staging: scratch (binary64, original-id order) <-> float4 device arrays
// ------------------------------------------------------------------------------------------------
__global__ void k_sp_load_state(const __grid_constant__ MdDev P)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const int pc = P.ctrl->p_dst, vc = P.ctrl->v_dst;
    const double *s = P.scratch + 3 * (size_t)i;
    if (!(isfinite(s[0]) && isfinite(s[1]) && isfinite(s[2]))) set_err(P, MD_ERR_NONFINITE);
    const float x = wrap1f((float)s[0], P.Lf), y = wrap1f((float)s[1], P.Lf), z = wrap1f((float)s[2], P.Lf);
    P.posf[pc][i] = make_float4(x, y, z, 0.0f);
    const double *v = P.scratch + 3 * (size_t)P.N + 3 * (size_t)i;
    P.velf[vc][i] = make_float4((float)v[0], (float)v[1], (float)v[2], 0.0f);
    P.id[vc][i] = i;
}

__global__ void k_sp_export(const __grid_constant__ MdDev P, int what, double *dst)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const int pc = P.ctrl->p_dst, vc = P.ctrl->v_dst;
    const int id = P.id[vc][i];
    double *o = dst + 3 * (size_t)id;
    if (what == 0) {
        const float4 r = P.posf[pc][i];
        o[0] = (double)wrap1f(r.x, P.Lf); o[1] = (double)wrap1f(r.y, P.Lf); o[2] = (double)wrap1f(r.z, P.Lf);
    } else {
        const float4 a = what == 1 ? P.velf[vc][i] : P.frcf[i];
        o[0] = (double)a.x; o[1] = (double)a.y; o[2] = (double)a.z;
    }
}

// ------------------------------------------------------------------------------------------------
// integration (opening half kick + drift; closing half kick of the split mode)
// ------------------------------------------------------------------------------------------------
// opening half kick + drift of atom i; returns |v|^2
__device__ __forceinline__ float sp_kick_drift_atom(const MdDev &P, int pc, int vc, int i)
{
    float4 r = P.posf[pc][i], v = P.velf[vc][i];
    const float4 f = P.frcf[i];
    v.x = __fadd_rn(v.x, __fmul_rn(P.hdtf, f.x)); v.y = __fadd_rn(v.y, __fmul_rn(P.hdtf, f.y)); v.z = __fadd_rn(v.z, __fmul_rn(P.hdtf, f.z));
    r.x = __fadd_rn(r.x, __fmul_rn(P.dtf, v.x)); r.y = __fadd_rn(r.y, __fmul_rn(P.dtf, v.y)); r.z = __fadd_rn(r.z, __fmul_rn(P.dtf, v.z));
    P.velf[vc][i] = v;
    P.posf[pc][i] = r;
    float v2 = v.x * v.x + v.y * v.y + v.z * v.z;
    if (!isfinite(v2 + r.x + r.y + r.z)) { set_err(P, MD_ERR_NONFINITE); v2 = 0.0f; }
    return v2;
}

__global__ void __launch_bounds__(256) k_sp_kick_drift(const __grid_constant__ MdDev P)
{
    __shared__ double sm[32];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    const float v2 = i < P.N ? sp_kick_drift_atom(P, pc, vc, i) : 0.0f;
    const double bm = block_max((double)v2, sm);
    if (threadIdx.x == 0) publish_vmax2(P, blockIdx.x, bm);
}

__global__ void __launch_bounds__(256) k_sp_kick(const __grid_constant__ MdDev P)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const int vc = __ldcg(&P.ctrl->v_dst);
    float4 v = P.velf[vc][i];
    const float4 f = P.frcf[i];
    v.x = __fadd_rn(v.x, __fmul_rn(P.hdtf, f.x)); v.y = __fadd_rn(v.y, __fmul_rn(P.hdtf, f.y)); v.z = __fadd_rn(v.z, __fmul_rn(P.hdtf, f.z));
    P.velf[vc][i] = v;
}

// ------------------------------------------------------------------------------------------------
// N1/N2: the cell of an atom is found in binary64 from its binary32 coordinate (cells are
// kept wider than r_n by 1e-5 relative at create time, far more than the rounding error of a binary32 r2)
// ------------------------------------------------------------------------------------------------
template <class LD>
__device__ __forceinline__ void sp_bin_body(const MdDev &P, const Bufs B)
{
    const float4 *pos = P.posf[B.ps];
    const int *idv = P.id[B.vs];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += gridDim.x * blockDim.x) {
        const float4 r = LD::f4(pos + i);
        const int cx = cell_coord((double)wrap1f(r.x, P.Lf), P.inv_wx, P.ncx), cy = cell_coord((double)wrap1f(r.y, P.Lf), P.inv_w, P.nc),
                  cz = cell_coord((double)wrap1f(r.z, P.Lf), P.inv_w, P.nc);
        const int sys = P.n_sys > 1 ? LD::i32(idv + i) / P.N1 : 0;
        const int c = sys * P.NC1 + cx + P.ncx * (cy + P.nc * cz);
        P.cell_of[i] = c;
        P.slot[i] = atomicAdd(&P.cell_count[c], 1);
    }
}

__global__ void __launch_bounds__(256) k_sp_bin(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    sp_bin_body<LdNC>(P, bufs_from_ctrl(P));
}

// cell-order gather, coordinates wrapped here; members of a cell ranked by previous slot
template <class LD>
__device__ __forceinline__ void sp_reorder_body(const MdDev &P, const Bufs B)
{
    const float4 *pin = P.posf[B.ps];
    const float4 *vin = P.velf[B.vs];
    const int *idin = P.id[B.vs];
    for (int p = blockIdx.x * blockDim.x + threadIdx.x; p < P.N; p += gridDim.x * blockDim.x) {
        const int a = P.perm[p];
        const float4 r = LD::f4(pin + a), v = LD::f4(vin + a);
        const int id = LD::i32(idin + a);
        const int c = P.cell_of[a];
        const int s = P.cell_start[c], e = P.cell_start[c + 1];
        int rank = 0;
        for (int q = s; q < e; q++) rank += (P.perm[q] < a);
        const int n = s + rank;
        P.posf[B.pd][n] = make_float4(wrap1f(r.x, P.Lf), wrap1f(r.y, P.Lf), wrap1f(r.z, P.Lf), 0.0f);
        P.velf[B.vd][n] = v;
        P.id[B.vd][n] = id;
        if (P.need_inv) P.inv[id] = n;
    }
}

__global__ void __launch_bounds__(256) k_sp_reorder(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    sp_reorder_body<LdNC>(P, bufs_from_ctrl(P));
}

// ------------------------------------------------------------------------------------------------
// N5: the gather form of md_kernels.cu:k_build in binary32
// ------------------------------------------------------------------------------------------------
// (A single flat loop over all candidates of an atom, its <= 18 segments tabulated in shared memory so that lanes
// idle only at the end of the whole list, was measured SLOWER -- 534 vs 390 us per build at wca_2m: lanes then sit
// in different runs, each gather request touches more lines, and the loop no longer unrolls.)
template <bool SHIFT, class LD>
__device__ __forceinline__ void scan_run_f(const MdDev &P, const float4 *pos, const float4 &ri, int i, int b, int e,
                                           float sx, float sy, float sz, unsigned fl, int &m)
{
    for (int j = b; j < e; j++) {
        const float4 rj = LD::f4(pos + j);
        float dx = __fsub_rn(ri.x, rj.x), dy = __fsub_rn(ri.y, rj.y), dz = __fsub_rn(ri.z, rj.z);
        if (SHIFT) { dx = __fadd_rn(dx, sx); dy = __fadd_rn(dy, sy); dz = __fadd_rn(dz, sz); }
        const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
        if (r2 < P.rn2f && j != i) {
            if (m < P.Mmax) P.W[(size_t)m * P.w_row + (size_t)i * P.w_col] = (int)((unsigned)j | (fl << W_FLAG_SHIFT));
            m++;
        }
    }
}

// all threads of the block call it (block reduction of the statistics at the end); blocks of <= 256 threads
template <class LD>
__device__ __forceinline__ void sp_build_body(const MdDev &P, const Bufs B)
{
    __shared__ int smx[8], scand[8];
    __shared__ int ssum[8];
    const float4 *pos = P.posf[B.pd];
    const int *cs = P.cell_start;
    const int *idv = P.id[B.vd];
    const int nc = P.nc, ncx = P.ncx;
    const float L = P.Lf;
    int tmax = 0, tsum = 0, tcand = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += gridDim.x * blockDim.x) {
        const float4 ri = LD::f4(pos + i);
        const int cx = cell_coord((double)ri.x, P.inv_wx, ncx), cy = cell_coord((double)ri.y, P.inv_w, nc), cz = cell_coord((double)ri.z, P.inv_w, nc);
        const RowGaps gaps = row_gaps(P, (double)ri.y, (double)ri.z, cy, cz);
        const int cell_base = P.n_sys > 1 ? (LD::i32(idv + i) / P.N1) * P.NC1 : 0;
        int m = 0;
        for (int dz = -1; dz <= 1; dz++) {
            int z = cz + dz;
            float sz = 0.0f;
            unsigned fz = 0u;
            if (z < 0) { z += nc; sz = L; fz = 4u; } else if (z >= nc) { z -= nc; sz = -L; fz = 4u; }
            for (int dy = -1; dy <= 1; dy++) {
                const int kr = row_halfwidth(P, gaps, dy, dz);
                if (kr < 0) continue;
                int y = cy + dy;
                float sy = 0.0f;
                unsigned fl = fz;
                if (y < 0) { y += nc; sy = L; fl |= 2u; } else if (y >= nc) { y -= nc; sy = -L; fl |= 2u; }
                const int row = cell_base + ncx * (y + nc * z);
                const int lo = cx - kr, hi = cx + kr;
                const int b = LD::i32(cs + row + (lo < 0 ? 0 : lo)), e = LD::i32(cs + row + (hi >= ncx ? ncx : hi + 1));
                tcand += e - b;
                if (fl) scan_run_f<true, LD>(P, pos, ri, i, b, e, 0.0f, sy, sz, fl, m);
                else scan_run_f<false, LD>(P, pos, ri, i, b, e, 0.0f, 0.0f, 0.0f, 0u, m);
                if (lo < 0) scan_run_f<true, LD>(P, pos, ri, i, LD::i32(cs + row + ncx + lo), LD::i32(cs + row + ncx), L, sy, sz, fl | 1u, m);
                if (hi >= ncx) scan_run_f<true, LD>(P, pos, ri, i, LD::i32(cs + row), LD::i32(cs + row + hi - ncx + 1), -L, sy, sz, fl | 1u, m);
            }
        }
        P.nnb[i] = m < P.Mmax ? m : P.Mmax;
        if (m > P.Mmax) set_err(P, MD_ERR_NEBR_OVERFLOW);
        // long columns (P.sp_pad): pad to a multiple of SP_PAD rows with the atom's own index (Mmax is a multiple): the
        // force kernel then walks whole groups of SP_PAD rows without per-row predicates; a self entry has r2 = 0
        // and is deselected there.  m_i = nnb[i] stays the true count for everything else.
        if (P.sp_pad > 1)
            for (int k = m; k < ((m + SP_PAD - 1) & ~(SP_PAD - 1)) && k < P.Mmax; k++)
                P.W[(size_t)k * P.w_row + (size_t)i * P.w_col] = i;
        tmax = max(tmax, m);
        tsum += m;
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int wm = warp_max_i(tmax), ws = warp_sum_i(tsum), wc = warp_sum_i(tcand);
    if (lane == 0) { smx[wid] = wm; ssum[wid] = ws; scand[wid] = wc; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int mx = 0, sm = 0, sc = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) { mx = max(mx, smx[w]); sm += ssum[w]; sc += scand[w]; }
        atomicMax(&P.ctrl->max_nnb, mx);
        atomicAdd(&P.ctrl->nnb_total, (unsigned long long)sm);
        atomicAdd(&P.ctrl->cand_total, (unsigned long long)sc);
    }
}

__global__ void __launch_bounds__(128) k_sp_build(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    sp_build_body<LdNC>(P, bufs_from_ctrl(P));
}

// ------------------------------------------------------------------------------------------------
// F1: column i of W, partner positions gathered as 16-byte records; the structure (W rows a block
// of D ahead, U gathers in flight) is that of md_kernels.cu:column_force
// ------------------------------------------------------------------------------------------------
struct PairAccF {
    float fx, fy, fz;
};

// One pair term, branch-free: the range test selects the coefficient instead of guarding the arithmetic (a warp
// almost always holds a lane in range, so a branch would only add its own instructions).
// Range test 0 < r2 < r_c^2 in ONE unsigned compare: non-negative floats order like their bit patterns, and
// bits - 1 wraps r2 = 0 (the self entries that pad a column) to the top.  The decision is exact.
// 1/r2 is the hardware approximation (MUFU.RCP, <= 1 ulp): the coefficient's error stays inside the rounding bound
// of the binary32 sum.  The factor 48 is applied once to the sums.
// The image flags of the W entry sit behind one branch that almost every warp skips.  (Two copies
// of the loop, with and without flag arithmetic, chosen per atom by its distance from the faces, were measured
// SLOWER: a quarter of the warps of an x-ordered system hold atoms of both kinds and ran both copies.)
__device__ __forceinline__ void pair_force_f(const float4 &ri, const float4 &rj, unsigned en, float L, unsigned rc2m1, PairAccF &a)
{
    float dx = __fsub_rn(ri.x, rj.x), dy = __fsub_rn(ri.y, rj.y), dz = __fsub_rn(ri.z, rj.z);
    const unsigned fl = en >> W_FLAG_SHIFT;
    if (fl) {
        if (fl & 1u) dx = __fsub_rn(dx, copysignf(L, dx));
        if (fl & 2u) dy = __fsub_rn(dy, copysignf(L, dy));
        if (fl & 4u) dz = __fsub_rn(dz, copysignf(L, dz));
    }
    const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
    float s;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(r2));
    const float s3 = s * s * s;
    float fc = s3 * (s3 - 0.5f) * s;
    fc = (__float_as_uint(r2) - 1u) < rc2m1 ? fc : 0.0f;
    a.fx = fmaf(fc, dx, a.fx); a.fy = fmaf(fc, dy, a.fy); a.fz = fmaf(fc, dz, a.fz);
}

__device__ __forceinline__ float mi_disp_f(const MdDev &P, const float4 &a, const float4 &b, float &dx, float &dy, float &dz)
{
    dx = minimgf(__fsub_rn(a.x, b.x), P.Lf, P.half_Lf); dy = minimgf(__fsub_rn(a.y, b.y), P.Lf, P.half_Lf);
    dz = minimgf(__fsub_rn(a.z, b.z), P.Lf, P.half_Lf);
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

// bond-angle terms in binary32: md_kernels.cu:angle_force (R19)
__device__ __forceinline__ void angle_force_f(const MdDev &P, const float4 *__restrict__ pos, const float4 &ri, int i, PairAccF &a)
{
    const int p[2] = {P.bond_dev[i], P.bond_dev[(size_t)P.N_pad + i]};
    const float k = (float)P.ang_k, c0 = (float)P.ang_c0;
    float4 rp[2];
#pragma unroll
    for (int q = 0; q < 2; q++)
        if (p[q] >= 0) rp[q] = ld4(pos + p[q]);
    if (p[0] >= 0 && p[1] >= 0) {
        float x1, y1, z1, x2, y2, z2;
        const float n1 = mi_disp_f(P, rp[0], ri, x1, y1, z1), n2 = mi_disp_f(P, rp[1], ri, x2, y2, z2);
        const float inv12 = 1.0f / sqrtf(n1 * n2), c = (x1 * x2 + y1 * y2 + z1 * z2) * inv12;
        const float g = -k * (c - c0), u1 = c / n1, u2 = c / n2;
        a.fx -= g * ((x2 * inv12 - u1 * x1) + (x1 * inv12 - u2 * x2));
        a.fy -= g * ((y2 * inv12 - u1 * y1) + (y1 * inv12 - u2 * y2));
        a.fz -= g * ((z2 * inv12 - u1 * z1) + (z1 * inv12 - u2 * z2));
    }
#pragma unroll
    for (int q = 0; q < 2; q++) {
        if (p[q] < 0) continue;
        const int q0 = P.bond_dev[p[q]], q1 = P.bond_dev[(size_t)P.N_pad + p[q]];
        const int o = q0 == i ? q1 : q0;
        if (o < 0) continue;
        const float4 ro = ld4(pos + o);
        float x1, y1, z1, x2, y2, z2;
        const float n1 = mi_disp_f(P, ri, rp[q], x1, y1, z1), n2 = mi_disp_f(P, ro, rp[q], x2, y2, z2);
        const float inv12 = 1.0f / sqrtf(n1 * n2), c = (x1 * x2 + y1 * y2 + z1 * z2) * inv12;
        const float g = -k * (c - c0), u1 = c / n1;
        a.fx += g * (x2 * inv12 - u1 * x1);
        a.fy += g * (y2 * inv12 - u1 * y1);
        a.fz += g * (z2 * inv12 - u1 * z1);
    }
}

// dihedral terms in binary32: md_kernels.cu:dihedral_term / dihedral_force (R19)
struct V3f {
    float x, y, z;
};
__device__ __forceinline__ V3f cross3f(const V3f &u, const V3f &v) { return {u.y * v.z - u.z * v.y, u.z * v.x - u.x * v.z, u.x * v.y - u.y * v.x}; }
__device__ __forceinline__ V3f mi_vec_f(const MdDev &P, const float4 &a, const float4 &b)
{
    V3f d;
    mi_disp_f(P, a, b, d.x, d.y, d.z);
    return d;
}

__device__ __forceinline__ float dihedral_term_f(const MdDev &P, const float4 &ra, const float4 &rb, const float4 &rc, const float4 &rd, int which,
                                                 PairAccF &acc)
{
    const V3f b1 = mi_vec_f(P, rb, ra), b2 = mi_vec_f(P, rc, rb), b3 = mi_vec_f(P, rd, rc);
    const V3f A = cross3f(b1, b2), B = cross3f(b2, b3);
    const float nA = A.x * A.x + A.y * A.y + A.z * A.z, nB = B.x * B.x + B.y * B.y + B.z * B.z;
    const float invAB = 1.0f / sqrtf(nA * nB), c = (A.x * B.x + A.y * B.y + A.z * B.z) * invAB;
    if (which < 0) return c;
    const float uA = c / nA, uB = c / nB;
    const V3f gA = {B.x * invAB - uA * A.x, B.y * invAB - uA * A.y, B.z * invAB - uA * A.z};
    const V3f gB = {A.x * invAB - uB * B.x, A.y * invAB - uB * B.y, A.z * invAB - uB * B.z};
    const V3f g1 = cross3f(b2, gA), t1 = cross3f(gA, b1), t2 = cross3f(b3, gB), g3 = cross3f(gB, b2);
    const V3f g2 = {t1.x + t2.x, t1.y + t2.y, t1.z + t2.z};
    V3f d;
    if (which == 0) d = {-g1.x, -g1.y, -g1.z};
    else if (which == 1) d = {g1.x - g2.x, g1.y - g2.y, g1.z - g2.z};
    else if (which == 2) d = {g2.x - g3.x, g2.y - g3.y, g2.z - g3.z};
    else d = g3;
    const float g = -(float)P.dih_k * (c - (float)P.dih_c0);
    acc.fx += g * d.x; acc.fy += g * d.y; acc.fz += g * d.z;
    return c;
}

__device__ __forceinline__ int chain_next_f(const MdDev &P, int x, int prev)
{
    const int q0 = P.bond_dev[x], q1 = P.bond_dev[(size_t)P.N_pad + x];
    return q0 == prev ? q1 : q0;
}

__device__ __noinline__ void dihedral_force_f(const MdDev &P, const float4 *__restrict__ pos, const float4 &ri, int i, PairAccF &a)
{
    const int L1 = P.bond_dev[i], R1 = P.bond_dev[(size_t)P.N_pad + i];
    const int L2 = L1 >= 0 ? chain_next_f(P, L1, i) : -1, L3 = L2 >= 0 ? chain_next_f(P, L2, L1) : -1;
    const int R2 = R1 >= 0 ? chain_next_f(P, R1, i) : -1, R3 = R2 >= 0 ? chain_next_f(P, R2, R1) : -1;
    float4 l1, l2, l3, r1, r2, r3;
    if (L1 >= 0) l1 = ld4(pos + L1);
    if (L2 >= 0) l2 = ld4(pos + L2);
    if (L3 >= 0) l3 = ld4(pos + L3);
    if (R1 >= 0) r1 = ld4(pos + R1);
    if (R2 >= 0) r2 = ld4(pos + R2);
    if (R3 >= 0) r3 = ld4(pos + R3);
    if (L3 >= 0) dihedral_term_f(P, l3, l2, l1, ri, 3, a);
    if (L2 >= 0 && R1 >= 0) dihedral_term_f(P, l2, l1, ri, r1, 2, a);
    if (L1 >= 0 && R2 >= 0) dihedral_term_f(P, l1, ri, r1, r2, 1, a);
    if (R3 >= 0) dihedral_term_f(P, ri, r1, r2, r3, 0, a);
}

// EXTRAS: angle / dihedral code compiled in (the FENE-only instantiation keeps its registers)
template <bool CHECK, bool EXTRAS = true, class LD = LdNC>
__device__ __forceinline__ void bond_force_f(const MdDev &P, const float4 *pos, const float4 &ri, int i, PairAccF &a)
{
    if (EXTRAS && P.has_angles) angle_force_f(P, pos, ri, i, a);
    if (EXTRAS && P.has_dihedrals) dihedral_force_f(P, pos, ri, i, a);
#pragma unroll
    for (int k = 0; k < 2; k++) {
        const int j = P.bond_dev[(size_t)k * P.N_pad + i];
        if (j < 0) continue;
        const float4 rj = LD::f4(pos + j);
        const float dx = minimgf(__fsub_rn(ri.x, rj.x), P.Lf, P.half_Lf), dy = minimgf(__fsub_rn(ri.y, rj.y), P.Lf, P.half_Lf),
                    dz = minimgf(__fsub_rn(ri.z, rj.z), P.Lf, P.half_Lf);
        const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
        if (!(r2 < P.fene_R02f)) { if (CHECK) set_err(P, MD_ERR_BOND_BROKEN); continue; }
        const float fc = __fdividef(-(P.fene_kf * P.fene_R02f), P.fene_R02f - r2);      // one approximate division (2 ulp) for two IEEE ones
        a.fx += fc * dx; a.fy += fc * dy; a.fz += fc * dz;
    }
}

#ifndef MD_SP_FORCE_D
#define MD_SP_FORCE_D 4
#endif
#ifndef MD_SP_FORCE_U
#define MD_SP_FORCE_U 4
#endif

// Column i of W.  W rows stream from HBM a block of D rows ahead of the gathers (md_kernels.cu:column_force).
// PADDED: the build padded every column to a multiple of SP_PAD rows with self entries (P.sp_pad; chosen at create
// time for long columns, e.g. LJ r_c = 2.5), so whole groups of SP_PAD rows run without per-row predicates: measured
// 197 -> 169 us per fused step at lj_1m.  For the short WCA columns the ~1.5 extra gather rows per warp cost more
// than the predicates save (94 -> 99 us at wca_2m: the kernel's time goes with its number of gather instructions),
// so there the rows past the column end are predicated off instead; such a lane carries r_j = r_i (r2 = 0).
template <int D, bool PADDED, class LD = LdNC>
__device__ __forceinline__ PairAccF column_force_f(const MdDev &P, const float4 *pos, const float4 &ri, int i)
{
    constexpr int U = PADDED ? SP_PAD : MD_SP_FORCE_U;       // gathers in flight per thread
    static_assert(D % U == 0, "D must be a multiple of the gather group");
    const int *__restrict__ w = P.W + (size_t)i * P.w_col;
    const size_t pitch = (size_t)P.w_row;
    const float L = P.Lf;
    const unsigned rc2m1 = __float_as_uint(P.rc2f) - 1u;
    PairAccF a = {0.0f, 0.0f, 0.0f};
    unsigned cur[D], nxt[D];
#pragma unroll
    for (int d = 0; d < D; d++) cur[d] = d < P.Mmax ? (unsigned)__ldcs(w + d * pitch) : 0u;
    const int m = PADDED ? (P.nnb[i] + U - 1) & ~(U - 1) : P.nnb[i];
    w += D * pitch;
    for (int rem = m; rem > 0; rem -= D, w += D * pitch) {
        if (PADDED) {
#pragma unroll
            for (int g = 0; g < D; g += U)
                if (D + g < rem) {
#pragma unroll
                    for (int u = 0; u < U; u++) nxt[g + u] = (unsigned)__ldcs(w + (g + u) * pitch);
                }
        } else {
#pragma unroll
            for (int d = 0; d < D; d++) nxt[d] = D + d < rem ? (unsigned)__ldcs(w + d * pitch) : 0u;
        }
#pragma unroll
        for (int g = 0; g < D; g += U) {
            if (g < rem) {
                float4 rj[U];
#pragma unroll
                for (int u = 0; u < U; u++) {
                    if (PADDED) rj[u] = LD::f4(pos + (cur[g + u] & W_INDEX_MASK));
                    else {
                        rj[u] = ri;
                        if (g + u < rem) rj[u] = LD::f4(pos + (cur[g + u] & W_INDEX_MASK));
                    }
                }
#pragma unroll
                for (int u = 0; u < U; u++) pair_force_f(ri, rj[u], cur[g + u], L, rc2m1, a);
            }
        }
#pragma unroll
        for (int d = 0; d < D; d++) cur[d] = nxt[d];
    }
    a.fx *= 48.0f; a.fy *= 48.0f; a.fz *= 48.0f;
    return a;
}

// MODE 0: store f.  MODE 1: fused leapfrog step (v += dt f; r' = r + dt v into the other position buffer; per-block
// max v^2 for k_decide).  MODE 2: store f and apply the closing half kick.
#ifndef MD_SP_MIN_THREADS
#define MD_SP_MIN_THREADS 1280       // resident threads per SM the register allocation must allow
#endif
// BONDS: 0 none, 1 FENE bonds, 2 FENE + angle / dihedral terms
// forces on atom i over column i of W (+ bonds) and the MODE's part of the integration; returns |v|^2 (MODE 1)
template <int MODE, int BONDS, bool PADDED, class LD>
__device__ __forceinline__ float sp_force_atom(const MdDev &P, int pc, int vc, int i)
{
    const float4 *pos = P.posf[pc];
    float v2 = 0.0f;
    const float4 ri = LD::f4(pos + i);
    float4 v = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    if (MODE != 0) v = P.velf[vc][i];               // in flight while the column is walked
    PairAccF a = column_force_f<MD_SP_FORCE_D, PADDED, LD>(P, pos, ri, i);
    if (BONDS == 1) bond_force_f<true, false, LD>(P, pos, ri, i, a);
    if (BONDS == 2) bond_force_f<true, true, LD>(P, pos, ri, i, a);
    if (MODE == 0 || MODE == 2) P.frcf[i] = make_float4(a.fx, a.fy, a.fz, 0.0f);
    if (MODE == 2) {
        v.x = __fadd_rn(v.x, __fmul_rn(P.hdtf, a.fx)); v.y = __fadd_rn(v.y, __fmul_rn(P.hdtf, a.fy)); v.z = __fadd_rn(v.z, __fmul_rn(P.hdtf, a.fz));
        P.velf[vc][i] = v;
    }
    if (MODE == 1) {
        // two half kicks of the oracle's step merged into one full kick (leapfrog form)
        v.x = __fadd_rn(v.x, __fmul_rn(P.dtf, a.fx)); v.y = __fadd_rn(v.y, __fmul_rn(P.dtf, a.fy)); v.z = __fadd_rn(v.z, __fmul_rn(P.dtf, a.fz));
        P.velf[vc][i] = v;
        const float x = __fadd_rn(ri.x, __fmul_rn(P.dtf, v.x)), y = __fadd_rn(ri.y, __fmul_rn(P.dtf, v.y)), z = __fadd_rn(ri.z, __fmul_rn(P.dtf, v.z));
        P.posf[pc ^ 1][i] = make_float4(x, y, z, 0.0f);
        v2 = v.x * v.x + v.y * v.y + v.z * v.z;
        if (!isfinite(v2 + x + y + z)) { set_err(P, MD_ERR_NONFINITE); v2 = 0.0f; }
    }
    return v2;
}

template <int MODE, int BONDS, int BLOCK, bool PADDED>
__global__ void __launch_bounds__(BLOCK, MD_SP_MIN_THREADS / BLOCK) k_sp_force(const __grid_constant__ MdDev P)
{
    __shared__ double sm[32];
    const int i = blockIdx.x * BLOCK + threadIdx.x;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    const float v2 = i < P.N ? sp_force_atom<MODE, BONDS, PADDED, LdNC>(P, pc, vc, i) : 0.0f;
    if (MODE == 1) {
        const double bm = block_max((double)v2, sm);
        if (threadIdx.x == 0) publish_vmax2(P, blockIdx.x, bm);
    }
}

// ---- the persistent kernel in binary32: md_kernels.cu:k_persist with the bodies above (see there for the structure) ----
namespace cg = cooperative_groups;

template <int BONDS, int MINB>
__global__ void __launch_bounds__(PERSIST_T, MINB) k_sp_persist(const __grid_constant__ MdDev P, long long n_steps)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ double sm[33];
    const int nblk = gridDim.x, tid = threadIdx.x;
    const int stride = nblk * PERSIST_T, first = blockIdx.x * PERSIST_T + tid;
    DecState c = dec_load(P);
    for (long long step = 0; step < n_steps; step++) {
        float v2 = 0.0f;
        for (int i = first; i < P.N; i += stride)
            v2 = fmaxf(v2, step == 0 ? sp_kick_drift_atom(P, c.p_dst, c.v_dst, i) : sp_force_atom<1, BONDS, false, LdPlain>(P, c.p_dst, c.v_dst, i));
        const double bm = block_max((double)v2, sm);
        double *vmax_buf = P.blk_vmax2 + DEC_SLOTS + (step & 1) * nblk;
        if (tid == 0) vmax_buf[blockIdx.x] = bm;
        grid.sync();
        double m = 0.0;
        for (int b = tid; b < nblk; b += PERSIST_T) m = fmax(m, __ldcg(vmax_buf + b));
        __syncthreads();
        m = block_max(m, sm);
        if (tid == 0) sm[32] = m;
        __syncthreads();
        decide_state(P, c, sm[32], step != 0);
        if (blockIdx.x == 0 && tid == 0) dec_store(P, c);
        if (c.need_rebuild) {
            const Bufs B = {c.p_src, c.p_dst, c.v_src, c.v_dst};
            sp_bin_body<LdPlain>(P, B);
            grid.sync();
            for (int t = blockIdx.x; t < P.scan_blocks; t += nblk) { scan_reduce_tile(P, t); __syncthreads(); }
            grid.sync();
            if (blockIdx.x == 0 && tid == 0) {
                int run = 0;
                for (int t = 0; t < P.scan_blocks; t++) { const int v = P.block_sums[t]; P.block_sums[t] = run; run += v; }
            }
            grid.sync();
            for (int t = blockIdx.x; t < P.scan_blocks; t += nblk) { scan_apply_tile<false>(P, t); __syncthreads(); }
            grid.sync();
            place_body(P);
            grid.sync();
            sp_reorder_body<LdPlain>(P, B);
            grid.sync();
            if (BONDS) { bonds_remap_body(P, B); grid.sync(); }
            sp_build_body<LdPlain>(P, B);
            grid.sync();
        }
    }
    for (int i = first; i < P.N; i += stride) sp_force_atom<2, BONDS, false, LdPlain>(P, c.p_dst, c.v_dst, i);
}

// F2 and the other sums: binary32 pair terms, binary64 accumulation
template <bool BONDS>
__global__ void __launch_bounds__(256) k_sp_energy(const __grid_constant__ MdDev P)
{
    __shared__ RedSmem S;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    const float4 *__restrict__ pos = P.posf[pc];
    double q[RED_N];
#pragma unroll
    for (int k = 0; k < RED_N; k++) q[k] = 0.0;
    if (i < P.N) {
        const float4 ri = ld4(pos + i);
        const int m = P.nnb[i];
        const int *__restrict__ w = P.W + (size_t)i * P.w_col;
        double u = 0.0, vir = 0.0;
#pragma unroll 2
        for (int k = 0; k < m; k++) {
            const unsigned en = (unsigned)__ldcs(w + (size_t)k * P.w_row);
            const float4 rj = ld4(pos + (en & W_INDEX_MASK));
            float dx, dy, dz;
            const float r2 = disp2f(ri, rj, en >> W_FLAG_SHIFT, P.Lf, dx, dy, dz);
            if (r2 < P.rc2f) {
                const float s = __frcp_rn(r2), s3 = s * s * s;
                u += (double)(4.0f * s3 * (s3 - 1.0f) - P.ucf);
                vir += (double)(48.0f * s3 * (s3 - 0.5f));          // fc * r^2
            }
        }
        q[RED_PE] = 0.5 * u;                                         // full list: every pair twice
        q[RED_VIR] = 0.5 * vir;
        if (BONDS) {
#pragma unroll
            for (int k = 0; k < 2; k++) {
                const int j = P.bond_dev[(size_t)k * P.N_pad + i];
                if (j < 0) continue;
                const float4 rj = ld4(pos + j);
                const float dx = minimgf(__fsub_rn(ri.x, rj.x), P.Lf, P.half_Lf), dy = minimgf(__fsub_rn(ri.y, rj.y), P.Lf, P.half_Lf),
                            dz = minimgf(__fsub_rn(ri.z, rj.z), P.Lf, P.half_Lf);
                const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                if (!(r2 < P.fene_R02f)) { set_err(P, MD_ERR_BOND_BROKEN); continue; }
                const float x = 1.0f - r2 / P.fene_R02f;
                q[RED_PEB] += 0.5 * (double)(-0.5f * P.fene_kf * P.fene_R02f * logf(x));
                q[RED_VIR] += 0.5 * (double)((-P.fene_kf / x) * r2);
            }
            if (P.has_dihedrals) {
#pragma unroll
                for (int k = 0; k < 2; k++) {
                    const int pk = P.bond_dev[(size_t)k * P.N_pad + i], qk = P.bond_dev[(size_t)(1 - k) * P.N_pad + i];
                    if (pk < 0 || qk < 0 || i > pk) continue;
                    const int o = chain_next_f(P, pk, i);
                    if (o < 0) continue;
                    PairAccF dummy = {0.0f, 0.0f, 0.0f};
                    const float c = dihedral_term_f(P, ld4(pos + qk), ri, ld4(pos + pk), ld4(pos + o), -1, dummy);
                    const float kf = (float)P.dih_k, c0 = (float)P.dih_c0;
                    q[RED_PEB] += (double)(0.5f * kf * (c - c0) * (c - c0));
                }
            }
            if (P.has_angles) {
                const int p0 = P.bond_dev[i], p1 = P.bond_dev[(size_t)P.N_pad + i];
                if (p0 >= 0 && p1 >= 0) {
                    float x1, y1, z1, x2, y2, z2;
                    const float n1 = mi_disp_f(P, ld4(pos + p0), ri, x1, y1, z1), n2 = mi_disp_f(P, ld4(pos + p1), ri, x2, y2, z2);
                    const float c = (x1 * x2 + y1 * y2 + z1 * z2) * (1.0f / sqrtf(n1 * n2));
                    const float k = (float)P.ang_k, c0 = (float)P.ang_c0;
                    q[RED_PEB] += (double)(0.5f * k * (c - c0) * (c - c0));
                }
            }
        }
        const float4 v = P.velf[vc][i];
        const double vx = v.x, vy = v.y, vz = v.z;
        const double v2 = vx * vx + vy * vy + vz * vz;
        q[RED_KE] = 0.5 * v2;
        q[RED_PX] = vx; q[RED_PY] = vy; q[RED_PZ] = vz;
        q[RED_VMAX2] = v2;
    }
    reduce_finish(P, q, S, blockIdx.x, gridDim.x);
}

inline int cdiv(long long a, int b) { return (int)((a + b - 1) / b); }
inline int capped_grid(const MdDev &P, long long n, int block, int per_sm) { return std::min(cdiv(n, block), P.sm_count * per_sm); }

template <int MODE, int BONDS, bool PADDED>
void launch_sp_force_p(const MdDev &P, int block, cudaStream_t st)
{
    switch (block) {
    case 64: k_sp_force<MODE, BONDS, 64, PADDED><<<cdiv(P.N, 64), 64, 0, st>>>(P); break;
    case 256: k_sp_force<MODE, BONDS, 256, PADDED><<<cdiv(P.N, 256), 256, 0, st>>>(P); break;
    case 512: k_sp_force<MODE, BONDS, 512, PADDED><<<cdiv(P.N, 512), 512, 0, st>>>(P); break;
    default: k_sp_force<MODE, BONDS, 128, PADDED><<<cdiv(P.N, 128), 128, 0, st>>>(P); break;
    }
}

template <int MODE, int BONDS>
void launch_sp_force(const MdDev &P, int block, cudaStream_t st)
{
    if (P.sp_pad > 1) launch_sp_force_p<MODE, BONDS, true>(P, block, st);
    else launch_sp_force_p<MODE, BONDS, false>(P, block, st);
}

}  // namespace

// the persistent launch of md_kernels.cu (mdk_persist_ok / mdk_persist_steps) in binary32: kernel and grid
namespace {
template <int MINB>
const void *sp_persist_kernel(const MdDev &P) { return P.has_bonds ? (const void *)k_sp_persist<1, MINB> : (const void *)k_sp_persist<0, MINB>; }
}  // namespace

int mdk_sp_persist_choice(const MdDev &P, const void **kernel)
{
    const int want = cdiv(P.N, PERSIST_T);
    int per_sm = 0;
    const void *k = sp_persist_kernel<2>(P);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, PERSIST_T, 0) == cudaSuccess && per_sm >= 1 && want <= per_sm * P.sm_count) {
        *kernel = k;
        return want;
    }
    k = sp_persist_kernel<4>(P);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, PERSIST_T, 0) == cudaSuccess && per_sm >= 1) {
        *kernel = k;
        return std::min(want, per_sm * P.sm_count);
    }
    cudaGetLastError();
    *kernel = nullptr;
    return 0;
}

void mdk_sp_load_state(const MdDev &P, cudaStream_t st) { k_sp_load_state<<<cdiv(P.N, 256), 256, 0, st>>>(P); }
void mdk_sp_export(const MdDev &P, int what, double *dst, cudaStream_t st) { k_sp_export<<<cdiv(P.N, 256), 256, 0, st>>>(P, what, dst); }
void mdk_sp_kick_drift(const MdDev &P, cudaStream_t st) { k_sp_kick_drift<<<cdiv(P.N, 256), 256, 0, st>>>(P); }
void mdk_sp_kick(const MdDev &P, cudaStream_t st) { k_sp_kick<<<cdiv(P.N, 256), 256, 0, st>>>(P); }
void mdk_sp_bin(const MdDev &P, cudaStream_t st) { k_sp_bin<<<capped_grid(P, P.N, 256, 8), 256, 0, st>>>(P); }
void mdk_sp_reorder(const MdDev &P, cudaStream_t st) { k_sp_reorder<<<capped_grid(P, P.N, 256, 8), 256, 0, st>>>(P); }
void mdk_sp_build(const MdDev &P, cudaStream_t st) { k_sp_build<<<capped_grid(P, P.N, 128, 16), 128, 0, st>>>(P); }

void mdk_sp_force(const MdDev &P, const MdLaunch &lc, int mode, cudaStream_t st)
{
    if (P.has_bonds && (P.has_angles || P.has_dihedrals)) {
        if (mode == 0) launch_sp_force<0, 2>(P, lc.block, st);
        else if (mode == 1) launch_sp_force<1, 2>(P, lc.block, st);
        else launch_sp_force<2, 2>(P, lc.block, st);
    } else if (P.has_bonds) {
        if (mode == 0) launch_sp_force<0, 1>(P, lc.block, st);
        else if (mode == 1) launch_sp_force<1, 1>(P, lc.block, st);
        else launch_sp_force<2, 1>(P, lc.block, st);
    } else {
        if (mode == 0) launch_sp_force<0, 0>(P, lc.block, st);
        else if (mode == 1) launch_sp_force<1, 0>(P, lc.block, st);
        else launch_sp_force<2, 0>(P, lc.block, st);
    }
}

void mdk_sp_energy(const MdDev &P, cudaStream_t st)
{
    const int grid = cdiv(P.N, 256);
    if (P.has_bonds) k_sp_energy<true><<<grid, 256, 0, st>>>(P);
    else k_sp_energy<false><<<grid, 256, 0, st>>>(P);
}
