// CUDA kernels (sm_100a) of the short-range MD hot path.  One thread per atom replaces every atom loop
// of the serial program.  Steps are named after the paper's list:
//   N1/N2  k_bin            cell assignment c_i and in-cell slot l_i by atomic occupancy counting
//   N3/N4  k_scan_*         prefix scan of the occupancies k_c (the GPU alternative the paper describes in
//                           sec. 2.4(4)) -> CSR cell_start; replaces the dense cell x layer matrix H
//          k_place/k_reorder  cell-order sort of the atoms at EVERY rebuild (paper: every 100 steps)
//   N5     k_build          neighbor matrix W[m][i], row m contiguous over atoms, with the
//                           periodic-image flag bits of PAPER.md:163 in the top 3 bits of every entry
//   F1     k_force          pair forces over W, no Newton-3 (variant A) / k_force_n3 half list + atomics (variant B)
//   F2     k_energy         block reductions finished by the last block
//          k_kick_drift / k_kick   leapfrog integration
// The model arithmetic follows DESIGN.md "Readings" (R1..R9).  No code is shared with oracle/.
//
// Periodic boundaries (R9).  Coordinates are wrapped into [0, L) only when the atoms are re-sorted
// (k_reorder) and on output (k_export); between rebuilds they may stray outside the box by at most
// r_shell/2.  That keeps the image flags frozen into W at build time valid for the life of the matrix,
// which is the condition the paper's flag-bit scheme needs.
#include <algorithm>

#include <cooperative_groups.h>

#include "md_device.cuh"
#include "md_rebuild.cuh"

namespace {

// ------------------------------------------------------------------------------------------------
// control / staging kernels
// ------------------------------------------------------------------------------------------------
__global__ void k_force_rebuild(const __grid_constant__ MdDev P)
{
    DevCtrl *c = P.ctrl;
    c->need_rebuild = 1;
    c->p_src = c->p_dst; c->p_dst ^= 1;
    c->v_src = c->v_dst; c->v_dst ^= 1;
    c->disp_acc = 0.0;
    c->max_occ = 0; c->max_nnb = 0; c->nnb_total = 0ull; c->cand_total = 0ull;
    c->do_reorder = !P.layer_H || P.reorder_interval >= 0;      // a forced rebuild sorts unless the system never does
    c->since_reorder = 0;
}

// md_set_state's argument check, on the device: every coordinate of scratch[0 .. 3N) must lie in [0, box] (NaN fails).
// (On the host this loop over 6.3 M doubles cost more than the H2D copy of the state at N = 2M.)
__global__ void k_check_range(const __grid_constant__ MdDev P, double box)
{
    const size_t n3 = 3 * (size_t)P.N;
    bool bad = false;
    for (size_t k = blockIdx.x * (size_t)blockDim.x + threadIdx.x; k < n3; k += (size_t)gridDim.x * blockDim.x) {
        const double x = P.scratch[k];
        bad |= !(x >= 0.0 && x <= box);
    }
    if (bad) set_err(P, MD_ERR_INVALID);
}

// scratch = [xyz (3N) | vxyz (3N)] in original-id order -> device arrays in identity order
__global__ void k_load_state(const __grid_constant__ MdDev P)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const int pc = P.ctrl->p_dst, vc = P.ctrl->v_dst;
    const double *s = P.scratch + 3 * (size_t)i;
    double x = wrap1(s[0], P.L), y = wrap1(s[1], P.L), z = wrap1(s[2], P.L);
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) set_err(P, MD_ERR_NONFINITE);
    st_pos(P.pos[pc] + i, x, y, z);
    const double *v = P.scratch + 3 * (size_t)P.N + 3 * (size_t)i;
    double *vel = P.vel[vc];
    vel[i] = v[0]; vel[P.N_pad + i] = v[1]; vel[2 * (size_t)P.N_pad + i] = v[2];
    P.id[vc][i] = i;
}

// device order -> dst (device, 3N doubles) in original-id order.  what: 0 positions (wrapped into [0, L)), 1 velocities, 2 forces
__global__ void k_export(const __grid_constant__ MdDev P, int what, double *dst)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const int pc = P.ctrl->p_dst, vc = P.ctrl->v_dst;
    const int id = P.id[vc][i];
    double *o = dst + 3 * (size_t)id;
    if (what == 0) {
        const pos_t r = ld_pos_rw(P.pos[pc] + i);
        o[0] = wrap1(r.x, P.L); o[1] = wrap1(r.y, P.L); o[2] = wrap1(r.z, P.L);
    } else {
        const double *a = what == 1 ? P.vel[vc] : P.frc;
        o[0] = a[i]; o[1] = a[P.N_pad + i]; o[2] = a[2 * (size_t)P.N_pad + i];
    }
}

// ------------------------------------------------------------------------------------------------
// integration (split mode): first half kick + drift + max velocity + rebuild decision
// ------------------------------------------------------------------------------------------------
// opening half kick + drift of atom i; returns |v|^2
__device__ __forceinline__ double kick_drift_atom(const MdDev &P, int pc, int vc, int i)
{
    pos_t *pp = P.pos[pc] + i;
    double *vx = P.vel[vc] + i, *vy = vx + P.N_pad, *vz = vy + P.N_pad;
    const double *fx = P.frc + i, *fy = fx + P.N_pad, *fz = fy + P.N_pad;
    const pos_t r = ld_pos_rw(pp);
    const double ax = *vx + P.hdt * *fx, ay = *vy + P.hdt * *fy, az = *vz + P.hdt * *fz;
    *vx = ax; *vy = ay; *vz = az;
    const double x = r.x + P.dt * ax, y = r.y + P.dt * ay, z = r.z + P.dt * az;
    st_pos(pp, x, y, z);
    double v2 = ax * ax + ay * ay + az * az;
    if (!isfinite(v2 + x + y + z)) { set_err(P, MD_ERR_NONFINITE); v2 = 0.0; }
    return v2;
}

__global__ void __launch_bounds__(256) k_kick_drift(const __grid_constant__ MdDev P)
{
    __shared__ double sm[32];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    const double v2 = i < P.N ? kick_drift_atom(P, pc, vc, i) : 0.0;
    const double bm = block_max(v2, sm);
    if (threadIdx.x == 0) publish_vmax2(P, blockIdx.x, bm);
}

// max over the per-block maxima of v^2, then the rebuild decision: one block, ordered after the drifting kernel
// by the stream.  Inside md_step's CUDA graph it also sets the condition of the IF node that holds the rebuild chain.
__global__ void __launch_bounds__(DEC_SLOTS) k_decide(const __grid_constant__ MdDev P, int pos_pingpong, cudaGraphConditionalHandle cond)
{
    __shared__ double sm[32];
    // read and clear this thread's slot (publish_vmax2): the next drifting kernel starts from zeros
    double m = __longlong_as_double((long long)atomicExch(reinterpret_cast<unsigned long long *>(P.blk_vmax2) + threadIdx.x, 0ull));
    m = block_max(m, sm);
    if (threadIdx.x == 0) {
        decide(P, m, pos_pingpong != 0);
        if (cond) cudaGraphSetConditional(cond, (unsigned)P.ctrl->need_rebuild);
    }
}

// second half kick
__global__ void __launch_bounds__(256) k_kick(const __grid_constant__ MdDev P)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const int vc = __ldcg(&P.ctrl->v_dst);
    double *v = P.vel[vc] + i;
    const double *f = P.frc + i;
#pragma unroll
    for (int k = 0; k < 3; k++) v[(size_t)k * P.N_pad] += P.hdt * f[(size_t)k * P.N_pad];
}

// ------------------------------------------------------------------------------------------------
// cells: N1/N2 binning with atomic occupancy counters, N3/N4 as a prefix scan.  The rebuild kernels use
// grid-stride loops over a capped grid: a launch that finds need_rebuild == 0 retires in ~2 us.
// ------------------------------------------------------------------------------------------------
template <class LD>
__device__ __forceinline__ void bin_body(const MdDev &P, const Bufs B)
{
    const pos_t *__restrict__ pos = P.pos[B.ps];
    const int *__restrict__ idv = P.id[B.vs];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += gridDim.x * blockDim.x) {
        const pos_t r = LD::pos(pos + i);
        const int cx = cell_coord(wrap1(r.x, P.L), P.inv_wx, P.ncx), cy = cell_coord(wrap1(r.y, P.L), P.inv_w, P.nc),
                  cz = cell_coord(wrap1(r.z, P.L), P.inv_w, P.nc);
        // batched independent systems: each has its own block of cells, found from the permanent id
        const int sys = P.n_sys > 1 ? LD::i32(idv + i) / P.N1 : 0;
        const int c = sys * P.NC1 + cx + P.ncx * (cy + P.nc * cz);
        P.cell_of[i] = c;
        P.slot[i] = atomicAdd(&P.cell_count[c], 1);  // l_i; "incrementing k_c requires an atomic operation" (N2)
    }
}

__global__ void __launch_bounds__(256) k_bin(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    bin_body<LdNC>(P, bufs_from_ctrl(P));
}

__global__ void __launch_bounds__(SCAN_T) k_scan_reduce(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    scan_reduce_tile(P, blockIdx.x);
}

__global__ void __launch_bounds__(SCAN_T) k_scan_apply(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    scan_apply_tile<true>(P, blockIdx.x);
}

__global__ void __launch_bounds__(256) k_place(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    if (P.layer_H && !__ldcg(&P.ctrl->do_reorder)) return;
    place_body(P);
}

// Cell-order gather of r, v and the permanent serial numbers; coordinates are wrapped into
// [0, L) here.  The atomics of N2 leave the order inside a cell indeterminate; ranking the
// cell's members by their previous slot makes the order -- and with it every floating-point sum downstream --
// reproducible run to run.
template <class LD>
__device__ __forceinline__ void reorder_body(const MdDev &P, const Bufs B)
{
    const int ps = B.ps, pd = B.pd, vs = B.vs, vd = B.vd;
    const pos_t *__restrict__ pin = P.pos[ps];
    const double *__restrict__ vin = P.vel[vs];
    const int *__restrict__ idin = P.id[vs];
    for (int p = blockIdx.x * blockDim.x + threadIdx.x; p < P.N; p += gridDim.x * blockDim.x) {
        const int a = P.perm[p];
        // issue the payload loads first; the rank search below overlaps with their latency
        const pos_t r = LD::pos(pin + a);
        const double vx = LD::f64(vin + a), vy = LD::f64(vin + P.N_pad + a), vz = LD::f64(vin + 2 * (size_t)P.N_pad + a);
        const int id = LD::i32(idin + a);
        const int c = P.cell_of[a];
        const int s = P.cell_start[c], e = P.cell_start[c + 1];
        int rank = 0;
        for (int q = s; q < e; q++) rank += (P.perm[q] < a);
        const int n = s + rank;
        st_pos(P.pos[pd] + n, wrap1(r.x, P.L), wrap1(r.y, P.L), wrap1(r.z, P.L));
        double *vo = P.vel[vd] + n;
        vo[0] = vx; vo[P.N_pad] = vy; vo[2 * (size_t)P.N_pad] = vz;
        P.id[vd][n] = id;
        if (P.need_inv) P.inv[id] = n;
    }
}

__global__ void __launch_bounds__(256) k_reorder(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    if (P.layer_H && !__ldcg(&P.ctrl->do_reorder)) return;
    reorder_body<LdNC>(P, bufs_from_ctrl(P));
}


__global__ void __launch_bounds__(256) k_bonds_remap(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    bonds_remap_body(P, bufs_from_ctrl(P));
}

// ------------------------------------------------------------------------------------------------
// N5: neighbor matrix.  With the atoms in cell order (x fastest) the stencil of an atom is 9 contiguous runs of the
// atom array, one per row of cells (dy, dz): the atoms of the 2 k + 1 fine cells around the atom's own (k <= kx, fewer
// where the row is too far for the full width: row_halfwidth), plus a wrapped piece at the periodic x faces.
// One thread per atom walks its candidates run by run; the next candidate's position is fetched while the current
// one is tested.
// The periodic image is a per-run shift (0, +L or -L per axis) added to the raw difference.  For every pair
// closer than r_n this is exactly the minimum-image arithmetic of DESIGN.md R5 (d0 = a - b rounded, then
// d0 -+ L rounded): with cells wider than r_n and >= 3 cells per edge the image reached through the
// stencil is the minimum image, and a pair for which it is not is farther than r_n in either form.
// ------------------------------------------------------------------------------------------------
// candidates j in [b, e) of one run, image shift (sx, sy, sz) and flag bits fl for the whole run
// EXCL: rigid molecules -- sites of the atom's own molecule (mol = original id / sites per molecule) are no neighbors
template <bool HALF, bool SHIFT, bool EXCL, class LD>
__device__ __forceinline__ void scan_run(const MdDev &P, const pos_t *__restrict__ pos, const pos_t &ri, int i, int b, int e,
                                         double sx, double sy, double sz, unsigned fl, int &m, const int *__restrict__ idv, int mol)
{
    for (int j = b; j < e; j++) {
        if (EXCL && LD::i32(idv + j) / P.rb_ns == mol) continue;
        const pos_t rj = LD::pos(pos + j);
        // d = (r_i - r_j) + shift, each operation rounded once
        double dx = __dsub_rn(ri.x, rj.x), dy = __dsub_rn(ri.y, rj.y), dz = __dsub_rn(ri.z, rj.z);
        if (SHIFT) { dx = __dadd_rn(dx, sx); dy = __dadd_rn(dy, sy); dz = __dadd_rn(dz, sz); }
        const double r2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
        if (r2 < P.rn2 && (HALF ? (j > i) : (j != i))) {
            if (m < P.Mmax) P.W[(size_t)m * P.w_row + (size_t)i * P.w_col] = (int)((unsigned)j | (fl << W_FLAG_SHIFT));
            m++;
        }
    }
}

template <bool HALF, bool EXCL, class LD>
__device__ __forceinline__ void build_body(const MdDev &P, const Bufs B)
{
    __shared__ int smx[32], scand[32];
    __shared__ int ssum[32];
    const pos_t *__restrict__ pos = P.pos[B.pd];
    const int *__restrict__ cs = P.cell_start;
    const int *__restrict__ idv = P.id[B.vd];
    const int nc = P.nc, ncx = P.ncx;
    const double L = P.L;
    int tmax = 0, tsum = 0, tcand = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += gridDim.x * blockDim.x) {
        const pos_t ri = LD::pos(pos + i);
        const int cx = cell_coord(ri.x, P.inv_wx, ncx), cy = cell_coord(ri.y, P.inv_w, nc), cz = cell_coord(ri.z, P.inv_w, nc);
        const RowGaps gaps = row_gaps(P, ri.y, ri.z, cy, cz);
        const int cell_base = P.n_sys > 1 ? (LD::i32(idv + i) / P.N1) * P.NC1 : 0;     // the atom's own system of cells
        const int mol = EXCL ? LD::i32(idv + i) / P.rb_ns : 0;
        int m = 0;
        for (int dz = -1; dz <= 1; dz++) {
            int z = cz + dz;
            double sz = 0.0;
            unsigned fz = 0u;
            if (z < 0) { z += nc; sz = L; fz = 4u; } else if (z >= nc) { z -= nc; sz = -L; fz = 4u; }
            for (int dy = -1; dy <= 1; dy++) {
                const int kr = row_halfwidth(P, gaps, dy, dz);
                if (kr < 0) continue;
                int y = cy + dy;
                double sy = 0.0;
                unsigned fl = fz;
                if (y < 0) { y += nc; sy = L; fl |= 2u; } else if (y >= nc) { y -= nc; sy = -L; fl |= 2u; }
                const int row = cell_base + ncx * (y + nc * z);
                const int lo = cx - kr, hi = cx + kr;
                const int b = LD::i32(cs + row + (lo < 0 ? 0 : lo)), e = LD::i32(cs + row + (hi >= ncx ? ncx : hi + 1));
                tcand += e - b;
                if (fl) scan_run<HALF, true, EXCL, LD>(P, pos, ri, i, b, e, 0.0, sy, sz, fl, m, idv, mol);
                else scan_run<HALF, false, EXCL, LD>(P, pos, ri, i, b, e, 0.0, 0.0, 0.0, 0u, m, idv, mol);
                // the part of the window beyond a periodic x face: the cells at the other end of the row, shifted by +-L
                if (lo < 0) scan_run<HALF, true, EXCL, LD>(P, pos, ri, i, LD::i32(cs + row + ncx + lo), LD::i32(cs + row + ncx), L, sy, sz, fl | 1u, m, idv, mol);
                if (hi >= ncx) scan_run<HALF, true, EXCL, LD>(P, pos, ri, i, LD::i32(cs + row), LD::i32(cs + row + hi - ncx + 1), -L, sy, sz, fl | 1u, m, idv, mol);
            }
        }
        P.nnb[i] = m < P.Mmax ? m : P.Mmax;
        if (m > P.Mmax) set_err(P, MD_ERR_NEBR_OVERFLOW);
        tmax = max(tmax, m);
        tsum += m;
    }
    // statistics of the matrix (md_energy.max_neighbors / mean_neighbors)
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

template <bool HALF, bool EXCL>
__global__ void __launch_bounds__(128) k_build(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    build_body<HALF, EXCL, LdNC>(P, bufs_from_ctrl(P));
}

// ------------------------------------------------------------------------------------------------
// Ablation MD_FLAG_LAYER_H: the paper's own cell structure and sort schedule.
//   N1/N2  k_bin as above: c_i and the layer l_i = atomicAdd(k_c)
//   N3     max occupancy from the scan kernels (ctrl->max_occ); H has a fixed N_l = P.n_layers columns
//   N4     k_layer_fill: H[c_i][l_i] = i
//   N5     k_build_layers: for every cell of the stencil, for every layer l < k_c: i' = H[c][l]
// The atoms are re-sorted into cell order only when decide() says so (every reorder_interval steps); at the
// other rebuilds k_copy_wrap moves them to the other buffers in place (the rebuild chain always changes buffers).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_copy_wrap(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild) || __ldcg(&P.ctrl->do_reorder)) return;
    const int ps = __ldcg(&P.ctrl->p_src), pd = __ldcg(&P.ctrl->p_dst);
    const int vs = __ldcg(&P.ctrl->v_src), vd = __ldcg(&P.ctrl->v_dst);
    const size_t np = (size_t)P.N_pad;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += gridDim.x * blockDim.x) {
        const pos_t r = ld_pos(P.pos[ps] + i);
        st_pos(P.pos[pd] + i, wrap1(r.x, P.L), wrap1(r.y, P.L), wrap1(r.z, P.L));
        const double *vi = P.vel[vs] + i;
        double *vo = P.vel[vd] + i;
        vo[0] = vi[0]; vo[np] = vi[np]; vo[2 * np] = vi[2 * np];
        const int id = P.id[vs][i];
        P.id[vd][i] = id;
        if (P.need_inv) P.inv[id] = i;
    }
}

__global__ void __launch_bounds__(256) k_layer_fill(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    const bool sorted = __ldcg(&P.ctrl->do_reorder) != 0;
    const pos_t *__restrict__ pos = P.pos[__ldcg(&P.ctrl->p_dst)];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += gridDim.x * blockDim.x) {
        int c, l;
        if (sorted) {        // after the sort the layer is the atom's rank inside its cell
            const pos_t r = ld_pos(pos + i);
            c = cell_coord(r.x, P.inv_w, P.nc) + P.nc * (cell_coord(r.y, P.inv_w, P.nc) + P.nc * cell_coord(r.z, P.inv_w, P.nc));
            l = i - P.cell_start[c];
        } else {             // atoms stayed in place: c_i and the atomic slot l_i of k_bin
            c = P.cell_of[i];
            l = P.slot[i];
        }
        if (l >= P.n_layers) { set_err(P, MD_ERR_CELL_OVERFLOW); continue; }
        P.H[(size_t)c * P.n_layers + l] = i;
    }
}

__global__ void __launch_bounds__(128) k_build_layers(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    __shared__ int smx[4];
    __shared__ int ssum[4];
    const pos_t *__restrict__ pos = P.pos[__ldcg(&P.ctrl->p_dst)];
    const int *__restrict__ cs = P.cell_start;
    const int nc = P.nc, NL = P.n_layers;
    const double L = P.L;
    int tmax = 0, tsum = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += gridDim.x * blockDim.x) {
        const pos_t ri = ld_pos(pos + i);
        const int cx = cell_coord(ri.x, P.inv_w, nc), cy = cell_coord(ri.y, P.inv_w, nc), cz = cell_coord(ri.z, P.inv_w, nc);
        int m = 0;
        for (int dz = -1; dz <= 1; dz++) {
            int z = cz + dz;
            double sz = 0.0;
            unsigned fz = 0u;
            if (z < 0) { z += nc; sz = L; fz = 4u; } else if (z >= nc) { z -= nc; sz = -L; fz = 4u; }
            for (int dy = -1; dy <= 1; dy++) {
                int y = cy + dy;
                double sy = 0.0;
                unsigned fy = fz;
                if (y < 0) { y += nc; sy = L; fy |= 2u; } else if (y >= nc) { y -= nc; sy = -L; fy |= 2u; }
                for (int dx = -1; dx <= 1; dx++) {
                    int x = cx + dx;
                    double sx = 0.0;
                    unsigned fl = fy;
                    if (x < 0) { x += nc; sx = L; fl |= 1u; } else if (x >= nc) { x -= nc; sx = -L; fl |= 1u; }
                    const int c = x + nc * (y + nc * z);
                    const int kc = min(__ldg(cs + c + 1) - __ldg(cs + c), NL);        // k_c: occupancy from the scan
                    const int *__restrict__ h = P.H + (size_t)c * NL;
                    for (int l = 0; l < kc; l++) {
                        const int j = __ldg(h + l);
                        const pos_t rj = ld_pos(pos + j);
                        // d = (r_i - r_j) + shift, each operation rounded once (+0.0 is exact): DESIGN.md R5
                        const double ddx = __dadd_rn(__dsub_rn(ri.x, rj.x), sx), ddy = __dadd_rn(__dsub_rn(ri.y, rj.y), sy),
                                     ddz = __dadd_rn(__dsub_rn(ri.z, rj.z), sz);
                        const double r2 = __fma_rn(ddz, ddz, __fma_rn(ddy, ddy, __dmul_rn(ddx, ddx)));
                        if (r2 < P.rn2 && j != i) {
                            if (m < P.Mmax) P.W[(size_t)m * P.w_row + (size_t)i * P.w_col] = (int)((unsigned)j | (fl << W_FLAG_SHIFT));
                            m++;
                        }
                    }
                }
            }
        }
        P.nnb[i] = m < P.Mmax ? m : P.Mmax;
        if (m > P.Mmax) set_err(P, MD_ERR_NEBR_OVERFLOW);
        tmax = max(tmax, m);
        tsum += m;
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int wm = warp_max_i(tmax), ws = warp_sum_i(tsum);
    if (lane == 0) { smx[wid] = wm; ssum[wid] = ws; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int mx = 0, sm = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) { mx = max(mx, smx[w]); sm += ssum[w]; }
        atomicMax(&P.ctrl->max_nnb, mx);
        atomicAdd(&P.ctrl->nnb_total, (unsigned long long)sm);
    }
}

// ------------------------------------------------------------------------------------------------
// F1: pair forces.  Thread i walks column i of W; row m is contiguous over i, so the 32 threads of a
// warp read 128 consecutive bytes of W per row; the partner positions are gathers.
// W streams from HBM once per step while the positions stay in L2, so the index loads run U rows ahead of
// the gathers that depend on them (two dependent memory latencies would otherwise serialise per neighbor).
// ------------------------------------------------------------------------------------------------
struct PairAcc {
    double fx, fy, fz;
};

__device__ __forceinline__ void pair_force(const MdDev &P, const pos_t &ri, const pos_t &rj, unsigned fl, PairAcc &a)
{
    double dx, dy, dz;
    const double r2 = disp2(ri, rj, fl, P.L, dx, dy, dz);
    if (r2 < P.rc2) {
        const double s = fast_rcp(r2), s3 = s * s * s;
        const double fc = s3 * (s3 - 0.5) * s;          // x 48 applied once to the sums
        a.fx += fc * dx; a.fy += fc * dy; a.fz += fc * dz;
    }
}

// minimum-image r_a - r_b (R5 arithmetic), squared length returned
__device__ __forceinline__ double mi_disp(const MdDev &P, const pos_t &a, const pos_t &b, double &dx, double &dy, double &dz)
{
    dx = minimg(a.x - b.x, P.L, P.half_L); dy = minimg(a.y - b.y, P.L, P.half_L); dz = minimg(a.z - b.z, P.L, P.half_L);
    return __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
}

// Bond-angle terms ("bond-angle torque"; R19): U = k/2 (cos(theta) - c0)^2 at every atom with
// two bonded partners.  "One thread per atom handles all its interactions": atom i collects its force
// from the angle it is the vertex of and from the (up to two) angles it ends, found through its partners' partners.
// With d1 = r_end - r_vertex, d2 = r_other_end - r_vertex, c = d1.d2/(|d1||d2|), g = -k (c - c0):
//   force on the end atom of d1: g (d2/(|d1||d2|) - c d1/|d1|^2);  on the vertex: minus the sum of both ends.
__device__ __forceinline__ void angle_force(const MdDev &P, const pos_t *__restrict__ pos, const pos_t &ri, int i, PairAcc &a)
{
    const int p[2] = {P.bond_dev[i], P.bond_dev[(size_t)P.N_pad + i]};
    pos_t rp[2];
#pragma unroll
    for (int k = 0; k < 2; k++)
        if (p[k] >= 0) rp[k] = ld_pos(pos + p[k]);
    if (p[0] >= 0 && p[1] >= 0) {                       // i is the vertex
        double x1, y1, z1, x2, y2, z2;
        const double n1 = mi_disp(P, rp[0], ri, x1, y1, z1), n2 = mi_disp(P, rp[1], ri, x2, y2, z2);
        const double inv12 = 1.0 / sqrt(n1 * n2), c = (x1 * x2 + y1 * y2 + z1 * z2) * inv12;
        const double g = -P.ang_k * (c - P.ang_c0), u1 = c / n1, u2 = c / n2;
        // -(f_a + f_c)
        a.fx -= g * ((x2 * inv12 - u1 * x1) + (x1 * inv12 - u2 * x2));
        a.fy -= g * ((y2 * inv12 - u1 * y1) + (y1 * inv12 - u2 * y2));
        a.fz -= g * ((z2 * inv12 - u1 * z1) + (z1 * inv12 - u2 * z2));
    }
#pragma unroll
    for (int k = 0; k < 2; k++) {                       // i ends the angle whose vertex is its partner p[k]
        if (p[k] < 0) continue;
        const int q0 = P.bond_dev[p[k]], q1 = P.bond_dev[(size_t)P.N_pad + p[k]];
        const int q = q0 == i ? q1 : q0;
        if (q < 0) continue;
        const pos_t rq = ld_pos(pos + q);
        double x1, y1, z1, x2, y2, z2;
        const double n1 = mi_disp(P, ri, rp[k], x1, y1, z1), n2 = mi_disp(P, rq, rp[k], x2, y2, z2);
        const double inv12 = 1.0 / sqrt(n1 * n2), c = (x1 * x2 + y1 * y2 + z1 * z2) * inv12;
        const double g = -P.ang_k * (c - P.ang_c0), u1 = c / n1;
        a.fx += g * (x2 * inv12 - u1 * x1);
        a.fy += g * (y2 * inv12 - u1 * y1);
        a.fz += g * (z2 * inv12 - u1 * z1);
    }
}

// Dihedral terms ("optional dihedral"; R19): U = k/2 (cos(phi) - c0)^2 for every four consecutive
// beads a-b-c-d, cos(phi) = A.B/(|A||B|), A = b1 x b2, B = b2 x b3, b1 = r_b - r_a, b2 = r_c - r_b, b3 = r_d - r_c.
// With gA = B/(|A||B|) - c A/|A|^2, gB = A/(|A||B|) - c B/|B|^2:
//   dc/db1 = b2 x gA, dc/db2 = gA x b1 + b3 x gB, dc/db3 = gB x b2,
//   dc/dr_a = -dc/db1, dc/dr_b = dc/db1 - dc/db2, dc/dr_c = dc/db2 - dc/db3, dc/dr_d = dc/db3;  f = -k (c - c0) dc/dr.
struct V3 {
    double x, y, z;
};
__device__ __forceinline__ V3 cross3(const V3 &u, const V3 &v) { return {u.y * v.z - u.z * v.y, u.z * v.x - u.x * v.z, u.x * v.y - u.y * v.x}; }
__device__ __forceinline__ V3 mi_vec(const MdDev &P, const pos_t &a, const pos_t &b)
{
    V3 d;
    mi_disp(P, a, b, d.x, d.y, d.z);
    return d;
}

// cos(phi) of a-b-c-d and, if WHICH >= 0, the force on atom WHICH (0 = a .. 3 = d) added to acc
__device__ __forceinline__ double dihedral_term(const MdDev &P, const pos_t &ra, const pos_t &rb, const pos_t &rc, const pos_t &rd, int which,
                                                PairAcc &acc)
{
    const V3 b1 = mi_vec(P, rb, ra), b2 = mi_vec(P, rc, rb), b3 = mi_vec(P, rd, rc);
    const V3 A = cross3(b1, b2), B = cross3(b2, b3);
    const double nA = A.x * A.x + A.y * A.y + A.z * A.z, nB = B.x * B.x + B.y * B.y + B.z * B.z;
    const double invAB = 1.0 / sqrt(nA * nB), c = (A.x * B.x + A.y * B.y + A.z * B.z) * invAB;
    if (which < 0) return c;
    const double uA = c / nA, uB = c / nB;
    const V3 gA = {B.x * invAB - uA * A.x, B.y * invAB - uA * A.y, B.z * invAB - uA * A.z};
    const V3 gB = {A.x * invAB - uB * B.x, A.y * invAB - uB * B.y, A.z * invAB - uB * B.z};
    const V3 g1 = cross3(b2, gA), t1 = cross3(gA, b1), t2 = cross3(b3, gB), g3 = cross3(gB, b2);
    const V3 g2 = {t1.x + t2.x, t1.y + t2.y, t1.z + t2.z};
    V3 d;
    if (which == 0) d = {-g1.x, -g1.y, -g1.z};
    else if (which == 1) d = {g1.x - g2.x, g1.y - g2.y, g1.z - g2.z};
    else if (which == 2) d = {g2.x - g3.x, g2.y - g3.y, g2.z - g3.z};
    else d = g3;
    const double g = -P.dih_k * (c - P.dih_c0);
    acc.fx += g * d.x; acc.fy += g * d.y; acc.fz += g * d.z;
    return c;
}

// the partner of x other than prev (-1 at a chain end)
__device__ __forceinline__ int chain_next(const MdDev &P, int x, int prev)
{
    const int q0 = P.bond_dev[x], q1 = P.bond_dev[(size_t)P.N_pad + x];
    return q0 == prev ? q1 : q0;
}

// atom i collects its force from the (up to four) dihedrals it belongs to, found by walking three bonds either way.
// Not inlined: its ~60 live fp64 values would otherwise spill inside the force kernels even when the terms are off.
__device__ __noinline__ void dihedral_force(const MdDev &P, const pos_t *__restrict__ pos, const pos_t &ri, int i, PairAcc &a)
{
    const int L1 = P.bond_dev[i], R1 = P.bond_dev[(size_t)P.N_pad + i];
    const int L2 = L1 >= 0 ? chain_next(P, L1, i) : -1, L3 = L2 >= 0 ? chain_next(P, L2, L1) : -1;
    const int R2 = R1 >= 0 ? chain_next(P, R1, i) : -1, R3 = R2 >= 0 ? chain_next(P, R2, R1) : -1;
    pos_t l1, l2, l3, r1, r2, r3;
    if (L1 >= 0) l1 = ld_pos(pos + L1);
    if (L2 >= 0) l2 = ld_pos(pos + L2);
    if (L3 >= 0) l3 = ld_pos(pos + L3);
    if (R1 >= 0) r1 = ld_pos(pos + R1);
    if (R2 >= 0) r2 = ld_pos(pos + R2);
    if (R3 >= 0) r3 = ld_pos(pos + R3);
    if (L3 >= 0) dihedral_term(P, l3, l2, l1, ri, 3, a);
    if (L2 >= 0 && R1 >= 0) dihedral_term(P, l2, l1, ri, r1, 2, a);
    if (L1 >= 0 && R2 >= 0) dihedral_term(P, l1, ri, r1, r2, 1, a);
    if (R3 >= 0) dihedral_term(P, ri, r1, r2, r3, 0, a);
}

// EXTRAS: the angle / dihedral code is compiled in (kernels instantiated without it keep the registers of the FENE-only path)
template <bool CHECK, bool EXTRAS = true, class LD = LdNC>
__device__ __forceinline__ void bond_force(const MdDev &P, const pos_t *__restrict__ pos, const pos_t &ri, int i, PairAcc &a)
{
    if (EXTRAS && P.has_angles) angle_force(P, pos, ri, i, a);
    if (EXTRAS && P.has_dihedrals) dihedral_force(P, pos, ri, i, a);
#pragma unroll
    for (int k = 0; k < 2; k++) {
        const int j = P.bond_dev[(size_t)k * P.N_pad + i];
        if (j < 0) continue;
        const pos_t rj = LD::pos(pos + j);
        const double dx = minimg(ri.x - rj.x, P.L, P.half_L), dy = minimg(ri.y - rj.y, P.L, P.half_L),
                     dz = minimg(ri.z - rj.z, P.L, P.half_L);
        const double r2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
        if (!(r2 < P.fene_R02)) { if (CHECK) set_err(P, MD_ERR_BOND_BROKEN); continue; }
        // -k / (1 - r^2 / R0^2) = -k R0^2 / (R0^2 - r^2) with the refined hardware reciprocal (md_device.cuh: fast_rcp, ~1 ulp):
        // two IEEE divisions per bond were as many instructions as five pair terms
        const double fc = -(P.fene_k * P.fene_R02) * fast_rcp(P.fene_R02 - r2);
        a.fx += fc * dx; a.fy += fc * dy; a.fz += fc * dz;
    }
}

// Sum of pair forces on atom i over column i of W.
// Two dependent streams feed the loop: the rows of W come from HBM (W is far larger than L2 and read once per
// step), the partner positions from L1/L2.  With the index loads only U rows ahead, every U rows waited one
// full HBM latency (measured: ~7 us per row of W at N = 2M, whatever the gathers touched).  So the W rows are
// loaded a block of D at a time, one block ahead: the next D rows are in flight while the gathers of the current
// block run U at a time.
#ifndef MD_FORCE_D
#define MD_FORCE_D 8
#endif
template <int U, int D, class LD = LdNC>
__device__ __forceinline__ PairAcc column_force(const MdDev &P, const pos_t *__restrict__ pos, const pos_t &ri, int i)
{
    static_assert(D % U == 0, "D must be a multiple of U");
    const int *__restrict__ w = P.W + (size_t)i * P.w_col;
    const size_t pitch = (size_t)P.w_row;
    PairAcc a = {0.0, 0.0, 0.0};
    unsigned cur[D], nxt[D];
    // the first block of rows does not wait for the column length: rows < Mmax exist, entries >= m are never used
#pragma unroll
    for (int d = 0; d < D; d++) cur[d] = d < P.Mmax ? (unsigned)__ldcs(w + d * pitch) : 0u;
    const int m = P.nnb[i];
    for (int base = 0; base < m; base += D) {
#pragma unroll
        for (int d = 0; d < D; d++) nxt[d] = base + D + d < m ? (unsigned)__ldcs(w + (base + D + d) * pitch) : 0u;
#pragma unroll
        for (int g = 0; g < D; g += U) {
            if (base + g < m) {
                pos_t rj[U];
#pragma unroll
                for (int u = 0; u < U; u++)
                    if (base + g + u < m) rj[u] = LD::pos(pos + (cur[g + u] & W_INDEX_MASK));
#pragma unroll
                for (int u = 0; u < U; u++)
                    if (base + g + u < m) pair_force(P, ri, rj[u], cur[g + u] >> W_FLAG_SHIFT, a);
            }
        }
#pragma unroll
        for (int d = 0; d < D; d++) cur[d] = nxt[d];
    }
    a.fx *= 48.0; a.fy *= 48.0; a.fz *= 48.0;
    return a;
}

// MODE 0: store f.  MODE 1: fused leapfrog step: v += dt f, r' = r + dt v into the other position
// buffer, max |v|, rebuild decision.  MODE 2: store f and apply the closing half kick v += dt/2 f.
// BONDS: 0 none, 1 FENE bonds, 2 FENE + angle / dihedral terms
// forces on atom i over column i of W (+ bonds) and the MODE's part of the integration; returns |v|^2 (MODE 1)
// Register budget and W prefetch depth of the fused / force kernels (measured): 1280 resident threads per SM
// with the W rows fetched 4 ahead gains 1.3-2.8 % at N >= 1M over 1024 threads and 8 rows; the kernels with angle /
// dihedral code (BONDS = 2) spill under the tighter cap and keep the round-1 setting.
constexpr int force_min_threads(int bonds) { return bonds == 2 ? MD_FORCE_MIN_THREADS : 1280; }

template <int MODE, int BONDS, class LD, int U = MD_FORCE_U, int D = MD_FORCE_D>
__device__ __forceinline__ double force_atom(const MdDev &P, int pc, int vc, int i)
{
    const pos_t *__restrict__ pos = P.pos[pc];
    double v2 = 0.0;
    const pos_t ri = LD::pos(pos + i);
    const size_t np = (size_t)P.N_pad;
    double *v = P.vel[vc] + i;
    double v0 = 0.0, v1 = 0.0, v2i = 0.0;
    if (MODE != 0) { v0 = v[0]; v1 = v[np]; v2i = v[2 * np]; }     // in flight while the column is walked
    PairAcc a = column_force<U, D, LD>(P, pos, ri, i);
    if (BONDS == 1) bond_force<true, false, LD>(P, pos, ri, i, a);
    if (BONDS == 2) bond_force<true, true, LD>(P, pos, ri, i, a);
    if (MODE == 0 || MODE == 2) {
        double *f = P.frc + i;
        f[0] = a.fx; f[np] = a.fy; f[2 * np] = a.fz;
    }
    if (MODE == 2) {
        v[0] = v0 + P.hdt * a.fx; v[np] = v1 + P.hdt * a.fy; v[2 * np] = v2i + P.hdt * a.fz;
    }
    if (MODE == 1) {
        const double vx = v0 + P.dt * a.fx, vy = v1 + P.dt * a.fy, vz = v2i + P.dt * a.fz;
        v[0] = vx; v[np] = vy; v[2 * np] = vz;
        const double x = ri.x + P.dt * vx, y = ri.y + P.dt * vy, z = ri.z + P.dt * vz;
        st_pos(P.pos[pc ^ 1] + i, x, y, z);
        v2 = vx * vx + vy * vy + vz * vz;
        if (!isfinite(v2 + x + y + z)) { set_err(P, MD_ERR_NONFINITE); v2 = 0.0; }
    }
    return v2;
}

template <int MODE, int BONDS, int BLOCK>
__global__ void __launch_bounds__(BLOCK, force_min_threads(BONDS) / BLOCK) k_force(const __grid_constant__ MdDev P)
{
    __shared__ double sm[32];
    const int i = blockIdx.x * BLOCK + threadIdx.x;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    constexpr int D = BONDS == 2 ? MD_FORCE_D : 4;      // W rows in flight (see force_min_threads)
    const double v2 = i < P.N ? force_atom<MODE, BONDS, LdNC, MD_FORCE_U, D>(P, pc, vc, i) : 0.0;
    if (MODE == 1) {
        const double bm = block_max(v2, sm);
        if (threadIdx.x == 0) publish_vmax2(P, blockIdx.x, bm);
    }
}

// Variant B: each pair once; f_i in registers, f_j by fp64 atomics.  f must be zero on entry.
template <bool BONDS>
__global__ void __launch_bounds__(256) k_force_n3(const __grid_constant__ MdDev P)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const pos_t *__restrict__ pos = P.pos[__ldcg(&P.ctrl->p_dst)];
    const pos_t ri = ld_pos(pos + i);
    const int *__restrict__ w = P.W + (size_t)i * P.w_col;
    const size_t pitch = (size_t)P.w_row;
    double *fx = P.frc, *fy = fx + P.N_pad, *fz = fy + P.N_pad;
    PairAcc a = {0.0, 0.0, 0.0};
    // same W prefetch as variant A (column_force): a block of D rows ahead, the first before the column length
    constexpr int D = MD_FORCE_D, U = MD_FORCE_U;
    unsigned cur[D], nxt[D];
#pragma unroll
    for (int d = 0; d < D; d++) cur[d] = d < P.Mmax ? (unsigned)__ldcs(w + d * pitch) : 0u;
    const int m = P.nnb[i];
    for (int base = 0; base < m; base += D) {
#pragma unroll
        for (int d = 0; d < D; d++) nxt[d] = base + D + d < m ? (unsigned)__ldcs(w + (base + D + d) * pitch) : 0u;
#pragma unroll
        for (int g = 0; g < D; g += U) {
            if (base + g < m) {
                pos_t rj[U];
#pragma unroll
                for (int u = 0; u < U; u++)
                    if (base + g + u < m) rj[u] = ld_pos(pos + (cur[g + u] & W_INDEX_MASK));
#pragma unroll
                for (int u = 0; u < U; u++)
                    if (base + g + u < m) {
                        const unsigned en = cur[g + u];
                        const int j = (int)(en & W_INDEX_MASK);
                        double dx, dy, dz;
                        const double r2 = disp2(ri, rj[u], en >> W_FLAG_SHIFT, P.L, dx, dy, dz);
                        if (r2 < P.rc2) {
                            const double s = fast_rcp(r2), s3 = s * s * s;
                            const double fc = 48.0 * s3 * (s3 - 0.5) * s;
                            const double gx = fc * dx, gy = fc * dy, gz = fc * dz;
                            a.fx += gx; a.fy += gy; a.fz += gz;
                            atomicAdd(fx + j, -gx); atomicAdd(fy + j, -gy); atomicAdd(fz + j, -gz);
                        }
                    }
            }
        }
#pragma unroll
        for (int d = 0; d < D; d++) cur[d] = nxt[d];
    }
    if (BONDS) bond_force<true>(P, pos, ri, i, a);
    atomicAdd(fx + i, a.fx); atomicAdd(fy + i, a.fy); atomicAdd(fz + i, a.fz);
}

__global__ void __launch_bounds__(256) k_zero_forces(const __grid_constant__ MdDev P)
{
    const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (i < 3 * (size_t)P.N_pad) P.frc[i] = 0.0;
}

// ------------------------------------------------------------------------------------------------
// F2 and the other global sums: warp shuffles -> shared memory -> one partial per block
// -> the last block (atomic ticket + memory fence) finishes in a fixed order, so results are reproducible.
// ------------------------------------------------------------------------------------------------
template <bool BONDS>
__global__ void __launch_bounds__(256) k_energy(const __grid_constant__ MdDev P)
{
    __shared__ RedSmem S;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    const pos_t *__restrict__ pos = P.pos[pc];
    double q[RED_N];
#pragma unroll
    for (int k = 0; k < RED_N; k++) q[k] = 0.0;
    if (i < P.N) {
        const pos_t ri = ld_pos(pos + i);
        const int m = P.nnb[i];
        const int *__restrict__ w = P.W + (size_t)i * P.w_col;
        double u = 0.0, vir = 0.0;
#pragma unroll 2
        for (int k = 0; k < m; k++) {
            const unsigned en = (unsigned)__ldcs(w + (size_t)k * P.w_row);
            const pos_t rj = ld_pos(pos + (en & W_INDEX_MASK));
            double dx, dy, dz;
            const double r2 = disp2(ri, rj, en >> W_FLAG_SHIFT, P.L, dx, dy, dz);
            if (r2 < P.rc2) {
                const double s = 1.0 / r2, s3 = s * s * s;
                u += 4.0 * s3 * (s3 - 1.0) - P.uc;
                vir += 48.0 * s3 * (s3 - 0.5);         // fc * r^2
            }
        }
        const double pair_scale = P.half_list ? 1.0 : 0.5;   // full list: u_i counts every pair twice
        q[RED_PE] = pair_scale * u;
        q[RED_VIR] = pair_scale * vir;
        if (BONDS) {
#pragma unroll
            for (int k = 0; k < 2; k++) {
                const int j = P.bond_dev[(size_t)k * P.N_pad + i];
                if (j < 0) continue;
                const pos_t rj = ld_pos(pos + j);
                const double dx = minimg(ri.x - rj.x, P.L, P.half_L), dy = minimg(ri.y - rj.y, P.L, P.half_L),
                             dz = minimg(ri.z - rj.z, P.L, P.half_L);
                const double r2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
                if (!(r2 < P.fene_R02)) { set_err(P, MD_ERR_BOND_BROKEN); continue; }
                const double x = 1.0 - r2 / P.fene_R02;
                q[RED_PEB] += 0.5 * (-0.5 * P.fene_k * P.fene_R02 * log(x));
                q[RED_VIR] += 0.5 * (-P.fene_k / x) * r2;
            }
            if (P.has_dihedrals) {   // the dihedral around the bond (i, partner), counted by the end with the smaller index
#pragma unroll
                for (int k = 0; k < 2; k++) {
                    const int pk = P.bond_dev[(size_t)k * P.N_pad + i], qk = P.bond_dev[(size_t)(1 - k) * P.N_pad + i];
                    if (pk < 0 || qk < 0 || i > pk) continue;
                    const int o = chain_next(P, pk, i);
                    if (o < 0) continue;
                    PairAcc dummy = {0.0, 0.0, 0.0};
                    const double c = dihedral_term(P, ld_pos(pos + qk), ri, ld_pos(pos + pk), ld_pos(pos + o), -1, dummy);
                    q[RED_PEB] += 0.5 * P.dih_k * (c - P.dih_c0) * (c - P.dih_c0);
                }
            }
            if (P.has_angles) {      // the angle i is the vertex of, counted once; cos(theta) is scale invariant: no virial
                const int p0 = P.bond_dev[i], p1 = P.bond_dev[(size_t)P.N_pad + i];
                if (p0 >= 0 && p1 >= 0) {
                    double x1, y1, z1, x2, y2, z2;
                    const double n1 = mi_disp(P, ld_pos(pos + p0), ri, x1, y1, z1), n2 = mi_disp(P, ld_pos(pos + p1), ri, x2, y2, z2);
                    const double c = (x1 * x2 + y1 * y2 + z1 * z2) / sqrt(n1 * n2);
                    q[RED_PEB] += 0.5 * P.ang_k * (c - P.ang_c0) * (c - P.ang_c0);
                }
            }
        }
        const double *v = P.vel[vc] + i;
        const double vx = v[0], vy = v[P.N_pad], vz = v[2 * (size_t)P.N_pad];
        const double v2 = vx * vx + vy * vy + vz * vz;
        q[RED_KE] = 0.5 * v2;
        q[RED_PX] = vx; q[RED_PY] = vy; q[RED_PZ] = vz;
        q[RED_VMAX2] = v2;
    }
    reduce_finish(P, q, S, blockIdx.x, gridDim.x);
}

// ------------------------------------------------------------------------------------------------
// Small systems: ALL n time steps of md_step in ONE cooperative launch.  A system of a few thousand atoms is a few
// dozen thread blocks: its step is not limited by memory or arithmetic but by kernel launches and by the conditional
// node of the step graph (wca_4k: 20 us per step for ~5 us of kernel work).  Here the blocks stay resident and meet at
// grid-wide barriers instead: per step the fused force + kick + drift of every atom, a barrier, the rebuild decision by
// block 0 (decide(), as k_decide takes it), a barrier; and, when the decision says so, the rebuild chain -- the bodies of
// k_bin, k_scan_*, k_place, k_reorder, k_bonds_remap and k_build, a barrier after each.  The arrays those phases rewrite
// are read with ordinary coherent loads (LdPlain), never through the read-only path.  Same arithmetic, same order of
// operations per atom as the graph path with MD_FLAG_GLOBAL_W: results are bitwise equal to it.
// fp64, global-index W (gathering build), variant A, fused steps, at most FENE bonds.
// ------------------------------------------------------------------------------------------------
namespace cg = cooperative_groups;

#ifndef MD_PERSIST_U
#define MD_PERSIST_U 4             // gathers in flight per thread: the phase is one latency chain per atom, not a bandwidth problem
#endif
// MINB: resident blocks per SM the register allocation must allow.  2 (116 registers, 512 threads per SM): every atom its own
// thread, the lowest latency per step -- systems of up to ~75,000 atoms.  4 (64 registers, 1024 threads per SM): larger
// systems, several atoms per thread in grid-stride loops.
template <int BONDS, int MINB>
__global__ void __launch_bounds__(PERSIST_T, MINB) k_persist(const __grid_constant__ MdDev P, long long n_steps)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ double sm[33];
    const int nblk = gridDim.x, tid = threadIdx.x;
    const int stride = nblk * PERSIST_T, first = blockIdx.x * PERSIST_T + tid;
    // Every thread keeps its own copy of the decision scalars and evaluates decide_state() on the same inputs, so no
    // second barrier is needed to publish the decision; block 0 mirrors it into the control block for the host.
    DecState c = dec_load(P);
    for (long long step = 0; step < n_steps; step++) {
        // ---- drifting phase: opening half kick + drift (first step), else forces + full kick + drift ----
        double v2 = 0.0;
        for (int i = first; i < P.N; i += stride)
            v2 = fmax(v2, step == 0 ? kick_drift_atom(P, c.p_dst, c.v_dst, i)
                                    : force_atom<1, BONDS, LdPlain, MD_PERSIST_U, 8>(P, c.p_dst, c.v_dst, i));
        const double bm = block_max(v2, sm);
        double *vmax_buf = P.blk_vmax2 + DEC_SLOTS + (step & 1) * nblk;       // (past k_decide's slots) double-buffered: a fast block may already be in the next step
        if (tid == 0) vmax_buf[blockIdx.x] = bm;
        grid.sync();
        // ---- the rebuild decision, replicated in every block ----
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
            bin_body<LdPlain>(P, B);
            grid.sync();
            for (int t = blockIdx.x; t < P.scan_blocks; t += nblk) { scan_reduce_tile(P, t); __syncthreads(); }
            grid.sync();
            if (blockIdx.x == 0 && tid == 0) {          // exclusive scan of the (few) tile sums
                int run = 0;
                for (int t = 0; t < P.scan_blocks; t++) { const int v = P.block_sums[t]; P.block_sums[t] = run; run += v; }
            }
            grid.sync();
            for (int t = blockIdx.x; t < P.scan_blocks; t += nblk) { scan_apply_tile<false>(P, t); __syncthreads(); }
            grid.sync();
            place_body(P);
            grid.sync();
            reorder_body<LdPlain>(P, B);
            grid.sync();
            if (BONDS) { bonds_remap_body(P, B); grid.sync(); }
            build_body<false, false, LdPlain>(P, B);
            grid.sync();
        }
    }
    // ---- closing: forces at the final positions + half kick ----
    for (int i = first; i < P.N; i += stride) force_atom<2, BONDS, LdPlain, MD_PERSIST_U, 8>(P, c.p_dst, c.v_dst, i);
}

inline int cdiv(long long a, int b) { return (int)((a + b - 1) / b); }

// grid of the rebuild kernels: at most one full wave of the device's SMs; they use grid-stride loops
inline int capped_grid(const MdDev &P, long long n, int block, int per_sm) { return std::min(cdiv(n, block), P.sm_count * per_sm); }

}  // namespace

// ------------------------------------------------------------------------------------------------
// launch wrappers
// ------------------------------------------------------------------------------------------------
void mdk_force_rebuild(const MdDev &P, cudaStream_t st) { k_force_rebuild<<<1, 1, 0, st>>>(P); }

void mdk_check_range(const MdDev &P, double box, cudaStream_t st)
{
    k_check_range<<<capped_grid(P, 3LL * P.N, 256, 8), 256, 0, st>>>(P, box);
}

// The control block into page-locked host memory, written by a kernel: a device-to-host cudaMemcpy would queue on the
// copy engine behind a bulk download in flight on another stream (md_get_state_async) and hold the status read -- and
// with it the next md_step -- for the length of that transfer (measured: 1.8 ms at N = 2M).
namespace {
__global__ void k_publish_ctrl(const DevCtrl *__restrict__ src, DevCtrl *dst)
{
    static_assert(sizeof(DevCtrl) % sizeof(int) == 0, "DevCtrl is copied word by word");
    const int *a = reinterpret_cast<const int *>(src);
    volatile int *b = reinterpret_cast<volatile int *>(dst);
    for (int k = threadIdx.x; k < (int)(sizeof(DevCtrl) / sizeof(int)); k += blockDim.x) b[k] = __ldcg(a + k);
    __threadfence_system();
}
}  // namespace
void mdk_publish_ctrl(const MdDev &P, DevCtrl *host_mapped, cudaStream_t st) { k_publish_ctrl<<<1, 64, 0, st>>>(P.ctrl, host_mapped); }

void mdk_load_state(const MdDev &P, cudaStream_t st)
{
    if (P.sp) return mdk_sp_load_state(P, st);
    k_load_state<<<cdiv(P.N, 256), 256, 0, st>>>(P);
}

void mdk_export(const MdDev &P, int what, double *dst, cudaStream_t st)
{
    if (P.sp) return mdk_sp_export(P, what, dst, st);
    k_export<<<cdiv(P.N, 256), 256, 0, st>>>(P, what, dst);
}

void mdk_decide(const MdDev &P, bool pos_pingpong, cudaStream_t st, unsigned long long cond)
{
    k_decide<<<1, DEC_SLOTS, 0, st>>>(P, pos_pingpong ? 1 : 0, (cudaGraphConditionalHandle)cond);
}

void mdk_kick_drift(const MdDev &P, const MdLaunch &, cudaStream_t st)
{
    if (P.sp) return mdk_sp_kick_drift(P, st);
    k_kick_drift<<<cdiv(P.N, 256), 256, 0, st>>>(P);
}

void mdk_kick(const MdDev &P, const MdLaunch &, cudaStream_t st)
{
    if (P.sp) return mdk_sp_kick(P, st);
    k_kick<<<cdiv(P.N, 256), 256, 0, st>>>(P);
}

void mdk_cells(const MdDev &P, const MdLaunch &, cudaStream_t st)
{
    if (P.sp) mdk_sp_bin(P, st);
    else k_bin<<<capped_grid(P, P.N, 256, 8), 256, 0, st>>>(P);
    k_scan_reduce<<<P.scan_blocks, SCAN_T, 0, st>>>(P);
    k_scan_apply<<<P.scan_blocks, SCAN_T, 0, st>>>(P);
    k_place<<<capped_grid(P, P.N, 256, 8), 256, 0, st>>>(P);
}

void mdk_reorder(const MdDev &P, const MdLaunch &, cudaStream_t st)
{
    if (P.sp) mdk_sp_reorder(P, st);
    else k_reorder<<<capped_grid(P, P.N, 256, 8), 256, 0, st>>>(P);
    if (P.layer_H) k_copy_wrap<<<capped_grid(P, P.N, 256, 8), 256, 0, st>>>(P);
    if (P.has_bonds) k_bonds_remap<<<capped_grid(P, P.N, 256, 8), 256, 0, st>>>(P);
    if (P.rigid) mdk_rigid_offsets(P, st);
}

void mdk_build(const MdDev &P, const MdLaunch &, cudaStream_t st)
{
    if (P.sp) return mdk_sp_build(P, st);
    if (P.layer_H) {
        k_layer_fill<<<capped_grid(P, P.N, 256, 8), 256, 0, st>>>(P);
        k_build_layers<<<capped_grid(P, P.N, 128, 16), 128, 0, st>>>(P);
        return;
    }
    if (P.rigid) k_build<false, true><<<capped_grid(P, P.N, 128, 16), 128, 0, st>>>(P);
    else if (P.half_list) k_build<true, false><<<capped_grid(P, P.N, 128, 16), 128, 0, st>>>(P);
    else k_build<false, false><<<capped_grid(P, P.N, 128, 16), 128, 0, st>>>(P);
}

template <int MODE, int BONDS>
static void launch_force_block(const MdDev &P, int block, cudaStream_t st)
{
    switch (block) {
    case 64: k_force<MODE, BONDS, 64><<<cdiv(P.N, 64), 64, 0, st>>>(P); break;
    case 128: k_force<MODE, BONDS, 128><<<cdiv(P.N, 128), 128, 0, st>>>(P); break;
    case 512: k_force<MODE, BONDS, 512><<<cdiv(P.N, 512), 512, 0, st>>>(P); break;
    default: k_force<MODE, BONDS, 256><<<cdiv(P.N, 256), 256, 0, st>>>(P); break;
    }
}

void mdk_force(const MdDev &P, const MdLaunch &lc, int mode, cudaStream_t st)
{
    if (P.sp) return mdk_sp_force(P, lc, mode, st);
    if (P.has_bonds && (P.has_angles || P.has_dihedrals)) {
        if (mode == 0) launch_force_block<0, 2>(P, lc.block, st);
        else if (mode == 1) launch_force_block<1, 2>(P, lc.block, st);
        else launch_force_block<2, 2>(P, lc.block, st);
    } else if (P.has_bonds) {
        if (mode == 0) launch_force_block<0, 1>(P, lc.block, st);
        else if (mode == 1) launch_force_block<1, 1>(P, lc.block, st);
        else launch_force_block<2, 1>(P, lc.block, st);
    } else {
        if (mode == 0) launch_force_block<0, 0>(P, lc.block, st);
        else if (mode == 1) launch_force_block<1, 0>(P, lc.block, st);
        else launch_force_block<2, 0>(P, lc.block, st);
    }
}

void mdk_force_newton3(const MdDev &P, const MdLaunch &, cudaStream_t st)
{
    k_zero_forces<<<cdiv(3LL * P.N_pad, 256), 256, 0, st>>>(P);
    if (P.has_bonds) k_force_n3<true><<<cdiv(P.N, 256), 256, 0, st>>>(P);
    else k_force_n3<false><<<cdiv(P.N, 256), 256, 0, st>>>(P);
}

void mdk_energy(const MdDev &P, const MdLaunch &, cudaStream_t st)
{
    if (P.sp) return mdk_sp_energy(P, st);
    const int grid = cdiv(P.N, 256);
    if (P.has_bonds) k_energy<true><<<grid, 256, 0, st>>>(P);
    else k_energy<false><<<grid, 256, 0, st>>>(P);
}

// ---- the persistent small-system kernel ----
#ifndef MD_PERSIST_MAX_N
#define MD_PERSIST_MAX_N 400000     // beyond ~450,000 atoms the graph path (tile-staged build, 1280 threads per SM in the force kernel) is faster
#endif
namespace {
struct PersistChoice {
    const void *kernel;
    int grid;
};
template <int MINB>
const void *persist_kernel(const MdDev &P) { return P.has_bonds ? (const void *)k_persist<1, MINB> : (const void *)k_persist<0, MINB>; }

// every atom its own thread if the low-latency instantiation holds them all at once, else the high-occupancy one with
// as many blocks as are resident together (a cooperative launch needs that) and grid-stride loops
PersistChoice persist_choice(const MdDev &P)
{
    if (P.sp) {
        const void *k = nullptr;
        const int grid = mdk_sp_persist_choice(P, &k);
        return {k, grid};
    }
    const int want = cdiv(P.N, PERSIST_T);
    int per_sm = 0;
    const void *k = persist_kernel<2>(P);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, PERSIST_T, 0) == cudaSuccess && per_sm >= 1 && want <= per_sm * P.sm_count)
        return {k, want};
    k = persist_kernel<4>(P);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, PERSIST_T, 0) == cudaSuccess && per_sm >= 1)
        return {k, std::min(want, per_sm * P.sm_count)};
    cudaGetLastError();
    return {nullptr, 0};
}
}  // namespace

bool mdk_persist_ok(const MdDev &P)
{
    if (P.tiled || P.half_list || P.layer_H || P.rigid || P.has_angles || P.has_dihedrals || P.w_col != 1) return false;
    if (P.sp && P.sp_pad > 1) return false;               // padded columns (long binary32 columns): step graph
    if (P.N > MD_PERSIST_MAX_N) return false;
    int dev = 0, coop = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop) { cudaGetLastError(); return false; }
    return persist_choice(P).grid > 0;
}

int mdk_persist_steps(const MdDev &P, long long n, cudaStream_t st)
{
    const PersistChoice c = persist_choice(P);
    if (c.grid <= 0) return -1;
    MdDev Pc = P;
    void *args[] = {(void *)&Pc, (void *)&n};
    return cudaLaunchCooperativeKernel(c.kernel, dim3(c.grid), dim3(PERSIST_T), args, 0, st) == cudaSuccess ? 0 : -1;
}

int mdk_launches_of(int which)
{
    switch (which) {
    case LK_CELLS: return 4;
    case LK_FORCE_N3: return 2;
    default: return 1;
    }
}
