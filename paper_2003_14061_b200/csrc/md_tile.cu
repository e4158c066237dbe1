// Tiled-W kernels (sm_100a): neighbor-matrix build (N5), pair forces (F1) and the
// energy sums (F2) with the partner positions staged in SHARED MEMORY instead of gathered
// through L1/L2.
//
// Why.  With W holding global atom indices the force kernel issues one 32-lane gather per row of W, and on
// sm_100a such a gather occupies the L1 wavefront queue for ~2 cycles per distinct 128-byte line it touches
// (~20 lines per gather here): profiles/r01a_ncu_full_wca2m.txt shows the kernel pinned on that queue at 21 %
// of DRAM bandwidth.  The paper meets the same wall ("r_i' ... are not stored consecutively")
// and answers it with cell-order sorting; its cell-block comparison (sec. 4.2(1)) stages cell
// contents in shared memory but abandons the neighbor matrix.  Here both are kept: atoms are in cell order
// (x fastest), a thread block owns the atoms of a box of S x R x RZ cells -- R*RZ contiguous index ranges --
// and the 27-cell neighbourhoods of all of them are (R+2)(RZ+2) contiguous runs of the position array, copied
// once per block, coalesced, into a shared-memory tile.  W keeps the paper's layout (row m contiguous over
// atoms i) but its entries are 16 bits: 13 bits of index into the block's tile + the 3
// periodic-image flag bits of PAPER.md:163, packed two rows per 32-bit word.  The random accesses then hit
// the shared-memory crossbar (128 B/cycle/SM, no tag look-ups) and W costs 2 bytes per neighbor.
//
// The tile layout is a pure function of (block index, cell_start); cell_start only changes at a rebuild,
// so the build kernel and every later force / energy kernel reconstruct the same layout.
#include <algorithm>

#include "md_device.cuh"

namespace {

struct TileMeta {
    int n_own, T;                                       // atoms owned by the block, atoms in the tile
    int own_base[TILE_OWN_MAX];                         // global index of the first own atom of own row k
    int own_loc[TILE_OWN_MAX];                          // its index in the tile
    int own_pre[TILE_OWN_MAX + 1];                      // exclusive prefix of the own-row lengths
    int row_off[TILE_Q_MAX + 1];                        // tile index of the first atom of tile row q
    int pg[TILE_Q_MAX][3], pn[TILE_Q_MAX][3];           // the (up to) 3 contiguous pieces of a tile row: start, length
    int row_cell[TILE_Q_MAX];                           // linear index of the x = 0 cell of the (wrapped) row
    int ysh[TILE_Q_MAX], zsh[TILE_Q_MAX];               // image shift of the row in units of L
};

// Build the tile of block blockIdx.x: fills M, copies positions into sx/sy/sz and (CELLS) the tile index of
// the first atom of every tile cell into tcs[q * (S + 3) + k], k = 0 .. sxc + 2.  Returns false, with nothing
// copied, when the tile would exceed the capacity.  All threads of the block must call it.
template <bool CELLS>
__device__ __forceinline__ bool tile_setup(const MdDev &P, const TileBox &B, const pos_t *__restrict__ pos, TileMeta &M,
                                           double *sx, double *sy, double *sz, int *tcs)
{
    const int nc = P.nc;
    const int *__restrict__ cs = P.cell_start;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
    if (tid < B.nq) {
        const int q = tid;
        int rowc, ysh, zsh, xa, xc;
        tile_row(B, nc, q, rowc, ysh, zsh, xa, xc);
        const int gA = __ldg(cs + rowc + xa), nA = __ldg(cs + rowc + xa + 1) - gA;
        const int gB = __ldg(cs + rowc + B.x0), nB = __ldg(cs + rowc + B.x0 + B.sxc) - gB;
        const int gC = __ldg(cs + rowc + xc), nC = __ldg(cs + rowc + xc + 1) - gC;
        M.pg[q][0] = gA; M.pg[q][1] = gB; M.pg[q][2] = gC;
        M.pn[q][0] = nA; M.pn[q][1] = nB; M.pn[q][2] = nC;
        M.row_cell[q] = rowc; M.ysh[q] = ysh; M.zsh[q] = zsh;
    }
    __syncthreads();
    if (tid == 0) {
        int off = 0, own = 0, k = 0;
        for (int q = 0; q < B.nq; q++) {
            M.row_off[q] = off;
            const int qy = q % B.nyq, qz = q / B.nyq;
            if (qy >= 1 && qy <= B.ny && qz >= 1 && qz <= B.nz) {      // a row of the box itself
                M.own_base[k] = M.pg[q][1];
                M.own_loc[k] = off + M.pn[q][0];
                M.own_pre[k] = own;
                own += M.pn[q][1];
                k++;
            }
            off += M.pn[q][0] + M.pn[q][1] + M.pn[q][2];
        }
        M.row_off[B.nq] = off;
        for (; k <= TILE_OWN_MAX; k++) M.own_pre[k] = own;
        M.n_own = own;
        M.T = off;
    }
    __syncthreads();
    if (M.T > P.tg.cap) return false;
    for (int q = wid; q < B.nq; q += nw) {
        const int off = M.row_off[q], nA = M.pn[q][0], nB = M.pn[q][1], nC = M.pn[q][2];
        const int gA = M.pg[q][0], gB = M.pg[q][1], gC = M.pg[q][2];
        const int tot = nA + nB + nC;
        for (int u = lane; u < tot; u += 32) {
            const int src = u < nA ? gA + u : (u < nA + nB ? gB + (u - nA) : gC + (u - nA - nB));
            const pos_t p = ld_pos(pos + src);
            sx[off + u] = p.x; sy[off + u] = p.y; sz[off + u] = p.z;
        }
        if (CELLS) {
            const int rowc = M.row_cell[q];
            for (int k = lane; k <= B.sxc + 2; k += 32) {
                int v;
                if (k == 0) v = off;
                else if (k == B.sxc + 2) v = off + tot;
                else v = off + nA + (__ldg(cs + rowc + B.x0 + k - 1) - gB);
                tcs[q * (P.tg.S + 3) + k] = v;
            }
        }
    }
    __syncthreads();
    return true;
}

// own atom number t of the block -> global index i and tile index li
__device__ __forceinline__ void own_atom(const TileMeta &M, int t, int &i, int &li)
{
    int k = 0;
#pragma unroll
    for (int r = 1; r < TILE_OWN_MAX; r++) k = t >= M.own_pre[r] ? r : k;
    // rows past the last one repeat own_pre = n_own > t, so k stops at the right row
    const int o = t - M.own_pre[k];
    i = M.own_base[k] + o;
    li = M.own_loc[k] + o;
}

// ------------------------------------------------------------------------------------------------
// N5 on the tile.  One thread per atom; the candidates of atom i in cell (cx, cy, cz) are, for
// each of the 9 (dy, dz), the 3 consecutive tile cells cx-1 .. cx+1 of tile row (cy+dy, cz+dz): one contiguous
// range of the shared arrays.  Lanes in the same cell read the same shared-memory words (broadcast).
// Accept test and image arithmetic are those of DESIGN.md R5, bit for bit: d = (r_i - r_j) rounded, + shift
// rounded, r^2 = fma(dz,dz, fma(dy,dy, dx*dx)) < r_n^2.
// ------------------------------------------------------------------------------------------------
struct Emit {
    unsigned *w;        // column i of W (32-bit words of two entries)
    size_t pitch;
    int m, Mmax;
    unsigned pend;
    __device__ __forceinline__ void put(unsigned e)
    {
        if (m & 1) { if (m < Mmax) w[(size_t)(m >> 1) * pitch] = pend | (e << 16); }
        else pend = e;
        m++;
    }
    __device__ __forceinline__ void flush()
    {
        if ((m & 1) && m < Mmax) w[(size_t)(m >> 1) * pitch] = pend;
    }
};

template <bool SHIFT>
__device__ __forceinline__ void tile_scan_run(const double *sx, const double *sy, const double *sz, double xi, double yi, double zi,
                                              int li, int b, int e, double shx, double shy, double shz, unsigned fl, double rn2, Emit &em)
{
    for (int j = b; j < e; j++) {
        double dx = __dsub_rn(xi, sx[j]), dy = __dsub_rn(yi, sy[j]), dz = __dsub_rn(zi, sz[j]);
        if (SHIFT) { dx = __dadd_rn(dx, shx); dy = __dadd_rn(dy, shy); dz = __dadd_rn(dz, shz); }
        const double r2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
        if (r2 < rn2 && j != li) em.put((unsigned)j | (fl << T_FLAG_SHIFT));
    }
}

template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) k_tile_build(const __grid_constant__ MdDev P)
{
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    extern __shared__ double dsm[];
    __shared__ TileMeta M;
    __shared__ int smx[32], ssum[32];
    const int cap = P.tg.cap;
    double *sx = dsm, *sy = sx + cap, *sz = sy + cap;
    int *tcs = (int *)(sz + cap);
    const int stride = P.tg.S + 3;
    const pos_t *__restrict__ pos = P.pos[__ldcg(&P.ctrl->p_dst)];
    const TileBox B = tile_box(P.tg, P.nc, blockIdx.x);
    const bool ok = tile_setup<true>(P, B, pos, M, sx, sy, sz, tcs);
    if (!ok) {
        if (threadIdx.x == 0) set_err(P, MD_ERR_TILE_OVERFLOW);
        return;
    }
    const int nc = P.nc;
    const double L = P.L, rn2 = P.rn2;
    int tmax = 0, tsum = 0;
    for (int t = threadIdx.x; t < M.n_own; t += BLOCK) {
        int i, li;
        own_atom(M, t, i, li);
        const double xi = sx[li], yi = sy[li], zi = sz[li];
        const int cx = cell_coord(xi, P.inv_w, nc), cy = cell_coord(yi, P.inv_w, nc), cz = cell_coord(zi, P.inv_w, nc);
        Emit em = {(unsigned *)P.W + i, (size_t)P.N_pad, 0, P.Mmax, 0u};
        const int k0 = cx - B.x0;
        for (int dz = -1; dz <= 1; dz++) {
            for (int dy = -1; dy <= 1; dy++) {
                const int q = (cy + dy - (B.y0 - 1)) + B.nyq * (cz + dz - (B.z0 - 1));
                const int ysh = M.ysh[q], zsh = M.zsh[q];
                const unsigned fl = (ysh ? 2u : 0u) | (zsh ? 4u : 0u);
                const double shy = ysh * L, shz = zsh * L;
                const int *tc = tcs + q * stride + k0;
                const int b = tc[0], e = tc[3];
                if (cx == 0) {
                    const int mid = tc[1];
                    tile_scan_run<true>(sx, sy, sz, xi, yi, zi, li, b, mid, L, shy, shz, fl | 1u, rn2, em);
                    if (fl) tile_scan_run<true>(sx, sy, sz, xi, yi, zi, li, mid, e, 0.0, shy, shz, fl, rn2, em);
                    else tile_scan_run<false>(sx, sy, sz, xi, yi, zi, li, mid, e, 0.0, 0.0, 0.0, 0u, rn2, em);
                } else if (cx == nc - 1) {
                    const int mid = tc[2];
                    if (fl) tile_scan_run<true>(sx, sy, sz, xi, yi, zi, li, b, mid, 0.0, shy, shz, fl, rn2, em);
                    else tile_scan_run<false>(sx, sy, sz, xi, yi, zi, li, b, mid, 0.0, 0.0, 0.0, 0u, rn2, em);
                    tile_scan_run<true>(sx, sy, sz, xi, yi, zi, li, mid, e, -L, shy, shz, fl | 1u, rn2, em);
                } else if (fl) {
                    tile_scan_run<true>(sx, sy, sz, xi, yi, zi, li, b, e, 0.0, shy, shz, fl, rn2, em);
                } else {
                    tile_scan_run<false>(sx, sy, sz, xi, yi, zi, li, b, e, 0.0, 0.0, 0.0, 0u, rn2, em);
                }
            }
        }
        em.flush();
        const int m = em.m;
        P.nnb[i] = m < P.Mmax ? m : P.Mmax;
        if (m > P.Mmax) set_err(P, MD_ERR_NEBR_OVERFLOW);
        tmax = max(tmax, m);
        tsum += m;
    }
    // statistics of the matrix (md_energy.max_neighbors / mean_neighbors)
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int wm = warp_max_i(tmax), ws = warp_sum_i(tsum);
    if (lane == 0) { smx[wid] = wm; ssum[wid] = ws; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int mx = 0, sm = 0;
        for (int w = 0; w < BLOCK / 32; w++) { mx = max(mx, smx[w]); sm += ssum[w]; }
        atomicMax(&P.ctrl->max_nnb, mx);
        atomicAdd(&P.ctrl->nnb_total, (unsigned long long)sm);
    }
}

// ------------------------------------------------------------------------------------------------
// F1 on the tile.  Thread i walks column i of W (coalesced 32-bit words, two neighbors each, streamed from HBM
// two words ahead of their use); the partner positions come from the shared-memory tile.
// ------------------------------------------------------------------------------------------------
struct PairAccT {
    double fx, fy, fz, u, vir;
};

template <bool ENERGY>
__device__ __forceinline__ void tile_pair(const MdDev &P, const double *sx, const double *sy, const double *sz, double xi, double yi,
                                          double zi, unsigned e, PairAccT &a)
{
    const unsigned l = e & T_INDEX_MASK, fl = e >> T_FLAG_SHIFT;
    double dx = xi - sx[l], dy = yi - sy[l], dz = zi - sz[l];
    if (fl) {                                   // only atoms next to a periodic face take this branch
        if (fl & 1u) dx -= copysign(P.L, dx);
        if (fl & 2u) dy -= copysign(P.L, dy);
        if (fl & 4u) dz -= copysign(P.L, dz);
    }
    const double r2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
    if (r2 < P.rc2) {
        if (ENERGY) {
            const double s = 1.0 / r2, s3 = s * s * s;
            a.u += 4.0 * s3 * (s3 - 1.0) - P.uc;
            a.vir += 48.0 * s3 * (s3 - 0.5);          // fc * r^2
        } else {
            const double s = fast_rcp(r2), s3 = s * s * s;
            const double fc = s3 * (s3 - 0.5) * s;    // x 48 applied once to the sums
            a.fx += fc * dx; a.fy += fc * dy; a.fz += fc * dz;
        }
    }
}

template <bool ENERGY>
__device__ __forceinline__ PairAccT tile_column(const MdDev &P, const double *sx, const double *sy, const double *sz, double xi,
                                                double yi, double zi, int i)
{
    const int m = P.nnb[i];
    const unsigned *__restrict__ w = (const unsigned *)P.W + i;
    const size_t pitch = (size_t)P.N_pad;
    const int nw = (m + 1) >> 1;
    PairAccT a = {0.0, 0.0, 0.0, 0.0, 0.0};
    unsigned cur = nw > 0 ? __ldcs(w) : 0u, nxt = nw > 1 ? __ldcs(w + pitch) : 0u;
    for (int k = 0; k < nw; k++) {
        const unsigned nn = k + 2 < nw ? __ldcs(w + (size_t)(k + 2) * pitch) : 0u;
        tile_pair<ENERGY>(P, sx, sy, sz, xi, yi, zi, cur & 0xffffu, a);
        if (2 * k + 1 < m) tile_pair<ENERGY>(P, sx, sy, sz, xi, yi, zi, cur >> 16, a);
        cur = nxt; nxt = nn;
    }
    if (!ENERGY) { a.fx *= 48.0; a.fy *= 48.0; a.fz *= 48.0; }
    return a;
}

// FENE bonds: partners by global index, read from the position array (2 per atom at most)
template <bool ENERGY>
__device__ __forceinline__ void tile_bonds(const MdDev &P, const pos_t *__restrict__ pos, double xi, double yi, double zi, int i,
                                           PairAccT &a, double &ub)
{
#pragma unroll
    for (int k = 0; k < 2; k++) {
        const int j = P.bond_dev[(size_t)k * P.N_pad + i];
        if (j < 0) continue;
        const pos_t rj = ld_pos(pos + j);
        const double dx = minimg(xi - rj.x, P.L, P.half_L), dy = minimg(yi - rj.y, P.L, P.half_L), dz = minimg(zi - rj.z, P.L, P.half_L);
        const double r2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
        if (!(r2 < P.fene_R02)) { set_err(P, MD_ERR_BOND_BROKEN); continue; }
        if (ENERGY) {
            const double x = 1.0 - r2 / P.fene_R02;
            ub += 0.5 * (-0.5 * P.fene_k * P.fene_R02 * log(x));
            a.vir += 0.5 * (-P.fene_k / x) * r2;
        } else {
            const double fc = -P.fene_k / (1.0 - r2 / P.fene_R02);
            a.fx += fc * dx; a.fy += fc * dy; a.fz += fc * dz;
        }
    }
}

// MODE 0: store f.  MODE 1: fused leapfrog step: v += dt f, r' = r + dt v into the other position buffer,
// max |v|, rebuild decision.  MODE 2: store f and apply the closing half kick v += dt/2 f.
template <int MODE, bool BONDS, int BLOCK>
__global__ void __launch_bounds__(BLOCK, 1024 / BLOCK) k_tile_force(const __grid_constant__ MdDev P)
{
    extern __shared__ double dsm[];
    __shared__ TileMeta M;
    __shared__ double red[32];
    const int cap = P.tg.cap;
    double *sx = dsm, *sy = sx + cap, *sz = sy + cap;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    const pos_t *__restrict__ pos = P.pos[pc];
    const TileBox B = tile_box(P.tg, P.nc, blockIdx.x);
    const bool ok = tile_setup<false>(P, B, pos, M, sx, sy, sz, nullptr);
    double v2 = 0.0;
    if (ok) {
        for (int t = threadIdx.x; t < M.n_own; t += BLOCK) {
            int i, li;
            own_atom(M, t, i, li);
            const double xi = sx[li], yi = sy[li], zi = sz[li];
            PairAccT a = tile_column<false>(P, sx, sy, sz, xi, yi, zi, i);
            double ub = 0.0;
            if (BONDS) tile_bonds<false>(P, pos, xi, yi, zi, i, a, ub);
            if (MODE == 0 || MODE == 2) {
                double *f = P.frc + i;
                f[0] = a.fx; f[P.N_pad] = a.fy; f[2 * (size_t)P.N_pad] = a.fz;
            }
            if (MODE == 2) {
                double *v = P.vel[vc] + i;
                v[0] += P.hdt * a.fx; v[P.N_pad] += P.hdt * a.fy; v[2 * (size_t)P.N_pad] += P.hdt * a.fz;
            }
            if (MODE == 1) {
                double *v = P.vel[vc] + i;
                const double vx = v[0] + P.dt * a.fx, vy = v[P.N_pad] + P.dt * a.fy, vz = v[2 * (size_t)P.N_pad] + P.dt * a.fz;
                v[0] = vx; v[P.N_pad] = vy; v[2 * (size_t)P.N_pad] = vz;
                const double x = xi + P.dt * vx, y = yi + P.dt * vy, z = zi + P.dt * vz;
                st_pos(P.pos[pc ^ 1] + i, x, y, z);
                double w2 = vx * vx + vy * vy + vz * vz;
                if (!isfinite(w2 + x + y + z)) { set_err(P, MD_ERR_NONFINITE); w2 = 0.0; }
                v2 = fmax(v2, w2);
            }
        }
    }
    if (MODE == 1) {
        const double bm = block_max(v2, red);
        if (threadIdx.x == 0) publish_vmax_and_decide(P, bm, true);
    }
}

template <bool BONDS, int BLOCK>
__global__ void __launch_bounds__(BLOCK) k_tile_energy(const __grid_constant__ MdDev P)
{
    extern __shared__ double dsm[];
    __shared__ TileMeta M;
    __shared__ RedSmem S;
    const int cap = P.tg.cap;
    double *sx = dsm, *sy = sx + cap, *sz = sy + cap;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    const pos_t *__restrict__ pos = P.pos[pc];
    const TileBox B = tile_box(P.tg, P.nc, blockIdx.x);
    const bool ok = tile_setup<false>(P, B, pos, M, sx, sy, sz, nullptr);
    double q[RED_N];
#pragma unroll
    for (int k = 0; k < RED_N; k++) q[k] = 0.0;
    if (ok) {
        for (int t = threadIdx.x; t < M.n_own; t += BLOCK) {
            int i, li;
            own_atom(M, t, i, li);
            const double xi = sx[li], yi = sy[li], zi = sz[li];
            PairAccT a = tile_column<true>(P, sx, sy, sz, xi, yi, zi, i);
            a.u *= 0.5; a.vir *= 0.5;               // full list: u_i counts every pair twice
            double ub = 0.0;
            if (BONDS) tile_bonds<true>(P, pos, xi, yi, zi, i, a, ub);
            const double *v = P.vel[vc] + i;
            const double vx = v[0], vy = v[P.N_pad], vz = v[2 * (size_t)P.N_pad];
            const double w2 = vx * vx + vy * vy + vz * vz;
            q[RED_PE] += a.u; q[RED_PEB] += ub; q[RED_VIR] += a.vir;
            q[RED_KE] += 0.5 * w2;
            q[RED_PX] += vx; q[RED_PY] += vy; q[RED_PZ] += vz;
            q[RED_VMAX2] = fmax(q[RED_VMAX2], w2);
        }
    }
    reduce_finish(P, q, S);
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// launch wrappers
// ------------------------------------------------------------------------------------------------
size_t mdk_tile_smem(const TileGeom &G, bool with_cells)
{
    size_t b = 3 * (size_t)G.cap * sizeof(double);
    if (with_cells) b += (size_t)TILE_Q_MAX * (G.S + 3) * sizeof(int);
    return b;
}

namespace {

inline int tile_grid(const MdDev &P) { return P.tg.nsx * P.tg.nsy * P.tg.nsz; }

template <typename K>
int opt_in(K kernel, size_t bytes)
{
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) == cudaSuccess ? 0 : -1;
}

template <int BLOCK>
int configure_block(const MdDev &P)
{
    const size_t sf = mdk_tile_smem(P.tg, false), sb = mdk_tile_smem(P.tg, true);
    int rc = 0;
    rc |= opt_in(k_tile_build<BLOCK>, sb);
    rc |= opt_in(k_tile_force<0, false, BLOCK>, sf);
    rc |= opt_in(k_tile_force<1, false, BLOCK>, sf);
    rc |= opt_in(k_tile_force<2, false, BLOCK>, sf);
    rc |= opt_in(k_tile_force<0, true, BLOCK>, sf);
    rc |= opt_in(k_tile_force<1, true, BLOCK>, sf);
    rc |= opt_in(k_tile_force<2, true, BLOCK>, sf);
    rc |= opt_in(k_tile_energy<false, BLOCK>, sf);
    rc |= opt_in(k_tile_energy<true, BLOCK>, sf);
    return rc;
}

template <int BLOCK>
void launch_force(const MdDev &P, int mode, cudaStream_t st)
{
    const int g = tile_grid(P);
    const size_t sm = mdk_tile_smem(P.tg, false);
    if (P.has_bonds) {
        if (mode == 0) k_tile_force<0, true, BLOCK><<<g, BLOCK, sm, st>>>(P);
        else if (mode == 1) k_tile_force<1, true, BLOCK><<<g, BLOCK, sm, st>>>(P);
        else k_tile_force<2, true, BLOCK><<<g, BLOCK, sm, st>>>(P);
    } else {
        if (mode == 0) k_tile_force<0, false, BLOCK><<<g, BLOCK, sm, st>>>(P);
        else if (mode == 1) k_tile_force<1, false, BLOCK><<<g, BLOCK, sm, st>>>(P);
        else k_tile_force<2, false, BLOCK><<<g, BLOCK, sm, st>>>(P);
    }
}

}  // namespace

int mdk_tile_configure(const MdDev &P)
{
    switch (P.tg.threads) {
    case 128: return configure_block<128>(P);
    case 256: return configure_block<256>(P);
    case 512: return configure_block<512>(P);
    default: return -1;
    }
}

void mdk_tile_build(const MdDev &P, cudaStream_t st)
{
    const int g = tile_grid(P);
    const size_t sm = mdk_tile_smem(P.tg, true);
    switch (P.tg.threads) {
    case 128: k_tile_build<128><<<g, 128, sm, st>>>(P); break;
    case 512: k_tile_build<512><<<g, 512, sm, st>>>(P); break;
    default: k_tile_build<256><<<g, 256, sm, st>>>(P); break;
    }
}

void mdk_tile_force(const MdDev &P, int mode, cudaStream_t st)
{
    switch (P.tg.threads) {
    case 128: launch_force<128>(P, mode, st); break;
    case 512: launch_force<512>(P, mode, st); break;
    default: launch_force<256>(P, mode, st); break;
    }
}

void mdk_tile_energy(const MdDev &P, cudaStream_t st)
{
    const int g = tile_grid(P);
    const size_t sm = mdk_tile_smem(P.tg, false);
#define MD_TE(B)                                                            \
    if (P.has_bonds) k_tile_energy<true, B><<<g, B, sm, st>>>(P);          \
    else k_tile_energy<false, B><<<g, B, sm, st>>>(P)
    switch (P.tg.threads) {
    case 128: MD_TE(128); break;
    case 512: MD_TE(512); break;
    default: MD_TE(256); break;
    }
#undef MD_TE
}
