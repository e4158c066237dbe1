// Bodies of the rebuild chain that do not touch coordinates (N3/N4: scan of the cell occupancies, place, bond-partner remap)
// and are shared by the binary64 and binary32 kernels: each is the body of a kernel of md_kernels.cu AND a phase of the
// persistent kernels (md_kernels.cu: k_persist, md_sp.cu: k_sp_persist), which run them between grid-wide barriers.
#pragma once
#include "md_device.cuh"

namespace {

// which of the ping-pong buffers a rebuild reads (ps, vs) and writes (pd, vd): from the control block, or from the
// persistent kernel's own copy of the decision
struct Bufs {
    int ps, pd, vs, vd;
};
__device__ __forceinline__ Bufs bufs_from_ctrl(const MdDev &P)
{
    return {__ldcg(&P.ctrl->p_src), __ldcg(&P.ctrl->p_dst), __ldcg(&P.ctrl->v_src), __ldcg(&P.ctrl->v_dst)};
}

constexpr int SCAN_T = 256, SCAN_V = 8, SCAN_TILE = SCAN_T * SCAN_V;

// the SCAN_V = 8 occupancies of a thread: two 128-bit loads where all 8 cells exist (the arrays are 256-byte aligned, base is
// a multiple of 8), else one by one with zeros past the last cell.  Plain loads: the persistent kernels rewrite cell_count.
__device__ __forceinline__ void scan_load8(const MdDev &P, int base, int (&c)[SCAN_V])
{
    static_assert(SCAN_V == 8, "two int4 per thread");
    if (base + SCAN_V <= P.NC) {
        const int4 a = *reinterpret_cast<const int4 *>(P.cell_count + base), b = *reinterpret_cast<const int4 *>(P.cell_count + base + 4);
        c[0] = a.x; c[1] = a.y; c[2] = a.z; c[3] = a.w; c[4] = b.x; c[5] = b.y; c[6] = b.z; c[7] = b.w;
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_V; k++) c[k] = base + k < P.NC ? P.cell_count[base + k] : 0;
    }
}

// occupancy sum and maximum of tile `tile` of SCAN_TILE cells; the block has SCAN_T threads
__device__ __forceinline__ void scan_reduce_tile(const MdDev &P, int tile)
{
    __shared__ int ssum[SCAN_T / 32], smax[SCAN_T / 32];
    const int base = tile * SCAN_TILE + threadIdx.x * SCAN_V;
    int c[SCAN_V], sum = 0, mx = 0;
    scan_load8(P, base, c);
#pragma unroll
    for (int k = 0; k < SCAN_V; k++) {
        sum += c[k];
        mx = max(mx, c[k]);
    }
    sum = warp_sum_i(sum);
    mx = warp_max_i(mx);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { ssum[wid] = sum; smax[wid] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int s = 0, m = 0;
        for (int w = 0; w < SCAN_T / 32; w++) { s += ssum[w]; m = max(m, smax[w]); }
        P.block_sums[tile] = s;
        atomicMax(&P.ctrl->max_occ, m);              // N3: the paper's layer count N_l = max_c k_c
    }
}

// RAW: block_sums holds the tiles' own sums and the block adds up the tiles before its own (the kernel chain: one launch less
// than with a separate scan of the tile sums); else block_sums holds the exclusive prefix already (persistent kernels).
template <bool RAW>
__device__ __forceinline__ void scan_apply_tile(const MdDev &P, int tile)
{
    __shared__ int wsum[SCAN_T / 32], psum[SCAN_T / 32];
    int before = 0;
    if (RAW) {
        for (int t = threadIdx.x; t < tile; t += SCAN_T) before += P.block_sums[t];
        before = warp_sum_i(before);
        if ((threadIdx.x & 31) == 0) psum[threadIdx.x >> 5] = before;
    }
    const int base = tile * SCAN_TILE + threadIdx.x * SCAN_V;
    int c[SCAN_V], sum = 0;
    scan_load8(P, base, c);
#pragma unroll
    for (int k = 0; k < SCAN_V; k++) sum += c[k];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(FULL_MASK, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    int woff = 0;
    for (int w = 0; w < wid; w++) woff += wsum[w];
    if (RAW) {
        before = 0;
        for (int w = 0; w < SCAN_T / 32; w++) before += psum[w];
    } else {
        before = P.block_sums[tile];
    }
    int run = before + woff + inc - sum;
    if (base + SCAN_V < P.NC) {      // all 8 cells exist and none is the last: 128-bit stores
        int st[SCAN_V];
#pragma unroll
        for (int k = 0; k < SCAN_V; k++) { st[k] = run; run += c[k]; }
        int4 *cs = reinterpret_cast<int4 *>(P.cell_start + base), *cc = reinterpret_cast<int4 *>(P.cell_count + base);
        cs[0] = make_int4(st[0], st[1], st[2], st[3]);
        cs[1] = make_int4(st[4], st[5], st[6], st[7]);
        cc[0] = make_int4(0, 0, 0, 0);               // ready for the next binning
        cc[1] = make_int4(0, 0, 0, 0);
        return;
    }
#pragma unroll
    for (int k = 0; k < SCAN_V; k++) {
        const int idx = base + k;
        if (idx < P.NC) {
            P.cell_start[idx] = run;
            P.cell_count[idx] = 0;                   // ready for the next binning
            run += c[k];
            if (idx == P.NC - 1) P.cell_start[P.NC] = run;
        }
    }
}

// N4 in CSR form: the atom's place in the cell-ordered sequence s
__device__ __forceinline__ void place_body(const MdDev &P)
{
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.N; i += gridDim.x * blockDim.x)
        P.perm[P.cell_start[P.cell_of[i]] + P.slot[i]] = i;
}

__device__ __forceinline__ void bonds_remap_body(const MdDev &P, const Bufs B)
{
    const int *idv = P.id[B.vd];
    for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < P.N; n += gridDim.x * blockDim.x) {
        const int id = idv[n];
#pragma unroll
        for (int k = 0; k < 2; k++) {
            const int partner = P.bond_orig[(size_t)k * P.N + id];
            P.bond_dev[(size_t)k * P.N_pad + n] = partner >= 0 ? P.inv[partner] : -1;
        }
    }
}

constexpr int PERSIST_T = SCAN_T;      // block size of the persistent kernels: the scan tiles need exactly SCAN_T threads

}  // namespace
