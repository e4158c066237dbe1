// Device helpers shared by the kernel translation units (md_kernels.cu, md_tile.cu): 256-bit position
// loads/stores, the exact displacement arithmetic of DESIGN.md R5, warp/block reductions and the device-side
// rebuild decision.  Internal; not part of the boundary.
#pragma once
#include "md_types.h"

#define FULL_MASK 0xffffffffu
#define W_INDEX_MASK 0x1fffffffu     // 29 index bits ("3 bits are sufficient" for the flags)
#define W_FLAG_SHIFT 29
#ifndef MD_FORCE_U
#define MD_FORCE_U 2                 // gathers in flight per thread in the force loop
#endif
#ifndef MD_FORCE_MIN_THREADS
#define MD_FORCE_MIN_THREADS 1024    // resident threads per SM the register allocation must allow
#endif

namespace {

// ------------------------------------------------------------------------------------------------
// small device helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double minimg(double d, double L, double half)
{
    return d > half ? d - L : (d < -half ? d + L : d);
}

__device__ __forceinline__ double wrap1(double x, double L)
{
    if (x >= L) x -= L;
    else if (x < 0.0) { x += L; if (x >= L) x = 0.0; }
    return x;
}

// 32-byte record = one L2 sector, moved by ONE 256-bit access (LDG.E.ENL2.256 / STG.E.ENL2.256 on sm_100a):
// a gather then costs one L1 tag look-up per lane instead of two with a pair of 128-bit loads.
// Read-only path: never used on a buffer the same kernel writes.
#ifndef MD_LDPOS
#define MD_LDPOS 0                   // cache policy of the position gathers (tuning experiments)
#endif
__device__ __forceinline__ pos_t ld_pos(const pos_t *p)
{
    pos_t r;
#if MD_LDPOS == 1
    asm("ld.global.cg.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
#elif MD_LDPOS == 2
    asm("ld.global.nc.L1::evict_last.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
#elif MD_LDPOS == 3
    asm("ld.global.nc.L1::no_allocate.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
#elif MD_LDPOS == 4
    asm("ld.global.nc.L1::evict_last.L2::256B.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
#else
    asm("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
#endif
    return r;
}

__device__ __forceinline__ pos_t ld_pos_rw(const pos_t *p)
{
    pos_t r;
    asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
    return r;
}

// How the kernels read arrays that the SAME launch never writes (LdNC: the non-coherent read-only path) -- and how the
// persistent small-system kernel (md_kernels.cu: k_persist), which rewrites those arrays between its grid-wide barriers,
// must read them instead (LdPlain: ordinary coherent loads).
__device__ __forceinline__ float4 ld_f4_rw(const float4 *p)
{
    float4 r;
    asm volatile("ld.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
struct LdNC {
    static __device__ __forceinline__ float4 f4(const float4 *p) { return __ldg(p); }
    static __device__ __forceinline__ pos_t pos(const pos_t *p) { return ld_pos(p); }
    static __device__ __forceinline__ int i32(const int *p) { return __ldg(p); }
    static __device__ __forceinline__ double f64(const double *p) { return __ldg(p); }
};
struct LdPlain {
    static __device__ __forceinline__ float4 f4(const float4 *p) { return ld_f4_rw(p); }
    static __device__ __forceinline__ pos_t pos(const pos_t *p) { return ld_pos_rw(p); }
    static __device__ __forceinline__ int i32(const int *p) { return *(const volatile int *)p; }
    static __device__ __forceinline__ double f64(const double *p) { return *(const volatile double *)p; }
};

__device__ __forceinline__ void st_pos(pos_t *p, double x, double y, double z)
{
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(x), "d"(y), "d"(z), "d"(0.0) : "memory");
}

// 1/x to within ~1 ulp without the IEEE-division slow path: hardware seed (relative error <= 2^-23) + one
// third-order (Halley) step, y (1 + e + e^2) with e = 1 - x y: error e^3 ~ 2^-69, i.e. rounding only.
// (Forces are compared with the oracle to 1e-10; the accept tests use r^2 itself.)
__device__ __forceinline__ double fast_rcp(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double t = fma(e, e, e);
    return fma(y, t, y);
}

// Displacement r_i - r_j with the image correction frozen into the W entry (flag bit k set = subtract +-L
// along axis k, sign taken from the raw difference).  On freshly wrapped coordinates this is
// bit-for-bit the minimum-image arithmetic of DESIGN.md R5 (d0 = a - b rounded; d0 -+ L rounded), so
// r^2 = fma(dz,dz, fma(dy,dy, dx*dx)) decides r^2 < r_c^2 on the same bits as any other implementation.
__device__ __forceinline__ double disp2(const pos_t &a, const pos_t &b, unsigned fl, double L, double &dx, double &dy, double &dz)
{
    dx = a.x - b.x;
    dy = a.y - b.y;
    dz = a.z - b.z;
    if (fl) {                                   // only atoms next to a periodic face take this branch
        if (fl & 1u) dx -= copysign(L, dx);
        if (fl & 2u) dy -= copysign(L, dy);
        if (fl & 4u) dz -= copysign(L, dz);
    }
    return __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
}

__device__ __forceinline__ int cell_coord(double x, double inv_w, int nc)
{
    int q = (int)floor(x * inv_w);
    q = q < 0 ? 0 : q;
    return q >= nc ? nc - 1 : q;
}

// Row pruning of the neighbor build (MdDev::kx): an atom at fractional height (fy, fz) in its cell is at least
// gyl = fy w below-row gap, gyh = (1 - fy) w above-row gap ... away from the rows of cells next to its own.  A partner
// in the row (dy, dz) can then differ by at most s = sqrt(r_n^2 - g^2) along x, i.e. lie at most floor(s / w_x) + 1
// fine cells away.  All quantities are binary32 rounded to the safe side (gaps shrunk, r_n^2 and 1 / w_x grown by
// 1e-5, against a binary32 rounding of 6e-8 and a cell margin of >= 1e-9), so the window never loses a partner; the
// accept test itself stays the exact arithmetic of DESIGN.md R5 / R18.
struct RowGaps {
    float yl, yh, zl, zh;
};

__device__ __forceinline__ RowGaps row_gaps(const MdDev &P, double y, double z, int cy, int cz)
{
    const float fy = (float)(y * P.inv_w - (double)cy), fz = (float)(z * P.inv_w - (double)cz);
    RowGaps G;
    G.yl = fmaxf(fy, 0.0f) * P.w_f; G.yh = fmaxf(1.0f - fy, 0.0f) * P.w_f;
    G.zl = fmaxf(fz, 0.0f) * P.w_f; G.zh = fmaxf(1.0f - fz, 0.0f) * P.w_f;
    return G;
}

// half-width of the x window (in fine cells) of the row (dy, dz) in {-1, 0, 1}^2; -1: the row is out of reach
__device__ __forceinline__ int row_halfwidth(const MdDev &P, const RowGaps &G, int dy, int dz)
{
    const float gy = dy < 0 ? G.yl : (dy > 0 ? G.yh : 0.0f), gz = dz < 0 ? G.zl : (dz > 0 ? G.zh : 0.0f);
    const float s2 = P.rn2_prune - (gy * gy + gz * gz);
    if (!(s2 > 0.0f)) return -1;
    const int k = (int)(sqrtf(s2) * P.inv_wx_f) + 1;
    return k < P.kx ? k : P.kx;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(FULL_MASK, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fmax(v, __shfl_xor_sync(FULL_MASK, v, o));
    return v;
}
__device__ __forceinline__ int warp_sum_i(int v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(FULL_MASK, v, o);
    return v;
}
__device__ __forceinline__ int warp_max_i(int v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v = max(v, __shfl_xor_sync(FULL_MASK, v, o));
    return v;
}

// block-wide max of a non-negative double; result valid in thread 0.  sm: >= 32 doubles.
__device__ __forceinline__ double block_max(double v, double *sm)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    v = warp_max(v);
    if (lane == 0) sm[wid] = v;
    __syncthreads();
    if (wid == 0) {
        v = lane < nw ? sm[lane] : 0.0;
        v = warp_max(v);
    }
    return v;
}

// A drifting kernel leaves its blocks' maxima of v^2 for k_decide in DEC_SLOTS words (block b in slot b mod DEC_SLOTS) with a
// fire-and-forget atomic maximum: v^2 is finite and >= +0, and the bit patterns of such doubles order as unsigned integers.
// k_decide then reads -- and clears -- 64 words instead of one entry per block (16,384 at N = 2M): 6.7 -> 5.1 us per step on top
// of the fused kernel.  A maximum does not depend on the order of the atomics: results stay bitwise reproducible.
constexpr int DEC_SLOTS = 64;
__device__ __forceinline__ void publish_vmax2(const MdDev &P, int bid, double bm)
{
    atomicMax(reinterpret_cast<unsigned long long *>(P.blk_vmax2) + (bid & (DEC_SLOTS - 1)), (unsigned long long)__double_as_longlong(bm));
}

// The rebuild decision (R8), taken on the device by k_decide from the per-block maxima of
// v^2 that the drifting kernel left in blk_vmax2.  It also fixes which buffers the rebuild kernels read and
// write, so the host never needs to know whether a rebuild happened.
// (A "last block done" ticket inside the drifting kernel, was measured at ~7.5 ns per block on
// B200 -- two same-address L2 atomics and a fence per block, ~75 us for the 10^4 blocks of N = 2M, more than
// the rest of the kernel -- so the decision moved to a one-block kernel ordered by the stream.)
// the scalars of the decision and the buffer roles it fixes (a copy of the corresponding DevCtrl fields)
struct DecState {
    double disp_acc;
    int p_src, p_dst, v_src, v_dst, need_rebuild, n_rebuilds, do_reorder, since_reorder;
};

__device__ __forceinline__ DecState dec_load(const MdDev &P)
{
    const volatile DevCtrl *c = P.ctrl;
    DecState d;
    d.disp_acc = c->disp_acc; d.p_src = c->p_src; d.p_dst = c->p_dst; d.v_src = c->v_src; d.v_dst = c->v_dst;
    d.need_rebuild = c->need_rebuild; d.n_rebuilds = c->n_rebuilds; d.do_reorder = c->do_reorder; d.since_reorder = c->since_reorder;
    return d;
}

__device__ __forceinline__ void dec_store(const MdDev &P, const DecState &d)
{
    volatile DevCtrl *c = P.ctrl;
    if (d.need_rebuild) { c->max_occ = 0; c->max_nnb = 0; c->nnb_total = 0ull; c->cand_total = 0ull; }
    c->disp_acc = d.disp_acc; c->p_src = d.p_src; c->p_dst = d.p_dst; c->v_src = d.v_src; c->v_dst = d.v_dst;
    c->need_rebuild = d.need_rebuild; c->n_rebuilds = d.n_rebuilds; c->do_reorder = d.do_reorder; c->since_reorder = d.since_reorder;
}

// pure: the same inputs give the same decision in every thread that evaluates it (k_persist replicates it per block)
__device__ __forceinline__ void decide_state(const MdDev &P, DecState &c, double vmax2, bool pos_pingpong)
{
    double acc = c.disp_acc + P.dt * sqrt(vmax2);
    const int need = acc > P.thresh;
    c.since_reorder += 1;
    if (need) {
        acc = 0.0;
        c.n_rebuilds += 1;
        // the paper sorts the atoms only every ~100 steps; the default path at every rebuild
        const int ro = !P.layer_H || P.reorder_interval == 0 || (P.reorder_interval > 0 && c.since_reorder >= P.reorder_interval);
        c.do_reorder = ro;
        if (ro) c.since_reorder = 0;
    }
    c.disp_acc = acc;
    c.need_rebuild = need;
    const int ps = pos_pingpong ? (c.p_dst ^ 1) : c.p_dst;
    c.p_src = ps;
    c.p_dst = need ? (ps ^ 1) : ps;
    const int vs = c.v_dst;
    c.v_src = vs;
    c.v_dst = need ? (vs ^ 1) : vs;
}

__device__ __forceinline__ void decide(const MdDev &P, double vmax2, bool pos_pingpong)
{
    DecState c = dec_load(P);
    decide_state(P, c, vmax2, pos_pingpong);
    dec_store(P, c);
}

__device__ __forceinline__ void set_err(const MdDev &P, int code) { atomicCAS(&P.ctrl->err, 0, code); }

// F2 and the other global sums: warp shuffles -> shared memory -> one partial per block
// -> the last block (atomic ticket + memory fence) finishes in a fixed order, so results are reproducible.
// q[k] = this thread's contribution (RED_VMAX2 is a max, the others sums).  All threads of the block call it.
struct RedSmem {
    double v[RED_N][32];
    bool last;
};

__device__ __forceinline__ void reduce_finish(const MdDev &P, const double (&q)[RED_N], RedSmem &S, int bid, int nblk)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int k = 0; k < RED_N; k++) {
        const double r = k == RED_VMAX2 ? warp_max(q[k]) : warp_sum(q[k]);
        if (lane == 0) S.v[k][wid] = r;
    }
    __syncthreads();
    if (threadIdx.x < RED_N) {
        const int k = threadIdx.x;
        double r = S.v[k][0];
        for (int w = 1; w < nw; w++) r = k == RED_VMAX2 ? fmax(r, S.v[k][w]) : r + S.v[k][w];
        P.partials[(size_t)k * P.max_grid + bid] = r;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned t = atomicInc(&P.ctrl->ticket[TK_ENERGY], nblk - 1);
        S.last = (t == (unsigned)(nblk - 1));
    }
    __syncthreads();
    if (!S.last) return;
    __threadfence();
    // the last block sums the partials of all blocks (itself included), fixed order
    for (int k = 0; k < RED_N; k++) {
        double r = 0.0;
        const volatile double *p = P.partials + (size_t)k * P.max_grid;
        for (int b = threadIdx.x; b < nblk; b += blockDim.x) r = k == RED_VMAX2 ? fmax(r, p[b]) : r + p[b];
        r = k == RED_VMAX2 ? warp_max(r) : warp_sum(r);
        __syncthreads();
        if (lane == 0) S.v[0][wid] = r;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = S.v[0][0];
            for (int w = 1; w < nw; w++) t = k == RED_VMAX2 ? fmax(t, S.v[0][w]) : t + S.v[0][w];
            P.ctrl->red[k] = t;
        }
    }
}

}  // namespace
