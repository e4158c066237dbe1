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
// The tile layout is a pure function of (block index, cell_start); cell_start only changes at a rebuild, so the
// build kernel computes it once per box, stores it as a TileDesc in global memory, and every later force /
// energy kernel reads it back with one coalesced load.  Inside a block the global-memory latencies are
// overlapped, not chained: descriptor -> {W words + velocities of the own atoms, position tile} -> compute.
#include <algorithm>

#include "md_device.cuh"

// Experiment: stage the BUILD kernel's fp64 tile with TMA bulk copies (cp.async.bulk, one per contiguous
// piece of a tile row, completion on an mbarrier) instead of LDG.256 + 3 STS through registers.  The tile then holds the
// 32-byte position records as they are in global memory (stride 4 doubles instead of the packed 3).
#ifndef MD_TILE_TMA
#define MD_TILE_TMA 0
#endif
constexpr int TSTR64 = MD_TILE_TMA ? 4 : 3;      // doubles per atom in the build kernel's fp64 tile

#ifndef MD_TILE_FORCE_THREADS
#define MD_TILE_FORCE_THREADS 1024     // resident threads per SM the register allocation of k_tile_force must allow
#endif

namespace {

__device__ __forceinline__ int tile_bid(const TileGeom &G) { return blockIdx.x + G.nsx * (blockIdx.y + G.nsy * blockIdx.z); }

// what only the build kernel needs per tile row: the row's x = 0 cell and its image shift in units of L
struct TileRowGeom {
    int row_cell[TILE_Q_MAX], ysh[TILE_Q_MAX], zsh[TILE_Q_MAX];
    int xa, xc;         // first cell of the halo before / after the box (the same in every row)
};

// Build kernel, step 1: the descriptor of box blockIdx.x from cell_start.  All threads of the block call it.
__device__ __forceinline__ void tile_describe(const MdDev &P, const TileBox &B, TileDesc &M, TileRowGeom &X)
{
    const int nc = P.nc, ncx = P.ncx, K = P.kx;
    const int *__restrict__ cs = P.cell_start;
    const int tid = threadIdx.x;
    if (tid < B.nq) {
        const int q = tid;
        int rowc, ysh, zsh, xa, xc;
        tile_row(B, nc, ncx, K, q, rowc, ysh, zsh, xa, xc);
        // the three contiguous pieces of the row: K halo cells, the box's own cells, K halo cells
        const int gA = __ldg(cs + rowc + xa), nA = __ldg(cs + rowc + xa + K) - gA;
        const int gB = __ldg(cs + rowc + B.x0), nB = __ldg(cs + rowc + B.x0 + B.sxc) - gB;
        const int gC = __ldg(cs + rowc + xc), nC = __ldg(cs + rowc + xc + K) - gC;
        M.row[q].g[0] = gA; M.row[q].g[1] = gB; M.row[q].g[2] = gC;
        M.row[q].n[0] = nA; M.row[q].n[1] = nB; M.row[q].n[2] = nC;
        X.row_cell[q] = rowc; X.ysh[q] = ysh; X.zsh[q] = zsh;
        if (q == 0) { X.xa = xa; X.xc = xc; }
        // piece 0 holds the far-face cells when the box starts at x = 0: d = (r_i - r_j) + L; piece 2 likewise with -L
        const int xshA = B.x0 == 0 ? 1 : 0, xshC = B.x0 + B.sxc == ncx ? -1 : 0;
        M.row[q].sh = (ysh + 1) | ((zsh + 1) << 2) | ((xshA + 1) << 4) | ((xshC + 1) << 6);
    }
    __syncthreads();
    if (tid < 32) {
        // prefix sums over the <= 25 tile rows by warp 0: tile offset of each row, and for the rows of the box itself
        // (own rows) their rank k and the prefix of their lengths
        const int q = tid;
        const bool in = q < B.nq;
        const int nA = in ? M.row[q].n[0] : 0, nB = in ? M.row[q].n[1] : 0, nC = in ? M.row[q].n[2] : 0;
        const int qy = q % B.nyq, qz = q / B.nyq;
        const bool own_row = in && qy >= 1 && qy <= B.ny && qz >= 1 && qz <= B.nz;
        const int tot = nA + nB + nC, ownn = own_row ? nB : 0;
        int inc = tot, oinc = ownn;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t1 = __shfl_up_sync(FULL_MASK, inc, o), t2 = __shfl_up_sync(FULL_MASK, oinc, o);
            if (tid >= o) { inc += t1; oinc += t2; }
        }
        const int off = inc - tot, opre = oinc - ownn;
        const unsigned ownmask = __ballot_sync(FULL_MASK, own_row);
        const int k = __popc(ownmask & ((1u << tid) - 1u)), nown_rows = __popc(ownmask);
        const int T = __shfl_sync(FULL_MASK, inc, 31), n_own = __shfl_sync(FULL_MASK, oinc, 31);
        if (in) M.row[q].off = off;
        if (own_row) { M.own_base[k] = M.row[q].g[1]; M.own_loc[k] = off + nA; M.own_pre[k] = opre; }
        if (tid >= nown_rows && tid <= TILE_OWN_MAX) {
            M.own_pre[tid] = n_own;
            if (tid < TILE_OWN_MAX) { M.own_base[tid] = 0; M.own_loc[tid] = 0; }
        }
        if (tid == 0) { M.n_own = n_own; M.T = T; M.nq = B.nq; M.pad = 0; }
    }
    __syncthreads();
}

// one tile row's copy parameters in registers (the descriptor lives in shared memory, which the staging stores
// alias, so the compiler would otherwise reload it inside the copy loop)
struct RowCopy {
    int tot, g0, n0, n01, b1, b2, off3;     // src = u + (u < n0 ? g0 : u < n01 ? b1 : b2);  dst = off3 + 3 u
    bool contiguous, xwrap;
    double shxA, shxC, shy, shz;            // image shifts (IMAGE only)
};

template <bool IMAGE>
__device__ __forceinline__ RowCopy row_copy(const TileDesc::Row &R, double L)
{
    RowCopy c;
    const int g0 = R.g[0], g1 = R.g[1], g2 = R.g[2], n0 = R.n[0], n1 = R.n[1], n2 = R.n[2], sh = R.sh;
    c.tot = n0 + n1 + n2; c.g0 = g0; c.n0 = n0; c.n01 = n0 + n1;
    c.b1 = g1 - n0; c.b2 = g2 - n0 - n1; c.off3 = 3 * R.off;
    c.contiguous = g0 + n0 == g1 && g1 + n1 == g2;
    c.xwrap = false; c.shxA = c.shxC = c.shy = c.shz = 0.0;
    if (IMAGE) {
        const int xa = ((sh >> 4) & 3) - 1, xc = ((sh >> 6) & 3) - 1;
        c.xwrap = (xa | xc) != 0;
        c.shxA = xa * L; c.shxC = xc * L; c.shy = ((sh & 3) - 1) * L; c.shz = (((sh >> 2) & 3) - 1) * L;
    }
    return c;
}

template <bool IMAGE>
__device__ __forceinline__ pos_t row_load(const RowCopy &c, const pos_t *__restrict__ pos, int u)
{
    const int src = c.contiguous ? c.g0 + u : u + (u < c.n0 ? c.g0 : (u < c.n01 ? c.b1 : c.b2));
    pos_t p = ld_pos(pos + src);
    if (IMAGE) {
        p.y -= c.shy; p.z -= c.shz;
        if (c.xwrap) p.x -= u < c.n0 ? c.shxA : (u >= c.n01 ? c.shxC : 0.0);
    }
    return p;
}

__device__ __forceinline__ void row_store(const RowCopy &c, double *st, int u, const pos_t &p)
{
    double *d = st + c.off3 + 3 * u;
    d[0] = p.x; d[1] = p.y; d[2] = p.z;
}

// Copy the positions of the tile into shared memory as packed (x, y, z) triples: st[3 j + k].  One warp per
// tile row, two rows and two 32-atom chunks of each in flight per lane (4 independent 256-bit loads) before
// the first shared-memory store.
// IMAGE: store the periodic IMAGE the box sees, r_j - shift (shift = 0 or +-L per axis, fixed per tile row and
// piece), so that the pair loop needs no flag handling.  r - L is exact (Sterbenz) and r + L is rounded once at
// magnitude L, the same size of error as the oracle's (r_i - r_j) at the far face: ~1e-16 relative to L, far
// inside the 1e-10 force tolerance.  The build kernel stages raw positions (IMAGE = false) and applies the
// shift to the difference, because its accept test must reproduce DESIGN.md R5 bit for bit.
template <bool IMAGE>
__device__ __forceinline__ void tile_stage(const TileDesc &M, const pos_t *__restrict__ pos, double *st, double L)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int nq = M.nq;
    for (int qa = wid; qa < nq; qa += 2 * nw) {
        const RowCopy A = row_copy<IMAGE>(M.row[qa], L);
        RowCopy B = A;
        B.tot = 0;
        if (qa + nw < nq) B = row_copy<IMAGE>(M.row[qa + nw], L);
        const int tmax = A.tot > B.tot ? A.tot : B.tot;
        for (int u = lane; u < tmax; u += 64) {
            pos_t a0, a1, b0, b1;
            const bool va0 = u < A.tot, va1 = u + 32 < A.tot, vb0 = u < B.tot, vb1 = u + 32 < B.tot;
            if (va0) a0 = row_load<IMAGE>(A, pos, u);
            if (va1) a1 = row_load<IMAGE>(A, pos, u + 32);
            if (vb0) b0 = row_load<IMAGE>(B, pos, u);
            if (vb1) b1 = row_load<IMAGE>(B, pos, u + 32);
            if (va0) row_store(A, st, u, a0);
            if (va1) row_store(A, st, u + 32, a1);
            if (vb0) row_store(B, st, u, b0);
            if (vb1) row_store(B, st, u + 32, b1);
        }
    }
}

// own atom number t of the block -> global index i and tile index li
__device__ __forceinline__ void own_atom(const TileDesc &M, int t, int &i, int &li)
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
// range of the shared array.  Lanes in the same cell read the same shared-memory words (broadcast).
// Accept test and image arithmetic are those of DESIGN.md R5, bit for bit: d = (r_i - r_j) rounded, + shift
// rounded, r^2 = fma(dz,dz, fma(dy,dy, dx*dx)) < r_n^2.
// LOCALW: W entries are 16-bit tile indices packed two per word (MD_W_TILED); otherwise 29-bit global atom
// indices, one per word (MD_W_GLOBAL) -- the same kernel then feeds the gathering force kernels.
// ------------------------------------------------------------------------------------------------
// Appending to column i of W is written so that it compiles to predicated instructions, not a divergent
// block: in a warp some lane accepts its candidate in most iterations, so a branch would be taken (by a few
// lanes, the others idling) nearly every time.  Tiled layout: entry m of the column is the 16-bit half
// (m & 1) of word (m >> 1) * pitch + i, written with a 16-bit store.
template <bool LOCALW>
struct Emit {
    char *wp;           // address of the next free entry of column i of W
    long long pitch4;   // bytes between consecutive word rows
    int m, Mmax;
    // candidate with tile index j; add = (flags << shift) + (global - tile index), constant over a run
    __device__ __forceinline__ void put(bool acc, int j, unsigned add)
    {
        const unsigned e = (unsigned)j + add;
        const bool st = acc && m < Mmax;
        if (LOCALW) {
            if (st) *(unsigned short *)wp = (unsigned short)e;
            const long long step = (m & 1) ? pitch4 - 2 : 2;
            wp += acc ? step : 0;
        } else {
            if (st) *(unsigned *)wp = e;
            wp += acc ? pitch4 : 0;
        }
        m += acc;
    }
    // an odd column leaves the upper half of its last word unwritten: clear it, the force kernel reads whole words
    __device__ __forceinline__ void flush()
    {
        if (LOCALW && (m & 1) && m < Mmax) *(unsigned short *)wp = 0;
    }
};

template <bool SHIFT, bool LOCALW>
__device__ __forceinline__ void tile_scan_run(const double *st, double xi, double yi, double zi, int li, int b, int e, double shx,
                                              double shy, double shz, unsigned add, double rn2, Emit<LOCALW> &em)
{
    const double *p = st + TSTR64 * b;
#pragma unroll 2
    for (int j = b; j < e; j++, p += TSTR64) {
        double dx = __dsub_rn(xi, p[0]), dy = __dsub_rn(yi, p[1]), dz = __dsub_rn(zi, p[2]);
        if (SHIFT) { dx = __dadd_rn(dx, shx); dy = __dadd_rn(dy, shy); dz = __dadd_rn(dz, shz); }
        const double r2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
        em.put(r2 < rn2 && j != li, j, add);
    }
}

// binary32 tile of the single-precision variant (md_sp.cu; R18): packed triples, raw positions
__device__ __forceinline__ void tile_stage_f(const TileDesc &M, const float4 *__restrict__ pos, float *st)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int q = wid; q < M.nq; q += nw) {
        const RowCopy A = row_copy<false>(M.row[q], 0.0);
        for (int u = lane; u < A.tot; u += 64) {
            const int u1 = u + 32;
            const int s0 = A.contiguous ? A.g0 + u : u + (u < A.n0 ? A.g0 : (u < A.n01 ? A.b1 : A.b2));
            const int s1 = A.contiguous ? A.g0 + u1 : u1 + (u1 < A.n0 ? A.g0 : (u1 < A.n01 ? A.b1 : A.b2));
            const float4 p0 = __ldg(pos + s0);
            float4 p1 = p0;
            if (u1 < A.tot) p1 = __ldg(pos + s1);
            float *d = st + A.off3 + 3 * u;
            d[0] = p0.x; d[1] = p0.y; d[2] = p0.z;
            if (u1 < A.tot) { d[96] = p1.x; d[97] = p1.y; d[98] = p1.z; }
        }
    }
}

// Packed binary32 arithmetic of sm_100 (FFMA2 / FADD2: two IEEE-rounded lanes per instruction): the accept test of TWO
// consecutive candidates at once.  Lane-wise the operations are those of DESIGN.md R18 (d = fl(x_i - x_j) as
// fma(-1, x_j, x_i), one rounding; + shift rounded once; r2 = fma(dz,dz, fma(dy,dy, fl(dx dx)))), so the sets stay exact.
__device__ __forceinline__ unsigned long long pack2(float a, float b)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void unpack2(unsigned long long v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long mul2(unsigned long long a, unsigned long long b)
{
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ unsigned long long add2(unsigned long long a, unsigned long long b)
{
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

template <bool SHIFT, bool LOCALW>
__device__ __forceinline__ void tile_scan_run(const float *st, float xi, float yi, float zi, int li, int b, int e, float shx, float shy,
                                              float shz, unsigned add, float rn2, Emit<LOCALW> &em)
{
    const unsigned long long m1 = pack2(-1.0f, -1.0f), x2 = pack2(xi, xi), y2 = pack2(yi, yi), z2 = pack2(zi, zi);
    const unsigned long long sx2 = pack2(shx, shx), sy2 = pack2(shy, shy), sz2 = pack2(shz, shz);
    const float *p = st + 3 * b;
    int j = b;
#pragma unroll 2
    for (; j + 1 < e; j += 2, p += 6) {
        unsigned long long dx = fma2(m1, pack2(p[0], p[3]), x2), dy = fma2(m1, pack2(p[1], p[4]), y2), dz = fma2(m1, pack2(p[2], p[5]), z2);
        if (SHIFT) { dx = add2(dx, sx2); dy = add2(dy, sy2); dz = add2(dz, sz2); }
        const unsigned long long r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
        float ra, rb;
        unpack2(r2, ra, rb);
        em.put(ra < rn2 && j != li, j, add);
        em.put(rb < rn2 && j + 1 != li, j + 1, add);
    }
    if (j < e) {
        float dx = __fsub_rn(xi, p[0]), dy = __fsub_rn(yi, p[1]), dz = __fsub_rn(zi, p[2]);
        if (SHIFT) { dx = __fadd_rn(dx, shx); dy = __fadd_rn(dy, shy); dz = __fadd_rn(dz, shz); }
        const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
        em.put(r2 < rn2 && j != li, j, add);
    }
}

// What differs between the two precisions of the tile build: the coordinate type, where the positions come from, how
// the tile is staged, and the constants of the accept test.  Everything else -- the box decomposition, the descriptor,
// the candidate windows, the append -- is ONE kernel (k_tile_build below).
#if MD_TILE_TMA
// TMA staging of the raw 32-byte records: warp 0 issues one bulk copy per non-empty piece of every tile row; all threads
// then wait on the mbarrier's phase 0.  (sm_90+ PTX; SASS UBLKCP.)
__device__ __forceinline__ void tile_stage_tma(const TileDesc &M, const pos_t *__restrict__ pos, double *st)
{
    __shared__ __align__(8) unsigned long long mbar;
    const unsigned mb = (unsigned)__cvta_generic_to_shared(&mbar);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        if (lane == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"((unsigned)M.T * 32u) : "memory");
        __syncwarp();
        for (int e = lane; e < 3 * M.nq; e += 32) {
            const int q = e / 3, k = e - 3 * q;
            const TileDesc::Row &R = M.row[q];
            const int n = R.n[k];
            if (n == 0) continue;
            const int toff = R.off + (k > 0 ? R.n[0] : 0) + (k > 1 ? R.n[1] : 0);
            const unsigned dst = (unsigned)__cvta_generic_to_shared(st + 4 * toff);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                         "l"(pos + R.g[k]), "r"((unsigned)n * 32u), "r"(mb)
                         : "memory");
        }
    }
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_TMA:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0;\n\t@!p bra WAIT_TMA;\n\t}" ::"r"(mb) : "memory");
}
#endif

struct PrecF64 {
    using real = double;
    static constexpr int STR = TSTR64;
    static __device__ __forceinline__ void stage(const MdDev &P, const TileDesc &M, int pc, real *st)
    {
#if MD_TILE_TMA
        tile_stage_tma(M, P.pos[pc], st);
#else
        tile_stage<false>(M, P.pos[pc], st, P.L);
#endif
    }
    static __device__ __forceinline__ real box(const MdDev &P) { return P.L; }
    static __device__ __forceinline__ real rn2(const MdDev &P) { return P.rn2; }
};
struct PrecF32 {
    using real = float;
    static constexpr int STR = 3;
    static __device__ __forceinline__ void stage(const MdDev &P, const TileDesc &M, int pc, real *st) { tile_stage_f(M, P.posf[pc], st); }
    static __device__ __forceinline__ real box(const MdDev &P) { return P.Lf; }
    static __device__ __forceinline__ real rn2(const MdDev &P) { return P.rn2f; }
};

// The block size is a run-time value (any multiple of 32 up to 512): it is picked so that the own atoms of a box
// fill the block's warps.
// Registers (measured): ptxas picks 56-64 under this bound; caps of 56 / 48 (a fifth resident block of the former
// 224-thread blocks) gained only in binary32 and nothing once the boxes were made for 256-thread blocks (4 blocks of 256 = 1024
// threads per SM need <= 64 registers anyway).
template <typename PR, bool LOCALW>
__global__ void __launch_bounds__(512) k_tile_build(const __grid_constant__ MdDev P)
{
    using real = typename PR::real;
    const int BLOCK = blockDim.x;
    if (!__ldcg(&P.ctrl->need_rebuild)) return;
    extern __shared__ double dsm[];
    __shared__ TileDesc M;
    __shared__ TileRowGeom X;
    __shared__ int smx[32], ssum[32], scand[32];
    struct RowC { real shy, shz; unsigned fl, add0; int e0, e1, d0, d1, d2, pad; };
    __shared__ RowC rc[TILE_Q_MAX];
    const int cap = P.tg.cap, K = P.kx;
    const int stride = P.tg.S + 2 * K + 1;
    real *st = (real *)dsm;
    int *tcs = (int *)(st + PR::STR * cap);           // tile index of the first atom of every tile cell
    const int *__restrict__ cs = P.cell_start;
    const TileBox B = tile_box3(P.tg, P.nc, P.ncx, blockIdx.x, blockIdx.y, blockIdx.z);
    const int bid = tile_bid(P.tg);
    tile_describe(P, B, M, X);
    if (LOCALW) {   // publish the descriptor for the force / energy kernels
        int *d = P.tile_desc + (size_t)bid * TILE_DESC_INTS;
        const int n = TILE_DESC_HEAD + TILE_ROW_INTS * B.nq;
        for (int k = threadIdx.x; k < n; k += BLOCK) d[k] = ((const int *)&M)[k];
    }
    if (M.T > cap) {
        if (threadIdx.x == 0) set_err(P, MD_ERR_TILE_OVERFLOW);
        return;
    }
    // tcs[q * stride + k], k = 0 .. sxc + 2 K  (K halo cells, the box's sxc cells, K halo cells; the last entry closes the row):
    // tile index of the first atom of tile cell k of row q = (start of the cell in the global order) + (tile offset - global
    // start of the row's piece)
    const int n_tcs = B.nq * stride;
    auto tcs_fetch = [&](int e, int &add) -> int {      // the global load of entry e; add: what turns it into the tile index
        const int q = e / stride, k = e - q * stride;
        const TileDesc::Row &R = M.row[q];
        if (k < K) { add = R.off - R.g[0]; return __ldg(cs + X.row_cell[q] + X.xa + k); }
        if (k < K + B.sxc) { add = R.off + R.n[0] - R.g[1]; return __ldg(cs + X.row_cell[q] + B.x0 + k - K); }
        add = R.off + R.n[0] + R.n[1] - R.g[2];
        return k <= B.sxc + 2 * K ? __ldg(cs + X.row_cell[q] + X.xc + k - K - B.sxc) : 0;       // past the closing entry: never read
    };
    PR::stage(P, M, __ldcg(&P.ctrl->p_dst), st);
    // in batches of four loads before their four stores: a shared-memory store that waits for its global load would otherwise
    // hold back the next entry's load (one round of latency per entry): build 0.357 -> 0.342 ms at wca_2m_dr03.  (Requesting them
    // BEFORE the tile is staged, 8 registers held across the staging, gained 3 % in binary32 with the former 224-thread boxes and
    // nothing with the present ones.)
    for (int e0 = threadIdx.x; e0 < n_tcs; e0 += 4 * BLOCK) {
        int v[4], add[4];
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const int e = e0 + k * BLOCK;
            v[k] = 0; add[k] = 0;
            if (e < n_tcs) v[k] = tcs_fetch(e, add[k]);
        }
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const int e = e0 + k * BLOCK;
            if (e < n_tcs) tcs[e] = v[k] + add[k];
        }
    }
    // per tile row: periodic shifts along y, z, their flag bits, the index offsets of the row's (up to) three contiguous
    // pieces (global index = tile index + delta) -- everything of a run's set-up that does not depend on the atom
    for (int q = threadIdx.x; q < B.nq; q += BLOCK) {
        const int ysh = X.ysh[q], zsh = X.zsh[q];
        const unsigned fl = (ysh ? 2u : 0u) | (zsh ? 4u : 0u);
        const TileDesc::Row &R = M.row[q];
        RowC c;
        c.shy = ysh * PR::box(P); c.shz = zsh * PR::box(P);
        c.fl = fl;
        c.e0 = R.off + R.n[0]; c.e1 = c.e0 + R.n[1];
        c.d0 = R.g[0] - R.off; c.d1 = R.g[1] - c.e0; c.d2 = R.g[2] - c.e1; c.pad = 0;
        c.add0 = LOCALW ? fl << T_FLAG_SHIFT : (fl << W_FLAG_SHIFT) + (unsigned)c.d0;
        rc[q] = c;
    }
    __syncthreads();
    const int nc = P.nc, ncx = P.ncx;
    const real L = PR::box(P), rn2 = PR::rn2(P);
    const bool low_face = B.x0 == 0, high_face = B.x0 + B.sxc == ncx;
    const bool interior = !low_face && !high_face;           // block-uniform: every tile row is ONE global range, no image along x
    int tmax = 0, tsum = 0, tcand = 0;
    for (int t = threadIdx.x; t < M.n_own; t += BLOCK) {
        int i, li;
        own_atom(M, t, i, li);
        const real xi = st[PR::STR * li], yi = st[PR::STR * li + 1], zi = st[PR::STR * li + 2];
        const int cx = cell_coord((double)xi, P.inv_wx, ncx), cy = cell_coord((double)yi, P.inv_w, nc), cz = cell_coord((double)zi, P.inv_w, nc);
        Emit<LOCALW> em = {(char *)((unsigned *)P.W + (size_t)i * P.w_col), 4ll * P.w_row, 0, P.Mmax};
        const int kc = cx - B.x0;                                  // the window of K cells either side starts at tile cell kc
        const int q0 = (cy - B.y0) + B.nyq * (cz - B.z0);          // tile row (cy - 1, cz - 1)
        // (Shortening the window of rows that are far from the atom -- row_halfwidth, as the gathering build does -- was
        // measured slower here, in round 1 and again in round 2: the lanes of a warp then walk runs of more unequal lengths.)
        if (interior) {
            // the per-run set-up is one 16-byte and two 4-byte shared-memory reads (measured: build 0.385 -> 0.362 ms at wca_2m_dr03)
#pragma unroll 1
            for (int rz = 0; rz < 3; rz++) {
#pragma unroll 1
                for (int ry = 0; ry < 3; ry++) {
                    const int q = q0 + ry + B.nyq * rz;
                    const RowC c = rc[q];
                    const int *tc = tcs + q * stride + kc;
                    const int b = tc[0], e = tc[2 * K + 1];       // tile cells [kc, kc + 2 K + 1)
                    tcand += e - b;
                    if (c.fl) tile_scan_run<true, LOCALW>(st, xi, yi, zi, li, b, e, (real)0, c.shy, c.shz, c.add0, rn2, em);
                    else tile_scan_run<false, LOCALW>(st, xi, yi, zi, li, b, e, (real)0, (real)0, (real)0, c.add0, rn2, em);
                }
            }
        } else {
#pragma unroll 1
            for (int r = 0; r < 9; r++) {
                const int q = q0 + (r % 3) + B.nyq * (r / 3);
                const RowC c = rc[q];
                const unsigned fl = c.fl;
                const real shy = c.shy, shz = c.shz;
                const int *tc = tcs + q * stride + kc;
                const int b = tc[0], e = tc[2 * K + 1];
                tcand += e - b;
                // split off the part of the window that is a periodic image along x (box at an x face, window reaching
                // into the halo that holds the cells of the other end of the row)
                const bool ima = low_face && kc < K, imb = high_face && kc + K + 1 > B.sxc;
                const int mid = ima ? tc[K - kc] : (imb ? tc[K + B.sxc - kc] : e);
                const int da = b < c.e0 ? c.d0 : (b < c.e1 ? c.d1 : c.d2), db = mid < c.e0 ? c.d0 : (mid < c.e1 ? c.d1 : c.d2);
                const real shxa = ima ? L : (real)0, shxb = imb ? -L : (real)0;
                const unsigned fla = fl | (ima ? 1u : 0u), flb = fl | (imb ? 1u : 0u);
                // what is added to the tile index to make the W entry: the flag bits, and for global W the index offset
                const unsigned adda = LOCALW ? fla << T_FLAG_SHIFT : (fla << W_FLAG_SHIFT) + (unsigned)da;
                const unsigned addb = LOCALW ? flb << T_FLAG_SHIFT : (flb << W_FLAG_SHIFT) + (unsigned)db;
                if (fla) tile_scan_run<true, LOCALW>(st, xi, yi, zi, li, b, mid, shxa, shy, shz, adda, rn2, em);
                else tile_scan_run<false, LOCALW>(st, xi, yi, zi, li, b, mid, (real)0, (real)0, (real)0, adda, rn2, em);
                if (mid < e) {
                    if (flb) tile_scan_run<true, LOCALW>(st, xi, yi, zi, li, mid, e, shxb, shy, shz, addb, rn2, em);
                    else tile_scan_run<false, LOCALW>(st, xi, yi, zi, li, mid, e, (real)0, (real)0, (real)0, addb, rn2, em);
                }
            }
        }
        em.flush();
        const int m = em.m;
        // single precision, long columns: padded to a multiple of P.sp_pad rows with self entries (md_sp.cu)
        if (!LOCALW && P.sp_pad > 1)
            for (int k = m; k < ((m + P.sp_pad - 1) / P.sp_pad) * P.sp_pad && k < P.Mmax; k++)
                P.W[(size_t)k * P.w_row + (size_t)i * P.w_col] = i;
        P.nnb[i] = m < P.Mmax ? m : P.Mmax;
        if (m > P.Mmax) set_err(P, MD_ERR_NEBR_OVERFLOW);
        tmax = max(tmax, m);
        tsum += m;
    }
    // statistics of the matrix (md_energy.max_neighbors / mean_neighbors) and of the search (md_info.candidates_per_atom)
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int wm = warp_max_i(tmax), ws = warp_sum_i(tsum), wc = warp_sum_i(tcand);
    if (lane == 0) { smx[wid] = wm; ssum[wid] = ws; scand[wid] = wc; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int mx = 0, sm = 0, sc = 0;
        for (int w = 0; w < BLOCK / 32; w++) { mx = max(mx, smx[w]); sm += ssum[w]; sc += scand[w]; }
        atomicMax(&P.ctrl->max_nnb, mx);
        atomicAdd(&P.ctrl->nnb_total, (unsigned long long)sm);
        atomicAdd(&P.ctrl->cand_total, (unsigned long long)sc);
    }
}

// ------------------------------------------------------------------------------------------------
// F1 on the tile.  Thread i walks column i of W (coalesced 32-bit words, two neighbors each, streamed from HBM
// two words ahead of their use); the partner positions come from the shared-memory tile.
// ------------------------------------------------------------------------------------------------
struct PairAccT {
    double fx, fy, fz, u, vir;
};

// One 32-bit word of W = two neighbors, evaluated together and branch-free so that their two dependent
// fp64 chains interleave.  The tile holds image positions (tile_stage<true>), so the flag bits are not needed.
// valid0 / valid1: the entry exists (n < m_i); an absent entry is index 0 of the tile, a harmless read.
template <bool ENERGY>
__device__ __forceinline__ void tile_pair2(const MdDev &P, const double *st, double xi, double yi, double zi, unsigned w,
                                           bool valid0, bool valid1, PairAccT &a)
{
    const double *p0 = st + 3 * (w & T_INDEX_MASK), *p1 = st + 3 * ((w >> 16) & T_INDEX_MASK);
    const double dx0 = xi - p0[0], dy0 = yi - p0[1], dz0 = zi - p0[2];
    const double dx1 = xi - p1[0], dy1 = yi - p1[1], dz1 = zi - p1[2];
    const double q0 = __fma_rn(dz0, dz0, __fma_rn(dy0, dy0, __dmul_rn(dx0, dx0)));
    const double q1 = __fma_rn(dz1, dz1, __fma_rn(dy1, dy1, __dmul_rn(dx1, dx1)));
    const bool in0 = valid0 && q0 < P.rc2, in1 = valid1 && q1 < P.rc2;
    if (!(in0 || in1)) return;
    if (ENERGY) {
        const double s0 = 1.0 / (in0 ? q0 : 1.0), s1 = 1.0 / (in1 ? q1 : 1.0);
        const double c0 = s0 * s0 * s0, c1 = s1 * s1 * s1;
        a.u += in0 ? 4.0 * c0 * (c0 - 1.0) - P.uc : 0.0;
        a.u += in1 ? 4.0 * c1 * (c1 - 1.0) - P.uc : 0.0;
        a.vir += in0 ? 48.0 * c0 * (c0 - 0.5) : 0.0;          // fc * r^2
        a.vir += in1 ? 48.0 * c1 * (c1 - 0.5) : 0.0;
    } else {
        const double s0 = fast_rcp(q0), s1 = fast_rcp(q1);     // q = 0 (an absent entry hitting the atom itself) gives inf / NaN, dropped by the select below
        const double c0 = s0 * s0 * s0, c1 = s1 * s1 * s1;
        const double f0 = in0 ? c0 * (c0 - 0.5) * s0 : 0.0, f1 = in1 ? c1 * (c1 - 0.5) * s1 : 0.0;   // x 48 applied to the sums
        a.fx += f0 * dx0; a.fy += f0 * dy0; a.fz += f0 * dz0;
        a.fx += f1 * dx1; a.fy += f1 * dy1; a.fz += f1 * dz1;
    }
}

// The first WPRE words (2 WPRE neighbors) of column i and its length, loaded BEFORE the position tile is staged
// so that their HBM latency overlaps the staging.
constexpr int WPRE = 4;
struct ColPre {
    int m;
    unsigned w[WPRE];
};

__device__ __forceinline__ ColPre tile_column_preload(const MdDev &P, int i)
{
    ColPre c;
    const unsigned *__restrict__ w = (const unsigned *)P.W + i;
    const int rows = P.Mmax >> 1;
    c.m = P.nnb[i];
#pragma unroll
    for (int k = 0; k < WPRE; k++) c.w[k] = k < rows ? __ldcs(w + (size_t)k * P.N_pad) : 0u;
    return c;
}

template <bool ENERGY>
__device__ __forceinline__ PairAccT tile_column(const MdDev &P, const double *st, double xi, double yi, double zi, int i,
                                                const ColPre &pre)
{
    const int m = pre.m;
    const unsigned *__restrict__ w = (const unsigned *)P.W + i;
    const size_t pitch = (size_t)P.N_pad;
    const int nw = (m + 1) >> 1;
    PairAccT a = {0.0, 0.0, 0.0, 0.0, 0.0};
    unsigned cur[WPRE];
#pragma unroll
    for (int k = 0; k < WPRE; k++) cur[k] = pre.w[k];
    for (int base = 0; base < nw; base += WPRE) {
        unsigned nxt[WPRE];
#pragma unroll
        for (int k = 0; k < WPRE; k++) nxt[k] = base + WPRE + k < nw ? __ldcs(w + (size_t)(base + WPRE + k) * pitch) : 0u;
#pragma unroll
        for (int k = 0; k < WPRE; k++) {
            const int n0 = 2 * (base + k);
            if (n0 < m) tile_pair2<ENERGY>(P, st, xi, yi, zi, cur[k], true, n0 + 1 < m, a);
        }
#pragma unroll
        for (int k = 0; k < WPRE; k++) cur[k] = nxt[k];
    }
    if (!ENERGY) { a.fx *= 48.0; a.fy *= 48.0; a.fz *= 48.0; }
    return a;
}

// one coalesced load of the box descriptor written by the build kernel
__device__ __forceinline__ void tile_load_desc(const MdDev &P, const TileBox &B, int bid, TileDesc &M)
{
    const int *__restrict__ d = P.tile_desc + (size_t)bid * TILE_DESC_INTS;
    const int n = TILE_DESC_HEAD + TILE_ROW_INTS * B.nq;
    for (int k = threadIdx.x; k < n; k += blockDim.x) ((int *)&M)[k] = __ldg(d + k);
    __syncthreads();
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
__global__ void __launch_bounds__(BLOCK, MD_TILE_FORCE_THREADS / BLOCK) k_tile_force(const __grid_constant__ MdDev P)
{
    extern __shared__ double dsm[];
    __shared__ TileDesc M;
    __shared__ double red[32];
    const int cap = P.tg.cap;
    double *st = dsm;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    const pos_t *__restrict__ pos = P.pos[pc];
    double *__restrict__ vel = P.vel[vc];
    const size_t np = (size_t)P.N_pad;
    const TileBox B = tile_box3(P.tg, P.nc, P.ncx, blockIdx.x, blockIdx.y, blockIdx.z);
    const int bid = tile_bid(P.tg);
    tile_load_desc(P, B, bid, M);
    const int n_own = M.T <= cap ? M.n_own : 0;          // an overflowing tile was reported by the build kernel
    int t = threadIdx.x, i = 0, li = 0;
    ColPre pre;
    double v0 = 0.0, v1 = 0.0, v2 = 0.0;
    if (t < n_own) {
        own_atom(M, t, i, li);
        pre = tile_column_preload(P, i);
        if (MODE != 0) { v0 = vel[i]; v1 = vel[np + i]; v2 = vel[2 * np + i]; }
    }
    if (n_own > 0) tile_stage<true>(M, pos, st, P.L);
    __syncthreads();
    double vm2 = 0.0;
    for (; t < n_own; t += BLOCK) {
        if (t != (int)threadIdx.x) {                      // boxes with more atoms than threads: rare
            own_atom(M, t, i, li);
            pre = tile_column_preload(P, i);
            if (MODE != 0) { v0 = vel[i]; v1 = vel[np + i]; v2 = vel[2 * np + i]; }
        }
        const double xi = st[3 * li], yi = st[3 * li + 1], zi = st[3 * li + 2];
        PairAccT a = tile_column<false>(P, st, xi, yi, zi, i, pre);
        double ub = 0.0;
        if (BONDS) tile_bonds<false>(P, pos, xi, yi, zi, i, a, ub);
        if (MODE == 0 || MODE == 2) {
            double *f = P.frc + i;
            f[0] = a.fx; f[np] = a.fy; f[2 * np] = a.fz;
        }
        if (MODE == 2) {
            vel[i] = v0 + P.hdt * a.fx; vel[np + i] = v1 + P.hdt * a.fy; vel[2 * np + i] = v2 + P.hdt * a.fz;
        }
        if (MODE == 1) {
            const double vx = v0 + P.dt * a.fx, vy = v1 + P.dt * a.fy, vz = v2 + P.dt * a.fz;
            vel[i] = vx; vel[np + i] = vy; vel[2 * np + i] = vz;
            const double x = xi + P.dt * vx, y = yi + P.dt * vy, z = zi + P.dt * vz;
            st_pos(P.pos[pc ^ 1] + i, x, y, z);
            double w2 = vx * vx + vy * vy + vz * vz;
            if (!isfinite(w2 + x + y + z)) { set_err(P, MD_ERR_NONFINITE); w2 = 0.0; }
            vm2 = fmax(vm2, w2);
        }
    }
    if (MODE == 1) {
        const double bm = block_max(vm2, red);
        if (threadIdx.x == 0) publish_vmax2(P, bid, bm);
    }
}

template <bool BONDS, int BLOCK>
__global__ void __launch_bounds__(BLOCK) k_tile_energy(const __grid_constant__ MdDev P)
{
    extern __shared__ double dsm[];
    __shared__ TileDesc M;
    __shared__ RedSmem S;
    const int cap = P.tg.cap;
    double *st = dsm;
    const int pc = __ldcg(&P.ctrl->p_dst), vc = __ldcg(&P.ctrl->v_dst);
    const pos_t *__restrict__ pos = P.pos[pc];
    const TileBox B = tile_box3(P.tg, P.nc, P.ncx, blockIdx.x, blockIdx.y, blockIdx.z);
    const int bid = tile_bid(P.tg);
    tile_load_desc(P, B, bid, M);
    const int n_own = M.T <= cap ? M.n_own : 0;
    if (n_own > 0) tile_stage<true>(M, pos, st, P.L);
    __syncthreads();
    double q[RED_N];
#pragma unroll
    for (int k = 0; k < RED_N; k++) q[k] = 0.0;
    for (int t = threadIdx.x; t < n_own; t += BLOCK) {
        int i, li;
        own_atom(M, t, i, li);
        const double xi = st[3 * li], yi = st[3 * li + 1], zi = st[3 * li + 2];
        const ColPre pre = tile_column_preload(P, i);
        PairAccT a = tile_column<true>(P, st, xi, yi, zi, i, pre);
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
    reduce_finish(P, q, S, bid, P.tg.nsx * P.tg.nsy * P.tg.nsz * P.tg.nsys);
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// launch wrappers
// ------------------------------------------------------------------------------------------------
size_t mdk_tile_smem(const MdDev &P, bool with_cells)
{
    size_t b = (size_t)P.tg.cap * (P.sp ? 3 * sizeof(float) : (with_cells ? TSTR64 : 3) * sizeof(double));
    // build kernel: + the tile index of the first atom of every tile cell
    if (with_cells) b += (size_t)TILE_Q_MAX * (P.tg.S + 2 * P.kx + 1) * sizeof(int);
    return b;
}

namespace {

inline dim3 tile_grid3(const MdDev &P) { return dim3(P.tg.nsx, P.tg.nsy, P.tg.nsz * P.tg.nsys); }

// The attribute belongs to the kernel, not to one md_system: opt in to the device maximum, so that systems with
// different tile capacities can coexist in a process.  `bytes` only checks that this system fits.
template <typename K>
int opt_in(K kernel, size_t bytes)
{
    int dev = 0, optin = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) return -1;
    optin -= 8192;                                   // room for the kernels' static shared memory (< 4 KB)
    if (optin < 0 || (size_t)optin < bytes) return -1;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, optin) == cudaSuccess ? 0 : -1;
}

template <int BLOCK>
int configure_block(const MdDev &P)
{
    const size_t sf = mdk_tile_smem(P, false);
    int rc = 0;
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
    const dim3 g = tile_grid3(P);
    const size_t sm = mdk_tile_smem(P, false);
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
    const size_t sb = mdk_tile_smem(P, true);
    if (opt_in(k_tile_build<PrecF64, true>, sb) || opt_in(k_tile_build<PrecF64, false>, sb) || opt_in(k_tile_build<PrecF32, false>, sb)) return -1;
    if (!P.tiled) return 0;                          // the force / energy kernels exist for 128, 256 and 512 threads
    switch (P.tg.threads) {
    case 128: return configure_block<128>(P);
    case 256: return configure_block<256>(P);
    case 512: return configure_block<512>(P);
    default: return -1;
    }
}

void mdk_tile_build(const MdDev &P, cudaStream_t st)
{
    const dim3 g = tile_grid3(P);
    const size_t sm = mdk_tile_smem(P, true);
    if (P.sp) k_tile_build<PrecF32, false><<<g, P.tg.threads, sm, st>>>(P);
    else if (P.tiled) k_tile_build<PrecF64, true><<<g, P.tg.threads, sm, st>>>(P);
    else k_tile_build<PrecF64, false><<<g, P.tg.threads, sm, st>>>(P);
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
    const dim3 g = tile_grid3(P);
    const size_t sm = mdk_tile_smem(P, false);
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
