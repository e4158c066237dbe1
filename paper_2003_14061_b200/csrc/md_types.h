// Internal types shared by the kernels (md_kernels.cu) and the C-ABI layer (md_api.cu).
// Not part of the public boundary (include/md_b200.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "md_b200.h"

// Position record: 32 bytes = one L2 sector per gather (the paper's float4 choice, in fp64).
struct __align__(32) pos_t {
    double x, y, z, w;
};

// Indices of the final reduction outputs in DevCtrl::red
enum { RED_KE = 0, RED_PE = 1, RED_PEB = 2, RED_VIR = 3, RED_PX = 4, RED_PY = 5, RED_PZ = 6, RED_VMAX2 = 7, RED_N = 8 };

// Device-resident control block.  Every decision that the paper's host loop takes (PAPER.md:64:
// "the maximal atom velocity needed to determine when the neighbor matrix needs rebuilding") is taken
// on the device by the last block of the integrating kernel and recorded here, so md_step(n) never
// synchronises with the host inside its loop.
struct DevCtrl {
    int p_src, p_dst;          // position ping-pong: a rebuild reads pos[p_src], writes pos[p_dst]; current = p_dst
    int v_src, v_dst;          // same for velocities and atom ids
    int need_rebuild;          // written every step by decide()
    int err;                   // first md_status error seen on the device (0 = none)
    int n_rebuilds;
    int max_nnb;               // max m_i of the current matrix
    int max_occ;               // max k_c of the last binning
    int do_reorder;            // MD_FLAG_LAYER_H: this rebuild re-sorts the atoms into cell order (else they stay in place)
    unsigned int ticket[6];    // "last block done" counters, one per kernel family
    int since_reorder;         // steps since the last sort
    int pad1;
    unsigned long long nnb_total;
    unsigned long long cand_total;   // candidates the last neighbor build tested (all atoms): md_info.candidates_per_atom
    long long step;
    double disp_acc;           // accumulated dt * max|v| since the last rebuild
    double red[RED_N];
};

enum { TK_INTEGRATE = 0, TK_ENERGY = 1, TK_FORCE = 2 };

// Shared-memory tile decomposition of the W layout MD_W_TILED.  The cells are cut into
// boxes of S x R x RZ cells (x fastest).  One thread block owns the atoms of one box -- R*RZ contiguous index
// ranges, because atoms are kept in cell order -- and stages the positions of the box plus one halo cell on
// every side (the 27-cell neighbourhoods of all its atoms) in shared memory: (R+2)(RZ+2) "tile
// rows", each the contiguous atoms of S+2 cells along x.  W then holds 16-bit entries: 13 bits of index
// into that tile + the 3 periodic-image flag bits of PAPER.md:163.
struct TileGeom {
    int S, R, RZ;            // cells per box along x (fine cells, see MdDev::kx), y, z
    int nsx, nsy, nsz;       // boxes per axis of ONE system
    int nsys;                // independent systems stacked along the grid's z axis (box index bz = sys * nsz + local)
    int cap;                 // tile capacity in atoms (<= 8192: 13 index bits)
    int threads;             // block size of the tile kernels
};

struct TileBox {
    int x0, sxc, y0, ny, z0, nz;   // first cell and number of cells of the box along each axis
    int nyq, nq;                   // tile rows per z plane (ny + 2) and in total
    int cell_base;                 // index of the first cell of the system the box belongs to (batched systems)
};

// nc: cells per edge along y, z; ncx: (fine) cells per edge along x
__host__ __device__ inline TileBox tile_box3(const TileGeom &G, int nc, int ncx, int bx, int by, int bzg)
{
    TileBox B;
    const int sys = bzg / G.nsz, bz = bzg - sys * G.nsz;
    B.cell_base = sys * ncx * nc * nc;
    B.x0 = bx * G.S;  B.sxc = ncx - B.x0 < G.S ? ncx - B.x0 : G.S;
    B.y0 = by * G.R;  B.ny = nc - B.y0 < G.R ? nc - B.y0 : G.R;
    B.z0 = bz * G.RZ; B.nz = nc - B.z0 < G.RZ ? nc - B.z0 : G.RZ;
    B.nyq = B.ny + 2;
    B.nq = B.nyq * (B.nz + 2);
    return B;
}

__host__ __device__ inline TileBox tile_box(const TileGeom &G, int nc, int ncx, int b)
{
    return tile_box3(G, nc, ncx, b % G.nsx, (b / G.nsx) % G.nsy, b / (G.nsx * G.nsy));
}

// Tile row q of a box: the row of cells (y0-1 + q % nyq, z0-1 + q / nyq), wrapped periodically.
// rowc = linear index of its x = 0 cell; ysh, zsh in {-1, 0, +1}: image shift of the row in units of L
// (added to r_i - r_j); xa, xc = x index of the FIRST of the kx halo cells before / after the box (wrapped at the
// faces: a box that starts at x = 0 sees the last kx cells of the row as its halo, shifted by one box edge).
// The box layout guarantees x0 >= kx for every box but the first and x0 + sxc + kx <= ncx for every box but the last,
// so each halo is ONE contiguous range of cells.
__host__ __device__ inline void tile_row(const TileBox &B, int nc, int ncx, int kx, int q, int &rowc, int &ysh, int &zsh, int &xa, int &xc)
{
    int y = B.y0 - 1 + q % B.nyq, z = B.z0 - 1 + q / B.nyq;
    ysh = 0; zsh = 0;
    if (y < 0) { y += nc; ysh = 1; } else if (y >= nc) { y -= nc; ysh = -1; }
    if (z < 0) { z += nc; zsh = 1; } else if (z >= nc) { z -= nc; zsh = -1; }
    rowc = B.cell_base + ncx * (y + nc * z);
    xa = B.x0 == 0 ? ncx - kx : B.x0 - kx;
    xc = B.x0 + B.sxc == ncx ? 0 : B.x0 + B.sxc;
}

constexpr int TILE_Q_MAX = 25;      // (R + 2)(RZ + 2) with R, RZ <= 3
constexpr int TILE_OWN_MAX = 9;     // R * RZ

// Tile descriptor of one box: written to global memory by the build kernel (the layout only changes when
// cell_start does, i.e. at a rebuild), read back with one coalesced load by every force / energy kernel.
struct TileDesc {
    int n_own, T, nq, pad;                              // atoms owned by the box, atoms in the tile, tile rows
    int own_base[TILE_OWN_MAX];                         // global index of the first own atom of own row k
    int own_loc[TILE_OWN_MAX];                          // its index in the tile
    int own_pre[TILE_OWN_MAX + 1];                      // exclusive prefix of the own-row lengths
    struct Row {
        int g[3], n[3];                                 // the (up to) 3 contiguous pieces of the row: start, length
        int off;                                        // tile index of the row's first atom
        int sh;                                         // periodic-image shifts in units of L, 2 bits each, biased by 1:
                                                        // bits 0-1 y, 2-3 z, 4-5 x of piece 0, 6-7 x of piece 2
    } row[TILE_Q_MAX];
};
constexpr int TILE_DESC_INTS = (int)(sizeof(TileDesc) / sizeof(int));
constexpr int TILE_DESC_HEAD = 4 + 2 * TILE_OWN_MAX + TILE_OWN_MAX + 1;     // ints before row[]
constexpr int TILE_ROW_INTS = 8;
#define T_INDEX_MASK 0x1fffu
#define T_FLAG_SHIFT 13

// The unvarying parameter block.  The paper copies it to constant memory; here it is a
// __grid_constant__ kernel argument, which lives in the same constant bank without a separate copy.
struct MdDev {
    int N, N_pad, Mmax, nc, NC;         // N, NC: atoms and cells of ALL systems; nc: cells per edge of one along y and z
    // Cells are anisotropic: at least r_n wide along y and z (3 x 3 rows of cells around an atom), but kx times finer
    // along x, the direction in which atoms are contiguous in memory: a row's candidates are then the atoms of the
    // 2 kx + 1 fine cells around the atom's own, a window ~(2 + 1/kx) r_n long instead of 3 cell widths, and shorter
    // still where the row's distance from the atom leaves less than r_n for x.  kx = 1: the paper's cubic cells.
    int kx, ncx;                        // fine cells per r_n-wide cell along x; cells per edge along x = kx * nc
    double inv_wx;                      // ncx / L
    float w_f, inv_wx_f, rn2_prune;     // cell width along y/z, ncx / L and r_n^2 in binary32, rounded to the safe side (row pruning)
    int n_sys, N1, NC1;                 // batched independent systems: count, atoms and cells of one
    int has_bonds, half_list, scan_blocks;
    int sm_count;                       // multiprocessors of the device (grid sizing of the grid-stride kernels)
    int tiled, tile_build, max_grid;    // W layout (1 = MD_W_TILED); shared-memory staged build kernel in use; row pitch of `partials`
    TileGeom tg;
    double L, half_L, inv_w;            // inv_w = nc / L
    double rc2, rn2, uc;
    double dt, hdt, thresh;             // thresh = r_shell / 2
    double fene_k, fene_R02;
    int has_angles;                     // bond-angle terms k/2 (cos(theta) - c0)^2 at atoms with two bonds (md_set_angles)
    double ang_k, ang_c0;
    int has_dihedrals;                  // dihedral terms k/2 (cos(phi) - c0)^2 for every four consecutive beads (md_set_dihedrals)
    double dih_k, dih_c0;
    pos_t *pos[2];
    double *vel[2];                     // SoA: vx = vel, vy = vel + N_pad, vz = vel + 2 N_pad
    double *frc;                        // SoA, same pitch
    int *id[2];                         // device slot -> original atom id
    int *cell_of, *slot, *cell_count, *cell_start, *perm, *block_sums;
    int *tile_desc;                     // tiled layout: TileDesc per box
    int w_row, w_col;                   // W[m * w_row + i * w_col]: (N_pad, 1) = atom-index-fastest; (1, Mmax) = transposed (ablation)
    int *W, *nnb;                       // neighbor matrix W[m * N_pad + i], counts m_i
                                        // (tiled layout: 32-bit words of two 16-bit entries, W[(m/2) * N_pad + i])
    int *inv, *bond_orig, *bond_dev;    // original id -> slot; bond partners by original id / by slot (2 x N_pad)
    double *blk_vmax2;                  // DEC_SLOTS maxima of v^2 from the drifting kernel (md_device.cuh: publish_vmax2; input of k_decide), then the
                                        // persistent kernels' 2 x grid per-block maxima
    double *partials;                   // RED_N x max_grid block partials
    double *scratch;                    // 6 N doubles, original-id order (get/set staging: xyz | vxyz)
    DevCtrl *ctrl;
    // ablation MD_FLAG_LAYER_H: the paper's dense cell x layer matrix H[c * n_layers + l] and its
    // every-100-steps sort
    int layer_H, n_layers, reorder_interval;
    int *H;
    // rigid molecules (md_rigid.cu; R20): molecule m = sites m rb_ns .. by original id
    int rigid, rb_ns, rb_nm, need_inv;  // need_inv: k_reorder keeps inv (original id -> slot) up to date (bonds or rigid molecules)
    double rb_body[24];                 // body-frame site positions (<= 8 sites), principal axes, centre of mass at the origin
    double rb_I[3], rb_M, rb_Imin, rb_bmax;
    double *rb_R, *rb_V, *rb_A, *rb_pi; // per molecule: centre of mass, its velocity, rotation matrix (row-major, body -> space), body-frame angular momentum
    double *rb_off;                     // per site (original id): multiple of L between the stored coordinate and R + A b_k
    // single-precision variant (md_sp.cu; MD_PREC_F32): float4 records r, v, f replace pos / vel / frc,
    // which stay null; L and inv_w above are then those of the binary32 box edge (double)(float)L
    int sp, sp_pad;                     // sp_pad = SP_PAD when the columns of W are padded with self entries (long columns), else 1
    float Lf, half_Lf, rc2f, rn2f, ucf, dtf, hdtf, fene_kf, fene_R02f;
    float4 *posf[2], *velf[2], *frcf;
};

// Launch wrappers (md_kernels.cu).  All are asynchronous on `st`.
struct MdLaunch {
    int block;          // threads per block of the per-atom kernels
    int grid_atoms;     // ceil(N / block)
};

void mdk_force_rebuild(const MdDev &P, cudaStream_t st);
void mdk_check_range(const MdDev &P, double box, cudaStream_t st);           // scratch xyz in [0, box] else ctrl->err = MD_ERR_INVALID
void mdk_load_state(const MdDev &P, cudaStream_t st);                        // scratch(xyz | vxyz) -> pos/vel/id
// rebuild decision from blk_vmax2[0..nblk); cond != 0: also set that CUDA-graph conditional handle to need_rebuild
void mdk_decide(const MdDev &P, bool pos_pingpong, cudaStream_t st, unsigned long long cond);
void mdk_kick_drift(const MdDev &P, const MdLaunch &lc, cudaStream_t st);     // v += dt/2 f; r += dt v; per-block max v^2
void mdk_kick(const MdDev &P, const MdLaunch &lc, cudaStream_t st);           // v += dt/2 f
void mdk_cells(const MdDev &P, const MdLaunch &lc, cudaStream_t st);          // bin + scan + place       (N1-N4)
void mdk_reorder(const MdDev &P, const MdLaunch &lc, cudaStream_t st);        // cell-order gather       (sec 2.4(4))
void mdk_build(const MdDev &P, const MdLaunch &lc, cudaStream_t st);          // neighbor matrix         (N5)
// mode 0: f only; 1: fused leapfrog step (f, kick dt, drift, per-block max v^2; follow with mdk_decide); 2: f and closing half kick
void mdk_force(const MdDev &P, const MdLaunch &lc, int mode, cudaStream_t st);
void mdk_force_newton3(const MdDev &P, const MdLaunch &lc, cudaStream_t st);  // zero f + half-list atomics
void mdk_energy(const MdDev &P, const MdLaunch &lc, cudaStream_t st);         // all reductions -> ctrl->red
void mdk_export(const MdDev &P, int what, double *dst, cudaStream_t st);
void mdk_publish_ctrl(const MdDev &P, DevCtrl *host_mapped, cudaStream_t st);
void mdk_set_error(const char *msg);     // md_last_error() text, for the translation units beside md_api.cu
int mdk_sp_persist_choice(const MdDev &P, const void **kernel);     // grid of the binary32 persistent kernel (0: not possible)       // 0 pos, 1 vel, 2 frc -> dst (device, 3N doubles, original-id order)
// tiled layout (md_tile.cu)
int mdk_tile_configure(const MdDev &P);                                       // opt in to the dynamic shared memory; 0 = ok
size_t mdk_tile_smem(const MdDev &P, bool with_cells);
void mdk_tile_build(const MdDev &P, cudaStream_t st);
void mdk_tile_force(const MdDev &P, int mode, cudaStream_t st);
void mdk_tile_energy(const MdDev &P, cudaStream_t st);
// single-precision variant (md_sp.cu); the wrappers above dispatch to these when P.sp
void mdk_sp_load_state(const MdDev &P, cudaStream_t st);
void mdk_sp_export(const MdDev &P, int what, double *dst, cudaStream_t st);
void mdk_sp_kick_drift(const MdDev &P, cudaStream_t st);
void mdk_sp_kick(const MdDev &P, cudaStream_t st);
void mdk_sp_bin(const MdDev &P, cudaStream_t st);
void mdk_sp_reorder(const MdDev &P, cudaStream_t st);
void mdk_sp_build(const MdDev &P, cudaStream_t st);
void mdk_sp_force(const MdDev &P, const MdLaunch &lc, int mode, cudaStream_t st);
void mdk_sp_energy(const MdDev &P, cudaStream_t st);
// push-off of an overlapping chain start (md_pushoff.cu; initialisation, not the hot path)
void mdk_po_kick_drift(const MdDev &P, double rcap2, double vlim2, double ke_target, int first, cudaStream_t st);
void mdk_po_force(const MdDev &P, double rcap2, cudaStream_t st);
void mdk_po_kick(const MdDev &P, cudaStream_t st);                             // + kinetic energy -> ctrl->red[RED_KE]
void mdk_po_check(const MdDev &P, unsigned long long *out, cudaStream_t st);  // out[0] min non-bonded r^2, out[1] max bond r^2 (bit patterns)
// small systems: all n steps of md_step in one cooperative launch (md_kernels.cu: k_persist); 0 = launched
bool mdk_persist_ok(const MdDev &P);
int mdk_persist_steps(const MdDev &P, long long n, cudaStream_t st);
// rigid molecules (md_rigid.cu)
void mdk_rigid_kick_drift(const MdDev &P, cudaStream_t st);
void mdk_rigid_kick(const MdDev &P, cudaStream_t st);
void mdk_rigid_offsets(const MdDev &P, cudaStream_t st);
// measured arithmetic ceilings (md_peaks.cu); scratch >= 8 * sms doubles
double mdk_peak_fp64(cudaStream_t st, int sms, double *scratch);
double mdk_peak_fp32(cudaStream_t st, int sms, double *scratch);
int mdk_launches_of(int which);   // number of kernels each wrapper launches (for md_info.kernel_launches)
enum { LK_REBUILD_FORCE = 0, LK_LOAD, LK_KICK_DRIFT, LK_KICK, LK_CELLS, LK_REORDER, LK_BUILD, LK_FORCE, LK_FORCE_N3,
       LK_ENERGY, LK_EXPORT };
