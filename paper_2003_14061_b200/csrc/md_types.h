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
    int pad0;
    unsigned int ticket[6];    // "last block done" counters, one per kernel family
    unsigned long long vmax2_bits;
    unsigned long long nnb_total;
    long long step;
    double disp_acc;           // accumulated dt * max|v| since the last rebuild
    double red[RED_N];
};

enum { TK_INTEGRATE = 0, TK_ENERGY = 1, TK_FORCE = 2 };

// The unvarying parameter block.  The paper copies it to constant memory; here it is a
// __grid_constant__ kernel argument, which lives in the same constant bank without a separate copy.
struct MdDev {
    int N, N_pad, Mmax, nc, NC;
    int has_bonds, half_list, scan_blocks;
    double L, half_L, inv_w;            // inv_w = nc / L
    double rc2, rn2, uc;
    double dt, hdt, thresh;             // thresh = r_shell / 2
    double fene_k, fene_R02;
    pos_t *pos[2];
    double *vel[2];                     // SoA: vx = vel, vy = vel + N_pad, vz = vel + 2 N_pad
    double *frc;                        // SoA, same pitch
    int *id[2];                         // device slot -> original atom id
    int *cell_of, *slot, *cell_count, *cell_start, *perm, *block_sums;
    int *W, *nnb;                       // neighbor matrix W[m * N_pad + i], counts m_i
    int *inv, *bond_orig, *bond_dev;    // original id -> slot; bond partners by original id / by slot (2 x N_pad)
    double *partials;                   // RED_N x max_grid block partials
    double *scratch;                    // 6 N doubles, original-id order (get/set staging: xyz | vxyz)
    DevCtrl *ctrl;
};

// Launch wrappers (md_kernels.cu).  All are asynchronous on `st`.
struct MdLaunch {
    int block;          // threads per block of the per-atom kernels
    int grid_atoms;     // ceil(N / block)
};

void mdk_force_rebuild(const MdDev &P, cudaStream_t st);
void mdk_load_state(const MdDev &P, cudaStream_t st);                        // scratch(xyz | vxyz) -> pos/vel/id
void mdk_kick_drift(const MdDev &P, const MdLaunch &lc, cudaStream_t st);     // v += dt/2 f; r += dt v; wrap; decide
void mdk_kick(const MdDev &P, const MdLaunch &lc, cudaStream_t st);           // v += dt/2 f
void mdk_cells(const MdDev &P, const MdLaunch &lc, cudaStream_t st);          // bin + scan + place       (N1-N4)
void mdk_reorder(const MdDev &P, const MdLaunch &lc, cudaStream_t st);        // cell-order gather       (sec 2.4(4))
void mdk_build(const MdDev &P, const MdLaunch &lc, cudaStream_t st);          // neighbor matrix         (N5)
// mode 0: f only; 1: fused leapfrog step (f, kick dt, drift, decide); 2: f and closing half kick
void mdk_force(const MdDev &P, const MdLaunch &lc, int mode, cudaStream_t st);
void mdk_force_newton3(const MdDev &P, const MdLaunch &lc, cudaStream_t st);  // zero f + half-list atomics
void mdk_energy(const MdDev &P, const MdLaunch &lc, cudaStream_t st);         // all reductions -> ctrl->red
void mdk_export(const MdDev &P, int what, size_t offset, cudaStream_t st);    // 0 pos, 1 vel, 2 frc -> scratch + offset
int mdk_launches_of(int which);   // number of kernels each wrapper launches (for md_info.kernel_launches)
enum { LK_REBUILD_FORCE = 0, LK_LOAD, LK_KICK_DRIFT, LK_KICK, LK_CELLS, LK_REORDER, LK_BUILD, LK_FORCE, LK_FORCE_N3,
       LK_ENERGY, LK_EXPORT };
