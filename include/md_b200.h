/*
 * md_b200.h -- C ABI of the B200 (sm_100a) short-range molecular-dynamics hot path.
 *
 * The library implements, in hand-written CUDA, the per-time-step path of
 * D. C. Rapaport, "GPU molecular dynamics: Algorithms and performance" (arXiv 2003.14061):
 *   cell assignment and occupancy counting          (steps N1-N2)
 *   cell ordering of the atoms by prefix scan        (N3-N4 and the reorder of sec. 2.4(4))
 *   neighbor-matrix construction W[m][i]             (N5; layout PAPER.md:68)
 *   pair forces over W without / with Newton's 3rd   (F1)
 *   leapfrog integration with periodic wrap          (Table 2 "integration")
 *   energy / virial / momentum / max-velocity sums   (F2 and the reductions of PAPER.md:58, 64-66)
 *   displacement-triggered rebuild of W
 *   optional FENE bond lists for polymer chains
 * The paper prints no equations; the model (truncated, energy-shifted Lennard-Jones; two-half-kick
 * leapfrog; rebuild when the accumulated dt*max|v| exceeds r_shell/2) is fixed in DESIGN.md, "Readings".
 *
 * Conventions
 *   - Reduced units (sigma = epsilon = m = 1).  Cubic periodic box [0, L)^3.  All arithmetic is fp64 unless
 *     md_params.precision = MD_PREC_F32 selects the single-precision variant.
 *   - Every array argument is a HOST pointer owned by the caller unless its name ends in `_device`.
 *     Page-locked (cudaHostAlloc / cudaHostRegister) arrays are copied to and from directly on the stream;
 *     pageable ones go through a pinned staging buffer inside the library.
 *     Layout of per-atom vectors at the boundary: xyz[3*i + k], i = ORIGINAL atom id (the device keeps
 *     atoms in cell order and re-sorts them at every rebuild; that is invisible here).
 *   - No C++ exceptions cross the boundary.  Functions returning int give MD_OK (0) or a negative
 *     md_status; md_last_error() returns a thread-local description of the last failure.
 *   - The library runs on the CUDA stream given in md_params.stream (0 = a stream it creates) and
 *     allocates device memory through the hooks given to md_set_allocator (default cudaMalloc/cudaFree).
 *   - There is no CPU fallback: without a CUDA device every call that needs one fails with MD_ERR_CUDA.
 */
#ifndef MD_B200_H
#define MD_B200_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define MD_API __attribute__((visibility("default")))
#else
#define MD_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct md_system md_system;

typedef enum md_status {
    MD_OK = 0,
    MD_ERR_INVALID = -1,        /* bad argument or call order */
    MD_ERR_NEBR_OVERFLOW = -2,  /* some atom has more than Mmax neighbors (never truncated silently) */
    MD_ERR_BOND_BROKEN = -3,    /* a FENE bond reached r >= R0 */
    MD_ERR_NONFINITE = -4,      /* NaN/Inf in the state */
    MD_ERR_CUDA = -5,           /* CUDA runtime error (text in md_last_error) */
    MD_ERR_UNSUPPORTED = -6,    /* e.g. fewer than 3 cells per edge, more than 2 bonds per atom */
    MD_ERR_NOMEM = -7,
    MD_ERR_TILE_OVERFLOW = -8,  /* tiled W: a block's cell neighbourhood holds more atoms than its shared-memory
                                   tile (strongly inhomogeneous density); re-create with MD_FLAG_GLOBAL_W */
    MD_ERR_CELL_OVERFLOW = -9   /* MD_FLAG_LAYER_H only: a cell holds more atoms than the layer count N_l of the dense
                                   cell x layer matrix H (the CSR default has no such bound) */
} md_status;

enum { MD_LATTICE_AUTO = 0, MD_LATTICE_SC = 1, MD_LATTICE_FCC = 2, MD_LATTICE_NONE = 3 };
/* force_variant: the trade-off of PAPER.md:68 */
enum { MD_FORCE_FULL_LIST = 0,      /* A: one thread per atom, every pair twice, no Newton-3, no atomics */
       MD_FORCE_NEWTON3_ATOMICS = 1 /* B: half list, f_j updated with fp64 atomics */ };
/* step_mode: how one time step is mapped to kernels */
enum { MD_STEP_FUSED = 0,           /* force + kick + drift in one kernel (leapfrog form), variant A only */
       MD_STEP_SPLIT = 1            /* the paper's structure: integrate / force / integrate as separate kernels */ };

/* Parameters of md_create_ex.  Fill with md_params_default() first.  The library copies it. */
typedef struct md_params {
    int64_t  n_atoms;
    double   box;            /* L; if <= 0 it is (n_atoms/density)^(1/3) */
    double   density;        /* used when box <= 0; if both are given they must agree to 1e-12 relative */
    double   r_cut;          /* r_c: pair cutoff (2^(1/6) gives the soft-sphere / WCA system) */
    double   r_shell;        /* delta: neighbor shell thickness */
    double   dt;
    uint64_t seed;           /* seed of the counter-based velocity generator */
    double   temperature;    /* initial velocities: Gaussian, zero net momentum, sum v^2 = 3(N-1)T */
    int32_t  lattice;        /* MD_LATTICE_*; NONE: call md_set_state before stepping */
    int32_t  force_variant;  /* MD_FORCE_* */
    int32_t  step_mode;      /* MD_STEP_* (NEWTON3 forces imply SPLIT) */
    int32_t  max_neighbors;  /* Mmax, rows of W; 0 = auto: multiple of 16 >= 1.35*(4/3)pi r_n^3 rho + 12 */
    int32_t  block_size;     /* threads per block of the per-atom kernels; 0 = default */
    int32_t  device;         /* CUDA device ordinal; -1 = current */
    void    *stream;         /* cudaStream_t to run on; NULL = the library creates its own */
    uint32_t flags;          /* MD_FLAG_* */
    int32_t  n_systems;      /* batch of independent, mutually invisible systems run by the same kernel launches
                                ("many separate simulations within a single run" to fill the GPU with
                                small systems); 0 or 1 = one.  n_atoms, box, density are PER SYSTEM; every per-atom
                                array at this boundary then has n_systems * n_atoms rows, system-major, and atom ids
                                (bond lists, md_get_neighbors) are global: id = system * n_atoms + i.  System b starts
                                from the same lattice with velocity seed + b.  One rebuild decision (the largest
                                velocity of any system) serves all; md_energies returns sums over all systems. */
    int32_t  precision;      /* MD_PREC_F64 (default) or MD_PREC_F32: the paper's own precision with
                                its float4 state arrays: coordinates, velocities, forces and the pair
                                arithmetic in binary32, every sum of energies in binary64.  Boundary arrays stay double and
                                are rounded to binary32 on entry; the box edge used is (float)box.  Variant A only
                                (fused or split steps), global-index W. */
    int32_t  reorder_interval; /* MD_FLAG_LAYER_H only.  > 0: the atoms are re-sorted into cell order at the first rebuild
                                that falls at least this many steps after the last sort (the paper: 100);
                                0: at every rebuild; < 0: never (not even at the start).  Ignored without the flag: the
                                default path sorts at every rebuild. */
    int32_t  cell_split_x;   /* cells are >= r_n wide along y and z and this many times finer along x, the direction atoms
                                are contiguous in after the cell-order sort, which shortens the candidate runs of the
                                neighbor build; 1 = the paper's cubic cells; 0 = auto (2; 1 with
                                MD_FLAG_LAYER_H).  1 .. 8. */
    int32_t  tile_cells[3];  /* shared-memory staged kernels: r_n-wide cells per thread block along x, y, z (y, z: 1..3); 0 = auto */
    int32_t  tile_threads;   /* their block size (multiple of 32 in [64, 512]; tiled W: 128, 256 or 512); 0 = auto */
    int32_t  tile_capacity;  /* atoms the shared-memory tile holds (<= 8192); 0 = auto (1.35 x mean + 6 sigma) */
} md_params;

enum { MD_PREC_F64 = 0, MD_PREC_F32 = 1 };

enum { MD_FLAG_NO_GRAPH = 1u, /* launch kernels one by one instead of replaying a captured CUDA graph */
       MD_FLAG_GLOBAL_W = 2u, /* the paper's literal data path: W holds global atom indices and BOTH
                                 the neighbor build and the force kernel gather partner positions through L1/L2.
                                 Without this flag the build kernel stages the cell neighbourhood of each thread
                                 block in shared memory; W is the same. */
       MD_FLAG_TILED_W = 4u,  /* W holds 16-bit indices into the per-block shared-memory tile, and the force / energy
                                 kernels stage that tile too.  Variant A only.  Without any of
                                 these flags the library picks this layout when the expected number of neighbors per
                                 atom is >= 32 (e.g. LJ with r_c = 2.5) and global indices otherwise. */
       MD_FLAG_GATHER_W = 8u, /* never pick the tiled layout automatically (the build kernel still stages tiles) */
       MD_FLAG_W_TRANSPOSED = 16u, /* ablation of PAPER.md:165-167: store W atom-index-SLOWEST, W[i * Mmax + m], so that
                                 the threads of a warp no longer read consecutive words (global-index layout only) */
       MD_FLAG_NO_PERSIST = 64u, /* Systems of <= 400,000 atoms (either precision, fused steps, no flag and no tile setting given) run
                                 md_step as ONE cooperative launch whose blocks stay resident over all n steps and meet at
                                 grid-wide barriers (md_info.use_graph = 2), with W built by the gathering
                                 kernel (one atom per thread up to ~75,000 atoms, several beyond).  This flag -- like any other
                                 flag or tile setting -- keeps the step graph that larger systems use. */
       MD_FLAG_LAYER_H = 32u  /* ablation: the paper's own cell structure (steps N1-N5): a dense cell x
                                 layer matrix H[c][l] = atom, filled from the atomic slot l_i, searched by the neighbor
                                 build; atoms are re-sorted into cell order only every md_params.reorder_interval steps
                                  and otherwise stay where they are.  Implies MD_FLAG_GLOBAL_W.  fp64,
                                 variant A only.  A cell holding more than N_l atoms gives MD_ERR_CELL_OVERFLOW. */ };
enum { MD_W_GLOBAL = 0, MD_W_TILED = 1 };

/* Totals (not per atom) at the current, synchronised time: r, v and f belong to the same instant. */
typedef struct md_energy {
    double  ke;                 /* 1/2 sum |v|^2 */
    double  pe_pair;            /* 1/2 sum_i u_i  (u_i counts each pair twice: "actually 2U") */
    double  pe_bond;            /* FENE energy */
    double  virial;             /* sum over pairs of f_ij . r_ij (pair + bond) */
    double  px, py, pz;         /* total momentum */
    double  vmax;               /* max |v| */
    int64_t step;               /* steps taken since creation / md_set_state */
    int64_t n_rebuilds;         /* neighbor-matrix rebuilds since then (initial build not counted) */
    int32_t max_neighbors;      /* max_i m_i of the current matrix */
    int32_t max_cell_occupancy; /* max_c k_c of the last binning (the paper's layer count N_l) */
    double  mean_neighbors;     /* mean m_i of the current matrix, FULL-list convention for both variants */
} md_energy;

typedef struct md_info {
    int64_t n_atoms, n_pad;     /* n_atoms PER SYSTEM; n_pad: row pitch of W (all atoms, rounded up to 128) */
    double  box, r_neighbor, cell_width;
    int32_t cells_per_edge, max_neighbors, block_size, force_variant, step_mode, n_bonds_per_atom_max;
    int64_t device_bytes;       /* device memory held by this system */
    int64_t kernel_launches;    /* kernels launched by this system since creation */
    char    device_name[64];
    int32_t w_layout;           /* MD_W_GLOBAL / MD_W_TILED */
    int32_t tile_cells[3];      /* tiled: cells per thread block along x, y, z */
    int32_t tile_capacity;      /* tiled: atoms the shared-memory tile can hold */
    int32_t tile_threads;       /* tiled: threads per block of the build / force kernels */
    int32_t use_graph;          /* 1 when md_step replays a CUDA graph with a conditional rebuild node; 2 when it runs all its
                                   steps in one cooperative launch (small systems) */
    int32_t n_systems;
    int32_t precision;          /* MD_PREC_* */
    int32_t n_layers;           /* MD_FLAG_LAYER_H: N_l, columns of H; else 0 */
    int32_t cells_x;            /* cells per edge along x (the direction atoms are contiguous in): cell_split_x * cells_per_edge */
    int32_t cell_split_x;       /* fine cells per r_n-wide cell along x; the build scans up to +-cell_split_x of them per row */
    int32_t sm_count;
    double  candidates_per_atom;/* mean number of candidates the neighbor build tests per atom with this cell geometry (upper bound) */
} md_info;

/* Kernel classes of md_get_timers, after Table 2 of the paper. */
enum { MD_T_INTEGRATE = 0, MD_T_CELLS = 1, MD_T_REORDER = 2, MD_T_NEBR = 3, MD_T_FORCE = 4, MD_T_ENERGY = 5,
       MD_T_FUSED_STEP = 6, MD_T_DECIDE = 7, MD_T_COUNT = 8 };

MD_API void md_params_default(md_params *p);

/* PAPER.md:107 states the problem as: N atoms on a cubic grid, density, cutoff, shell, time step, random
 * velocities.  Lattice: SC when N is a perfect cube, else FCC when N/4 is; T = 1; variant A, fused steps.
 * Returns NULL on failure.  On return the neighbor matrix, forces and energies at t = 0 are valid. */
MD_API md_system *md_create(int64_t n_atoms, double box, double density, double r_cut, double r_shell, double dt,
                     uint64_t seed);
MD_API md_system *md_create_ex(const md_params *p);
MD_API void md_destroy(md_system *s);

/* Optional bond list for the chain workload: n_bonds pairs ij[2*b], ij[2*b+1] of ORIGINAL
 * atom ids, FENE force -k r / (1 - r^2/R0^2) on top of the pair force (which also acts on bonded pairs).
 * At most 2 bonds per atom (linear chains).  Only before the first md_step after create / md_set_state.
 * Forces and energies are re-evaluated. */
MD_API int md_set_bonds(md_system *s, int64_t n_bonds, const int32_t *ij, double k, double R0);

/* Chain start "grown as seeded random walks then pushed apart" (BASELINE.json configs[4]; R12).
 * INITIALISATION, not part of the time-step path: xyz (host, 3*N, original-id order, in [0, L]) is an OVERLAPPING start,
 * e.g. random walks; the library runs its own MD kernels on it with the pair force capped (for r < r_cap the force keeps
 * the magnitude it has at r_cap), r_cap ramped from r_cap_start to r_cap_end over ramp_steps, the FENE force clamped
 * short of its pole, no atom moving more than max_move per step, and the velocities rescaled to `temperature` every
 * step, until the smallest distance between atoms that are not bonded exceeds min_nonbonded and the longest bond is
 * below max_bond (checked every check_interval steps once the ramp is over).  Then it loads the pushed-off positions,
 * fresh velocities (the generator of md_create with `seed`: Gaussian, zero net momentum, sum v^2 = 3(N-1)T) and the bond
 * list into `s` exactly as md_set_state + md_set_bonds would.  The work runs in a temporary system of its own (global-index
 * W with room for the crowded start), so `s` may have any layout or precision.  Zero fields of opts take the defaults
 * given below; opts may be NULL.  MD_ERR_UNSUPPORTED if the criteria are not met within max_steps. */
typedef struct md_pushoff_opts {
    double   r_cap_start, r_cap_end;   /* 1.0, 0.8 */
    int32_t  ramp_steps;               /* 3000 */
    int32_t  max_steps;                /* 40000 */
    int32_t  check_interval;           /* 100 */
    double   min_nonbonded, max_bond;  /* 0.85, 1.3 */
    double   max_move;                 /* 0.05 */
    double   temperature;              /* 1.0 */
    uint64_t seed;                     /* fresh velocities after the push-off; the push-off itself starts from seed + 1 */
} md_pushoff_opts;
typedef struct md_pushoff_report {
    int64_t steps;                     /* push-off steps run */
    double  min_nonbonded, max_bond;   /* of the state loaded into s */
    double  min_nonbonded_start;       /* of the overlapping start */
} md_pushoff_report;
MD_API int md_pushoff(md_system *s, const double *xyz, int64_t n_bonds, const int32_t *ij, double k, double R0,
                      const md_pushoff_opts *opts, md_pushoff_report *report);

/* Rigid molecules (sec. 4.3(1): "rigid bodies with multiple interaction sites ... e.g., four SP spheres
 * in a rigid tetrahedral configuration ... rotation matrices ... a generalization of the symplectic leapfrog"; the paper
 * gives no equations: DESIGN.md R20 states the textbook forms used).  The n_atoms atoms of the system become the
 * interaction SITES of n_atoms / n_sites molecules: molecule m owns the atoms m*n_sites .. m*n_sites + n_sites - 1 (original
 * ids), unit mass each, at the fixed body-frame positions body_xyz[3*k .. 3*k+2] (host; centre of mass at the origin,
 * axes = principal axes, all three moments > 0, else MD_ERR_INVALID).  Sites of different molecules interact through the
 * system's pair potential; sites of one molecule do not.  After this call load a state with md_set_rigid_state; md_step
 * then integrates the molecules (half kick of V and of the body-frame angular momentum, free rotation of the rotation matrix
 * by the splitting Rx Ry Rz Ry Rx, drift, rebuild decision from a bound on the largest site speed, site forces, half kick).
 * md_energies: ke = translational + rotational kinetic energy, vmax = the largest site speed; md_get_positions /
 * _velocities / _forces return the sites.  fp64, full-list forces, global-index W, one system, no bond terms
 * (MD_ERR_UNSUPPORTED otherwise). */
MD_API int md_set_rigid(md_system *s, int32_t n_sites, const double *body_xyz);
/* Molecule state, all host arrays in molecule order: com[3*m], rot[9*m] (row-major rotation matrix A, body -> space: site k
 * of molecule m sits at com + A b_k), vcom[3*m], angmom_body[3*m] (angular momentum in the body frame).  Setting a state
 * bins the sites, builds W and evaluates the forces, like md_set_state. */
MD_API int md_set_rigid_state(md_system *s, const double *com, const double *rot, const double *vcom, const double *angmom_body);
MD_API int md_get_rigid_state(md_system *s, double *com, double *rot, double *vcom, double *angmom_body);

/* Optional bond-angle terms for the chain workload ("bond force, bond-angle torque"; the paper gives
 * no form: the textbook cosine-harmonic U = k_theta/2 (cos(theta) - cos_theta0)^2 is used, R19) at every
 * atom that has two bonded partners, theta the angle between its two bonds.  Call after md_set_bonds and before the
 * first md_step.  Forces and energies are re-evaluated; md_energy.pe_bond then holds FENE + angle energy (the terms
 * have no virial).  Global-index W layouts only, either precision (MD_ERR_UNSUPPORTED with MD_FLAG_TILED_W). */
MD_API int md_set_angles(md_system *s, double k_theta, double cos_theta0);

/* Optional dihedral terms ("optional dihedral"; R19): U = k_phi/2 (cos(phi) - cos_phi0)^2 for
 * every four consecutive bonded atoms a-b-c-d, phi the angle between the planes (a,b,c) and (b,c,d) (cos(phi) = -1 for a
 * planar zig-zag).  Same call order, reporting and restrictions as md_set_angles. */
MD_API int md_set_dihedrals(md_system *s, double k_phi, double cos_phi0);

/* Advance n time steps.  Asynchronous on the stream except for one status read at the end.
 * After an error other than MD_ERR_INVALID the state is undefined; only md_destroy is valid. */
MD_API int md_step(md_system *s, int64_t n);

/* Energy / virial / momentum / max-velocity reductions of the current state.  Synchronises. */
MD_API int md_energies(md_system *s, md_energy *out);

/* xyz: host, 3*N doubles, original-id order.  Positions are wrapped into [0, L).  Synchronise. */
MD_API int md_get_positions(md_system *s, double *xyz);
MD_API int md_get_velocities(md_system *s, double *xyz);
MD_API int md_get_forces(md_system *s, double *xyz);

/* Positions and velocities in one call (one synchronisation; a single device-to-host transfer when vxyz == xyz + 3*N
 * and the array is page-locked). */
MD_API int md_get_state(md_system *s, double *xyz, double *vxyz);

/* Zero-copy read-out: the same arrays (3*N doubles, original-id order, positions wrapped into [0, L)) written by one
 * kernel into a caller-owned DEVICE buffer, e.g. the data_ptr() of a torch tensor on the system's device.  Enqueued on
 * the system's stream and NOT synchronised: order later work after that stream.  MD_ERR_INVALID for a host pointer. */
MD_API int md_get_positions_device(md_system *s, double *xyz_device);
MD_API int md_get_velocities_device(md_system *s, double *xyz_device);
MD_API int md_get_forces_device(md_system *s, double *xyz_device);

/* Replace positions and velocities (host, 3*N each, original-id order; vxyz may be NULL = keep).
 * Positions must lie in [0, L].  Re-bins, rebuilds W, re-evaluates forces, resets step and rebuild
 * counters and the displacement accumulator; bonds are kept. */
MD_API int md_set_state(md_system *s, const double *xyz, const double *vxyz);
/* The same from DEVICE arrays (e.g. torch tensors on the system's device): no host transfer.  vxyz_device may be NULL. */
MD_API int md_set_state_device(md_system *s, const double *xyz_device, const double *vxyz_device);

/* Pipelined host I/O (SURVEY.md 8(b) extension): the two directions of the host link run on the
 * library's own copy streams, concurrently with each other and with the kernels on the system's stream, so that a
 * service loop over independent host-resident states pays max(upload, download, compute) per state, not their sum.
 * All host arrays of these calls must be PAGE-LOCKED (cudaHostAlloc / cudaHostRegister / torch pin_memory), 3*N doubles
 * each, original-id order, and must stay valid and untouched until the transfer is known to be complete;
 * MD_ERR_INVALID for pageable memory.  Not for rigid-molecule systems.  The first call allocates four staging buffers
 * of 6*N doubles on the device (through the system's allocator hooks).
 *   md_stage_state      starts the upload of a NEXT state (positions and velocities) into a device staging buffer and
 *                       returns at once; the system's current state and its kernels are not affected.  Up to TWO states
 *                       can be staged (a FIFO; MD_ERR_INVALID for a third), so that the next upload runs while the
 *                       previous one is being installed.
 *   md_commit_state     makes the OLDEST staged state the system's state, exactly as md_set_state would (range check on
 *                       the device before the old state is touched, re-bin, rebuild W, forces, counters reset).  Waits
 *                       for that upload; after it returns the host arrays of that upload may be reused.  A state that
 *                       fails the range check is dropped from the FIFO.  MD_ERR_INVALID if nothing is staged.
 *   md_get_state_async  exports positions and velocities of the CURRENT state (stream-ordered after the kernels enqueued so
 *                       far) and starts their download; returns at once.  Downloads complete in the order they were
 *                       started; two can be in flight before a third makes the system's stream wait for the first.
 *   md_wait_io          max_pending = 0: blocks until every transfer started by the calls above is complete.
 *                       max_pending = 1 .. 3: blocks until at most that many of the NEWEST downloads are still in flight
 *                       (1: everything but the download started last is complete).  Returns MD_ERR_CUDA if a transfer
 *                       failed.  md_destroy waits for everything. */
MD_API int md_stage_state(md_system *s, const double *xyz, const double *vxyz);
MD_API int md_commit_state(md_system *s);
MD_API int md_get_state_async(md_system *s, double *xyz, double *vxyz);
MD_API int md_wait_io(md_system *s, int32_t max_pending);

/* Test hooks.  md_rebuild_neighbors forces a rebuild now.  md_get_neighbors returns the matrix by ORIGINAL
 * ids: counts[N]; list[N * max_neighbors] with row i = neighbors of atom i (unordered, -1 padded); for the
 * Newton-3 variant the half list is symmetrised so both variants return the full relation.
 * list may be NULL (counts only). */
MD_API int md_rebuild_neighbors(md_system *s);
MD_API int md_get_neighbors(md_system *s, int32_t *counts, int32_t *list, int32_t *max_neighbors_out);

MD_API int md_get_info(md_system *s, md_info *out);

/* Per-kernel-class device timers (CUDA events on the library's stream around every launch while enabled).
 * ms[MD_T_COUNT], launches[MD_T_COUNT] accumulate since the last md_reset_timers.  Synchronises. */
MD_API int md_set_profiling(md_system *s, int enabled);
MD_API int md_get_timers(md_system *s, double *ms, int64_t *launches);
MD_API int md_reset_timers(md_system *s);

/* Arithmetic ceilings of the device, MEASURED with register-resident FMA loops (CUDA events on the system's stream):
 * the denominators for kernels bound by the fp64 pipe / instruction issue rather than HBM.  Not on the time-step path. */
typedef struct md_peaks {
    double  fp64_tflops;        /* DFMA loop, 2 flops per instruction */
    double  fp32_tflops;        /* FFMA loop */
    int32_t sm_count;
    int32_t sm_clock_khz;       /* cudaDevAttrClockRate */
} md_peaks;
MD_API int md_measure_peaks(md_system *s, md_peaks *out);

/* Device-memory hooks for the systems created AFTER the call (each system records the pair in force at its creation
 * and frees through it, so systems created under different hooks can coexist).  alloc(bytes, stream, user) returns a
 * device pointer or NULL; free_(ptr, user).  NULL, NULL = cudaMalloc / cudaFree.  The Python binding routes these to
 * torch's caching allocator. */
typedef void *(*md_alloc_fn)(size_t bytes, void *stream, void *user);
typedef void (*md_free_fn)(void *ptr, void *user);
MD_API void md_set_allocator(md_alloc_fn alloc, md_free_fn free_, void *user);

/* Allocation-free reduction for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid it): the velocity part of the sums of md_energies -- kinetic energy, total
 * momentum and the largest speed, the input of the rebuild rule -- of ANY device array of velocities, without an
 * md_system.  vxyz_device: 3*n_atoms doubles, v[3*i + k] (what md_get_velocities_device writes).  out5_device: 5 doubles
 * on the device: ke = sum 1/2 |v|^2, px, py, pz, vmax.  stream: cudaStream_t (NULL = the default stream).  Both arrays must
 * be device memory of the CURRENT device.  The call enqueues one 256-byte memset and one kernel on the stream and returns;
 * it does not synchronise and calls no cudaMalloc / cudaFree or allocating routine: the block partials and the "last block
 * done" ticket live in a static device array inside the library (0.64 MB, held by every GPU that loads the library until
 * the process exits), which is why n_atoms is limited: MD_ERR_INVALID above MD_NOALLOC_MAX_ATOMS (or for a host pointer,
 * n_atoms < 1).  ALL calls share that array: calls that overlap on the GPU (two streams, two host threads) race -- serialise
 * them.  Results are reproducible (fixed summation order) and agree with md_energies to summation rounding. */
#define MD_NOALLOC_MAX_ATOMS 16777216
MD_API int md_velocity_sums_noalloc(const double *vxyz_device, int64_t n_atoms, double *out5_device, void *stream);

MD_API const char *md_last_error(void);
MD_API const char *md_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MD_B200_H */
