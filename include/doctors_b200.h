/* doctors_b200.h — C ABI of the B200-native DOCTORS hot path (arXiv 1910.11335).
 *
 * The one thing this library computes: the 3-D Cartesian discrete-ordinates transport
 * sweep of the paper's Eq. (2) inside the multigroup source iteration
 * (PAPER.md:149, :183), driven by the ray-traced first-collision source of Eqs. (4)-(7)
 * (PAPER.md:44-62).  Every step runs in hand-written sm_100a CUDA kernels; there is no
 * CPU fallback: without a CUDA device every call that needs one returns DOCTORS_CUDA.
 *
 * Conventions (DESIGN.md §2 gives the readings R1-R16 of the paper behind them)
 *   - cell index c = i + nx*(j + ny*k), x fastest; the mesh is centred on the origin,
 *     x_i = (i + 1/2) dx - nx dx / 2 (same for y, z).
 *   - energy group g = 0 is the HIGHEST energy; scattering g_from -> g_to only for
 *     g_to >= g_from (in-scatter from equal or higher energy).
 *   - quadrature weights sum to 4 pi; moment index lm = l*l + l + m, real harmonics
 *     Y_l0 = P_l(xi), Y_l,+-m = sqrt(2 (l-m)!/(l+m)!) P_l^m(xi) {cos, sin}(m phi), no
 *     Condon-Shortley phase; moment 0 is the scalar flux of Eq. (3).
 *   - sigma_s,l normalisation: sigma_s(mu0) = sum_l (2l+1)/(4 pi) sigma_s,l P_l(mu0).
 *   - all cross sections are per unit density: sigma(c) = density(c) * table[material(c)].
 *
 * Ownership: every `set_*` call copies its inputs before returning (the caller may free
 * them); every output goes to a caller-allocated buffer.  Pointers are HOST pointers
 * unless the argument is named `device_*` or has an `*_is_device` flag.  The library
 * allocates no large device memory: the caller asks `doctors_workspace_bytes` and hands
 * a device buffer (e.g. a torch tensor's data_ptr) to `doctors_set_workspace`.
 *
 * Errors: every call returns a status; `doctors_last_error` gives the text.  No C++
 * exception crosses the ABI.  A handle is not thread-safe.
 */
#ifndef DOCTORS_B200_H
#define DOCTORS_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    DOCTORS_OK = 0,
    DOCTORS_INVALID_ARG = 1,
    DOCTORS_BAD_STATE = 2,      /* call order / inconsistent inputs (e.g. material id >= n_materials of the XS table) */
    DOCTORS_ALLOC = 3,          /* workspace missing or too small */
    DOCTORS_CUDA = 4,           /* CUDA runtime / driver error, or no device */
    DOCTORS_NOT_CONVERGED = 5,  /* warning class: outputs valid, some (source, group) hit max_iters */
    DOCTORS_NOT_RETAINED = 6    /* higher moments of a source solved in an earlier chunk were overwritten */
};

typedef struct doctors_problem doctors_problem;

/* Library version string, e.g. "doctors-b200 0.1 (sm_100a)". */
const char* doctors_version(void);

/* sizeof(doctors_source), sizeof(doctors_solve_opts), sizeof(doctors_solve_info) as this library was compiled:
 * out_sizes[3] (host).  A binding checks its own struct declarations against them. */
void doctors_abi_sizes(int* out_sizes);

/* Create / destroy a problem bound to `cuda_device` and to `stream` (a cudaStream_t passed as
 * void*, e.g. torch.cuda.current_stream().cuda_stream; NULL = the legacy default stream).
 * All kernels and copies of this handle are issued on that stream.
 * Errors: DOCTORS_CUDA if the device cannot be selected (no GPU, bad ordinal). */
int  doctors_create_problem(int cuda_device, void* stream, doctors_problem** out);
void doctors_destroy_problem(doctors_problem* p);
const char* doctors_last_error(const doctors_problem* p);

/* Voxel mesh and material map (PAPER.md:37 mesh, :155-159 material + density per voxel).
 *   material_id [nz][ny][nx] uint8 (host), density same shape float g/cm^3 or NULL (= 1).
 * Errors: INVALID_ARG for n <= 0, pitch <= 0, non-finite / negative density,
 *         id >= n_materials, n_materials > 16. */
int doctors_set_mesh_materials(doctors_problem* p, int nx, int ny, int nz,
                               double dx, double dy, double dz,
                               const uint8_t* material_id, const float* density,
                               int n_materials);

/* Multigroup total cross section and P_L scattering tables (Figs. 6-7), per unit
 * density.  sigma_t [n_mat][G];  sigma_s [n_mat][L+1][G_from][G_to].
 * Errors: INVALID_ARG for G <= 0, pl_order outside 0..3, negative sigma_t, or any non-zero
 *         upscatter entry (g_to < g_from). */
int doctors_set_xs(doctors_problem* p, int n_materials, int n_groups, int pl_order,
                   const double* sigma_t, const double* sigma_s);

/* Built-in level-symmetric S_N set, N in {2,4,6,8,12,16} -> N(N+2) directions (PAPER.md:39-42,
 * :208; the rule that fixes weights is DESIGN.md App. A).  Directions are stored octant-major,
 * octant bit0/1/2 set = negative x/y/z component. */
int doctors_set_quadrature(doctors_problem* p, int sn_order);
/* User quadrature: omega_xyz [n][3] unit vectors, w [n] with sum = 4 pi (checked to 1e-10).
 * Requirements: no zero component, the same number of directions in each octant.  The set is
 * re-ordered octant-major (stable); doctors_get_quadrature returns the stored order. */
int doctors_set_quadrature_points(doctors_problem* p, int n_dir, const double* omega_xyz, const double* w);
/* omega_xyz / w may be NULL to query n_dir only. */
int doctors_get_quadrature(const doctors_problem* p, int* n_dir, double* omega_xyz, double* w);

/* Source description (reading R12).  The mesh is centred on the origin. */
typedef struct {
    int kind;                 /* 0 isotropic volume source, 1 isotropic point, 2 cone (hard edge), 3 fan (hard edges) */
    double pos[3];            /* kinds 1, 2, 3: source position, cm */
    double axis[3];           /* kinds 2, 3: beam axis (need not be normalised) */
    double half_angle_rad;    /* kind 2: half angle of the cone; kind 3: half of the azimuthal angle the fan subtends IN its plane */
    const double* spectrum;   /* kinds 1, 2, 3: [G] photons emitted per group */
    const float* volume;      /* kind 0: [G][nz][ny][nx] photons/cm^3, 4pi-integrated (host) */
    double up[3];             /* kind 3: a vector out of the fan plane (not parallel to axis); the plane is spanned by axis and up x axis */
    double half_angle2_rad;   /* kind 3: half of the polar angle the fan subtends OUT of its plane, in (0, pi/2] (R18) */
} doctors_source;
/* mode 0: the n sources are independent problems, solved batched.
 * mode 1: the n sources are summed into ONE problem (the paper's CT scan).
 * Errors: INVALID_ARG for n_sources <= 0 or > 64, unknown kind, a point source within
 *         1e-9 pitch of a cell centre (1/R^2 singularity). */
int doctors_set_source(doctors_problem* p, int n_sources, const doctors_source* src, int mode);

typedef struct {
    double tol;               /* stop when max|dphi_0| / max|phi_0| < tol (reading R8); <= 0 -> 1e-5 */
    int max_iters;            /* <= 0 -> 100 */
    const int* fixed_iters;   /* NULL, or [n_problems][G]: entry > 0 = exactly that many sweeps (R10) */
    int closure;              /* 0 pure diamond difference; 1 + set-to-zero fix-up with rebalance (R2).
                               * The face recurrence is fp64 either way; faces that cross a brick boundary are stored as fp32 with
                               * closure 1 and as fp64 with closure 0 */
    int deterministic;        /* 1: octants swept one after another, fixed summation order (bit-reproducible) */
    int source_chunk;         /* problems solved together (HBM capacity); 0 = all that fit the workspace */
    int sweep_mode;           /* 0 brick wavefront kernel (product path); 1 the paper's one-launch-per-sub-sweep scheme,
                               * kept as a comparison arm */
    int brick[3];             /* sweep_mode 0: brick extents in cells; 0 = automatic.  brick[0] % 4 == 0, brick[1]*brick[2] <= 32 */
    int ctas_per_sm;          /* sweep_mode 0: persistent CTAs per SM; 0 = occupancy maximum */
    int check_window;         /* tolerance mode: sweeps enqueued between host reads of the device flag; 0 = adaptive
                               * (first read one sweep before the count the previous group needed, then every sweep) */
    int projection;           /* sweep_mode 0, the two projections of Eq. (2) rhs / Eq. (3) inside the sweep kernel:
                               * 0 automatic: tensor cores for more than 16 directions per octant (S12, S16), else the FMA loops
                               *   (the faster of the two as measured on B200); 1 packed fp32 FMA loops;
                               * 2 tensor cores (mma TF32, 3-product split, fp32 accumulate) when P3, <= 48 directions per
                               *   octant and a brick of a multiple of 8 cells; else the FMA loops */
} doctors_solve_opts;

typedef struct {
    int* iters;               /* [n_problems][G] caller-allocated, or NULL */
    double* residual;         /* [n_problems][G] last delta_k, or NULL */
    double* balance;          /* [n_problems][G][3] = sum Q_00 V, sum sigma_t phi_0 V, leakage of the last sweep; or NULL */
    double ms_raytrace, ms_fixed_source, ms_sweep, ms_iterate, ms_total;   /* CUDA-event times */
    unsigned long long updates;        /* cell*direction updates performed: sum_k cells * n_dir over all sweeps */
    unsigned long long sweep_launches; /* sweep kernel launches */
    unsigned long long kernel_launches;/* all kernel launches of this solve */
    int n_chunks;
    int brick[3];
    int ctas_per_sm;
    int sweep_kernel;         /* kernel that swept: 0 brick, 1 paper scheme */
    int projection_mtiles;    /* > 0: the projections ran on the tensor cores (16-direction m-tiles per octant); 0: fp32 FMA loops */
    unsigned long long timed_sweeps;   /* sweep iterations whose CUDA-event time is in ms_sweep (= all of them) */
    int pl_exceeds_quadrature;/* warning flag: 1 if the quadrature does not integrate Y_lm Y_l'm' exactly up to pl_order
                               * (level-symmetric sets: exact up to P1 / P2 / P3 / P4 at S2 / S4 / S6 / S8, >= P5 at S12 / S16;
                               * e.g. P3 with S4).  The solve runs; the scattering-source moments are then not Galerkin-consistent. */
} doctors_solve_info;

/* n_problems = n_sources (mode 0) or 1 (mode 1). */
int    doctors_n_problems(const doctors_problem* p);
/* Device bytes `doctors_solve` needs with these options (0 on error; see last_error). */
size_t doctors_workspace_bytes(doctors_problem* p, const doctors_solve_opts* opts);
/* `device_ptr` must be 256-byte aligned device memory that outlives the handle's use of it. */
int    doctors_set_workspace(doctors_problem* p, void* device_ptr, size_t bytes);

/* Whole hot path: ray trace (Eq. 4) -> per group, high to low energy: fixed source (Eq. 5 + downscatter)
 * -> source iteration { Q = sigma_s phi + fixed; sweep all 8 octants (Eq. 2); moments (Eq. 3);
 * convergence on the device }.  Blocks until the stream has finished.
 * Errors: BAD_STATE if mesh / xs / quadrature / source are missing or disagree (n_materials,
 * G), ALLOC if the workspace is missing or too small, CUDA on a runtime error.
 * Returns NOT_CONVERGED (outputs valid) if any (problem, group) stopped at max_iters. */
int doctors_solve(doctors_problem* p, const doctors_solve_opts* opts, doctors_solve_info* info);

/* Collided-flux moments of one (problem, group): out [(l_max+1)^2][nz][ny][nx] fp32, to a host
 * (out_is_device = 0) or device buffer.  l_max = 0 (scalar flux, Eq. 3) is retained for every
 * problem; l_max > 0 only for problems of the last chunk solved (else NOT_RETAINED).
 * Errors: BAD_STATE before a successful solve; INVALID_ARG for bad indices / l_max > L. */
int doctors_get_flux_moments(doctors_problem* p, int problem, int group, int l_max,
                             float* out, int out_is_device);
/* Uncollided scalar flux of Eq. (4) for one SOURCE and group: out [nz][ny][nx] fp32. */
int doctors_get_uncollided_flux(doctors_problem* p, int source, int group, float* out, int out_is_device);

/* Post-processing hook ("a conversion of photon fluence to an absorbed dose"): a response per group folded
 * with the scalar fluence of one PROBLEM on the device,
 *   out[nz][ny][nx] = sum_g response[g] * (phi_00,g + (include_uncollided ? sum over the problem's sources of phi_u,g : 0)),
 * fp64 accumulation over the groups, fp32 result.  response: [G] doubles (host, copied).  The collided flux alone is what
 * the sweep computes; the total fluence of the first-collision method is collided + uncollided.
 * Errors: BAD_STATE before a successful solve, INVALID_ARG for a bad problem index or NULL pointers. */
int doctors_get_response(doctors_problem* p, int problem, const double* response, int include_uncollided,
                         float* out, int out_is_device);

/* Test hooks: the integer schedules the kernels consume (Eqs. 8-22, Table 1),
 * for the bit-exact check against the oracle.
 *   level 0: cells of the whole mesh in sub-sweep order (what sweep_mode 1 launches over)
 *   level 1: bricks of the brick grid in sub-sweep order (the task order of sweep_mode 0)
 *   level 2: cells of one full brick in sub-sweep order, local index li + bx*(lj + by*lk).  The kernel
 *            needs no table at this level (lane (j',k') at step s updates i' = s - j' - k'); the planes it
 *            actually visits are checked with doctors_debug_device_brick_steps
 * dims = extents the schedule runs over; plane_offset has dims[0]+dims[1]+dims[2]-1 entries,
 * cell_of has dims[0]*dims[1]*dims[2].  Uses opts->brick (NULL opts = automatic). */
int doctors_debug_schedule_dims(doctors_problem* p, const doctors_solve_opts* opts, int level, int dims[3]);
int doctors_debug_get_schedule(doctors_problem* p, const doctors_solve_opts* opts, int octant, int level,
                               int32_t* plane_offset, int32_t* cell_of);
/* Device-side check of the in-brick wavefront (level 2): runs the product sweep kernel on one full
 * bx x by x bz brick for `octant` and returns, per cell (local index li + bx*(lj + by*lk)), the step at
 * which the kernel updated it.  By Eq. (8) that step must equal the cell's sub-sweep
 * index i'+j'+k' in the octant's sweep-space coordinates.  The same launch bounds-checks every shared-memory address of the
 * wavefront loop, idle lanes included (they load from their running addresses): an address outside the CTA's allocation makes
 * the call return DOCTORS_CUDA (compute-sanitizer is closed on this pool; this is the repo's own check).  Needs a CUDA device. */
int doctors_debug_device_brick_steps(doctors_problem* p, int bx, int by, int bz, int octant, int32_t* step_of_cell);
/* P(S) of Eq. (9) as the library evaluates it. */
long long doctors_wavefront_size(int nx, int ny, int nz, int S);
/* Projection tables the kernels use (fp32 copies of these doubles):
 * Mtab [n_dir][nm] = (2l+1)/(4pi) Y_lm(Omega_n), Dtab [n_dir][nm] = w_n Y_lm(Omega_n). */
int doctors_debug_get_tables(const doctors_problem* p, int pl_order, double* Mtab, double* Dtab);


/* Host-only helpers (no device needed): the generators behind set_quadrature and the schedules,
 * callable without a handle so that the host logic can be tested on a machine without a GPU.
 * doctors_host_level_symmetric: omega_xyz [N(N+2)][3], w [N(N+2)]; returns INVALID_ARG for an
 * unsupported N.  doctors_host_schedule: as doctors_debug_get_schedule over an nx x ny x nz box.
 * doctors_host_projection_tables: Mtab / Dtab [n_dir][(L+1)^2] for the given directions. */
int doctors_host_level_symmetric(int sn_order, double* omega_xyz, double* w);
int doctors_host_schedule(int nx, int ny, int nz, int octant, int32_t* plane_offset, int32_t* cell_of);
int doctors_host_projection_tables(int pl_order, int n_dir, const double* omega_xyz, const double* w,
                                   double* Mtab, double* Dtab);
/* The warning doctors_solve_info.pl_exceeds_quadrature as a host function: returns 1 if the set does NOT integrate the
 * products Y_lm Y_l'm' exactly for all l, l' <= pl_order (defect = max |sum_n w_n Y_lm (2l'+1)/(4 pi) Y_l'm' - delta| > 1e-9),
 * 0 if it does, -1 for bad arguments; *defect (may be NULL) receives the defect.  Level-symmetric sets are exact up to
 * P1 / P2 / P3 / P4 at S2 / S4 / S6 / S8 and beyond P3 at S12 / S16 (quadrature rule). */
int doctors_host_pl_exceeds_quadrature(int pl_order, int n_dir, const double* omega_xyz, const double* w, double* defect);


/* Allocation-free entry point (for callers that may not allocate: CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc).  The convergence measure of the source iteration (reading R8), per problem q:
 *     delta_q = max_c |phi_new[q][c] - phi_old[q][c]| / max_c |phi_new[q][c]|       (0 if phi_new is identically 0)
 * i.e. what doctors_solve evaluates on the device after every sweep, offered for fluxes the caller holds.
 *   device_phi_new, device_phi_old : DEVICE pointers, fp32, problem q at offset q * problem_stride, n_cells values each
 *                                    (any cell order; padding cells must hold equal values in both, e.g. 0)
 *   device_out                     : DEVICE pointer, [n_problems][3] fp32 = delta, max |new - old|, max |new|; a NaN input gives inf
 * The call enqueues a 256-byte memset node and one kernel on the handle's stream and returns without synchronising; it calls
 * no cudaMalloc / cudaFree / allocating routine.  Its cross-block scratch is a static __device__ array of 33,024 bytes that
 * every GPU which loads the library holds until exit.  Limit: n_problems <= 64 per call (INVALID_ARG beyond, with a message).
 * ALL calls on a device share that array: calls that overlap on the GPU (other streams, other handles) race — serialise them.
 * The first call per device looks up the array's device address (cudaGetSymbolAddress): make it outside a graph capture.
 * Errors: INVALID_ARG (NULL pointer, n_problems outside 1..64, n_cells < 1, stride < n_cells), CUDA on a runtime error. */
int doctors_convergence_delta_no_alloc(doctors_problem* p, const float* device_phi_new, const float* device_phi_old,
                                       long long n_cells, long long problem_stride, int n_problems, float* device_out);

#ifdef __cplusplus
}
#endif
#endif /* DOCTORS_B200_H */
