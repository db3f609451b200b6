/*
 * sph.h -- C ABI of the B200-native WCSPH particle-interaction sweep (libsph_b200.so).
 *
 * The library implements the per-time-step hot path of the fully coupled fluid-solid-thermal
 * weakly-compressible SPH solver of arxiv/paper_2512_09904 (citations are PAPER.md:<line>):
 * neighbour build, Riemann-based continuity / momentum sums (Eq. 10-13), density
 * re-initialisation (Eq. 14-15, :123-133), one-sided-Riemann wall forces (Eq. 16-19, :137-155),
 * thermal diffusion (Eq. 22, :169), dual-criteria time stepping (Eq. 25-26, :189-200), prescribed
 * gear rotation (:276, :336) and churning torque (:336-338).  Readings of passages the paper
 * leaves open are the R-numbers of DESIGN.md section 3.
 *
 * Conventions
 *  - plain pointers and sizes only; every array argument says whether it is HOST or DEVICE memory
 *    through `mem_kind`.  The context owns all device memory it allocates; callers own every
 *    buffer they pass; input buffers are copied before the call returns.
 *  - one context <-> one CUDA device + one stream (the stream handed in `sph_params.cuda_stream`,
 *    NULL = legacy default stream).  Not thread-safe per context; no global state.
 *  - all functions return 0 (SPH_OK) or a negative error code; sph_last_error gives text.
 *  - sph_step is asynchronous on the stream.  Device-detected errors (particle outside the grid,
 *    NaN, neighbour-list overflow) surface at the next synchronising call (sph_get_fields,
 *    sph_get_torque, sph_synchronize).
 *  - there is no CPU fallback: without a CUDA device sph_create fails with SPH_ECUDA.
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPH_MAX_BODIES 8

/* error codes */
#define SPH_OK 0
#define SPH_EINVAL (-1)   /* bad argument */
#define SPH_ENOMEM (-2)   /* device or host allocation failed */
#define SPH_ECUDA (-3)    /* CUDA runtime error (text in sph_last_error) */
#define SPH_EDOMAIN (-4)  /* a particle left the grid domain (it was clamped into the border cell) */
#define SPH_ENAN (-5)     /* a non-finite position was met */
#define SPH_ESTATE (-6)   /* call out of order (e.g. step before load) */
#define SPH_ENEIGH (-7)   /* a neighbour list exceeded max_neigh_fluid / max_neigh_wall */

/* sph_params.flags */
#define SPH_FLAG_FREE_SURFACE 1u    /* Eq. 14 (max form) for EVERY particle instead of Eq. 15 in the density re-initialisation
                                       (the whole fluid is one free-surface flow: DESIGN.md reading R12) */
#define SPH_FLAG_DENSITY_REINIT 2u  /* apply Eq. 14/15 at every neighbour rebuild */
#define SPH_FLAG_THERMAL 4u         /* Eq. 22 heat conduction, fluid-fluid and fluid-wall */
#define SPH_FLAG_VISCOUS 8u         /* viscous sums of Eq. 10 l.2 and Eq. 18 l.2 */
#define SPH_FLAG_HYDRO 16u          /* off: particles are static, only the heat equation advances */
#define SPH_FLAG_DUAL_CRITERIA 32u  /* informational; the rebuild policy is `rebuild_every` */
#define SPH_FLAG_PRESSURE 64u       /* pressure sums of Eq. 10 l.2 and Eq. 18 l.1 */
#define SPH_FLAG_VISCOUS_HELD 128u  /* with SPH_FLAG_VISCOUS: the viscous sums are evaluated by the first acoustic step after each
                                       neighbour rebuild and held until the next one, as in the dual-criteria scheme of ref [45]
                                       (reading R26); off: every acoustic step (R8) */
#define SPH_FLAG_FREE_SURFACE_LOCAL 256u /* Eq. 14 only "in regions identified as free-surface flow", Eq. 15 elsewhere
                                       (:129).  DESIGN.md reading R27: surface particle = kernel sum sigma_i < fs_threshold * sigma0;
                                       region = the surface particles and all their fluid neighbours.  Wins over
                                       SPH_FLAG_FREE_SURFACE when both are set */

#define SPH_MEM_HOST 0
#define SPH_MEM_DEVICE 1

/* sph_get_fields field ids.  Element type and count per particle in brackets; fluid fields have
 * n_fluid entries, WALL_* fields n_wall entries, all in ORIGINAL (caller) particle order. */
enum sph_field {
    SPH_FIELD_POS = 0,          /* [f32 x3] current positions r */
    SPH_FIELD_VEL = 1,          /* [f32 x3] velocities v */
    SPH_FIELD_RHO = 2,          /* [f32] density rho = rho0 + drho */
    SPH_FIELD_P = 3,            /* [f32] pressure, Eq. 2: c0^2 (rho - rho0) */
    SPH_FIELD_T = 4,            /* [f32] temperature */
    SPH_FIELD_ACC = 5,          /* [f32 x3] dv/dt of the last sweep A (incl. g) */
    SPH_FIELD_DRHO_DT = 6,      /* [f32] drho/dt of the last sweep B */
    SPH_FIELD_DT_DT = 7,        /* [f32] dT/dt of the last sweep B */
    SPH_FIELD_CELL = 8,         /* [i32 x3] cell coordinates at the last rebuild */
    SPH_FIELD_NEIGH_COUNT = 9,  /* [u32 x2] number of fluid, wall neighbours at the last rebuild */
    SPH_FIELD_NEIGH_DIGEST = 10,/* [u64] order-independent digest of the neighbour set (R1) */
    SPH_FIELD_DRHO = 11,        /* [f32] rho - rho0 exactly as stored */
    SPH_FIELD_WALL_POS = 12,    /* [f32 x3] wall positions at the last rebuild */
    SPH_FIELD_WALL_NORMAL = 13, /* [f32 x3] wall normals at the last rebuild */
    SPH_FIELD_STATS = 14,       /* [f64 x SPH_STATS_COUNT] see below; not per particle */
    SPH_FIELD_NEIGH_CSR_FLUID = 15, /* [i32] concatenated fluid-neighbour original ids, particle by particle in
                                       original order, each list ascending; size = sum of counts */
    SPH_FIELD_NEIGH_CSR_WALL = 16,  /* [i32] same for wall neighbours (original wall ids) */
    SPH_FIELD_DRHO_SAVED = 17,  /* [f32] drho/dt saved for the next first half step (R7) */
    SPH_FIELD_THETA = 18,       /* [f32] T - T_ref exactly as stored */
    SPH_FIELD_CONTACT_FACTOR = 19, /* [f32 per WALL particle, original wall order] zeta_C of Eq. 24:
                                   sum_j V_j W_wj over the lubricant neighbours of solid particle w (V_j = m / rho_j now,
                                   distances of the last rebuild) / the same sum with every place of w's support that no
                                   solid particle takes filled with lubricant, dx^3 (sigma0 - sum_w' W_ww') (R22);
                                   0 for buried particles.  Needs a completed step (SPH_ESTATE otherwise). */
    SPH_FIELD_WALL_T = 20,      /* [f32 per WALL particle, original wall order] wall temperature (evolves for bodies with
                                   thermal_mode = 1, R23; held otherwise) */
    SPH_FIELD_WALL_DT_DT = 21,  /* [f32 per WALL particle] dT_w/dt of the last step (0 for held bodies) */
    SPH_FIELD_FS_REGION = 22,   /* [u32] which form the last density re-initialisation took for the particle: 0 = Eq. 15,
                                   1 = Eq. 14 as a neighbour of a surface particle, 2 = Eq. 14 as a surface particle
                                   (R27; all 0 without SPH_FLAG_FREE_SURFACE_LOCAL) */
    SPH_FIELD_SORT_CELL_COUNT = 23, /* [u32 x n_sort_cells] fluid particles per sort cell at the last rebuild (row a3's
                                   histogram; n_sort_cells = 4 ncell_x ncell_y ncell_z: every contract cell is cut into 4
                                   sub-cells along x, x fastest).  Not per particle; needs a completed rebuild */
    SPH_FIELD_SORT_CELL_START = 24, /* [u32 x (n_sort_cells + 1)] its exclusive prefix sum = first sorted fluid index of
                                   every sort cell, last entry = n_fluid (row a3's cell_start) */
};

/* SPH_FIELD_STATS layout (doubles) */
enum sph_stat {
    SPH_STAT_T = 0, SPH_STAT_DT = 1, SPH_STAT_DT_AD = 2, SPH_STAT_ELAPSED = 3, SPH_STAT_VMAX = 4,
    SPH_STAT_STEPS = 5, SPH_STAT_REBUILDS = 6, SPH_STAT_SIGMA0 = 7, SPH_STAT_NCELL_X = 8,
    SPH_STAT_NCELL_Y = 9, SPH_STAT_NCELL_Z = 10, SPH_STAT_ERROR_BITS = 11, SPH_STAT_LAUNCHES = 12,
    SPH_STAT_DEVICE_BYTES = 13, SPH_STAT_MAX_NEIGH_FLUID = 14, SPH_STAT_MAX_NEIGH_WALL = 15,
    SPH_STAT_TILES = 16, SPH_STAT_DIRECT_TILES = 17,   /* tiles of the last rebuild; those gathering from global memory */
    SPH_STAT_SPLIT_TILES = 18,                         /* tiles processed as 2 or 4 sub-tile passes */
    SPH_STAT_T_MEAN = 19,                              /* average lubricant temperature (Fig. 10): mean of T
                                                          over the fluid particles, reduced on the device in fp64 */
    SPH_STAT_SPLIT4_TILES = 20,                        /* of the split tiles, those processed as 4 sub-tile passes */
    SPH_STATS_COUNT = 21
};

/* kernel classes for sph_get_profile */
enum sph_kernel_class {
    SPH_K_CONTROL = 0, SPH_K_WALL_KINEMATICS = 1, SPH_K_HASH = 2, SPH_K_SCAN = 3, SPH_K_SCATTER = 4,
    SPH_K_REORDER = 5, SPH_K_BUILD_LISTS = 6, SPH_K_REINIT = 7, SPH_K_PRE = 8, SPH_K_SWEEP_A = 9,
    SPH_K_SWEEP_B = 10, SPH_K_FINISH = 11, SPH_K_OTHER = 12, SPH_K_COUNT = 13
};

typedef struct sph_body_params {
    double k_s;            /* conductivity seen by the fluid, W/mK; 0 = adiabatic (R10) */
    double rho_s, cp_s;    /* solid density and specific heat: used by thermal_mode 1 */
    int32_t thermal_mode;  /* 0 = wall temperature held (the paper's runs); 1 = evolving by Eq. 20 with the
                              fluid and solid neighbours (R23) */
    int32_t reserved;
} sph_body_params;

typedef struct sph_params {
    uint32_t struct_size;  /* = sizeof(sph_params), checked */
    uint32_t flags;
    double dx;             /* initial particle spacing; m = rho0 dx^3, V_w = dx^3 (dx^2 when dim = 2) */
    double h;              /* smoothing length (Wendland C2, support 2h; R2) */
    double rho0, c0, nu;   /* Eq. 2 reference density and sound speed; kinematic viscosity */
    double g[3];
    double k_f, cp_f;      /* fluid conductivity, specific heat (Table 6) */
    double T_ref;          /* temperatures are stored as T - T_ref in fp32 */
    double cfl_ac, cfl_ad; /* Eq. 25; 0 -> 0.6 and 0.25 */
    double u_ref;          /* floor of |v|max in Eq. 25 (R13); < 0 -> c0/10 */
    double dt_fixed;       /* > 0: fixed acoustic step; 0: Eq. 25 */
    int32_t rebuild_every; /* K >= 1: rebuild every K acoustic steps; 0: when dt_ad has elapsed */
    int32_t n_bodies;      /* 1..SPH_MAX_BODIES; body 0 = housing by convention */
    double domain_min[3], domain_max[3];   /* grid covers this box; cell edge 2h(1+2^-10) */
    uint64_t max_fluid, max_wall;          /* capacities (0 -> sized at the first load) */
    uint32_t max_neigh_fluid, max_neigh_wall; /* list capacities per particle; 0 -> 160 / 96 */
    sph_body_params body[SPH_MAX_BODIES];
    int32_t device;        /* CUDA device ordinal */
    int32_t dim;           /* 0 or 3: three-dimensional; 2: planar run (R25): all particles share one z, the
                              kernel takes its 2-D normalisation 7 / (4 pi h^2), volumes are dx^2 */
    void *cuda_stream;     /* cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream */
    double fs_threshold;   /* theta of the surface test sigma_i < theta sigma0 under SPH_FLAG_FREE_SURFACE_LOCAL (R27); 0 -> 0.9 */
} sph_params;

typedef struct sph_ctx sph_ctx;

/* Create a context for one problem statement: the parameters are those the paper tabulates for its cases (Tables 5-6,
 * spacing, oil density / viscosity / conductivity / specific heat; c0 = 10 U_max, Eq. 2) plus
 * the switches of the scheme.  Checks params, selects the device, computes the grid of R1 and sigma0, the full-lattice kernel
 * sum that is the "sum W^0" of Eq. 14-15 (R12).  `p` and `out` are HOST pointers; the context is owned by
 * the library until sph_destroy.  Errors: SPH_EINVAL (bad parameter or struct_size), SPH_ECUDA (no device), SPH_ENOMEM;
 * *out is NULL on failure and sph_last_error(NULL) gives the text. */
int sph_create(const sph_params *p, sph_ctx **out);

/* Free everything the context owns (device memory, graphs, streams, events).  NULL is allowed.  Always SPH_OK. */
int sph_destroy(sph_ctx *ctx);

/* Load the particle state: the fluid particles (r, v, rho, T: the symbols of Eq. 1-4 and 10) and
 * the dummy wall particles of the solids with their unit normals pointing from the solid into the fluid (Eq. 16,
 * PAPER.md:137-141; R16), body index in [0, n_bodies) and temperature (Eq. 22).  AoS [n][3] / [n] fp32 arrays
 * in caller order; rho_f may be NULL (-> rho0), vel_f may be NULL (-> 0); the wall arrays may be NULL iff n_w == 0.  Uniform mass
 * m = rho0 dx^3 and wall volume dx^3.  Resets t = 0, the saved drho/dt, the body angles and the materials.
 * All pointers are `mem_kind` memory; the buffers are copied before the call returns (it synchronises the stream).
 * Errors: SPH_EINVAL (NULL / counts above the capacity / body index out of range), SPH_ENOMEM, SPH_ECUDA. */
int sph_load_particles(sph_ctx *ctx, uint64_t n_f, const float *pos_f, const float *vel_f,
                       const float *rho_f, const float *T_f, uint64_t n_w, const float *pos_w,
                       const float *normal_w, const int32_t *body_w, const float *T_w, int mem_kind);

/* Per-particle materials of the heat equation.  Eq. 20-22 are written for particles of different
 * conductivity, K_ij = 4 k_i k_j / (k_i + k_j), and the benchmark of section 3.2 (Table 3) has two materials of
 * different density, conductivity and specific heat.  Arrays of n_fluid floats in caller order, `mem_kind` memory: mass m_i
 * (V_i = m_i / rho_i in the heat sums), conductivity k_i, specific heat cp_i; a NULL array keeps the uniform value of sph_params
 * (m = rho0 dx^3, k_f, cp_f); all three NULL returns to uniform materials.  With materials set, dT/dt of Eq. 22 is summed with
 * them (fluid-fluid and fluid-wall pairs; the wall side keeps sph_body_params.k_s).  The hydrodynamic sums (Eq. 10-19) are
 * written for one fluid: mass_f must be NULL when SPH_FLAG_HYDRO is set (SPH_EINVAL otherwise).  Call after
 * sph_load_particles (a load resets to uniform materials).  Synchronises. */
int sph_set_materials(sph_ctx *ctx, const float *mass_f, const float *k_f, const float *cp_f, int mem_kind);

/* Overwrite the fluid state of the loaded particles WITHOUT restarting the run: positions, velocities, densities and temperatures
 * in caller (original) order, `mem_kind` memory; a NULL array leaves that quantity as it is.  The clock, the body angles, the wall
 * particles, the saved drho/dt of the position-Verlet first half (R7) and the particle count are kept.  If any uploaded position
 * differs from the one the library holds, the neighbour configuration is rebuilt by the next sph_step (positions may have moved
 * arbitrarily: "neighbor lists ... are updated"); positions that come back bit for bit (a host loop that acts on
 * velocities or temperatures only) leave it standing.  This is the per-step upload of a host-coupled run (sph_get_fields is
 * its read-back).  Synchronises. */
int sph_set_state(sph_ctx *ctx, const float *pos_f, const float *vel_f, const float *rho_f, const float *T_f, int mem_kind);

/* Prescribed rigid rotation of body `body` about the line (origin, axis) with angular speed omega
 * (PAPER.md:276, :293-308).  HOST pointers.  axis is normalised.  Takes effect at the next step;
 * wall positions move at neighbour rebuilds (the configuration is frozen in between). */
int sph_set_gear_kinematics(sph_ctx *ctx, int body, const double origin[3], const double axis[3],
                            double omega);

/* Advance n acoustic steps of the dual-criteria scheme (section 2.8): each step = dt from Eq. 25 (bounded by
 * Eq. 26), neighbour configuration + density re-initialisation (Eq. 14-15) when the advection step has elapsed
 * ("neighbor lists and kernel-related quantities are updated based on the advection time step"), position-Verlet
 * first half (R7), momentum sums of Eq. 10 l.2 with Eq. 11-12 and the wall forces of Eq. 16-19, kick and
 * drift, continuity of Eq. 10 l.1 with Eq. 13 and heat conduction of Eq. 22, second half, torque.
 * Asynchronous on the context's stream: returns when the work is enqueued; device-detected errors surface at the next
 * synchronising call.  Errors here: SPH_ESTATE (nothing loaded), SPH_EINVAL (n < 0), SPH_ECUDA. */
int sph_step(sph_ctx *ctx, int n);

/* Copy one field (enum sph_field: the state and the rates of Eq. 10 / 22, the neighbour configuration of PAPER.md:191, the
 * contact factor of Eq. 24, statistics) to dst in ORIGINAL particle order.  dst is `mem_kind` memory owned by the caller and
 * dst_bytes must be at least the field size (sph_field_bytes gives it, also for the two variable-size NEIGH_CSR fields).
 * Synchronises.  Errors: SPH_EINVAL (unknown field, NULL or too small dst), SPH_ESTATE, or the pending device error
 * (SPH_EDOMAIN / SPH_ENAN / SPH_ENEIGH), which is cleared by reporting it. */
int sph_get_fields(sph_ctx *ctx, uint32_t field, void *dst, uint64_t dst_bytes, int mem_kind);

/* Size in bytes of a field for the currently loaded particles (synchronises for the CSR fields). */
int sph_field_bytes(sph_ctx *ctx, uint32_t field, uint64_t *bytes);

/* Churning torque (no formula is printed: reading R15): moment about the body's origin of the forces
 * the fluid exerted on the wall particles of body `body` during the last completed step, F_w = -sum_i m_i (pressure + viscous
 * pair accelerations of Eq. 18); axial = axis . torque (negative = resisting for omega > 0).  `torque` (3 doubles) and `axial`
 * (may be NULL) are HOST pointers.  Synchronises; returns the pending device error if one was raised. */
int sph_get_torque(sph_ctx *ctx, int body, double torque[3], double *axial);

/* n steps of the physics-driven particle relaxation of Eq. 6-9 with the constant background
 * pressure p0 > 0, without the level set (R24): per step a neighbour configuration of the present positions,
 * F_p,i = -(2/m_i) sum_j V_i V_j p0 grad_i W_ij over fluid and wall neighbours (V = dx^3, m = rho0 dx^3), one global
 * dt = 0.25 sqrt(h / max|F_p|), r_i += F_p,i dt^2 / 2.  Only fluid positions change (v, rho, T, walls, clock untouched);
 * the next sph_step rebuilds the neighbour configuration.  Asynchronous on the stream like sph_step. */
int sph_relax(sph_ctx *ctx, int n, double p0);

/* Wait for the stream; returns the pending device error, if any, and clears it. */
int sph_synchronize(sph_ctx *ctx);

/* Per-kernel-class device timing with CUDA events on the context's stream.  enable != 0 starts a
 * fresh recording (every later launch is bracketed by an event pair), enable == 0 stops it. */
int sph_profile(sph_ctx *ctx, int enable);

/* Total device milliseconds and launch count of one kernel class since sph_profile(ctx, 1).
 * HOST pointers.  Synchronises. */
int sph_get_profile(sph_ctx *ctx, int kernel_class, double *ms_total, uint64_t *launches);

/* Row a3 on its own, for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the exclusive prefix sum of a per-cell histogram ("histogram per cell ->
 * exclusive scan -> cell_start[n_cells + 1]"; the neighbour search the paper only names),
 *     starts[c] = counts[0] + ... + counts[c - 1]  (c = 0 .. n_cells - 1),   starts[n_cells] = n_items,
 * by the library's three scan kernels, with their scratch (one partial sum per 2048 cells) in a file-scope
 * `static __device__` array of SPH_SCAN_STATIC_SCRATCH_BYTES instead of context memory.  No context is needed.
 *   device          CUDA device ordinal; it must be the device that owns the two buffers and the stream
 *   counts_dev      DEVICE pointer, uint32 [n_cells], read only
 *   starts_dev      DEVICE pointer, uint32 [n_cells + 1], written; must not overlap counts_dev
 *   n_cells         0 < n_cells <= SPH_SCAN_STATIC_MAX_CELLS, else SPH_EINVAL with a text that names the limit
 *   n_items         the value stored in starts[n_cells] (the caller's particle count; it is not checked against the sum)
 *   cuda_stream     cudaStream_t the kernels are enqueued on (NULL = default stream); asynchronous, no synchronisation
 * The call allocates and frees nothing: no cudaMalloc / cudaFree / cudaMallocAsync, no allocating library routine; the
 * caller owns both buffers.  The first call on a device resolves the scratch array's device address once
 * (cudaGetSymbolAddress with that device current; the current device of the calling thread is restored) -- make that
 * first call outside a stream capture.  The scratch array is ONE per device and process, shared by every call and every
 * thread and holding the last call's partial sums: calls on the same device that can overlap on the GPU (different
 * streams without an ordering between them) race on it and give wrong prefix sums; calls on one stream are ordered and
 * safe.  Nothing in it has to start at zero (every entry a call reads it has written itself first).  Every GPU that loads
 * the library carries the array until the process exits.
 * Returns SPH_OK, SPH_EINVAL (NULL pointer, bad size, overlap, bad device) or SPH_ECUDA; the text is read with
 * sph_last_error(NULL) on the calling thread. */
#define SPH_SCAN_STATIC_MAX_CELLS (1u << 24)              /* 16,777,216 sort cells (cfg4 has 6.4 M) */
#define SPH_SCAN_STATIC_SCRATCH_BYTES (32768u + 256u)     /* 8192 partial sums + padding */
int sph_cell_scan_static(int device, const uint32_t *counts_dev, uint32_t *starts_dev, uint32_t n_cells, uint32_t n_items,
                         void *cuda_stream);

/* Measurement helper for bench.py's roofline (not part of the step): the plain fp32 FMA rate this device sustains, in
 * TFLOP/s (FMA = 2 flops), from a kernel of independent FFMA chains that fills every SM, timed with CUDA events on
 * `cuda_stream` (best of three launches after a warm-up).  It stands beside the derived ALU peak (SMs x 128 lanes x 2 x
 * clock).  tflops: HOST pointer.  Allocates and frees a small device buffer; synchronises. */
int sph_measure_fma_peak(int device, double *tflops, void *cuda_stream);

/* Text of the last error of this context ("" if none).  ctx may be NULL (-> create-time error, or the error of the last
 * context-free call, sph_cell_scan_static, on this thread). */
const char *sph_last_error(const sph_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
