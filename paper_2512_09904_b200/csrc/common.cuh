// common.cuh -- device-side parameter blocks and small helpers shared by the CUDA kernels.
// Part of libsph_b200 (sm_100a).  Notation follows PAPER.md: i fluid particle, j fluid neighbour,
// w wall neighbour, r_ij = r_i - r_j, e_ij = r_ij/|r_ij|, F_ij = W'(r_ij)/r_ij, V = m/rho.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define SPH_MAXB 8
#define SPH_SX 4                   // sort cells per contract cell along x (see fine_coord)

// flag bits (mirror include/sph.h)
#define F_FREE_SURFACE 1u
#define F_DENSITY_REINIT 2u
#define F_THERMAL 4u
#define F_VISCOUS 8u
#define F_HYDRO 16u
#define F_PRESSURE 64u
#define F_VISCOUS_HELD 128u
#define F_FREE_SURFACE_LOCAL 256u

// device error bits
#define ERR_DOMAIN 1u
#define ERR_NAN 2u
#define ERR_NEIGH 4u
#define ERR_BOUNDS 8u
// Debug build (-DSPH_BOUNDS_CHECK; compute-sanitizer is not available on the GPU pool): the index checks the kernels can make
// themselves -- staged gathers inside the staged records, hit-buffer and scatter-array positions inside their arrays, headers
// inside the budget.  A failed check sets ERR_BOUNDS in a device word that sync_and_check() reports as SPH_ECUDA.  The release
// build compiles the checks away.
#ifdef SPH_BOUNDS_CHECK
__device__ unsigned int g_sph_bounds_err = 0u;
#define SPH_DBG_CHECK(cond, bit) do { if (!(cond)) atomicOr(&g_sph_bounds_err, 1u << (bit)); } while (0)
#else
#define SPH_DBG_CHECK(cond, bit) do { } while (0)
#endif

struct BodyF {                 // per body, float copy used inside the pair sweeps
    float ox, oy, oz;          // origin o_b
    float wx, wy, wz;          // omega_b * a_b  (v_w = wvec x (r_w - o_b))
    float K;                   // K_in = 4 k_f k_n / (k_f + k_n), Eq. 22 (0 if adiabatic)
    float pad;
};

struct DevParams {
    // grid (reading R1)
    float xmin[3];
    float inv_ell;
    int ng[3];
    int n_cells;               // sort cells: SPH_SX * ng[0] * ng[1] * ng[2]
    float rc2;
    float inv_ell4;            // SPH_SX * inv_ell (exact: a power of two)
    int nfx;                   // SPH_SX * ng[0]: sort cells per row
    float rcu2;                // (rc * inv_ell)^2 (1 + 1e-4): squared cut-off in contract-cell units, rounded up
    // kernel (R2): F = CF (1 - q/2)^3, W = CW (1 - q/2)^4 (1 + 2q)
    float h, inv_h, half_inv_h, CF, CW;
    // fluid
    float rho0, inv_rho0, c0, c0sq, inv_c0, inv_c0sq, eta, mass, Vw, gx, gy, gz, k2f, inv_cp;
    uint32_t flags;
    int n_f, n_w;
    int KF, KW;                // list capacities per particle (multiples of 8)
    int dummy_f, dummy_w;      // index of the far-away dummy record at the end of the sorted fluid / wall arrays
    BodyF body[SPH_MAXB];
    // evolving solid temperature (R23): conductivity, 1 / (rho_s c_s dx^3), mode (1 = evolving) per body
    float bk[SPH_MAXB], binvC[SPH_MAXB];
    int bmode[SPH_MAXB];
};

struct BodyD {                 // per body, double state owned by the control kernel
    double origin[3], axis[3], omega, theta, cs, sn;
};

struct Clock {                 // device-resident clock; one instance per context
    double t, t_kin, dt, dt_ad, elapsed;
    double cfl_ac, cfl_ad, u_ref, dt_fixed, h, c0, nu;
    double dt_T;                     // Eq. 26 bound of the explicit thermal step (0: none)
    double torque[SPH_MAXB][3];      // accumulated by sweep A of the current step
    double torque_done[SPH_MAXB][3]; // torque of the last completed step
    double torque_visc[SPH_MAXB][3]; // R26: viscous part, summed by the step that rebuilt and held until the next rebuild (else 0)
    long long steps, rebuilds, since_rebuild;
    long long last_adv_steps;        // acoustic steps of the advection step that ended at the last rebuild (0 before the second rebuild)
    long long graph_rebuilds;        // rebuilds taken through the conditional node of the step graph
    float dt_f;
    unsigned int work_A, work_B;   // tile counters of the persistent sweeps (reset by k_control)
    unsigned int relax_f2_bits; // max |F_p|^2 of the current relaxation step (Eq. 8), as float bits
    unsigned int vmax2_bits;   // max |v|^2 of the last kick, as float bits (non-negative floats order as uints)
    float vmax;
    int rebuild_every;
    int have_config;
    int rebuild;               // decided by the control kernel for the current step
    unsigned int err;
    unsigned int state_moved;  // sph_set_state: some uploaded position differs from the one held
    int walls_moving;
    BodyD body[SPH_MAXB];
};

__device__ __forceinline__ float4 ldg4(const float4* p) { return __ldg(p); }

// Canonical cell coordinate (R1): c = floor(fl(fl(x - xmin) * inv_ell)), clamped.
__device__ __forceinline__ int cell_coord(float x, float xmin, float inv_ell, int n, unsigned int& err)
{
    float rel = __fsub_rn(x, xmin);
    float s = __fmul_rn(rel, inv_ell);
    int c = (int)floorf(s);
    if (!(s == s) || fabsf(s) > 1e9f) { err |= ERR_NAN; c = 0; }
    if (c < 0) { c = 0; err |= ERR_DOMAIN; }
    if (c > n - 1) { c = n - 1; err |= ERR_DOMAIN; }
    return c;
}

// Sort grid.  The contract grid of R1 (cell edge ell = 2h(1 + 2^-10)) is kept for y and z; along x every
// contract cell is cut into SPH_SX sort cells: fx = floor(fl(fl(x - xmin) * SPH_SX inv_ell)).  Scaling by a power
// of two is exact, so fx >> 2 is the contract cell coordinate of R1 bit for bit.  The sorted arrays are ordered by
// (z, y, fx, original id); a stencil row's candidates for one particle are then ONE contiguous range
// [f0, f1] of sort cells around the particle, trimmed to the chord of the cut-off sphere in that row
// (stencil_row): ~250 candidates per particle instead of the ~475 of the full 27 contract cells.
__device__ __forceinline__ float fine_coord(float x, float xmin, float inv_ell4)
{
    return __fmul_rn(__fsub_rn(x, xmin), inv_ell4);
}
__device__ __forceinline__ int fine_cell(float u4, int nfx)
{
    int c = (int)floorf(u4);
    if (!(u4 == u4) || fabsf(u4) > 4e9f) c = 0;
    return min(max(c, 0), nfx - 1);
}

// Canonical squared distance (R1): d2 = fma(dz,dz, fma(dy,dy, fl(dx*dx))).
__device__ __forceinline__ float dist2(float dx, float dy, float dz)
{
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

__device__ __forceinline__ uint64_t mix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__device__ __forceinline__ float warp_max(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ int warp_max_i(int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
