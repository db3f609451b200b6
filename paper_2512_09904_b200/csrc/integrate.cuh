// integrate.cuh -- time stepping and reductions (steps a1, a6, a7, a11 of DESIGN.md section 2):
// device-resident clock and dt criteria (Eq. 25), rigid wall kinematics
// (PAPER.md:276, :336), the own-particle half steps of the position-Verlet scheme (R7), and the
// read-back helpers that put fields into original particle order.
#pragma once
#include "common.cuh"

// ---------------------------------------------------------------------------------------------
// a6  control kernel, one thread, first launch of every acoustic step.
//  - closes the previous step's reductions (max |v| from the kick, torque)
//  - decides whether the neighbour configuration is rebuilt (rebuild_every K, or Eq. 25 l.1 / R14)
//  - on rebuild: advances the body angles to the present time, dt_ad = CFL_ad min(h/|v|max, h^2/nu)
//  - dt = dt_fixed or CFL_ac h / (c0 + |v|max), truncated to hit the advection step (R14)
// ---------------------------------------------------------------------------------------------
// `cond`: when the step runs as a CUDA graph, the rebuild chain is the body of a conditional IF node and this kernel
// sets its condition (use_cond = 1); otherwise the rebuild kernels are launched predicated on c.rebuild.
__global__ void k_control(Clock* clk, int hydro, cudaGraphConditionalHandle cond, int use_cond)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    Clock& c = *clk;
    if (hydro && c.steps > 0) {
        c.vmax = sqrtf(__uint_as_float(c.vmax2_bits));
    }
    c.vmax2_bits = 0u;
    c.work_A = 0u; c.work_B = 0u;
    double ur = c.u_ref < 0.0 ? 0.1 * c.c0 : c.u_ref;
    double vm = (double)c.vmax > ur ? (double)c.vmax : ur;
    int due = !c.have_config;
    if (c.rebuild_every >= 1) due |= (c.since_rebuild >= c.rebuild_every);
    else due |= (c.elapsed >= c.dt_ad);
    c.rebuild = due;
    if (due) {
        double dtk = c.t - c.t_kin;
        for (int b = 0; b < SPH_MAXB; ++b) {
            c.body[b].theta += c.body[b].omega * dtk;
            c.body[b].cs = cos(c.body[b].theta);
            c.body[b].sn = sin(c.body[b].theta);
        }
        c.t_kin = c.t;
        double a = c.h / vm, b2 = c.nu > 0.0 ? c.h * c.h / c.nu : a;
        c.dt_ad = c.cfl_ad * (a < b2 ? a : b2);
        if (c.have_config) c.last_adv_steps = c.since_rebuild;       // (kept across sph_set_state, which only drops the configuration)
        c.elapsed = 0.0; c.since_rebuild = 0; c.rebuilds++; c.have_config = 1;
        for (int b = 0; b < SPH_MAXB; ++b) for (int d = 0; d < 3; ++d) c.torque_visc[b][d] = 0.0;      // R26: re-summed by this step
    }
    double dt;
    if (c.dt_fixed > 0.0) dt = c.dt_fixed;
    else {
        dt = c.cfl_ac * c.h / (c.c0 + vm);
        if (c.rebuild_every < 1) { double rem = c.dt_ad - c.elapsed; if (rem < dt) dt = rem; }
        // Eq. 26: the explicit thermal step is bounded by dt_T; without hydrodynamics (static particles, heat
        // only) there is no acoustic criterion to obey and the step IS dt_T
        if (c.dt_T > 0.0 && (!hydro || dt > c.dt_T)) dt = c.dt_T;
    }
    c.dt = dt; c.dt_f = (float)dt;
    for (int b = 0; b < SPH_MAXB; ++b) for (int d = 0; d < 3; ++d) c.torque[b][d] = 0.0;
    if (use_cond) {
        cudaGraphSetConditional(cond, due ? 1u : 0u);
        if (due) c.graph_rebuilds++;
    }
}

// end-of-step bookkeeping (one thread of k_finish: nothing else in that kernel reads these fields, and the torque sums of the
// step are complete since sweep A)
__device__ __forceinline__ void clock_advance(Clock& c)
{
    c.t += c.dt; c.elapsed += c.dt; c.steps++; c.since_rebuild++;
    for (int b = 0; b < SPH_MAXB; ++b) for (int d = 0; d < 3; ++d) c.torque_done[b][d] = c.torque[b][d] + c.torque_visc[b][d];
}

// ---------------------------------------------------------------------------------------------
// a1  wall kinematics: r_w = o_b + R(a_b, theta_b)(r_ref - o_b), n_w = R n_ref (Rodrigues), fp64
// rotation of the fp32 reference arrays, rounded once to fp32.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_wall_kinematics(int n, const float4* __restrict__ ref_pos, const float4* __restrict__ ref_nrm,
                                                          const int* __restrict__ body, float4* __restrict__ wpos, float4* __restrict__ wnrm,
                                                          Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= n) return;
    const BodyD& bd = clk->body[body[w]];
    float4 rp = ref_pos[w], rn = ref_nrm[w];
    if (bd.theta == 0.0) { wpos[w] = rp; wnrm[w] = rn; return; }
    const double ax = bd.axis[0], ay = bd.axis[1], az = bd.axis[2], cs = bd.cs, sn = bd.sn;
    {
        double px = (double)rp.x - bd.origin[0], py = (double)rp.y - bd.origin[1], pz = (double)rp.z - bd.origin[2];
        double ap = ax * px + ay * py + az * pz;
        double cx = ay * pz - az * py, cy = az * px - ax * pz, cz = ax * py - ay * px;
        wpos[w] = make_float4((float)(bd.origin[0] + px * cs + cx * sn + ax * ap * (1.0 - cs)),
                              (float)(bd.origin[1] + py * cs + cy * sn + ay * ap * (1.0 - cs)),
                              (float)(bd.origin[2] + pz * cs + cz * sn + az * ap * (1.0 - cs)), 0.f);
    }
    {
        double px = rn.x, py = rn.y, pz = rn.z;
        double ap = ax * px + ay * py + az * pz;
        double cx = ay * pz - az * py, cy = az * px - ax * pz, cz = ax * py - ay * px;
        wnrm[w] = make_float4((float)(px * cs + cx * sn + ax * ap * (1.0 - cs)),
                              (float)(py * cs + cy * sn + ay * ap * (1.0 - cs)),
                              (float)(pz * cs + cz * sn + az * ap * (1.0 - cs)), 0.f);
    }
}

// ---------------------------------------------------------------------------------------------
// a7  first half step (own particle): rho^{n+1/2} = rho^n + dt/2 (drho/dt)^saved ; r += dt/2 v
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_pre(int n, float4* __restrict__ A, const float4* __restrict__ B, float4* __restrict__ posc, const Clock* clk)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float hdt = 0.5f * clk->dt_f;
    float4 pc = posc[i];
    const float4 b = B[i];
    reinterpret_cast<float*>(A + i)[3] += hdt * pc.w;
    pc.x += hdt * b.x; pc.y += hdt * b.y; pc.z += hdt * b.z;
    posc[i] = pc;
}

// ---------------------------------------------------------------------------------------------
// a11  second half (own particle): rho^{n+1} = rho^{n+1/2} + dt/2 drho/dt (saved for the next
// step); T^{n+1} = T^n + dt dT/dt (forward Euler, R11)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_finish(int n, int hydro, float4* __restrict__ A, float4* __restrict__ B, float4* __restrict__ posc,
                                                 const float2* __restrict__ rates, Clock* clk)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    const float dt = clk->dt_f;
    if (i == 0) clock_advance(*clk);                 // t, elapsed, counters; torque of the completed step latched for sph_get_torque
    if (i >= n) return;
    const float2 r = rates[i];
    if (hydro) {
        reinterpret_cast<float*>(A + i)[3] += 0.5f * dt * r.x;
        reinterpret_cast<float*>(posc + i)[3] = r.x;
    }
    reinterpret_cast<float*>(B + i)[3] += dt * r.y;
}

// ---------------------------------------------------------------------------------------------
// load: caller AoS arrays -> device state in original order (sorted index = original index)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_init_fluid(int n, const float* __restrict__ pos, const float* __restrict__ vel, const float* __restrict__ rho,
                                                     const float* __restrict__ T, float rho0, float T_ref,
                                                     float4* __restrict__ posc, float4* __restrict__ A, float4* __restrict__ B, uint32_t* __restrict__ orig,
                                                     Clock* clk)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    float v2 = 0.f;
    if (i < n) {
        float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
        float vx = vel ? vel[3 * i] : 0.f, vy = vel ? vel[3 * i + 1] : 0.f, vz = vel ? vel[3 * i + 2] : 0.f;
        float drho = rho ? rho[i] - rho0 : 0.f;
        float th = T ? T[i] - T_ref : 0.f;
        posc[i] = make_float4(x, y, z, 0.f);
        A[i] = make_float4(x, y, z, drho);
        B[i] = make_float4(vx, vy, vz, th);
        orig[i] = (uint32_t)i;
        v2 = vx * vx + vy * vy + vz * vz;
    }
    v2 = warp_max(v2);
    if ((threadIdx.x & 31) == 0 && v2 > 0.f) atomicMax(&clk->vmax2_bits, __float_as_uint(v2));
}

// sph_set_state: caller-order arrays -> the sorted records (sorted slot s holds original particle orig[s]); NULL keeps a quantity
__global__ void __launch_bounds__(256) k_set_state(int n, const float* __restrict__ pos, const float* __restrict__ vel, const float* __restrict__ rho,
                                                    const float* __restrict__ T, float rho0, float T_ref, const uint32_t* __restrict__ orig,
                                                    float4* __restrict__ posc, float4* __restrict__ A, float4* __restrict__ B, Clock* clk)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    float v2 = 0.f;
    unsigned int moved = 0u;
    if (s < n) {
        const size_t o = orig[s];
        if (pos) {
            float4 pc = posc[s];
            const float x = pos[3 * o], y = pos[3 * o + 1], z = pos[3 * o + 2];
            if (x != pc.x || y != pc.y || z != pc.z) moved = 1u;         // (a NaN counts as moved)
            pc.x = x; pc.y = y; pc.z = z;
            posc[s] = pc;
        }
        if (rho) reinterpret_cast<float*>(A + s)[3] = rho[o] - rho0;
        float4 b = B[s];
        if (vel) { b.x = vel[3 * o]; b.y = vel[3 * o + 1]; b.z = vel[3 * o + 2]; }
        if (T) b.w = T[o] - T_ref;
        if (vel || T) B[s] = b;
        v2 = b.x * b.x + b.y * b.y + b.z * b.z;
    }
    v2 = warp_max(v2);
    if ((threadIdx.x & 31) == 0 && v2 > 0.f) atomicMax(&clk->vmax2_bits, __float_as_uint(v2));
    if (__any_sync(0xffffffffu, moved != 0u) && (threadIdx.x & 31) == 0) atomicOr(&clk->state_moved, 1u);
}

// around k_set_state.  begin = 1: forget the max |v|^2 of the last kick (k_set_state reduces over all particles, new or kept).
// begin = 0: the next step rebuilds IF a position has changed; |v|max of Eq. 25 is that of the state as it now stands (k_control takes it from the bits
// once a step has been taken, from Clock.vmax before the first step)
__global__ void k_state_changed(Clock* clk, int begin)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    if (begin) { clk->vmax2_bits = 0u; clk->state_moved = 0u; return; }
    clk->vmax = sqrtf(__uint_as_float(clk->vmax2_bits));
    if (!clk->state_moved) return;           // every position came back bit for bit: the neighbour configuration stands
    // the advection step that this upload cuts short had `since_rebuild` acoustic steps: a host loop that moves particles at every
    // step uses each neighbour configuration once, and k_build_tiles then leaves the list re-ordering out (pair.cuh: bank_order_one)
    if (clk->have_config && clk->since_rebuild > 0) clk->last_adv_steps = clk->since_rebuild;
    clk->have_config = 0;
}

// sph_set_materials: {m, k, cp, 0} per particle in original order; NULL arrays take the uniform values
__global__ void __launch_bounds__(256) k_set_materials(int n, const float* __restrict__ m, const float* __restrict__ k, const float* __restrict__ cp,
                                                        float m0, float k0, float cp0, float4* __restrict__ mat)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) mat[i] = make_float4(m ? m[i] : m0, k ? k[i] : k0, cp ? cp[i] : cp0, 0.f);
}

// sph_load_particles with DEVICE buffers: body indices outside [0, n_bodies) raise a flag the host reads after the load's
// synchronisation (HOST buffers are checked on the host while the copies are in flight)
__global__ void __launch_bounds__(256) k_check_body(int n, const int* __restrict__ body, int n_bodies, unsigned int* __restrict__ bad)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && (body[i] < 0 || body[i] >= n_bodies)) atomicOr(bad, 1u);
}

__global__ void k_init_vmax(Clock* clk)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) { clk->vmax = sqrtf(__uint_as_float(clk->vmax2_bits)); clk->vmax2_bits = 0u; }
}

__global__ void __launch_bounds__(256) k_init_wall(int n, const float* __restrict__ pos, const float* __restrict__ nrm, const float* __restrict__ T,
                                                    float T_ref, float4* __restrict__ ref_pos, float4* __restrict__ ref_nrm,
                                                    float4* __restrict__ wpos, float4* __restrict__ wnrm, float* __restrict__ Tw)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 p = make_float4(pos[3 * i], pos[3 * i + 1], pos[3 * i + 2], 0.f);
    float4 q = make_float4(nrm[3 * i], nrm[3 * i + 1], nrm[3 * i + 2], 0.f);
    ref_pos[i] = p; ref_nrm[i] = q; wpos[i] = p; wnrm[i] = q;
    Tw[i] = T ? T[i] - T_ref : 0.f;
}

// ---------------------------------------------------------------------------------------------
// read-back in original order.  what: see the switch.
// ---------------------------------------------------------------------------------------------
enum { X_POS = 0, X_VEL, X_RHO, X_P, X_T, X_ACC, X_DRHO_DT, X_DT_DT, X_CELL, X_NCOUNT, X_DRHO, X_DRHO_SAVED, X_THETA, X_FS_REGION };

__global__ void __launch_bounds__(256) k_extract(DevParams P, int what, float T_ref, const float4* __restrict__ posc, const float4* __restrict__ A,
                                                  const float4* __restrict__ B, const float4* __restrict__ acc, const float2* __restrict__ rates,
                                                  const uint32_t* __restrict__ ncnt, const unsigned char* __restrict__ fs_region, const uint32_t* __restrict__ orig,
                                                  void* __restrict__ out)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.n_f) return;
    const size_t o = orig[s];
    float* of = reinterpret_cast<float*>(out);
    switch (what) {
    case X_POS: { float4 p = posc[s]; of[3 * o] = p.x; of[3 * o + 1] = p.y; of[3 * o + 2] = p.z; break; }
    case X_VEL: { float4 b = B[s]; of[3 * o] = b.x; of[3 * o + 1] = b.y; of[3 * o + 2] = b.z; break; }
    case X_RHO: of[o] = P.rho0 + A[s].w; break;
    case X_P: of[o] = P.c0sq * A[s].w; break;
    case X_T: of[o] = T_ref + B[s].w; break;
    case X_ACC: { float4 a = acc[s]; of[3 * o] = a.x; of[3 * o + 1] = a.y; of[3 * o + 2] = a.z; break; }
    case X_DRHO_DT: of[o] = rates[s].x; break;
    case X_DT_DT: of[o] = rates[s].y; break;
    case X_DRHO: of[o] = A[s].w; break;
    case X_DRHO_SAVED: of[o] = posc[s].w; break;
    case X_THETA: of[o] = B[s].w; break;
    case X_FS_REGION: reinterpret_cast<uint32_t*>(out)[o] = (P.flags & F_FREE_SURFACE_LOCAL) ? (uint32_t)fs_region[s] : 0u; break;
    case X_CELL: {
        float4 a = A[s]; unsigned int err = 0;
        int* oi = reinterpret_cast<int*>(out);
        oi[3 * o] = cell_coord(a.x, P.xmin[0], P.inv_ell, P.ng[0], err);
        oi[3 * o + 1] = cell_coord(a.y, P.xmin[1], P.inv_ell, P.ng[1], err);
        oi[3 * o + 2] = cell_coord(a.z, P.xmin[2], P.inv_ell, P.ng[2], err);
        break; }
    case X_NCOUNT: { uint32_t c = ncnt[s]; uint32_t* ou = reinterpret_cast<uint32_t*>(out); ou[2 * o] = c & 0xffffu; ou[2 * o + 1] = c >> 16; break; }
    default: break;
    }
}

__global__ void __launch_bounds__(256) k_extract_wall(int n, const float4* __restrict__ src, float* __restrict__ out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 p = src[i];
    out[3 * i] = p.x; out[3 * i + 1] = p.y; out[3 * i + 2] = p.z;
}

// wall scalars in original wall order: what = 1: T_w = T_ref + wT (kept in original order); 0: dT_w/dt of the last step
// (sorted order -> original through worig; zero when no body evolves)
__global__ void __launch_bounds__(256) k_extract_wall_scalar(int n, int what, float T_ref, const float* __restrict__ wT, const float* __restrict__ wrate,
                                                             const uint32_t* __restrict__ worig, int have_rate, float* __restrict__ out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (what == 1) out[i] = T_ref + wT[i];
    else out[worig[i]] = have_rate ? wrate[i] : 0.0f;
}

// ---------------------------------------------------------------------------------------------
// Particle relaxation by a constant background pressure, Eq. 6-9 (reading R24).  One step =
// k_relax_begin -> rebuild chain (lists and the fp64 gradient sums G_i = dx^3 sum_j grad_i W_ij over fluid and wall
// neighbours, no density re-initialisation) -> k_relax_force (F_p,i = -(2 p0 / rho0) G_i, Eq. 7 with V = dx^3,
// m = rho0 dx^3; max |F_p|^2) -> k_relax_move (dt^2 = h / (16 max |F_p|), Eq. 8; r += F_p dt^2 / 2, Eq. 9).
// ---------------------------------------------------------------------------------------------
__global__ void k_relax_begin(Clock* clk)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) { clk->rebuild = 1; clk->relax_f2_bits = 0u; }
}
__global__ void k_relax_end(Clock* clk)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) { clk->rebuild = 0; clk->have_config = 0; }
}
__global__ void __launch_bounds__(256) k_relax_force(int n, float c /* -2 p0 / rho0 */, const float4* __restrict__ G, Clock* clk)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    float f2 = 0.f;
    if (i < n) {
        const float4 g = G[i];
        const float fx = c * g.x, fy = c * g.y, fz = c * g.z;
        f2 = fx * fx + fy * fy + fz * fz;
    }
    f2 = warp_max(f2);
    if ((threadIdx.x & 31) == 0 && f2 > 0.f) atomicMax(&clk->relax_f2_bits, __float_as_uint(f2));
}
__global__ void __launch_bounds__(256) k_relax_move(int n, float c, float h, const float4* __restrict__ G, float4* __restrict__ posc, const Clock* clk)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float fmax = sqrtf(__uint_as_float(clk->relax_f2_bits));
    if (!(fmax > 0.f)) return;
    const float half_dt2 = 0.5f * 0.0625f * h / fmax;          // dt = 0.25 sqrt(h / fmax)
    const float4 g = G[i];
    float4 p = posc[i];
    p.x = fmaf(half_dt2, c * g.x, p.x); p.y = fmaf(half_dt2, c * g.y, p.y); p.z = fmaf(half_dt2, c * g.z, p.z);
    posc[i] = p;
}

// average lubricant temperature (Fig. 10): sum of theta = T - T_ref over the fluid particles in fp64
// (warp shuffle -> one atomic per warp); the host divides by n and adds T_ref
__global__ void __launch_bounds__(256) k_sum_theta(int n, const float4* __restrict__ B, double* __restrict__ out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    double s = i < n ? (double)B[i].w : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0 && s != 0.0) atomicAdd(out, s);
}
