// sweeps.cuh -- neighbour-pair summations (steps a5, a8, a10 of DESIGN.md section 2).
// One thread per sorted fluid particle i; a warp walks the 32 neighbour lists of its tile row by
// row (coalesced 128-byte list loads), gathers the neighbour records {x,y,z,drho} / {v,T} through
// L1/L2 and accumulates in registers.  Geometry comes from the positions frozen at the last
// rebuild.  fp32 arithmetic; density enters as drho = rho - rho0 so that
// p = c0^2 drho carries full fp32 precision.
#pragma once
#include "common.cuh"

struct PairGeom { float dx, dy, dz, rinv, r, F; };

// F = W'(r)/r = CF (1 - q/2)^3 for the 3-D Wendland C2 kernel (R2), q = r/h.
__device__ __forceinline__ PairGeom pair_geom(const DevParams& P, float4 ai, float4 aj)
{
    PairGeom g;
    g.dx = ai.x - aj.x; g.dy = ai.y - aj.y; g.dz = ai.z - aj.z;
    float d2 = dist2(g.dx, g.dy, g.dz);
    g.rinv = rsqrtf(d2);
    g.r = d2 * g.rinv;
    float t = fmaxf(1.0f - g.r * P.half_inv_h, 0.0f);
    g.F = P.CF * t * t * t;
    return g;
}

// ---------------------------------------------------------------------------------------------
// a5  density re-initialisation, Eq. 14-15, reading R12.  The kernel sum is
// taken in fp64: rho0 (sigma/sigma0 - 1) is a small difference of O(1) sums, and its fp32
// rounding would enter the pressure at 1e-4 relative.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double W_f64(double d2, double inv_h, double CW)
{
    double q = sqrt(d2) * inv_h;
    double s = 1.0 - 0.5 * q;
    if (s <= 0.0) return 0.0;
    double s2 = s * s;
    return CW * s2 * s2 * (1.0 + 2.0 * q);
}

__global__ void __launch_bounds__(128) k_density_reinit(DevParams P, double inv_h, double CW, double sigma0, double rho0,
                                                         float4* __restrict__ A, const float4* __restrict__ WA,
                                                         const uint32_t* __restrict__ list_f, const uint32_t* __restrict__ list_w,
                                                         const uint32_t* __restrict__ ncnt, Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.n_f) return;
    const int lane = threadIdx.x & 31;
    const size_t tile = (size_t)(i >> 5);
    const uint32_t* lf = list_f + tile * (size_t)P.KF * SPH_TILE + lane;
    const uint32_t* lw = list_w + tile * (size_t)P.KW * SPH_TILE + lane;
    const float4 ai = A[i];
    const uint32_t c = ncnt[i];
    const int nf = c & 0xffffu, nw = c >> 16;
    double sig = CW;                                   // W(0)
    for (int k = 0; k < nf; ++k) {
        float4 aj = ldg4(A + lf[(size_t)k * SPH_TILE]);
        double dx = (double)ai.x - (double)aj.x, dy = (double)ai.y - (double)aj.y, dz = (double)ai.z - (double)aj.z;
        sig += W_f64(dx * dx + dy * dy + dz * dz, inv_h, CW);
    }
    for (int k = 0; k < nw; ++k) {
        float4 aj = ldg4(WA + lw[(size_t)k * SPH_TILE]);
        double dx = (double)ai.x - (double)aj.x, dy = (double)ai.y - (double)aj.y, dz = (double)ai.z - (double)aj.z;
        sig += W_f64(dx * dx + dy * dy + dz * dz, inv_h, CW);
    }
    float dn = (float)(rho0 * (sig - sigma0) / sigma0);
    float d = (P.flags & F_FREE_SURFACE) ? fmaxf(ai.w, dn) : dn;
    // only the .w lane changes; neighbours read .xyz of A concurrently, never .w, in this kernel
    reinterpret_cast<float*>(A + i)[3] = d;
}

// ---------------------------------------------------------------------------------------------
// a8 + a9  sweep A: momentum equation (Eq. 10 l.2) with the Riemann pressure of
// Eq. 12 (:114), wall forces of Eq. 18-19 (:148-155), then the kick v += dt a and the second-half
// drift r += dt/2 v (R7).  Also: max |v|^2 for Eq. 25 and the per-body torque partials (R15).
//   a_i = g - 2 sum_j (V_j/rho_i) p*_ij F_ij r_ij + 2 sum_j (V_j/rho_i) eta F_ij v_ij
//           - 2 sum_w (V_w/rho_i) p*_iw F_iw r_iw + 2 sum_w (V_w/rho_i) eta F_iw (v_i - v_w)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_sweep_A(DevParams P, const float4* __restrict__ A, const float4* __restrict__ Bc,
                                                  float4* __restrict__ Bn, float4* __restrict__ posc, float4* __restrict__ acc_out,
                                                  const float4* __restrict__ WA,
                                                  const uint32_t* __restrict__ list_f, const uint32_t* __restrict__ list_w,
                                                  const uint32_t* __restrict__ ncnt, Clock* clk)
{
    __shared__ float s_tq[SPH_MAXB * 3];
    __shared__ int s_tq_used;
    if (threadIdx.x < SPH_MAXB * 3) s_tq[threadIdx.x] = 0.0f;
    if (threadIdx.x == 0) s_tq_used = 0;
    __syncthreads();

    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < P.n_f;
    const int ii = valid ? i : P.n_f - 1;
    const int lane = threadIdx.x & 31;
    const size_t tile = (size_t)(ii >> 5);
    const uint32_t* lf = list_f + tile * (size_t)P.KF * SPH_TILE + lane;
    const uint32_t* lw = list_w + tile * (size_t)P.KW * SPH_TILE + lane;
    const float4 ai = A[ii], bi = Bc[ii];
    const uint32_t c = valid ? ncnt[ii] : 0u;
    const int nf = c & 0xffffu, nw = c >> 16;
    const float dt = clk->dt_f;
    const bool do_p = (P.flags & F_PRESSURE) != 0, do_v = (P.flags & F_VISCOUS) != 0;

    const float rho_i = P.rho0 + ai.w, p_i = P.c0sq * ai.w;
    const float inv_rho_i = 1.0f / rho_i;
    const float kp = do_p ? -2.0f * inv_rho_i : 0.0f;          // pressure prefactor, times V p* F
    const float kv = do_v ? 2.0f * inv_rho_i * P.eta : 0.0f;   // viscous prefactor, times V F
    float ax = 0.f, ay = 0.f, az = 0.f;

    const int nf_max = warp_max_i(nf);
#pragma unroll 2
    for (int k = 0; k < nf_max; ++k) {
        if (k < nf) {
            const uint32_t j = lf[(size_t)k * SPH_TILE];
            const float4 aj = ldg4(A + j), bj = ldg4(Bc + j);
            const PairGeom g = pair_geom(P, ai, aj);
            const float vx = bi.x - bj.x, vy = bi.y - bj.y, vz = bi.z - bj.z;
            const float vr = vx * g.dx + vy * g.dy + vz * g.dz;
            const float rho_j = P.rho0 + aj.w, p_j = P.c0sq * aj.w;
            const float du = -vr * g.rinv;                                   // U_L - U_R (Eq. 11)
            const float beta = fminf(3.0f * fmaxf(du, 0.0f), P.c0);          // limiter
            const float rs_inv = 1.0f / (rho_i + rho_j);
            const float pstar = (rho_i * p_j + rho_j * p_i + rho_i * rho_j * beta * du) * rs_inv;   // Eq. 12
            const float VF = P.mass / rho_j * g.F;                           // V_j F_ij
            const float cp = kp * VF * pstar, cv = kv * VF;
            ax += cp * g.dx + cv * vx;
            ay += cp * g.dy + cv * vy;
            az += cp * g.dz + cv * vz;
        }
    }

    // walls: torque accumulated for the body of the current run of wall neighbours
    int cur_b = -1;
    float tqx = 0.f, tqy = 0.f, tqz = 0.f;
    const int nw_max = warp_max_i(nw);
    for (int k = 0; k < nw_max; ++k) {
        if (k < nw) {
            const uint32_t w = lw[(size_t)k * SPH_TILE];
            const float4 wa = ldg4(WA + w);
            const PairGeom g = pair_geom(P, ai, wa);
            const int b = __float_as_int(wa.w);
            const BodyF bd = P.body[b];
            const float px = wa.x - bd.ox, py = wa.y - bd.oy, pz = wa.z - bd.oz;        // r_w - o_b
            const float vwx = bd.wy * pz - bd.wz * py, vwy = bd.wz * px - bd.wx * pz, vwz = bd.wx * py - bd.wy * px;
            const float pR = p_i - rho_i * (P.gx * g.dx + P.gy * g.dy + P.gz * g.dz);     // Eq. 17, r_fw = -r_iw
            const float rhoR = P.rho0 + pR * P.inv_c0sq;
            const float pstar = (rho_i * pR + rhoR * p_i) / (rho_i + rhoR);               // Eq. 19
            const float VF = P.Vw * g.F;
            const float cp = kp * VF * pstar, cv = kv * VF;
            const float fx = cp * g.dx + cv * (bi.x - vwx);
            const float fy = cp * g.dy + cv * (bi.y - vwy);
            const float fz = cp * g.dz + cv * (bi.z - vwz);
            ax += fx; ay += fy; az += fz;
            if (b != cur_b) {
                if (cur_b >= 0) {
                    atomicAdd(&s_tq[cur_b * 3 + 0], tqx); atomicAdd(&s_tq[cur_b * 3 + 1], tqy); atomicAdd(&s_tq[cur_b * 3 + 2], tqz);
                }
                cur_b = b; tqx = tqy = tqz = 0.f;
            }
            // force on the wall particle = -m_i (pair acceleration); moment about o_b
            const float Fx = -P.mass * fx, Fy = -P.mass * fy, Fz = -P.mass * fz;
            tqx += py * Fz - pz * Fy; tqy += pz * Fx - px * Fz; tqz += px * Fy - py * Fx;
        }
    }
    if (cur_b >= 0) {
        atomicAdd(&s_tq[cur_b * 3 + 0], tqx); atomicAdd(&s_tq[cur_b * 3 + 1], tqy); atomicAdd(&s_tq[cur_b * 3 + 2], tqz);
        s_tq_used = 1;
    }

    float v2 = 0.f;
    if (valid) {
        ax += P.gx; ay += P.gy; az += P.gz;
        const float vx = bi.x + dt * ax, vy = bi.y + dt * ay, vz = bi.z + dt * az;      // a9 kick
        Bn[i] = make_float4(vx, vy, vz, bi.w);
        float4 pc = posc[i];
        const float hdt = 0.5f * dt;
        pc.x += hdt * vx; pc.y += hdt * vy; pc.z += hdt * vz;                            // a9 drift
        posc[i] = pc;
        acc_out[i] = make_float4(ax, ay, az, 0.f);
        v2 = vx * vx + vy * vy + vz * vz;
    }
    v2 = warp_max(v2);
    if (lane == 0 && v2 > 0.f) atomicMax(&clk->vmax2_bits, __float_as_uint(v2));
    __syncthreads();
    if (s_tq_used && threadIdx.x < SPH_MAXB * 3) {
        float t = s_tq[threadIdx.x];
        if (t != 0.f) atomicAdd(&clk->torque[threadIdx.x / 3][threadIdx.x % 3], (double)t);
    }
}

// ---------------------------------------------------------------------------------------------
// a10  sweep B: continuity (Eq. 10 l.1; v* of Eq. 13 under R3; wall term R6) and
// heat conduction (Eq. 22; R9-R10), using v^{n+1}, rho^{n+1/2}, T^n.
//   drho_i/dt = 2 rho_i [ sum_j V_j ( rho_j v_ij.e_ij + (p_i - p_j)/c0 ) / (rho_i + rho_j) W'_ij
//                         + sum_w V_w (U*_iw - U_L)(n_w.e_iw) W'_iw ]
//   dT_i/dt   = 1/(rho_i cp) [ 2 k_f sum_j V_j T_ij F_ij + sum_w V_w K_w T_iw F_iw ]
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_sweep_B(DevParams P, const float4* __restrict__ A, const float4* __restrict__ B,
                                                  const float4* __restrict__ WA, const float4* __restrict__ WB,
                                                  const uint32_t* __restrict__ list_f, const uint32_t* __restrict__ list_w,
                                                  const uint32_t* __restrict__ ncnt, float2* __restrict__ rates, Clock* clk)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < P.n_f;
    const int ii = valid ? i : P.n_f - 1;
    const int lane = threadIdx.x & 31;
    const size_t tile = (size_t)(ii >> 5);
    const uint32_t* lf = list_f + tile * (size_t)P.KF * SPH_TILE + lane;
    const uint32_t* lw = list_w + tile * (size_t)P.KW * SPH_TILE + lane;
    const float4 ai = A[ii], bi = B[ii];
    const uint32_t c = valid ? ncnt[ii] : 0u;
    const int nf = c & 0xffffu, nw = c >> 16;
    const bool hydro = (P.flags & F_HYDRO) != 0, thermal = (P.flags & F_THERMAL) != 0;
    const float rho_i = P.rho0 + ai.w, p_i = P.c0sq * ai.w;
    float sr = 0.f, sT = 0.f;

    const int nf_max = warp_max_i(nf);
#pragma unroll 2
    for (int k = 0; k < nf_max; ++k) {
        if (k < nf) {
            const uint32_t j = lf[(size_t)k * SPH_TILE];
            const float4 aj = ldg4(A + j), bj = ldg4(B + j);
            const PairGeom g = pair_geom(P, ai, aj);
            const float rho_j = P.rho0 + aj.w;
            const float VF = P.mass / rho_j * g.F;                            // V_j F_ij
            const float vr = (bi.x - bj.x) * g.dx + (bi.y - bj.y) * g.dy + (bi.z - bj.z) * g.dz;
            // (v_i - v*).e_ij W' = [rho_j v_ij.e_ij + (p_i - p_j)/c0] / (rho_i + rho_j) * F r
            const float num = rho_j * vr * g.rinv + P.c0 * (ai.w - aj.w);     // (p_i - p_j)/c0 = c0 (drho_i - drho_j)
            sr += VF * g.r * num / (rho_i + rho_j);
            sT += VF * (bi.w - bj.w);
        }
    }
    sT *= P.k2f;                                                              // K_ij = 4 k k/(2k) = 2 k_f
    const int nw_max = warp_max_i(nw);
    for (int k = 0; k < nw_max; ++k) {
        if (k < nw) {
            const uint32_t w = lw[(size_t)k * SPH_TILE];
            const float4 wa = ldg4(WA + w), wb = ldg4(WB + w);
            const PairGeom g = pair_geom(P, ai, wa);
            const int b = __float_as_int(wa.w);
            const BodyF bd = P.body[b];
            const float px = wa.x - bd.ox, py = wa.y - bd.oy, pz = wa.z - bd.oz;
            const float vwx = bd.wy * pz - bd.wz * py, vwy = bd.wz * px - bd.wx * pz, vwz = bd.wx * py - bd.wy * px;
            const float UL = -(wb.x * bi.x + wb.y * bi.y + wb.z * bi.z);               // Eq. 16
            const float uw = -(wb.x * vwx + wb.y * vwy + wb.z * vwz);
            const float UR = -UL + 2.0f * uw;                                          // Eq. 17
            const float dpg = rho_i * (P.gx * g.dx + P.gy * g.dy + P.gz * g.dz);       // p_L - p_R (Eq. 17)
            const float pR = p_i - dpg;
            const float rhoR = P.rho0 + pR * P.inv_c0sq;
            const float rs_inv = 1.0f / (rho_i + rhoR);
            const float Ustar = (rho_i * UL + rhoR * UR) * rs_inv + dpg * P.inv_c0 * rs_inv;           // Eq. 12 l.1
            const float ne = (wb.x * g.dx + wb.y * g.dy + wb.z * g.dz) * g.rinv;       // n_w . e_iw
            const float VF = P.Vw * g.F;
            sr += VF * g.r * (Ustar - UL) * ne;                                        // R6
            sT += VF * bd.K * (bi.w - wb.w);
        }
    }
    if (valid) {
        float drho = hydro ? 2.0f * rho_i * sr : 0.0f;
        float dT = thermal ? sT * P.inv_cp / rho_i : 0.0f;
        rates[i] = make_float2(drho, dT);
    }
}
