/*
 * sph_oracle.c -- plain, slow, fp64 CPU oracle for the WCSPH particle-interaction sweep of
 * arxiv/paper_2512_09904.  TEST INFRASTRUCTURE ONLY: it is imported by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs, never by the
 * product path.  It shares no code, header, table or constant generator with the CUDA library
 * (paper_2512_09904_b200/csrc); only the seeded input generators serve both.
 *
 * Every function cites the passage of PAPER.md it follows; readings of silent / ambiguous
 * passages are the R-numbers of DESIGN.md section 3 (taken from SURVEY.md section 8(c)).
 * Gather form everywhere: particle i sums over its neighbours j (fluid) and w (wall); nothing
 * is blocked, fused or reordered beyond the step order of DESIGN.md section 2.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force O(N^2) neighbour sets (P1),
 * kernel normalisation / partition of unity (P2), pairwise momentum conservation (P3), thermal
 * energy conservation (P4), hydrostatic tank (P5), 1-D two-material conduction vs the erfc
 * solution (P6), linear-field consistency of continuity / heat / viscous sums (P7), Riemann
 * signs and limiter (P8), zero viscous force in linear shear (P9), rigid rotation (P10),
 * action-reaction torque (P11), dt formulae (P12), sort invariants (P13); the position-Verlet half steps and the hand-over of
 * the saved rate (I1, I2), the wall part of the density re-initialisation (I3), the wall continuity term in closed form
 * (I4), the acoustic wave speed (I5), the Eq. 26 step bound (I6) in tests/test_oracle_pins_integrator.py; the free-surface
 * region of the re-initialisation (F1-F5, reading R27) in tests/test_oracle_pins_free_surface.py; pairs at zero distance
 * (C1-C3, reading R28) in tests/test_oracle_pins_coincident.py.  tests/oracle_mutations.py
 * applies the one-token mutations those pins name and checks that each pin fails on its mutant.
 * Parity unpinned (the arithmetic is pinned, the choice of reading is fixed by DESIGN.md only): wall p* without limiter (R6),
 * viscous term per acoustic step (R8) or held per advection step by flag (R26: the evaluation point is a reading), u_ref
 * floor (R13), denominator of the contact factor (R22), evolving solid temperature (R23), relaxation without the level set
 * (R24), indicator and threshold of the free-surface region (R27), the limit taken for two particles at the same place (R28).
 *
 * Precision: all state and arithmetic in double, except the two predicates that decide integers
 * (cell coordinate, neighbour membership), which are evaluated in float exactly as DESIGN.md
 * R1 states so that an fp32 device can reproduce the same integers.
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC sph_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_BODIES 8

enum {
    ORC_FREE_SURFACE = 1, ORC_DENSITY_REINIT = 2, ORC_THERMAL = 4, ORC_VISCOUS = 8,
    ORC_HYDRO = 16, ORC_DUAL_CRITERIA = 32, ORC_PRESSURE = 64,
    ORC_VISCOUS_HELD = 128,    /* R26: viscous sums evaluated once per advection step and held (ref [45]) */
    ORC_FREE_SURFACE_LOCAL = 256   /* R27: Eq. 14 only in the identified free-surface region, Eq. 15 elsewhere */
};

typedef struct {
    uint32_t flags;
    int32_t rebuild_every;     /* K >= 1: rebuild every K acoustic steps; 0: dt_ad rule (Eq. 25) */
    int32_t n_bodies;
    int32_t neigh_backend;     /* 0 = cell list, 1 = brute force O(N^2) */
    double dx, h, rho0, c0, nu;
    double g[3];
    double k_f, cp_f;
    double cfl_ac, cfl_ad, u_ref, dt_fixed;
    double domain_min[3], domain_max[3];
    double body_k[ORC_MAX_BODIES];
    double body_rho[ORC_MAX_BODIES], body_cp[ORC_MAX_BODIES];   /* solid density, specific heat (evolving bodies) */
    int32_t body_mode[ORC_MAX_BODIES];                          /* 0: temperature held (R10); 1: evolving (R23) */
    int32_t dim;                                                /* 0 or 3: three-dimensional; 2: planar (R25) */
    double fs_threshold;                                        /* R27: theta of the surface test sigma_i < theta sigma0; 0 -> 0.9 */
} orc_params;

typedef struct {
    orc_params p;
    int64_t n_f, n_w;
    /* fluid state, original order */
    double *r, *v, *rho, *T, *drho_saved, *mass, *k, *cp;
    double *acc, *acc_p, *acc_v, *acc_wp, *acc_wv, *drho_dt, *dT_dt;
    /* wall state */
    double *rw_ref, *nw_ref, *rw, *nw, *Tw, *Fw, *Fw_v, *dTw_dt;
    int32_t *body_w;
    unsigned char *fs_region;         /* R27 / R12: 1 where the last re-initialisation took the max form of Eq. 14 */
    /* configuration frozen at the last rebuild */
    double *r_frz;
    int32_t *cell_f, *cell_w;         /* canonical fp32 cell coordinates, [n][3] */
    int64_t *ff_start, *fw_start;
    int32_t *ff_idx, *fw_idx;
    /* bodies (prescribed rigid rotation) */
    double origin[ORC_MAX_BODIES][3], axis[ORC_MAX_BODIES][3], omega[ORC_MAX_BODIES],
        theta[ORC_MAX_BODIES], torque[ORC_MAX_BODIES][3];
    /* clock */
    double t, t_kin, dt, dt_ad, elapsed, vmax;
    int64_t steps, rebuilds, since_rebuild;
    int have_config;
    int visc_fresh;                   /* R26: this evaluation recomputes the viscous sums (always 1 without ORC_VISCOUS_HELD) */
    double sigma0;
} orc;

/* ---------------------------------------------------------------------------------------------
 * Kernel function.  The paper is silent (only "kernel function W(|r_ij|, h)");
 * BASELINE.json fixes the 3-D Wendland C2 kernel with support 2h (reading R2):
 *   W(r,h) = alpha (1 - q/2)^4 (1 + 2q), q = r/h < 2, alpha = 21 / (16 pi h^3).
 * ------------------------------------------------------------------------------------------- */
double orc_W(double r, double h)
{
    double q = r / h;
    if (q >= 2.0) return 0.0;
    double a = 21.0 / (16.0 * M_PI * h * h * h);
    double s = 1.0 - 0.5 * q;
    return a * s * s * s * s * (1.0 + 2.0 * q);
}

/* dW/dr, the "partial W_ij / partial r_ij" of Eq. 10. */
double orc_dWdr(double r, double h)
{
    double q = r / h;
    if (q >= 2.0) return 0.0;
    double a = 21.0 / (16.0 * M_PI * h * h * h);
    double s = 1.0 - 0.5 * q;
    return -(5.0 * a / h) * q * s * s * s;
}

/* Sum of W over a full cubic lattice of spacing dx including the self term: the constant
 * denominator "sum W_ij^0" of Eq. 14-15 under reading R12. */
double orc_sigma0(double dx, double h)
{
    int m = (int)ceil(2.0 * h / dx) + 1;
    double s = 0.0;
    for (int a = -m; a <= m; ++a)
        for (int b = -m; b <= m; ++b)
            for (int c = -m; c <= m; ++c) {
                double r = dx * sqrt((double)(a * a + b * b + c * c));
                s += orc_W(r, h);
            }
    return s;
}

/* Planar mode (reading R25; the paper's section 3.2 benchmark is two-dimensional): the same
 * Wendland C2 shape with the two-dimensional normalisation alpha = 7 / (4 pi h^2), particle volume dx^2, square-lattice
 * sigma0; all particles share one z and the grid has one cell layer. */
double orc_W2d(double r, double h)
{
    double q = r / h;
    if (q >= 2.0) return 0.0;
    double a = 7.0 / (4.0 * M_PI * h * h);
    double s = 1.0 - 0.5 * q;
    return a * s * s * s * s * (1.0 + 2.0 * q);
}
double orc_dWdr2d(double r, double h)
{
    double q = r / h;
    if (q >= 2.0) return 0.0;
    double a = 7.0 / (4.0 * M_PI * h * h);
    double s = 1.0 - 0.5 * q;
    return -(5.0 * a / h) * q * s * s * s;
}
double orc_sigma0_2d(double dx, double h)
{
    int m = (int)ceil(2.0 * h / dx) + 1;
    double s = 0.0;
    for (int a = -m; a <= m; ++a)
        for (int b = -m; b <= m; ++b) s += orc_W2d(dx * sqrt((double)(a * a + b * b)), h);
    return s;
}
static int orc_planar(const orc_params *p) { return p->dim == 2; }
static double orc_Wd(const orc_params *p, double r, double h) { return orc_planar(p) ? orc_W2d(r, h) : orc_W(r, h); }
static double orc_dWdrd(const orc_params *p, double r, double h) { return orc_planar(p) ? orc_dWdr2d(r, h) : orc_dWdr(r, h); }
static double orc_vol(const orc_params *p) { return orc_planar(p) ? p->dx * p->dx : p->dx * p->dx * p->dx; }

/* Reading R28: two particles at the same place.  The pair terms of Eq. 10-13, 16-22 carry the unit vector
 * e_ij = r_ij / r_ij and the factor W'(r_ij) / r_ij, both 0/0 at r_ij = 0; the paper is silent.  Reading: the limit
 * eps -> 0+ of e_ij = r_ij / (r_ij + eps), i.e. the zero vector, and the finite limit of W'(r)/r, -5 alpha / h^2 for the Wendland C2
 * kernel (W' = -(5 alpha / h) q (1 - q/2)^3).  Such a pair then exchanges no pressure force and no mass flux (both act along
 * e_ij) but still viscous force and heat (both proportional to W'/r).  For r > 0 nothing changes. */
static double orc_inv_r(double r) { return r > 0.0 ? 1.0 / r : 0.0; }
static double orc_Fd(const orc_params *p, double r, double h)
{
    if (r > 0.0) return orc_dWdrd(p, r, h) / r;
    const double a = orc_planar(p) ? 7.0 / (4.0 * M_PI * h * h) : 21.0 / (16.0 * M_PI * h * h * h);
    return -5.0 * a / (h * h);
}

/* ---------------------------------------------------------------------------------------------
 * Integer predicates (reading R1).  Evaluated in float, operation by operation.
 *   cut-off:   rc = (float)(2h);  rc2 = rc*rc (float product)
 *   distance:  d = x_i - x_j per axis (float);  d2 = fmaf(dz,dz, fmaf(dy,dy, dx*dx))
 *   member:    d2 < rc2, j != i
 *   cell:      ell = 2h (1 + 2^-10);  inv = (float)(1/ell);  xmin = (float)domain_min
 *              c = (int)floorf( (float)((x - xmin) * inv) ), clamped to [0, n-1]
 *              n = (int)floorf( ((float)domain_max - xmin) * inv ) + 1
 * ------------------------------------------------------------------------------------------- */
static float orc_rc2(double h)
{
    float rc = (float)(2.0 * h);
    volatile float rc2 = rc * rc;
    return rc2;
}

static int orc_member(const float *a, const float *b, float rc2)
{
    /* x86-64 evaluates float expressions in float (FLT_EVAL_METHOD 0); with -ffp-contract=off
     * the product below is rounded on its own and the two fmaf calls are the only fusions. */
    float dx = a[0] - b[0], dy = a[1] - b[1], dz = a[2] - b[2];
    float xx = dx * dx;
    float d2 = fmaf(dz, dz, fmaf(dy, dy, xx));
    return d2 < rc2;
}

static void orc_grid(const orc_params *p, float xmin[3], float *inv, int n[3])
{
    double ell = 2.0 * p->h * (1.0 + 1.0 / 1024.0);
    *inv = (float)(1.0 / ell);
    for (int d = 0; d < 3; ++d) {
        xmin[d] = (float)p->domain_min[d];
        volatile float ext = (float)p->domain_max[d] - xmin[d];
        volatile float s = ext * (*inv);
        n[d] = (int)floorf(s) + 1;
    }
}

static int orc_cell1(float x, float xmin, float inv, int n, int *outside)
{
    volatile float rel = x - xmin;
    volatile float s = rel * inv;
    int c = (int)floorf(s);
    if (c < 0) { c = 0; *outside = 1; }
    if (c > n - 1) { c = n - 1; *outside = 1; }
    return c;
}

void orc_grid_dims(const orc_params *p, int n[3])
{
    float xmin[3], inv;
    orc_grid(p, xmin, &inv, n);
}

/* order-independent digest of a neighbour set: sum over members of mix64(id + 1), where fluid
 * neighbours use their original index and wall neighbours n_f + original wall index. */
static uint64_t orc_mix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

/* ---------------------------------------------------------------------------------------------
 * life cycle
 * ------------------------------------------------------------------------------------------- */
orc *orc_create(const orc_params *p)
{
    orc *o = (orc *)calloc(1, sizeof(orc));
    if (!o) return NULL;
    o->p = *p;
    for (int b = 0; b < ORC_MAX_BODIES; ++b) { o->axis[b][2] = 1.0; }
    o->sigma0 = orc_planar(p) ? orc_sigma0_2d(p->dx, p->h) : orc_sigma0(p->dx, p->h);
    return o;
}

static void orc_free_arrays(orc *o)
{
    void *ptrs[] = {o->r, o->v, o->rho, o->T, o->drho_saved, o->mass, o->k, o->cp, o->acc,
                    o->acc_p, o->acc_v, o->acc_wp, o->acc_wv, o->drho_dt, o->dT_dt, o->rw_ref,
                    o->nw_ref, o->rw, o->nw, o->Tw, o->Fw, o->body_w, o->r_frz, o->cell_f,
                    o->cell_w, o->ff_start, o->fw_start, o->ff_idx, o->fw_idx, o->dTw_dt, o->Fw_v, o->fs_region};
    for (size_t i = 0; i < sizeof(ptrs) / sizeof(ptrs[0]); ++i) free(ptrs[i]);
}

void orc_destroy(orc *o)
{
    if (!o) return;
    orc_free_arrays(o);
    free(o);
}

static double *dalloc(int64_t n) { return (double *)calloc((size_t)(n > 0 ? n : 1), sizeof(double)); }

/* Inputs: AoS [n][3] float arrays in original order (the same buffers the device path loads).
 * rho_f == NULL -> rho0.  Uniform mass m = rho0 dx^3 and wall volume V_w = dx^3 (PAPER.md:105
 * "V is particle volume, m is the particle mass"; lattice initialisation). */
int orc_load(orc *o, int64_t n_f, const float *pos_f, const float *vel_f, const float *rho_f,
             const float *T_f, int64_t n_w, const float *pos_w, const float *nrm_w,
             const int32_t *body_w, const float *T_w)
{
    orc_free_arrays(o);
    o->n_f = n_f; o->n_w = n_w;
    o->r = dalloc(3 * n_f); o->v = dalloc(3 * n_f); o->rho = dalloc(n_f); o->T = dalloc(n_f);
    o->drho_saved = dalloc(n_f); o->mass = dalloc(n_f); o->k = dalloc(n_f); o->cp = dalloc(n_f);
    o->acc = dalloc(3 * n_f); o->acc_p = dalloc(3 * n_f); o->acc_v = dalloc(3 * n_f);
    o->acc_wp = dalloc(3 * n_f); o->acc_wv = dalloc(3 * n_f);
    o->drho_dt = dalloc(n_f); o->dT_dt = dalloc(n_f);
    o->rw_ref = dalloc(3 * n_w); o->nw_ref = dalloc(3 * n_w); o->rw = dalloc(3 * n_w);
    o->nw = dalloc(3 * n_w); o->Tw = dalloc(n_w); o->Fw = dalloc(3 * n_w); o->Fw_v = dalloc(3 * n_w); o->dTw_dt = dalloc(n_w);
    o->body_w = (int32_t *)calloc((size_t)(n_w > 0 ? n_w : 1), sizeof(int32_t));
    o->r_frz = dalloc(3 * n_f);
    o->fs_region = (unsigned char *)calloc((size_t)(n_f > 0 ? n_f : 1), 1);
    o->cell_f = (int32_t *)calloc((size_t)(3 * n_f + 1), sizeof(int32_t));
    o->cell_w = (int32_t *)calloc((size_t)(3 * n_w + 1), sizeof(int32_t));
    o->ff_start = (int64_t *)calloc((size_t)(n_f + 1), sizeof(int64_t));
    o->fw_start = (int64_t *)calloc((size_t)(n_f + 1), sizeof(int64_t));
    o->ff_idx = NULL; o->fw_idx = NULL;
    double m = o->p.rho0 * orc_vol(&o->p);
    for (int64_t i = 0; i < n_f; ++i) {
        for (int d = 0; d < 3; ++d) {
            o->r[3 * i + d] = pos_f[3 * i + d];
            o->v[3 * i + d] = vel_f ? vel_f[3 * i + d] : 0.0;
        }
        o->rho[i] = rho_f ? (double)rho_f[i] : o->p.rho0;
        o->T[i] = T_f ? (double)T_f[i] : 0.0;
        o->mass[i] = m; o->k[i] = o->p.k_f; o->cp[i] = o->p.cp_f;
    }
    for (int64_t w = 0; w < n_w; ++w) {
        for (int d = 0; d < 3; ++d) {
            o->rw_ref[3 * w + d] = o->rw[3 * w + d] = pos_w[3 * w + d];
            o->nw_ref[3 * w + d] = o->nw[3 * w + d] = nrm_w[3 * w + d];
        }
        o->body_w[w] = body_w ? body_w[w] : 0;
        o->Tw[w] = T_w ? (double)T_w[w] : 0.0;
    }
    o->t = o->t_kin = o->dt = o->dt_ad = o->elapsed = 0.0;
    o->steps = o->rebuilds = o->since_rebuild = 0;
    o->have_config = 0;
    for (int b = 0; b < ORC_MAX_BODIES; ++b) {
        o->theta[b] = 0.0;
        o->torque[b][0] = o->torque[b][1] = o->torque[b][2] = 0.0;
    }
    return 0;
}

/* optional per-particle materials (Eq. 20-22 are written for general k_i, k_j; the two-slab
 * benchmark of section 3.2, needs them).  NULL leaves a property unchanged. */
int orc_set_materials(orc *o, const double *mass, const double *k, const double *cp)
{
    for (int64_t i = 0; i < o->n_f; ++i) {
        if (mass) o->mass[i] = mass[i];
        if (k) o->k[i] = k[i];
        if (cp) o->cp[i] = cp[i];
    }
    return 0;
}

int orc_set_state(orc *o, const double *r, const double *v, const double *rho, const double *T,
                  const double *drho_saved)
{
    int64_t n = o->n_f;
    if (r) memcpy(o->r, r, sizeof(double) * 3 * n);
    if (v) memcpy(o->v, v, sizeof(double) * 3 * n);
    if (rho) memcpy(o->rho, rho, sizeof(double) * n);
    if (T) memcpy(o->T, T, sizeof(double) * n);
    if (drho_saved) memcpy(o->drho_saved, drho_saved, sizeof(double) * n);
    o->have_config = 0;
    return 0;
}

/* after orc_set_state in the MIDDLE of an advection step: keep the neighbour configuration, the frozen geometry and the held
 * viscous sums (R26) that this oracle built at its last rebuild, so that a state handed over between two rebuilds is
 * advanced as the step after it would be.  No arithmetic of the method; returns -1 if there is no configuration. */
int orc_keep_config(orc *o)
{
    if (!o->ff_start) return -1;
    o->have_config = 1;
    return 0;
}

/* move the clock (not the state) to time t: a state taken over at time t (orc_set_state) then sees the bodies
 * rotated to theta_b = omega_b t at its first rebuild.  No arithmetic of the method changes. */
int orc_set_time(orc *o, double t)
{
    o->t = t;
    return 0;
}

int orc_set_kinematics(orc *o, int body, const double origin[3], const double axis[3], double omega)
{
    if (body < 0 || body >= ORC_MAX_BODIES) return -1;
    double n = sqrt(axis[0] * axis[0] + axis[1] * axis[1] + axis[2] * axis[2]);
    if (!(n > 0.0)) return -1;
    /* bring every body's angle up to the present time with the speeds valid so far */
    for (int b = 0; b < ORC_MAX_BODIES; ++b) o->theta[b] += o->omega[b] * (o->t - o->t_kin);
    o->t_kin = o->t;
    for (int d = 0; d < 3; ++d) { o->origin[body][d] = origin[d]; o->axis[body][d] = axis[d] / n; }
    o->omega[body] = omega;
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * a1  wall kinematics: prescribed rigid rotation about a fixed axis.
 *     theta_b += omega_b (t - t_kin);  r_w = o_b + R(a_b, theta_b)(r_ref - o_b);  n_w = R n_ref
 *     (Rodrigues' formula);  v_w = omega_b a_b x (r_w - o_b) is evaluated where it is used.
 * ------------------------------------------------------------------------------------------- */
static void rodrigues(const double a[3], double th, const double p[3], double out[3])
{
    double c = cos(th), s = sin(th);
    double ap = a[0] * p[0] + a[1] * p[1] + a[2] * p[2];
    double cr[3] = {a[1] * p[2] - a[2] * p[1], a[2] * p[0] - a[0] * p[2], a[0] * p[1] - a[1] * p[0]};
    for (int d = 0; d < 3; ++d) out[d] = p[d] * c + cr[d] * s + a[d] * ap * (1.0 - c);
}

static void orc_wall_kinematics(orc *o)
{
    double dtk = o->t - o->t_kin;
    for (int b = 0; b < ORC_MAX_BODIES; ++b) o->theta[b] += o->omega[b] * dtk;
    o->t_kin = o->t;
    for (int64_t w = 0; w < o->n_w; ++w) {
        int b = o->body_w[w];
        if (o->omega[b] == 0.0 && o->theta[b] == 0.0) continue;
        double p[3], q[3];
        for (int d = 0; d < 3; ++d) p[d] = o->rw_ref[3 * w + d] - o->origin[b][d];
        rodrigues(o->axis[b], o->theta[b], p, q);
        /* R21: wall positions and normals are fp32 particle state like every array of the C ABI: the rotation is
         * evaluated in double and its result rounded once to float, so that the pair geometry uses the very
         * position the fp32 neighbour predicate (R1) sees */
        for (int d = 0; d < 3; ++d) o->rw[3 * w + d] = (double)(float)(o->origin[b][d] + q[d]);
        rodrigues(o->axis[b], o->theta[b], &o->nw_ref[3 * w], q);
        for (int d = 0; d < 3; ++d) o->nw[3 * w + d] = (double)(float)q[d];
    }
}

static void wall_velocity(const orc *o, int64_t w, double vw[3])
{
    int b = o->body_w[w];
    const double *a = o->axis[b];
    double om = o->omega[b];
    double p[3];
    for (int d = 0; d < 3; ++d) p[d] = o->rw[3 * w + d] - o->origin[b][d];
    vw[0] = om * (a[1] * p[2] - a[2] * p[1]);
    vw[1] = om * (a[2] * p[0] - a[0] * p[2]);
    vw[2] = om * (a[0] * p[1] - a[1] * p[0]);
}

/* ---------------------------------------------------------------------------------------------
 * a2-a4  neighbour configuration ("neighbor lists and kernel-related quantities are updated
 * based on the advection time step").  The oracle keeps original order and stores
 * the sets as CSR lists; membership is the R1 predicate.  Two back-ends: all pairs, and the
 * 27-cell stencil of the R1 grid.  Returns 1 if some particle lay outside the grid.
 * ------------------------------------------------------------------------------------------- */
typedef struct { int32_t *v; int64_t n, cap; } ivec;
static void ipush(ivec *a, int32_t x)
{
    if (a->n == a->cap) { a->cap = a->cap ? 2 * a->cap : 64; a->v = (int32_t *)realloc(a->v, sizeof(int32_t) * (size_t)a->cap); }
    a->v[a->n++] = x;
}
static int cmp_i32(const void *a, const void *b)
{
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

static int orc_build_config(orc *o)
{
    const int64_t nf = o->n_f, nw = o->n_w;
    float xmin[3], inv; int ng[3];
    orc_grid(&o->p, xmin, &inv, ng);
    const float rc2 = orc_rc2(o->p.h);
    float *pf = (float *)malloc(sizeof(float) * (size_t)(3 * nf + 3));
    float *pw = (float *)malloc(sizeof(float) * (size_t)(3 * nw + 3));
    int outside = 0;
    for (int64_t i = 0; i < 3 * nf; ++i) pf[i] = (float)o->r[i];
    for (int64_t i = 0; i < 3 * nw; ++i) pw[i] = (float)o->rw[i];
    for (int64_t i = 0; i < nf; ++i)
        for (int d = 0; d < 3; ++d) o->cell_f[3 * i + d] = orc_cell1(pf[3 * i + d], xmin[d], inv, ng[d], &outside);
    for (int64_t i = 0; i < nw; ++i)
        for (int d = 0; d < 3; ++d) o->cell_w[3 * i + d] = orc_cell1(pw[3 * i + d], xmin[d], inv, ng[d], &outside);
    memcpy(o->r_frz, o->r, sizeof(double) * (size_t)(3 * nf));

    ivec *lf = (ivec *)calloc((size_t)(nf + 1), sizeof(ivec));
    ivec *lw = (ivec *)calloc((size_t)(nf + 1), sizeof(ivec));
    if (o->p.neigh_backend == 1) {
#pragma omp parallel for schedule(dynamic, 64)
        for (int64_t i = 0; i < nf; ++i) {
            for (int64_t j = 0; j < nf; ++j)
                if (j != i && orc_member(&pf[3 * i], &pf[3 * j], rc2)) ipush(&lf[i], (int32_t)j);
            for (int64_t w = 0; w < nw; ++w)
                if (orc_member(&pf[3 * i], &pw[3 * w], rc2)) ipush(&lw[i], (int32_t)w);
        }
    } else {
        /* linked cells: head/next chains per cell, x fastest */
        int64_t nc = (int64_t)ng[0] * ng[1] * ng[2];
        int32_t *head_f = (int32_t *)malloc(sizeof(int32_t) * (size_t)nc);
        int32_t *head_w = (int32_t *)malloc(sizeof(int32_t) * (size_t)nc);
        int32_t *next_f = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nf + 1));
        int32_t *next_w = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nw + 1));
        for (int64_t c = 0; c < nc; ++c) head_f[c] = head_w[c] = -1;
        for (int64_t i = 0; i < nf; ++i) {
            int64_t c = o->cell_f[3 * i] + (int64_t)ng[0] * (o->cell_f[3 * i + 1] + (int64_t)ng[1] * o->cell_f[3 * i + 2]);
            next_f[i] = head_f[c]; head_f[c] = (int32_t)i;
        }
        for (int64_t w = 0; w < nw; ++w) {
            int64_t c = o->cell_w[3 * w] + (int64_t)ng[0] * (o->cell_w[3 * w + 1] + (int64_t)ng[1] * o->cell_w[3 * w + 2]);
            next_w[w] = head_w[c]; head_w[c] = (int32_t)w;
        }
#pragma omp parallel for schedule(dynamic, 256)
        for (int64_t i = 0; i < nf; ++i) {
            const int32_t *ci = &o->cell_f[3 * i];
            for (int dz = -1; dz <= 1; ++dz)
                for (int dy = -1; dy <= 1; ++dy)
                    for (int dx = -1; dx <= 1; ++dx) {
                        int cx = ci[0] + dx, cy = ci[1] + dy, cz = ci[2] + dz;
                        if (cx < 0 || cy < 0 || cz < 0 || cx >= ng[0] || cy >= ng[1] || cz >= ng[2]) continue;
                        int64_t c = cx + (int64_t)ng[0] * (cy + (int64_t)ng[1] * cz);
                        for (int32_t j = head_f[c]; j >= 0; j = next_f[j])
                            if (j != i && orc_member(&pf[3 * i], &pf[3 * j], rc2)) ipush(&lf[i], j);
                        for (int32_t w = head_w[c]; w >= 0; w = next_w[w])
                            if (orc_member(&pf[3 * i], &pw[3 * w], rc2)) ipush(&lw[i], w);
                    }
            qsort(lf[i].v, (size_t)lf[i].n, sizeof(int32_t), cmp_i32);
            qsort(lw[i].v, (size_t)lw[i].n, sizeof(int32_t), cmp_i32);
        }
        free(head_f); free(head_w); free(next_f); free(next_w);
    }
    o->ff_start[0] = o->fw_start[0] = 0;
    for (int64_t i = 0; i < nf; ++i) {
        o->ff_start[i + 1] = o->ff_start[i] + lf[i].n;
        o->fw_start[i + 1] = o->fw_start[i] + lw[i].n;
    }
    free(o->ff_idx); free(o->fw_idx);
    o->ff_idx = (int32_t *)malloc(sizeof(int32_t) * (size_t)(o->ff_start[nf] + 1));
    o->fw_idx = (int32_t *)malloc(sizeof(int32_t) * (size_t)(o->fw_start[nf] + 1));
    for (int64_t i = 0; i < nf; ++i) {
        if (lf[i].n) memcpy(&o->ff_idx[o->ff_start[i]], lf[i].v, sizeof(int32_t) * (size_t)lf[i].n);
        if (lw[i].n) memcpy(&o->fw_idx[o->fw_start[i]], lw[i].v, sizeof(int32_t) * (size_t)lw[i].n);
        free(lf[i].v); free(lw[i].v);
    }
    free(lf); free(lw); free(pf); free(pw);
    o->have_config = 1;
    return outside;
}

/* ---------------------------------------------------------------------------------------------
 * a5  density re-initialisation, Eq. 14 (free surface) / Eq. 15, reading R12:
 *     sigma_i = W(0) + sum_j W_ij + sum_w W_iw ;   rho_i <- max(rho_i, rho0 sigma_i / sigma0)      (Eq. 14)
 *     or rho_i <- rho0 sigma_i / sigma0                                                            (Eq. 15).
 * Which particles take which form ("the fluid density in regions identified as free-surface flow is reinitialized
 * according to [Eq. 14] ... In the absence of a free surface [Eq. 15]"; the paper gives no
 * identification rule):
 *   ORC_FREE_SURFACE        (R12) the whole fluid is one free-surface flow: Eq. 14 for every particle;
 *   ORC_FREE_SURFACE_LOCAL  (R27) a particle is a SURFACE particle when its support is visibly truncated,
 *                           sigma_i < theta sigma0 (theta = fs_threshold, default 0.9: the first layer under a flat
 *                           surface of the lattice has sigma / sigma0 = 0.789, the second 0.9965, deeper ones 1); the
 *                           free-surface REGION is the surface particles and all their fluid neighbours (R1 sets), i.e.
 *                           every particle whose support may reach across the surface; Eq. 14 in the region, Eq. 15
 *                           elsewhere.  Wins over ORC_FREE_SURFACE when both are set;
 *   neither                 no free surface: Eq. 15 for every particle.
 * ------------------------------------------------------------------------------------------- */
static void orc_density_reinit(orc *o)
{
    const double h = o->p.h;
    const int64_t n = o->n_f;
    double *sig = dalloc(n);
    unsigned char *region = (unsigned char *)calloc((size_t)(n > 0 ? n : 1), 1);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double s = orc_Wd(&o->p, 0.0, h);
        const double *ri = &o->r_frz[3 * i];
        for (int64_t q = o->ff_start[i]; q < o->ff_start[i + 1]; ++q) {
            const double *rj = &o->r_frz[3 * o->ff_idx[q]];
            double d0 = ri[0] - rj[0], d1 = ri[1] - rj[1], d2 = ri[2] - rj[2];
            s += orc_Wd(&o->p, sqrt(d0 * d0 + d1 * d1 + d2 * d2), h);
        }
        for (int64_t q = o->fw_start[i]; q < o->fw_start[i + 1]; ++q) {
            const double *rj = &o->rw[3 * o->fw_idx[q]];
            double d0 = ri[0] - rj[0], d1 = ri[1] - rj[1], d2 = ri[2] - rj[2];
            s += orc_Wd(&o->p, sqrt(d0 * d0 + d1 * d1 + d2 * d2), h);
        }
        sig[i] = s;
    }
    if (o->p.flags & ORC_FREE_SURFACE_LOCAL) {                       /* R27 */
        const double theta = o->p.fs_threshold > 0.0 ? o->p.fs_threshold : 0.9;
        for (int64_t i = 0; i < n; ++i) {
            if (!(sig[i] < theta * o->sigma0)) continue;             /* not a surface particle */
            region[i] = 1;
            for (int64_t q = o->ff_start[i]; q < o->ff_start[i + 1]; ++q) region[o->ff_idx[q]] = 1;
        }
    } else if (o->p.flags & ORC_FREE_SURFACE) {                      /* R12 */
        memset(region, 1, (size_t)n);
    }
    for (int64_t i = 0; i < n; ++i) {
        double rn = o->p.rho0 * sig[i] / o->sigma0;
        if (region[i]) o->rho[i] = o->rho[i] > rn ? o->rho[i] : rn;  /* Eq. 14 */
        else o->rho[i] = rn;                                         /* Eq. 15 */
        o->fs_region[i] = region[i];
    }
    free(sig); free(region);
}

/* ---------------------------------------------------------------------------------------------
 * Inter-particle Riemann problem, Eq. 11-13, readings R3, R4:
 *   U_L = -v_i.e_ij, U_R = -v_j.e_ij;  Ubar, Pbar density-weighted means;
 *   beta = min(3 max(U_L - U_R, 0), c0);
 *   U* = Ubar + (p_L - p_R) / (c0 (rho_L + rho_R));
 *   p* = Pbar + rho_L rho_R beta (U_L - U_R) / (rho_L + rho_R).
 * Exposed for the P8 pins.
 * ------------------------------------------------------------------------------------------- */
void orc_riemann(double rhoL, double UL, double pL, double rhoR, double UR, double pR, double c0,
                 double *Ustar, double *pstar, double *Ubar)
{
    double rs = rhoL + rhoR;
    double Ub = (rhoL * UL + rhoR * UR) / rs;
    double Pb = (rhoL * pR + rhoR * pL) / rs;
    double du = UL - UR;
    double beta = 3.0 * (du > 0.0 ? du : 0.0);
    if (beta > c0) beta = c0;
    *Ustar = Ub + (pL - pR) / (c0 * rs);
    *pstar = Pb + rhoL * rhoR * beta * du / rs;
    *Ubar = Ub;
}

/* ---------------------------------------------------------------------------------------------
 * a8  sweep A: momentum equation, Eq. 10 line 2 with the wall forces of Eq. 18-19
 *     (PAPER.md:148-155); geometry (r_ij, e_ij, W') frozen at the last rebuild.
 *       a_i = g - (2/m_i) sum_j V_i V_j p*_ij grad_i W_ij + (2/m_i) sum_j V_i V_j eta_ij v_ij/r_ij W'_ij
 *             - (2/m_i) sum_w V_i V_w p*_iw grad_i W_iw + (2/m_i) sum_w V_i V_w eta (v_i - v_w)/r_iw W'_iw
 *     with V = m / rho, grad_i W_ij = e_ij W'_ij, eta_ij = eta_w = rho0 nu (R6, R8), the wall
 *     one-sided Riemann states of Eq. 16-17 (R6), p*_iw of Eq. 19.
 * ------------------------------------------------------------------------------------------- */
static void orc_sweep_A(orc *o)
{
    const orc_params *p = &o->p;
    const double h = p->h, c0 = p->c0, rho0 = p->rho0, eta = p->rho0 * p->nu;
    const int do_p = (p->flags & ORC_PRESSURE) != 0, do_v = (p->flags & ORC_VISCOUS) != 0;
    const int fresh = o->visc_fresh;      /* R26: 0 = keep acc_v / acc_wv of the advection step's first evaluation */
    const double Vw = orc_vol(p);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < o->n_f; ++i) {
        const double *ri = &o->r_frz[3 * i], *vi = &o->v[3 * i];
        const double rho_i = o->rho[i], p_i = c0 * c0 * (rho_i - rho0), m_i = o->mass[i];
        const double V_i = m_i / rho_i;
        double ap[3] = {0, 0, 0}, av[3] = {0, 0, 0}, awp[3] = {0, 0, 0}, awv[3] = {0, 0, 0};
        for (int64_t q = o->ff_start[i]; q < o->ff_start[i + 1]; ++q) {
            int64_t j = o->ff_idx[q];
            const double *rj = &o->r_frz[3 * j], *vj = &o->v[3 * j];
            double rij[3] = {ri[0] - rj[0], ri[1] - rj[1], ri[2] - rj[2]};
            double r = sqrt(rij[0] * rij[0] + rij[1] * rij[1] + rij[2] * rij[2]);
            const double ir = orc_inv_r(r);                            /* R28: e_ij = 0 at r = 0 */
            double e[3] = {rij[0] * ir, rij[1] * ir, rij[2] * ir};
            double dW = orc_dWdrd(&o->p, r, h);
            double rho_j = o->rho[j], p_j = c0 * c0 * (rho_j - rho0), V_j = o->mass[j] / rho_j;
            double UL = -(vi[0] * e[0] + vi[1] * e[1] + vi[2] * e[2]);
            double UR = -(vj[0] * e[0] + vj[1] * e[1] + vj[2] * e[2]);
            double Us, ps, Ub;
            orc_riemann(rho_i, UL, p_i, rho_j, UR, p_j, c0, &Us, &ps, &Ub);
            for (int d = 0; d < 3; ++d) {
                if (do_p) ap[d] += -(2.0 / m_i) * V_i * V_j * ps * e[d] * dW;
                if (do_v && fresh) av[d] += (2.0 / m_i) * V_i * V_j * eta * (vi[d] - vj[d]) * orc_Fd(&o->p, r, h);
            }
        }
        for (int64_t q = o->fw_start[i]; q < o->fw_start[i + 1]; ++q) {
            int64_t w = o->fw_idx[q];
            const double *rw = &o->rw[3 * w];
            double riw[3] = {ri[0] - rw[0], ri[1] - rw[1], ri[2] - rw[2]};
            double r = sqrt(riw[0] * riw[0] + riw[1] * riw[1] + riw[2] * riw[2]);
            const double ir = orc_inv_r(r);                            /* R28 */
            double e[3] = {riw[0] * ir, riw[1] * ir, riw[2] * ir};
            double dW = orc_dWdrd(&o->p, r, h);
            double vw[3];
            wall_velocity(o, w, vw);
            /* Eq. 17: P_R = P_L + rho_f g . r_fw with r_fw = r_w - r_f ; rho_R from the EoS (Eq. 2) */
            double pR = p_i + rho_i * (p->g[0] * (-riw[0]) + p->g[1] * (-riw[1]) + p->g[2] * (-riw[2]));
            double rhoR = rho0 + pR / (c0 * c0);
            double ps = (rho_i * pR + rhoR * p_i) / (rho_i + rhoR);          /* Eq. 19 */
            for (int d = 0; d < 3; ++d) {
                if (do_p) awp[d] += -(2.0 / m_i) * V_i * Vw * ps * e[d] * dW;                 /* Eq. 18 l.1 */
                if (do_v && fresh) awv[d] += (2.0 / m_i) * V_i * Vw * eta * (vi[d] - vw[d]) * orc_Fd(&o->p, r, h);  /* Eq. 18 l.2 */
            }
        }
        for (int d = 0; d < 3; ++d) {
            o->acc_p[3 * i + d] = ap[d]; o->acc_wp[3 * i + d] = awp[d];
            if (fresh) { o->acc_v[3 * i + d] = av[d]; o->acc_wv[3 * i + d] = awv[d]; }
            o->acc[3 * i + d] = p->g[d] + ap[d] + o->acc_v[3 * i + d] + awp[d] + o->acc_wv[3 * i + d];
        }
    }
}

/* ---------------------------------------------------------------------------------------------
 * a12  churning torque (no formula in the paper; reading R15):
 *      force on wall particle w: F_w = - sum_i m_i (a^p_{i<-w} + a^nu_{i<-w});
 *      tau_b = sum_{w in b} (r_w - o_b) x F_w.  Wall-centric accumulation (serial scatter).
 * ------------------------------------------------------------------------------------------- */
static void orc_torque_reduce(orc *o)
{
    const orc_params *p = &o->p;
    const double h = p->h, c0 = p->c0, rho0 = p->rho0, eta = p->rho0 * p->nu;
    const int do_p = (p->flags & ORC_PRESSURE) != 0, do_v = (p->flags & ORC_VISCOUS) != 0;
    const double Vw = orc_vol(p);
    const int fresh = o->visc_fresh;      /* R26: 0 = the viscous wall forces Fw_v of the advection step's first evaluation are kept */
    memset(o->Fw, 0, sizeof(double) * (size_t)(3 * o->n_w));
    if (fresh) memset(o->Fw_v, 0, sizeof(double) * (size_t)(3 * o->n_w));
    for (int64_t i = 0; i < o->n_f; ++i) {
        const double *ri = &o->r_frz[3 * i], *vi = &o->v[3 * i];
        const double rho_i = o->rho[i], p_i = c0 * c0 * (rho_i - rho0), m_i = o->mass[i];
        const double V_i = m_i / rho_i;
        for (int64_t q = o->fw_start[i]; q < o->fw_start[i + 1]; ++q) {
            int64_t w = o->fw_idx[q];
            const double *rw = &o->rw[3 * w];
            double riw[3] = {ri[0] - rw[0], ri[1] - rw[1], ri[2] - rw[2]};
            double r = sqrt(riw[0] * riw[0] + riw[1] * riw[1] + riw[2] * riw[2]);
            double dW = orc_dWdrd(&o->p, r, h);
            double vw[3];
            wall_velocity(o, w, vw);
            double pR = p_i - rho_i * (p->g[0] * riw[0] + p->g[1] * riw[1] + p->g[2] * riw[2]);
            double rhoR = rho0 + pR / (c0 * c0);
            double ps = (rho_i * pR + rhoR * p_i) / (rho_i + rhoR);
            for (int d = 0; d < 3; ++d) {
                if (do_p) o->Fw[3 * w + d] += -m_i * (-(2.0 / m_i) * V_i * Vw * ps * (riw[d] * orc_inv_r(r)) * dW);
                if (do_v && fresh) o->Fw_v[3 * w + d] += -m_i * ((2.0 / m_i) * V_i * Vw * eta * (vi[d] - vw[d]) * orc_Fd(&o->p, r, h));
            }
        }
    }
    for (int64_t k = 0; k < 3 * o->n_w; ++k) o->Fw[k] += o->Fw_v[k];
    for (int b = 0; b < ORC_MAX_BODIES; ++b) o->torque[b][0] = o->torque[b][1] = o->torque[b][2] = 0.0;
    for (int64_t w = 0; w < o->n_w; ++w) {
        int b = o->body_w[w];
        double a[3] = {o->rw[3 * w] - o->origin[b][0], o->rw[3 * w + 1] - o->origin[b][1], o->rw[3 * w + 2] - o->origin[b][2]};
        const double *F = &o->Fw[3 * w];
        o->torque[b][0] += a[1] * F[2] - a[2] * F[1];
        o->torque[b][1] += a[2] * F[0] - a[0] * F[2];
        o->torque[b][2] += a[0] * F[1] - a[1] * F[0];
    }
}

/* ---------------------------------------------------------------------------------------------
 * a10  sweep B: continuity, Eq. 10 line 1 with v* of Eq. 13 under reading R3
 *      (v* = vbar - (U* - Ubar) e_ij), the wall term of reading R6, and thermal diffusion,
 *      Eq. 22 under readings R9-R10:
 *        drho_i/dt = 2 rho_i [ sum_j V_j (v_i - v*_ij) . grad_i W_ij
 *                              + sum_w V_w (U*_iw - U_L) (n_w . e_iw) W'_iw ]
 *        dT_i/dt  = 1/(rho_i cp_i) [ sum_j V_j K_ij T_ij / r_ij W'_ij + sum_n V_n K_in T_in / r_in W'_in ],
 *        K_ab = 4 k_a k_b / (k_a + k_b)   (0 if either conductivity is 0).
 * ------------------------------------------------------------------------------------------- */
static void orc_sweep_B(orc *o)
{
    const orc_params *p = &o->p;
    const double h = p->h, c0 = p->c0, rho0 = p->rho0;
    const int hydro = (p->flags & ORC_HYDRO) != 0, thermal = (p->flags & ORC_THERMAL) != 0;
    const double Vw = orc_vol(p);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < o->n_f; ++i) {
        const double *ri = &o->r_frz[3 * i], *vi = &o->v[3 * i];
        const double rho_i = o->rho[i], p_i = c0 * c0 * (rho_i - rho0);
        double sr = 0.0, sT = 0.0;
        for (int64_t q = o->ff_start[i]; q < o->ff_start[i + 1]; ++q) {
            int64_t j = o->ff_idx[q];
            const double *rj = &o->r_frz[3 * j], *vj = &o->v[3 * j];
            double rij[3] = {ri[0] - rj[0], ri[1] - rj[1], ri[2] - rj[2]};
            double r = sqrt(rij[0] * rij[0] + rij[1] * rij[1] + rij[2] * rij[2]);
            const double ir = orc_inv_r(r);                            /* R28: e_ij = 0 at r = 0 */
            double e[3] = {rij[0] * ir, rij[1] * ir, rij[2] * ir};
            double dW = orc_dWdrd(&o->p, r, h);
            double rho_j = o->rho[j], p_j = c0 * c0 * (rho_j - rho0), V_j = o->mass[j] / rho_j;
            if (hydro) {
                double UL = -(vi[0] * e[0] + vi[1] * e[1] + vi[2] * e[2]);
                double UR = -(vj[0] * e[0] + vj[1] * e[1] + vj[2] * e[2]);
                double Us, ps, Ub;
                orc_riemann(rho_i, UL, p_i, rho_j, UR, p_j, c0, &Us, &ps, &Ub);
                double dot = 0.0;
                for (int d = 0; d < 3; ++d) {
                    double vbar = (rho_i * vi[d] + rho_j * vj[d]) / (rho_i + rho_j);
                    double vstar = vbar - (Us - Ub) * e[d];              /* Eq. 13, sign per R3 */
                    dot += (vi[d] - vstar) * e[d] * dW;
                }
                sr += V_j * dot;
            }
            if (thermal) {
                double ki = o->k[i], kj = o->k[j];
                double K = (ki + kj) > 0.0 ? 4.0 * ki * kj / (ki + kj) : 0.0;
                sT += V_j * K * (o->T[i] - o->T[j]) * orc_Fd(&o->p, r, h);
            }
        }
        for (int64_t q = o->fw_start[i]; q < o->fw_start[i + 1]; ++q) {
            int64_t w = o->fw_idx[q];
            const double *rw = &o->rw[3 * w], *nw = &o->nw[3 * w];
            double riw[3] = {ri[0] - rw[0], ri[1] - rw[1], ri[2] - rw[2]};
            double r = sqrt(riw[0] * riw[0] + riw[1] * riw[1] + riw[2] * riw[2]);
            const double ir = orc_inv_r(r);                            /* R28 */
            double e[3] = {riw[0] * ir, riw[1] * ir, riw[2] * ir};
            double dW = orc_dWdrd(&o->p, r, h);
            if (hydro) {
                double vw[3];
                wall_velocity(o, w, vw);
                double UL = -(nw[0] * vi[0] + nw[1] * vi[1] + nw[2] * vi[2]);        /* Eq. 16 */
                double uw = -(nw[0] * vw[0] + nw[1] * vw[1] + nw[2] * vw[2]);
                double UR = -UL + 2.0 * uw;                                            /* Eq. 17 */
                double pR = p_i - rho_i * (p->g[0] * riw[0] + p->g[1] * riw[1] + p->g[2] * riw[2]);
                double rhoR = rho0 + pR / (c0 * c0);
                double Us, ps, Ub;
                orc_riemann(rho_i, UL, p_i, rhoR, UR, pR, c0, &Us, &ps, &Ub);
                double ne = nw[0] * e[0] + nw[1] * e[1] + nw[2] * e[2];
                sr += Vw * (Us - UL) * ne * dW;                                        /* R6 */
            }
            if (thermal) {
                double ki = o->k[i], kn = p->body_k[o->body_w[w]];
                double K = (ki + kn) > 0.0 ? 4.0 * ki * kn / (ki + kn) : 0.0;
                sT += Vw * K * (o->T[i] - o->Tw[w]) * orc_Fd(&o->p, r, h);
            }
        }
        o->drho_dt[i] = hydro ? 2.0 * rho_i * sr : 0.0;
        o->dT_dt[i] = thermal ? sT / (rho_i * o->cp[i]) : 0.0;
    }
}

/* ---------------------------------------------------------------------------------------------
 * Evolving solid temperature (reading R23): Eq. 20 applied to a solid particle w of a body
 * whose temperature is not held:
 *     m_w c_s dT_w/dt = sum_i V_w V_i K_wi T_wi F_wi  +  sum_u V_w V_u K_wu T_wu F_wu ,   F = W'(r)/r,
 * i = fluid neighbours (V_i = m_i / rho_i, the mirror image of the wall term of Eq. 22, so that the pair
 * exchange is antisymmetric), u = solid neighbours of any body (K_wu = 4 k_w k_u / (k_w + k_u), V = dx^3),
 * m_w = rho_s dx^3; neighbours under the R1 predicate, geometry of the last rebuild, T^n (R11).
 * ------------------------------------------------------------------------------------------- */
static int orc_any_evolving(const orc *o)
{
    for (int b = 0; b < o->p.n_bodies; ++b) if (o->p.body_mode[b] == 1) return 1;
    return 0;
}

static void orc_wall_heat(orc *o)
{
    const orc_params *p = &o->p;
    const int64_t nf = o->n_f, nw = o->n_w;
    const double h = p->h, V0 = orc_vol(p);
    for (int64_t w = 0; w < nw; ++w) o->dTw_dt[w] = 0.0;
    if (!(p->flags & ORC_THERMAL) || !orc_any_evolving(o)) return;
    double *flux = dalloc(nw);
    /* fluid neighbours: transpose of the fluid -> wall lists */
    for (int64_t i = 0; i < nf; ++i) {
        const double *ri = &o->r_frz[3 * i];
        const double Vi = o->mass[i] / o->rho[i], ki = o->k[i];
        for (int64_t q = o->fw_start[i]; q < o->fw_start[i + 1]; ++q) {
            const int64_t w = o->fw_idx[q];
            const int b = o->body_w[w];
            if (p->body_mode[b] != 1) continue;
            const double kn = p->body_k[b];
            const double K = (ki + kn) > 0.0 ? 4.0 * ki * kn / (ki + kn) : 0.0;
            const double *rw = &o->rw[3 * w];
            double d0 = rw[0] - ri[0], d1 = rw[1] - ri[1], d2 = rw[2] - ri[2];
            double r = sqrt(d0 * d0 + d1 * d1 + d2 * d2);
            flux[w] += V0 * Vi * K * (o->Tw[w] - o->T[i]) * orc_Fd(&o->p, r, h);
        }
    }
    /* solid neighbours: linked cells over the wall particles, fp32 predicate of R1 */
    const float rc2 = orc_rc2(h);
    float *pw = (float *)malloc(sizeof(float) * (size_t)(3 * nw + 3));
    for (int64_t i = 0; i < 3 * nw; ++i) pw[i] = (float)o->rw[i];
    float xmin[3], inv; int ng[3];
    orc_grid(p, xmin, &inv, ng);
    int64_t nc = (int64_t)ng[0] * ng[1] * ng[2];
    int32_t *head = (int32_t *)malloc(sizeof(int32_t) * (size_t)nc);
    int32_t *next = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nw + 1));
    for (int64_t c = 0; c < nc; ++c) head[c] = -1;
    for (int64_t w = 0; w < nw; ++w) {
        int64_t c = o->cell_w[3 * w] + (int64_t)ng[0] * (o->cell_w[3 * w + 1] + (int64_t)ng[1] * o->cell_w[3 * w + 2]);
        next[w] = head[c]; head[c] = (int32_t)w;
    }
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t w = 0; w < nw; ++w) {
        const int b = o->body_w[w];
        if (p->body_mode[b] != 1) continue;
        const int32_t *cw = &o->cell_w[3 * w];
        const double *rw = &o->rw[3 * w];
        const double kw = p->body_k[b];
        double s = 0.0;
        for (int dz = -1; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int cx = cw[0] + dx, cy = cw[1] + dy, cz = cw[2] + dz;
                    if (cx < 0 || cy < 0 || cz < 0 || cx >= ng[0] || cy >= ng[1] || cz >= ng[2]) continue;
                    int64_t c = cx + (int64_t)ng[0] * (cy + (int64_t)ng[1] * cz);
                    for (int32_t u = head[c]; u >= 0; u = next[u]) {
                        if (u == w || !orc_member(&pw[3 * w], &pw[3 * u], rc2)) continue;
                        const double ku = p->body_k[o->body_w[u]];
                        const double K = (kw + ku) > 0.0 ? 4.0 * kw * ku / (kw + ku) : 0.0;
                        const double *ru = &o->rw[3 * u];
                        double d0 = rw[0] - ru[0], d1 = rw[1] - ru[1], d2 = rw[2] - ru[2];
                        double r = sqrt(d0 * d0 + d1 * d1 + d2 * d2);
                        s += V0 * V0 * K * (o->Tw[w] - o->Tw[u]) * orc_Fd(&o->p, r, h);
                    }
                }
        o->dTw_dt[w] = (flux[w] + s) / (p->body_rho[b] * V0 * p->body_cp[b]);
    }
    free(flux); free(pw); free(head); free(next);
}

/* ---------------------------------------------------------------------------------------------
 * a6  time-step criteria, Eq. 25-26, readings R13-R14.
 * ------------------------------------------------------------------------------------------- */
double orc_dt_ad(double h, double vmax, double nu, double cfl_ad)
{
    double a = h / vmax, b = nu > 0.0 ? h * h / nu : a;
    return cfl_ad * (a < b ? a : b);
}
double orc_dt_ac(double h, double c0, double vmax, double cfl_ac) { return cfl_ac * h / (c0 + vmax); }
double orc_dt_thermal(double rho, double cp, double h, double k) { return 0.5 * rho * cp * h * h / k; }

static double orc_vmax(const orc *o)
{
    double m = 0.0;
    for (int64_t i = 0; i < o->n_f; ++i) {
        const double *v = &o->v[3 * i];
        double s = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        if (s > m) m = s;
    }
    return m;
}

static double orc_uref(const orc *o) { return o->p.u_ref < 0.0 ? 0.1 * o->p.c0 : o->p.u_ref; }

int orc_rebuild(orc *o)
{
    orc_wall_kinematics(o);                                  /* a1 */
    int outside = orc_build_config(o);                       /* a2-a4 */
    if (o->p.flags & ORC_DENSITY_REINIT) orc_density_reinit(o);   /* a5 */
    double vm = orc_vmax(o), ur = orc_uref(o);
    o->vmax = vm;
    o->dt_ad = orc_dt_ad(o->p.h, vm > ur ? vm : ur, o->p.nu, o->p.cfl_ad);
    o->elapsed = 0.0; o->since_rebuild = 0; o->rebuilds++;
    return outside;
}

/* ---------------------------------------------------------------------------------------------
 * Physics-driven particle relaxation, Eq. 6-9, without the level set (reading R24): one step =
 *   neighbour configuration of the present positions (R1);
 *   F_p,i = -(2 / m_i) sum_j V_i V_j p0 grad_i W_ij  (Eq. 7), j = fluid and wall neighbours, every volume dx^3 and
 *           m_i = rho0 dx^3 (the reference state that is being built; wall particles confine the fluid in place of
 *           the level-set "static confinement" of ref. [42]);
 *   dt = 0.25 sqrt(h / max_i |F_p,i|)  (Eq. 8, one global step);   r_i += F_p,i dt^2 / 2  (Eq. 9).
 * Velocities, densities and temperatures are untouched.  Returns the last max |F_p|.
 * ------------------------------------------------------------------------------------------- */
double orc_relax(orc *o, int n_steps, double p0)
{
    const int64_t nf = o->n_f;
    const double h = o->p.h, V0 = orc_vol(&o->p), m0 = o->p.rho0 * V0;
    double *F = dalloc(3 * nf);
    double fmax = 0.0;
    for (int s = 0; s < n_steps; ++s) {
        orc_wall_kinematics(o);
        orc_build_config(o);
        fmax = 0.0;
        for (int64_t i = 0; i < nf; ++i) {
            const double *ri = &o->r_frz[3 * i];
            double g[3] = {0.0, 0.0, 0.0};
            for (int64_t q = o->ff_start[i]; q < o->ff_start[i + 1]; ++q) {
                const double *rj = &o->r_frz[3 * o->ff_idx[q]];
                double d[3] = {ri[0] - rj[0], ri[1] - rj[1], ri[2] - rj[2]};
                double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                double c = orc_Fd(&o->p, r, h);
                for (int k = 0; k < 3; ++k) g[k] += V0 * c * d[k];              /* V_j grad_i W_ij */
            }
            for (int64_t q = o->fw_start[i]; q < o->fw_start[i + 1]; ++q) {
                const double *rj = &o->rw[3 * o->fw_idx[q]];
                double d[3] = {ri[0] - rj[0], ri[1] - rj[1], ri[2] - rj[2]};
                double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                double c = orc_Fd(&o->p, r, h);
                for (int k = 0; k < 3; ++k) g[k] += V0 * c * d[k];
            }
            for (int k = 0; k < 3; ++k) F[3 * i + k] = -2.0 / m0 * V0 * p0 * g[k];   /* Eq. 7 */
            double a = sqrt(F[3 * i] * F[3 * i] + F[3 * i + 1] * F[3 * i + 1] + F[3 * i + 2] * F[3 * i + 2]);
            if (a > fmax) fmax = a;
        }
        if (fmax > 0.0) {
            const double dt = 0.25 * sqrt(h / fmax);                            /* Eq. 8 */
            for (int64_t i = 0; i < 3 * nf; ++i) o->r[i] += 0.5 * F[i] * dt * dt;   /* Eq. 9 */
        }
        o->have_config = 0;                                                      /* positions moved */
    }
    free(F);
    return fmax;
}

/* ---------------------------------------------------------------------------------------------
 * One acoustic step: position-Verlet halves of the dual-criteria scheme (ref [45];
 * reading R7), steps a6-a12 of DESIGN.md section 2.
 * ------------------------------------------------------------------------------------------- */
static int orc_step_once(orc *o)
{
    const orc_params *p = &o->p;
    int rc = 0;
    int due = !o->have_config;
    if (p->rebuild_every >= 1) due |= (o->since_rebuild >= p->rebuild_every);
    else due |= (o->elapsed >= o->dt_ad);
    if (due) rc = orc_rebuild(o);

    const int hydro = (p->flags & ORC_HYDRO) != 0;
    double dt;
    if (p->dt_fixed > 0.0) dt = p->dt_fixed;
    else {
        double vm = orc_vmax(o), ur = orc_uref(o);
        o->vmax = vm;
        dt = orc_dt_ac(p->h, p->c0, vm > ur ? vm : ur, p->cfl_ac);          /* Eq. 25 l.2 */
        if (p->rebuild_every < 1) { double rem = o->dt_ad - o->elapsed; if (rem < dt) dt = rem; }  /* R14 */
        /* Eq. 26: the explicit thermal step may not exceed dt_T = 0.5 rho C_p h^2 / k, the smallest over the
         * fluid and the bodies whose temperature evolves (R23); with the hydrodynamics off (static particles, heat only) there is
         * no acoustic criterion and the step is dt_T itself */
        if (p->flags & ORC_THERMAL) {
            double dtT = p->k_f > 0.0 ? orc_dt_thermal(p->rho0, p->cp_f, p->h, p->k_f) : 0.0;
            for (int b = 0; b < p->n_bodies; ++b)
                if (p->body_mode[b] == 1 && p->body_k[b] > 0.0 && p->body_rho[b] > 0.0 && p->body_cp[b] > 0.0) {
                    double d = orc_dt_thermal(p->body_rho[b], p->body_cp[b], p->h, p->body_k[b]);
                    if (dtT == 0.0 || d < dtT) dtT = d;
                }
            if (dtT > 0.0 && (!hydro || dt > dtT)) dt = dtT;
        }
    }
    o->dt = dt;
    const int64_t n = o->n_f;
    /* R26 (ref [45]): with ORC_VISCOUS_HELD the viscous sums are evaluated by the first acoustic step of an
     * advection step (the one that rebuilt), from v^n and the densities that sweep sees, and held until the next rebuild */
    o->visc_fresh = !(p->flags & ORC_VISCOUS_HELD) || o->since_rebuild == 0;
    if (hydro) {
        for (int64_t i = 0; i < n; ++i) {                                    /* a7 */
            o->rho[i] += 0.5 * dt * o->drho_saved[i];
            for (int d = 0; d < 3; ++d) o->r[3 * i + d] += 0.5 * dt * o->v[3 * i + d];
        }
        orc_sweep_A(o);                                                      /* a8 */
        orc_torque_reduce(o);                                                /* a12 */
        for (int64_t i = 0; i < n; ++i)                                      /* a9 */
            for (int d = 0; d < 3; ++d) {
                o->v[3 * i + d] += dt * o->acc[3 * i + d];
                o->r[3 * i + d] += 0.5 * dt * o->v[3 * i + d];
            }
    }
    orc_sweep_B(o);                                                          /* a10 */
    orc_wall_heat(o);                                                        /* R23, with T^n on both sides */
    for (int64_t w = 0; w < o->n_w; ++w) o->Tw[w] += dt * o->dTw_dt[w];
    for (int64_t i = 0; i < n; ++i) {                                        /* a11 */
        if (hydro) { o->rho[i] += 0.5 * dt * o->drho_dt[i]; o->drho_saved[i] = o->drho_dt[i]; }
        o->T[i] += dt * o->dT_dt[i];                                         /* R11: forward Euler */
    }
    o->t += dt; o->elapsed += dt; o->steps++; o->since_rebuild++;
    return rc;
}

int orc_step(orc *o, int n)
{
    int rc = 0;
    for (int s = 0; s < n; ++s) rc |= orc_step_once(o);
    return rc;
}

/* evaluate the pair sums on the current state without advancing it (pins P3, P4, P7-P9, P11) */
int orc_eval_rates(orc *o)
{
    int rc = 0;
    if (!o->have_config) rc = orc_rebuild(o);
    o->visc_fresh = 1;
    orc_sweep_A(o);
    orc_torque_reduce(o);
    orc_sweep_B(o);
    orc_wall_heat(o);
    return rc;
}

/* ---------------------------------------------------------------------------------------------
 * Contact factor of the solid particles, Eq. 24:
 *     zeta_C(w) = sum_j V_j W_wj / sum_{j in N_w^full} V_j W_wj ,  j = lubricant particles around solid particle w.
 * Numerator: V_j = m_j / rho_j (current density), W at the distance of the frozen configuration,
 * over the fluid neighbours of w under the R1 predicate (the transpose of the fluid -> wall lists).
 * Denominator (reading R22; the paper only says "the case where the gear particle is fully immersed"): every place
 * in the support of w that is not taken by a solid particle is filled with lubricant at the reference spacing, so
 *     sum_full(w) = dx^3 sigma0 - sum_{w' solid, incl. w itself} V_w' W_ww' ,   V_w' = dx^3,
 * sigma0 = full cubic-lattice kernel sum incl. W(0) (R12).  Where less than 1e-3 of the support is open
 * (sum_full <= 1e-3 dx^3 sigma0: particles buried in the solid) zeta_C = 0.
 * ------------------------------------------------------------------------------------------- */
int orc_contact_factor(const orc *o, double *zeta)
{
    const int64_t nf = o->n_f, nw = o->n_w;
    if (!o->have_config) return -1;
    const double h = o->p.h, V0 = orc_vol(&o->p);
    const float rc2 = orc_rc2(h);
    double *num = dalloc(nw), *solid = dalloc(nw);
    /* numerator: transpose of the fluid -> wall neighbour lists */
    for (int64_t i = 0; i < nf; ++i) {
        const double Vi = o->mass[i] / o->rho[i];
        const double *ri = &o->r_frz[3 * i];
        for (int64_t q = o->fw_start[i]; q < o->fw_start[i + 1]; ++q) {
            const int64_t w = o->fw_idx[q];
            const double *rw = &o->rw[3 * w];
            double d0 = ri[0] - rw[0], d1 = ri[1] - rw[1], d2 = ri[2] - rw[2];
            num[w] += Vi * orc_Wd(&o->p, sqrt(d0 * d0 + d1 * d1 + d2 * d2), h);
        }
    }
    /* solid part of the support: wall-wall pairs under the same fp32 predicate, self included (W(0)) */
    float *pw = (float *)malloc(sizeof(float) * (size_t)(3 * nw + 3));
    for (int64_t i = 0; i < 3 * nw; ++i) pw[i] = (float)o->rw[i];
    float xmin[3], inv; int ng[3];
    orc_grid(&o->p, xmin, &inv, ng);
    int64_t nc = (int64_t)ng[0] * ng[1] * ng[2];
    int32_t *head = (int32_t *)malloc(sizeof(int32_t) * (size_t)nc);
    int32_t *next = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nw + 1));
    for (int64_t c = 0; c < nc; ++c) head[c] = -1;
    for (int64_t w = 0; w < nw; ++w) {
        int64_t c = o->cell_w[3 * w] + (int64_t)ng[0] * (o->cell_w[3 * w + 1] + (int64_t)ng[1] * o->cell_w[3 * w + 2]);
        next[w] = head[c]; head[c] = (int32_t)w;
    }
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t w = 0; w < nw; ++w) {
        const int32_t *cw = &o->cell_w[3 * w];
        const double *rw = &o->rw[3 * w];
        double s = 0.0;
        for (int dz = -1; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int cx = cw[0] + dx, cy = cw[1] + dy, cz = cw[2] + dz;
                    if (cx < 0 || cy < 0 || cz < 0 || cx >= ng[0] || cy >= ng[1] || cz >= ng[2]) continue;
                    int64_t c = cx + (int64_t)ng[0] * (cy + (int64_t)ng[1] * cz);
                    for (int32_t u = head[c]; u >= 0; u = next[u])
                        if (orc_member(&pw[3 * w], &pw[3 * u], rc2)) {
                            const double *ru = &o->rw[3 * u];
                            double d0 = rw[0] - ru[0], d1 = rw[1] - ru[1], d2 = rw[2] - ru[2];
                            s += orc_Wd(&o->p, sqrt(d0 * d0 + d1 * d1 + d2 * d2), h);
                        }
                }
        solid[w] = V0 * s;
    }
    for (int64_t w = 0; w < nw; ++w) {
        const double full = V0 * o->sigma0 - solid[w];
        zeta[w] = full > 1.0e-3 * V0 * o->sigma0 ? num[w] / full : 0.0;
    }
    free(num); free(solid); free(pw); free(head); free(next);
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * read-back
 * ------------------------------------------------------------------------------------------- */
enum {
    ORC_F_POS = 0, ORC_F_VEL, ORC_F_RHO, ORC_F_P, ORC_F_T, ORC_F_ACC, ORC_F_DRHO_DT, ORC_F_DT_DT,
    ORC_F_ACC_P, ORC_F_ACC_V, ORC_F_ACC_WP, ORC_F_ACC_WV, ORC_F_WALL_POS, ORC_F_WALL_NORMAL,
    ORC_F_WALL_FORCE, ORC_F_DRHO_SAVED, ORC_F_WALL_T, ORC_F_WALL_DT_DT
};

int64_t orc_get_f64(const orc *o, int field, double *dst)
{
    const int64_t n = o->n_f, nw = o->n_w;
    switch (field) {
    case ORC_F_POS: memcpy(dst, o->r, sizeof(double) * 3 * n); return 3 * n;
    case ORC_F_VEL: memcpy(dst, o->v, sizeof(double) * 3 * n); return 3 * n;
    case ORC_F_RHO: memcpy(dst, o->rho, sizeof(double) * n); return n;
    case ORC_F_P: for (int64_t i = 0; i < n; ++i) dst[i] = o->p.c0 * o->p.c0 * (o->rho[i] - o->p.rho0); return n;  /* Eq. 2 */
    case ORC_F_T: memcpy(dst, o->T, sizeof(double) * n); return n;
    case ORC_F_ACC: memcpy(dst, o->acc, sizeof(double) * 3 * n); return 3 * n;
    case ORC_F_DRHO_DT: memcpy(dst, o->drho_dt, sizeof(double) * n); return n;
    case ORC_F_DT_DT: memcpy(dst, o->dT_dt, sizeof(double) * n); return n;
    case ORC_F_ACC_P: memcpy(dst, o->acc_p, sizeof(double) * 3 * n); return 3 * n;
    case ORC_F_ACC_V: memcpy(dst, o->acc_v, sizeof(double) * 3 * n); return 3 * n;
    case ORC_F_ACC_WP: memcpy(dst, o->acc_wp, sizeof(double) * 3 * n); return 3 * n;
    case ORC_F_ACC_WV: memcpy(dst, o->acc_wv, sizeof(double) * 3 * n); return 3 * n;
    case ORC_F_WALL_POS: memcpy(dst, o->rw, sizeof(double) * 3 * nw); return 3 * nw;
    case ORC_F_WALL_NORMAL: memcpy(dst, o->nw, sizeof(double) * 3 * nw); return 3 * nw;
    case ORC_F_WALL_FORCE: memcpy(dst, o->Fw, sizeof(double) * 3 * nw); return 3 * nw;
    case ORC_F_DRHO_SAVED: memcpy(dst, o->drho_saved, sizeof(double) * n); return n;
    case ORC_F_WALL_T: memcpy(dst, o->Tw, sizeof(double) * nw); return nw;
    case ORC_F_WALL_DT_DT: memcpy(dst, o->dTw_dt, sizeof(double) * nw); return nw;
    default: return -1;
    }
}

int orc_get_cells(const orc *o, int32_t *cell_f, int32_t *cell_w)
{
    if (cell_f) memcpy(cell_f, o->cell_f, sizeof(int32_t) * (size_t)(3 * o->n_f));
    if (cell_w) memcpy(cell_w, o->cell_w, sizeof(int32_t) * (size_t)(3 * o->n_w));
    return 0;
}

/* which form the last density re-initialisation took: 1 = Eq. 14 (free-surface region), 0 = Eq. 15 */
int orc_get_fs_region(const orc *o, unsigned char *dst)
{
    memcpy(dst, o->fs_region, (size_t)o->n_f);
    return 0;
}

/* neighbour counts (fluid + wall) and digests of the frozen configuration */
int orc_get_neigh(const orc *o, uint32_t *count_ff, uint32_t *count_fw, uint64_t *digest)
{
    for (int64_t i = 0; i < o->n_f; ++i) {
        uint64_t dg = 0;
        for (int64_t q = o->ff_start[i]; q < o->ff_start[i + 1]; ++q) dg += orc_mix64((uint64_t)o->ff_idx[q] + 1);
        for (int64_t q = o->fw_start[i]; q < o->fw_start[i + 1]; ++q) dg += orc_mix64((uint64_t)o->n_f + (uint64_t)o->fw_idx[q] + 1);
        if (count_ff) count_ff[i] = (uint32_t)(o->ff_start[i + 1] - o->ff_start[i]);
        if (count_fw) count_fw[i] = (uint32_t)(o->fw_start[i + 1] - o->fw_start[i]);
        if (digest) digest[i] = dg;
    }
    return 0;
}

/* CSR copy-out: which = 0 fluid-fluid, 1 fluid-wall.  idx == NULL -> only the total is returned. */
int64_t orc_get_csr(const orc *o, int which, int64_t *start, int32_t *idx)
{
    const int64_t *s = which ? o->fw_start : o->ff_start;
    const int32_t *x = which ? o->fw_idx : o->ff_idx;
    if (start) memcpy(start, s, sizeof(int64_t) * (size_t)(o->n_f + 1));
    if (idx) memcpy(idx, x, sizeof(int32_t) * (size_t)s[o->n_f]);
    return s[o->n_f];
}

int orc_get_torque(const orc *o, int body, double torque[3], double *axial)
{
    if (body < 0 || body >= ORC_MAX_BODIES) return -1;
    for (int d = 0; d < 3; ++d) torque[d] = o->torque[body][d];
    if (axial) *axial = o->axis[body][0] * torque[0] + o->axis[body][1] * torque[1] + o->axis[body][2] * torque[2];
    return 0;
}

/* stats: t, dt, dt_ad, elapsed, vmax, steps, rebuilds, sigma0 */
int orc_get_stats(const orc *o, double out[8])
{
    out[0] = o->t; out[1] = o->dt; out[2] = o->dt_ad; out[3] = o->elapsed; out[4] = o->vmax;
    out[5] = (double)o->steps; out[6] = (double)o->rebuilds; out[7] = o->sigma0;
    return 0;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
