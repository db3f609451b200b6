// sph_b200.cu -- host side of libsph_b200.so: the C ABI of include/sph.h, device memory
// management and the launch sequence of one acoustic step.
// Every step of the path runs in the CUDA kernels of neighbour.cuh / pair.cuh / integrate.cuh;
// there is no CPU fallback.
#include "../../include/sph.h"
#include "common.cuh"
#include "integrate.cuh"
#include "neighbour.cuh"
#include "pair.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <utility>
#include <vector>

namespace {

thread_local char g_create_error[512] = "";

struct ProfRec { int cls; cudaEvent_t e0, e1; };

}  // namespace

struct sph_ctx {
    sph_params prm;
    DevParams P;
    cudaStream_t stream;
    int device;
    char err[512];
    uint64_t cap_f, cap_w, n_f, n_w;
    int n_cells;
    double sigma0;
    bool loaded, walls_sorted, walls_moving, any_evolving;
    bool have_config;
    long long since_rebuild;
    uint64_t launches, device_bytes;
    // bodies (host copy)
    double origin[SPH_MAX_BODIES][3], axis[SPH_MAX_BODIES][3], omega[SPH_MAX_BODIES];
    // fluid state (sorted order) + sort scratch
    float4 *posc, *posc_s, *A, *A_s, *Bc, *Bn, *B_s, *acc, *G;
    float4* mat;                   // sph_set_materials: {m, k, cp, 0} per fluid particle, original order (NULL: uniform fluid)
    bool have_mat;
    float4* avisc;                 // R26: held viscous acceleration (allocated with SPH_FLAG_VISCOUS_HELD)
    uint32_t *orig, *orig_s;
    float2* rates;
    uint32_t* ncnt;
    unsigned char* fs_region;      // R27: free-surface region of the last density re-initialisation (sorted order)
    uint4 *list_f, *list_w;
    TileHdr* hdr;
    uint32_t *tile_bin, *tile_order;      // tile schedule of the sweeps (k_tile_order)
    int n_tiles, KF8, KW8;
    uint32_t *cell_id_f, *rank_f, *perm_f, *ccount_f, *cstart_f;
    // walls
    float4 *wref_pos, *wref_nrm, *wpos, *wnrm, *WA, *WB;
    int* wbody;
    float *wT, *wrate;
    uint32_t *cell_id_w, *rank_w, *perm_w, *ccount_w, *cstart_w;
    uint32_t* block_sums;
    int n_scan_blocks;
    Clock* clk;
    void* out_buf;
    uint64_t out_bytes;
    unsigned char* stage_buf;        // device staging of HOST inputs of sph_load_particles (allocated at the first such call)
    uint64_t stage_bytes;
    std::vector<void*> allocs;
    // the acoustic step as a CUDA graph (device-decided rebuild = body of a conditional IF node); one executable per
    // parity of the Bc / Bn ping-pong
    cudaStream_t aux_stream, cap_stream;   // private streams used only while capturing (the caller's may be the legacy default stream)
    cudaGraphExec_t gexec[2];
    uint64_t g_fixed[2], g_body[2];      // kernels per graph launch outside / inside the conditional body
    int parity;
    bool use_graph;
    int bank_order;                // bank-aware list order at the end of k_build_tiles (pair.cuh: bank_order_one); 0 = off
    int n_sm;
    uint64_t graph_fixed_launches, graph_body_per_rebuild;
    // profiling
    bool prof_on;
    std::vector<ProfRec> prof;
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used;
};

namespace {

int fail(sph_ctx* c, int code, const char* fmt, ...)
{
    char* dst = c ? c->err : g_create_error;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess)                                                                    \
            return fail(ctx, SPH_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__, __LINE__); \
    } while (0)

template <typename T>
int dev_alloc(sph_ctx* ctx, T** p, uint64_t count)
{
    void* q = nullptr;
    uint64_t bytes = (count ? count : 1) * sizeof(T);
    cudaError_t e = cudaMalloc(&q, bytes);
    if (e != cudaSuccess) return fail(ctx, SPH_ENOMEM, "cudaMalloc(%llu bytes) failed: %s", (unsigned long long)bytes, cudaGetErrorString(e));
    ctx->allocs.push_back(q);
    ctx->device_bytes += bytes;
    *p = reinterpret_cast<T*>(q);
    return SPH_OK;
}

void free_all(sph_ctx* ctx)
{
    for (void* p : ctx->allocs) cudaFree(p);
    ctx->allocs.clear();
    ctx->device_bytes = 0;
}

cudaEvent_t next_event(sph_ctx* ctx)
{
    if (ctx->ev_used == ctx->ev_pool.size()) {
        cudaEvent_t e;
        cudaEventCreate(&e);
        ctx->ev_pool.push_back(e);
    }
    return ctx->ev_pool[ctx->ev_used++];
}

struct Launch {
    sph_ctx* ctx; int cls; cudaEvent_t e1;
    Launch(sph_ctx* c, int k) : ctx(c), cls(k), e1(nullptr)
    {
        if (ctx->prof_on) {
            cudaEvent_t e0 = next_event(ctx);
            e1 = next_event(ctx);
            cudaEventRecord(e0, ctx->stream);
            ctx->prof.push_back({cls, e0, e1});
        }
        ctx->launches++;
    }
    ~Launch() { if (e1) cudaEventRecord(e1, ctx->stream); }
};
#define LAUNCH(cls, kernel, grid, block, ...)                          \
    do {                                                               \
        Launch l__(ctx, cls);                                          \
        kernel<<<(grid), (block), 0, ctx->stream>>>(__VA_ARGS__);      \
    } while (0)

#define LAUNCH_SMEM(cls, kernel, grid, block, smem, ...)                \
    do {                                                               \
        Launch l__(ctx, cls);                                          \
        kernel<<<(grid), (block), (smem), ctx->stream>>>(__VA_ARGS__); \
    } while (0)

inline int cdiv(uint64_t a, int b) { return (int)((a + b - 1) / b); }

// Wendland C2 normalisation: 21 / (16 pi h^3) in three dimensions, 7 / (4 pi h^2) in the plane (R2, R25)
double wendland_alpha(double h, bool planar) { return planar ? 7.0 / (4.0 * M_PI * h * h) : 21.0 / (16.0 * M_PI * h * h * h); }

double wendland_W(double r, double h, bool planar)
{
    double q = r / h;
    if (q >= 2.0) return 0.0;
    double s = 1.0 - 0.5 * q;
    return wendland_alpha(h, planar) * s * s * s * s * (1.0 + 2.0 * q);
}

// sigma0: kernel sum over the full cubic lattice of spacing dx, self term included (R12)
double lattice_sigma0(double dx, double h, bool planar)
{
    int m = (int)std::ceil(2.0 * h / dx) + 1;
    double s = 0.0;
    for (int a = -m; a <= m; ++a)
        for (int b = -m; b <= m; ++b)
            for (int c = planar ? 0 : -m; c <= (planar ? 0 : m); ++c) s += wendland_W(dx * std::sqrt((double)(a * a + b * b + c * c)), h, planar);
    return s;
}

bool is_planar(const sph_params& p) { return p.dim == 2; }

// Eq. 26: dt_T = 0.5 rho C_p h^2 / k, the smallest over the fluid and the bodies whose temperature evolves
// (R23); 0 when the heat equation is off or nothing conducts
double thermal_dt_bound(const sph_params& p)
{
    if (!(p.flags & SPH_FLAG_THERMAL)) return 0.0;
    double best = 0.0;
    auto take = [&](double rho, double cp, double k) {
        if (k > 0.0 && rho > 0.0 && cp > 0.0) { const double d = 0.5 * rho * cp * p.h * p.h / k; if (best == 0.0 || d < best) best = d; }
    };
    take(p.rho0, p.cp_f, p.k_f);
    for (int b = 0; b < p.n_bodies; ++b)
        if (p.body[b].thermal_mode == 1) take(p.body[b].rho_s, p.body[b].cp_s, p.body[b].k_s);
    return best;
}
double particle_volume(const sph_params& p) { return is_planar(p) ? p.dx * p.dx : p.dx * p.dx * p.dx; }

void refresh_bodies(sph_ctx* ctx)
{
    const sph_params& p = ctx->prm;
    ctx->walls_moving = false;
    ctx->any_evolving = false;
    for (int b = 0; b < SPH_MAX_BODIES; ++b) {
        BodyF& f = ctx->P.body[b];
        f.ox = (float)ctx->origin[b][0]; f.oy = (float)ctx->origin[b][1]; f.oz = (float)ctx->origin[b][2];
        f.wx = (float)(ctx->omega[b] * ctx->axis[b][0]);
        f.wy = (float)(ctx->omega[b] * ctx->axis[b][1]);
        f.wz = (float)(ctx->omega[b] * ctx->axis[b][2]);
        double kn = b < p.n_bodies ? p.body[b].k_s : 0.0;
        f.K = (float)((p.k_f + kn) > 0.0 ? 4.0 * p.k_f * kn / (p.k_f + kn) : 0.0);     // Eq. 22
        f.pad = 0.f;
        if (ctx->omega[b] != 0.0) ctx->walls_moving = true;
        // evolving solid temperature (R23)
        const double C = b < p.n_bodies ? p.body[b].rho_s * p.body[b].cp_s * particle_volume(p) : 0.0;
        const int mode = (b < p.n_bodies && p.body[b].thermal_mode == 1 && C > 0.0 && (p.flags & SPH_FLAG_THERMAL)) ? 1 : 0;
        ctx->P.bk[b] = (float)kn; ctx->P.binvC[b] = mode ? (float)(1.0 / C) : 0.f; ctx->P.bmode[b] = mode;
        if (mode) ctx->any_evolving = true;
    }
}

int alloc_particles(sph_ctx* ctx, uint64_t cap_f, uint64_t cap_w)
{
    int rc;
    const uint64_t tiles = (cap_f + SPH_TP - 1) / SPH_TP;
    ctx->cap_f = cap_f; ctx->cap_w = cap_w;
    ctx->KF8 = ctx->P.KF / 8; ctx->KW8 = ctx->P.KW / 8;
    ctx->P.dummy_f = (int)cap_f; ctx->P.dummy_w = (int)cap_w;     // one extra record at the end of every sorted array
#define A_(ptr, n) if ((rc = dev_alloc(ctx, &ctx->ptr, (n))) != SPH_OK) return rc
    A_(posc, cap_f); A_(posc_s, cap_f); A_(A, cap_f + 1); A_(A_s, cap_f + 1); A_(Bc, cap_f + 1); A_(Bn, cap_f + 1); A_(B_s, cap_f + 1);
    if ((ctx->prm.flags & SPH_FLAG_VISCOUS_HELD) && (ctx->prm.flags & SPH_FLAG_VISCOUS)) { A_(avisc, cap_f); }
    A_(acc, cap_f); A_(G, cap_f); A_(orig, cap_f); A_(orig_s, cap_f); A_(rates, cap_f); A_(ncnt, cap_f); A_(fs_region, cap_f);
    A_(list_f, tiles * SPH_TP * (uint64_t)ctx->KF8); A_(list_w, tiles * SPH_TP * (uint64_t)ctx->KW8); A_(hdr, tiles * SPH_SMAX);
    A_(tile_bin, tiles); A_(tile_order, tiles);
    A_(cell_id_f, cap_f); A_(rank_f, cap_f); A_(perm_f, cap_f);
    A_(ccount_f, (uint64_t)ctx->n_cells + 1); A_(cstart_f, (uint64_t)ctx->n_cells + 1);
    A_(wref_pos, cap_w); A_(wref_nrm, cap_w); A_(wpos, cap_w); A_(wnrm, cap_w); A_(WA, cap_w + 1); A_(WB, cap_w + 1);
    A_(wbody, cap_w); A_(wT, cap_w); A_(wrate, cap_w); A_(cell_id_w, cap_w); A_(rank_w, cap_w); A_(perm_w, cap_w);
    A_(ccount_w, (uint64_t)ctx->n_cells + 1); A_(cstart_w, (uint64_t)ctx->n_cells + 1);
    ctx->n_scan_blocks = cdiv((uint64_t)ctx->n_cells, SCAN_CHUNK);
    A_(block_sums, (uint64_t)ctx->n_scan_blocks + 1);
    ctx->out_bytes = (cap_f > cap_w ? cap_f : cap_w) * 16 + 256;
    {
        char* ob = nullptr;
        if ((rc = dev_alloc(ctx, &ob, ctx->out_bytes)) != SPH_OK) return rc;
        ctx->out_buf = ob;
    }
#undef A_
    {   // dummy records (pair.cuh): far away, zero state; they survive the buffer swaps of the rebuild
        const float4 far4 = make_float4(SPH_FAR, SPH_FAR, SPH_FAR, 0.f), zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
        float4* pa[] = {ctx->A, ctx->A_s};
        float4* pb[] = {ctx->Bc, ctx->Bn, ctx->B_s};
        for (float4* q : pa) CU(cudaMemcpy(q + cap_f, &far4, sizeof(float4), cudaMemcpyHostToDevice));
        for (float4* q : pb) CU(cudaMemcpy(q + cap_f, &zero4, sizeof(float4), cudaMemcpyHostToDevice));
        CU(cudaMemcpy(ctx->WA + cap_w, &far4, sizeof(float4), cudaMemcpyHostToDevice));
        CU(cudaMemcpy(ctx->WB + cap_w, &zero4, sizeof(float4), cudaMemcpyHostToDevice));
    }
    CU(cudaFuncSetAttribute(k_build_tiles, cudaFuncAttributeMaxDynamicSharedMemorySize, SPH_BUILD_SMEM));
    CU(cudaFuncSetAttribute(k_sweep_A<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, SPH_STAGE_BYTES));
    CU(cudaFuncSetAttribute(k_sweep_A<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, SPH_STAGE_BYTES));
    CU(cudaFuncSetAttribute(k_sweep_A<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SPH_STAGE_BYTES));
    CU(cudaFuncSetAttribute(k_sweep_B, cudaFuncAttributeMaxDynamicSharedMemorySize, SPH_STAGE_BYTES));
    ctx->bank_order = getenv("SPH_NO_BANK_ORDER") ? 0 : 1;            // debugging switch
    return SPH_OK;
}

int scan_cells(sph_ctx* ctx, const uint32_t* counts, uint32_t* starts, uint32_t n_items, int pred)
{
    const int nb = ctx->n_scan_blocks;
    LAUNCH(SPH_K_SCAN, k_scan_local, nb, SCAN_THREADS, counts, starts, ctx->block_sums, ctx->n_cells, ctx->clk, pred);
    LAUNCH(SPH_K_SCAN, k_scan_sums, 1, SCAN_THREADS, ctx->block_sums, nb, ctx->clk, pred);
    LAUNCH(SPH_K_SCAN, k_scan_add, nb, SCAN_THREADS, starts, ctx->block_sums, ctx->n_cells, n_items, ctx->clk, pred);
    return SPH_OK;
}

// a1-a5: wall kinematics, cell hash, counting sort, SoA reorder, neighbour lists, density re-init
// mode 0: unconditional, sorted scratch buffers swapped in by the host;  1: every kernel predicated on Clock.rebuild,
// copy-back instead of the swap;  2: body of the step graph's conditional node (runs only when a rebuild is due):
// unpredicated kernels, copy-back
int rebuild(sph_ctx* ctx, int mode)
{
    const int pred = mode == 1 ? 1 : 0;
    const int nf = (int)ctx->n_f, nw = (int)ctx->n_w, nc = ctx->n_cells;
    Clock* clk = ctx->clk;
    if (nw > 0 && (!ctx->walls_sorted || ctx->walls_moving)) {
        LAUNCH(SPH_K_WALL_KINEMATICS, k_wall_kinematics, cdiv(nw, 256), 256, nw, ctx->wref_pos, ctx->wref_nrm, ctx->wbody, ctx->wpos,
               ctx->wnrm, clk, pred);
        CU(cudaMemsetAsync(ctx->ccount_w, 0, sizeof(uint32_t) * (size_t)(nc + 1), ctx->stream));
        LAUNCH(SPH_K_HASH, k_hash_count, cdiv(nw, 256), 256, ctx->P, ctx->wpos, nw, ctx->cell_id_w, ctx->rank_w, ctx->ccount_w, clk, pred);
        scan_cells(ctx, ctx->ccount_w, ctx->cstart_w, (uint32_t)nw, pred);
        LAUNCH(SPH_K_SCATTER, k_scatter, cdiv(nw, 256), 256, ctx->cell_id_w, ctx->rank_w, ctx->cstart_w, ctx->perm_w, nw, clk, pred);
        LAUNCH(SPH_K_SCATTER, k_cell_sort, cdiv(nc, 128), 128, ctx->cstart_w, ctx->perm_w, (const uint32_t*)nullptr, nc, clk, pred);
        LAUNCH(SPH_K_REORDER, k_reorder_wall, cdiv(nw, 256), 256, ctx->perm_w, nw, ctx->wpos, ctx->wnrm, ctx->wbody, ctx->wT, ctx->WA,
               ctx->WB, clk, pred);
        ctx->walls_sorted = true;
    }
    CU(cudaMemsetAsync(ctx->ccount_f, 0, sizeof(uint32_t) * (size_t)(nc + 1), ctx->stream));
    LAUNCH(SPH_K_HASH, k_hash_count, cdiv(nf, 256), 256, ctx->P, ctx->posc, nf, ctx->cell_id_f, ctx->rank_f, ctx->ccount_f, clk, pred);
    scan_cells(ctx, ctx->ccount_f, ctx->cstart_f, (uint32_t)nf, pred);
    LAUNCH(SPH_K_SCATTER, k_scatter, cdiv(nf, 256), 256, ctx->cell_id_f, ctx->rank_f, ctx->cstart_f, ctx->perm_f, nf, clk, pred);
    LAUNCH(SPH_K_SCATTER, k_cell_sort, cdiv(nc, 128), 128, ctx->cstart_f, ctx->perm_f, (const uint32_t*)ctx->orig, nc, clk, pred);
    LAUNCH(SPH_K_REORDER, k_reorder_fluid, cdiv(nf, 256), 256, ctx->perm_f, nf, ctx->posc, ctx->A, ctx->Bc, ctx->orig, ctx->posc_s,
           ctx->A_s, ctx->B_s, ctx->orig_s, clk, pred);
    if (mode != 0) {
        LAUNCH(SPH_K_REORDER, k_copy_back_fluid, cdiv(nf, 256), 256, nf, ctx->posc_s, ctx->A_s, ctx->B_s, ctx->orig_s, ctx->posc, ctx->A,
               ctx->Bc, ctx->orig, clk);
    } else {
        std::swap(ctx->posc, ctx->posc_s); std::swap(ctx->A, ctx->A_s); std::swap(ctx->Bc, ctx->B_s); std::swap(ctx->orig, ctx->orig_s);
    }
    {
        const double h = ctx->prm.h;
        BuildArgs a;
        a.inv_h = 1.0 / h; a.CW = wendland_alpha(h, is_planar(ctx->prm)); a.CF = -5.0 * a.CW / (h * h);
        a.sigma0 = ctx->sigma0; a.rho0 = ctx->prm.rho0; a.V0 = particle_volume(ctx->prm);
        a.A = ctx->A; a.WA = ctx->WA; a.cstart_f = ctx->cstart_f; a.cstart_w = ctx->cstart_w;
        a.list_f = ctx->list_f; a.list_w = ctx->list_w; a.ncnt = ctx->ncnt; a.G = ctx->G; a.hdr = ctx->hdr; a.clk = clk;
        a.KF8 = ctx->KF8; a.KW8 = ctx->KW8; a.pred = pred;
        a.tile_bin = ctx->tile_bin; a.order = ctx->tile_order;
        const double theta = ctx->prm.fs_threshold > 0.0 ? ctx->prm.fs_threshold : 0.9;      // R27
        a.fs_sigma = theta * ctx->sigma0; a.fs_region = ctx->fs_region;
        a.order_lists = ctx->bank_order ? 1 : 0; a.skip_short = 2;
        LAUNCH_SMEM(SPH_K_BUILD_LISTS, k_build_tiles, ctx->n_tiles, SPH_TP, SPH_BUILD_SMEM, ctx->P, a);
        if ((ctx->P.flags & F_DENSITY_REINIT) && (ctx->P.flags & F_FREE_SURFACE_LOCAL)) {       // R27: Eq. 14 in the region, Eq. 15 elsewhere
            LAUNCH(SPH_K_REINIT, k_fs_mark, ctx->n_tiles, SPH_TP, ctx->P, ctx->hdr, ctx->A, ctx->cstart_f, ctx->cstart_w, ctx->list_f, ctx->KF8,
                   ctx->ncnt, ctx->fs_region, clk, pred);
            LAUNCH(SPH_K_REINIT, k_fs_apply, cdiv(nf, 256), 256, nf, ctx->A, ctx->G, ctx->fs_region, clk, pred);
        }
        LAUNCH(SPH_K_BUILD_LISTS, k_tile_order, 1, 1024, ctx->n_tiles, SPH_TAIL_FACTOR * SPH_MINB * ctx->n_sm, ctx->tile_bin, ctx->tile_order, clk, pred);
    }
    return SPH_OK;
}

void drop_graphs(sph_ctx* ctx)
{
    for (int p = 0; p < 2; ++p)
        if (ctx->gexec[p]) { cudaGraphExecDestroy(ctx->gexec[p]); ctx->gexec[p] = nullptr; }
}

int sync_and_check(sph_ctx* ctx)
{
    CU(cudaStreamSynchronize(ctx->stream));
    unsigned int err = 0;
#ifdef SPH_BOUNDS_CHECK
    {   // debug build: the kernels' own index checks (common.cuh)
        unsigned int b = 0, zero = 0;
        CU(cudaMemcpyFromSymbol(&b, g_sph_bounds_err, sizeof(b)));
        if (b) {
            CU(cudaMemcpyToSymbol(g_sph_bounds_err, &zero, sizeof(zero)));
            return fail(ctx, SPH_ECUDA, "SPH_BOUNDS_CHECK: an index check failed in a kernel (check bits 0x%x, common.cuh / pair.cuh)", b);
        }
    }
#endif
    CU(cudaMemcpy(&err, &ctx->clk->err, sizeof(err), cudaMemcpyDeviceToHost));
    if (err) {
        unsigned int zero = 0;
        CU(cudaMemcpy(&ctx->clk->err, &zero, sizeof(zero), cudaMemcpyHostToDevice));
        if (err & ERR_NAN) return fail(ctx, SPH_ENAN, "non-finite particle position met during a neighbour rebuild");
        if (err & ERR_DOMAIN) return fail(ctx, SPH_EDOMAIN, "a particle left the grid domain (clamped into the border cell)");
        if (err & ERR_NEIGH) return fail(ctx, SPH_ENEIGH, "a neighbour list exceeded its capacity (max_neigh_fluid=%d, max_neigh_wall=%d)", ctx->P.KF, ctx->P.KW);
    }
    return SPH_OK;
}

int copy_out(sph_ctx* ctx, void* dst, const void* src_dev, uint64_t bytes, uint64_t dst_bytes, int mem_kind)
{
    if (dst_bytes < bytes) return fail(ctx, SPH_EINVAL, "destination too small: %llu < %llu bytes", (unsigned long long)dst_bytes, (unsigned long long)bytes);
    CU(cudaMemcpyAsync(dst, src_dev, bytes, mem_kind == SPH_MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    return SPH_OK;
}

uint64_t plain_field_bytes(const sph_ctx* ctx, uint32_t field)
{
    const uint64_t nf = ctx->n_f, nw = ctx->n_w;
    switch (field) {
    case SPH_FIELD_POS: case SPH_FIELD_VEL: case SPH_FIELD_ACC: case SPH_FIELD_CELL: return nf * 12;
    case SPH_FIELD_RHO: case SPH_FIELD_P: case SPH_FIELD_T: case SPH_FIELD_DRHO_DT: case SPH_FIELD_DT_DT:
    case SPH_FIELD_DRHO: case SPH_FIELD_DRHO_SAVED: case SPH_FIELD_THETA: case SPH_FIELD_FS_REGION: return nf * 4;
    case SPH_FIELD_NEIGH_COUNT: case SPH_FIELD_NEIGH_DIGEST: return nf * 8;
    case SPH_FIELD_WALL_POS: case SPH_FIELD_WALL_NORMAL: return nw * 12;
    case SPH_FIELD_CONTACT_FACTOR: case SPH_FIELD_WALL_T: case SPH_FIELD_WALL_DT_DT: return nw * 4;
    case SPH_FIELD_STATS: return SPH_STATS_COUNT * sizeof(double);
    case SPH_FIELD_SORT_CELL_COUNT: return (uint64_t)ctx->n_cells * 4;
    case SPH_FIELD_SORT_CELL_START: return ((uint64_t)ctx->n_cells + 1) * 4;
    default: return 0;
    }
}

}  // namespace

// =================================================================================================
extern "C" {

const char* sph_last_error(const sph_ctx* ctx) { return ctx ? ctx->err : g_create_error; }

int sph_create(const sph_params* p, sph_ctx** out)
{
    sph_ctx* ctx = nullptr;       // CU() reports into g_create_error until the context exists
    if (!out) return fail(nullptr, SPH_EINVAL, "out is NULL");
    *out = nullptr;
    if (!p || p->struct_size != sizeof(sph_params))
        return fail(nullptr, SPH_EINVAL, "sph_params.struct_size = %u, expected %zu", p ? p->struct_size : 0u, sizeof(sph_params));
    if (p->dim != 0 && p->dim != 2 && p->dim != 3) return fail(nullptr, SPH_EINVAL, "dim must be 0, 2 or 3");
    if (!(p->dx > 0) || !(p->h > 0) || !(p->rho0 > 0) || !(p->c0 > 0) || p->nu < 0 || p->n_bodies < 1 || p->n_bodies > SPH_MAX_BODIES)
        return fail(nullptr, SPH_EINVAL, "dx, h, rho0, c0 must be > 0, nu >= 0, 1 <= n_bodies <= %d", SPH_MAX_BODIES);
    if ((p->flags & SPH_FLAG_THERMAL) && !(p->cp_f > 0)) return fail(nullptr, SPH_EINVAL, "cp_f must be > 0 with SPH_FLAG_THERMAL");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return fail(nullptr, SPH_ECUDA, "no CUDA device: %s (this library has no CPU fallback)", cudaGetErrorString(e));
    if (p->device < 0 || p->device >= ndev) return fail(nullptr, SPH_EINVAL, "device %d out of range (%d devices)", p->device, ndev);
    CU(cudaSetDevice(p->device));

    ctx = new sph_ctx();
    ctx->prm = *p;
    ctx->stream = (cudaStream_t)p->cuda_stream;
    ctx->device = p->device;
    ctx->err[0] = 0;
    ctx->cap_f = ctx->cap_w = ctx->n_f = ctx->n_w = 0;
    ctx->loaded = ctx->walls_sorted = ctx->walls_moving = ctx->have_config = false;
    ctx->since_rebuild = 0; ctx->launches = 0; ctx->device_bytes = 0;
    ctx->prof_on = false; ctx->ev_used = 0;
    ctx->mat = nullptr; ctx->have_mat = false;
    ctx->clk = nullptr; ctx->out_buf = nullptr; ctx->stage_buf = nullptr; ctx->stage_bytes = 0;
    ctx->aux_stream = nullptr; ctx->gexec[0] = ctx->gexec[1] = nullptr; ctx->parity = 0;
    ctx->graph_fixed_launches = ctx->graph_body_per_rebuild = 0;
    {
        cudaDeviceProp prop;
        ctx->n_sm = cudaGetDeviceProperties(&prop, p->device) == cudaSuccess ? prop.multiProcessorCount : 148;
    }
    ctx->bank_order = 0;
    ctx->use_graph = getenv("SPH_NO_GRAPH") == nullptr;        // debugging switch: predicated launches instead of the step graph
    ctx->cap_stream = nullptr;
    if (cudaStreamCreateWithFlags(&ctx->aux_stream, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { ctx->use_graph = false; cudaGetLastError(); }
    if (ctx->prm.cfl_ac <= 0) ctx->prm.cfl_ac = 0.6;
    if (ctx->prm.cfl_ad <= 0) ctx->prm.cfl_ad = 0.25;
    for (int b = 0; b < SPH_MAX_BODIES; ++b) {
        for (int d = 0; d < 3; ++d) { ctx->origin[b][d] = 0.0; ctx->axis[b][d] = d == 2 ? 1.0 : 0.0; }
        ctx->omega[b] = 0.0;
    }

    DevParams& P = ctx->P;
    memset(&P, 0, sizeof(P));
    // grid (R1): cell edge 2h(1 + 2^-10), inverse rounded once to fp32; sizes from fp32 arithmetic
    const double ell = 2.0 * p->h * (1.0 + 1.0 / 1024.0);
    P.inv_ell = (float)(1.0 / ell);
    long long nc = 1;
    for (int d = 0; d < 3; ++d) {
        P.xmin[d] = (float)p->domain_min[d];
        volatile float ext = (float)p->domain_max[d] - P.xmin[d];
        volatile float s = ext * P.inv_ell;
        if (!(s >= 0.0f) || s > 2047.0f) {
            delete ctx;
            return fail(nullptr, SPH_EINVAL, "domain axis %d spans %g cells; must be within [0, 2047]", d, (double)s);
        }
        P.ng[d] = (int)floorf(s) + 1;
        nc *= P.ng[d];
    }
    if (nc > 500000000ll) { delete ctx; return fail(nullptr, SPH_EINVAL, "grid has %lld cells (> 5e8)", nc); }
    P.n_cells = ctx->n_cells = (int)nc * SPH_SX;      // sort cells (common.cuh: fine_coord)
    P.inv_ell4 = P.inv_ell * (float)SPH_SX;
    P.nfx = P.ng[0] * SPH_SX;
    {
        const double rcu = (double)(float)(2.0 * p->h) * (double)P.inv_ell;
        P.rcu2 = (float)(rcu * rcu * (1.0 + 1.0e-4));
    }
    {
        float rc = (float)(2.0 * p->h);
        volatile float rc2 = rc * rc;
        P.rc2 = rc2;
    }
    const double h = p->h;
    P.h = (float)h; P.inv_h = (float)(1.0 / h); P.half_inv_h = (float)(0.5 / h);
    P.CW = (float)wendland_alpha(h, is_planar(*p));
    P.CF = (float)(-5.0 * wendland_alpha(h, is_planar(*p)) / (h * h));      // W'/r = -(5 alpha / h^2)(1 - q/2)^3
    P.rho0 = (float)p->rho0; P.c0 = (float)p->c0; P.c0sq = (float)(p->c0 * p->c0);
    P.inv_c0 = (float)(1.0 / p->c0); P.inv_c0sq = (float)(1.0 / (p->c0 * p->c0));
    P.eta = (float)(p->rho0 * p->nu);
    P.mass = (float)(p->rho0 * particle_volume(*p));
    P.Vw = (float)particle_volume(*p);
    P.gx = (float)p->g[0]; P.gy = (float)p->g[1]; P.gz = (float)p->g[2];
    P.k2f = (float)(2.0 * p->k_f);
    P.inv_cp = p->cp_f > 0 ? (float)(1.0 / p->cp_f) : 0.f;
    P.flags = p->flags;
    P.KF = ((p->max_neigh_fluid ? (int)p->max_neigh_fluid : 160) + 7) & ~7;
    P.KW = ((p->max_neigh_wall ? (int)p->max_neigh_wall : 96) + 7) & ~7;
    P.inv_rho0 = (float)(1.0 / p->rho0);
    if (P.KF > 65535 || P.KW > 65535) { delete ctx; return fail(nullptr, SPH_EINVAL, "max_neigh_* must be < 65536"); }
    ctx->sigma0 = lattice_sigma0(p->dx, p->h, is_planar(*p));
    refresh_bodies(ctx);

    int rc = dev_alloc(ctx, &ctx->clk, 1);
    if (rc != SPH_OK) { strncpy(g_create_error, ctx->err, 511); delete ctx; return rc; }
    if (p->max_fluid) {
        rc = alloc_particles(ctx, p->max_fluid, p->max_wall);
        if (rc != SPH_OK) { strncpy(g_create_error, ctx->err, 511); free_all(ctx); delete ctx; return rc; }
    }
    *out = ctx;
    return SPH_OK;
}

int sph_destroy(sph_ctx* ctx)
{
    if (!ctx) return SPH_OK;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (cudaEvent_t e : ctx->ev_pool) cudaEventDestroy(e);
    drop_graphs(ctx);
    if (ctx->aux_stream) cudaStreamDestroy(ctx->aux_stream);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    free_all(ctx);
    delete ctx;
    return SPH_OK;
}

int sph_load_particles(sph_ctx* ctx, uint64_t n_f, const float* pos_f, const float* vel_f, const float* rho_f, const float* T_f,
                       uint64_t n_w, const float* pos_w, const float* normal_w, const int32_t* body_w, const float* T_w, int mem_kind)
{
    if (!ctx) return SPH_EINVAL;
    if (n_f == 0 || !pos_f) return fail(ctx, SPH_EINVAL, "n_f must be > 0 and pos_f non-NULL");
    if (n_w > 0 && (!pos_w || !normal_w)) return fail(ctx, SPH_EINVAL, "pos_w and normal_w are required when n_w > 0");
    if (n_f > 2000000000ull || n_w > 2000000000ull) return fail(ctx, SPH_EINVAL, "particle counts must be < 2e9");
    if (mem_kind != SPH_MEM_HOST && mem_kind != SPH_MEM_DEVICE) return fail(ctx, SPH_EINVAL, "bad mem_kind %d", mem_kind);
    CU(cudaSetDevice(ctx->device));
    if (ctx->cap_f == 0) {
        int rc = alloc_particles(ctx, n_f, n_w);
        if (rc != SPH_OK) return rc;
    }
    if (n_f > ctx->cap_f || n_w > ctx->cap_w)
        return fail(ctx, SPH_EINVAL, "n_f=%llu / n_w=%llu exceed the capacity %llu / %llu", (unsigned long long)n_f, (unsigned long long)n_w,
                    (unsigned long long)ctx->cap_f, (unsigned long long)ctx->cap_w);
    if (ctx->n_f != n_f || ctx->n_w != n_w) drop_graphs(ctx);   // grids and counts are baked into the step graphs
    ctx->n_f = n_f; ctx->n_w = n_w;
    ctx->P.n_f = (int)n_f; ctx->P.n_w = (int)n_w;
    ctx->n_tiles = cdiv(n_f, SPH_TP);
    if (ctx->n_tiles > 0)       // tile schedule before the first rebuild: index order (k_build_tiles walks the previous schedule)
        LAUNCH(SPH_K_OTHER, k_tile_order_identity, cdiv((uint64_t)ctx->n_tiles, 256), 256, ctx->n_tiles, ctx->tile_order);

    // stage host inputs on the device: one persistent buffer (no allocation or free on the per-call path)
    if (mem_kind == SPH_MEM_HOST) {
        const uint64_t need = ctx->cap_f * 32 + ctx->cap_w * 32 + 8 * 256;
        if (ctx->stage_bytes < need) {
            int rc0 = dev_alloc(ctx, &ctx->stage_buf, need);
            if (rc0 != SPH_OK) return rc0;
            ctx->stage_bytes = need;
        }
    }
    uint64_t stage_off = 0;
    auto stage = [&](const void* src, uint64_t bytes, const void** dev) -> int {
        *dev = nullptr;
        if (!src || bytes == 0) return SPH_OK;
        if (mem_kind == SPH_MEM_DEVICE) { *dev = src; return SPH_OK; }
        void* q = ctx->stage_buf + stage_off;
        stage_off += (bytes + 255) & ~(uint64_t)255;
        cudaError_t e = cudaMemcpyAsync(q, src, bytes, cudaMemcpyHostToDevice, ctx->stream);
        if (e != cudaSuccess) return fail(ctx, SPH_ECUDA, "H2D copy failed: %s", cudaGetErrorString(e));
        *dev = q;
        return SPH_OK;
    };
    const void *d_pos, *d_vel, *d_rho, *d_T, *d_pw, *d_nw, *d_bw, *d_Tw;
    int rc = SPH_OK;
    if ((rc = stage(pos_f, n_f * 12, &d_pos)) || (rc = stage(vel_f, n_f * 12, &d_vel)) || (rc = stage(rho_f, n_f * 4, &d_rho)) ||
        (rc = stage(T_f, n_f * 4, &d_T)) || (rc = stage(pos_w, n_w * 12, &d_pw)) || (rc = stage(normal_w, n_w * 12, &d_nw)) ||
        (rc = stage(body_w, n_w * 4, &d_bw)) || (rc = stage(T_w, n_w * 4, &d_Tw)))
        return rc;

    // clock
    Clock hc;
    memset(&hc, 0, sizeof(hc));
    const sph_params& p = ctx->prm;
    hc.cfl_ac = p.cfl_ac; hc.cfl_ad = p.cfl_ad; hc.u_ref = p.u_ref; hc.dt_fixed = p.dt_fixed; hc.h = p.h; hc.c0 = p.c0; hc.nu = p.nu;
    hc.rebuild_every = p.rebuild_every;
    hc.dt_T = thermal_dt_bound(p);
    for (int b = 0; b < SPH_MAX_BODIES; ++b) {
        for (int d = 0; d < 3; ++d) { hc.body[b].origin[d] = ctx->origin[b][d]; hc.body[b].axis[d] = ctx->axis[b][d]; }
        hc.body[b].omega = ctx->omega[b]; hc.body[b].theta = 0.0; hc.body[b].cs = 1.0; hc.body[b].sn = 0.0;
    }
    hc.walls_moving = ctx->walls_moving;
    CU(cudaMemcpyAsync(ctx->clk, &hc, sizeof(hc), cudaMemcpyHostToDevice, ctx->stream));
    if (body_w && mem_kind == SPH_MEM_HOST)      // host-side check of the body indices while the copies are in flight
        for (uint64_t w = 0; w < n_w; ++w)
            if (body_w[w] < 0 || body_w[w] >= p.n_bodies) {
                cudaStreamSynchronize(ctx->stream);          // the copies read the caller's buffers
                ctx->loaded = false;
                return fail(ctx, SPH_EINVAL, "body_w[%llu] = %d outside [0, %d)", (unsigned long long)w, body_w[w], p.n_bodies);
            }
    // (hc is pageable stack memory: cudaMemcpyAsync has staged it before returning, no synchronisation is needed for it)

    const int nf = (int)n_f, nw = (int)n_w;
    unsigned int bad_body = 0u;
    LAUNCH(SPH_K_OTHER, k_init_fluid, cdiv(nf, 256), 256, nf, (const float*)d_pos, (const float*)d_vel, (const float*)d_rho, (const float*)d_T,
           (float)p.rho0, (float)p.T_ref, ctx->posc, ctx->A, ctx->Bc, ctx->orig, ctx->clk);
    LAUNCH(SPH_K_OTHER, k_init_vmax, 1, 1, ctx->clk);
    if (nw > 0) {
        LAUNCH(SPH_K_OTHER, k_init_wall, cdiv(nw, 256), 256, nw, (const float*)d_pw, (const float*)d_nw, (const float*)d_Tw, (float)p.T_ref,
               ctx->wref_pos, ctx->wref_nrm, ctx->wpos, ctx->wnrm, ctx->wT);
        if (d_bw) CU(cudaMemcpyAsync(ctx->wbody, d_bw, n_w * 4, cudaMemcpyDeviceToDevice, ctx->stream));
        else CU(cudaMemsetAsync(ctx->wbody, 0, n_w * 4, ctx->stream));
        if (d_bw && mem_kind == SPH_MEM_DEVICE) {          // the host cannot read the caller's device array: check it on the device
            CU(cudaMemsetAsync(ctx->out_buf, 0, sizeof(unsigned int), ctx->stream));
            LAUNCH(SPH_K_OTHER, k_check_body, cdiv(nw, 256), 256, nw, ctx->wbody, p.n_bodies, (unsigned int*)ctx->out_buf);
            CU(cudaMemcpyAsync(&bad_body, ctx->out_buf, sizeof(unsigned int), cudaMemcpyDeviceToHost, ctx->stream));
        }
    }
    CU(cudaMemsetAsync(ctx->acc, 0, n_f * sizeof(float4), ctx->stream));
    CU(cudaMemsetAsync(ctx->rates, 0, n_f * sizeof(float2), ctx->stream));
    CU(cudaMemsetAsync(ctx->ncnt, 0, n_f * sizeof(uint32_t), ctx->stream));
    CU(cudaMemsetAsync(ctx->fs_region, 0, n_f, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));          // the caller's buffers may be reused on return
    if (bad_body) { ctx->loaded = false; return fail(ctx, SPH_EINVAL, "body_w holds an index outside [0, %d)", p.n_bodies); }
    ctx->loaded = true; ctx->walls_sorted = false; ctx->have_config = false; ctx->since_rebuild = 0;
    if (ctx->have_mat) { ctx->have_mat = false; drop_graphs(ctx); }      // a load returns to uniform materials
    CU(cudaGetLastError());
    return SPH_OK;
}

int sph_set_materials(sph_ctx* ctx, const float* mass_f, const float* k_f, const float* cp_f, int mem_kind)
{
    if (!ctx) return SPH_EINVAL;
    if (!ctx->loaded) return fail(ctx, SPH_ESTATE, "sph_set_materials before sph_load_particles");
    if (mem_kind != SPH_MEM_HOST && mem_kind != SPH_MEM_DEVICE) return fail(ctx, SPH_EINVAL, "bad mem_kind %d", mem_kind);
    if (mass_f && (ctx->prm.flags & SPH_FLAG_HYDRO))
        return fail(ctx, SPH_EINVAL, "per-particle masses enter the heat equation only (Eq. 20-22); mass_f must be NULL with SPH_FLAG_HYDRO");
    CU(cudaSetDevice(ctx->device));
    drop_graphs(ctx);                                 // the step graphs are captured with or without the materials kernel
    if (!mass_f && !k_f && !cp_f) { ctx->have_mat = false; return SPH_OK; }
    const uint64_t n_f = ctx->n_f;
    if (!ctx->mat) {
        int rc = dev_alloc(ctx, &ctx->mat, ctx->cap_f);
        if (rc != SPH_OK) return rc;
    }
    float* stage = nullptr;
    const float* dev[3] = {mass_f, k_f, cp_f};
    if (mem_kind == SPH_MEM_HOST) {
        CU(cudaMalloc(&stage, 3 * n_f * sizeof(float)));
        for (int k = 0; k < 3; ++k)
            if (dev[k]) {
                cudaError_t e = cudaMemcpyAsync(stage + k * n_f, dev[k], n_f * sizeof(float), cudaMemcpyHostToDevice, ctx->stream);
                if (e != cudaSuccess) { cudaFree(stage); return fail(ctx, SPH_ECUDA, "H2D copy failed: %s", cudaGetErrorString(e)); }
                dev[k] = stage + k * n_f;
            }
    }
    const sph_params& p = ctx->prm;
    LAUNCH(SPH_K_OTHER, k_set_materials, cdiv(n_f, 256), 256, (int)n_f, dev[0], dev[1], dev[2], (float)(p.rho0 * particle_volume(p)), (float)p.k_f,
           (float)p.cp_f, ctx->mat);
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    if (stage) cudaFree(stage);
    if (e != cudaSuccess) return fail(ctx, SPH_ECUDA, "sph_set_materials: %s", cudaGetErrorString(e));
    ctx->have_mat = true;
    return SPH_OK;
}

int sph_set_state(sph_ctx* ctx, const float* pos_f, const float* vel_f, const float* rho_f, const float* T_f, int mem_kind)
{
    if (!ctx) return SPH_EINVAL;
    if (!ctx->loaded) return fail(ctx, SPH_ESTATE, "sph_set_state before sph_load_particles");
    if (mem_kind != SPH_MEM_HOST && mem_kind != SPH_MEM_DEVICE) return fail(ctx, SPH_EINVAL, "bad mem_kind %d", mem_kind);
    CU(cudaSetDevice(ctx->device));
    const uint64_t n_f = ctx->n_f;
    if (mem_kind == SPH_MEM_HOST) {
        const uint64_t need = ctx->cap_f * 32 + ctx->cap_w * 32 + 8 * 256;
        if (ctx->stage_bytes < need) {
            int rc0 = dev_alloc(ctx, &ctx->stage_buf, need);
            if (rc0 != SPH_OK) return rc0;
            ctx->stage_bytes = need;
        }
    }
    uint64_t off = 0;
    const void* dev[4] = {nullptr, nullptr, nullptr, nullptr};
    const void* src[4] = {pos_f, vel_f, rho_f, T_f};
    const uint64_t bytes[4] = {n_f * 12, n_f * 12, n_f * 4, n_f * 4};
    for (int k = 0; k < 4; ++k) {
        if (!src[k]) continue;
        if (mem_kind == SPH_MEM_DEVICE) { dev[k] = src[k]; continue; }
        void* q = ctx->stage_buf + off;
        off += (bytes[k] + 255) & ~(uint64_t)255;
        CU(cudaMemcpyAsync(q, src[k], bytes[k], cudaMemcpyHostToDevice, ctx->stream));
        dev[k] = q;
    }
    const int nf = (int)n_f;
    LAUNCH(SPH_K_OTHER, k_state_changed, 1, 1, ctx->clk, 1);
    LAUNCH(SPH_K_OTHER, k_set_state, cdiv(nf, 256), 256, nf, (const float*)dev[0], (const float*)dev[1], (const float*)dev[2], (const float*)dev[3],
           (float)ctx->prm.rho0, (float)ctx->prm.T_ref, ctx->orig, ctx->posc, ctx->A, ctx->Bc, ctx->clk);
    LAUNCH(SPH_K_OTHER, k_state_changed, 1, 1, ctx->clk, 0);
    unsigned int moved = 1u;
    CU(cudaMemcpyAsync(&moved, &ctx->clk->state_moved, sizeof(moved), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));          // the caller's buffers may be reused on return
    if (moved) { ctx->have_config = false; ctx->since_rebuild = 0; }      // else the configuration (and the step graph) stand
    CU(cudaGetLastError());
    return SPH_OK;
}

int sph_set_gear_kinematics(sph_ctx* ctx, int body, const double origin[3], const double axis[3], double omega)
{
    if (!ctx) return SPH_EINVAL;
    if (body < 0 || body >= ctx->prm.n_bodies || !origin || !axis) return fail(ctx, SPH_EINVAL, "bad body %d or NULL origin/axis", body);
    double n = std::sqrt(axis[0] * axis[0] + axis[1] * axis[1] + axis[2] * axis[2]);
    if (!(n > 0.0)) return fail(ctx, SPH_EINVAL, "axis must be non-zero");
    for (int d = 0; d < 3; ++d) { ctx->origin[body][d] = origin[d]; ctx->axis[body][d] = axis[d] / n; }
    ctx->omega[body] = omega;
    refresh_bodies(ctx);
    drop_graphs(ctx);                              // DevParams (body table) is a by-value kernel argument of the graph nodes
    if (ctx->loaded) {
        // bring all body angles up to the present time with the speeds valid so far, then switch
        CU(cudaSetDevice(ctx->device));
        CU(cudaStreamSynchronize(ctx->stream));
        Clock hc;
        CU(cudaMemcpy(&hc, ctx->clk, sizeof(hc), cudaMemcpyDeviceToHost));
        for (int b = 0; b < SPH_MAX_BODIES; ++b) hc.body[b].theta += hc.body[b].omega * (hc.t - hc.t_kin);
        hc.t_kin = hc.t;
        for (int d = 0; d < 3; ++d) { hc.body[body].origin[d] = ctx->origin[body][d]; hc.body[body].axis[d] = ctx->axis[body][d]; }
        hc.body[body].omega = omega;
        hc.walls_moving = ctx->walls_moving;
        CU(cudaMemcpy(ctx->clk, &hc, sizeof(hc), cudaMemcpyHostToDevice));
    }
    return SPH_OK;
}

}  // extern "C"

namespace {

// a7-a11 + clock of one acoustic step (everything after the control kernel and the rebuild)
int enqueue_step_tail(sph_ctx* ctx)
{
    const int nf = (int)ctx->n_f;
    const int hydro = (ctx->prm.flags & SPH_FLAG_HYDRO) ? 1 : 0;
    if (hydro) {
        LAUNCH(SPH_K_PRE, k_pre, cdiv(nf, 256), 256, nf, ctx->A, ctx->Bc, ctx->posc, ctx->clk);
        SweepAArgs a;
        a.A = ctx->A; a.Bc = ctx->Bc; a.WA = ctx->WA; a.G = ctx->G; a.Bn = ctx->Bn; a.posc = ctx->posc; a.acc = ctx->acc;
        a.list_f = ctx->list_f; a.list_w = ctx->list_w; a.ncnt = ctx->ncnt; a.cstart_f = ctx->cstart_f; a.cstart_w = ctx->cstart_w;
        a.hdr = ctx->hdr; a.order = ctx->tile_order; a.clk = ctx->clk; a.KF8 = ctx->KF8; a.KW8 = ctx->KW8; a.avisc = ctx->avisc;
        const int grid = std::min(SPH_MINB * ctx->n_sm, ctx->n_tiles);
        if (ctx->avisc) {       // R26: the step that rebuilt renews the viscous sums (<1>), the others add the held ones (<2>);
                                // Clock.rebuild decides on the device which of the two runs, the other returns at once
            LAUNCH_SMEM(SPH_K_SWEEP_A, k_sweep_A<1>, grid, SPH_TP, SPH_STAGE_BYTES, ctx->P, a, ctx->n_tiles, &ctx->clk->work_A);
            LAUNCH_SMEM(SPH_K_SWEEP_A, k_sweep_A<2>, grid, SPH_TP, SPH_STAGE_BYTES, ctx->P, a, ctx->n_tiles, &ctx->clk->work_A);
        } else {
            LAUNCH_SMEM(SPH_K_SWEEP_A, k_sweep_A<0>, grid, SPH_TP, SPH_STAGE_BYTES, ctx->P, a, ctx->n_tiles, &ctx->clk->work_A);
        }
        std::swap(ctx->Bc, ctx->Bn);
        ctx->parity ^= 1;
    }
    {
        SweepBArgs b;
        b.A = ctx->A; b.B = ctx->Bc; b.WA = ctx->WA; b.WB = ctx->WB; b.list_f = ctx->list_f; b.list_w = ctx->list_w; b.ncnt = ctx->ncnt;
        b.cstart_f = ctx->cstart_f; b.cstart_w = ctx->cstart_w; b.hdr = ctx->hdr; b.order = ctx->tile_order; b.rates = ctx->rates; b.KF8 = ctx->KF8; b.KW8 = ctx->KW8;
        LAUNCH_SMEM(SPH_K_SWEEP_B, k_sweep_B, std::min(SPH_MINB * ctx->n_sm, ctx->n_tiles), SPH_TP, SPH_STAGE_BYTES, ctx->P, b, ctx->n_tiles, &ctx->clk->work_B);
    }
    if (ctx->have_mat && (ctx->prm.flags & SPH_FLAG_THERMAL))      // Eq. 20-22 with per-particle m, k, cp: replaces sweep B's dT/dt
        LAUNCH(SPH_K_SWEEP_B, k_heat_materials, ctx->n_tiles, SPH_TP, ctx->P, ctx->hdr, ctx->A, ctx->Bc, ctx->WA, ctx->WB, ctx->cstart_f, ctx->cstart_w,
               ctx->list_f, ctx->list_w, ctx->KF8, ctx->KW8, ctx->ncnt, ctx->orig, ctx->mat, ctx->rates);
    const bool wall_heat = ctx->any_evolving && ctx->n_w > 0;
    if (wall_heat)                                   // R23: T^n on both sides, so before the finish kernels
        LAUNCH(SPH_K_OTHER, k_wall_heat, cdiv(ctx->n_w, 128), 128, ctx->P, ctx->A, ctx->Bc, ctx->WA, ctx->WB, ctx->cstart_f, ctx->cstart_w, ctx->wrate);
    LAUNCH(SPH_K_FINISH, k_finish, cdiv(nf, 256), 256, nf, hydro, ctx->A, ctx->Bc, ctx->posc, ctx->rates, ctx->clk);
    if (wall_heat)
        LAUNCH(SPH_K_FINISH, k_finish_wall, cdiv(ctx->n_w, 256), 256, (int)ctx->n_w, ctx->WB, ctx->wT, ctx->wrate, ctx->perm_w, ctx->clk);
    return SPH_OK;
}

// Capture one acoustic step for the current ping-pong parity:
//   k_control (sets the condition) -> IF (rebuild due) { a1-a5 } -> a7 ... a11, clock.
// Nothing executes during capture; host-side pointer roles and counters are restored afterwards.
int capture_step_graph(sph_ctx* ctx)
{
    const int p = ctx->parity;
    const int hydro = (ctx->prm.flags & SPH_FLAG_HYDRO) ? 1 : 0;
    float4 *sBc = ctx->Bc, *sBn = ctx->Bn;
    const uint64_t l0 = ctx->launches;
    const bool ws = ctx->walls_sorted;
    cudaStream_t user_stream = ctx->stream, main_stream = ctx->cap_stream;
    ctx->stream = main_stream;
    cudaGraph_t graph = nullptr, body = nullptr;
    cudaError_t e;
    auto bail = [&](const char* what, cudaError_t err) {
        cudaGraph_t junk = nullptr;
        cudaStreamCaptureStatus st;
        if (cudaStreamIsCapturing(main_stream, &st) == cudaSuccess && st != cudaStreamCaptureStatusNone) cudaStreamEndCapture(main_stream, &junk);
        if (junk) cudaGraphDestroy(junk);
        ctx->stream = user_stream; ctx->Bc = sBc; ctx->Bn = sBn; ctx->parity = p; ctx->launches = l0; ctx->walls_sorted = ws;
        cudaGetLastError();
        ctx->use_graph = false;                        // fall back to predicated launches for good
        fprintf(stderr, "libsph_b200: step graph disabled (%s failed: %s); using predicated launches\n", what, cudaGetErrorString(err));
        return fail(ctx, SPH_OK, "step graph disabled: %s failed: %s", what, cudaGetErrorString(err));
    };
    if ((e = cudaStreamBeginCapture(main_stream, cudaStreamCaptureModeThreadLocal)) != cudaSuccess) return bail("cudaStreamBeginCapture", e);
    cudaStreamCaptureStatus st;
    const cudaGraphNode_t* deps = nullptr;
    size_t ndeps = 0;
    if ((e = cudaStreamGetCaptureInfo(main_stream, &st, nullptr, &graph, &deps, &ndeps)) != cudaSuccess) return bail("cudaStreamGetCaptureInfo", e);
    cudaGraphConditionalHandle handle;
    if ((e = cudaGraphConditionalHandleCreate(&handle, graph, 0, cudaGraphCondAssignDefault)) != cudaSuccess) return bail("cudaGraphConditionalHandleCreate", e);
    LAUNCH(SPH_K_CONTROL, k_control, 1, 1, ctx->clk, hydro, handle, 1);
    if ((e = cudaStreamGetCaptureInfo(main_stream, &st, nullptr, &graph, &deps, &ndeps)) != cudaSuccess) return bail("cudaStreamGetCaptureInfo", e);
    cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = handle;
    np.conditional.type = cudaGraphCondTypeIf;
    np.conditional.size = 1;
    cudaGraphNode_t cond_node;
    if ((e = cudaGraphAddNode(&cond_node, graph, deps, ndeps, &np)) != cudaSuccess) return bail("cudaGraphAddNode(conditional)", e);
    body = np.conditional.phGraph_out[0];
    const uint64_t lb0 = ctx->launches;
    if ((e = cudaStreamBeginCaptureToGraph(ctx->aux_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal)) != cudaSuccess)
        return bail("cudaStreamBeginCaptureToGraph", e);
    ctx->stream = ctx->aux_stream;
    int rc = rebuild(ctx, 2);
    ctx->stream = main_stream;
    cudaGraph_t body_out = nullptr;
    e = cudaStreamEndCapture(ctx->aux_stream, &body_out);
    if (rc != SPH_OK || e != cudaSuccess) return bail("capture of the rebuild chain", e);
    const uint64_t body_launches = ctx->launches - lb0;
    if ((e = cudaStreamUpdateCaptureDependencies(main_stream, &cond_node, 1, cudaStreamSetCaptureDependencies)) != cudaSuccess)
        return bail("cudaStreamUpdateCaptureDependencies", e);
    if (enqueue_step_tail(ctx) != SPH_OK) return bail("capture of the step tail", cudaGetLastError());
    if ((e = cudaStreamEndCapture(main_stream, &graph)) != cudaSuccess) return bail("cudaStreamEndCapture", e);
    e = cudaGraphInstantiate(&ctx->gexec[p], graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { ctx->gexec[p] = nullptr; return bail("cudaGraphInstantiate", e); }
    ctx->g_body[p] = body_launches;
    ctx->g_fixed[p] = ctx->launches - l0 - body_launches;
    ctx->stream = user_stream; ctx->Bc = sBc; ctx->Bn = sBn; ctx->parity = p; ctx->launches = l0; ctx->walls_sorted = ws;
    return SPH_OK;
}

}  // namespace

extern "C" {

int sph_step(sph_ctx* ctx, int n)
{
    if (!ctx) return SPH_EINVAL;
    if (!ctx->loaded) return fail(ctx, SPH_ESTATE, "sph_step before sph_load_particles");
    if (n < 0) return fail(ctx, SPH_EINVAL, "n must be >= 0");
    CU(cudaSetDevice(ctx->device));
    const int hydro = (ctx->prm.flags & SPH_FLAG_HYDRO) ? 1 : 0;
    const int K = ctx->prm.rebuild_every;
    for (int s = 0; s < n; ++s) {
        // device-decided rebuilds (K = 0), configuration and sorted walls present, no per-kernel timing: one graph launch
        if (K < 1 && ctx->use_graph && ctx->have_config && !ctx->prof_on && hydro) {
            const int p = ctx->parity;
            if (!ctx->gexec[p]) capture_step_graph(ctx);
            if (ctx->gexec[p]) {
                CU(cudaGraphLaunch(ctx->gexec[p], ctx->stream));
                std::swap(ctx->Bc, ctx->Bn);
                ctx->parity ^= 1;
                ctx->graph_fixed_launches += ctx->g_fixed[p];
                ctx->graph_body_per_rebuild = ctx->g_body[p];
                ctx->since_rebuild++;
                continue;
            }
        }
        LAUNCH(SPH_K_CONTROL, k_control, 1, 1, ctx->clk, hydro, (cudaGraphConditionalHandle)0, 0);
        if (K >= 1) {                                   // rebuild schedule known to the host
            if (!ctx->have_config || ctx->since_rebuild >= K) {
                int rc = rebuild(ctx, 0);
                if (rc != SPH_OK) return rc;
                ctx->have_config = true; ctx->since_rebuild = 0;
            }
        } else {                                        // Eq. 25 l.1 decides on the device: predicated launches
            int rc = rebuild(ctx, 1);
            if (rc != SPH_OK) return rc;
            ctx->have_config = true;
        }
        int rc = enqueue_step_tail(ctx);
        if (rc != SPH_OK) return rc;
        ctx->since_rebuild++;
    }
    CU(cudaGetLastError());
    return SPH_OK;
}

int sph_relax(sph_ctx* ctx, int n, double p0)
{
    if (!ctx) return SPH_EINVAL;
    if (!ctx->loaded) return fail(ctx, SPH_ESTATE, "sph_relax before sph_load_particles");
    if (n < 0 || !(p0 > 0.0)) return fail(ctx, SPH_EINVAL, "n must be >= 0 and p0 > 0");
    CU(cudaSetDevice(ctx->device));
    const int nf = (int)ctx->n_f;
    const float c = (float)(-2.0 * p0 / ctx->prm.rho0);
    const uint32_t flags = ctx->P.flags;
    ctx->P.flags &= ~F_DENSITY_REINIT;               // relaxation moves particles only (R24)
    int rc = SPH_OK;
    for (int s = 0; s < n && rc == SPH_OK; ++s) {
        LAUNCH(SPH_K_CONTROL, k_relax_begin, 1, 1, ctx->clk);
        rc = rebuild(ctx, 2);                        // unpredicated kernels, copy-back: buffer roles stay as the step graphs know them
        LAUNCH(SPH_K_OTHER, k_relax_force, cdiv(nf, 256), 256, nf, c, ctx->G, ctx->clk);
        LAUNCH(SPH_K_OTHER, k_relax_move, cdiv(nf, 256), 256, nf, c, (float)ctx->prm.h, ctx->G, ctx->posc, ctx->clk);
    }
    LAUNCH(SPH_K_CONTROL, k_relax_end, 1, 1, ctx->clk);
    ctx->P.flags = flags;
    ctx->have_config = false;                        // the next sph_step rebuilds for the moved particles
    ctx->since_rebuild = 0;
    if (rc != SPH_OK) return rc;
    CU(cudaGetLastError());
    return SPH_OK;
}

int sph_synchronize(sph_ctx* ctx)
{
    if (!ctx) return SPH_EINVAL;
    CU(cudaSetDevice(ctx->device));
    return sync_and_check(ctx);
}

int sph_field_bytes(sph_ctx* ctx, uint32_t field, uint64_t* bytes)
{
    if (!ctx || !bytes) return SPH_EINVAL;
    if (!ctx->loaded) return fail(ctx, SPH_ESTATE, "no particles loaded");
    if (field == SPH_FIELD_NEIGH_CSR_FLUID || field == SPH_FIELD_NEIGH_CSR_WALL) {
        CU(cudaSetDevice(ctx->device));
        CU(cudaStreamSynchronize(ctx->stream));
        std::vector<uint32_t> c(ctx->n_f);
        CU(cudaMemcpy(c.data(), ctx->ncnt, ctx->n_f * 4, cudaMemcpyDeviceToHost));
        uint64_t tot = 0;
        for (uint32_t x : c) tot += field == SPH_FIELD_NEIGH_CSR_FLUID ? (x & 0xffffu) : (x >> 16);
        *bytes = tot * 4;
        return SPH_OK;
    }
    uint64_t b = plain_field_bytes(ctx, field);
    if (b == 0 && !(field == SPH_FIELD_WALL_POS || field == SPH_FIELD_WALL_NORMAL || field == SPH_FIELD_CONTACT_FACTOR || field == SPH_FIELD_WALL_T || field == SPH_FIELD_WALL_DT_DT)) return fail(ctx, SPH_EINVAL, "unknown field %u", field);
    *bytes = b;
    return SPH_OK;
}

int sph_get_fields(sph_ctx* ctx, uint32_t field, void* dst, uint64_t dst_bytes, int mem_kind)
{
    if (!ctx) return SPH_EINVAL;
    if (!ctx->loaded) return fail(ctx, SPH_ESTATE, "sph_get_fields before sph_load_particles");
    if (!dst) return fail(ctx, SPH_EINVAL, "dst is NULL");
    if (mem_kind != SPH_MEM_HOST && mem_kind != SPH_MEM_DEVICE) return fail(ctx, SPH_EINVAL, "bad mem_kind %d", mem_kind);
    CU(cudaSetDevice(ctx->device));
    const int nf = (int)ctx->n_f, nw = (int)ctx->n_w;
    int rc = SPH_OK;
    int what = -1;
    switch (field) {
    case SPH_FIELD_POS: what = X_POS; break;
    case SPH_FIELD_VEL: what = X_VEL; break;
    case SPH_FIELD_RHO: what = X_RHO; break;
    case SPH_FIELD_P: what = X_P; break;
    case SPH_FIELD_T: what = X_T; break;
    case SPH_FIELD_ACC: what = X_ACC; break;
    case SPH_FIELD_DRHO_DT: what = X_DRHO_DT; break;
    case SPH_FIELD_DT_DT: what = X_DT_DT; break;
    case SPH_FIELD_CELL: what = X_CELL; break;
    case SPH_FIELD_NEIGH_COUNT: what = X_NCOUNT; break;
    case SPH_FIELD_DRHO: what = X_DRHO; break;
    case SPH_FIELD_DRHO_SAVED: what = X_DRHO_SAVED; break;
    case SPH_FIELD_THETA: what = X_THETA; break;
    case SPH_FIELD_FS_REGION: what = X_FS_REGION; break;
    default: break;
    }
    if (what >= 0) {
        LAUNCH(SPH_K_OTHER, k_extract, cdiv(nf, 256), 256, ctx->P, what, (float)ctx->prm.T_ref, ctx->posc, ctx->A, ctx->Bc, ctx->acc, ctx->rates,
               ctx->ncnt, ctx->fs_region, ctx->orig, ctx->out_buf);
        if ((rc = copy_out(ctx, dst, ctx->out_buf, plain_field_bytes(ctx, field), dst_bytes, mem_kind)) != SPH_OK) return rc;
        return sync_and_check(ctx);
    }
    switch (field) {
    case SPH_FIELD_NEIGH_DIGEST:
        LAUNCH(SPH_K_OTHER, k_neigh_digest, ctx->n_tiles, SPH_TP, ctx->P, ctx->hdr, ctx->A, ctx->cstart_f, ctx->cstart_w, ctx->list_f, ctx->list_w,
               ctx->KF8, ctx->KW8, ctx->ncnt, ctx->orig, ctx->perm_w, (uint64_t*)ctx->out_buf);
        if ((rc = copy_out(ctx, dst, ctx->out_buf, (uint64_t)nf * 8, dst_bytes, mem_kind)) != SPH_OK) return rc;
        return sync_and_check(ctx);
    case SPH_FIELD_SORT_CELL_COUNT:
    case SPH_FIELD_SORT_CELL_START:             // row a3 as the last rebuild left it (k_hash_count's histogram, scan_cells' output)
        if (!ctx->have_config) return fail(ctx, SPH_ESTATE, "the sort-cell arrays need a completed rebuild (sph_step)");
        if ((rc = copy_out(ctx, dst, field == SPH_FIELD_SORT_CELL_COUNT ? ctx->ccount_f : ctx->cstart_f, plain_field_bytes(ctx, field), dst_bytes,
                           mem_kind)) != SPH_OK)
            return rc;
        return sync_and_check(ctx);
    case SPH_FIELD_WALL_POS:
    case SPH_FIELD_WALL_NORMAL:
        if (nw > 0) {
            LAUNCH(SPH_K_OTHER, k_extract_wall, cdiv(nw, 256), 256, nw, field == SPH_FIELD_WALL_POS ? ctx->wpos : ctx->wnrm, (float*)ctx->out_buf);
            if ((rc = copy_out(ctx, dst, ctx->out_buf, (uint64_t)nw * 12, dst_bytes, mem_kind)) != SPH_OK) return rc;
        }
        return sync_and_check(ctx);
    case SPH_FIELD_WALL_T:
    case SPH_FIELD_WALL_DT_DT:
        if (nw > 0) {
            if (field == SPH_FIELD_WALL_DT_DT && !ctx->have_config) return fail(ctx, SPH_ESTATE, "WALL_DT_DT needs a completed step");
            LAUNCH(SPH_K_OTHER, k_extract_wall_scalar, cdiv(nw, 256), 256, nw, field == SPH_FIELD_WALL_T ? 1 : 0, (float)ctx->prm.T_ref, ctx->wT,
                   ctx->wrate, ctx->perm_w, ctx->any_evolving ? 1 : 0, (float*)ctx->out_buf);
            if ((rc = copy_out(ctx, dst, ctx->out_buf, (uint64_t)nw * 4, dst_bytes, mem_kind)) != SPH_OK) return rc;
        }
        return sync_and_check(ctx);
    case SPH_FIELD_CONTACT_FACTOR: {
        if (!ctx->have_config) return fail(ctx, SPH_ESTATE, "CONTACT_FACTOR needs a neighbour configuration: call sph_step first");
        if (nw > 0) {
            const double h = ctx->prm.h;
            LAUNCH(SPH_K_OTHER, k_contact_factor, cdiv(nw, 128), 128, ctx->P, 1.0 / h, wendland_alpha(h, is_planar(ctx->prm)), ctx->sigma0,
                   particle_volume(ctx->prm), ctx->prm.rho0 * particle_volume(ctx->prm), ctx->prm.rho0, ctx->A, ctx->WA, ctx->cstart_f, ctx->cstart_w, ctx->perm_w,
                   (float*)ctx->out_buf);
            if ((rc = copy_out(ctx, dst, ctx->out_buf, (uint64_t)nw * 4, dst_bytes, mem_kind)) != SPH_OK) return rc;
        }
        return sync_and_check(ctx);
    }
    case SPH_FIELD_STATS: {
        if ((rc = sync_and_check(ctx)) != SPH_OK) return rc;
        Clock hc;
        CU(cudaMemcpy(&hc, ctx->clk, sizeof(hc), cudaMemcpyDeviceToHost));
        double s[SPH_STATS_COUNT];
        const uint64_t graph_launches = ctx->graph_fixed_launches + (uint64_t)hc.graph_rebuilds * ctx->graph_body_per_rebuild;
        s[SPH_STAT_T] = hc.t; s[SPH_STAT_DT] = hc.dt; s[SPH_STAT_DT_AD] = hc.dt_ad; s[SPH_STAT_ELAPSED] = hc.elapsed;
        s[SPH_STAT_VMAX] = hc.vmax; s[SPH_STAT_STEPS] = (double)hc.steps; s[SPH_STAT_REBUILDS] = (double)hc.rebuilds;
        s[SPH_STAT_SIGMA0] = ctx->sigma0; s[SPH_STAT_NCELL_X] = ctx->P.ng[0]; s[SPH_STAT_NCELL_Y] = ctx->P.ng[1];
        s[SPH_STAT_NCELL_Z] = ctx->P.ng[2]; s[SPH_STAT_ERROR_BITS] = 0.0; s[SPH_STAT_LAUNCHES] = (double)(ctx->launches + graph_launches);
        s[SPH_STAT_DEVICE_BYTES] = (double)ctx->device_bytes; s[SPH_STAT_MAX_NEIGH_FLUID] = ctx->P.KF; s[SPH_STAT_MAX_NEIGH_WALL] = ctx->P.KW;
        s[SPH_STAT_TILES] = (double)ctx->n_tiles; s[SPH_STAT_DIRECT_TILES] = 0.0; s[SPH_STAT_SPLIT_TILES] = 0.0; s[SPH_STAT_SPLIT4_TILES] = 0.0;
        if (ctx->have_config && ctx->n_tiles > 0) {
            std::vector<uint32_t> st((size_t)ctx->n_tiles);
            CU(cudaMemcpy2D(st.data(), 4, &ctx->hdr[0].S, sizeof(TileHdr) * SPH_SMAX, 4, (size_t)ctx->n_tiles, cudaMemcpyDeviceToHost));
            for (uint32_t x : st) { s[SPH_STAT_DIRECT_TILES] += x ? 0.0 : 1.0; s[SPH_STAT_SPLIT_TILES] += x > 1 ? 1.0 : 0.0; s[SPH_STAT_SPLIT4_TILES] += x == 4 ? 1.0 : 0.0; }
        }
        {
            double sum = 0.0;
            CU(cudaMemsetAsync(ctx->out_buf, 0, sizeof(double), ctx->stream));
            LAUNCH(SPH_K_OTHER, k_sum_theta, cdiv(nf, 256), 256, nf, ctx->Bc, (double*)ctx->out_buf);
            ctx->launches--;                         // a read-out, not part of the step count reported above
            CU(cudaMemcpyAsync(&sum, ctx->out_buf, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
            CU(cudaStreamSynchronize(ctx->stream));
            s[SPH_STAT_T_MEAN] = ctx->prm.T_ref + sum / (double)nf;
        }
        if (dst_bytes < sizeof(s)) return fail(ctx, SPH_EINVAL, "destination too small for STATS");
        CU(cudaMemcpy(dst, s, sizeof(s), mem_kind == SPH_MEM_DEVICE ? cudaMemcpyHostToDevice : cudaMemcpyHostToHost));
        return SPH_OK;
    }
    case SPH_FIELD_NEIGH_CSR_FLUID:
    case SPH_FIELD_NEIGH_CSR_WALL: {
        const int which = field == SPH_FIELD_NEIGH_CSR_WALL;
        if ((rc = sync_and_check(ctx)) != SPH_OK) return rc;
        std::vector<uint32_t> cnt_sorted(nf), org(nf);
        CU(cudaMemcpy(cnt_sorted.data(), ctx->ncnt, (size_t)nf * 4, cudaMemcpyDeviceToHost));
        CU(cudaMemcpy(org.data(), ctx->orig, (size_t)nf * 4, cudaMemcpyDeviceToHost));
        std::vector<uint64_t> offs((size_t)nf + 1, 0);
        for (int s = 0; s < nf; ++s) offs[org[s] + 1] = which ? (cnt_sorted[s] >> 16) : (cnt_sorted[s] & 0xffffu);
        for (int i = 0; i < nf; ++i) offs[i + 1] += offs[i];
        const uint64_t total = offs[nf];
        if (dst_bytes < total * 4) return fail(ctx, SPH_EINVAL, "destination too small for the CSR field: %llu < %llu", (unsigned long long)dst_bytes, (unsigned long long)(total * 4));
        uint64_t* d_offs = nullptr; int32_t* d_out = nullptr;
        CU(cudaMalloc(&d_offs, ((size_t)nf + 1) * 8));
        CU(cudaMalloc(&d_out, (size_t)(total ? total : 1) * 4));
        CU(cudaMemcpy(d_offs, offs.data(), ((size_t)nf + 1) * 8, cudaMemcpyHostToDevice));
        LAUNCH(SPH_K_OTHER, k_neigh_csr, ctx->n_tiles, SPH_TP, ctx->P, which, ctx->hdr, ctx->A, ctx->cstart_f, ctx->cstart_w,
               which ? ctx->list_w : ctx->list_f, which ? ctx->KW8 : ctx->KF8, ctx->ncnt, ctx->orig, which ? ctx->perm_w : ctx->orig, d_offs, d_out);
        cudaError_t e1 = cudaMemcpyAsync(dst, d_out, total * 4, mem_kind == SPH_MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream);
        cudaError_t e2 = cudaStreamSynchronize(ctx->stream);
        cudaFree(d_offs); cudaFree(d_out);
        if (e1 != cudaSuccess || e2 != cudaSuccess) return fail(ctx, SPH_ECUDA, "CSR read-back failed: %s", cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
        return SPH_OK;
    }
    default: return fail(ctx, SPH_EINVAL, "unknown field %u", field);
    }
}

int sph_get_torque(sph_ctx* ctx, int body, double torque[3], double* axial)
{
    if (!ctx) return SPH_EINVAL;
    if (!ctx->loaded) return fail(ctx, SPH_ESTATE, "sph_get_torque before sph_load_particles");
    if (body < 0 || body >= ctx->prm.n_bodies || !torque) return fail(ctx, SPH_EINVAL, "bad body %d or NULL torque", body);
    CU(cudaSetDevice(ctx->device));
    int rc = sync_and_check(ctx);
    if (rc != SPH_OK) return rc;
    double t[3];
    CU(cudaMemcpy(t, &ctx->clk->torque_done[body][0], sizeof(t), cudaMemcpyDeviceToHost));
    for (int d = 0; d < 3; ++d) torque[d] = t[d];
    if (axial) *axial = ctx->axis[body][0] * t[0] + ctx->axis[body][1] * t[1] + ctx->axis[body][2] * t[2];
    return SPH_OK;
}

int sph_profile(sph_ctx* ctx, int enable)
{
    if (!ctx) return SPH_EINVAL;
    CU(cudaSetDevice(ctx->device));
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->prof.clear();
    ctx->ev_used = 0;
    ctx->prof_on = enable != 0;
    if (enable && ctx->ev_pool.size() < 4096) {
        ctx->ev_pool.reserve(4096);
        while (ctx->ev_pool.size() < 4096) { cudaEvent_t e; CU(cudaEventCreate(&e)); ctx->ev_pool.push_back(e); }
    }
    return SPH_OK;
}

int sph_get_profile(sph_ctx* ctx, int kernel_class, double* ms_total, uint64_t* launches)
{
    if (!ctx || kernel_class < 0 || kernel_class >= SPH_K_COUNT) return SPH_EINVAL;
    CU(cudaSetDevice(ctx->device));
    CU(cudaStreamSynchronize(ctx->stream));
    double ms = 0.0; uint64_t n = 0;
    for (const ProfRec& r : ctx->prof) {
        if (r.cls != kernel_class) continue;
        float t = 0.f;
        CU(cudaEventElapsedTime(&t, r.e0, r.e1));
        ms += t; ++n;
    }
    if (ms_total) *ms_total = ms;
    if (launches) *launches = n;
    return SPH_OK;
}

}  // extern "C"

// =================================================================================================
// sph_cell_scan_static (include/sph.h): row a3's exclusive scan for callers that may not allocate.  The scan kernels'
// scratch -- one partial sum per SCAN_CHUNK cells -- lives in this file-scope device array: every GPU that loads the
// library holds SPH_SCAN_STATIC_SCRATCH_BYTES of it until the process exits.  In HOST code the name `g_scan_scratch` is a
// host-side stand-in, not a device address: the address the kernels get is resolved once per device with
// cudaGetSymbolAddress (that device current) and kept in g_scan_scratch_dev[].
// =================================================================================================
#define SPH_SCAN_STATIC_MAX_BLOCKS ((int)(SPH_SCAN_STATIC_MAX_CELLS / SCAN_CHUNK))
static_assert(SPH_SCAN_STATIC_MAX_CELLS % SCAN_CHUNK == 0, "whole scan blocks");
static_assert(((size_t)SPH_SCAN_STATIC_MAX_BLOCKS + 1) * sizeof(uint32_t) <= SPH_SCAN_STATIC_SCRATCH_BYTES, "scratch size stated in sph.h");
static __device__ __align__(256) uint32_t g_scan_scratch[SPH_SCAN_STATIC_SCRATCH_BYTES / sizeof(uint32_t)];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_scan_mutex;
uint32_t* g_scan_scratch_dev[kMaxDevices] = {};       // device address of g_scan_scratch on device d (nullptr: not resolved yet)

// once per device, with that device current; the calling thread's current device is restored
int scan_scratch_address(int device, uint32_t** out)
{
    std::lock_guard<std::mutex> lock(g_scan_mutex);
    if (!g_scan_scratch_dev[device]) {
        int prev = -1;
        cudaError_t e = cudaGetDevice(&prev);
        if (e == cudaSuccess) e = cudaSetDevice(device);
        void* ptr = nullptr;
        if (e == cudaSuccess) e = cudaGetSymbolAddress(&ptr, g_scan_scratch);
        if (prev >= 0 && prev != device) cudaSetDevice(prev);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            return fail(nullptr, SPH_ECUDA, "sph_cell_scan_static: cudaGetSymbolAddress on device %d failed: %s", device, cudaGetErrorString(e));
        }
        g_scan_scratch_dev[device] = static_cast<uint32_t*>(ptr);
    }
    *out = g_scan_scratch_dev[device];
    return SPH_OK;
}
}  // namespace

extern "C" int sph_cell_scan_static(int device, const uint32_t* counts_dev, uint32_t* starts_dev, uint32_t n_cells, uint32_t n_items,
                                    void* cuda_stream)
{
    if (!counts_dev || !starts_dev) return fail(nullptr, SPH_EINVAL, "sph_cell_scan_static: counts_dev / starts_dev is NULL");
    if (device < 0 || device >= kMaxDevices) return fail(nullptr, SPH_EINVAL, "sph_cell_scan_static: device %d out of range", device);
    if (n_cells == 0 || n_cells > SPH_SCAN_STATIC_MAX_CELLS)
        return fail(nullptr, SPH_EINVAL, "sph_cell_scan_static: n_cells = %u, the static scratch array serves 1 .. %u cells (SPH_SCAN_STATIC_MAX_CELLS)",
                    n_cells, (unsigned)SPH_SCAN_STATIC_MAX_CELLS);
    {
        const uintptr_t a = reinterpret_cast<uintptr_t>(counts_dev), b = reinterpret_cast<uintptr_t>(starts_dev);
        if (a < b + ((uintptr_t)n_cells + 1) * 4 && b < a + (uintptr_t)n_cells * 4)
            return fail(nullptr, SPH_EINVAL, "sph_cell_scan_static: counts_dev and starts_dev overlap");
    }
    uint32_t* scratch = nullptr;
    int rc = scan_scratch_address(device, &scratch);
    if (rc != SPH_OK) return rc;
    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e == cudaSuccess && prev != device) e = cudaSetDevice(device);
    if (e != cudaSuccess) return fail(nullptr, SPH_ECUDA, "sph_cell_scan_static: cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int n = (int)n_cells, nb = (n + SCAN_CHUNK - 1) / SCAN_CHUNK;          // nb <= SPH_SCAN_STATIC_MAX_BLOCKS
    // the library's scan kernels, unpredicated (pred = 0: the Clock pointer is not read); every scratch entry that is read
    // (0 .. nb - 1) is written by k_scan_local first, so the last call's contents do not matter
    k_scan_local<<<nb, SCAN_THREADS, 0, st>>>(counts_dev, starts_dev, scratch, n, nullptr, 0);
    k_scan_sums<<<1, SCAN_THREADS, 0, st>>>(scratch, nb, nullptr, 0);
    k_scan_add<<<nb, SCAN_THREADS, 0, st>>>(starts_dev, scratch, n, n_items, nullptr, 0);
    e = cudaPeekAtLastError();
    if (prev >= 0 && prev != device) cudaSetDevice(prev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(nullptr, SPH_ECUDA, "sph_cell_scan_static: kernel launch failed: %s", cudaGetErrorString(e));
    }
    return SPH_OK;
}

// =================================================================================================
// sph_measure_fma_peak (include/sph.h): measured fp32 FMA rate, for the roofline of the ALU-bound sweeps
// =================================================================================================
#define SPH_PEAK_CHAINS 8
__global__ void __launch_bounds__(256) k_fma_peak(float* __restrict__ out, int iters, float a, float b)
{
    float x[SPH_PEAK_CHAINS];
#pragma unroll
    for (int k = 0; k < SPH_PEAK_CHAINS; ++k) x[k] = 1.0e-3f * (float)threadIdx.x + (float)k;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int k = 0; k < SPH_PEAK_CHAINS; ++k) x[k] = fmaf(x[k], a, b);          // independent chains: latency hidden inside one warp
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < SPH_PEAK_CHAINS; ++k) s += x[k];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" int sph_measure_fma_peak(int device, double* tflops, void* cuda_stream)
{
    if (!tflops) return fail(nullptr, SPH_EINVAL, "sph_measure_fma_peak: tflops is NULL");
    *tflops = 0.0;
    cudaDeviceProp prop;
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) return fail(nullptr, SPH_ECUDA, "sph_measure_fma_peak: device %d: %s", device, cudaGetErrorString(e));
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int grid = prop.multiProcessorCount * 8, block = 256, iters = 4096;
    float* buf = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    e = cudaMalloc(&buf, (size_t)grid * block * sizeof(float));
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    float best = 0.f;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {            // rep 0 = warm-up
        cudaEventRecord(e0, st);
        k_fma_peak<<<grid, block, 0, st>>>(buf, iters, 0.999f, 1.0e-3f);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms > 0.f && (best == 0.f || ms < best)) best = ms;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (buf) cudaFree(buf);
    if (e != cudaSuccess || best <= 0.f) {
        cudaGetLastError();
        return fail(nullptr, SPH_ECUDA, "sph_measure_fma_peak: %s", cudaGetErrorString(e));
    }
    const double flops = 2.0 * SPH_PEAK_CHAINS * 8.0 * (double)iters * (double)grid * (double)block;
    *tflops = flops / ((double)best * 1.0e-3) / 1.0e12;
    return SPH_OK;
}
