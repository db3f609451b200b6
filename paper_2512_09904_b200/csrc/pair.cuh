// pair.cuh -- tile-staged neighbour lists and the fused neighbour-pair sweeps (steps a4b, a5, a8-a10,
// a12 of DESIGN.md section 1).
//
// Tiles.  A tile is SPH_TP consecutive particles of the cell-sorted fluid arrays, handled by one CTA of
// SPH_TP threads.  Its particles lie in the linear cells [c_first, c_last] (x fastest), so every neighbour
// candidate lies in one of nine CONTIGUOUS index ranges of the sorted arrays: for each (dy, dz) the cells
// [c_first - 1 + s, c_last + 1 + s], s = dy nx + dz nx ny (clamped to the grid; cells that wrap around a
// row end are harmless extras).  The same holds for the sorted wall arrays.  A sweep copies those ranges
// into shared memory once per CTA with 1-D TMA bulk copies (cp.async.bulk + mbarrier), so each stencil
// record leaves L2 once per tile instead of once per pair, and all gathers are LDS.128.
//
// Shared-memory layout.  Two halves of SPH_HALF_BYTES each with the same layout
//   [fluid records: tot_f + SPH_ND][wall records: tot_w + SPH_ND]
// half 0 holds the A records ({x, y, z, drho} / wall {x, y, z, body}), half 1 the B records
// ({vx, vy, vz, theta} / wall {nx, ny, nz, theta_w}), so the B record of a neighbour sits at a
// compile-time offset from its A record (one address computation per pair).
//
// Lists.  The neighbour list of a particle holds 16-bit indices into its tile's staged order
// ("local" index = lbase[range] + offset in range), eight per 16-byte word, laid out [tile][k/8][lane] so
// a warp reads 512 contiguous bytes per eight neighbours; the next word is in flight while the current
// one is processed (the list stream comes from HBM and would otherwise expose its latency).  Lists are
// padded to the warp's longest list (rounded up to 4) with the index of a dummy record placed far away,
// whose kernel weight is exactly 0: the pair loops carry no per-lane predicate.  Tiles whose ranges
// exceed the shared-memory budget (crowded or very sparse regions, any cell span) run in "direct" mode:
// their list entries index the particle's own 27-cell stencil instead and the records are gathered from
// global memory.
//
// Arithmetic: fp32; the pressure sum is re-associated as  sum_j V_j F_ij r_ij p*_ij =
// p_i G_i + sum_j V_j F_ij r_ij [(p*_ij - p_i) - p_i drho_j / rho0]  (+ the same for walls) with the purely
// geometric G_i = dx^3 sum F r summed once per rebuild in fp64, so that a large
// uniform pressure level does not cancel in fp32.
#pragma once
#include "common.cuh"

#ifndef SPH_TP
#define SPH_TP 256                 // particles per tile = threads per CTA
#endif
#ifndef SPH_STAGE_BYTES
#define SPH_STAGE_BYTES (108 * 1024)   // shared-memory budget of the staged records (2 CTAs per SM)
#endif
#ifndef SPH_MINB
#define SPH_MINB 2                 // resident CTAs per SM the sweeps are compiled for
#endif
#ifndef SPH_MINB_BUILD
#define SPH_MINB_BUILD 2           // resident CTAs per SM of k_build_tiles (its shared memory allows two)
#endif
#define SPH_HALF_BYTES (SPH_STAGE_BYTES / 2)
#define SPH_NR 9                   // ranges per row run and species (the 3 x 3 neighbouring cell rows)
#ifndef SPH_RUNS
#define SPH_RUNS 4                 // a staged tile may touch up to this many cell rows
#endif
#define SPH_NRMAX (SPH_NR * SPH_RUNS)
#define SPH_ND 1                   // dummy records behind each species' staged records
#define SPH_NWARP (SPH_TP / 32)
#define SPH_COST_CLASSES 4         // cost classes of the tile schedule (k_tile_order)
#ifndef SPH_TAIL_FACTOR
#define SPH_TAIL_FACTOR 16         // tiles per persistent CTA at the end of the schedule that are sorted by cost class
#endif

// A tile's particles form up to SPH_RUNS "row runs": maximal stretches lying in one cell row (same y, z).
// Run k occupies the cells [c_lo, c_hi] of its row; its candidates lie in the nine ranges
// [c_lo - 1, c_hi + 1] (clamped to the row) of the rows (y + dy, z + dz).  Ranges of different runs may
// overlap (the records are then staged twice); a particle only ever indexes the ranges of its own run.
// A tile whose ranges do not fit the shared-memory budget (sparse cell rows make a 256-particle tile long) is
// processed as S = 2 or 4 consecutive SUB-TILES of SPH_TP / S particles, one pass each, every pass with its own
// header and staging; in a pass all SPH_TP threads work, S threads per particle, each on every S-th list word.
// Header slot q of tile t is hdr[t * SPH_SMAX + q]; slot 0 carries S.
#ifndef SPH_SMAX
#define SPH_SMAX 4
#endif
struct TileHdr {
    uint32_t n_ranges;                 // SPH_NR * number of runs; meaningful for staged tiles
    uint32_t staged;                   // 1: <= SPH_RUNS runs and the ranges fit in shared memory
    uint32_t S;                        // slot 0: passes of this tile (1, 2, 4); 0 = direct mode (global gathers)
    uint32_t pad;
    uint32_t tot_f, tot_w;             // staged records per species (= lbase[n_ranges]); the dummy slot
    uint32_t gstart_f[SPH_NRMAX];      // first sorted fluid index of range q = 9 run + r
    uint32_t lbase_f[SPH_NRMAX + 1];   // local (staged) index of range q's first record
    uint32_t gstart_w[SPH_NRMAX];
    uint32_t lbase_w[SPH_NRMAX + 1];
};

// ---------------------------------------------------------------------------------------------
// PTX helpers: mbarrier + 1-D bulk copy global -> shared (TMA), approximate reciprocals
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ float rcp_fast(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float2 dup2(float x) { return make_float2(x, x); }
__device__ __forceinline__ float rsqrt_fast(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// dummy record: far enough that 1 - r/(2h) < 0 for any h, near enough that d2 stays finite in fp32
#define SPH_FAR 1.0e15f
// Reading R28 (two particles at the same place): e_ij = r_ij / (r_ij + eps) -> 0 and W'/r -> its finite limit.
// The squared distance that feeds a reciprocal square root starts from this tiny value instead of from zero (the first
// multiply of the chain becomes an FMA: no extra instruction): d2 = 0 gives 1/r = 1e15 and r = 1e-15, every term along e_ij
// vanishes with r_ij = 0 and nothing turns into NaN; for any real pair (d2 > 1e-22) the sum rounds to d2 itself.
#define SPH_D2_TINY 1.0e-30f

// ---------------------------------------------------------------------------------------------
// tile context in shared memory
// ---------------------------------------------------------------------------------------------
struct TileSmem {
    TileHdr hdr;
    uint64_t bar;
    float tq[SPH_NWARP][SPH_MAXB * 3];     // per-warp torque partials (sweep A)
    float tv[SPH_NWARP][SPH_MAXB * 3];     // same, viscous part on its own (sweep A of a rebuilding step under R26)
};

// dynamic shared memory of the staged kernels: the staged records (sweeps: A half, B half; build: A records + hit buffers)
extern __shared__ __align__(128) unsigned char sph_dyn_smem[];

// Index tables.  Staged tiles index the tile's nine ranges (TileHdr); direct tiles index the
// particle's OWN nine sub-ranges (its 27 cells), so a direct tile works whatever its cell span.
struct RangeTab { uint32_t gs[SPH_NR]; uint32_t lb[SPH_NR + 1]; };

// local -> global sorted index; L == total maps to the dummy slot
__device__ __forceinline__ uint32_t resolve_local(const uint32_t* lb, const uint32_t* gs, uint32_t L, uint32_t dummy)
{
    if (L >= lb[SPH_NR]) return dummy;
    uint32_t g = gs[0], b = 0;
#pragma unroll
    for (int q = 1; q < SPH_NR; ++q)
        if (L >= lb[q]) { g = gs[q]; b = lb[q]; }
    return g + (L - b);
}
__device__ __forceinline__ uint32_t resolve_local_n(const uint32_t* lb, const uint32_t* gs, int nr, uint32_t L)
{
    uint32_t g = gs[0], b = 0;
    for (int q = 1; q < nr; ++q)
        if (L >= lb[q]) { g = gs[q]; b = lb[q]; }
    return g + (L - b);
}

// A particle's position in the sort grid and the window of sort cells it can have neighbours in, per stencil row.
// Row r = (dy + 1) + 3 (dz + 1).  In contract-cell units the particle sits at (ry, rz) in [0, 1) inside its cell; a
// particle j of row (dy, dz) is at least dmin_y (dy = -1: ry, dy = +1: 1 - ry) and dmin_z away in y and z, so
// |x_i - x_j| <= sqrt(rc^2 - dmin_y^2 - dmin_z^2).  Margins: 1e-3 cell on dmin and 1e-2 sort cell on the window
// cover the rounding of the scaled fp32 coordinates (<= 2.5e-4 cell at 2047 cells); the window never leaves
// [fx - SPH_SX, fx + SPH_SX], which contains every neighbour because rc < ell.  The result is a superset of the
// fp32 cut-off ball (R1); the exact predicate is applied to every candidate.
struct Stencil {
    int cy, cz, fx;
    float ux4, ry, rz;
};
__device__ __forceinline__ Stencil make_stencil(const DevParams& P, float4 pi)
{
    unsigned int err = 0;
    Stencil st;
    st.cy = cell_coord(pi.y, P.xmin[1], P.inv_ell, P.ng[1], err);
    st.cz = cell_coord(pi.z, P.xmin[2], P.inv_ell, P.ng[2], err);
    st.ux4 = fine_coord(pi.x, P.xmin[0], P.inv_ell4);
    st.fx = fine_cell(st.ux4, P.nfx);
    st.ry = __fmul_rn(__fsub_rn(pi.y, P.xmin[1]), P.inv_ell) - (float)st.cy;
    st.rz = __fmul_rn(__fsub_rn(pi.z, P.xmin[2]), P.inv_ell) - (float)st.cz;
    return st;
}
// first sort cell of row r's window in the cstart arrays and its length in sort cells (0: nothing in reach)
__device__ __forceinline__ int stencil_row(const DevParams& P, const Stencil& st, int r, int& ncell)
{
    const int dy = r % 3 - 1, dz = r / 3 - 1;
    const int y = st.cy + dy, z = st.cz + dz;
    ncell = 0;
    if (y < 0 || y >= P.ng[1] || z < 0 || z >= P.ng[2]) return 0;
    const float my = dy < 0 ? st.ry : (dy > 0 ? 1.0f - st.ry : 0.0f), mz = dz < 0 ? st.rz : (dz > 0 ? 1.0f - st.rz : 0.0f);
    const float ay = dy ? fmaxf(my - 1.0e-3f, 0.0f) : 0.0f, az = dz ? fmaxf(mz - 1.0e-3f, 0.0f) : 0.0f;
    const float w2 = P.rcu2 - ay * ay - az * az;
    if (!(w2 > 0.0f)) return 0;
    const float wk = sqrtf(w2) * (float)SPH_SX + 1.0e-2f;
    const int f0 = max(max((int)floorf(st.ux4 - wk), st.fx - SPH_SX), 0);
    const int f1 = min(min((int)floorf(st.ux4 + wk), st.fx + SPH_SX), P.nfx - 1);
    ncell = max(f1 - f0 + 1, 0);                  // a particle far outside the grid (clamped cell) reaches nothing
    return P.nfx * (y + P.ng[1] * z) + min(f0, P.nfx - 1);
}

// the particle's own stencil as nine sub-ranges of a sorted array (rows out of reach are empty)
__device__ __forceinline__ void own_table(const DevParams& P, float4 pi, const uint32_t* __restrict__ cstart, bool active, RangeTab& t)
{
    const Stencil st = make_stencil(P, pi);
    uint32_t acc = 0;
#pragma unroll
    for (int r = 0; r < SPH_NR; ++r) {
        int nc;
        const int c0 = stencil_row(P, st, r, nc);
        uint32_t s = 0, n = 0;
        if (active && nc > 0) {
            s = cstart[c0];
            n = cstart[c0 + nc] - s;
        }
        t.gs[r] = s; t.lb[r] = acc; acc += n;
    }
    t.lb[SPH_NR] = acc;
}

// Record access.  STAGED: shared memory, tile-local index, B record at a constant offset from the A
// record.  Direct: global memory, own-stencil index resolved through the thread's range table.
template <bool STAGED>
struct Recs {
    const float4* smA;       // staged A records of this species (half 0)
    const float4* gA;        // global sorted A array
    const float4* gB;        // global sorted B array
    const RangeTab* tab;     // direct mode: this thread's own table
    uint32_t dummy;          // global index of the dummy record
    __device__ __forceinline__ float4 A(uint32_t L) const
    {
        if (STAGED) SPH_DBG_CHECK(reinterpret_cast<const unsigned char*>(smA + L + 1) <= sph_dyn_smem + SPH_HALF_BYTES, 0);
        if (STAGED) return smA[L];
        return __ldg(gA + resolve_local(tab->lb, tab->gs, L, dummy));
    }
    __device__ __forceinline__ void AB(uint32_t L, float4& a, float4& b) const
    {
        if (STAGED) {
            SPH_DBG_CHECK(reinterpret_cast<const unsigned char*>(smA + L + 1) <= sph_dyn_smem + SPH_HALF_BYTES, 1);
            const float4* p = smA + L;
            a = *p;
            b = *reinterpret_cast<const float4*>(reinterpret_cast<const unsigned char*>(p) + SPH_HALF_BYTES);
        } else {
            const uint32_t g = resolve_local(tab->lb, tab->gs, L, dummy);
            a = __ldg(gA + g);
            b = __ldg(gB + g);
        }
    }
};

// Issue the bulk copy of range q of one species (one thread per range).
__device__ __forceinline__ void stage_range(const uint32_t* gstart, const uint32_t* lbase, int q, const float4* src, float4* dst, uint64_t* bar)
{
    const uint32_t n = lbase[q + 1] - lbase[q];
    if (n) bulk_g2s(dst + lbase[q], src + gstart[q], n * 16u, bar);
}

// ---------------------------------------------------------------------------------------------
// tile header: the nine fluid and nine wall ranges of a tile (threads 0..17 of the CTA)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int linear_cell(const DevParams& P, float4 p)       // sort-cell id (x sub-cell fastest)
{
    unsigned int err = 0;
    const int fx = fine_cell(fine_coord(p.x, P.xmin[0], P.inv_ell4), P.nfx);
    const int cy = cell_coord(p.y, P.xmin[1], P.inv_ell, P.ng[1], err);
    const int cz = cell_coord(p.z, P.xmin[2], P.inv_ell, P.ng[2], err);
    return fx + P.nfx * (cy + P.ng[1] * cz);
}

// Builds the header of `tile` in shared memory.  Every thread of the CTA passes the linear cell of its
// particle (c) and whether it holds one; returns the thread's run index.
__device__ int make_tile_header(const DevParams& P, int tile, int c, bool valid_all, int lo, int hi, const uint32_t* __restrict__ cstart_f,
                                const uint32_t* __restrict__ cstart_w, TileHdr* h /* shared */)
{
    const bool valid = valid_all && (int)threadIdx.x >= lo && (int)threadIdx.x < hi;      // threads [lo, hi): this (sub-)tile
    __shared__ int s_last_cell[SPH_NWARP];
    __shared__ uint32_t s_warp_runs[SPH_NWARP];
    __shared__ int s_run_lo[SPH_RUNS], s_run_hi[SPH_RUNS];
    __shared__ uint32_t s_cnt[2][SPH_NRMAX];
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5, nx = P.nfx;
    // run starts: first particle of the tile, or a particle whose cell row differs from its predecessor's
    int prev_c = __shfl_up_sync(0xffffffffu, c, 1);
    if (lane == 31) s_last_cell[wid] = c;
    __syncthreads();
    if (lane == 0 && wid > 0) prev_c = s_last_cell[wid - 1];
    const bool start = valid && (t == lo || prev_c / nx != c / nx);
    const uint32_t bal = __ballot_sync(0xffffffffu, start);
    if (lane == 0) s_warp_runs[wid] = __popc(bal);
    __syncthreads();
    int before = 0, n_runs = 0;
#pragma unroll
    for (int w = 0; w < SPH_NWARP; ++w) { const int k = (int)s_warp_runs[w]; n_runs += k; if (w < wid) before += k; }
    const int run = before + __popc(bal & (0xffffffffu >> (31 - lane))) - 1;       // starts at or before this lane
    if (start) {
        if (run < SPH_RUNS) s_run_lo[run] = c;
        if (run >= 1 && run - 1 < SPH_RUNS) s_run_hi[run - 1] = prev_c;
    }
    const bool last_valid = valid && (t == hi - 1 || tile * SPH_TP + t == P.n_f - 1);
    if (last_valid && run < SPH_RUNS) s_run_hi[run] = c;
    __syncthreads();
    const int nr = n_runs <= SPH_RUNS ? SPH_NR * n_runs : 0;
    if (t < 2 * nr) {
        const int sp = t / nr, q = t % nr, k = q / SPH_NR, r = q % SPH_NR;
        const int clo = s_run_lo[k], chi = s_run_hi[k];
        const int row = clo / nx, cy = row % P.ng[1], cz = row / P.ng[1];
        const int y = cy + r % 3 - 1, z = cz + r / 3 - 1;
        uint32_t g = 0, n = 0;
        if (y >= 0 && y < P.ng[1] && z >= 0 && z < P.ng[2] && (sp == 0 || P.n_w > 0)) {
            const int x0 = max(clo - row * nx - SPH_SX, 0), x1 = min(chi - row * nx + SPH_SX, nx - 1);
            const int base = nx * (y + P.ng[1] * z);
            const uint32_t* cs = sp ? cstart_w : cstart_f;
            g = cs[base + x0];
            n = cs[base + x1 + 1] - g;
        }
        (sp ? h->gstart_w : h->gstart_f)[q] = g;
        s_cnt[sp][q] = n;
    }
    __syncthreads();
    if (t < 2) {
        uint32_t* lb = t ? h->lbase_w : h->lbase_f;
        uint32_t acc = 0;
        for (int q = 0; q < nr; ++q) { lb[q] = acc; acc += s_cnt[t][q]; }
        lb[nr] = acc;
        if (t) h->tot_w = acc; else h->tot_f = acc;
    }
    __syncthreads();
    if (t == 0) {
        const unsigned long long need = ((unsigned long long)h->tot_f + SPH_ND + (unsigned long long)h->tot_w + SPH_ND) * 16ull;
        h->n_ranges = (uint32_t)nr;
        h->S = 1u; h->pad = 0u;
        h->staged = (nr > 0 && need <= (unsigned long long)SPH_HALF_BYTES && h->tot_f < 65535u - SPH_ND && h->tot_w < 65535u - SPH_ND) ? 1u : 0u;
    }
    __syncthreads();
    return run;
}

// ---------------------------------------------------------------------------------------------
// list words: eight 16-bit entries per uint4
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t word_entry(const uint4& w, int q /* 0..7 */)
{
    const uint32_t half = (q & 4) ? ((q & 2) ? w.w : w.z) : ((q & 2) ? w.y : w.x);
    return (q & 1) ? (half >> 16) : (half & 0xffffu);
}
__device__ __forceinline__ uint32_t list_entry(const uint4* col, int k) { return word_entry(col[(size_t)(k >> 3) * SPH_TP], k & 7); }

__device__ __forceinline__ void unpack4(uint32_t lo, uint32_t hi, uint32_t L[4])
{
    L[0] = lo & 0xffffu; L[1] = lo >> 16; L[2] = hi & 0xffffu; L[3] = hi >> 16;
}

// ---------------------------------------------------------------------------------------------
// k_build_tiles: tile header, neighbour lists (R1 predicate) and -- for every list word as it is written, in
// fp64 -- the kernel sum of the density re-initialisation (Eq. 14-15, R12) and the
// geometric gradient sum G_i = dx^3 sum F r used by sweep A.
// ---------------------------------------------------------------------------------------------
// fp64 Wendland C2 value and F = W'/r at squared distance d2 (0 outside the support), WITHOUT the constants
// CW, CF (applied once to the sums).  sqrt(d2) from the fp32 reciprocal square root refined by one Newton step
// in fp64 (relative error ~1e-13).  W / CW = s^4 (1 + 2q) = s^4 (5 - 4s), s = 1 - q/2.
__device__ __forceinline__ void WF_f64(double d2, double half_inv_h, double& W, double& F)
{
    const double y0 = (double)rsqrt_fast((float)d2 + SPH_D2_TINY);      // R28: d2 = 0 -> r = 0, W / CW = 1, F / CF = 1
    const double r0 = d2 * y0;                                          // sqrt(d2) to fp32 accuracy
    const double r = r0 * fma(-0.5, r0 * y0, 1.5);                      // = d2 y0 (1.5 - 0.5 d2 y0^2)
    const double s = fmax(fma(-r, half_inv_h, 1.0), 0.0);
    const double s2 = s * s;
    W = (s2 * s2) * (5.0 - 4.0 * s);
    F = s2 * s;
}

struct GeomSums { double sig, gx, gy, gz; };       // sum W / CW;  sum F r / CF

// One lane's list under construction.  Hits go into a ring of RC 16-bit entries in shared memory (one predicated
// store per candidate); complete 8-entry words are drained to the lane's global list column, and the fp64 sums of
// their entries are taken on the way (the records are still staged).  All control flow around it is warp-uniform.
#define SPH_RING_F 64              // ring sizes (entries, powers of two, multiples of 8) and strides in 4-byte words
#define SPH_RING_W 32              // (odd strides: the 32 lanes' equal ring positions fall on 32 banks)
#define SPH_RING_F_STRIDE 33
#define SPH_RING_W_STRIDE 17
#define SPH_RING_BYTES (SPH_TP * 4 * (SPH_RING_F_STRIDE + SPH_RING_W_STRIDE))
#define SPH_BUILD_SMEM (SPH_HALF_BYTES + SPH_RING_BYTES)      // k_build_tiles: staged A records + the hit buffers behind them
#define SPH_CAND_UNROLL 4          // candidates tested per round of the scan loop (8 measured 1 % slower: more rejected slots at the row ends)
struct ListRing {
    uint16_t* buf;      // this thread's buffer (RC entries); entry n lives at buf[n - fl]
    uint32_t wn;        // entries in the buffer = n - fl (an index, not a pointer: 32-bit shared-memory addressing in the scan loop)
    uint4* col;         // this lane's global list column: word k8 at col[k8 * SPH_TP]
    int rc;             // buffer size in entries
    int cap8;           // capacity in words
    int fl;             // entries drained (multiple of 8)
    __device__ __forceinline__ void push(uint32_t L, bool hit)
    {
        SPH_DBG_CHECK(!hit || (int)wn < rc, 2);
        if (hit) buf[wn] = (uint16_t)L;
        wn += hit ? 1u : 0u;
    }
    __device__ __forceinline__ int pending() const { return (int)wn; }
    __device__ __forceinline__ int n() const { return fl + pending(); }
    __device__ __forceinline__ bool nearly_full() const { return pending() > rc - SPH_CAND_UNROLL; }      // room for one more round of candidates
};

// Drain: every lane writes its complete words (final: also the partial one, padded with `dummy`) and adds their
// entries to the fp64 sums.  Warp-uniform loop; lanes without a word to write idle in it.
template <bool STAGED>
__device__ __forceinline__ void drain_ring(ListRing& w, bool final, uint32_t dummy, const Recs<STAGED>& R, float4 pi, double half_inv_h, GeomSums& g)
{
    const double xi = pi.x, yi = pi.y, zi = pi.z;
    int done = 0;                                   // entries of the buffer written out by this call
    const int pend = w.pending();
    for (;;) {
        const bool have = (pend - done >= 8) || (final && pend > done);
        if (!__any_sync(0xffffffffu, have)) break;
        if (have) {
            const uint32_t* src = reinterpret_cast<const uint32_t*>(w.buf + done);
            uint32_t e[8];
#pragma unroll
            for (int k = 0; k < 4; ++k) { const uint32_t v = src[k]; e[2 * k] = v & 0xffffu; e[2 * k + 1] = v >> 16; }
#pragma unroll
            for (int k = 0; k < 8; ++k) e[k] = (done + k < pend) ? e[k] : dummy;
            const int k8 = (w.fl + done) >> 3;
            if (k8 < w.cap8)
                __stcs(w.col + (size_t)k8 * SPH_TP, make_uint4(e[0] | (e[1] << 16), e[2] | (e[3] << 16), e[4] | (e[5] << 16), e[6] | (e[7] << 16)));
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const float4 pj = R.A(e[k]);
                const double dx = xi - (double)pj.x, dy = yi - (double)pj.y, dz = zi - (double)pj.z;
                double W, F;
                WF_f64(dx * dx + dy * dy + dz * dz, half_inv_h, W, F);
                g.sig += W;
                g.gx += F * dx; g.gy += F * dy; g.gz += F * dz;
            }
            done += 8;
        }
    }
    // keep the incomplete word: move it to the front of the buffer
    const int left = max(pend - done, 0);
    if (left > 0 && done > 0) {
        const uint32_t* src = reinterpret_cast<const uint32_t*>(w.buf + done);
        uint32_t* dst = reinterpret_cast<uint32_t*>(w.buf);
#pragma unroll
        for (int k = 0; k < 4; ++k) dst[k] = src[k];           // done is a multiple of 8: both 4-byte aligned, no overlap
    }
    w.fl += final ? pend : done;
    w.wn = final ? 0u : (uint32_t)left;
}

// dist2 (common.cuh: the canonical fma chain of R1) of N candidates, two at a time in 64-bit registers (FMUL2 / FFMA2
// round each half like the scalar instructions: the results are bit-identical)
template <int N>
__device__ __forceinline__ void dist2xN(float4 pi, const float4 (&pj)[N], float (&d2)[N])
{
    static_assert(N % 2 == 0, "pairs of candidates");
#pragma unroll
    for (int u = 0; u < N; u += 2) {
        const float2 dx = make_float2(pi.x - pj[u].x, pi.x - pj[u + 1].x), dy = make_float2(pi.y - pj[u].y, pi.y - pj[u + 1].y),
                     dz = make_float2(pi.z - pj[u].z, pi.z - pj[u + 1].z);
        const float2 d = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
        d2[u] = d.x; d2[u + 1] = d.y;
    }
}

// candidate tests of one particle.  STAGED: candidates are read from the staged ranges of the particle's
// row run, list entries index the tile's staged order.  Direct: candidates come from global memory and
// list entries index the particle's own nine sub-ranges (own_table order).  Loop bounds are made warp-uniform
// (maximum over the lanes) so that the rings can be drained by the whole warp whenever one is nearly full.
template <bool STAGED>
__device__ __forceinline__ void build_one(const DevParams& P, const TileHdr& h, int run, const float4* sA, const float4* sWA,
                                          const float4* __restrict__ A, const float4* __restrict__ WA, int i, bool valid, float4 pi,
                                          const uint32_t* __restrict__ cstart_f, const uint32_t* __restrict__ cstart_w, ListRing& wf, ListRing& ww,
                                          uint32_t dummy_f, uint32_t dummy_w, const Recs<STAGED>& RF, const Recs<STAGED>& RW, double half_inv_h,
                                          GeomSums& g)
{
    const Stencil stc = make_stencil(P, pi);
    uint32_t dbase_f = 0, dbase_w = 0;            // direct mode: running local base of the own sub-ranges
    const uint32_t dummy_f_g = (uint32_t)P.dummy_f, dummy_w_g = (uint32_t)P.dummy_w;
    // the window of row r in the sorted arrays: [sf, ef) fluid, [sw, ew) wall.  The four cell_start words of row r + 1 are
    // fetched before the candidate loops of row r, so that their L2 round trips run behind those loops instead of in front of
    // every row (round 2: 10 % of the kernel's warp time was spent waiting for them, profiles/r02e.md)
    struct RowWin { uint32_t sf, ef, sw, ew; bool on; };
    auto fetch_row = [&](int r) {
        RowWin w = {0u, 0u, 0u, 0u, false};
        int nc;
        const int c0 = stencil_row(P, stc, r, nc);
        w.on = valid && nc > 0;
        if (w.on) {
            w.sf = __ldg(cstart_f + c0); w.ef = __ldg(cstart_f + c0 + nc);
            if (P.n_w > 0) { w.sw = __ldg(cstart_w + c0); w.ew = __ldg(cstart_w + c0 + nc); }
        }
        return w;
    };
    RowWin win = fetch_row(0);
#pragma unroll 1
    for (int r = 0; r < SPH_NR; ++r) {
        const RowWin cw = win;
        if (r + 1 < SPH_NR) win = fetch_row(r + 1);
        const bool on = cw.on;
        const int q = STAGED ? run * SPH_NR + r : 0;
        {
            const uint32_t s = cw.sf, cnt = cw.ef - cw.sf;
            const uint32_t L0 = STAGED ? (on ? h.lbase_f[q] + (s - h.gstart_f[q]) : 0u) : dbase_f;
            const uint32_t self = (uint32_t)i - s;                       // offset of i in this window, if it is there
            const uint32_t cmax = __reduce_max_sync(0xffffffffu, cnt);
#pragma unroll 1
            for (uint32_t o0 = 0; o0 < cmax; o0 += SPH_CAND_UNROLL) {
                if (__any_sync(0xffffffffu, wf.nearly_full())) drain_ring<STAGED>(wf, false, dummy_f, RF, pi, half_inv_h, g);
                // lanes past their own window read on (inside the staging buffer; direct mode: clamped) and reject by `o < cnt`
                float4 pj[SPH_CAND_UNROLL];
#pragma unroll
                if (STAGED) SPH_DBG_CHECK(reinterpret_cast<const unsigned char*>(sA + L0 + o0 + SPH_CAND_UNROLL) <= sph_dyn_smem + SPH_BUILD_SMEM, 6);
                for (uint32_t u = 0; u < SPH_CAND_UNROLL; ++u) pj[u] = STAGED ? sA[L0 + o0 + u] : __ldg(A + min(s + o0 + u, dummy_f_g));
                float d2[SPH_CAND_UNROLL];
                dist2xN(pi, pj, d2);
#pragma unroll
                for (uint32_t u = 0; u < SPH_CAND_UNROLL; ++u) {
                    const uint32_t o = o0 + u;
                    wf.push(L0 + o, d2[u] < P.rc2 && o != self && o < cnt);
                }
            }
            dbase_f += cnt;
        }
        if (P.n_w > 0) {
            const uint32_t s = cw.sw, cnt = cw.ew - cw.sw;
            const uint32_t L0 = STAGED ? (on ? h.lbase_w[q] + (s - h.gstart_w[q]) : 0u) : dbase_w;
            const uint32_t cmax = __reduce_max_sync(0xffffffffu, cnt);
#pragma unroll 1
            for (uint32_t o0 = 0; o0 < cmax; o0 += SPH_CAND_UNROLL) {
                if (__any_sync(0xffffffffu, ww.nearly_full())) drain_ring<STAGED>(ww, false, dummy_w, RW, pi, half_inv_h, g);
                float4 pj[SPH_CAND_UNROLL];
#pragma unroll
                if (STAGED) SPH_DBG_CHECK(reinterpret_cast<const unsigned char*>(sWA + L0 + o0 + SPH_CAND_UNROLL) <= sph_dyn_smem + SPH_BUILD_SMEM, 6);
                for (uint32_t u = 0; u < SPH_CAND_UNROLL; ++u) pj[u] = STAGED ? sWA[L0 + o0 + u] : __ldg(WA + min(s + o0 + u, dummy_w_g));
                float d2[SPH_CAND_UNROLL];
                dist2xN(pi, pj, d2);
#pragma unroll
                for (uint32_t u = 0; u < SPH_CAND_UNROLL; ++u) {
                    const uint32_t o = o0 + u;
                    ww.push(L0 + o, d2[u] < P.rc2 && o < cnt);
                }
            }
            dbase_w += cnt;
        }
    }
    if (dbase_f >= 65535u || dbase_w >= 65535u) wf.fl = 0x3fffffff;     // own stencil not addressable with 16 bits: ERR_NEIGH
}

// after the last drain: dummy words up to the warp's longest list (m8 entries, a multiple of 8)
__device__ __forceinline__ void pad_list(const ListRing& w, int m8, uint32_t dummy)
{
    const uint32_t d2 = dummy | (dummy << 16);
    for (int k8 = (min(w.n(), w.cap8 * 8) + 7) >> 3; k8 < (m8 >> 3) && k8 < w.cap8; ++k8) __stcs(w.col + (size_t)k8 * SPH_TP, make_uint4(d2, d2, d2, d2));
}

// ---------------------------------------------------------------------------------------------
// bank_order_one: bank-aware order of a finished neighbour list (once per rebuild, last phase of k_build_tiles).
// In the sweeps the 8 lanes of a quarter warp gather one 16-byte record each per LDS.128; the request takes one
// shared-memory wavefront when the 8 records lie in 8 different 16-byte bank groups (record index mod 8) and up to 8
// otherwise -- 2.4 on average for lists in candidate order (profiles/r01f.md), which made the sweeps LDS-bound.
// The order of a list is free (R20), so every list is re-ordered such that entry k of the particle in lane slot s has
// index = (s + k) mod 8 wherever the list still holds such an entry: the lanes of a quarter warp then read 8 different
// bank groups at every step (1.27 wavefronts per ideal one measured, profiles/r02a.md).
// One thread per list.  Class of an entry: c = (index - s) mod 8, so that slot q of EVERY 8-entry word wants class q.
// Pass A scatters entry number r of class c to position 8 r + c of a per-thread shared-memory array (the wanted order,
// with holes where a class is short); pass B reads it back word by word, fills the holes below n with the entries
// that landed at positions >= n, and writes the words (coalesced 16 bytes per lane); dummy padding stays behind the
// real entries.  The eight running class counts live in two registers (a byte each; one PRMT reads a count, one
// 8-byte table look-up adds to it).  Lists with more than SPH_BO_RANKS entries in one class and direct tiles (global
// gathers) are left in candidate order.  The pass is left out when the advection step that just ended had fewer than
// BuildArgs.skip_short acoustic steps (Eq. 25 with a fast flow asks for a rebuild at almost every step: the lists live for
// one step and the pass would cost more than it wins).
// ---------------------------------------------------------------------------------------------
#define SPH_BO_RANKS 24                                      // positions per class in the scatter array
#define SPH_BO_STRIDE (SPH_BO_RANKS * 4 + 1)                 // per-thread stride in 4-byte words (odd: lanes spread over the banks)
#define SPH_BO_SMEM (SPH_TP * SPH_BO_STRIDE * 4)
#define SPH_BO_BATCH 6                                       // list words fetched at once in pass A

__device__ __forceinline__ void bank_order_one(uint4* __restrict__ col, int n, uint16_t* pos, const uint2* onehot, uint32_t shift)
{
    const int nfull = n >> 3, rest = n & 7;
    uint32_t lo = 0u, hi = 0u, over = 0u, dummy = 0u;
    auto put = [&](uint32_t e) {
        const uint32_t c = (e + shift) & 7u;
        const uint32_t r = __byte_perm(lo, hi, c) & 0xffu;                 // entries of class c so far
        const uint2 one = onehot[c];
        lo += one.x; hi += one.y;
        over |= r >= SPH_BO_RANKS ? 1u : 0u;                               // (the clamped store below is then discarded with the list)
        SPH_DBG_CHECK(8u * min(r, (uint32_t)SPH_BO_RANKS - 1u) + c < 8u * SPH_BO_RANKS, 3);
        pos[8u * min(r, (uint32_t)SPH_BO_RANKS - 1u) + c] = (uint16_t)e;
    };
    // pass A.  The list words come from L2 / HBM (~1 us away) and a word feeds only ~130 instructions: they are fetched in
    // batches of SPH_BO_BATCH independent loads so that their latency is paid once per batch, not once per word
    const int nwords = nfull + (rest ? 1 : 0);
    for (int b0 = 0; b0 < nwords; b0 += SPH_BO_BATCH) {
        uint4 w[SPH_BO_BATCH];
#pragma unroll
        for (int u = 0; u < SPH_BO_BATCH; ++u)
            if (b0 + u < nwords) w[u] = col[(size_t)(b0 + u) * SPH_TP];
#pragma unroll
        for (int u = 0; u < SPH_BO_BATCH; ++u) {
            if (b0 + u < nfull) {
                put(w[u].x & 0xffffu); put(w[u].x >> 16); put(w[u].y & 0xffffu); put(w[u].y >> 16);
                put(w[u].z & 0xffffu); put(w[u].z >> 16); put(w[u].w & 0xffffu); put(w[u].w >> 16);
            } else if (b0 + u == nfull && rest) {
#pragma unroll
                for (int q = 0; q < 8; ++q) { const uint32_t e = word_entry(w[u], q); if (q < rest) put(e); else dummy = e; }
            }
        }
    }
    if (over) return;                                                      // a crowded class: the list keeps its candidate order
    uint32_t cnt[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) cnt[q] = __byte_perm(lo, hi, q) & 0xffu;
    // fillers: the entries that landed at positions >= n, as many as there are holes below n.  They are first compacted in
    // place to pos[n], pos[n + 1], ... (the write index never passes the read index), so that pass B is branch-free: a slot
    // takes its own position or the next filler (a search loop per hole diverged across the lanes: 13 % of the kernel's time)
    uint32_t mx = cnt[0];
#pragma unroll
    for (int q = 1; q < 8; ++q) mx = max(mx, cnt[q]);
    {
        uint32_t nq = (uint32_t)n;
        for (uint32_t t = (uint32_t)n; t < 8u * mx; ++t) {
            const bool f = (t >> 3) < (__byte_perm(lo, hi, t & 7u) & 0xffu);
            SPH_DBG_CHECK(t < 8u * SPH_BO_RANKS && nq <= t, 4);
            const uint16_t v = pos[t];
            if (f) pos[nq] = v;
            nq += f ? 1u : 0u;
        }
    }
    uint32_t fi = (uint32_t)n;                                              // next filler
    for (int k8 = 0; k8 < nfull; ++k8) {                                    // pass B
        uint32_t e[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const bool f = (uint32_t)k8 < cnt[q];
            SPH_DBG_CHECK((f ? (uint32_t)(8 * k8 + q) : fi) < 8u * SPH_BO_RANKS, 5);
            e[q] = (uint32_t)pos[f ? (uint32_t)(8 * k8 + q) : fi];
            fi += f ? 0u : 1u;
        }
        col[(size_t)k8 * SPH_TP] = make_uint4(e[0] | (e[1] << 16), e[2] | (e[3] << 16), e[4] | (e[5] << 16), e[6] | (e[7] << 16));
    }
    if (rest) {
        uint32_t e[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const bool f = (uint32_t)nfull < cnt[q];
            e[q] = q >= rest ? dummy : (uint32_t)pos[f ? (uint32_t)(8 * nfull + q) : fi];
            fi += (q < rest && !f) ? 1u : 0u;
        }
        col[(size_t)nfull * SPH_TP] = make_uint4(e[0] | (e[1] << 16), e[2] | (e[3] << 16), e[4] | (e[5] << 16), e[6] | (e[7] << 16));
    }
}

struct BuildArgs {
    double inv_h, CW, CF, sigma0, rho0, V0;
    double fs_sigma;                 // R27: a particle with sigma_i < fs_sigma (= theta sigma0) is a surface particle
    unsigned char* fs_region;        // R27: 2 = surface particle, 1 = fluid neighbour of one (k_fs_mark), 0 = neither
    float4* A;                       // {x, y, z frozen, drho}; .w updated by the re-initialisation
    const float4* WA;
    const uint32_t *cstart_f, *cstart_w;
    uint4 *list_f, *list_w;
    uint32_t* ncnt;
    float4* G;                       // {G_x, G_y, G_z, 0}
    TileHdr* hdr;
    uint32_t* tile_bin;              // cost class of every tile (k_tile_order)
    const uint32_t* order;           // schedule of the PREVIOUS rebuild: the expensive tiles of the tail region start first here too
    Clock* clk;
    int KF8, KW8;                    // list capacities in 8-entry words
    int pred;
    int order_lists;                 // 1: re-order this tile's lists for the sweeps' bank groups at the end of the kernel (bank_order_one)
    int skip_short;                  // ... unless the advection step that just ended had fewer acoustic steps than this
};


struct BuildSmem {
    TileHdr hdr[SPH_SMAX];
    uint64_t bar;
};

__global__ void __launch_bounds__(SPH_TP, SPH_MINB_BUILD) k_build_tiles(DevParams P, BuildArgs a)
{
    if (a.pred && !a.clk->rebuild) return;
    __shared__ BuildSmem ts;
    const int tile = (int)__ldg(a.order + blockIdx.x), tid = threadIdx.x;       // any permutation of the tiles will do
    const int i = tile * SPH_TP + tid;
    const bool valid = i < P.n_f;
    const float4 pi = a.A[valid ? i : P.n_f - 1];
    const int cell = linear_cell(P, pi);
    // whole tile first; when its ranges exceed the budget, 2 or 4 sub-tiles; else direct mode (S = 0)
    int S = 1;
    int run = make_tile_header(P, tile, cell, valid, 0, SPH_TP, a.cstart_f, a.cstart_w, &ts.hdr[0]);
    if (!ts.hdr[0].staged) {
        for (S = 2; S <= SPH_SMAX; S *= 2) {
            const int np = SPH_TP / S;
            bool all = true;
            for (int q = 0; q < S; ++q) {
                const int r = make_tile_header(P, tile, cell, valid, q * np, (q + 1) * np, a.cstart_f, a.cstart_w, &ts.hdr[q]);
                if (tid / np == q) run = r;
                // a sub-tile beyond the last particle has no runs: nothing to stage, nothing to do
                all = all && (ts.hdr[q].staged || tile * SPH_TP + q * np >= P.n_f);
            }
            if (all) break;
        }
        if (S > SPH_SMAX) {
            S = 0;
            run = make_tile_header(P, tile, cell, valid, 0, SPH_TP, a.cstart_f, a.cstart_w, &ts.hdr[0]);
        }
        __syncthreads();
        if (tid == 0) ts.hdr[0].S = (uint32_t)S;
        __syncthreads();
    }
    const int n_slots = S > 1 ? S : 1;
    for (int k = tid; k < n_slots * (int)(sizeof(TileHdr) / 4); k += SPH_TP)
        reinterpret_cast<uint32_t*>(a.hdr + (size_t)tile * SPH_SMAX)[k] = reinterpret_cast<const uint32_t*>(&ts.hdr[0])[k];
    const bool staged = S >= 1;
    const int np = SPH_TP / n_slots;                 // particles per pass
    const int myq = tid / np;
    if (staged && tid == 0) mbar_init(&ts.bar, 1);

    static_assert(SPH_BUILD_SMEM * SPH_MINB_BUILD <= 226 * 1024, "SPH_MINB_BUILD build CTAs per SM");
    uint32_t* ring_base = reinterpret_cast<uint32_t*>(sph_dyn_smem + SPH_HALF_BYTES);
    ListRing wf, ww;
    wf.buf = reinterpret_cast<uint16_t*>(ring_base + tid * SPH_RING_F_STRIDE); wf.wn = 0u;
    ww.buf = reinterpret_cast<uint16_t*>(ring_base + SPH_TP * SPH_RING_F_STRIDE + tid * SPH_RING_W_STRIDE); ww.wn = 0u;
    wf.col = a.list_f + (size_t)tile * a.KF8 * SPH_TP + tid; wf.rc = SPH_RING_F; wf.cap8 = a.KF8; wf.fl = 0;
    ww.col = a.list_w + (size_t)tile * a.KW8 * SPH_TP + tid; ww.rc = SPH_RING_W; ww.cap8 = a.KW8; ww.fl = 0;
    const uint32_t gdummy_f = (uint32_t)P.dummy_f, gdummy_w = (uint32_t)P.dummy_w;
    const double half_inv_h = 0.5 * a.inv_h;
    GeomSums g = {0.0, 0.0, 0.0, 0.0};
    unsigned int err = 0;
    int nf = 0, nw = 0;

    if (!staged) {
        RangeTab tf, tw;
        own_table(P, pi, a.cstart_f, valid, tf);
        own_table(P, pi, a.cstart_w, valid && P.n_w > 0, tw);
        const uint32_t df = tf.lb[SPH_NR], dw = tw.lb[SPH_NR];
        const Recs<false> RF{nullptr, a.A, nullptr, &tf, gdummy_f}, RW{nullptr, a.WA, nullptr, &tw, gdummy_w};
        build_one<false>(P, ts.hdr[0], run, nullptr, nullptr, a.A, a.WA, i, valid, pi, a.cstart_f, a.cstart_w, wf, ww, df, dw, RF, RW, half_inv_h, g);
        drain_ring<false>(wf, true, df, RF, pi, half_inv_h, g);
        drain_ring<false>(ww, true, dw, RW, pi, half_inv_h, g);
        if (wf.n() > wf.cap8 * 8 || ww.n() > ww.cap8 * 8) err |= ERR_NEIGH;
        nf = min(wf.n(), wf.cap8 * 8); nw = min(ww.n(), ww.cap8 * 8);
        pad_list(wf, (warp_max_i(nf) + 7) & ~7, df);
        pad_list(ww, (warp_max_i(nw) + 7) & ~7, dw);
    } else {
        for (int q = 0; q < n_slots; ++q) {
            const TileHdr& h = ts.hdr[q];
            const uint32_t tot_f = h.tot_f, tot_w = h.tot_w;
            float4* sA = reinterpret_cast<float4*>(sph_dyn_smem);
            float4* sWA = sA + (tot_f + SPH_ND);
            SPH_DBG_CHECK((tot_f + tot_w + 2u * SPH_ND) * 16u <= SPH_HALF_BYTES && h.n_ranges <= SPH_NRMAX, 7);
            if (q > 0) __syncthreads();                          // everyone is done with the previous pass's records
            if (tid == 0) {
                sA[tot_f] = make_float4(SPH_FAR, SPH_FAR, SPH_FAR, 0.f);
                sWA[tot_w] = make_float4(SPH_FAR, SPH_FAR, SPH_FAR, 0.f);
            }
            __syncthreads();
            if (tid == 0) mbar_arrive_expect_tx(&ts.bar, (tot_f + tot_w) * 16u);
            if (tid < (int)h.n_ranges) {
                stage_range(h.gstart_f, h.lbase_f, tid, a.A, sA, &ts.bar);
                stage_range(h.gstart_w, h.lbase_w, tid, a.WA, sWA, &ts.bar);
            }
            if (myq != q) continue;                              // whole warps: np is a multiple of 32
            mbar_wait(&ts.bar, (uint32_t)(q & 1));
            const Recs<true> RF{sA, a.A, nullptr, nullptr, gdummy_f}, RW{sWA, a.WA, nullptr, nullptr, gdummy_w};
            build_one<true>(P, h, run, sA, sWA, a.A, a.WA, i, valid, pi, a.cstart_f, a.cstart_w, wf, ww, tot_f, tot_w, RF, RW, half_inv_h, g);
            drain_ring<true>(wf, true, tot_f, RF, pi, half_inv_h, g);
            drain_ring<true>(ww, true, tot_w, RW, pi, half_inv_h, g);
            if (wf.n() > wf.cap8 * 8 || ww.n() > ww.cap8 * 8) err |= ERR_NEIGH;
            nf = min(wf.n(), wf.cap8 * 8); nw = min(ww.n(), ww.cap8 * 8);
            // pad every lane's lists to the warp maximum (a whole number of words) with the dummy index
            pad_list(wf, (warp_max_i(nf) + 7) & ~7, tot_f);
            pad_list(ww, (warp_max_i(nw) + 7) & ~7, tot_w);
        }
    }
    {   // cost class of the tile for the sweeps' schedule (0 = most expensive): direct tiles (global gathers), tiles split
        // in four / in two (a staging round trip per pass), wall-rich tiles (torque, body data), the rest
        unsigned int c = valid ? (unsigned int)nf | ((unsigned int)nw << 16) : 0u;       // both sums stay below 2^16
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        __shared__ unsigned int s_cost[SPH_NWARP];
        if ((tid & 31) == 0) s_cost[tid >> 5] = c;
        __syncthreads();
        if (tid == 0) {
            unsigned int sf = 0u, sw = 0u;
            for (int k = 0; k < SPH_NWARP; ++k) { sf += s_cost[k] & 0xffffu; sw += s_cost[k] >> 16; }
            a.tile_bin[tile] = S == 0 ? 0u : S == 4 ? 1u : (S == 2 || 4u * sw > sf) ? 2u : 3u;
        }
    }
    const double sig = a.CW * (1.0 + g.sig);                     // W(0) / CW = 1: self term (R12)
    const double gx = a.CF * g.gx, gy = a.CF * g.gy, gz = a.CF * g.gz;
    if (err) atomicOr(&a.clk->err, err);
    if (valid) {
        a.ncnt[i] = (uint32_t)nf | ((uint32_t)nw << 16);
        a.G[i] = make_float4((float)(a.V0 * gx), (float)(a.V0 * gy), (float)(a.V0 * gz), 0.f);
        if (P.flags & F_DENSITY_REINIT) {
            const float dn = (float)(a.rho0 * (sig - a.sigma0) / a.sigma0);
            if (P.flags & F_FREE_SURFACE_LOCAL) {
                // R27: which form applies is known only when the surface particles have marked their neighbours
                // (k_fs_mark); the re-initialised value waits in G.w for k_fs_apply
                reinterpret_cast<float*>(a.G + i)[3] = dn;
                a.fs_region[i] = sig < a.fs_sigma ? 2 : 0;
            } else {
                const float d = (P.flags & F_FREE_SURFACE) ? fmaxf(pi.w, dn) : dn;
                // only .w changes; other CTAs read .xyz of A in this kernel, never .w
                reinterpret_cast<float*>(a.A + i)[3] = d;
            }
        }
    }
    // bank-aware order of the tile's finished lists (see bank_order_one): done here, while the lists are still in L2 and the
    // other CTA of the SM is busy with its candidate scan (this phase is latency-bound, that one issue-bound); the staged
    // records and the hit buffers are no longer needed and give room to the 256 scatter arrays
    if (a.order_lists && staged && !(a.clk->last_adv_steps > 0 && a.clk->last_adv_steps < a.skip_short)) {
        static_assert(SPH_BO_SMEM <= SPH_BUILD_SMEM, "the scatter arrays reuse the build kernel's dynamic shared memory");
        __shared__ uint2 onehot[8];                                        // byte c of the pair = 1
        __syncthreads();                                                   // every warp is done with the records and its hit buffers
        if (tid < 8) onehot[tid] = tid < 4 ? make_uint2(1u << (8 * tid), 0u) : make_uint2(0u, 1u << (8 * (tid - 4)));
        __syncthreads();
        uint16_t* pos = reinterpret_cast<uint16_t*>(reinterpret_cast<uint32_t*>(sph_dyn_smem) + (size_t)tid * SPH_BO_STRIDE);
        const uint32_t shift = 8u - ((uint32_t)tid & 7u);
        if (valid && nf >= 2) bank_order_one(a.list_f + (size_t)tile * a.KF8 * SPH_TP + tid, nf, pos, onehot, shift);
        if (valid && nw >= 2) bank_order_one(a.list_w + (size_t)tile * a.KW8 * SPH_TP + tid, nw, pos, onehot, shift);
    }
}

__global__ void __launch_bounds__(256) k_tile_order_identity(int n_tiles, uint32_t* __restrict__ order)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n_tiles) order[t] = (uint32_t)t;
}

// Tile schedule of the sweeps: the first n_tiles - n_tail tiles in their natural (spatial) order, then the last n_tail
// tiles STABLY sorted by cost class (most expensive first), so that no expensive tile is started late while tiles drawn at
// about the same time still share staged ranges in L2 (measured: sorting ALL tiles costs ~1 % on workloads with > 100
// tiles per CTA, where there is no tail to win back; profiles/r01e.md).  One CTA of 1024 threads; thread t takes the
// t-th contiguous chunk of the tail region.
__global__ void __launch_bounds__(1024) k_tile_order(int n_tiles, int n_tail, const uint32_t* __restrict__ tile_bin, uint32_t* __restrict__ order,
                                                      const Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    __shared__ unsigned int warp_off[SPH_COST_CLASSES][32];
    __shared__ unsigned int class_base[SPH_COST_CLASSES];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int head = max(n_tiles - n_tail, 0);
    for (int t = tid; t < head; t += 1024) order[t] = (uint32_t)t;
    const int chunk = (n_tiles - head + 1023) / 1024;
    const int t0 = min(head + tid * chunk, n_tiles), t1 = min(t0 + chunk, n_tiles);
    unsigned int c[SPH_COST_CLASSES], pre[SPH_COST_CLASSES];
#pragma unroll
    for (int k = 0; k < SPH_COST_CLASSES; ++k) c[k] = 0u;
    for (int t = t0; t < t1; ++t) {
        const uint32_t b = tile_bin[t];
#pragma unroll
        for (int k = 0; k < SPH_COST_CLASSES; ++k) c[k] += b == (uint32_t)k ? 1u : 0u;
    }
#pragma unroll
    for (int k = 0; k < SPH_COST_CLASSES; ++k) {
        unsigned int x = c[k];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const unsigned int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        pre[k] = x - c[k];
        if (lane == 31) warp_off[k][wid] = x;
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int k = 0; k < SPH_COST_CLASSES; ++k) {
            const unsigned int v = warp_off[k][lane];
            unsigned int x = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const unsigned int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
            warp_off[k][lane] = x - v;
            if (lane == 31) class_base[k] = x;               // class total, turned into a base below
        }
    }
    __syncthreads();
    if (tid == 0) {
        unsigned int run = (unsigned int)head;
        for (int k = 0; k < SPH_COST_CLASSES; ++k) { const unsigned int n = class_base[k]; class_base[k] = run; run += n; }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < SPH_COST_CLASSES; ++k) pre[k] += class_base[k] + warp_off[k][wid];
    for (int t = t0; t < t1; ++t) {
        const uint32_t b = tile_bin[t];
        unsigned int pos = 0u;
#pragma unroll
        for (int k = 0; k < SPH_COST_CLASSES; ++k)
            if (b == (uint32_t)k) { pos = pre[k]; pre[k] += 1u; }
        order[pos] = (uint32_t)t;
    }
}

// ---------------------------------------------------------------------------------------------
// shared prologue of the sweeps: header -> shared memory, TMA staging, dummy records
// ---------------------------------------------------------------------------------------------
struct Staged {
    float4 *sA, *sWA;        // half 0; the B records sit SPH_HALF_BYTES behind
};

__device__ __forceinline__ float4* half1(float4* p) { return reinterpret_cast<float4*>(reinterpret_cast<unsigned char*>(p) + SPH_HALF_BYTES); }

// Staging of one pass of a tile from a header that sits in SHARED memory: the dummy records and the expected byte count
// (thread 0), one thread per range issues its bulk copies (completion on `bar`).  No CTA barrier inside: the caller has
// synchronised the CTA since the last gather from the staging area.  The dummy records reach the readers through the
// mbarrier (released by thread 0's arrive, acquired by every waiter).
__device__ __forceinline__ void issue_staging(uint64_t* bar, const TileHdr& h, const float4* A, const float4* B, const float4* WA,
                                              const float4* WB, bool need_WB)
{
    const int tid = threadIdx.x;
    const uint32_t tot_f = h.tot_f, tot_w = h.tot_w;
    SPH_DBG_CHECK((tot_f + tot_w + 2u * SPH_ND) * 16u <= SPH_HALF_BYTES && h.n_ranges <= SPH_NRMAX, 7);
    float4* sA = reinterpret_cast<float4*>(sph_dyn_smem);
    float4* sWA = sA + (tot_f + SPH_ND);
    if (tid == 0) {
        sA[tot_f] = make_float4(SPH_FAR, SPH_FAR, SPH_FAR, 0.f);
        half1(sA)[tot_f] = make_float4(0.f, 0.f, 0.f, 0.f);
        sWA[tot_w] = make_float4(SPH_FAR, SPH_FAR, SPH_FAR, __int_as_float(0));
        half1(sWA)[tot_w] = make_float4(0.f, 0.f, 0.f, 0.f);
        mbar_arrive_expect_tx(bar, (2 * tot_f + (need_WB ? 2 * tot_w : tot_w)) * 16u);
    }
    // one thread per range issues its bulk copies; the ranges are dealt out across the warps (range q -> lane q / NWARP of warp
    // q % NWARP) so that no single warp carries the whole issue cost into its pair loop
    const int q = (tid & 31) * SPH_NWARP + (tid >> 5);
    if (q < (int)h.n_ranges) {                           // the staging area was last touched through the generic proxy
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        stage_range(h.gstart_f, h.lbase_f, q, A, sA, bar);
        stage_range(h.gstart_f, h.lbase_f, q, B, half1(sA), bar);
        stage_range(h.gstart_w, h.lbase_w, q, WA, sWA, bar);
        if (need_WB) stage_range(h.gstart_w, h.lbase_w, q, WB, half1(sWA), bar);
    }
}

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

__device__ __forceinline__ Staged staged_ptrs(uint32_t tot_f)
{
    Staged s;
    s.sA = reinterpret_cast<float4*>(sph_dyn_smem);
    s.sWA = s.sA + (tot_f + SPH_ND);
    return s;
}

// every warp clears its own torque partials (TileSmem.tq / tv rows): no CTA barrier needed before its wall loop
__device__ __forceinline__ void clear_warp_torque(TileSmem& ts)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane < SPH_MAXB * 3) { ts.tq[wid][lane] = 0.0f; ts.tv[wid][lane] = 0.0f; }
    __syncwarp();
}

struct PairGeom { float dx, dy, dz, rinv, r, F; };

// F = W'(r)/r = CF (1 - q/2)^3 for the 3-D Wendland C2 kernel (R2), q = r/h; 0 beyond the support
__device__ __forceinline__ PairGeom pair_geom(const DevParams& P, float4 ai, float4 aj)
{
    PairGeom g;
    g.dx = ai.x - aj.x; g.dy = ai.y - aj.y; g.dz = ai.z - aj.z;
    const float d2 = fmaf(g.dz, g.dz, fmaf(g.dy, g.dy, fmaf(g.dx, g.dx, SPH_D2_TINY)));      // R28
    g.rinv = rsqrt_fast(d2);
    g.r = d2 * g.rinv;
    const float t = fmaxf(fmaf(g.r, -P.half_inv_h, 1.0f), 0.0f);
    g.F = (P.CF * t) * (t * t);
    return g;
}

// ---------------------------------------------------------------------------------------------
// a8 + a9 + a12  sweep A: momentum equation (Eq. 10 l.2) with the Riemann pressure of
// Eq. 12 (:114), wall forces of Eq. 18-19 (:148-155), the kick v += dt a and the second-half drift
// r += dt/2 v (R7); max |v|^2 for Eq. 25; per-body torque partials (R15).
//   a_i = g - (2/rho_i) [ p_i G_i + sum_j V_j F_ij r_ij ((p*_ij - p_i) - p_i drho_j/rho0) + sum_w V_w F_iw r_iw (p*_iw - p_i) ]
//           + (2 eta/rho_i) [ sum_j V_j F_ij v_ij + sum_w V_w F_iw (v_i - v_w) ]
//   p*_ij - p_i = rho_i [c0^2 (drho_j - drho_i) + rho_j beta (U_L - U_R)] / (rho_i + rho_j)
//   p*_iw - p_i = -rho_i [rho_i g.r_iw] / (rho_i + rho_R)
// ---------------------------------------------------------------------------------------------
// MODE (R26, SPH_FLAG_VISCOUS_HELD): 0 = pressure and viscous sums every step (R8);  1 = the step that rebuilt
// (Clock.rebuild): both sums, the viscous one in accumulators of its own and kept in `avisc` / Clock.torque_visc;
// 2 = the other steps: pressure sums + the held `avisc`.  Under the flag both 1 and 2 are launched every step and the one
// whose turn it is not returns at once.
struct SweepAArgs {
    const float4 *A, *Bc, *WA, *G;
    float4 *Bn, *posc, *acc;
    float4* avisc;                 // held viscous acceleration a^nu_i, sorted order (MODE 1 writes, MODE 2 reads)
    const uint4 *list_f, *list_w;
    const uint32_t* ncnt;
    const uint32_t *cstart_f, *cstart_w;
    const TileHdr* hdr;
    const uint32_t* order;         // tile schedule (k_tile_order)
    Clock* clk;
    int KF8, KW8;
};

// `slot` = the particle's lane slot in its tile (list column); `part` of `S`: this thread takes list words
// part, part + S, ... of the particle (S threads per particle in a sub-tile pass, S = 1 otherwise).
template <bool STAGED, int MODE>
__device__ __forceinline__ void sweepA_body(const DevParams& P, const SweepAArgs& a, TileSmem& ts, const Staged& st, int tile, int slot, int part,
                                            int S, bool valid, float4 ai, float4 bi, int nf, int nw, uint4 first_f, float& ax,
                                            float& ay, float& az, float& avx, float& avy, float& avz)
{
    const int tid = threadIdx.x;
    RangeTab tf, tw;
    if (!STAGED) {
        own_table(P, ai, a.cstart_f, valid, tf);
        own_table(P, ai, a.cstart_w, valid && P.n_w > 0, tw);
    }
    const Recs<STAGED> RF{st.sA, a.A, a.Bc, &tf, (uint32_t)P.dummy_f};
    const Recs<STAGED> RW{st.sWA, a.WA, nullptr, &tw, (uint32_t)P.dummy_w};
    const bool do_p = (P.flags & F_PRESSURE) != 0, do_v = MODE != 2 && (P.flags & F_VISCOUS) != 0;
    const float rho_i = P.rho0 + ai.w, p_i = P.c0sq * ai.w;
    const float inv_rho_i = 1.0f / rho_i;
    const float kpm = do_p ? -2.0f * inv_rho_i * P.mass : 0.0f;          // pressure prefactor times m
    const float kvm = do_v ? 2.0f * inv_rho_i * P.eta * P.mass : 0.0f;   // viscous prefactor times m
    const float pib = p_i * P.inv_rho0;

    // Two pairs at a time in the two halves of 64-bit registers (FFMA2 / FMUL2 / FADD2 of sm_100: one issue slot for two fp32
    // operations; the differences r_ij, v_ji, drho_j - drho_i are scalar subtractions whose results the compiler places in
    // adjacent registers).  With w = v_j - v_i, dd = drho_j - drho_i, F' = t^3 (CF folded into the prefactors), sb = beta / c0
    // = sat(3 du / c0) (3 max(du, 0) = max(3 du, 0) exactly):
    //   du = (w . r_ij) / r,  w1' = rho_j sb du + c0 dd,  q = (rho_i c0 / (rho_i + rho_j)) w1' - (p_i / rho0)(dd + drho_i)
    // cp = kpm CF (F' / rho_j) q: the prefactor kpm CF is folded into q's three coefficients
    const float kq = kpm * P.CF;
    const float2 rhoi2 = dup2(rho_i), c0_2 = dup2(P.c0), K1 = dup2(kq * rho_i * P.c0), K2 = dup2(-kq * pib), K3 = dup2(-kq * pib * ai.w);
    const float2 nkvmCF2 = dup2(-kvm * P.CF);
    const float k3 = 3.0f * P.inv_c0;
    float2 ax2 = dup2(0.f), ay2 = dup2(0.f), az2 = dup2(0.f), avx2 = dup2(0.f), avy2 = dup2(0.f), avz2 = dup2(0.f);
    auto pair2 = [&](const float4& a0, const float4& b0, const float4& a1, const float4& b1) {
        const float2 dx = make_float2(ai.x - a0.x, ai.x - a1.x), dy = make_float2(ai.y - a0.y, ai.y - a1.y), dz = make_float2(ai.z - a0.z, ai.z - a1.z);
        const float2 d2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __ffma2_rn(dx, dx, dup2(SPH_D2_TINY))));      // R28
        const float2 rinv = make_float2(rsqrt_fast(d2.x), rsqrt_fast(d2.y));
        const float2 r = __fmul2_rn(d2, rinv);
        const float2 t = make_float2(__saturatef(fmaf(r.x, -P.half_inv_h, 1.0f)), __saturatef(fmaf(r.y, -P.half_inv_h, 1.0f)));
        const float2 F3 = __fmul2_rn(__fmul2_rn(t, t), t);                                  // F / CF
        const float2 dd = make_float2(a0.w - ai.w, a1.w - ai.w);
        const float2 rhoj = __fadd2_rn(rhoi2, dd);
        const float2 VF = __fmul2_rn(make_float2(rcp_fast(rhoj.x), rcp_fast(rhoj.y)), F3);  // V_j F_ij / (m CF)
        const float2 wx = make_float2(b0.x - bi.x, b1.x - bi.x), wy = make_float2(b0.y - bi.y, b1.y - bi.y), wz = make_float2(b0.z - bi.z, b1.z - bi.z);
        if (MODE == 2) {
            (void)wx;
        }
        const float2 du = __fmul2_rn(__ffma2_rn(wz, dz, __ffma2_rn(wy, dy, __fmul2_rn(wx, dx))), rinv);     // U_L - U_R (Eq. 11)
        const float2 sb = make_float2(__saturatef(du.x * k3), __saturatef(du.y * k3));                        // limiter / c0
        const float2 w1 = __ffma2_rn(__fmul2_rn(rhoj, sb), du, __fmul2_rn(c0_2, dd));
        const float2 rs = __fadd2_rn(rhoj, rhoi2);
        const float2 rr = make_float2(rcp_fast(rs.x), rcp_fast(rs.y));
        const float2 q = __ffma2_rn(__fmul2_rn(K1, rr), w1, __ffma2_rn(K2, dd, K3));          // kpm CF q
        const float2 cp = __fmul2_rn(VF, q);
        if (MODE == 0) {
            const float2 cvn = __fmul2_rn(nkvmCF2, VF);
            ax2 = __ffma2_rn(cp, dx, __ffma2_rn(cvn, wx, ax2));
            ay2 = __ffma2_rn(cp, dy, __ffma2_rn(cvn, wy, ay2));
            az2 = __ffma2_rn(cp, dz, __ffma2_rn(cvn, wz, az2));
        } else {
            ax2 = __ffma2_rn(cp, dx, ax2); ay2 = __ffma2_rn(cp, dy, ay2); az2 = __ffma2_rn(cp, dz, az2);
            if (MODE == 1) {
                const float2 cvn = __fmul2_rn(nkvmCF2, VF);
                avx2 = __ffma2_rn(cvn, wx, avx2); avy2 = __ffma2_rn(cvn, wy, avy2); avz2 = __ffma2_rn(cvn, wz, avz2);
            }
        }
    };
    auto fluid4 = [&](uint32_t lo, uint32_t hi) {
        uint32_t L[4];
        unpack4(lo, hi, L);
        float4 aj[4], bj[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) RF.AB(L[e], aj[e], bj[e]);
        pair2(aj[0], bj[0], aj[1], bj[1]);
        pair2(aj[2], bj[2], aj[3], bj[3]);
    };
    {
        const int n4 = (warp_max_i(nf) + 3) & ~3, n8 = (n4 + 7) >> 3;
        const uint4* lf = a.list_f + (size_t)tile * a.KF8 * SPH_TP + slot;
        uint4 nxt = first_f;
#pragma unroll 1
        for (int k8 = part; k8 < n8; k8 += S) {
            const uint4 cur = nxt;
            if (k8 + S < n8) nxt = __ldcs(lf + (size_t)(k8 + S) * SPH_TP);
            fluid4(cur.x, cur.y);
            if (8 * k8 + 4 < n4) fluid4(cur.z, cur.w);
        }
    }

    ax += ax2.x + ax2.y; ay += ay2.x + ay2.y; az += az2.x + az2.y;
    if (MODE == 1) { avx += avx2.x + avx2.y; avy += avy2.x + avy2.y; avz += avz2.x + avz2.y; }
    // walls: torque accumulated for the body of the current run of wall neighbours
    const float kp = do_p ? -2.0f * inv_rho_i * P.Vw : 0.0f;
    const float kv = do_v ? 2.0f * inv_rho_i * P.eta * P.Vw : 0.0f;
    int cur_b = -1;
    float tqx = 0.f, tqy = 0.f, tqz = 0.f;
    float tvx = 0.f, tvy = 0.f, tvz = 0.f;            // MODE 1: moment of the viscous forces on its own
    float* tqw = ts.tq[tid >> 5];
    float* tvw = ts.tv[tid >> 5];
    auto wall4 = [&](uint32_t lo, uint32_t hi) {
        uint32_t L[4];
        unpack4(lo, hi, L);
        float4 wa4[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) wa4[e] = RW.A(L[e]);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float4 wa = wa4[e];
            const PairGeom g = pair_geom(P, ai, wa);
            const int b = __float_as_int(wa.w);
            const BodyF bd = P.body[b];
            const float px = wa.x - bd.ox, py = wa.y - bd.oy, pz = wa.z - bd.oz;        // r_w - o_b
            const float vwx = bd.wy * pz - bd.wz * py, vwy = bd.wz * px - bd.wx * pz, vwz = bd.wx * py - bd.wy * px;
            const float dpg = rho_i * (P.gx * g.dx + P.gy * g.dy + P.gz * g.dz);       // p_L - p_R (Eq. 17, r_fw = -r_iw)
            const float rsum = fmaf(-dpg, P.inv_c0sq, 2.0f * rho_i);                    // rho_i + rho_R
            const float q = -rho_i * dpg * rcp_fast(rsum);                              // p*_iw - p_i (Eq. 19)
            const float cpq = kp * g.F * q, cpi = kp * g.F * p_i, cv = kv * g.F;
            // acceleration of i: small-term part here, p_i part through G_i
            const float vx = bi.x - vwx, vy = bi.y - vwy, vz = bi.z - vwz;
            // force on the wall particle = -m_i (full pair acceleration); moment about o_b
            const float cpt = cpq + cpi;
            float Fx, Fy, Fz;
            if (MODE == 1) {
                ax = fmaf(cpq, g.dx, ax); ay = fmaf(cpq, g.dy, ay); az = fmaf(cpq, g.dz, az);
                avx = fmaf(cv, vx, avx); avy = fmaf(cv, vy, avy); avz = fmaf(cv, vz, avz);
                Fx = -P.mass * (cpt * g.dx); Fy = -P.mass * (cpt * g.dy); Fz = -P.mass * (cpt * g.dz);
            } else {
                ax = fmaf(cpq, g.dx, fmaf(cv, vx, ax));
                ay = fmaf(cpq, g.dy, fmaf(cv, vy, ay));
                az = fmaf(cpq, g.dz, fmaf(cv, vz, az));
                Fx = -P.mass * fmaf(cpt, g.dx, cv * vx); Fy = -P.mass * fmaf(cpt, g.dy, cv * vy); Fz = -P.mass * fmaf(cpt, g.dz, cv * vz);
            }
            if (b != cur_b && g.F != 0.0f) {                // padding (F = 0) never switches the body
                if (cur_b >= 0) {
                    atomicAdd(&tqw[cur_b * 3 + 0], tqx); atomicAdd(&tqw[cur_b * 3 + 1], tqy); atomicAdd(&tqw[cur_b * 3 + 2], tqz);
                    if (MODE == 1) { atomicAdd(&tvw[cur_b * 3 + 0], tvx); atomicAdd(&tvw[cur_b * 3 + 1], tvy); atomicAdd(&tvw[cur_b * 3 + 2], tvz); }
                }
                cur_b = b; tqx = tqy = tqz = 0.f; tvx = tvy = tvz = 0.f;
            }
            tqx += py * Fz - pz * Fy; tqy += pz * Fx - px * Fz; tqz += px * Fy - py * Fx;
            if (MODE == 1) {
                const float Gx = -P.mass * (cv * vx), Gy = -P.mass * (cv * vy), Gz = -P.mass * (cv * vz);
                tvx += py * Gz - pz * Gy; tvy += pz * Gx - px * Gz; tvz += px * Gy - py * Gx;
            }
        }
    };
    {
        const int n4 = (warp_max_i(nw) + 3) & ~3, n8 = (n4 + 7) >> 3;
        const uint4* lw = a.list_w + (size_t)tile * a.KW8 * SPH_TP + slot;
        uint4 nxt = make_uint4(0u, 0u, 0u, 0u);
        if (part < n8) nxt = __ldcs(lw + (size_t)part * SPH_TP);          // (prefetched to L2 a tile ago; not held across the fluid loop)
#pragma unroll 1
        for (int k8 = part; k8 < n8; k8 += S) {
            const uint4 cur = nxt;
            if (k8 + S < n8) nxt = __ldcs(lw + (size_t)(k8 + S) * SPH_TP);
            wall4(cur.x, cur.y);
            if (8 * k8 + 4 < n4) wall4(cur.z, cur.w);
        }
        if (n8 > 0) {                                                    // warp-uniform: this warp met walls
            // close the open runs: one shuffle reduction per body present in the warp (the warp's slot of
            // ts.tq is private to it), then one fp64 atomic per body and component
            const int lane = tid & 31;
            __syncwarp();                                                // mid-loop shared atomics of other lanes are done
            unsigned open = __ballot_sync(0xffffffffu, cur_b >= 0);
            while (open) {
                const int bb = __shfl_sync(0xffffffffu, cur_b, __ffs(open) - 1);
                const bool mine = cur_b == bb;
                float x = mine ? tqx : 0.f, y = mine ? tqy : 0.f, z = mine ? tqz : 0.f;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    x += __shfl_xor_sync(0xffffffffu, x, o); y += __shfl_xor_sync(0xffffffffu, y, o); z += __shfl_xor_sync(0xffffffffu, z, o);
                }
                if (lane == 0) { tqw[bb * 3 + 0] += x; tqw[bb * 3 + 1] += y; tqw[bb * 3 + 2] += z; }
                if (MODE == 1) {
                    x = mine ? tvx : 0.f; y = mine ? tvy : 0.f; z = mine ? tvz : 0.f;
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        x += __shfl_xor_sync(0xffffffffu, x, o); y += __shfl_xor_sync(0xffffffffu, y, o); z += __shfl_xor_sync(0xffffffffu, z, o);
                    }
                    if (lane == 0) { tvw[bb * 3 + 0] += x; tvw[bb * 3 + 1] += y; tvw[bb * 3 + 2] += z; }
                }
                open &= ~__ballot_sync(0xffffffffu, mine);
            }
            __syncwarp();
            if (lane < SPH_MAXB * 3) {
                const float t = tqw[lane];
                if (t != 0.f) atomicAdd(&a.clk->torque[lane / 3][lane % 3], (double)t);
                if (MODE == 1) {
                    const float tv = tvw[lane];
                    if (tv != 0.f) atomicAdd(&a.clk->torque_visc[lane / 3][lane % 3], (double)tv);
                }
            }
        }
    }
}

// Persistent CTAs (2 per SM) draw tiles from an atomic counter.  Pipeline of one CTA (round 2: a CTA spent 30 % of its time
// waiting at tile boundaries, profiles/r02c.md):
//   * tickets run two tiles ahead, so the id of the NEXT tile is known when a tile starts and its pass-0 header is read from
//     global memory during the pair loop (one word per thread) and parked in the other half of s_hdr;
//   * one CTA barrier per tile ("all gathers from the staging area are done"); right behind it the staging of the next tile is
//     issued (TMA bulk copies on ts.bar), and only then the finished tile's own-particle work (kick, drift, global stores) and
//     the next tile's own-record loads run, i.e. they overlap the staging round trip instead of preceding it.
// Split tiles (S = 2, 4) take their passes q >= 1 the plain way (header from global memory into ts.hdr, barrier, staging).
#define SPH_HDR_WORDS ((int)(sizeof(TileHdr) / 4))
// Order in which the persistent CTAs draw tiles: ticket t of the atomic counter -> tile order[t], the tiles sorted by
// cost class at every rebuild (k_build_tiles + k_tile_order), so that the expensive tiles (split or direct tiles,
// wall-rich tiles) are not the ones the last CTAs are still working on when the others have run dry.
#define SPH_TILE_OK(t) ((t) < n_tiles)
#define SPH_TILE_NONE n_tiles
__device__ __forceinline__ int ticket_tile(unsigned int t, int n_tiles, const uint32_t* __restrict__ order)
{
    return t < (unsigned int)n_tiles ? (int)__ldg(order + t) : n_tiles;
}

// shared state of the tile pipeline of one persistent CTA
struct SweepPipe {
    TileHdr hdr[2];          // pass-0 header of the current tile (hdr[it & 1]) and of the next one
    int ticket[2];           // tickets handed from thread 0 to the CTA across the per-tile barrier
};

// start of a sweep kernel: the first two tickets, the first header, the first staging.  Returns the first tile.
__device__ __forceinline__ int pipe_begin(SweepPipe& pp, TileSmem& ts, const TileHdr* __restrict__ hdr, const uint32_t* __restrict__ order,
                                          unsigned int* work, int n_tiles, int& next, bool& issued, const float4* A, const float4* B,
                                          const float4* WA, const float4* WB, bool need_WB)
{
    const int tid = threadIdx.x;
    if (tid == 0) {
        pp.ticket[0] = (int)atomicAdd(work, 1u);
        pp.ticket[1] = (int)atomicAdd(work, 1u);
        mbar_init(&ts.bar, 1);
    }
    __syncthreads();
    const int tile = ticket_tile((unsigned int)pp.ticket[0], n_tiles, order);
    next = ticket_tile((unsigned int)pp.ticket[1], n_tiles, order);
    if (SPH_TILE_OK(tile) && tid < SPH_HDR_WORDS)
        reinterpret_cast<uint32_t*>(&pp.hdr[0])[tid] = __ldg(reinterpret_cast<const uint32_t*>(hdr + (size_t)tile * SPH_SMAX) + tid);
    __syncthreads();
    issued = SPH_TILE_OK(tile) && pp.hdr[0].S != 0u;
    if (issued) issue_staging(&ts.bar, pp.hdr[0], A, B, WA, WB, need_WB);
    return tile;
}

// passes q >= 1 of a split tile: header slot from global memory, barrier, staging
__device__ __forceinline__ void stage_later_pass(TileSmem& ts, const TileHdr* __restrict__ slot, const float4* A, const float4* B, const float4* WA,
                                                 const float4* WB, bool need_WB)
{
    const int tid = threadIdx.x;
    if (tid < SPH_HDR_WORDS) reinterpret_cast<uint32_t*>(&ts.hdr)[tid] = __ldg(reinterpret_cast<const uint32_t*>(slot) + tid);
    __syncthreads();
    issue_staging(&ts.bar, ts.hdr, A, B, WA, WB, need_WB);
}

template <int MODE>
__global__ void __launch_bounds__(SPH_TP, SPH_MINB) k_sweep_A(DevParams P, SweepAArgs a, int n_tiles, unsigned int* work)
{
    if (MODE != 0 && (a.clk->rebuild != 0) != (MODE == 1)) return;      // R26: 1 = the step that rebuilt, 2 = the others
    __shared__ TileSmem ts;
    __shared__ SweepPipe pp;
    static_assert(SPH_HDR_WORDS <= SPH_TP, "one header word per thread");
    const int tid = threadIdx.x, lane = tid & 31;
    int next, it = 0;
    bool issued;
    int tile = pipe_begin(pp, ts, a.hdr, a.order, work, n_tiles, next, issued, a.A, a.Bc, a.WA, nullptr, false);
    uint32_t use = 0;                                         // staged passes so far: mbarrier phase parity
    const float dt = a.clk->dt_f;
    float v2 = 0.f;
#pragma unroll 1
    while (SPH_TILE_OK(tile)) {
    const TileHdr& h0 = pp.hdr[it & 1];
    const TileHdr* slots = a.hdr + (size_t)tile * SPH_SMAX;
    const int S0 = (int)h0.S;                             // 0: direct mode
    const int S = S0 > 1 ? S0 : 1, np = SPH_TP / S;
    const int part = tid / np, slot0 = tid - part * np;
    const uint32_t tot_f0 = h0.tot_f;
    int tk = 0;
    if (tid == 0) tk = (int)atomicAdd(work, 1u);          // ticket of the tile after the next one
    // the next tile's pass-0 header: one word per thread, lands during the pair loop
    uint32_t hreg = 0u;
    if (SPH_TILE_OK(next) && tid < SPH_HDR_WORDS) hreg = __ldg(reinterpret_cast<const uint32_t*>(a.hdr + (size_t)next * SPH_SMAX) + tid);
    if (SPH_TILE_OK(next)) {                              // the next tile's own records and first list words: on their way to L2 now,
        const size_t j = min((size_t)next * SPH_TP + tid, (size_t)P.n_f - 1);      // read right after this tile's barrier
        prefetch_l2(a.A + j); prefetch_l2(a.Bc + j); prefetch_l2(a.G + j); prefetch_l2(a.posc + j);
        if ((tid & 3) == 0) prefetch_l2(a.ncnt + j);
        prefetch_l2(a.list_f + (size_t)next * a.KF8 * SPH_TP + tid);
        prefetch_l2(a.list_w + (size_t)next * a.KW8 * SPH_TP + tid);
    }
#pragma unroll 1
    for (int q = 0; q < S; ++q) {
        // own records and first list words: issued before the staging wait so that their latency overlaps it
        // (an unused list word is never dereferenced)
        const int slot = q * np + slot0;
        const int i = tile * SPH_TP + slot;
        const bool valid = i < P.n_f;
        const int ii = valid ? i : P.n_f - 1;
        const float4 ai = a.A[ii], bi = a.Bc[ii];
        const uint32_t c = valid ? a.ncnt[ii] : 0u;
        const uint4 first_f = __ldcs(a.list_f + ((size_t)tile * a.KF8 + min(part, a.KF8 - 1)) * SPH_TP + slot);      // list words: read once, evict first
        uint32_t tot_f = tot_f0;
        if (q > 0) {                                       // (the barrier at the end of pass q - 1 has been passed)
            stage_later_pass(ts, slots + q, a.A, a.Bc, a.WA, nullptr, false);
            tot_f = ts.hdr.tot_f;
        }
        const Staged st = staged_ptrs(tot_f);
        clear_warp_torque(ts);
        const int nf = c & 0xffffu, nw = c >> 16;
        float ax = 0.f, ay = 0.f, az = 0.f, avx = 0.f, avy = 0.f, avz = 0.f;
        if (S0 != 0) {
            mbar_wait(&ts.bar, use & 1u);
            ++use;
            sweepA_body<true, MODE>(P, a, ts, st, tile, slot, part, S, valid, ai, bi, nf, nw, first_f, ax, ay, az, avx, avy, avz);
        } else {
            sweepA_body<false, MODE>(P, a, ts, st, tile, slot, part, S, valid, ai, bi, nf, nw, first_f, ax, ay, az, avx, avy, avz);
        }
        if (S > 1) {                                       // sum the S partial accelerations of each particle
            float4* red = reinterpret_cast<float4*>(sph_dyn_smem);
            __syncthreads();                               // all gathers from the staged records are done
            if (part > 0) { red[tid] = make_float4(ax, ay, az, 0.f); if (MODE == 1) red[SPH_TP + tid] = make_float4(avx, avy, avz, 0.f); }
            __syncthreads();
            if (part == 0)
                for (int k = 1; k < S; ++k) {
                    const float4 r = red[tid + k * np]; ax += r.x; ay += r.y; az += r.z;
                    if (MODE == 1) { const float4 rv = red[SPH_TP + tid + k * np]; avx += rv.x; avy += rv.y; avz += rv.z; }
                }
        }
        if (q == S - 1) {                                  // hand the next header and the new ticket to the CTA
            if (SPH_TILE_OK(next) && tid < SPH_HDR_WORDS) reinterpret_cast<uint32_t*>(&pp.hdr[(it + 1) & 1])[tid] = hreg;
            if (tid == 0) pp.ticket[it & 1] = tk;
        }
        __syncthreads();                                   // the staging area is free: next pass or next tile
        if (q == S - 1) {
            issued = SPH_TILE_OK(next) && pp.hdr[(it + 1) & 1].S != 0u;
            if (issued) issue_staging(&ts.bar, pp.hdr[(it + 1) & 1], a.A, a.Bc, a.WA, nullptr, false);
        }
        if (valid && part == 0) {                          // own-particle work of this pass: overlaps the staging round trip
            const float4 G = a.G[i];                       // (prefetched to L2 a tile ago; loaded here, not across the pair loop)
            float4 pc = a.posc[i];
            if (MODE == 1) { a.avisc[i] = make_float4(avx, avy, avz, 0.f); ax += avx; ay += avy; az += avz; }
            if (MODE == 2) { const float4 av = a.avisc[i]; ax += av.x; ay += av.y; az += av.z; }
            if (P.flags & F_PRESSURE) {                                          // p_i G_i: the uniform-pressure part
                const float cg = -2.0f * (P.c0sq * ai.w) / (P.rho0 + ai.w);
                ax = fmaf(cg, G.x, ax); ay = fmaf(cg, G.y, ay); az = fmaf(cg, G.z, az);
            }
            ax += P.gx; ay += P.gy; az += P.gz;
            const float vx = fmaf(dt, ax, bi.x), vy = fmaf(dt, ay, bi.y), vz = fmaf(dt, az, bi.z);      // a9 kick
            a.Bn[i] = make_float4(vx, vy, vz, bi.w);
            const float hdt = 0.5f * dt;
            pc.x = fmaf(hdt, vx, pc.x); pc.y = fmaf(hdt, vy, pc.y); pc.z = fmaf(hdt, vz, pc.z);        // a9 drift
            a.posc[i] = pc;
            a.acc[i] = make_float4(ax, ay, az, 0.f);
            v2 = fmaxf(v2, vx * vx + vy * vy + vz * vz);
        }
    }
    tile = next;
    next = ticket_tile((unsigned int)pp.ticket[it & 1], n_tiles, a.order);
    ++it;
    }
    (void)issued;
    v2 = warp_max(v2);
    if (lane == 0 && v2 > 0.f) atomicMax(&a.clk->vmax2_bits, __float_as_uint(v2));
}

// ---------------------------------------------------------------------------------------------
// a10  sweep B: continuity (Eq. 10 l.1; v* of Eq. 13 under R3; wall term R6) and heat
// conduction (Eq. 22; R9-R10), using v^{n+1}, rho^{n+1/2}, T^n.
//   drho_i/dt = 2 rho_i [ sum_j V_j ( rho_j v_ij.e_ij + (p_i - p_j)/c0 ) / (rho_i + rho_j) W'_ij
//                         + sum_w V_w (U*_iw - U_L)(n_w.e_iw) W'_iw ]
//   dT_i/dt   = 1/(rho_i cp) [ 2 k_f sum_j V_j T_ij F_ij + sum_w V_w K_w T_iw F_iw ]
// ---------------------------------------------------------------------------------------------
struct SweepBArgs {
    const float4 *A, *B, *WA, *WB;
    const uint4 *list_f, *list_w;
    const uint32_t* ncnt;
    const uint32_t *cstart_f, *cstart_w;
    const TileHdr* hdr;
    const uint32_t* order;         // tile schedule (k_tile_order)
    float2* rates;
    int KF8, KW8;
};

template <bool STAGED>
__device__ __forceinline__ void sweepB_body(const DevParams& P, const SweepBArgs& a, const Staged& st, int tile, int slot, int part, int S,
                                            bool valid, float4 ai, float4 bi, int nf, int nw, uint4 first_f, uint4 first_w, float& sr, float& sT)
{
    RangeTab tf, tw;
    if (!STAGED) {
        own_table(P, ai, a.cstart_f, valid, tf);
        own_table(P, ai, a.cstart_w, valid && P.n_w > 0, tw);
    }
    const Recs<STAGED> RF{st.sA, a.A, a.B, &tf, (uint32_t)P.dummy_f};
    const Recs<STAGED> RW{st.sWA, a.WA, a.WB, &tw, (uint32_t)P.dummy_w};
    const float rho_i = P.rho0 + ai.w, p_i = P.c0sq * ai.w;
    // two pairs at a time in 64-bit registers (see sweepA_body); w = v_j - v_i, dd = drho_j - drho_i, F' = t^3:
    //   sr += (V_j F / m) r [rho_j v_ij.e_ij + c0 (drho_i - drho_j)] / (rho_i + rho_j)
    //       = CF (F' / rho_j) [rho_j (w . r_ij) (-1) + (-c0 dd) r] / (rho_i + rho_j)          (v_ij.e_ij r = -(w . r_ij))
    const float2 rhoi2 = dup2(rho_i), nc0_2 = dup2(-P.c0);
    float2 sr2 = dup2(0.f), sT2 = dup2(0.f);
    auto pair2 = [&](const float4& a0, const float4& b0, const float4& a1, const float4& b1) {
        const float2 dx = make_float2(ai.x - a0.x, ai.x - a1.x), dy = make_float2(ai.y - a0.y, ai.y - a1.y), dz = make_float2(ai.z - a0.z, ai.z - a1.z);
        const float2 d2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __ffma2_rn(dx, dx, dup2(SPH_D2_TINY))));      // R28
        const float2 rinv = make_float2(rsqrt_fast(d2.x), rsqrt_fast(d2.y));
        const float2 r = __fmul2_rn(d2, rinv);
        const float2 t = make_float2(__saturatef(fmaf(r.x, -P.half_inv_h, 1.0f)), __saturatef(fmaf(r.y, -P.half_inv_h, 1.0f)));
        const float2 F3 = __fmul2_rn(__fmul2_rn(t, t), t);                                  // F / CF
        const float2 dd = make_float2(a0.w - ai.w, a1.w - ai.w);
        const float2 rhoj = __fadd2_rn(rhoi2, dd);
        const float2 VF = __fmul2_rn(make_float2(rcp_fast(rhoj.x), rcp_fast(rhoj.y)), F3);  // V_j F_ij / (m CF)
        const float2 vx = make_float2(bi.x - b0.x, bi.x - b1.x), vy = make_float2(bi.y - b0.y, bi.y - b1.y), vz = make_float2(bi.z - b0.z, bi.z - b1.z);
        const float2 vr = __ffma2_rn(vz, dz, __ffma2_rn(vy, dy, __fmul2_rn(vx, dx)));
        // (v_i - v*).e_ij W' = [rho_j v_ij.e_ij + (p_i - p_j)/c0] / (rho_i + rho_j) * F r;  (p_i - p_j)/c0 = -c0 dd
        const float2 num = __ffma2_rn(__fmul2_rn(rhoj, vr), rinv, __fmul2_rn(nc0_2, dd));
        const float2 rs = __fadd2_rn(rhoj, rhoi2);
        const float2 rr = make_float2(rcp_fast(rs.x), rcp_fast(rs.y));
        sr2 = __ffma2_rn(__fmul2_rn(VF, r), __fmul2_rn(num, rr), sr2);
        sT2 = __ffma2_rn(VF, make_float2(bi.w - b0.w, bi.w - b1.w), sT2);
    };
    auto fluid4 = [&](uint32_t lo, uint32_t hi) {
        uint32_t L[4];
        unpack4(lo, hi, L);
        float4 aj[4], bj[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) RF.AB(L[e], aj[e], bj[e]);
        pair2(aj[0], bj[0], aj[1], bj[1]);
        pair2(aj[2], bj[2], aj[3], bj[3]);
    };
    {
        const int n4 = (warp_max_i(nf) + 3) & ~3, n8 = (n4 + 7) >> 3;
        const uint4* lf = a.list_f + (size_t)tile * a.KF8 * SPH_TP + slot;
        uint4 nxt = first_f;
#pragma unroll 1
        for (int k8 = part; k8 < n8; k8 += S) {
            const uint4 cur = nxt;
            if (k8 + S < n8) nxt = __ldcs(lf + (size_t)(k8 + S) * SPH_TP);
            fluid4(cur.x, cur.y);
            if (8 * k8 + 4 < n4) fluid4(cur.z, cur.w);
        }
    }
    sr = (sr2.x + sr2.y) * (P.mass * P.CF);
    sT = (sT2.x + sT2.y) * (P.mass * P.CF) * P.k2f;                           // K_ij = 4 k k/(2k) = 2 k_f
    auto wall4 = [&](uint32_t lo, uint32_t hi) {
        uint32_t L[4];
        unpack4(lo, hi, L);
        float4 wa4[4], wb4[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) RW.AB(L[e], wa4[e], wb4[e]);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float4 wa = wa4[e], wb = wb4[e];
            const PairGeom g = pair_geom(P, ai, wa);
            const int b = __float_as_int(wa.w);
            const BodyF bd = P.body[b];
            const float px = wa.x - bd.ox, py = wa.y - bd.oy, pz = wa.z - bd.oz;
            const float vwx = bd.wy * pz - bd.wz * py, vwy = bd.wz * px - bd.wx * pz, vwz = bd.wx * py - bd.wy * px;
            const float UL = -(wb.x * bi.x + wb.y * bi.y + wb.z * bi.z);               // Eq. 16
            const float uw = -(wb.x * vwx + wb.y * vwy + wb.z * vwz);
            const float UR = -UL + 2.0f * uw;                                          // Eq. 17
            const float dpg = rho_i * (P.gx * g.dx + P.gy * g.dy + P.gz * g.dz);       // p_L - p_R (Eq. 17)
            const float rhoR = P.rho0 + (p_i - dpg) * P.inv_c0sq;
            const float rs_inv = rcp_fast(rho_i + rhoR);
            const float Ustar = (rho_i * UL + rhoR * UR) * rs_inv + dpg * P.inv_c0 * rs_inv;           // Eq. 12 l.1
            const float ne = (wb.x * g.dx + wb.y * g.dy + wb.z * g.dz) * g.rinv;       // n_w . e_iw
            const float VF = P.Vw * g.F;
            sr = fmaf(VF * g.r, (Ustar - UL) * ne, sr);                                // R6
            sT = fmaf(VF * bd.K, bi.w - wb.w, sT);
        }
    };
    {
        const int n4 = (warp_max_i(nw) + 3) & ~3, n8 = (n4 + 7) >> 3;
        const uint4* lw = a.list_w + (size_t)tile * a.KW8 * SPH_TP + slot;
        uint4 nxt = first_w;
#pragma unroll 1
        for (int k8 = part; k8 < n8; k8 += S) {
            const uint4 cur = nxt;
            if (k8 + S < n8) nxt = __ldcs(lw + (size_t)(k8 + S) * SPH_TP);
            wall4(cur.x, cur.y);
            if (8 * k8 + 4 < n4) wall4(cur.z, cur.w);
        }
    }
}

__global__ void __launch_bounds__(SPH_TP, SPH_MINB) k_sweep_B(DevParams P, SweepBArgs a, int n_tiles, unsigned int* work)
{
    __shared__ TileSmem ts;
    __shared__ SweepPipe pp;                              // tile pipeline: see k_sweep_A
    const int tid = threadIdx.x;
    int next, it = 0;
    bool issued;
    int tile = pipe_begin(pp, ts, a.hdr, a.order, work, n_tiles, next, issued, a.A, a.B, a.WA, a.WB, true);
    uint32_t use = 0;
#pragma unroll 1
    while (SPH_TILE_OK(tile)) {
    const TileHdr& h0 = pp.hdr[it & 1];
    const TileHdr* slots = a.hdr + (size_t)tile * SPH_SMAX;
    const int S0 = (int)h0.S;
    const int S = S0 > 1 ? S0 : 1, np = SPH_TP / S;
    const int part = tid / np, slot0 = tid - part * np;
    const uint32_t tot_f0 = h0.tot_f;
    int tk = 0;
    if (tid == 0) tk = (int)atomicAdd(work, 1u);          // ticket of the tile after the next one
    uint32_t hreg = 0u;
    if (SPH_TILE_OK(next) && tid < SPH_HDR_WORDS) hreg = __ldg(reinterpret_cast<const uint32_t*>(a.hdr + (size_t)next * SPH_SMAX) + tid);
    if (SPH_TILE_OK(next)) {                              // the next tile's own records and first list words -> L2
        const size_t j = min((size_t)next * SPH_TP + tid, (size_t)P.n_f - 1);
        prefetch_l2(a.A + j); prefetch_l2(a.B + j);
        if ((tid & 3) == 0) prefetch_l2(a.ncnt + j);
        prefetch_l2(a.list_f + (size_t)next * a.KF8 * SPH_TP + tid);
        prefetch_l2(a.list_w + (size_t)next * a.KW8 * SPH_TP + tid);
    }
#pragma unroll 1
    for (int q = 0; q < S; ++q) {
        const int slot = q * np + slot0;
        const int i = tile * SPH_TP + slot;
        const bool valid = i < P.n_f;
        const int ii = valid ? i : P.n_f - 1;
        const float4 ai = a.A[ii], bi = a.B[ii];
        const uint32_t c = valid ? a.ncnt[ii] : 0u;
        const uint4 first_f = __ldcs(a.list_f + ((size_t)tile * a.KF8 + min(part, a.KF8 - 1)) * SPH_TP + slot);      // list words: read once, evict first
        const uint4 first_w = __ldcs(a.list_w + ((size_t)tile * a.KW8 + min(part, a.KW8 - 1)) * SPH_TP + slot);
        uint32_t tot_f = tot_f0;
        if (q > 0) {
            stage_later_pass(ts, slots + q, a.A, a.B, a.WA, a.WB, true);
            tot_f = ts.hdr.tot_f;
        }
        const Staged st = staged_ptrs(tot_f);
        const int nf = c & 0xffffu, nw = c >> 16;
        float sr = 0.f, sT = 0.f;
        if (S0 != 0) {
            mbar_wait(&ts.bar, use & 1u);
            ++use;
            sweepB_body<true>(P, a, st, tile, slot, part, S, valid, ai, bi, nf, nw, first_f, first_w, sr, sT);
        } else {
            sweepB_body<false>(P, a, st, tile, slot, part, S, valid, ai, bi, nf, nw, first_f, first_w, sr, sT);
        }
        if (S > 1) {
            float2* red = reinterpret_cast<float2*>(sph_dyn_smem);
            __syncthreads();
            if (part > 0) red[tid] = make_float2(sr, sT);
            __syncthreads();
            if (part == 0)
                for (int k = 1; k < S; ++k) { const float2 r = red[tid + k * np]; sr += r.x; sT += r.y; }
        }
        if (q == S - 1) {
            if (SPH_TILE_OK(next) && tid < SPH_HDR_WORDS) reinterpret_cast<uint32_t*>(&pp.hdr[(it + 1) & 1])[tid] = hreg;
            if (tid == 0) pp.ticket[it & 1] = tk;
        }
        __syncthreads();                                   // the staging area is free: next pass or next tile
        if (q == S - 1) {
            issued = SPH_TILE_OK(next) && pp.hdr[(it + 1) & 1].S != 0u;
            if (issued) issue_staging(&ts.bar, pp.hdr[(it + 1) & 1], a.A, a.B, a.WA, a.WB, true);
        }
        if (valid && part == 0) {
            const bool hydro = (P.flags & F_HYDRO) != 0, thermal = (P.flags & F_THERMAL) != 0;
            const float rho_i = P.rho0 + ai.w;
            a.rates[i] = make_float2(hydro ? 2.0f * rho_i * sr : 0.0f, thermal ? sT * P.inv_cp / rho_i : 0.0f);
        }
    }
    tile = next;
    next = ticket_tile((unsigned int)pp.ticket[it & 1], n_tiles, a.order);
    ++it;
    }
    (void)issued;
}

// ---------------------------------------------------------------------------------------------
// Contact factor of the solid particles, Eq. 24, reading R22: one thread per sorted wall
// particle walks its candidate windows in the sorted fluid and wall arrays (frozen positions of the last
// rebuild, R1 predicate in fp32), sums in fp64.  A diagnostic evaluated on request, not part of the step.
//   zeta_C(w) = sum_j (m / rho_j) W_wj / (dx^3 sigma0 - dx^3 sum_w' W_ww'),  0 where the open part is <= 1e-3
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double W_f64(double d2, double inv_h, double CW)
{
    const double q = sqrt(d2) * inv_h;
    const double s = fmax(1.0 - 0.5 * q, 0.0);
    const double s2 = s * s;
    return CW * s2 * s2 * (1.0 + 2.0 * q);
}

__global__ void __launch_bounds__(128) k_contact_factor(DevParams P, double inv_h, double CW, double sigma0, double V0, double mass, double rho0,
                                                        const float4* __restrict__ A, const float4* __restrict__ WA,
                                                        const uint32_t* __restrict__ cstart_f, const uint32_t* __restrict__ cstart_w,
                                                        const uint32_t* __restrict__ worig, float* __restrict__ out /* original wall order */)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.n_w) return;
    const float4 pw = WA[s];
    const Stencil st = make_stencil(P, pw);
    const double xw = pw.x, yw = pw.y, zw = pw.z;
    double num = 0.0, solid = 0.0;
#pragma unroll 1
    for (int r = 0; r < SPH_NR; ++r) {
        int nc;
        const int c0 = stencil_row(P, st, r, nc);
        if (nc == 0) continue;
        for (uint32_t j = cstart_f[c0], e = cstart_f[c0 + nc]; j < e; ++j) {
            const float4 pj = __ldg(A + j);
            if (dist2(pw.x - pj.x, pw.y - pj.y, pw.z - pj.z) < P.rc2) {
                const double dx = xw - (double)pj.x, dy = yw - (double)pj.y, dz = zw - (double)pj.z;
                num += mass / (rho0 + (double)pj.w) * W_f64(dx * dx + dy * dy + dz * dz, inv_h, CW);
            }
        }
        for (uint32_t j = cstart_w[c0], e = cstart_w[c0 + nc]; j < e; ++j) {
            const float4 pj = __ldg(WA + j);
            if (dist2(pw.x - pj.x, pw.y - pj.y, pw.z - pj.z) < P.rc2) {       // includes w itself: W(0)
                const double dx = xw - (double)pj.x, dy = yw - (double)pj.y, dz = zw - (double)pj.z;
                solid += W_f64(dx * dx + dy * dy + dz * dz, inv_h, CW);
            }
        }
    }
    const double full = V0 * (sigma0 - solid);
    out[worig[s]] = full > 1.0e-3 * V0 * sigma0 ? (float)(num / full) : 0.0f;
}

// ---------------------------------------------------------------------------------------------
// Evolving solid temperature (Eq. 20; reading R23): one thread per sorted wall particle of a body with
// thermal_mode = 1 walks its candidate windows in the sorted fluid and wall arrays (frozen positions, R1 predicate):
//   m_w c_s dT_w/dt = sum_i V_w (m / rho_i) K_wi (T_w - T_i) F_wi + sum_u V_w V_u K_wu (T_w - T_u) F_wu
// fp32 pair terms as in the sweeps, fp64 accumulation.  Temperatures are those of time n on both sides: it runs
// after sweep B and before the finish kernels.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_wall_heat(DevParams P, const float4* __restrict__ A, const float4* __restrict__ B,
                                                   const float4* __restrict__ WA, const float4* __restrict__ WB,
                                                   const uint32_t* __restrict__ cstart_f, const uint32_t* __restrict__ cstart_w,
                                                   float* __restrict__ wrate /* sorted wall order */)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.n_w) return;
    const float4 pw = WA[s];
    const int b = __float_as_int(pw.w);
    if (P.bmode[b] != 1) { wrate[s] = 0.0f; return; }
    const float th_w = WB[s].w, kw = P.bk[b], Kf = P.body[b].K;
    const Stencil st = make_stencil(P, pw);
    double flux_f = 0.0, flux_s = 0.0;
#pragma unroll 1
    for (int r = 0; r < SPH_NR; ++r) {
        int nc;
        const int c0 = stencil_row(P, st, r, nc);
        if (nc == 0) continue;
        for (uint32_t j = cstart_f[c0], e = cstart_f[c0 + nc]; j < e; ++j) {
            const float4 pj = __ldg(A + j);
            if (dist2(pw.x - pj.x, pw.y - pj.y, pw.z - pj.z) < P.rc2) {
                const PairGeom g = pair_geom(P, pw, pj);
                flux_f += (double)(g.F * (th_w - __ldg(&B[j].w)) / (P.rho0 + pj.w));
            }
        }
        for (uint32_t j = cstart_w[c0], e = cstart_w[c0 + nc]; j < e; ++j) {
            const float4 pj = __ldg(WA + j);
            if ((int)j != s && dist2(pw.x - pj.x, pw.y - pj.y, pw.z - pj.z) < P.rc2) {
                const PairGeom g = pair_geom(P, pw, pj);
                const float ku = P.bk[__float_as_int(pj.w)];
                const float K = (kw + ku) > 0.0f ? 4.0f * kw * ku / (kw + ku) : 0.0f;
                flux_s += (double)(g.F * K * (th_w - __ldg(&WB[j].w)));
            }
        }
    }
    // V_w = dx^3 on every term; fluid: V_i = m / rho_i, K_wi of the body; solid: V_u = dx^3
    const double flux = (double)P.Vw * ((double)P.mass * (double)Kf * flux_f + (double)P.Vw * flux_s);
    wrate[s] = (float)(flux * (double)P.binvC[b]);
}

// T_w += dt dT_w/dt in the sorted records and in the original-order copy a later wall sort starts from
__global__ void __launch_bounds__(256) k_finish_wall(int n, float4* __restrict__ WB, float* __restrict__ wT, const float* __restrict__ wrate,
                                                     const uint32_t* __restrict__ worig, const Clock* clk)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const float r = wrate[s];
    if (r == 0.0f) return;
    const float th = WB[s].w + clk->dt_f * r;
    reinterpret_cast<float*>(WB + s)[3] = th;
    wT[worig[s]] = th;
}

// ---------------------------------------------------------------------------------------------
// read-outs of the configuration (tests): digest and CSR in original ids
// ---------------------------------------------------------------------------------------------
// local list entry -> global sorted index for either tile mode (tests only)
struct Resolver {
    const TileHdr* h;
    RangeTab tf, tw;
    bool staged;
    // `slots` = the tile's header slots; `slot` = the particle's lane slot in the tile
    __device__ __forceinline__ void init(const DevParams& P, const TileHdr* slots, int slot, float4 pi, const uint32_t* cstart_f, const uint32_t* cstart_w)
    {
        const int S = (int)slots[0].S;
        staged = S >= 1;
        h = slots + (S > 1 ? slot / (SPH_TP / S) : 0);
        if (!staged) { own_table(P, pi, cstart_f, true, tf); own_table(P, pi, cstart_w, P.n_w > 0, tw); }
    }
    __device__ __forceinline__ uint32_t fluid(uint32_t L) const { return staged ? resolve_local_n(h->lbase_f, h->gstart_f, (int)h->n_ranges, L) : resolve_local(tf.lb, tf.gs, L, 0); }
    __device__ __forceinline__ uint32_t wall(uint32_t L) const { return staged ? resolve_local_n(h->lbase_w, h->gstart_w, (int)h->n_ranges, L) : resolve_local(tw.lb, tw.gs, L, 0); }
};

__global__ void __launch_bounds__(SPH_TP) k_neigh_digest(DevParams P, const TileHdr* __restrict__ hdr, const float4* __restrict__ A,
                                                          const uint32_t* __restrict__ cstart_f, const uint32_t* __restrict__ cstart_w,
                                                          const uint4* __restrict__ list_f, const uint4* __restrict__ list_w, int KF8, int KW8,
                                                          const uint32_t* __restrict__ ncnt, const uint32_t* __restrict__ orig,
                                                          const uint32_t* __restrict__ worig, uint64_t* __restrict__ out /* original order */)
{
    const int tile = blockIdx.x, tid = threadIdx.x, i = tile * SPH_TP + tid;
    if (i >= P.n_f) return;
    Resolver R;
    R.init(P, hdr + (size_t)tile * SPH_SMAX, tid, A[i], cstart_f, cstart_w);
    const uint4* lf = list_f + (size_t)tile * KF8 * SPH_TP + tid;
    const uint4* lw = list_w + (size_t)tile * KW8 * SPH_TP + tid;
    const uint32_t c = ncnt[i];
    const int nf = c & 0xffffu, nw = c >> 16;
    uint64_t dg = 0;
    for (int k = 0; k < nf; ++k) dg += mix64((uint64_t)orig[R.fluid(list_entry(lf, k))] + 1ull);
    for (int k = 0; k < nw; ++k) dg += mix64((uint64_t)P.n_f + (uint64_t)worig[R.wall(list_entry(lw, k))] + 1ull);
    out[orig[i]] = dg;
}

// which = 0: fluid lists, 1: wall lists.  offs[original i] = start of i's list in `out`.
__global__ void __launch_bounds__(SPH_TP) k_neigh_csr(DevParams P, int which, const TileHdr* __restrict__ hdr, const float4* __restrict__ A,
                                                       const uint32_t* __restrict__ cstart_f, const uint32_t* __restrict__ cstart_w,
                                                       const uint4* __restrict__ list, int K8, const uint32_t* __restrict__ ncnt,
                                                       const uint32_t* __restrict__ orig, const uint32_t* __restrict__ id_of,
                                                       const uint64_t* __restrict__ offs, int32_t* __restrict__ out)
{
    const int tile = blockIdx.x, tid = threadIdx.x, i = tile * SPH_TP + tid;
    if (i >= P.n_f) return;
    Resolver R;
    R.init(P, hdr + (size_t)tile * SPH_SMAX, tid, A[i], cstart_f, cstart_w);
    const uint4* l = list + (size_t)tile * K8 * SPH_TP + tid;
    const uint32_t c = ncnt[i];
    const int m = which ? (int)(c >> 16) : (int)(c & 0xffffu);
    int32_t* dst = out + offs[orig[i]];
    for (int k = 0; k < m; ++k) {                 // insertion sort by original id while copying
        const uint32_t g = which ? R.wall(list_entry(l, k)) : R.fluid(list_entry(l, k));
        const int32_t id = (int32_t)id_of[g];
        int q = k - 1;
        while (q >= 0 && dst[q] > id) { dst[q + 1] = dst[q]; --q; }
        dst[q + 1] = id;
    }
}

// ---------------------------------------------------------------------------------------------
// a5 under SPH_FLAG_FREE_SURFACE_LOCAL (reading R27 of PAPER.md:123-129): k_build_tiles left the re-initialised density
// offset in G.w and fs_region = 2 on the surface particles (sigma_i < theta sigma0).  k_fs_mark: every surface particle
// marks its fluid neighbours (region 1; only bytes that are 0 are written, with the same value by every writer).
// k_fs_apply: Eq. 14 (max form) in the region, Eq. 15 elsewhere.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SPH_TP) k_fs_mark(DevParams P, const TileHdr* __restrict__ hdr, const float4* __restrict__ A,
                                                     const uint32_t* __restrict__ cstart_f, const uint32_t* __restrict__ cstart_w,
                                                     const uint4* __restrict__ list_f, int KF8, const uint32_t* __restrict__ ncnt,
                                                     unsigned char* fs_region, const Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    const int tile = blockIdx.x, tid = threadIdx.x, i = tile * SPH_TP + tid, lane = tid & 31;
    const bool surf = i < P.n_f && fs_region[i] == 2;
    // the few surface particles of a warp are served by the whole warp, one after the other: 32 list entries at a time
    // instead of one (the walk is a chain of dependent global loads: header ranges, then the mark)
    unsigned todo = __ballot_sync(0xffffffffu, surf);
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const int slot = (tid & ~31) + src, is = tile * SPH_TP + slot;
        Resolver R;
        R.init(P, hdr + (size_t)tile * SPH_SMAX, slot, A[is], cstart_f, cstart_w);
        const uint4* lf = list_f + (size_t)tile * KF8 * SPH_TP + slot;
        const int nf = (int)(ncnt[is] & 0xffffu);
        for (int k = lane; k < nf; k += 32) {
            const uint32_t g = R.fluid(list_entry(lf, k));
            if (fs_region[g] == 0) fs_region[g] = 1;
        }
    }
}

__global__ void __launch_bounds__(256) k_fs_apply(int n, float4* __restrict__ A, const float4* __restrict__ G,
                                                   const unsigned char* __restrict__ fs_region, const Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float dn = G[i].w;
    float* d = reinterpret_cast<float*>(A + i) + 3;
    *d = fs_region[i] ? fmaxf(*d, dn) : dn;
}

// ---------------------------------------------------------------------------------------------
// Heat conduction with per-particle materials (sph_set_materials; Eq. 20-22, written for k_i != k_j, and
// the two-material benchmark of section 3.2, Table 3): replaces the dT/dt that sweep B summed for a uniform fluid.
//   dT_i/dt = 1 / (rho_i cp_i) [ sum_j (m_j / rho_j) K_ij (T_i - T_j) F_ij + sum_w V_w K_iw (T_i - T_w) F_iw ],
//   K_ab = 4 k_a k_b / (k_a + k_b)  (0 when either conductivity is 0).
// One thread per sorted fluid particle walks its lists (records gathered from global memory through the tile header);
// mat = {m, k, cp, 0} per particle in ORIGINAL order.  An option for multi-material heat problems, not tuned.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SPH_TP) k_heat_materials(DevParams P, const TileHdr* __restrict__ hdr, const float4* __restrict__ A,
                                                            const float4* __restrict__ B, const float4* __restrict__ WA, const float4* __restrict__ WB,
                                                            const uint32_t* __restrict__ cstart_f, const uint32_t* __restrict__ cstart_w,
                                                            const uint4* __restrict__ list_f, const uint4* __restrict__ list_w, int KF8, int KW8,
                                                            const uint32_t* __restrict__ ncnt, const uint32_t* __restrict__ orig,
                                                            const float4* __restrict__ mat, float2* __restrict__ rates)
{
    const int tile = blockIdx.x, tid = threadIdx.x, i = tile * SPH_TP + tid;
    if (i >= P.n_f) return;
    const float4 ai = A[i];
    Resolver R;
    R.init(P, hdr + (size_t)tile * SPH_SMAX, tid, ai, cstart_f, cstart_w);
    const uint4* lf = list_f + (size_t)tile * KF8 * SPH_TP + tid;
    const uint4* lw = list_w + (size_t)tile * KW8 * SPH_TP + tid;
    const uint32_t c = ncnt[i];
    const int nf = c & 0xffffu, nw = c >> 16;
    const float4 mi = mat[orig[i]];
    const float th_i = B[i].w;
    float s = 0.f;
    for (int k = 0; k < nf; ++k) {
        const uint32_t g = R.fluid(list_entry(lf, k));
        const float4 aj = A[g], mj = mat[orig[g]];
        const PairGeom pg = pair_geom(P, ai, aj);
        const float K = (mi.y + mj.y) > 0.f ? 4.0f * mi.y * mj.y / (mi.y + mj.y) : 0.f;
        s = fmaf(mj.x / (P.rho0 + aj.w) * K, (th_i - B[g].w) * pg.F, s);
    }
    for (int k = 0; k < nw; ++k) {
        const uint32_t g = R.wall(list_entry(lw, k));
        const float4 wa = WA[g];
        const PairGeom pg = pair_geom(P, ai, wa);
        const float kn = P.bk[__float_as_int(wa.w)];
        const float K = (mi.y + kn) > 0.f ? 4.0f * mi.y * kn / (mi.y + kn) : 0.f;
        s = fmaf(P.Vw * K, (th_i - WB[g].w) * pg.F, s);
    }
    rates[i].y = (P.flags & F_THERMAL) ? s / ((P.rho0 + ai.w) * mi.z) : 0.f;
}
