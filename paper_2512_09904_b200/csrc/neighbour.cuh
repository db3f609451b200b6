// neighbour.cuh -- cell-linked-list neighbour build (steps a2-a4 of DESIGN.md section 2):
// cell hash, counting sort (histogram, scan, scatter, deterministic intra-cell order),
// structure-of-arrays reorder of fluid and wall particles.  The per-particle neighbour lists that
// the pair sweeps consume until the next rebuild ("neighbor lists and kernel-related quantities are
// updated based on the advection time step") are built per tile in pair.cuh.
#pragma once
#include "common.cuh"

// ---------------------------------------------------------------------------------------------
// a2  cell hash + histogram.  pos.xyz = position; rank = arrival order inside the cell (arbitrary,
// made deterministic by k_cell_sort).  PRED: skip when the control kernel decided "no rebuild".
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_hash_count(DevParams P, const float4* __restrict__ pos, int n,
                                                     uint32_t* __restrict__ cell_id, uint32_t* __restrict__ rank,
                                                     uint32_t* __restrict__ cell_count, Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 p = pos[i];
    unsigned int err = 0;
    int cx = cell_coord(p.x, P.xmin[0], P.inv_ell, P.ng[0], err);
    int cy = cell_coord(p.y, P.xmin[1], P.inv_ell, P.ng[1], err);
    int cz = cell_coord(p.z, P.xmin[2], P.inv_ell, P.ng[2], err);
    (void)cx;                                     // contract cell (error flags); the sort key uses the x sub-cell
    const uint32_t fx = (uint32_t)fine_cell(fine_coord(p.x, P.xmin[0], P.inv_ell4), P.nfx);
    uint32_t c = fx + (uint32_t)P.nfx * ((uint32_t)cy + (uint32_t)P.ng[1] * (uint32_t)cz);
    cell_id[i] = c;
    rank[i] = atomicAdd(&cell_count[c], 1u);
    if (err) atomicOr(&clk->err, err);
}

// ---------------------------------------------------------------------------------------------
// a3  exclusive scan of the histogram -> cell_start[n_cells + 1]; three small kernels.
// ---------------------------------------------------------------------------------------------
#define SCAN_THREADS 256
#define SCAN_ITEMS 8
#define SCAN_CHUNK (SCAN_THREADS * SCAN_ITEMS)

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total)
{
    __shared__ uint32_t warp_sums[SCAN_THREADS / 32];
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) warp_sums[wid] = x;
    __syncthreads();
    if (wid == 0) {
        uint32_t s = lane < SCAN_THREADS / 32 ? warp_sums[lane] : 0u;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += y;
        }
        if (lane < SCAN_THREADS / 32) warp_sums[lane] = s;
    }
    __syncthreads();
    uint32_t base = wid ? warp_sums[wid - 1] : 0u;
    *total = warp_sums[SCAN_THREADS / 32 - 1];
    __syncthreads();
    return base + x - v;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_local(const uint32_t* __restrict__ in, uint32_t* __restrict__ out,
                                                             uint32_t* __restrict__ block_sums, int n, Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    int base = blockIdx.x * SCAN_CHUNK + threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = (base + k < n) ? in[base + k] : 0u; s += v[k]; }
    uint32_t total;
    uint32_t off = block_exclusive_scan(s, &total);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { if (base + k < n) out[base + k] = off; off += v[k]; }
    if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_sums(uint32_t* block_sums, int nb, Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    __shared__ uint32_t carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += SCAN_THREADS) {
        int i = base + threadIdx.x;
        uint32_t v = i < nb ? block_sums[i] : 0u, total;
        uint32_t off = block_exclusive_scan(v, &total);
        uint32_t carry = carry_s;
        if (i < nb) block_sums[i] = carry + off;
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + total;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_add(uint32_t* __restrict__ out, const uint32_t* __restrict__ block_sums,
                                                           int n, uint32_t n_items, Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    int base = blockIdx.x * SCAN_CHUNK + threadIdx.x * SCAN_ITEMS;
    uint32_t add = block_sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k)
        if (base + k < n) out[base + k] += add;
    if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = n_items;       // cell_start[n_cells] = N
}

// scatter: perm[cell_start[c] + rank] = source index
__global__ void __launch_bounds__(256) k_scatter(const uint32_t* __restrict__ cell_id, const uint32_t* __restrict__ rank,
                                                  const uint32_t* __restrict__ cell_start, uint32_t* __restrict__ perm, int n,
                                                  Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    perm[cell_start[cell_id[i]] + rank[i]] = (uint32_t)i;
}

// deterministic intra-cell order: ascending original id (R1).  One thread per cell; cells hold
// ~18 particles, so an insertion sort on (key, src) pairs in registers / local memory is enough.
// key_of == NULL: the key is the source index itself (walls are always sorted from original order).
#define CELL_SORT_LOCAL 24
__global__ void __launch_bounds__(128) k_cell_sort(const uint32_t* __restrict__ cell_start, uint32_t* __restrict__ perm,
                                                    const uint32_t* __restrict__ key_of, int n_cells, Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cells) return;
    uint32_t s = cell_start[c], e = cell_start[c + 1];
    int m = (int)(e - s);
    if (m <= 1) return;
    if (m <= CELL_SORT_LOCAL) {
        uint64_t a[CELL_SORT_LOCAL];
        for (int k = 0; k < m; ++k) {
            uint32_t src = perm[s + k];
            uint32_t key = key_of ? key_of[src] : src;
            uint64_t x = ((uint64_t)key << 32) | src;
            int q = k - 1;
            while (q >= 0 && a[q] > x) { a[q + 1] = a[q]; --q; }
            a[q + 1] = x;
        }
        for (int k = 0; k < m; ++k) perm[s + k] = (uint32_t)a[k];
    } else {                                   // crowded cell (e.g. escaped particles clamped into a border cell): heap sort in
                                               // place in global memory, O(m log m) (keys are distinct: ascending original id)
        auto key = [&](int k) { const uint32_t src = perm[s + k]; return key_of ? key_of[src] : src; };
        auto sift = [&](int root, int end) {
            const uint32_t src = perm[s + root], kr = key_of ? key_of[src] : src;
            for (;;) {
                int child = 2 * root + 1;
                if (child >= end) break;
                uint32_t kc = key(child);
                if (child + 1 < end) { const uint32_t k2 = key(child + 1); if (k2 > kc) { kc = k2; ++child; } }
                if (kc <= kr) break;
                perm[s + root] = perm[s + child];
                root = child;
            }
            perm[s + root] = src;
        };
        for (int k = m / 2 - 1; k >= 0; --k) sift(k, m);
        for (int end = m - 1; end > 0; --end) {
            const uint32_t top = perm[s], last = perm[s + end];
            perm[s + end] = top; perm[s] = last;
            sift(0, end);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// a4  SoA reorder.  Fluid state lives in sorted order between rebuilds:
//   posc = {x, y, z, drho/dt saved}   current (drifting) position + saved continuity rate (R7)
//   A    = {x, y, z, drho}            position FROZEN at this rebuild + density offset rho - rho0
//   B    = {vx, vy, vz, T - T_ref}
//   orig = original (caller) index
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_reorder_fluid(const uint32_t* __restrict__ perm, int n,
                                                        const float4* __restrict__ posc_in, const float4* __restrict__ A_in,
                                                        const float4* __restrict__ B_in, const uint32_t* __restrict__ orig_in,
                                                        float4* __restrict__ posc_out, float4* __restrict__ A_out,
                                                        float4* __restrict__ B_out, uint32_t* __restrict__ orig_out,
                                                        Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    uint32_t src = perm[s];
    float4 p = posc_in[src];
    float drho = A_in[src].w;
    posc_out[s] = p;
    A_out[s] = make_float4(p.x, p.y, p.z, drho);
    B_out[s] = B_in[src];
    orig_out[s] = orig_in[src];
}

// copy-back used when the rebuild decision is taken on the device (buffers cannot be swapped by
// the host): sorted scratch -> primary arrays.
__global__ void __launch_bounds__(256) k_copy_back_fluid(int n, const float4* __restrict__ posc_s, const float4* __restrict__ A_s,
                                                          const float4* __restrict__ B_s, const uint32_t* __restrict__ orig_s,
                                                          float4* __restrict__ posc, float4* __restrict__ A, float4* __restrict__ B,
                                                          uint32_t* __restrict__ orig, Clock* clk)
{
    if (!clk->rebuild) return;
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    posc[s] = posc_s[s]; A[s] = A_s[s]; B[s] = B_s[s]; orig[s] = orig_s[s];
}

// walls: original-order current position / normal -> sorted records
//   WA = {x, y, z, body (int bits)}   WB = {nx, ny, nz, T_w - T_ref}
__global__ void __launch_bounds__(256) k_reorder_wall(const uint32_t* __restrict__ perm, int n,
                                                       const float4* __restrict__ wpos, const float4* __restrict__ wnrm,
                                                       const int* __restrict__ body, const float* __restrict__ Tw,
                                                       float4* __restrict__ WA, float4* __restrict__ WB, Clock* clk, int pred)
{
    if (pred && !clk->rebuild) return;
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    uint32_t src = perm[s];
    float4 p = wpos[src], q = wnrm[src];
    WA[s] = make_float4(p.x, p.y, p.z, __int_as_float(body[src]));
    WB[s] = make_float4(q.x, q.y, q.z, Tw[src]);
}

