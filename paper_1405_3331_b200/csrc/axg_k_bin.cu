// axg_k_bin.cu -- P2c reorder + P2d cell ranges (DESIGN.md §3 O5, O6).
// Paper: "position and velocity arrays were also sorted" and identifyCellStart / its reverse
// (PAPER.md:265).  HBM layout chosen here: ONE array cell_lo[cells+1] with
// cell_lo[c] = number of particles whose key is < c, written by "gap filling" from the sorted keys, so that
//   count(c) = cell_lo[c+1] - cell_lo[c]  and a run of consecutive cells is one subtraction,
// and no per-step clear of 2 x cells words is needed.  The paper's cellStart / cellEnd (0 / 0 for an empty cell,
// reading A-10) are produced from it on read by k_cell_export.
#include "axg_dev.cuh"

namespace {

constexpr int BIN_THREADS = 256;
constexpr uint32_t INLINE_GAP = 4;   // gaps up to this many cells are filled by the owning thread

// the whole warp fills cell_lo[lo..hi] = v for every lane that has a long gap (warp-synchronous, no shared memory)
__device__ __forceinline__ void warp_fill(uint32_t* __restrict__ cell_lo, bool mine, uint32_t lo, uint32_t hi,
                                          uint32_t v, int lane) {
    uint32_t bal = __ballot_sync(0xffffffffu, mine);
    while (bal) {
        const int src = __ffs(bal) - 1;
        bal &= bal - 1u;
        const uint32_t lo_ = __shfl_sync(0xffffffffu, lo, src), hi_ = __shfl_sync(0xffffffffu, hi, src),
                       v_ = __shfl_sync(0xffffffffu, v, src);
        for (unsigned long long c = (unsigned long long)lo_ + lane; c <= hi_; c += 32ull) cell_lo[c] = v_;
    }
}

__global__ void __launch_bounds__(BIN_THREADS, 8) k_reorder(const AxgParams p) {
    const AxgDev* dev = p.dev;
    const uint32_t n = dev->n_live;
    const uint32_t* __restrict__ keys = p.skey[p.final_buf];
    const uint32_t* __restrict__ perm = p.sidx[p.final_buf];
    const float4* __restrict__ rec = p.Brec;
    uint32_t* __restrict__ cell_lo = p.cell_lo;
    const int tid = threadIdx.x, lane = tid & 31;

    if (n == 0u) {  // nothing alive: every prefix is 0
        for (uint32_t c = blockIdx.x * BIN_THREADS + tid; c <= p.cells; c += gridDim.x * BIN_THREADS) cell_lo[c] = 0u;
        return;
    }
    // One sorted slot per thread (measured faster than four per thread with 128-bit accesses: the gather is
    // latency-bound and wants warps in flight).  Warp-uniform trip count: j0 is the slot of lane 0.
    for (uint32_t j0 = blockIdx.x * BIN_THREADS + (tid & ~31); j0 < n; j0 += gridDim.x * BIN_THREADS) {
        const uint32_t j = j0 + lane;
        const bool ok = j < n;
        const uint32_t k = ok ? __ldg(keys + j) : 0u;
        const uint32_t v = ok ? __ldg(perm + j) : 0u;
        // O5: A[j] = B[perm[j]] -- one 16 B record gather per particle, species from the top bits of the value
        if (ok) {
            const float4 r = __ldg(rec + (v & AXG_IDX_MASK));
            p.A.x[j] = r.x;
            p.A.y[j] = r.y;
            p.A.z[j] = r.z;
            p.A.id[j] = __float_as_uint(r.w);
            p.A.species[j] = (uint8_t)(v >> 30);
        }
        // O6 as prefix counts: cells (k_prev, k] have exactly j particles below them
        uint32_t kprev = __shfl_up_sync(0xffffffffu, k, 1);
        if (lane == 0) kprev = (j0 > 0u) ? __ldg(keys + j0 - 1u) : 0u;
        const uint32_t lo = (j == 0u) ? 0u : kprev + 1u;
        const bool gap = ok && lo <= k;
        const bool lng = gap && (k - lo >= INLINE_GAP);
        if (gap && !lng)
            for (uint32_t c = lo; c <= k; ++c) cell_lo[c] = j;
        warp_fill(cell_lo, lng, lo, k, j, lane);
        // cells above the last key, and the end sentinel cell_lo[cells] = n
        warp_fill(cell_lo, ok && j == n - 1u, k + 1u, p.cells, n, lane);
    }
}

constexpr int BIN_ITEMS = 4;
// Four consecutive sorted slots per thread, 128-bit loads and stores on every column: the better variant when the
// streams do not fit the L2 (measured: C4 1.33 vs 1.42 ms, C5 4.43 vs 5.26 ms; at C3 the one-slot kernel wins, 0.171 vs
// 0.211 ms).  Same results.
__global__ void __launch_bounds__(BIN_THREADS) k_reorder4(const AxgParams p) {
    const AxgDev* dev = p.dev;
    const uint32_t n = dev->n_live;
    const uint32_t* __restrict__ keys = p.skey[p.final_buf];
    const uint32_t* __restrict__ perm = p.sidx[p.final_buf];
    const float4* __restrict__ rec = p.Brec;
    uint32_t* __restrict__ cell_lo = p.cell_lo;
    const int tid = threadIdx.x, lane = tid & 31;

    if (n == 0u) {  // nothing alive: every prefix is 0
        for (uint32_t c = blockIdx.x * BIN_THREADS + tid; c <= p.cells; c += gridDim.x * BIN_THREADS) cell_lo[c] = 0u;
        return;
    }
    const uint32_t n_groups = (n + BIN_ITEMS - 1) / BIN_ITEMS;
    // warp-uniform trip count: g0 is the group of lane 0
    for (uint32_t g0 = blockIdx.x * BIN_THREADS + (tid & ~31); g0 < n_groups; g0 += gridDim.x * BIN_THREADS) {
        const uint32_t grp = g0 + lane;
        const uint32_t j0 = grp * BIN_ITEMS;
        const bool full = grp < n_groups && j0 + BIN_ITEMS <= n;
        uint32_t k[BIN_ITEMS], v[BIN_ITEMS];
        if (full) {
            const uint4 kk = __ldg(reinterpret_cast<const uint4*>(keys + j0));
            const uint4 vv = __ldg(reinterpret_cast<const uint4*>(perm + j0));
            k[0] = kk.x; k[1] = kk.y; k[2] = kk.z; k[3] = kk.w;
            v[0] = vv.x; v[1] = vv.y; v[2] = vv.z; v[3] = vv.w;
        } else {
#pragma unroll
            for (int i = 0; i < BIN_ITEMS; ++i) {
                const bool ok = grp < n_groups && j0 + i < n;
                k[i] = ok ? __ldg(keys + j0 + i) : 0u;
                v[i] = ok ? __ldg(perm + j0 + i) : 0u;
            }
        }
        // O5: A[j] = B[perm[j]] -- one 16 B record gather per particle, species from the top bits of the value
        float4 r[BIN_ITEMS];
#pragma unroll
        for (int i = 0; i < BIN_ITEMS; ++i)
            r[i] = (grp < n_groups && j0 + i < n) ? __ldg(rec + (v[i] & AXG_IDX_MASK)) : make_float4(0.f, 0.f, 0.f, 0.f);
        if (full) {
            *reinterpret_cast<float4*>(p.A.x + j0) = make_float4(r[0].x, r[1].x, r[2].x, r[3].x);
            *reinterpret_cast<float4*>(p.A.y + j0) = make_float4(r[0].y, r[1].y, r[2].y, r[3].y);
            *reinterpret_cast<float4*>(p.A.z + j0) = make_float4(r[0].z, r[1].z, r[2].z, r[3].z);
            *reinterpret_cast<float4*>(p.A.id + j0) = make_float4(r[0].w, r[1].w, r[2].w, r[3].w);
            *reinterpret_cast<uchar4*>(p.A.species + j0) =
                make_uchar4((unsigned char)(v[0] >> 30), (unsigned char)(v[1] >> 30), (unsigned char)(v[2] >> 30),
                            (unsigned char)(v[3] >> 30));
        } else {
#pragma unroll
            for (int i = 0; i < BIN_ITEMS; ++i)
                if (grp < n_groups && j0 + i < n) {
                    p.A.x[j0 + i] = r[i].x;
                    p.A.y[j0 + i] = r[i].y;
                    p.A.z[j0 + i] = r[i].z;
                    p.A.id[j0 + i] = __float_as_uint(r[i].w);
                    p.A.species[j0 + i] = (uint8_t)(v[i] >> 30);
                }
        }
        // O6 as prefix counts: cells (k_prev, k] have exactly j particles below them
        uint32_t kprev = __shfl_up_sync(0xffffffffu, k[BIN_ITEMS - 1], 1);
        if (lane == 0) kprev = (j0 > 0u && j0 - 1u < n) ? __ldg(keys + j0 - 1u) : 0u;
#pragma unroll
        for (int i = 0; i < BIN_ITEMS; ++i) {
            const uint32_t j = j0 + i;
            const bool ok = grp < n_groups && j < n;
            const uint32_t lo = (j == 0u) ? 0u : kprev + 1u;
            const bool gap = ok && lo <= k[i];
            const bool lng = gap && (k[i] - lo >= INLINE_GAP);
            if (gap && !lng)
                for (uint32_t c = lo; c <= k[i]; ++c) cell_lo[c] = j;
            warp_fill(cell_lo, lng, lo, k[i], j, lane);
            // cells above the last key, and the end sentinel cell_lo[cells] = n
            warp_fill(cell_lo, ok && j == n - 1u, k[i] + 1u, p.cells, n, lane);
            kprev = k[i];
        }
    }
}

// ---- read path of the pre-sort array and the permutation ----------------------------------------------------------
// Radix binning keeps the pre-sort array dense.  Count binning keeps it in the chunked layout of k_diffuse_chunked
// (holes at the end of every 128-row chunk); the ABI's pre-sort index of physical row o is chunk_base[o / 128] + o % 128
// (newborns: survivors + offset), with chunk_base = exclusive scan of chunk_cnt, computed here on demand.
__global__ void __launch_bounds__(1024) k_chunk_scan(const AxgParams p) {
    __shared__ uint32_t s_sum[1024];
    const uint32_t n_chunks = p.dev->n_phys / AXG_CHUNK;
    const uint32_t per = (n_chunks + 1023u) / 1024u;
    const uint32_t lo = min(threadIdx.x * per, n_chunks), hi = min(lo + per, n_chunks);
    uint32_t sum = 0u;
    for (uint32_t q = lo; q < hi; ++q) sum += p.chunk_cnt[q];
    s_sum[threadIdx.x] = sum;
    __syncthreads();
    for (uint32_t d = 1u; d < 1024u; d <<= 1) {  // Hillis-Steele inclusive scan of the 1024 partial sums
        const uint32_t v = threadIdx.x >= d ? s_sum[threadIdx.x - d] : 0u;
        __syncthreads();
        s_sum[threadIdx.x] += v;
        __syncthreads();
    }
    uint32_t run = s_sum[threadIdx.x] - sum;
    for (uint32_t q = lo; q < hi; ++q) {
        p.chunk_base[q] = run;
        run += p.chunk_cnt[q];
    }
}

__device__ __forceinline__ bool axg_is_hole(const AxgParams& p, uint32_t o, uint32_t n_phys) {
    return o < n_phys && (o % AXG_CHUNK) >= p.chunk_cnt[o / AXG_CHUNK];
}
__device__ __forceinline__ uint32_t axg_dense_index(const AxgParams& p, uint32_t o, uint32_t n_phys, uint32_t n_surv) {
    return o >= n_phys ? n_surv + (o - n_phys) : p.chunk_base[o / AXG_CHUNK] + (o % AXG_CHUNK);
}

// one column of the pre-sort array in dense order: component 0..2 = x, y, z (f32 bits), 3 = id, 4 = key (all to
// uint32 dst), 5 = species (to uint8 dst)
__global__ void k_pre_export(const AxgParams p, int component, int chunked, void* __restrict__ dst) {
    const uint32_t n_live = p.dev->n_live;
    const uint32_t n_phys = chunked ? p.dev->n_phys : 0u, n_rows = chunked ? p.dev->n_pp : n_live;
    const uint32_t n_surv = n_live - (n_rows - n_phys);
    const uint32_t* __restrict__ rec = reinterpret_cast<const uint32_t*>(p.Brec);
    for (uint32_t o = blockIdx.x * blockDim.x + threadIdx.x; o < n_rows; o += gridDim.x * blockDim.x) {
        if (chunked && axg_is_hole(p, o, n_phys)) continue;
        const uint32_t i = chunked ? axg_dense_index(p, o, n_phys, n_surv) : o;
        if (component < 4) static_cast<uint32_t*>(dst)[i] = rec[(size_t)o * 4 + component];
        else if (component == 4) static_cast<uint32_t*>(dst)[i] = chunked ? p.kw[o].x : p.key_pre[o];
        else static_cast<uint8_t*>(dst)[i] = chunked ? (uint8_t)(p.kw[o].y >> 30) : p.Bsp[o];
    }
}
// the permutation (sorted slot -> pre-sort index) without the species bits
__global__ void k_perm_export(const AxgParams p, int chunked, uint32_t* __restrict__ dst) {
    const uint32_t n = p.dev->n_live;
    const uint32_t n_phys = p.dev->n_phys, n_surv = n - (p.dev->n_pp - n_phys);
    const uint32_t* __restrict__ src = p.sidx[p.final_buf];
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const uint32_t o = src[i] & AXG_IDX_MASK;
        dst[i] = chunked ? axg_dense_index(p, o, n_phys, n_surv) : o;
    }
}

// cellStart / cellEnd in the paper's convention from cell_lo (read path only)
__global__ void k_cell_export(const AxgParams p, uint32_t* __restrict__ start, uint32_t* __restrict__ end) {
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < p.cells; c += gridDim.x * blockDim.x) {
        const uint32_t a = p.cell_lo[c], b = p.cell_lo[c + 1];
        const bool ne = b > a;
        if (start) start[c] = ne ? a : 0u;
        if (end) end[c] = ne ? b : 0u;
    }
}

}  // namespace

void axg_launch_reorder(const AxgParams& p, int grid, int wide, cudaStream_t s) {
    if (wide) k_reorder4<<<grid, BIN_THREADS, 0, s>>>(p); else k_reorder<<<grid, BIN_THREADS, 0, s>>>(p);
}

void axg_launch_pre_export(const AxgParams& p, int component, int chunked, void* dst, cudaStream_t s) {
    if (chunked) k_chunk_scan<<<1, 1024, 0, s>>>(p);
    k_pre_export<<<148 * 8, 256, 0, s>>>(p, component, chunked, dst);
}
void axg_launch_perm_export(const AxgParams& p, int chunked, uint32_t* dst, cudaStream_t s) {
    if (chunked) k_chunk_scan<<<1, 1024, 0, s>>>(p);
    k_perm_export<<<148 * 8, 256, 0, s>>>(p, chunked, dst);
}

void axg_launch_cell_export(const AxgParams& p, uint32_t* start, uint32_t* end, cudaStream_t s) {
    k_cell_export<<<148 * 8, 256, 0, s>>>(p, start, end);
}
