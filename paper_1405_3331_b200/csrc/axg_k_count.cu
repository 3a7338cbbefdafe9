// axg_k_count.cu -- P2 by cell counts (AXG_BIN_COUNT): the same outputs as the radix path (axg_k_sort.cu +
// k_reorder) -- stable sorted permutation, sorted keys, reordered SoA, cell ranges -- computed as a counting sort
// over the cells themselves (DESIGN.md §3 O4..O6, §6 "binning modes").
//
// Why it exists: on B200 the radix passes are issue-bound, not HBM-bound (profiles/), while the array of per-cell
// counts (4 B x cells: 67 MB at C3) sits in the 126 MB L2.  So P1 counts particles per cell with one L2 atomic each,
// and P2 is
//   k_cell_scan2 cell_lo = exclusive scan of cnt over the cells (block sums, grid barrier, scan; cooperative launch)
//                -> O6 for free; cnt is re-zeroed on the way.  k_cell_scan (single pass, decoupled look-back) is the
//                fallback where a cooperative launch is not available
//   k_place      slot[cell_lo[key] + arrival rank] = pre-sort row (| species << 30): cells are contiguous, the order
//                INSIDE a cell is the arbitrary order in which P1's counting atomics arrived (they return the rank)
//   k_settle     every slot finds its rank among the members of its cell by pre-sort index (the order std::stable_sort
//                gives equal keys, reading A-9), and the record moves to cell_lo + rank: O4 + O5.  Deterministic:
//                nothing of the arrival order survives.
// The paper's scheme sorts (cell hash, id) pairs and then finds cell starts; here the cell starts
// come first and the sort is what is left inside a cell (mean occupancy of a non-empty cell is ~1.6 at C3).
#include "axg_dev.cuh"

namespace {

// ---- exclusive scan of cnt[0 .. cells] --------------------------------------------------------------------------
constexpr int SCAN_THREADS = 512;
constexpr int SCAN_ITEMS = AXG_SCAN_TILE / SCAN_THREADS;  // 16 consecutive cells per thread: 4 x 128-bit
constexpr int SCAN_WARPS = SCAN_THREADS / 32;

__global__ void __launch_bounds__(SCAN_THREADS) k_cell_scan(const AxgParams p) {
    __shared__ uint32_t s_warp[SCAN_WARPS];
    __shared__ uint32_t s_tile, s_base;
    AxgDev* dev = p.dev;
    const uint32_t epoch = dev->epoch;
    const uint32_t n_el = p.cells + 1u;  // cell_lo[cells] = n_live
    const uint32_t n_tiles = (n_el + AXG_SCAN_TILE - 1) / AXG_SCAN_TILE;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (blockIdx.x == 0 && tid == 0) dev->n_big = 0u;  // the list of crowded cells that k_place builds for k_settle

    while (true) {
        __syncthreads();
        if (tid == 0) s_tile = atomicAdd(&dev->ticket, 1u);
        __syncthreads();
        const uint32_t tile = s_tile;
        if (tile >= n_tiles) break;
        // the arrays are padded to a whole tile (zeros in cnt), so the vector accesses never leave them.  Every warp
        // owns 512 consecutive cells; chunk c of a lane is the 4 cells at (32 c + lane) * 4: each load and store
        // instruction of the warp covers 512 contiguous bytes.
        const size_t at4 = ((size_t)tile * AXG_SCAN_TILE + (size_t)warp * (32 * SCAN_ITEMS)) / 4 + lane;
        uint4 v[SCAN_ITEMS / 4];
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS / 4; ++k) v[k] = reinterpret_cast<const uint4*>(p.cnt)[at4 + 32 * k];
        uint32_t pre[SCAN_ITEMS / 4];  // particles before my 4 cells of chunk k, inside the warp's segment
        uint32_t carry = 0u;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS / 4; ++k) {
            const uint32_t mine = v[k].x + v[k].y + v[k].z + v[k].w;
            uint32_t incl = mine;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += u;
            }
            pre[k] = carry + incl - mine;
            carry += __shfl_sync(0xffffffffu, incl, 31);
        }
        const uint32_t inc = carry;  // the warp's total, in every lane
        if (lane == 31) s_warp[warp] = inc;
        __syncthreads();
        uint32_t woff = 0u, ttotal = 0u;
#pragma unroll
        for (int w = 0; w < SCAN_WARPS; ++w) {
            const uint32_t c = s_warp[w];
            woff += (w < warp) ? c : 0u;
            ttotal += c;
        }
        if (warp == 0) {  // decoupled look-back, 32 predecessors per probe
            uint32_t excl = 0u;
            if (tile == 0) {
                if (lane == 0) axg_st_state(p.scan_state + tile, axg_pack(epoch, AXG_FLAG_INCL, ttotal));
            } else {
                if (lane == 0) axg_st_state(p.scan_state + tile, axg_pack(epoch, AXG_FLAG_AGG, ttotal));
                excl = axg_lookback(p.scan_state, tile, epoch, lane);
                if (lane == 0) axg_st_state(p.scan_state + tile, axg_pack(epoch, AXG_FLAG_INCL, excl + ttotal));
            }
            if (lane == 0) s_base = excl;
        }
        __syncthreads();
        // cell_lo[j] = particles below cell j = where cell j starts; cell_lo[cells] = n_live.  cnt is re-zeroed on the way.
        const uint32_t wbase = s_base + woff;
        const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS / 4; ++k) {
            uint32_t run = wbase + pre[k];
            uint4 o;
            o.x = run; run += v[k].x;
            o.y = run; run += v[k].y;
            o.z = run; run += v[k].z;
            o.w = run;
            reinterpret_cast<uint4*>(p.cell_lo)[at4 + 32 * k] = o;
            reinterpret_cast<uint4*>(p.cnt)[at4 + 32 * k] = zero;
        }
    }
    if (axg_last_block(dev) && tid == 0) {
        dev->ticket = 0u;
        dev->done = 0u;
        dev->epoch = epoch + 1u;
    }
}

// ---- the same scan without a chain: reduce, grid barrier, scan ------------------------------------------------------
// In k_cell_scan 59 % of the stall samples sit at the barrier behind the look-back: 1 025 tiles chained through 296
// resident blocks.  Here every block owns a CONTIGUOUS run of tiles: it sums them (phase 1), all blocks meet at a grid
// barrier, every block adds up the sums of the blocks before it and scans its own run (phase 2, cnt re-read from the
// L2).  Needs all blocks co-resident (2 per SM: axg_launch_cell_scan checks the occupancy and falls back otherwise).
constexpr int SCAN2_BLOCKS_PER_SM = 2;

__global__ void __launch_bounds__(SCAN_THREADS, SCAN2_BLOCKS_PER_SM) k_cell_scan2(const AxgParams p) {
    __shared__ uint32_t s_warp[SCAN_WARPS];
    __shared__ uint32_t s_red[SCAN_WARPS];
    __shared__ uint32_t s_bcast;
    AxgDev* dev = p.dev;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t G = gridDim.x, b = blockIdx.x;
    const uint32_t gen = *(volatile uint32_t*)&dev->epoch;  // read before this block arrives at the barrier
    if (b == 0 && tid == 0) dev->n_big = 0u;  // the list of crowded cells that k_place builds for k_settle
    const uint32_t n_el = p.cells + 1u;
    const uint32_t n_tiles = (n_el + AXG_SCAN_TILE - 1) / AXG_SCAN_TILE;
    const uint32_t per = (n_tiles + G - 1u) / G;
    const uint32_t t0 = min(b * per, n_tiles), t1 = min(t0 + per, n_tiles);
    const uint4* __restrict__ cnt4 = reinterpret_cast<const uint4*>(p.cnt);

    // ---- phase 1: sum of my tiles ----
    uint32_t acc = 0u;
    for (uint32_t tile = t0; tile < t1; ++tile) {
        const size_t at4 = (size_t)tile * (AXG_SCAN_TILE / 4) + tid;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS / 4; ++k) {
            const uint4 v = cnt4[at4 + (size_t)SCAN_THREADS * k];
            acc += v.x + v.y + v.z + v.w;
        }
    }
    acc = __reduce_add_sync(0xffffffffu, acc);
    if (lane == 0) s_red[warp] = acc;
    __syncthreads();
    if (tid == 0) {
        uint32_t total = 0u;
        for (int w = 0; w < SCAN_WARPS; ++w) total += s_red[w];
        axg_st_state(p.scan_state + b, (unsigned long long)total);
        __threadfence();
        if (atomicAdd(&dev->ticket, 1u) == G - 1u) {  // last to arrive: open the barrier
            dev->ticket = 0u;
            __threadfence();
            atomicAdd(&dev->epoch, 1u);
        } else {
            while (*(volatile uint32_t*)&dev->epoch == gen) __nanosleep(64);
        }
        __threadfence();
    }
    __syncthreads();

    // ---- phase 2: particles before my first tile, then the scan of my tiles ----
    uint32_t before = 0u;
    for (uint32_t i = tid; i < b; i += SCAN_THREADS) before += (uint32_t)axg_ld_state(p.scan_state + i);
    before = __reduce_add_sync(0xffffffffu, before);
    __syncthreads();
    if (lane == 0) s_red[warp] = before;
    __syncthreads();
    if (tid == 0) {
        uint32_t t = 0u;
        for (int w = 0; w < SCAN_WARPS; ++w) t += s_red[w];
        s_bcast = t;
    }
    __syncthreads();
    uint32_t base = s_bcast;
    for (uint32_t tile = t0; tile < t1; ++tile) {
        const size_t at4 = ((size_t)tile * AXG_SCAN_TILE + (size_t)warp * (32 * SCAN_ITEMS)) / 4 + lane;
        uint4 v[SCAN_ITEMS / 4];
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS / 4; ++k) v[k] = cnt4[at4 + 32 * k];
        uint32_t pre[SCAN_ITEMS / 4];
        uint32_t carry = 0u;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS / 4; ++k) {
            const uint32_t mine = v[k].x + v[k].y + v[k].z + v[k].w;
            uint32_t incl = mine;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += u;
            }
            pre[k] = carry + incl - mine;
            carry += __shfl_sync(0xffffffffu, incl, 31);
        }
        __syncthreads();  // s_warp of the previous tile has been read
        if (lane == 31) s_warp[warp] = carry;
        __syncthreads();
        uint32_t woff = 0u, ttotal = 0u;
#pragma unroll
        for (int w = 0; w < SCAN_WARPS; ++w) {
            const uint32_t c = s_warp[w];
            woff += (w < warp) ? c : 0u;
            ttotal += c;
        }
        const uint32_t wbase = base + woff;
        const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS / 4; ++k) {
            uint32_t run = wbase + pre[k];
            uint4 o;
            o.x = run; run += v[k].x;
            o.y = run; run += v[k].y;
            o.z = run; run += v[k].z;
            o.w = run;
            reinterpret_cast<uint4*>(p.cell_lo)[at4 + 32 * k] = o;
            reinterpret_cast<uint4*>(p.cnt)[at4 + 32 * k] = zero;
        }
        base += ttotal;
    }
}

// ---- slot[cell start + arrival rank] = pre-sort row | species << 30 ---------------------------------------------------------
constexpr int PLACE_THREADS = 256;
// Cells with more members than this are not ranked member by member (a loop over the cell per member: quadratic in the
// occupancy) but as a whole, by one block (settle_big_cell below).  k_place lists them: the row whose arrival rank is
// exactly SETTLE_INLINE exists once in every cell with more than SETTLE_INLINE members.
constexpr uint32_t SETTLE_INLINE = 32u;

template <bool CS>
__global__ void __launch_bounds__(PLACE_THREADS) k_place(const AxgParams p) {
    // B is in the chunked layout of k_diffuse_chunked: every physical row below n_pp is visited, the holes at the end
    // of each chunk are skipped, and the slot value is the PHYSICAL row (it orders the rows like the dense index)
    const uint32_t n_phys = p.dev->n_phys, n_pp = p.dev->n_pp;
    uint32_t* __restrict__ slot = p.sidx[p.final_buf ^ 1];
    const uint32_t* __restrict__ cell_lo = p.cell_lo;
    // one particle per thread: the kernel is bound by L2 transactions (one random 4-byte read of the cell start + one
    // scattered 4-byte store each) and wants many warps in flight.  No atomic: the counting atomic of P1 already
    // returned every row's arrival rank inside its cell (kw.y), in the arbitrary order of the atomics.
    for (uint32_t o = blockIdx.x * PLACE_THREADS + threadIdx.x; o < n_pp; o += gridDim.x * PLACE_THREADS) {
        if (o < n_phys && (o % AXG_CHUNK) >= __ldg(p.chunk_cnt + o / AXG_CHUNK)) continue;  // a hole
        const uint2 w = axg_ld_stream<CS>(p.kw + o);  // key, arrival rank | species << 30: one 8-byte load
        const uint32_t arr = w.y & AXG_IDX_MASK;
        slot[__ldg(cell_lo + w.x) + arr] = o | (w.y & ~AXG_IDX_MASK);
        if (arr == SETTLE_INLINE) p.big_list[atomicAdd(&p.dev->n_big, 1u)] = w.x;  // at most n_live / 33 entries
    }
}

// ---- rank inside the cell by pre-sort index, then O5: A[cell_lo + rank] = B[index] -------------------------------
constexpr int SETTLE_THREADS = 256;
constexpr int SETTLE_ITEMS = 1;  // warp-striped (item i of lane l is slot base + 32 i + l).  Measured at C3: 1 item and
                                 // 8 blocks per SM 0.188 ms, 2 items 0.198, 4 items / 6 blocks 0.227, 8 items 0.272 --
                                 // the kernel lives on many independent warps in flight, not on ILP inside one
#ifndef AXG_SETTLE_SORT_MAX
#define AXG_SETTLE_SORT_MAX 4096
#endif
constexpr uint32_t SETTLE_SORT_MAX = AXG_SETTLE_SORT_MAX;
#ifndef AXG_SETTLE_PREFETCH
#define AXG_SETTLE_PREFETCH 3   // look-ahead of the record prefetch in half grid sweeps (0 = off)
#endif  // members of a cell that one block sorts in shared memory

template <bool WITH_KP>
__device__ __forceinline__ void settle_store(const AxgParams& p, uint32_t dst, const float4& r, uint32_t v, uint32_t k) {
    p.A.x[dst] = r.x;  // (streaming hints measured on these stores and on the slot loads: no gain at C4 / C5)
    p.A.y[dst] = r.y;
    p.A.z[dst] = r.z;
    p.A.id[dst] = __float_as_uint(r.w);
    p.A.species[dst] = (uint8_t)(v >> 30);
    if (WITH_KP) {
        p.skey[p.final_buf][dst] = k;
        p.sidx[p.final_buf][dst] = v;
    }
}

// One block puts ONE crowded cell (more than SETTLE_INLINE members) into pre-sort order.
//  m <= SETTLE_SORT_MAX: the members' slot values are sorted in shared memory (bitonic network: O(m log^2 m)), then
//     gathered in that order.
//  larger: tile by tile -- SETTLE_SORT_MAX members are sorted in shared memory, and EVERY member adds to its rank the
//     number of entries of that tile below it (a binary search in shared memory); after the last tile a member's rank is
//     its position.  O(m^2 / SETTLE_SORT_MAX x log): 2e5 members take a few milliseconds of one block instead of the
//     seconds of the member-by-member loop (D = 0 piles a source's whole emission into one cell: SURVEY.md §8(a) P2b-P2d,
//     reading A-9).  The ranks accumulate in the cell's own range of skey[final_buf ^ 1], which count binning does not use.
// The slot value is rotated left by two first: index in the top 30 bits, species in the low 2 -> integer order = order
// of the pre-sort index.
__device__ __forceinline__ void settle_bitonic(uint32_t* s_sort, uint32_t n2) {
    for (uint32_t size = 2u; size <= n2; size <<= 1)
        for (uint32_t stride = size >> 1; stride > 0u; stride >>= 1) {
            for (uint32_t t = threadIdx.x; t < (n2 >> 1); t += SETTLE_THREADS) {
                const uint32_t i = 2u * t - (t & (stride - 1u)), j = i + stride;
                const uint32_t a = s_sort[i], b = s_sort[j];
                if ((a > b) == ((i & size) == 0u)) { s_sort[i] = b; s_sort[j] = a; }
            }
            __syncthreads();
        }
}

template <bool WITH_KP>
__device__ void settle_big_cell(const AxgParams& p, uint32_t key, uint32_t* s_sort) {
    const uint32_t* __restrict__ slot = p.sidx[p.final_buf ^ 1];
    const uint32_t lo = p.cell_lo[key], hi = p.cell_lo[key + 1u], m = hi - lo;
    const int tid = threadIdx.x;
    if (m <= SETTLE_SORT_MAX) {
        uint32_t n2 = 64u;
        while (n2 < m) n2 <<= 1;
        for (uint32_t i = tid; i < n2; i += SETTLE_THREADS) {
            const uint32_t v = i < m ? slot[lo + i] : 0u;
            s_sort[i] = i < m ? ((v << 2) | (v >> 30)) : 0xffffffffu;
        }
        __syncthreads();
        settle_bitonic(s_sort, n2);
        for (uint32_t i = tid; i < m; i += SETTLE_THREADS) {
            const uint32_t w = s_sort[i], v = (w >> 2) | (w << 30);
            settle_store<WITH_KP>(p, lo + i, p.Brec[v & AXG_IDX_MASK], v, key);
        }
        __syncthreads();
        return;
    }
    uint32_t* __restrict__ rank = p.skey[p.final_buf ^ 1] + lo;
    for (uint32_t i = tid; i < m; i += SETTLE_THREADS) rank[i] = 0u;  // member i is always handled by thread i % 256
    for (uint32_t t0 = 0u; t0 < m; t0 += SETTLE_SORT_MAX) {
        const uint32_t tn = min(SETTLE_SORT_MAX, m - t0);
        for (uint32_t i = tid; i < SETTLE_SORT_MAX; i += SETTLE_THREADS) {
            const uint32_t v = i < tn ? slot[lo + t0 + i] : 0u;
            s_sort[i] = i < tn ? ((v << 2) | (v >> 30)) : 0xffffffffu;
        }
        __syncthreads();
        settle_bitonic(s_sort, SETTLE_SORT_MAX);
        for (uint32_t i = tid; i < m; i += SETTLE_THREADS) {
            const uint32_t v = slot[lo + i], x = (v << 2) | (v >> 30);
            uint32_t a = 0u, b = tn;  // entries of the tile below x
            while (a < b) {
                const uint32_t mid = (a + b) >> 1;
                if (s_sort[mid] < x) a = mid + 1u; else b = mid;
            }
            rank[i] += a;
        }
        __syncthreads();
    }
    for (uint32_t i = tid; i < m; i += SETTLE_THREADS) {
        const uint32_t v = slot[lo + i];
        settle_store<WITH_KP>(p, lo + rank[i], p.Brec[v & AXG_IDX_MASK], v, key);
    }
    __syncthreads();
}

// WITH_KP: also store the sorted keys and the permutation.  Nothing on the path reads them (P1 recomputes the key, P3
// works from cell_lo), so the step runs the lean kernel and axg_read_state(AXG_KEYS_SORTED / AXG_PERM) replays the
// full one on the intact inputs (slot list, records, cell_lo): the same values land in the same places.
template <bool WITH_KP>
__global__ void __launch_bounds__(SETTLE_THREADS, 8) k_settle(const AxgParams p) {
    __shared__ uint32_t s_sort[SETTLE_SORT_MAX];
    const uint32_t n = p.dev->n_live;
    const uint32_t* __restrict__ slot = p.sidx[p.final_buf ^ 1];
    const float4* __restrict__ rec = p.Brec;
    const uint32_t* __restrict__ cell_lo = p.cell_lo;
    const int lane = threadIdx.x & 31;
    const uint32_t warps_total = (gridDim.x * SETTLE_THREADS) >> 5;
    const uint32_t chunk = 32u * SETTLE_ITEMS;
#if AXG_SETTLE_PREFETCH
    // The record gather is the one access of this kernel that misses the L2: a slot's record sits within a few cell
    // planes of the slot's own index in the pre-sort array (a particle moves a few cells per step), and every 32-byte
    // sector of that array is first touched by a random 16-byte read, i.e. at DRAM latency.  So the array is swept into
    // the L2 sequentially, AXG_SETTLE_PREFETCH / 2 grid sweeps ahead of the gathers (one 512-byte bulk prefetch per warp
    // trip), and the gathers hit.
    const uint32_t n_pp = p.dev->n_pp;
    const uint32_t look = (warps_total * chunk / 2u) * AXG_SETTLE_PREFETCH;
#endif
    for (uint32_t base = ((blockIdx.x * SETTLE_THREADS + threadIdx.x) >> 5) * chunk; base < n;
         base += warps_total * chunk) {
        uint32_t v[SETTLE_ITEMS];
        float4 r[SETTLE_ITEMS];
#if AXG_SETTLE_PREFETCH
        if (lane == 0) {
            const uint32_t row = base + look;
            if (row + chunk <= n_pp) axg_prefetch_l2(rec + row, chunk * (uint32_t)sizeof(float4));
            if (base < warps_total * chunk && look > warps_total * chunk)   // first sweep: also what lies before `look`
                for (uint32_t q = base + warps_total * chunk; q < look + base && q + chunk <= n_pp; q += warps_total * chunk)
                    axg_prefetch_l2(rec + q, chunk * (uint32_t)sizeof(float4));
        }
#endif
#pragma unroll
        for (int i = 0; i < SETTLE_ITEMS; ++i) {
            const uint32_t j = base + 32u * i + lane;
            v[i] = (j < n) ? __ldg(slot + j) : 0u;
        }
#pragma unroll
        for (int i = 0; i < SETTLE_ITEMS; ++i) {
            const uint32_t j = base + 32u * i + lane;
            r[i] = (j < n) ? __ldg(rec + (v[i] & AXG_IDX_MASK)) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int i = 0; i < SETTLE_ITEMS; ++i) {
            const uint32_t j = base + 32u * i + lane;
            if (j >= n) continue;
            const uint32_t idx = v[i] & AXG_IDX_MASK;
            const uint32_t k = axg_cell_key(p, r[i].x, r[i].y, r[i].z);
            const uint32_t lo = __ldg(cell_lo + k), hi = __ldg(cell_lo + k + 1u);
            if (hi - lo > SETTLE_INLINE) continue;  // a crowded cell: settle_big_cell below
            uint32_t rank = 0u;  // members of my cell with a smaller pre-sort index (reading A-9: ties keep that order)
            if (hi - lo > 1u)  // alone in the cell (the common case): nothing to rank against
                for (uint32_t q = lo; q < hi; ++q) rank += ((__ldg(slot + q) & AXG_IDX_MASK) < idx) ? 1u : 0u;
            settle_store<WITH_KP>(p, lo + rank, r[i], v[i], k);
        }
    }
    // the crowded cells that k_place listed (a few hundred at C3..C5: the cells next to a source), one block each
    const uint32_t n_big = p.dev->n_big;
    for (uint32_t w = blockIdx.x; w < n_big; w += gridDim.x) settle_big_cell<WITH_KP>(p, p.big_list[w], s_sort);
}

}  // namespace

void axg_launch_cell_scan(const AxgParams& p, int grid, cudaStream_t s) {
    static int resident = -1;  // blocks of k_cell_scan2 that fit one SM
    if (resident < 0 &&
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, k_cell_scan2, SCAN_THREADS, 0) != cudaSuccess) {
        cudaGetLastError();
        resident = 0;
    }
    // (The chained single-pass kernel reads cnt once instead of twice -- 12 instead of 16 B per cell -- but loses also where
    // the scan is DRAM-bound: C4 0.518 vs 0.355 ms, C5 1.03 vs 0.69 ms; the two-phase kernel runs at the copy roofline.)
    if (resident >= SCAN2_BLOCKS_PER_SM) {
        // cooperative launch: the driver schedules all blocks of the grid together or not at all, so the grid barrier
        // cannot deadlock against another context's kernels
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(148 * SCAN2_BLOCKS_PER_SM);
        cfg.blockDim = dim3(SCAN_THREADS);
        cfg.stream = s;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeCooperative;
        attr[0].val.cooperative = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        if (cudaLaunchKernelEx(&cfg, k_cell_scan2, p) == cudaSuccess) return;
        cudaGetLastError();
        resident = 0;  // not supported here: the chained kernel from now on
    }
    k_cell_scan<<<grid, SCAN_THREADS, 0, s>>>(p);
}
void axg_launch_place(const AxgParams& p, int grid, cudaStream_t s) {
    if (p.cs) k_place<true><<<grid, PLACE_THREADS, 0, s>>>(p); else k_place<false><<<grid, PLACE_THREADS, 0, s>>>(p);
}
void axg_launch_settle(const AxgParams& p, int grid, int with_keys_perm, cudaStream_t s) {
    if (with_keys_perm) k_settle<true><<<grid, SETTLE_THREADS, 0, s>>>(p);
    else k_settle<false><<<grid, SETTLE_THREADS, 0, s>>>(p);
}
