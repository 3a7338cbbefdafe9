// axg_k_sort.cu -- P2b: stable LSD radix sort of (key, pre-sort index), 8- or 9-bit digits, one kernel per digit pass
// (DESIGN.md §3 O4, reading A-9).  The paper sorts (cell hash, particle id) pairs with a
// library radix sort; this is a hand-written single-pass-per-digit ("onesweep"-style) sort:
//   - digit histograms of ALL passes are known before the first pass (accumulated by k_diffuse / k_emit),
//   - inside a tile every warp ranks its keys in memory order by warp ballots + popc (stable),
//   - per-tile per-digit counts chain across tiles by decoupled look-back (one 64-bit word per tile and digit,
//     epoch-tagged so the words never need clearing),
//   - the tile is sorted through shared memory so that global stores run along digit runs.
#include "axg_dev.cuh"

namespace {

constexpr int SORT_THREADS = 512;
constexpr int SORT_ITEMS = 12;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;
// digits of BITS bits: 8 by default; 9 where that saves a pass ("9-bit digits would take C4 to 3 passes":
// 27 = 9 + 9 + 9) -- one more ballot per key in the peer search, 512 instead of 256 counters per warp
constexpr size_t sort_smem(int bits) {
    return (size_t)(2 * SORT_TILE + SORT_WARPS * (1 << bits) + 2 * (1 << bits) + 32) * sizeof(uint32_t);
}

// One bit of the peer search: keep in m the lanes whose digit agrees with mine on `bitmask`.  Four instructions
// (LOP3 -> predicate, VOTE, two predicated LOP3: m & b / m & ~b); the C++ form `m &= bit ? bal : ~bal` compiled to seven.
__device__ __forceinline__ uint32_t peers_step(uint32_t m, uint32_t d, uint32_t bitmask) {
    asm("{\n\t"
        ".reg .pred p;\n\t"
        ".reg .b32 t, b;\n\t"
        "and.b32 t, %1, %2;\n\t"
        "setp.ne.u32 p, t, 0;\n\t"
        "vote.sync.ballot.b32 b, p, 0xffffffff;\n\t"
        "@p and.b32 %0, %0, b;\n\t"
        "@!p lop3.b32 %0, %0, b, 0, 0x30;\n\t"
        "}"
        : "+r"(m)
        : "r"(d), "r"(bitmask));
    return m;
}

template <bool FIRST, int BITS>
__global__ void __launch_bounds__(SORT_THREADS, 2)
k_sort_pass(const AxgParams p, const int pass, const uint32_t* __restrict__ kin, const uint32_t* __restrict__ vin,
            uint32_t* __restrict__ kout, uint32_t* __restrict__ vout) {
    constexpr int RADIX = 1 << BITS;
    constexpr uint32_t DMASK = RADIX - 1;
    static_assert(RADIX <= SORT_THREADS && RADIX <= AXG_RADIX, "one thread per digit");
    extern __shared__ uint32_t smem[];
    uint32_t* s_key = smem;
    uint32_t* s_val = s_key + SORT_TILE;
    uint32_t* s_wh = s_val + SORT_TILE;             // [SORT_WARPS][RADIX] per-warp digit counts -> offsets
    uint32_t* s_dstart = s_wh + SORT_WARPS * RADIX; // [RADIX] first tile-local slot of the digit
    uint32_t* s_gbase = s_dstart + RADIX;           // [RADIX] global slot of tile-local slot 0 of the digit run
    uint32_t* s_misc = s_gbase + RADIX;             // [0] tile ticket, [1..16] warp scan partials, [20..21] tickets

    AxgDev* dev = p.dev;
    const uint32_t n = dev->n_live, epoch = dev->epoch;
    const uint32_t n_tiles = (n + SORT_TILE - 1) / SORT_TILE;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t lt = axg_lanemask_lt();
    const int shift = BITS * pass;
    uint32_t* my_wh = s_wh + warp * RADIX;
    uint32_t* s_tk = s_misc + 20;  // [2] tile tickets, double-buffered: the next ticket is drawn a tile ahead

    uint32_t key[SORT_ITEMS], val[SORT_ITEMS], rank[SORT_ITEMS];
    auto load_tile = [&](uint32_t tile) {
        const uint32_t first = tile * SORT_TILE + warp * (32 * SORT_ITEMS) + lane;
#pragma unroll
        for (int i = 0; i < SORT_ITEMS; ++i) {
            const uint32_t g = first + i * 32;
            const bool ok = tile < n_tiles && g < n;
            key[i] = ok ? __ldg(kin + g) : 0xffffffffu;
            if (FIRST) {  // value = pre-sort index | species << 30 (the species byte rides along to P2c)
                val[i] = ok ? (g | ((uint32_t)__ldg(p.Bsp + g) << 30)) : 0u;
            } else {
                val[i] = ok ? __ldg(vin + g) : 0u;
            }
        }
    };

#pragma unroll
    for (int i = 0; i < RADIX / 32; ++i) my_wh[i * 32 + lane] = 0u;
    if (tid == 0) s_tk[0] = atomicAdd(&dev->ticket, 1u);
    __syncthreads();
    uint32_t tile = s_tk[0];
    int par = 0;
    load_tile(tile);

    while (tile < n_tiles) {
        if (tid == 0) s_tk[par ^ 1] = atomicAdd(&dev->ticket, 1u);  // read by everyone after barrier B
        // ---- lanes with the same digit, by BITS ballots per item (independent across items: no MATCH latency chain)
#pragma unroll
        for (int i = 0; i < SORT_ITEMS; ++i) {
            const uint32_t d = (key[i] >> shift) & DMASK;
            uint32_t m = 0xffffffffu;
#pragma unroll
            for (int b = 0; b < BITS; ++b) m = peers_step(m, d, 1u << b);
            rank[i] = m;
        }
        // ---- rank inside the warp chunk, in memory order (item, lane): per-warp digit counters in shared memory
#pragma unroll
        for (int i = 0; i < SORT_ITEMS; ++i) {
            const uint32_t d = (key[i] >> shift) & DMASK;
            const uint32_t m = rank[i];
            const int leader = __ffs(m) - 1;
            uint32_t old = 0u;
            if (lane == leader) {
                old = my_wh[d];
                my_wh[d] = old + __popc(m);
            }
            __syncwarp();
            old = __shfl_sync(0xffffffffu, old, leader);
            rank[i] = old + __popc(m & lt);
        }
        __syncthreads();  // barrier A
        // ---- per digit: scan over warps, scan over digits, publish the tile aggregate ---------------------------
        uint32_t count = 0u;
        unsigned long long* st = p.sort_state + (size_t)tile * RADIX + tid;
        if (tid < RADIX) {
            const int d = tid;
            uint32_t run = 0u;
#pragma unroll
            for (int w = 0; w < SORT_WARPS; ++w) {
                const uint32_t c = s_wh[w * RADIX + d];
                s_wh[w * RADIX + d] = run;
                run += c;
            }
            count = run;
            axg_st_state(st, axg_pack(epoch, tile == 0 ? AXG_FLAG_INCL : AXG_FLAG_AGG, count));
            uint32_t inc = count;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += v;
            }
            if (lane == 31) s_misc[1 + warp] = inc;
            asm volatile("bar.sync 1, %0;" ::"n"(RADIX));  // the warps that own the digits
            uint32_t off = 0u;
            for (int w = 0; w < warp; ++w) off += s_misc[1 + w];
            s_dstart[d] = off + inc - count;
        }
        __syncthreads();  // barrier B
        // ---- sort the tile through shared memory; the warp's counter row is zeroed for the next tile ------------
#pragma unroll
        for (int i = 0; i < SORT_ITEMS; ++i) {
            const uint32_t d = (key[i] >> shift) & DMASK;
            const uint32_t pos = s_dstart[d] + my_wh[d] + rank[i];
            s_key[pos] = key[i];
            s_val[pos] = val[i];
        }
        __syncwarp();
#pragma unroll
        for (int i = 0; i < RADIX / 32; ++i) my_wh[i * 32 + lane] = 0u;
        // ---- the registers are free: prefetch the next tile while the look-back and the write-out run ----------
        const uint32_t next_tile = s_tk[par ^ 1];
        load_tile(next_tile);
        // ---- decoupled look-back over the predecessor tiles, one thread per digit, 4 predecessors per probe -----
        if (tid < RADIX) {
            const int d = tid;
            uint32_t excl = 0u;
            if (tile > 0) {
                int q = (int)tile - 1;
                const unsigned long long* base = p.sort_state + d;
                const unsigned long long zero_incl = axg_pack(epoch, AXG_FLAG_INCL, 0u);
                while (true) {
                    unsigned long long w[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        w[j] = (q - j >= 0) ? axg_ld_state(base + (size_t)(q - j) * RADIX) : zero_incl;
                    bool done = false;
                    int adv = 0;
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        if (!done && adv == j) {
                            const uint32_t f = axg_flag(w[j], epoch);
                            if (f != 0u) {
                                excl += (uint32_t)w[j];
                                adv = j + 1;
                                done = (f == (uint32_t)AXG_FLAG_INCL);
                            }
                        }
                    }
                    if (done) break;
                    q -= adv;
                }
                axg_st_state(st, axg_pack(epoch, AXG_FLAG_INCL, excl + count));
            }
            s_gbase[d] = dev->base[pass][d] + excl - s_dstart[d];
        }
        __syncthreads();  // barrier C
        const uint32_t tile_n = min((uint32_t)SORT_TILE, n - tile * SORT_TILE);
#pragma unroll
        for (int i = 0; i < SORT_ITEMS; ++i) {
            const uint32_t pos = tid + i * SORT_THREADS;
            if (pos < tile_n) {
                const uint32_t k = s_key[pos];
                const uint32_t g = s_gbase[(k >> shift) & DMASK] + pos;
                kout[g] = k;
                vout[g] = s_val[pos];
            }
        }
        tile = next_tile;
        par ^= 1;
        // no barrier here: the next tile's shared-memory writes (s_wh scan, s_key scatter, s_gbase) all sit behind
        // its barriers A / B, which every thread reaches only after it has finished this write-out
    }
    if (axg_last_block(dev) && tid == 0) {
        dev->ticket = 0u;
        dev->done = 0u;
        dev->epoch = epoch + 1u;
    }
}

}  // namespace

int axg_sort_tile() { return SORT_TILE; }

template <int BITS>
static void launch_sort_pass(const AxgParams& p, int pass, int grid, cudaStream_t s) {
    static bool attr_set = false;
    constexpr size_t SMEM = sort_smem(BITS);
    if (!attr_set) {
        cudaFuncSetAttribute(k_sort_pass<true, BITS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM);
        cudaFuncSetAttribute(k_sort_pass<false, BITS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM);
        attr_set = true;
    }
    if (pass == 0) {
        k_sort_pass<true, BITS><<<grid, SORT_THREADS, SMEM, s>>>(p, 0, p.key_pre, nullptr, p.skey[0], p.sidx[0]);
    } else {
        const int in = (pass - 1) & 1, out = pass & 1;
        k_sort_pass<false, BITS><<<grid, SORT_THREADS, SMEM, s>>>(p, pass, p.skey[in], p.sidx[in], p.skey[out], p.sidx[out]);
    }
}

void axg_launch_sort_pass(const AxgParams& p, int pass, int grid, cudaStream_t s) {
    if (p.digit_bits == 9) launch_sort_pass<9>(p, pass, grid, s);
    else launch_sort_pass<8>(p, pass, grid, s);
}
