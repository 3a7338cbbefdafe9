// axg_k_diffuse.cu -- P1 of the step (SURVEY.md §8(a) P1a..P1d + P2a; DESIGN.md §3 O1..O3):
//   k_diffuse  Brownian step of every live particle (Philox4x32-10 keyed on (seed, id, t) -> Box-Muller -> fma),
//              absorbing-boundary test, ORDER-PRESERVING compaction (warp ballot/popc ranks, block scan, one
//              decoupled look-back word per tile), cell key, per-pass digit histograms for the radix sort.
//   emit_and_close  newborns of every owned source appended after the survivors, counters, histogram scan: run by
//              the last block of k_diffuse to finish (k_emit = the same after k_rekey, harness path).
//   k_rekey    harness path (AXG_PHASE_BIN without AXG_PHASE_DIFFUSE): copy A -> B and key it.
// Paper: integration kernel + calculateHash, PAPER.md:263 (§3.5); particles "generated ... and die".
#include "axg_dev.cuh"

namespace {

constexpr int DIFF_THREADS = 256;
constexpr int DIFF_ITEMS = 4;   // measured at C3 after the compaction was pipelined: 4 items / 4 blocks per SM 0.264 ms,
                                // 8 / 3 0.280, 4 / 5 0.267, 8 / 4 0.293
constexpr int DIFF_TILE = DIFF_THREADS * DIFF_ITEMS;
constexpr int DIFF_WARPS = DIFF_THREADS / 32;

// What P1 leaves for P2 besides the key: radix mode -- the digit histograms of every pass (shared memory, flushed
// once per block); count mode -- one more particle in cnt[key] (L2 reduction, no return value).
__device__ __forceinline__ void tally(const AxgParams& p, uint32_t (*s_hist)[AXG_RADIX], uint32_t key) {
    if (p.bin_mode == AXG_BIN_COUNT_D) {
        atomicAdd(p.cnt + key + 1u, 1u);  // shifted by one cell (see k_cell_scan); result unused: a fire-and-forget RED
    } else {
#pragma unroll
        for (int q = 0; q < AXG_MAX_PASSES; ++q)
            if (q < p.n_pass) atomicAdd(&s_hist[q][(key >> (8 * q)) & 0xffu], 1u);
    }
}

// O2: newborns (reading A-5: exactly at the source, not moved in their birth step; A-6: after the survivors, in
// (source, j) order), counters, and -- radix mode -- the exclusive scans of the digit histograms that the sort passes
// start from.  Run by ONE block: the last block of k_diffuse to finish, or k_emit (do_emit == 0: harness path after
// k_rekey).  s_hist must hold AXG_MAX_PASSES x AXG_RADIX words; its contents are overwritten.  Brec = the pre-sort
// record buffer of THIS step (the fused kernel writes the other one of the pair).
__device__ void emit_and_close(const AxgParams& p, int do_emit, uint32_t (*s_hist)[AXG_RADIX], float4* Brec) {
    __shared__ uint32_t s_scan[AXG_RADIX / 32];
    AxgDev* dev = p.dev;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const uint32_t n_in = dev->n_live;
    const uint32_t n_surv = do_emit ? (n_in ? dev->n_surv : 0u) : n_in;
    const uint32_t next_id = dev->next_id;
    const bool fits = (unsigned long long)n_surv + p.e_owned <= (unsigned long long)p.capacity;
    __syncthreads();
    for (int i = tid; i < AXG_MAX_PASSES * AXG_RADIX; i += nthr) (&s_hist[0][0])[i] = 0u;
    __syncthreads();
    if (do_emit && fits) {
        for (uint32_t e = tid; e < p.e_owned; e += nthr) {
            // source s with src_emit_prefix[s] <= e < src_emit_prefix[s+1]
            uint32_t lo = 0u, hi = p.n_src;
            while (hi - lo > 1u) {
                const uint32_t mid = (lo + hi) >> 1;
                if (p.src_emit_prefix[mid] <= e) lo = mid; else hi = mid;
            }
            const uint32_t s = lo, j = e - p.src_emit_prefix[s];
            const AxgSourceDev sd = p.src[s];
            const uint32_t o = n_surv + e;
            const uint32_t key = axg_cell_key(p, sd.x, sd.y, sd.z);
            Brec[o] = make_float4(sd.x, sd.y, sd.z, __uint_as_float(next_id + p.src_id_prefix[s] + j));
            p.Bsp[o] = (uint8_t)(sd.species_polarity & 0xffu);
            p.key_pre[o] = key;
            if (p.bin_mode != AXG_BIN_COUNT_D) {
                tally(p, s_hist, key);
            } else if (j == 0u) {  // all newborns of a source share its cell: one reduction per source, not per particle
                atomicAdd(p.cnt + key + 1u, p.src_emit_prefix[s + 1] - p.src_emit_prefix[s]);
            }
        }
    }
    __syncthreads();
    if (p.bin_mode != AXG_BIN_COUNT_D) {
        // total histogram -> exclusive scan per pass; needs >= 256 threads (one digit each)
        for (int q = 0; q < p.n_pass; ++q) {
            const int d = tid, lane = tid & 31, wq = tid >> 5;
            uint32_t c = 0u, inc = 0u;
            if (d < AXG_RADIX) {
                c = dev->hist[q][d] + s_hist[q][d];
                inc = c;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += v;
                }
                if (lane == 31) s_scan[wq] = inc;
            }
            __syncthreads();
            if (d < AXG_RADIX) {
                uint32_t off = 0u;
                for (int w = 0; w < wq; ++w) off += s_scan[w];
                dev->base[q][d] = off + inc - c;
                dev->hist[q][d] = 0u;
            }
            __syncthreads();
        }
    }
    if (tid == 0 && do_emit) {
        dev->pstep += 1u;  // P1 of step t is done: the next k_diffuse draws from (id, t + 1)
        if (!fits) atomicOr(&dev->err, 1u);
        dev->n_live = fits ? n_surv + p.e_owned : n_surv;
        dev->next_id = next_id + p.e_total;
        dev->emitted += fits ? p.e_owned : 0u;
        dev->absorbed += n_in - n_surv;
        dev->particle_steps += n_in;
    }
}

// ---- settle phase of the fused kernel: O4/O5 for the sorted rows [T0, T0 + DIFF_TILE) --------------------------------
// k_place left, for every cell, its members in slot[cell_lo[c] .. cell_lo[c+1]) in the arbitrary order of the atomics.
// The row of sorted position lo + rank is the member with `rank` members of smaller pre-sort index before it (reading
// A-9), exactly as in k_settle; here the row goes to the shared staging area instead of the SoA.  Every thread settles
// the slots j of its own tile; a cell that straddles the tile boundary also has members in slots OUTSIDE the tile
// whose rows fall inside it: the in-tile members of that cell share those slots among themselves (strided), so no
// barrier and no search is needed.
__device__ __forceinline__ void stage_row(uint32_t dst, uint32_t T0, uint32_t Tend, const float4& r, uint32_t v,
                                          float4* s_in_rec, uint32_t* s_in_v) {
    if (dst >= T0 && dst < Tend) {
        s_in_rec[dst - T0] = r;
        s_in_v[dst - T0] = v;
    }
}

__device__ __forceinline__ void settle_outside(const AxgParams& p, const uint32_t* __restrict__ slot, uint32_t e,
                                               uint32_t lo, uint32_t hi, uint32_t T0, uint32_t Tend, float4* s_in_rec,
                                               uint32_t* s_in_v) {
    const uint32_t ve = __ldg(slot + e), idxe = ve & AXG_IDX_MASK;
    uint32_t rank = 0u;
    for (uint32_t q = lo; q < hi; ++q) rank += ((__ldg(slot + q) & AXG_IDX_MASK) < idxe) ? 1u : 0u;
    const uint32_t dst = lo + rank;
    if (dst >= T0 && dst < Tend) stage_row(dst, T0, Tend, __ldg(p.Brec + idxe), ve, s_in_rec, s_in_v);
}

// named barriers of the fused kernel (id 0 = __syncthreads of the whole block)
constexpr int BAR_FULL = 1;     // producers arrive, compute warps wait: the staging area holds the next tile
constexpr int BAR_EMPTY = 2;    // compute warps arrive, producers wait: the staged rows have been taken into registers
constexpr int BAR_COMPUTE = 3;  // the compute warps among themselves
constexpr int BAR_PROD = 4;     // the producer warps among themselves
constexpr int PROD_THREADS = 64;
constexpr int PROD_ROWS = 8;    // rows per producer thread per batch: eight independent chains of dependent loads
constexpr int PROD_BATCH = PROD_THREADS * PROD_ROWS;
constexpr int FUSED_THREADS = DIFF_THREADS + PROD_THREADS;
static_assert(DIFF_TILE % PROD_BATCH == 0, "a tile is a whole number of producer batches");

__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// One batch of the settle phase by the producer warps: slots j0 + i * PROD_THREADS.  All global loads and the rank
// loops come first; the staging area is written only after the compute warps have released it (wait_empty).
__device__ __forceinline__ void settle_batch(const AxgParams& p, uint32_t T0, uint32_t Tend, uint32_t n_in, uint32_t j0,
                                             bool wait_empty, float4* s_in_rec, uint32_t* s_in_v) {
    const uint32_t* __restrict__ slot = p.sidx[p.final_buf ^ 1];
    const uint32_t* __restrict__ cell_lo = p.cell_lo;
    uint32_t v[PROD_ROWS], lo[PROD_ROWS], hi[PROD_ROWS], dst[PROD_ROWS];
    float4 r[PROD_ROWS];
#pragma unroll
    for (int i = 0; i < PROD_ROWS; ++i) v[i] = (j0 + i * PROD_THREADS < n_in) ? __ldg(slot + j0 + i * PROD_THREADS) : 0u;
#pragma unroll
    for (int i = 0; i < PROD_ROWS; ++i)
        r[i] = (j0 + i * PROD_THREADS < n_in) ? __ldg(p.Brec + (v[i] & AXG_IDX_MASK)) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int i = 0; i < PROD_ROWS; ++i) {
        const uint32_t k = axg_cell_key(p, r[i].x, r[i].y, r[i].z);
        lo[i] = __ldg(cell_lo + k);
        hi[i] = __ldg(cell_lo + k + 1u);
    }
#pragma unroll
    for (int i = 0; i < PROD_ROWS; ++i) {
        const uint32_t j = j0 + i * PROD_THREADS;
        const uint32_t idx = v[i] & AXG_IDX_MASK;
        if (hi[i] - lo[i] > AXG_BIG_CELL) {  // crowded cell: its slots are sorted (k_sort_big_cells), row = slot
            dst[i] = j;
        } else {
            uint32_t rank = 0u;
            if (hi[i] - lo[i] > 1u)  // alone in the cell (the common case): nothing to rank against
                for (uint32_t q = lo[i]; q < hi[i]; ++q) rank += ((__ldg(slot + q) & AXG_IDX_MASK) < idx) ? 1u : 0u;
            dst[i] = lo[i] + rank;
        }
    }
    if (wait_empty) bar_sync(BAR_EMPTY, FUSED_THREADS);
#pragma unroll
    for (int i = 0; i < PROD_ROWS; ++i) {
        const uint32_t j = j0 + i * PROD_THREADS;
        if (j >= n_in) continue;
        stage_row(dst[i], T0, Tend, r[i], v[i], s_in_rec, s_in_v);
        if (hi[i] - lo[i] > AXG_BIG_CELL) continue;
        if (lo[i] < T0) {  // my cell starts before the tile: slots [lo, T0) belong to no thread of this block
            const uint32_t mine = min(hi[i], Tend) - T0;  // its members among the tile's slots; I am number j - T0
            for (uint32_t e = lo[i] + (j - T0); e < T0; e += mine)
                settle_outside(p, slot, e, lo[i], hi[i], T0, Tend, s_in_rec, s_in_v);
        }
        if (hi[i] > Tend) {  // my cell ends after the tile: slots [Tend, hi)
            const uint32_t from = max(lo[i], T0), mine = Tend - from;
            for (uint32_t e = Tend + (j - from); e < hi[i]; e += mine)
                settle_outside(p, slot, e, lo[i], hi[i], T0, Tend, s_in_rec, s_in_v);
        }
    }
}

// The producer warps of the fused kernel: draw the block's tiles, settle each into the staging area one tile ahead
// of the compute warps.  The chain of dependent loads (slot -> record -> cell range -> members of the cell) runs while
// the compute warps do the arithmetic of the previous tile; only the final shared-memory stores wait for them.
__device__ void produce_tiles(const AxgParams& p, uint32_t n_in, uint32_t n_tiles, int ptid, float4* s_in_rec,
                              uint32_t* s_in_v, uint32_t* s_pt, uint32_t* s_ptile) {
    for (uint32_t n = 0u;; ++n) {
        if (ptid == 0) s_pt[n & 1u] = atomicAdd(&p.dev->ticket, 1u);
        bar_sync(BAR_PROD, PROD_THREADS);
        const uint32_t tile = s_pt[n & 1u];
        const bool have = tile < n_tiles;
        bool wait_empty = n > 0u;  // the previous tile of this block is still being read
        if (have) {
            const uint32_t T0 = tile * DIFF_TILE, Tend = min(T0 + (uint32_t)DIFF_TILE, n_in);
#pragma unroll 1
            for (int b = 0; b < DIFF_TILE / PROD_BATCH; ++b) {
                settle_batch(p, T0, Tend, n_in, T0 + b * PROD_BATCH + ptid, wait_empty, s_in_rec, s_in_v);
                wait_empty = false;
            }
        } else if (wait_empty) {
            bar_sync(BAR_EMPTY, FUSED_THREADS);
        }
        if (ptid == 0) *s_ptile = tile;  // >= n_tiles: the block is done
        bar_arrive(BAR_FULL, FUSED_THREADS);
        if (!have) break;
    }
}

// FUSED (count binning only, axg_step(n > 1)): the kernel starts from the slot list that k_place left for step t-1
// instead of the sorted SoA -- it first does what k_settle does (rank inside the cell by pre-sort index, O4/O5), stages
// the tile's sorted rows in shared memory, and diffuses them from there.  The sorted SoA of step t-1 never makes the
// round trip through HBM (17 B written + 17 B read per particle).  Warp-specialised: two PRODUCER warps per block run
// the latency-bound settle phase of tile k+1 (produce_tiles) while the eight compute warps do the Philox / Box-Muller
// arithmetic of tile k; they meet at two named barriers (staging full / staging empty).  Without the producers every
// block alternated between waiting for its gather and computing, in lock-step with all the others along the
// compaction chain, and the fused kernel was slower than the two kernels it replaces (0.52 vs 0.42 ms at C3).
template <bool FUSED>
__global__ void __launch_bounds__(FUSED ? FUSED_THREADS : DIFF_THREADS, FUSED ? 3 : 4) k_diffuse(const AxgParams p) {
    // FUSED: staging area of the settle phase (records + sort values of the tile, in sorted order); it doubles as the
    // histogram scratch of emit_and_close.  Not FUSED: the digit histograms.
    constexpr int RAW_BYTES = FUSED ? DIFF_TILE * 20 : AXG_MAX_PASSES * AXG_RADIX * 4;
    static_assert(RAW_BYTES >= AXG_MAX_PASSES * AXG_RADIX * 4, "emit_and_close needs the histogram scratch");
    __shared__ __align__(16) unsigned char s_raw[RAW_BYTES];
    uint32_t (*s_hist)[AXG_RADIX] = reinterpret_cast<uint32_t (*)[AXG_RADIX]>(s_raw);
    float4* s_in_rec = reinterpret_cast<float4*>(s_raw);
    uint32_t* s_in_v = reinterpret_cast<uint32_t*>(s_raw + (FUSED ? DIFF_TILE * 16 : 0));
    __shared__ float4 s_rec[DIFF_TILE];     // the tile's survivors, compacted inside the tile, waiting for their base
    __shared__ uint32_t s_key[DIFF_TILE];
    __shared__ uint8_t s_sp[DIFF_TILE];
    __shared__ uint32_t s_warp[DIFF_WARPS];
    __shared__ uint32_t s_tk[2], s_base;
    __shared__ uint32_t s_pt[2], s_ptile;   // FUSED: the producers' ticket ring, and the tile that is staged

    AxgDev* dev = p.dev;
    const uint32_t n_in = dev->n_live, t = dev->pstep, epoch = dev->epoch;
    const uint32_t n_tiles = (n_in + DIFF_TILE - 1) / DIFF_TILE;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t lt = axg_lanemask_lt();
    const AxgRoundKeys rk = axg_round_keys(p.seed_lo, p.seed_hi);

    if (!FUSED)
        for (int i = tid; i < AXG_MAX_PASSES * AXG_RADIX; i += DIFF_THREADS) (&s_hist[0][0])[i] = 0u;
    if (!FUSED && tid == 0) s_tk[0] = atomicAdd(&dev->ticket, 1u);
    __syncthreads();
    // the compute warps' own barrier: the two producer warps of the fused kernel never take part in it
    auto cbar = [&]() {
        if (FUSED) bar_sync(BAR_COMPUTE, DIFF_THREADS); else __syncthreads();
    };

    // The chained compaction is software-pipelined over the tiles of a block: tile T's survivors are parked in shared
    // memory and its aggregate is published at once, but its look-back -- which has to wait for EVERY tile in flight
    // before it -- is resolved only after the arithmetic of the block's next tile, when those predecessors have long
    // published.  (Resolving it right away cost ~40 polls per tile with all eight warps parked at a barrier.)
    bool pending = false;
    uint32_t ptile = 0u, ptotal = 0u;
    int par = 0;
    const bool producer = FUSED && tid >= DIFF_THREADS;
    if (producer) produce_tiles(p, n_in, n_tiles, tid - DIFF_THREADS, s_in_rec, s_in_v, s_pt, &s_ptile);
    while (!producer) {
        uint32_t tile;
        if (FUSED) {
            bar_sync(BAR_FULL, FUSED_THREADS);  // the producers have staged the block's next tile
            tile = s_ptile;
        } else {
            tile = s_tk[par];
            if (tid == 0) s_tk[par ^ 1] = atomicAdd(&dev->ticket, 1u);  // next trip's tile, drawn a trip ahead
        }
        const bool have = tile < n_tiles;

        float x[DIFF_ITEMS], y[DIFF_ITEMS], z[DIFF_ITEMS];
        uint32_t id[DIFF_ITEMS];
        uint32_t sp_pack[DIFF_ITEMS / 4];
        uint32_t alive = 0u, wtotal = 0u;
        if (have) {
            const uint32_t first = tile * DIFF_TILE + warp * (32 * DIFF_ITEMS) + lane;
#pragma unroll
            for (int k = 0; k < DIFF_ITEMS / 4; ++k) sp_pack[k] = 0u;
            if (FUSED) {
                // ---- load: the staged rows, in sorted order (what k_settle would have written to the SoA) ----------
#pragma unroll
                for (int i = 0; i < DIFF_ITEMS; ++i) {
                    const uint32_t g = first + i * 32;
                    const bool v = g < n_in;
                    const uint32_t q = warp * (32 * DIFF_ITEMS) + i * 32 + lane;
                    const float4 r = v ? s_in_rec[q] : make_float4(-1.0f, -1.0f, -1.0f, 0.0f);
                    const uint32_t sv = v ? s_in_v[q] : 0u;
                    x[i] = r.x; y[i] = r.y; z[i] = r.z;
                    id[i] = __float_as_uint(r.w);
                    sp_pack[i >> 2] |= (sv >> 30) << (8 * (i & 3));
                    if (p.materialize && v) {  // O5 of step t-1, stored as k_settle stores it
                        p.A.x[g] = r.x; p.A.y[g] = r.y; p.A.z[g] = r.z;
                        p.A.id[g] = id[i];
                        p.A.species[g] = (uint8_t)(sv >> 30);
                        p.skey[p.final_buf][g] = axg_cell_key(p, r.x, r.y, r.z);
                        p.sidx[p.final_buf][g] = sv;
                    }
                }
                bar_arrive(BAR_EMPTY, FUSED_THREADS);  // the rows are in registers: the producers may stage the next tile
            } else {
                // ---- load: warp-striped, 128 B per warp request per column ---------------------------------------
#pragma unroll
                for (int i = 0; i < DIFF_ITEMS; ++i) {
                    const uint32_t g = first + i * 32;
                    const bool v = g < n_in;
                    x[i] = v ? __ldg(p.A.x + g) : -1.0f;
                    y[i] = v ? __ldg(p.A.y + g) : -1.0f;
                    z[i] = v ? __ldg(p.A.z + g) : -1.0f;
                    id[i] = v ? __ldg(p.A.id + g) : 0u;
                    const uint32_t s = v ? (uint32_t)__ldg(p.A.species + g) : 0u;
                    sp_pack[i >> 2] |= s << (8 * (i & 3));
                }
            }
            // ---- O1: diffuse; P1b: absorb -----------------------------------------------------------------------
#pragma unroll
            for (int i = 0; i < DIFF_ITEMS; ++i) {
                const bool v = (first + i * 32) < n_in;
                float z0, z1, z2;
                axg_normals3(id[i], t, 0u, rk, z0, z1, z2);
                x[i] = fmaf(p.sigma, z0, x[i]);
                y[i] = fmaf(p.sigma, z1, y[i]);
                z[i] = fmaf(p.sigma, z2, z[i]);
                const bool in = x[i] >= 0.0f && x[i] < p.fnx && y[i] >= 0.0f && y[i] < p.fny && z[i] >= 0.0f &&
                                z[i] < p.fnz;
                alive |= (v && in) ? (1u << i) : 0u;
            }
            // ---- P1d: order-preserving ranks.  Order inside a warp chunk is (item, lane) = memory order. -----------
#pragma unroll
            for (int i = 0; i < DIFF_ITEMS; ++i) wtotal += __popc(__ballot_sync(0xffffffffu, (alive >> i) & 1u));
            if (lane == 0) s_warp[warp] = wtotal;
        }
        cbar();  // barrier A: warp totals
        uint32_t woff = 0u, ttotal = 0u;
        if (have) {
#pragma unroll
            for (int w = 0; w < DIFF_WARPS; ++w) {
                const uint32_t c = s_warp[w];
                woff += (w < warp) ? c : 0u;
                ttotal += c;
            }
            if (tid == 0)  // tile 0 has nothing before it: its aggregate is its inclusive prefix
                axg_st_state(p.tile_state + tile, axg_pack(epoch, tile == 0 ? AXG_FLAG_INCL : AXG_FLAG_AGG, ttotal));
        }
        // ---- the parked tile: look-back (its predecessors had a whole tile's time to publish), then flush ----------
        if (pending) {
            if (warp == 0) {
                uint32_t excl = 0u;
                if (ptile > 0) {
                    excl = axg_lookback(p.tile_state, ptile, epoch, lane);
                    if (lane == 0) axg_st_state(p.tile_state + ptile, axg_pack(epoch, AXG_FLAG_INCL, excl + ptotal));
                }
                if (lane == 0) {
                    s_base = excl;
                    if (ptile == n_tiles - 1) dev->n_surv = excl + ptotal;
                }
            }
            cbar();  // barrier B: base known
            const uint32_t base = s_base;
            for (uint32_t q = tid; q < ptotal; q += DIFF_THREADS) {  // contiguous in global memory: 128-bit records
                (FUSED ? p.Brec_alt : p.Brec)[base + q] = s_rec[q];
                p.key_pre[base + q] = s_key[q];
                p.Bsp[base + q] = s_sp[q];
            }
            cbar();  // barrier C: the parking area is free
        } else {
            cbar();  // first trip: s_warp has been read by everyone before the next trip rewrites it
        }
        if (!have) break;
        // ---- park my survivors at their tile-local slots; key; histograms / cell counts ---------------------------
        uint32_t out = woff;
#pragma unroll
        for (int i = 0; i < DIFF_ITEMS; ++i) {
            const uint32_t a = (alive >> i) & 1u;
            const uint32_t b = __ballot_sync(0xffffffffu, a);
            if (a) {
                const uint32_t o = out + __popc(b & lt);
                const uint32_t key = axg_cell_key(p, x[i], y[i], z[i]);
                s_rec[o] = make_float4(x[i], y[i], z[i], __uint_as_float(id[i]));
                s_sp[o] = (uint8_t)((sp_pack[i >> 2] >> (8 * (i & 3))) & 0xffu);
                s_key[o] = key;
                tally(p, s_hist, key);
            }
            out += __popc(b);
        }
        pending = true;
        ptile = tile;
        ptotal = ttotal;
        par ^= 1;
    }

    __syncthreads();
    if (!FUSED)
        for (int i = tid; i < p.n_pass * AXG_RADIX; i += DIFF_THREADS) {
            const uint32_t c = (&s_hist[0][0])[i];
            if (c) atomicAdd(&dev->hist[0][0] + i, c);
        }
    if (axg_last_block(dev)) {  // every block's survivors, keys and histogram flushes are visible here
        if (tid == 0) {
            dev->ticket = 0u;
            dev->done = 0u;
            dev->epoch = epoch + 1u;
        }
        __threadfence();
        emit_and_close(p, 1, s_hist, FUSED ? p.Brec_alt : p.Brec);  // the buffer this kernel's survivors went to
    }
}

// harness path: B = A, key_pre = key(A), histograms.  No RNG, no compaction.
__global__ void __launch_bounds__(256) k_rekey(const AxgParams p) {
    __shared__ uint32_t s_hist[AXG_MAX_PASSES][AXG_RADIX];
    AxgDev* dev = p.dev;
    const uint32_t n = dev->n_live;
    for (int i = threadIdx.x; i < AXG_MAX_PASSES * AXG_RADIX; i += blockDim.x) (&s_hist[0][0])[i] = 0u;
    __syncthreads();
    for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < n; g += gridDim.x * blockDim.x) {
        const float x = p.A.x[g], y = p.A.y[g], z = p.A.z[g];
        const uint32_t key = axg_cell_key(p, x, y, z);
        p.Brec[g] = make_float4(x, y, z, __uint_as_float(p.A.id[g]));
        p.Bsp[g] = p.A.species[g];
        p.key_pre[g] = key;
        tally(p, s_hist, key);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < p.n_pass * AXG_RADIX; i += blockDim.x) {
        const uint32_t c = (&s_hist[0][0])[i];
        if (c) atomicAdd(&dev->hist[0][0] + i, c);
    }
}

constexpr int EMIT_THREADS = 256;
__global__ void __launch_bounds__(EMIT_THREADS) k_emit(const AxgParams p, int do_emit) {
    __shared__ uint32_t s_hist[AXG_MAX_PASSES][AXG_RADIX];
    emit_and_close(p, do_emit, s_hist, p.Brec);
}

}  // namespace

int axg_diffuse_tile() { return DIFF_TILE; }

void axg_launch_diffuse(const AxgParams& p, int grid, cudaStream_t s) { k_diffuse<false><<<grid, DIFF_THREADS, 0, s>>>(p); }
void axg_launch_settle_diffuse(const AxgParams& p, int grid, cudaStream_t s) {
    k_diffuse<true><<<grid, FUSED_THREADS, 0, s>>>(p);
}
void axg_launch_rekey(const AxgParams& p, int grid, cudaStream_t s) { k_rekey<<<grid, 256, 0, s>>>(p); }
void axg_launch_emit(const AxgParams& p, int do_emit, cudaStream_t s) { k_emit<<<1, EMIT_THREADS, 0, s>>>(p, do_emit); }
