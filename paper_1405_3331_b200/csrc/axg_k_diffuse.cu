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
__device__ __forceinline__ void tally(const AxgParams& p, uint32_t (*s_hist)[AXG_RADIX], uint32_t key, uint32_t o,
                                      uint32_t species) {
    if (p.bin_mode == AXG_BIN_COUNT_D) {
        // the old count = this row's arrival rank inside its cell; the species rides in its top two bits (no Bsp column)
        p.kw[o] = make_uint2(key, atomicAdd(p.cnt + key, 1u) | (species << 30));
    } else {
#pragma unroll
        for (int q = 0; q < AXG_MAX_PASSES; ++q)
            if (q < p.n_pass) atomicAdd(&s_hist[q][(key >> (p.digit_bits * q)) & ((1u << p.digit_bits) - 1u)], 1u);
    }
}

// O2: newborns (reading A-5: exactly at the source, not moved in their birth step; A-6: after the survivors, in
// (source, j) order), counters, and -- radix mode -- the exclusive scans of the digit histograms that the sort passes
// start from.  Run by ONE block: the last block of k_diffuse to finish, or k_emit (do_emit == 0: harness path after
// k_rekey).  s_hist must hold AXG_MAX_PASSES x AXG_RADIX words; its contents are overwritten.
__device__ void emit_and_close(const AxgParams& p, int do_emit, uint32_t (*s_hist)[AXG_RADIX]) {
    __shared__ uint32_t s_scan[AXG_RADIX / 32];
    AxgDev* dev = p.dev;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const uint32_t n_in = dev->n_live;
    // volatile: written by other blocks of this kernel; the line may sit in this SM's L1 from the read of n_live
    const uint32_t n_surv = do_emit ? (n_in ? *(volatile uint32_t*)&dev->n_surv : 0u) : n_in;
    const uint32_t next_id = dev->next_id;
    // count binning: B is in the chunked layout, the newborns follow the last chunk (AxgDev::n_phys)
    const bool chunked = p.bin_mode == AXG_BIN_COUNT_D;
    const uint32_t n_phys = chunked ? ((n_in + AXG_CHUNK - 1u) / AXG_CHUNK) * AXG_CHUNK : n_surv;
    const bool fits = (unsigned long long)n_surv + p.e_owned <= (unsigned long long)p.capacity &&
                      (unsigned long long)n_phys + p.e_owned <= (unsigned long long)p.capacity + AXG_CHUNK;
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
            const uint32_t o = n_phys + e;
            const uint32_t key = axg_cell_key(p, sd.x, sd.y, sd.z);
            p.Brec[o] = make_float4(sd.x, sd.y, sd.z, __uint_as_float(next_id + p.src_id_prefix[s] + j));
            if (p.bin_mode != AXG_BIN_COUNT_D) p.Bsp[o] = (uint8_t)(sd.species_polarity & 0xffu);
            if (p.bin_mode != AXG_BIN_COUNT_D) {
                p.key_pre[o] = key;
                tally(p, s_hist, key, o, 0u);
            } else if (j == 0u) {  // all newborns of a source share its cell: one atomic per source, not per particle
                p.src_arr[s] = atomicAdd(p.cnt + key, p.src_emit_prefix[s + 1] - p.src_emit_prefix[s]);
            }
        }
    }
    __syncthreads();
    if (do_emit && fits && p.bin_mode == AXG_BIN_COUNT_D) {  // arrival ranks of the newborns: source base + j
        for (uint32_t e = tid; e < p.e_owned; e += nthr) {
            uint32_t lo = 0u, hi = p.n_src;
            while (hi - lo > 1u) {
                const uint32_t mid = (lo + hi) >> 1;
                if (p.src_emit_prefix[mid] <= e) lo = mid; else hi = mid;
            }
            const AxgSourceDev sd = p.src[lo];
            p.kw[n_phys + e] = make_uint2(axg_cell_key(p, sd.x, sd.y, sd.z),
                                          (p.src_arr[lo] + (e - p.src_emit_prefix[lo])) | ((sd.species_polarity & 0xffu) << 30));
        }
    }
    if (p.bin_mode != AXG_BIN_COUNT_D) {
        // total histogram -> exclusive scan per pass: the block's 256 threads take the digits 256 at a time
        const int n_digits = 1 << p.digit_bits;
        for (int q = 0; q < p.n_pass; ++q) {
            uint32_t carry = 0u;
            for (int d0 = 0; d0 < n_digits; d0 += 256) {
                const int d = d0 + tid, lane = tid & 31, wq = tid >> 5;
                uint32_t c = 0u, inc = 0u;
                if (tid < 256) {
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
                uint32_t off = 0u, total = 0u;
                for (int w = 0; w < 8; ++w) {
                    off += w < wq ? s_scan[w] : 0u;
                    total += s_scan[w];
                }
                if (tid < 256) {
                    dev->base[q][d] = carry + off + inc - c;
                    dev->hist[q][d] = 0u;
                }
                carry += total;
                __syncthreads();
            }
        }
    }
    if (tid == 0 && !do_emit) {  // harness path after k_rekey: B is dense, which is a valid chunked layout too
        dev->n_surv = 0u;
        dev->n_phys = n_phys;
        dev->n_pp = n_phys;
    }
    if (tid == 0 && do_emit) {
        dev->pstep += 1u;  // P1 of step t is done: the next k_diffuse draws from (id, t + 1)
        if (!fits) atomicOr(&dev->err, 1u);
        dev->n_live = fits ? n_surv + p.e_owned : n_surv;
        dev->n_surv = 0u;  // k_diffuse_chunked accumulates into it
        dev->n_phys = n_phys;
        dev->n_pp = n_phys + (do_emit && fits ? p.e_owned : 0u);
        dev->next_id = next_id + p.e_total;
        dev->emitted += fits ? p.e_owned : 0u;
        dev->absorbed += n_in - n_surv;
        dev->particle_steps += n_in;
    }
}

__global__ void __launch_bounds__(DIFF_THREADS, 4) k_diffuse(const AxgParams p) {
    __shared__ uint32_t s_hist[AXG_MAX_PASSES][AXG_RADIX];
    __shared__ float4 s_rec[DIFF_TILE];     // the tile's survivors, compacted inside the tile, waiting for their base
    __shared__ uint32_t s_key[DIFF_TILE];
    __shared__ uint8_t s_sp[DIFF_TILE];
    __shared__ uint32_t s_warp[DIFF_WARPS];
    __shared__ uint32_t s_tk[2], s_base;

    AxgDev* dev = p.dev;
    const uint32_t n_in = dev->n_live, t = dev->pstep, epoch = dev->epoch;
    const uint32_t n_tiles = (n_in + DIFF_TILE - 1) / DIFF_TILE;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t lt = axg_lanemask_lt();
    const AxgRoundKeys rk = axg_round_keys(p.seed_lo, p.seed_hi);

    for (int i = tid; i < AXG_MAX_PASSES * AXG_RADIX; i += DIFF_THREADS) (&s_hist[0][0])[i] = 0u;
    if (tid == 0) s_tk[0] = atomicAdd(&dev->ticket, 1u);
    __syncthreads();

    // The chained compaction is software-pipelined over the tiles of a block: tile T's survivors are parked in shared
    // memory and its aggregate is published at once, but its look-back -- which has to wait for EVERY tile in flight
    // before it -- is resolved only after the arithmetic of the block's next tile, when those predecessors have long
    // published.  (Resolving it right away cost ~40 polls per tile with all eight warps parked at a barrier.)
    bool pending = false;
    uint32_t ptile = 0u, ptotal = 0u;
    int par = 0;
    while (true) {
        const uint32_t tile = s_tk[par];
        const bool have = tile < n_tiles;
        if (tid == 0) s_tk[par ^ 1] = atomicAdd(&dev->ticket, 1u);  // next trip's tile, drawn a trip ahead

        float x[DIFF_ITEMS], y[DIFF_ITEMS], z[DIFF_ITEMS];
        uint32_t id[DIFF_ITEMS];
        uint32_t sp_pack[DIFF_ITEMS / 4];
        uint32_t alive = 0u, wtotal = 0u;
        if (have) {
            // ---- load: warp-striped, 128 B per warp request per column ---------------------------------------
            const uint32_t first = tile * DIFF_TILE + warp * (32 * DIFF_ITEMS) + lane;
#pragma unroll
            for (int k = 0; k < DIFF_ITEMS / 4; ++k) sp_pack[k] = 0u;
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
        __syncthreads();  // barrier A: warp totals
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
            __syncthreads();  // barrier B: base known
            const uint32_t base = s_base;
            for (uint32_t q = tid; q < ptotal; q += DIFF_THREADS) {  // contiguous in global memory: 128-bit records
                p.Brec[base + q] = s_rec[q];
                p.key_pre[base + q] = s_key[q];
                p.Bsp[base + q] = s_sp[q];
            }
            __syncthreads();  // barrier C: the parking area is free
        } else {
            __syncthreads();  // first trip: s_warp has been read by everyone before the next trip rewrites it
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
                tally(p, s_hist, key, 0u, 0u);  // radix binning only: count binning runs k_diffuse_chunked
            }
            out += __popc(b);
        }
        pending = true;
        ptile = tile;
        ptotal = ttotal;
        par ^= 1;
    }

    __syncthreads();
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
        emit_and_close(p, 1, s_hist);
    }
}

// ---- P1 for count binning: compaction inside chunks, no chain ------------------------------------------------------
// The chained kernel above produces a DENSE pre-sort array, which makes every tile wait for the survivor count of every
// tile before it: all blocks march in lock-step, and at C3 a third of the issue slots go to the barriers around the
// look-back and to the burst of stores after it (profiles/).  Count binning never reads the pre-sort array
// sequentially by index -- k_place only needs to visit every row once, k_settle gathers by position -- so here each
// warp compacts its own chunk of 128 rows in place: chunk q's survivors go to B[128 q .. 128 q + chunk_cnt[q]), in
// input order (ballot / popc ranks, reading A-6), straight from registers.  No shared memory, no block barrier, no
// look-back.  The position of a row in this layout orders the rows exactly as the dense index would, so the stable
// order of P2 is unchanged; the dense index itself (the permutation the ABI reports) is chunk_base + offset, computed
// by the export kernels only.
#ifndef AXG_CHUNKED_BLOCKS
#define AXG_CHUNKED_BLOCKS 4
#endif
#ifndef AXG_P1_STAGES
#define AXG_P1_STAGES 0   // chunks in flight per warp (bulk-async staging); 0 = per-lane loads held in registers
#endif
// One stage = the five column runs of one chunk: x, y, z, id (512 B each) and species (128 B).  A chunk column is one
// 16-byte-aligned run of global memory, so each is ONE 1-D bulk copy (cp.async.bulk -> SASS UBLKCP) whose completion
// is counted on the stage's mbarrier: the bytes in flight no longer sit in registers behind the scoreboard, and a warp
// only ever waits for data that was requested two chunks ago.
constexpr int CH_ITEMS = AXG_CHUNK_ITEMS;            // rows per lane and trip; one warp trip = one chunk
constexpr uint32_t CH_COL = AXG_CHUNK * 4u;          // bytes of one 4-byte column of a chunk
constexpr int P1_STAGE_BYTES = 4 * (int)CH_COL + (int)AXG_CHUNK;
constexpr int P1_SMEM = AXG_P1_STAGES > 0 ? DIFF_WARPS * AXG_P1_STAGES * P1_STAGE_BYTES
                                          : (int)(AXG_MAX_PASSES * AXG_RADIX * sizeof(uint32_t));  // scratch of emit_and_close
static_assert(P1_SMEM >= (int)(AXG_MAX_PASSES * AXG_RADIX * sizeof(uint32_t)), "emit_and_close reuses the staging area");

template <bool CS>
__global__ void __launch_bounds__(DIFF_THREADS, AXG_CHUNKED_BLOCKS) k_diffuse_chunked(const AxgParams p) {
    extern __shared__ __align__(128) unsigned char s_raw[];
    __shared__ __align__(8) unsigned long long s_bar[DIFF_WARPS][AXG_P1_STAGES > 0 ? AXG_P1_STAGES : 1];
    __shared__ uint32_t s_surv;
    AxgDev* dev = p.dev;
    const uint32_t n_in = dev->n_live, t = dev->pstep;
    const uint32_t n_chunks = (n_in + AXG_CHUNK - 1u) / AXG_CHUNK;
    const int tid = threadIdx.x, lane = tid & 31;
    const uint32_t lt = axg_lanemask_lt();
    const AxgRoundKeys rk = axg_round_keys(p.seed_lo, p.seed_hi);
    static_assert(32 * CH_ITEMS == AXG_CHUNK, "one warp trip = one chunk");
    if (tid == 0) s_surv = 0u;

    uint32_t mine = 0u;  // survivors of my warp's chunks (lane 0)
    const uint32_t warps_total = (gridDim.x * DIFF_THREADS) >> 5;
    const uint32_t gw = (blockIdx.x * DIFF_THREADS + tid) >> 5;
#if AXG_P1_STAGES > 0
    unsigned char* const my_stage = s_raw + (size_t)(tid >> 5) * AXG_P1_STAGES * P1_STAGE_BYTES;
    const uint32_t my_stage_u32 = axg_smem_u32(my_stage), my_bar_u32 = axg_smem_u32(&s_bar[tid >> 5][0]);
    auto request = [&](uint32_t chunk, int st) {  // lane 0: arm the stage's barrier, then the five bulk copies
        const uint32_t bar = my_bar_u32 + 8u * st, dst = my_stage_u32 + (uint32_t)st * P1_STAGE_BYTES;
        const size_t r0 = (size_t)chunk * AXG_CHUNK;  // the arrays are padded: the last chunk may read past n_in
        axg_mbar_expect_tx(bar, P1_STAGE_BYTES);
        axg_bulk_g2s(dst, p.A.x + r0, CH_COL, bar);
        axg_bulk_g2s(dst + CH_COL, p.A.y + r0, CH_COL, bar);
        axg_bulk_g2s(dst + 2u * CH_COL, p.A.z + r0, CH_COL, bar);
        axg_bulk_g2s(dst + 3u * CH_COL, p.A.id + r0, CH_COL, bar);
        axg_bulk_g2s(dst + 4u * CH_COL, p.A.species + r0, AXG_CHUNK, bar);
    };
    if (lane == 0) {
#pragma unroll
        for (int st = 0; st < AXG_P1_STAGES; ++st) axg_mbar_init(my_bar_u32 + 8u * st, 1u);
        axg_fence_mbar_init();
#pragma unroll
        for (int st = 0; st < AXG_P1_STAGES; ++st)
            if (gw + st * warps_total < n_chunks) request(gw + st * warps_total, st);
    }
    __syncwarp();
    int st = 0;
    uint32_t parity = 0u;
#endif
    __syncthreads();  // s_surv

    for (uint32_t chunk = gw; chunk < n_chunks; chunk += warps_total) {
        const uint32_t first = chunk * AXG_CHUNK + lane;
        float x[CH_ITEMS], y[CH_ITEMS], z[CH_ITEMS];
        uint32_t id[CH_ITEMS], sp[CH_ITEMS];
#if AXG_P1_STAGES > 0
        axg_mbar_wait(my_bar_u32 + 8u * st, parity);
        {
            const unsigned char* sb = my_stage + (size_t)st * P1_STAGE_BYTES;
#pragma unroll
            for (int i = 0; i < CH_ITEMS; ++i) {  // warp-striped rows, as in memory: conflict-free
                const int r = i * 32 + lane;
                x[i] = reinterpret_cast<const float*>(sb)[r];
                y[i] = reinterpret_cast<const float*>(sb + CH_COL)[r];
                z[i] = reinterpret_cast<const float*>(sb + 2 * CH_COL)[r];
                id[i] = reinterpret_cast<const uint32_t*>(sb + 3 * CH_COL)[r];
                sp[i] = sb[4 * CH_COL + r];
            }
        }
#else
#pragma unroll
        for (int i = 0; i < CH_ITEMS; ++i) {
            const uint32_t g = first + i * 32;
            const bool v = g < n_in;
            // volatile asm: all twenty loads of the chunk are ISSUED here, before the arithmetic of its first row (left
            // to itself the compiler sinks each row's loads to their use, behind the previous row's divergent stores,
            // and every row then pays a full memory latency: 42 % of the stall samples)
            x[i] = -1.0f; y[i] = -1.0f; z[i] = -1.0f; id[i] = 0u; sp[i] = 0u;
            if (v) {
                if constexpr (CS) {
                    asm volatile("ld.global.cs.f32 %0, [%1];" : "=f"(x[i]) : "l"(p.A.x + g) : "memory");
                    asm volatile("ld.global.cs.f32 %0, [%1];" : "=f"(y[i]) : "l"(p.A.y + g) : "memory");
                    asm volatile("ld.global.cs.f32 %0, [%1];" : "=f"(z[i]) : "l"(p.A.z + g) : "memory");
                    asm volatile("ld.global.cs.u32 %0, [%1];" : "=r"(id[i]) : "l"(p.A.id + g) : "memory");
                    asm volatile("ld.global.cs.u8 %0, [%1];" : "=r"(sp[i]) : "l"(p.A.species + g) : "memory");
                } else {
                    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(x[i]) : "l"(p.A.x + g) : "memory");
                    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(y[i]) : "l"(p.A.y + g) : "memory");
                    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(z[i]) : "l"(p.A.z + g) : "memory");
                    asm volatile("ld.global.nc.u32 %0, [%1];" : "=r"(id[i]) : "l"(p.A.id + g) : "memory");
                    asm volatile("ld.global.nc.u8 %0, [%1];" : "=r"(sp[i]) : "l"(p.A.species + g) : "memory");
                }
            }
        }
#endif
        // O1 + P1b for the four rows first, as straight-line code (the compiler interleaves the four Philox chains);
        // the divergent part -- ranks and stores -- comes after
        uint32_t alive = 0u;
#pragma unroll
        for (int i = 0; i < CH_ITEMS; ++i) {
            float z0, z1, z2;
            axg_normals3(id[i], t, 0u, rk, z0, z1, z2);
            x[i] = fmaf(p.sigma, z0, x[i]);
            y[i] = fmaf(p.sigma, z1, y[i]);
            z[i] = fmaf(p.sigma, z2, z[i]);
            const bool in = x[i] >= 0.0f && x[i] < p.fnx && y[i] >= 0.0f && y[i] < p.fny && z[i] >= 0.0f && z[i] < p.fnz;
            alive |= ((first + i * 32) < n_in && in) ? (1u << i) : 0u;  // rows past n_in hold padding: never alive
        }
#if AXG_P1_STAGES > 0
        // every lane has its rows in registers (the arithmetic above consumed them): the stage is free for the chunk
        // AXG_P1_STAGES trips ahead
        __syncwarp();
        if (lane == 0 && chunk + AXG_P1_STAGES * warps_total < n_chunks) request(chunk + AXG_P1_STAGES * warps_total, st);
        if (++st == AXG_P1_STAGES) { st = 0; parity ^= 1u; }
#endif
        uint32_t out = chunk * AXG_CHUNK;
        uint32_t dst[CH_ITEMS], arr[CH_ITEMS], key[CH_ITEMS];
#pragma unroll
        for (int i = 0; i < CH_ITEMS; ++i) {  // P1d + P2a
            const bool a = (alive >> i) & 1u;
            const uint32_t b = __ballot_sync(0xffffffffu, a);
            dst[i] = out + __popc(b & lt);
            key[i] = 0u;
            arr[i] = 0u;
            if (a) {
                key[i] = axg_cell_key(p, x[i], y[i], z[i]);
                arr[i] = atomicAdd(p.cnt + key[i], 1u);  // old count = arrival rank inside the cell (see tally)
                axg_st_stream<CS>(p.Brec + dst[i], make_float4(x[i], y[i], z[i], __uint_as_float(id[i])));
            }
            out += __popc(b);
        }
#pragma unroll
        for (int i = 0; i < CH_ITEMS; ++i)  // the four atomics have been in flight together: one wait, not four
            if ((alive >> i) & 1u) axg_st_stream<CS>(p.kw + dst[i], make_uint2(key[i], arr[i] | (sp[i] << 30)));  // species: top two bits
        if (lane == 0) {
            const uint32_t c = out - chunk * AXG_CHUNK;
            p.chunk_cnt[chunk] = c;
            mine += c;
        }
    }
    if (lane == 0 && mine) atomicAdd(&s_surv, mine);
    __syncthreads();
    if (tid == 0 && s_surv) atomicAdd(&dev->n_surv, s_surv);
    if (axg_last_block(dev)) {  // every block's survivors, keys and counts are visible here
        if (tid == 0) dev->done = 0u;
        __threadfence();
        emit_and_close(p, 1, reinterpret_cast<uint32_t(*)[AXG_RADIX]>(s_raw));
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
        // axg_load_particles does not validate positions: a row outside the domain has no cell.  It is flagged (the
        // call reports AXG_EINVAL) and binned into cell 0 so that nothing is written out of bounds.
        const bool in = x >= 0.0f && x < p.fnx && y >= 0.0f && y < p.fny && z >= 0.0f && z < p.fnz;
        if (!in) atomicOr(&dev->err, 4u);
        const uint32_t key = in ? axg_cell_key(p, x, y, z) : 0u;
        p.Brec[g] = make_float4(x, y, z, __uint_as_float(p.A.id[g]));
        const uint32_t sp = p.A.species[g];
        if (p.bin_mode != AXG_BIN_COUNT_D) {
            p.Bsp[g] = (uint8_t)sp;
            p.key_pre[g] = key;
        }
        if (p.bin_mode == AXG_BIN_COUNT_D && (g % AXG_CHUNK) == 0u) p.chunk_cnt[g / AXG_CHUNK] = min(AXG_CHUNK, n - g);
        tally(p, s_hist, key, g, sp);
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
    emit_and_close(p, do_emit, s_hist);
}

}  // namespace

int axg_diffuse_tile() { return DIFF_TILE; }

void axg_launch_diffuse(const AxgParams& p, int grid, cudaStream_t s) {
    if (p.bin_mode == AXG_BIN_COUNT_D) {
        static bool attr_set = false;  // dynamic shared memory above 48 KB needs the opt-in once per process
        if (!attr_set) {
            cudaFuncSetAttribute(k_diffuse_chunked<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, P1_SMEM);
            cudaFuncSetAttribute(k_diffuse_chunked<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, P1_SMEM);
            attr_set = true;
        }
        if (p.cs) k_diffuse_chunked<true><<<148 * AXG_CHUNKED_BLOCKS, DIFF_THREADS, P1_SMEM, s>>>(p);
        else k_diffuse_chunked<false><<<148 * AXG_CHUNKED_BLOCKS, DIFF_THREADS, P1_SMEM, s>>>(p);
    } else {
        k_diffuse<<<grid, DIFF_THREADS, 0, s>>>(p);
    }
}
void axg_launch_rekey(const AxgParams& p, int grid, cudaStream_t s) { k_rekey<<<grid, 256, 0, s>>>(p); }
void axg_launch_emit(const AxgParams& p, int do_emit, cudaStream_t s) { k_emit<<<1, EMIT_THREADS, 0, s>>>(p, do_emit); }
