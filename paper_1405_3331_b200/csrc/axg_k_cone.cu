// axg_k_cone.cu -- P3 sensing, P4 advance, P5 append (DESIGN.md §3 O7..O10).
// Paper: neighbour-cell loop over the uniform grid, "vector addition" steering and "continue
// on the current direction" when nothing is in range, a predefined distance per step
// (PAPER.md:282), capsule appended at the end of the previous one, growth stops near a target or out of bounds
// (PAPER.md:239), squared-distance test.
#include "axg_dev.cuh"

namespace {

// ---- P3: one warp per cone; lanes take stencil cells; integer sums only (bit-exact) --------------------------
// sense[c][s] = (n_s, Mx_s, My_s, Mz_s), M_s = sum over stencil offsets d of count_s(cell + d) * d   (reading A-12)
#ifndef AXG_SENSE_STAGE
#define AXG_SENSE_STAGE 0
#endif
__global__ void __launch_bounds__(256) k_sense(const AxgParams p) {
#if AXG_SENSE_STAGE
    __shared__ uint32_t s_stage[256][2];
#endif
    const int lane = threadIdx.x & 31;
    const uint32_t warps_total = (gridDim.x * blockDim.x) >> 5;
    const uint32_t* __restrict__ cell_lo = p.cell_lo;
    for (uint32_t c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; c < p.n_cones; c += warps_total) {
        if (p.cone_state[c] != 0) {  // frozen cones skip P3..P5 (reading A-16)
            if (p.sharded && lane < 16) p.sense[(size_t)c * 16 + lane] = 0;
            continue;
        }
        const int ci = (int)p.cone_pos[c * 3 + 0], cj = (int)p.cone_pos[c * 3 + 1], ck = (int)p.cone_pos[c * 3 + 2];
        int acc[AXG_MAX_SPECIES_D][4];
#pragma unroll
        for (int s = 0; s < AXG_MAX_SPECIES_D; ++s)
#pragma unroll
            for (int a = 0; a < 4; ++a) acc[s][a] = 0;
        for (uint32_t e = lane; e < p.n_stencil; e += 32) {
            const int32_t o = __ldg(p.stencil + e);
            const int dx = (int)(int8_t)(o & 0xff), dy = (int)(int8_t)((o >> 8) & 0xff),
                      dz = (int)(int8_t)((o >> 16) & 0xff);
            const int x = ci + dx, y = cj + dy, z = ck + dz;
            if (x < 0 || y < 0 || z < 0 || x >= (int)p.nx || y >= (int)p.ny || z >= (int)p.nz) continue;
            const uint32_t cell = axg_key_of_cell(p, (uint32_t)x, (uint32_t)y, (uint32_t)z);
#if AXG_SENSE_STAGE
            // north_star's form: the cell range staged in shared memory by cp.async (two 4-byte copies: the pair sits at an
            // arbitrary 4-byte alignment), read back after the group has landed.  Measured against the direct loads below
            // (profiles/r02_experiments.md §8): not faster -- the pair is used once, by the lane that asked for it.
            const uint32_t sm = axg_smem_u32(&s_stage[threadIdx.x][0]);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sm), "l"(cell_lo + cell) : "memory");
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sm + 4u), "l"(cell_lo + cell + 1) : "memory");
            asm volatile("cp.async.wait_all;" ::: "memory");
            const uint32_t a = s_stage[threadIdx.x][0], b = s_stage[threadIdx.x][1];
#else
            const uint32_t a = __ldg(cell_lo + cell), b = __ldg(cell_lo + cell + 1);
#endif
            if (p.single_species >= 0) {
                const int cnt = (int)(b - a);
#pragma unroll
                for (int s = 0; s < AXG_MAX_SPECIES_D; ++s)
                    if (s == p.single_species) {
                        acc[s][0] += cnt; acc[s][1] += cnt * dx; acc[s][2] += cnt * dy; acc[s][3] += cnt * dz;
                    }
            } else {
                for (uint32_t j = a; j < b; ++j) {
                    const int sp = (int)__ldg(p.A.species + j);
#pragma unroll
                    for (int s = 0; s < AXG_MAX_SPECIES_D; ++s)
                        if (s == sp) { acc[s][0] += 1; acc[s][1] += dx; acc[s][2] += dy; acc[s][3] += dz; }
                }
            }
        }
        int mine = 0;
        long long G[3] = {0, 0, 0};
#pragma unroll
        for (int s = 0; s < AXG_MAX_SPECIES_D; ++s)
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const int v = __reduce_add_sync(0xffffffffu, acc[s][a]);
                if (lane == s * 4 + a) mine = v;
                if (a > 0) G[a - 1] += (long long)p.polarity[s] * v;
            }
        if (lane < 16) p.sense[(size_t)c * 16 + lane] = mine;
        if (lane < 3) p.cone_gradient[c * 3 + lane] = (float)G[lane] / p.s2;  // g = G / S2(R)
    }
}

// ---- P3, per-particle rule (section 5.3; reading A-26; axg_set_sensing) ------------------
// A particle at x is detected by the cone at q iff |x - q|^2 <= R^2 (fp32, operations and order fixed below); it adds
// rint(256 (x - q)) -- or, weighted, rint(16 w) rint(16 (x - q)) with w = 1 - d^2 / R^2 -- to the first moment of its
// species.  Integer sums: bit-exact, order-free, additive over shards.
// One warp per cone.  The candidates are the particles of the cells that the ball can reach; in the sorted SoA the
// cells x0..x1 of one (y, z) row are ONE contiguous run [cell_lo[key(x0, y, z)], cell_lo[key(x1, y, z) + 1]), so a lane
// takes a row: two cell_lo loads and a short serial walk (~0.6 particles per cell away from the sources).  Rows with
// AXG_PS_BIG or more particles (next to a source) are walked by the whole warp instead, 32 particles per request.
// Rows and x ranges are clipped to the ball with a margin far above the fp32 rounding of the exact test, which alone
// decides: the candidate set only has to be a superset.
#define AXG_PS_BIG 24u

__device__ __forceinline__ void axg_ps_add(const AxgParams& p, int (&acc)[AXG_MAX_SPECIES_D][4], uint32_t j, float qx,
                                           float qy, float qz) {
    const float dx = __fsub_rn(__ldg(p.A.x + j), qx), dy = __fsub_rn(__ldg(p.A.y + j), qy),
                dz = __fsub_rn(__ldg(p.A.z + j), qz);
    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
    if (!(d2 <= p.r2f)) return;
    int mx, my, mz;
    if (p.sense_mode == 1) {
        mx = __float2int_rn(__fmul_rn(dx, 256.0f));
        my = __float2int_rn(__fmul_rn(dy, 256.0f));
        mz = __float2int_rn(__fmul_rn(dz, 256.0f));
    } else {
        const int wq = __float2int_rn(__fmul_rn(__fsub_rn(1.0f, __fdiv_rn(d2, p.r2f)), 16.0f));
        mx = wq * __float2int_rn(__fmul_rn(dx, 16.0f));
        my = wq * __float2int_rn(__fmul_rn(dy, 16.0f));
        mz = wq * __float2int_rn(__fmul_rn(dz, 16.0f));
    }
    const int sp = (p.single_species >= 0) ? p.single_species : (int)__ldg(p.A.species + j);
#pragma unroll
    for (int s = 0; s < AXG_MAX_SPECIES_D; ++s)
        if (s == sp) { acc[s][0] += 1; acc[s][1] += mx; acc[s][2] += my; acc[s][3] += mz; }
}

__global__ void __launch_bounds__(256) k_sense_particles(const AxgParams p) {
    const int lane = threadIdx.x & 31;
    const uint32_t warps_total = (gridDim.x * blockDim.x) >> 5;
    const uint32_t* __restrict__ cell_lo = p.cell_lo;
    const float Rm = p.radius * 1.00001f + 1e-5f;  // margin of the candidate box (not of the test)
    for (uint32_t c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; c < p.n_cones; c += warps_total) {
        if (p.cone_state[c] != 0) {  // frozen cones skip P3..P5 (reading A-16)
            if (p.sharded && lane < 16) p.sense[(size_t)c * 16 + lane] = 0;
            continue;
        }
        const float qx = p.cone_pos[c * 3 + 0], qy = p.cone_pos[c * 3 + 1], qz = p.cone_pos[c * 3 + 2];
        const int y0 = max(0, (int)floorf(qy - Rm)), y1 = min((int)p.ny - 1, (int)floorf(qy + Rm));
        const int z0 = max(0, (int)floorf(qz - Rm)), z1 = min((int)p.nz - 1, (int)floorf(qz + Rm));
        const int ny_rows = y1 - y0 + 1, n_rows = (y1 >= y0 && z1 >= z0) ? ny_rows * (z1 - z0 + 1) : 0;
        int acc[AXG_MAX_SPECIES_D][4];
#pragma unroll
        for (int s = 0; s < AXG_MAX_SPECIES_D; ++s)
#pragma unroll
            for (int a = 0; a < 4; ++a) acc[s][a] = 0;
        // bricked cell order: the x range of a row crosses at most max_seg bricks, one contiguous run in each (Z-order:
        // runs of two cells -- x bit 0 is key bit 0)
        const int seg_shift = p.key_order == 1 ? 3 : 1;
        const int max_seg = p.key_order ? ((2 * (int)ceilf(Rm) + (1 << seg_shift)) >> seg_shift) + 1 : 1;
        for (int r0 = 0; r0 < n_rows; r0 += 32)
        for (int seg = 0; seg < max_seg; ++seg) {
            const int r = r0 + lane;
            uint32_t a = 0, b = 0;
            if (r < n_rows) {
                const int y = y0 + r % ny_rows, z = z0 + r / ny_rows;
                // squared distance from the cone to the slab of cells (y, z), then the half width left along x
                const float ey = fmaxf(fmaxf((float)y - qy, qy - (float)(y + 1)), 0.0f);
                const float ez = fmaxf(fmaxf((float)z - qz, qz - (float)(z + 1)), 0.0f);
                const float left = Rm * Rm - (ey * ey + ez * ez);
                if (left >= 0.0f) {
                    const float hw = sqrtf(left) * 1.00001f + 1e-5f;
                    int x0 = max(0, (int)floorf(qx - hw)), x1 = min((int)p.nx - 1, (int)floorf(qx + hw));
                    if (p.key_order) {  // the seg-th brick (run) of the range
                        const int bx = (x0 >> seg_shift) + seg;
                        x0 = max(x0, bx << seg_shift);
                        x1 = min(x1, (bx << seg_shift) + (1 << seg_shift) - 1);
                    }
                    if (x1 >= x0) {
                        a = __ldg(cell_lo + axg_key_of_cell(p, (uint32_t)x0, (uint32_t)y, (uint32_t)z));
                        b = __ldg(cell_lo + axg_key_of_cell(p, (uint32_t)x1, (uint32_t)y, (uint32_t)z) + 1u);
                    }
                }
            }
            const bool big = (b - a) >= AXG_PS_BIG;
            uint32_t bigs = __ballot_sync(0xffffffffu, big);
            while (bigs) {  // crowded rows: the whole warp, coalesced
                const int src = __ffs(bigs) - 1;
                bigs &= bigs - 1;
                const uint32_t ra = __shfl_sync(0xffffffffu, a, src), rb = __shfl_sync(0xffffffffu, b, src);
                for (uint32_t j = ra + lane; j < rb; j += 32) axg_ps_add(p, acc, j, qx, qy, qz);
            }
            if (!big)
                for (uint32_t j = a; j < b; ++j) axg_ps_add(p, acc, j, qx, qy, qz);
        }
        int mine = 0;
        long long G[3] = {0, 0, 0};
#pragma unroll
        for (int s = 0; s < AXG_MAX_SPECIES_D; ++s)
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const int v = __reduce_add_sync(0xffffffffu, acc[s][a]);
                if (lane == s * 4 + a) mine = v;
                if (a > 0) G[a - 1] += (long long)p.polarity[s] * v;
            }
        if (lane < 16) p.sense[(size_t)c * 16 + lane] = mine;
        if (lane < 3) p.cone_gradient[c * 3 + lane] = (float)G[lane] / p.s2;
    }
}

// ---- P4 + P5: one thread per cone ------------------------------------------------------------------------------
// Every fp32 operation that the specification fixes is written with the explicit round-to-nearest intrinsics so
// that nvcc cannot contract it into an fma (reading A-22); only the normals may differ by an ulp.
// commit != 0: the last block to finish also does O10 (t += 1), which saves the one-thread k_commit launch
__global__ void __launch_bounds__(128) k_advance(const AxgParams p, int commit) {
    AxgDev* dev = p.dev;
    const uint32_t t = dev->step;
    const AxgRoundKeys rk = axg_round_keys(p.seed_lo, p.seed_hi);
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < p.n_cones; c += gridDim.x * blockDim.x) {
        if (p.cone_state[c] != 0) continue;
        long long G[3] = {0, 0, 0}, n_all = 0;
#pragma unroll
        for (int s = 0; s < AXG_MAX_SPECIES_D; ++s) {
            const int4 v = *reinterpret_cast<const int4*>(p.sense + (size_t)c * 16 + s * 4);
            n_all += v.x;
            G[0] += (long long)p.polarity[s] * v.y;
            G[1] += (long long)p.polarity[s] * v.z;
            G[2] += (long long)p.polarity[s] * v.w;
        }
        float h[3] = {p.cone_heading[c * 3 + 0], p.cone_heading[c * 3 + 1], p.cone_heading[c * 3 + 2]};
        float q[3] = {p.cone_pos[c * 3 + 0], p.cone_pos[c * 3 + 1], p.cone_pos[c * 3 + 2]};
        float g[3];
        const float gx = (float)G[0], gy = (float)G[1], gz = (float)G[2];
        p.cone_gradient[c * 3 + 0] = __fdiv_rn(gx, p.s2);  // rewritten here: with sharding the sums were
        p.cone_gradient[c * 3 + 1] = __fdiv_rn(gy, p.s2);  // all-reduced after k_sense
        p.cone_gradient[c * 3 + 2] = __fdiv_rn(gz, p.s2);
        if (G[0] == 0 && G[1] == 0 && G[2] == 0) {  // reading A-14: keep the current direction
            g[0] = h[0]; g[1] = h[1]; g[2] = h[2];
        } else {
            const float len = __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(gx, gx), __fmul_rn(gy, gy)), __fmul_rn(gz, gz)));
            g[0] = __fdiv_rn(gx, len); g[1] = __fdiv_rn(gy, len); g[2] = __fdiv_rn(gz, len);
        }
        float xi[3];
        axg_normals3(c, t, 1u, rk, xi[0], xi[1], xi[2]);  // stream 1 = cone noise (A-2)
        if (p.steer_mode == 1) {
            // the paper's first steering rule (Eq. 5; reading A-25): fixed turn towards / away from the
            // gradient direction by the sign of a draw from N(SNR, 1).  Same operations, in the same order, as the oracle.
            const float dot = __fadd_rn(__fadd_rn(__fmul_rn(h[0], g[0]), __fmul_rn(h[1], g[1])), __fmul_rn(h[2], g[2]));
            float w[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) w[a] = __fsub_rn(g[a], __fmul_rn(dot, h[a]));
            const float sinphi =
                __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(w[0], w[0]), __fmul_rn(w[1], w[1])), __fmul_rn(w[2], w[2])));
            const bool have_g = !(G[0] == 0 && G[1] == 0 && G[2] == 0);
            if (have_g && n_all > 0 && sinphi > 0.0f) {
                const float glen = __fdiv_rn(
                    __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(gx, gx), __fmul_rn(gy, gy)), __fmul_rn(gz, gz))), p.s2);
                const float gamma = __fdiv_rn((float)n_all, (float)p.n_stencil);
                const float mu = __fdiv_rn(glen, gamma);
                const float one = __fadd_rn(1.0f, gamma);
                const float root = __fsqrt_rn(__fdiv_rn(gamma, __fmul_rn(__fmul_rn(one, one), one)));
                const float snr = __fmul_rn(__fmul_rn(__fmul_rn(p.snr_gain, mu), root), sinphi);
                const float sgn = (__fadd_rn(snr, xi[0]) > 0.0f) ? 1.0f : -1.0f;
                const float st = __fmul_rn(sgn, p.sin_turn);
                float v[3];
#pragma unroll
                for (int a = 0; a < 3; ++a)
                    v[a] = __fadd_rn(__fmul_rn(p.cos_turn, h[a]), __fmul_rn(st, __fdiv_rn(w[a], sinphi)));
                const float vlen =
                    __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(v[0], v[0]), __fmul_rn(v[1], v[1])), __fmul_rn(v[2], v[2])));
#pragma unroll
                for (int a = 0; a < 3; ++a) h[a] = __fdiv_rn(v[a], vlen);
            }
        } else {
            float v[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) v[a] = __fadd_rn(g[a], __fmul_rn(p.noise, xi[a]));  // reading A-15
            const float vlen =
                __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(v[0], v[0]), __fmul_rn(v[1], v[1])), __fmul_rn(v[2], v[2])));
#pragma unroll
            for (int a = 0; a < 3; ++a) h[a] = (vlen > 0.0f) ? __fdiv_rn(v[a], vlen) : g[a];
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) q[a] = __fadd_rn(q[a], __fmul_rn(p.speed, h[a]));
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            p.cone_heading[c * 3 + a] = h[a];
            p.cone_pos[c * 3 + a] = q[a];
        }
        // O9 append: step-major planes so that one step's appends of neighbouring cones coalesce
        const uint32_t len = p.poly_len[c];
        if (len <= p.max_segments) {
#pragma unroll
            for (int a = 0; a < 3; ++a) p.poly[((size_t)len * 3 + a) * p.n_cones + c] = q[a];
            p.poly_len[c] = len + 1u;
        } else {
            atomicOr(&dev->err, 2u);
        }
        uint8_t state = 0;
        if (!(q[0] >= 0.0f && q[0] < p.fnx && q[1] >= 0.0f && q[1] < p.fny && q[2] >= 0.0f && q[2] < p.fnz)) {
            state = 2;  // exited
        } else {
            for (uint32_t s = 0; s < p.n_src; ++s) {  // reading A-16: targets = attractive sources, r_cap = 1
                const AxgSourceDev sd = p.src[s];
                if (!(sd.species_polarity & 0x100u)) continue;
                const float dx = __fsub_rn(q[0], sd.x), dy = __fsub_rn(q[1], sd.y), dz = __fsub_rn(q[2], sd.z);
                const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
                if (d2 <= 1.0f) { state = 1; break; }
            }
        }
        if (state) p.cone_state[c] = state;
    }
    if (commit && axg_last_block(&dev->done2) && threadIdx.x == 0) {  // every block has read dev->step by now
        dev->done2 = 0u;
        dev->step = t + 1u;  // NOT pstep: the next step's P1 may already have bumped it (see AxgDev::pstep)
    }
}

// O10; bump == 0: only re-align P1's step index with the committed one (phase calls that commit without a P1)
__global__ void k_commit(const AxgParams p, int bump) {
    p.dev->step += (uint32_t)bump;
    p.dev->pstep = p.dev->step;
}

__global__ void k_census(const AxgParams p) {
    __shared__ uint32_t s_c[4];
    if (threadIdx.x < 4) s_c[threadIdx.x] = 0u;
    __syncthreads();
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < p.n_cones; c += gridDim.x * blockDim.x) {
        const uint32_t st = p.cone_state[c];
        if (st < 3u) atomicAdd(&s_c[st], 1u);
        if (st == 3u) atomicAdd(&p.dev->n_connected, 1u);  // connection formation only: rare
        if (st == 0u) atomicMax(&s_c[3], p.poly_len[c]);  // longest ACTIVE polyline (capacity pre-check)
    }
    __syncthreads();
    if (threadIdx.x < 3 && s_c[threadIdx.x]) atomicAdd(&p.dev->cone_census[threadIdx.x], s_c[threadIdx.x]);
    if (threadIdx.x == 3) atomicMax(&p.dev->cone_census[3], s_c[3]);
}

// widen the int32 sensing sums to the ABI's int64 layouts
__global__ void k_sense_export(const AxgParams p, long long* counts, long long* moment) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < p.n_cones * 4u; i += gridDim.x * blockDim.x) {
        const int4 v = *reinterpret_cast<const int4*>(p.sense + (size_t)i * 4);
        if (counts) counts[i] = v.x;
        if (moment) { moment[(size_t)i * 3 + 0] = v.y; moment[(size_t)i * 3 + 1] = v.z; moment[(size_t)i * 3 + 2] = v.w; }
    }
}

// step-major planes -> neuron-major AoS [C][max_segments+1][3]; entries >= poly_len are 0
__global__ void k_poly_export(const AxgParams p, float* __restrict__ dst) {
    const size_t rows = (size_t)p.max_segments + 1;
    const size_t total = (size_t)p.n_cones * rows;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const uint32_t c = (uint32_t)(i / rows);
        const size_t k = i % rows;
        const bool live = k < p.poly_len[c];
#pragma unroll
        for (int a = 0; a < 3; ++a) dst[i * 3 + a] = live ? p.poly[(k * 3 + a) * p.n_cones + c] : 0.0f;
    }
}

// poly[len-1] = current position (axg_place_neurons / axg_load_cones)
__global__ void k_poly_init(const AxgParams p) {
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < p.n_cones; c += gridDim.x * blockDim.x) {
        const uint32_t len = p.poly_len[c];
        if (len >= 1u && len <= p.max_segments + 1u)
            for (int a = 0; a < 3; ++a) p.poly[((size_t)(len - 1) * 3 + a) * p.n_cones + c] = p.cone_pos[c * 3 + a];
    }
}

inline int grid_for(uint32_t n, int threads, int cap) {
    long long g = ((long long)n + threads - 1) / threads;
    if (g < 1) g = 1;
    if (g > cap) g = cap;
    return (int)g;
}

}  // namespace

void axg_launch_sense(const AxgParams& p, cudaStream_t s) {
    if (!p.n_cones) return;
    if (p.sense_mode != 0)
        k_sense_particles<<<grid_for(p.n_cones, 8, 148 * 8), 256, 0, s>>>(p);
    else
        k_sense<<<grid_for(p.n_cones, 8, 148 * 8), 256, 0, s>>>(p);
}
void axg_launch_advance(const AxgParams& p, int commit, cudaStream_t s) {
    if (!p.n_cones) return;
    k_advance<<<grid_for(p.n_cones, 128, 148 * 16), 128, 0, s>>>(p, commit);
}
void axg_launch_commit(const AxgParams& p, int bump, cudaStream_t s) { k_commit<<<1, 1, 0, s>>>(p, bump); }
void axg_launch_census(const AxgParams& p, cudaStream_t s) {
    if (!p.n_cones) return;
    k_census<<<grid_for(p.n_cones, 256, 148 * 4), 256, 0, s>>>(p);
}
void axg_launch_sense_export(const AxgParams& p, long long* counts, long long* moment, cudaStream_t s) {
    if (!p.n_cones) return;
    k_sense_export<<<grid_for(p.n_cones * 4u, 256, 148 * 8), 256, 0, s>>>(p, counts, moment);
}
void axg_launch_poly_export(const AxgParams& p, float* dst, cudaStream_t s) {
    if (!p.n_cones) return;
    k_poly_export<<<148 * 8, 256, 0, s>>>(p, dst);
}
void axg_launch_poly_init(const AxgParams& p, cudaStream_t s) {
    if (!p.n_cones) return;
    k_poly_init<<<grid_for(p.n_cones, 256, 148 * 8), 256, 0, s>>>(p);
}
