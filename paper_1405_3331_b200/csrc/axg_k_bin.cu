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
constexpr uint32_t INLINE_GAP = 4;  // gaps up to this many cells are filled by the owning thread

__global__ void __launch_bounds__(BIN_THREADS) k_reorder(const AxgParams p) {
    __shared__ uint32_t s_qlo[2 * BIN_THREADS], s_qhi[2 * BIN_THREADS], s_qval[2 * BIN_THREADS];
    __shared__ uint32_t s_qn;
    const AxgDev* dev = p.dev;
    const uint32_t n = dev->n_live;
    const uint32_t* __restrict__ keys = p.skey[p.final_buf];
    const uint32_t* __restrict__ perm = p.sidx[p.final_buf];
    uint32_t* __restrict__ cell_lo = p.cell_lo;
    const int tid = threadIdx.x;

    if (n == 0u) {  // nothing alive: every prefix is 0
        for (uint32_t c = blockIdx.x * BIN_THREADS + tid; c <= p.cells; c += gridDim.x * BIN_THREADS) cell_lo[c] = 0u;
        return;
    }
    const uint32_t n_round = (n + BIN_THREADS - 1) / BIN_THREADS;
    for (uint32_t r = blockIdx.x; r < n_round; r += gridDim.x) {
        if (tid == 0) s_qn = 0u;
        __syncthreads();
        const uint32_t j = r * BIN_THREADS + tid;
        if (j < n) {
            const uint32_t k = __ldg(keys + j);
            const uint32_t src = __ldg(perm + j);
            // O5: A[j] = B[perm[j]]
            p.A.x[j] = __ldg(p.B.x + src);
            p.A.y[j] = __ldg(p.B.y + src);
            p.A.z[j] = __ldg(p.B.z + src);
            p.A.id[j] = __ldg(p.B.id + src);
            p.A.species[j] = __ldg(p.B.species + src);
            // O6 as prefix counts: cells (k_prev, k] have exactly j particles below them
            const uint32_t lo = (j == 0u) ? 0u : __ldg(keys + j - 1) + 1u;
            if (lo <= k) {
                if (k - lo < INLINE_GAP) {
                    for (uint32_t c = lo; c <= k; ++c) cell_lo[c] = j;
                } else {
                    const uint32_t q = atomicAdd(&s_qn, 1u);
                    s_qlo[q] = lo; s_qhi[q] = k; s_qval[q] = j;
                }
            }
            if (j == n - 1u) {  // cells above the last key, and the end sentinel cell_lo[cells] = n
                const uint32_t q = atomicAdd(&s_qn, 1u);
                s_qlo[q] = k + 1u; s_qhi[q] = p.cells; s_qval[q] = n;
            }
        }
        __syncthreads();
        const uint32_t qn = s_qn;
        for (uint32_t q = 0; q < qn; ++q) {  // long gaps: the whole block fills, coalesced
            const uint32_t lo = s_qlo[q], hi = s_qhi[q], v = s_qval[q];
            for (uint32_t c = lo + tid; c <= hi && c >= lo; c += BIN_THREADS) cell_lo[c] = v;
        }
        __syncthreads();
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

void axg_launch_reorder(const AxgParams& p, int grid, cudaStream_t s) { k_reorder<<<grid, BIN_THREADS, 0, s>>>(p); }

void axg_launch_cell_export(const AxgParams& p, uint32_t* start, uint32_t* end, cudaStream_t s) {
    k_cell_export<<<148 * 8, 256, 0, s>>>(p, start, end);
}
