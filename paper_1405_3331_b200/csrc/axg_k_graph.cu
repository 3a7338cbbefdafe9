// axg_k_graph.cu -- connection formation, the compact adjacency list and the level-synchronous BFS
// (readings A-28..A-30).
//   PAPER.md:223-233 (§3.3)  sphere-sphere collision on SQUARED distances, broadphase + narrowphase
//   PAPER.md:239      (§3.4)  the axon grows until its end is within reach of another neuron
//   PAPER.md:241-247  (§3.4)  compact adjacency list: Va = heads, Ea = edges, vertex i+1's edges follow vertex i's
//   PAPER.md:249-255  (Fig. 5) CUDA_BFS_KERNEL(Va, Ea, Fa, Xa, Ca): one thread per vertex, frontier / visited / cost
//   PAPER.md:443      (§5.1)  "the neurons would be sorted and stored in a grid data structure entirely computed on the
//                             GPU": the broadphase here -- the somata binned into a uniform grid whose cell edge is at
//                             least the collision reach (the paper's rule "cell size = object size"), so a
//                             tip only meets the somata of its 27 neighbouring cells
// The somata are the first polyline points (where axg_place_neurons put the neurons); they never move, so the soma grid
// is built once.  All kernels here are far off the bandwidth path (C <= 10^6 cones against 10^8 particles).
#include "axg_dev.cuh"

namespace {

constexpr uint32_t NO_TARGET = 0xffffffffu;
constexpr int G_THREADS = 256;

__device__ __forceinline__ uint32_t soma_cell(const AxgParams& p, float x, float y, float z) {
    const uint32_t cx = ((uint32_t)x) >> p.ng_shift, cy = ((uint32_t)y) >> p.ng_shift, cz = ((uint32_t)z) >> p.ng_shift;
    return (cz * p.ngy + cy) * p.ngx + cx;
}
__device__ __forceinline__ float soma_coord(const AxgParams& p, uint32_t n, int axis) {
    return p.poly[(size_t)axis * p.n_cones + n];  // step-major planes: plane 0 = where the neurons were placed
}

// ---- exclusive scan of n words into out[0..n] (out[n] = total): one block, every thread a contiguous slice --------
__global__ void __launch_bounds__(1024) k_scan_small(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, uint32_t n) {
    __shared__ uint32_t s_sum[1024];
    const uint32_t per = (n + 1023u) / 1024u;
    const uint32_t lo = min(threadIdx.x * per, n), hi = min(lo + per, n);
    uint32_t sum = 0u;
    for (uint32_t q = lo; q < hi; ++q) sum += in[q];
    s_sum[threadIdx.x] = sum;
    __syncthreads();
    for (uint32_t d = 1u; d < 1024u; d <<= 1) {
        const uint32_t v = threadIdx.x >= d ? s_sum[threadIdx.x - d] : 0u;
        __syncthreads();
        s_sum[threadIdx.x] += v;
        __syncthreads();
    }
    uint32_t run = s_sum[threadIdx.x] - sum;
    for (uint32_t q = lo; q < hi; ++q) {
        const uint32_t v = in[q];
        out[q] = run;
        run += v;
    }
    if (threadIdx.x == 1023u) out[n] = s_sum[1023];
}

// ---- soma grid (broadphase) -------------------------------------------------------------------------------------------
__global__ void k_soma_count(const AxgParams p, uint32_t* __restrict__ cnt) {
    for (uint32_t n = blockIdx.x * blockDim.x + threadIdx.x; n < p.n_cones; n += gridDim.x * blockDim.x)
        atomicAdd(cnt + soma_cell(p, soma_coord(p, n, 0), soma_coord(p, n, 1), soma_coord(p, n, 2)), 1u);
}
__global__ void k_soma_fill(const AxgParams p, uint32_t* __restrict__ cursor, uint32_t* __restrict__ list) {
    // the order inside a cell is the arbitrary order of the atomics: k_connect's choice does not depend on it
    for (uint32_t n = blockIdx.x * blockDim.x + threadIdx.x; n < p.n_cones; n += gridDim.x * blockDim.x) {
        const uint32_t cc = soma_cell(p, soma_coord(p, n, 0), soma_coord(p, n, 1), soma_coord(p, n, 2));
        list[p.ng_lo[cc] + atomicAdd(cursor + cc, 1u)] = n;
    }
}

// ---- narrowphase: reading A-28 ------------------------------------------------------------------------------------------
// Every cone still ACTIVE after P4 / P5 against the somata of the 27 soma-grid cells around its tip; d2 = (dx dx + dy dy)
// + dz dz with every operation rounded once (fp32 decides an integer: the oracle takes the same operations in the same
// order), strict '<' against fl(fl(r_cone + r_soma)^2); the nearest soma wins, equal distances go to the lowest index.
__global__ void __launch_bounds__(G_THREADS) k_connect(const AxgParams p) {
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < p.n_cones; c += gridDim.x * blockDim.x) {
        if (p.cone_state[c] != 0) continue;
        const float px = p.cone_pos[c * 3 + 0], py = p.cone_pos[c * 3 + 1], pz = p.cone_pos[c * 3 + 2];
        const int cx = (int)(((uint32_t)px) >> p.ng_shift), cy = (int)(((uint32_t)py) >> p.ng_shift),
                  cz = (int)(((uint32_t)pz) >> p.ng_shift);
        float best = 0.0f;
        uint32_t who = NO_TARGET;
        for (int dz = -1; dz <= 1; ++dz) {
            const int z = cz + dz;
            if (z < 0 || z >= (int)p.ngz) continue;
            for (int dy = -1; dy <= 1; ++dy) {
                const int y = cy + dy;
                if (y < 0 || y >= (int)p.ngy) continue;
                const int x0 = max(cx - 1, 0), x1 = min(cx + 1, (int)p.ngx - 1);
                const uint32_t row = ((uint32_t)z * p.ngy + (uint32_t)y) * p.ngx;
                // the three cells of a row are consecutive: one range
                for (uint32_t j = p.ng_lo[row + x0], e = p.ng_lo[row + x1 + 1]; j < e; ++j) {
                    const uint32_t n = p.ng_list[j];
                    if (n == c) continue;  // not its own neuron
                    const float dx_ = __fsub_rn(px, soma_coord(p, n, 0)), dy_ = __fsub_rn(py, soma_coord(p, n, 1)),
                                dz_ = __fsub_rn(pz, soma_coord(p, n, 2));
                    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx_, dx_), __fmul_rn(dy_, dy_)), __fmul_rn(dz_, dz_));
                    if (d2 < p.conn_thr && (who == NO_TARGET || d2 < best || (d2 == best && n < who))) {
                        best = d2;
                        who = n;
                    }
                }
            }
        }
        if (who != NO_TARGET) {
            p.cone_target[c] = who;
            p.cone_state[c] = 3;  // AXG_CONE_CONNECTED: frozen from here on
        }
    }
}

__global__ void k_fill_u32(uint32_t* __restrict__ a, uint32_t v, uint32_t n) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) a[i] = v;
}

// ---- adjacency list: reading A-29 ----------------------------------------------------------------------------------------
// Undirected: list(v) = {u : target[u] = v} + {target[v]}, ascending, without duplicates.  The in-lists are gathered by a
// counting sort over the targets (count -> scan -> fill in the arbitrary order of the atomics -> sort each list), the
// same construction as the particle binning of axg_k_count.cu, one level up.
__global__ void k_g_indeg(const AxgGraph g) {
    for (uint32_t u = blockIdx.x * blockDim.x + threadIdx.x; u < g.n; u += gridDim.x * blockDim.x) {
        const uint32_t t = g.target[u];
        if (t != NO_TARGET) atomicAdd(g.cnt + t, 1u);
    }
}
__global__ void k_g_fill(const AxgGraph g) {
    for (uint32_t u = blockIdx.x * blockDim.x + threadIdx.x; u < g.n; u += gridDim.x * blockDim.x) {
        const uint32_t t = g.target[u];
        if (t != NO_TARGET) g.in_list[g.in_lo[t] + atomicAdd(g.cursor + t, 1u)] = u;
    }
}
constexpr uint32_t G_SORT_INLINE = 32u, G_SORT_SMEM = 2048u;
// short lists: insertion sort by the owning thread; long ones are queued for k_g_sort_big
__global__ void k_g_sort(const AxgGraph g) {
    for (uint32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < g.n; v += gridDim.x * blockDim.x) {
        const uint32_t lo = g.in_lo[v], d = g.in_lo[v + 1] - lo;
        if (d > G_SORT_INLINE) {
            g.big[atomicAdd(g.n_big, 1u)] = v;  // at most n / 33 entries
            continue;
        }
        uint32_t* a = g.in_list + lo;
        for (uint32_t i = 1; i < d; ++i) {
            const uint32_t x = a[i];
            uint32_t j = i;
            while (j > 0 && a[j - 1] > x) { a[j] = a[j - 1]; --j; }
            a[j] = x;
        }
    }
}
// one block per long list: bitonic network in shared memory up to G_SORT_SMEM entries; above that every entry's rank is
// counted against the whole list (the entries are distinct), through a scratch copy
__global__ void __launch_bounds__(G_THREADS) k_g_sort_big(const AxgGraph g) {
    __shared__ uint32_t s[G_SORT_SMEM];
    const uint32_t n_big = *g.n_big;
    for (uint32_t w = blockIdx.x; w < n_big; w += gridDim.x) {
        const uint32_t v = g.big[w], lo = g.in_lo[v], d = g.in_lo[v + 1] - lo;
        uint32_t* a = g.in_list + lo;
        if (d <= G_SORT_SMEM) {
            uint32_t n2 = 64u;
            while (n2 < d) n2 <<= 1;
            for (uint32_t i = threadIdx.x; i < n2; i += G_THREADS) s[i] = i < d ? a[i] : 0xffffffffu;
            __syncthreads();
            for (uint32_t size = 2u; size <= n2; size <<= 1)
                for (uint32_t stride = size >> 1; stride > 0u; stride >>= 1) {
                    for (uint32_t t = threadIdx.x; t < (n2 >> 1); t += G_THREADS) {
                        const uint32_t i = 2u * t - (t & (stride - 1u)), j = i + stride;
                        const uint32_t x = s[i], y = s[j];
                        if ((x > y) == ((i & size) == 0u)) { s[i] = y; s[j] = x; }
                    }
                    __syncthreads();
                }
            for (uint32_t i = threadIdx.x; i < d; i += G_THREADS) a[i] = s[i];
            __syncthreads();
        } else {
            uint32_t* tmp = g.scratch + lo;
            for (uint32_t i = threadIdx.x; i < d; i += G_THREADS) tmp[i] = a[i];
            __syncthreads();
            for (uint32_t i = threadIdx.x; i < d; i += G_THREADS) {
                const uint32_t x = tmp[i];
                uint32_t rank = 0u;
                for (uint32_t j = 0; j < d; ++j) rank += tmp[j] < x ? 1u : 0u;
                a[rank] = x;
            }
            __syncthreads();
        }
    }
}
__device__ __forceinline__ bool g_contains(const uint32_t* a, uint32_t d, uint32_t x) {
    uint32_t lo = 0u, hi = d;
    while (lo < hi) {
        const uint32_t mid = (lo + hi) >> 1;
        if (a[mid] < x) lo = mid + 1u; else hi = mid;
    }
    return lo < d && a[lo] == x;
}
__global__ void k_g_degree(const AxgGraph g) {
    for (uint32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < g.n; v += gridDim.x * blockDim.x) {
        const uint32_t t = g.target[v];
        if (g.directed) {
            g.cnt[v] = t != NO_TARGET ? 1u : 0u;
        } else {
            const uint32_t lo = g.in_lo[v], d = g.in_lo[v + 1] - lo;
            g.cnt[v] = d + ((t != NO_TARGET && !g_contains(g.in_list + lo, d, t)) ? 1u : 0u);
        }
    }
}
__global__ void k_g_write(const AxgGraph g) {
    for (uint32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < g.n; v += gridDim.x * blockDim.x) {
        const uint32_t t = g.target[v];
        uint32_t o = g.Va[v];
        if (g.directed) {
            if (t != NO_TARGET) g.Ea[o] = t;
            continue;
        }
        const uint32_t lo = g.in_lo[v], d = g.in_lo[v + 1] - lo;
        const uint32_t* a = g.in_list + lo;
        const bool extra = t != NO_TARGET && !g_contains(a, d, t);
        bool placed = !extra;
        for (uint32_t i = 0; i < d; ++i) {  // merge of the sorted in-list with the one out-neighbour
            if (!placed && t < a[i]) { g.Ea[o++] = t; placed = true; }
            g.Ea[o++] = a[i];
        }
        if (!placed) g.Ea[o++] = t;
    }
}

// ---- BFS: reading A-30 ------------------------------------------------------------------------------------------------------
// Fig. 5 of the paper with the updating-frontier array of the algorithm it cites: as printed (one frontier array) a vertex
// switched on in this pass could be expanded in the same pass.  Pass 1 expands the frontier F: C[nid] = C[tid] + 1 for
// every unvisited neighbour (all writers of one pass write the same level), Fu[nid] = true; pass 2 moves Fu into F, marks
// X and raises the "frontier not empty" flag.
__global__ void k_bfs_init(const AxgGraph g, uint32_t root) {
    for (uint32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < g.n; v += gridDim.x * blockDim.x) {
        g.C[v] = v == root ? 0 : -1;
        g.F[v] = v == root ? 1 : 0;
        g.X[v] = v == root ? 1 : 0;
        g.Fu[v] = 0;
    }
}
__global__ void k_bfs_expand(const AxgGraph g) {
    for (uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x; tid < g.n; tid += gridDim.x * blockDim.x) {
        if (!g.F[tid]) continue;
        g.F[tid] = 0;
        const int c = g.C[tid] + 1;
        for (uint32_t e = g.Va[tid]; e < g.Va[tid + 1]; ++e) {
            const uint32_t nid = g.Ea[e];
            if (!g.X[nid]) {
                g.C[nid] = c;
                g.Fu[nid] = 1;
            }
        }
    }
}
__global__ void k_bfs_advance(const AxgGraph g) {
    for (uint32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < g.n; v += gridDim.x * blockDim.x) {
        if (!g.Fu[v]) continue;
        g.Fu[v] = 0;
        g.F[v] = 1;
        g.X[v] = 1;
        *g.flag = 1u;
    }
}

int grid_for(uint32_t n) { return (int)max(1u, min((n + G_THREADS - 1) / G_THREADS, 148u * 8u)); }

}  // namespace

void axg_launch_scan_small(const uint32_t* in, uint32_t* out, uint32_t n, cudaStream_t s) {
    k_scan_small<<<1, 1024, 0, s>>>(in, out, n);
}
void axg_launch_soma_grid(const AxgParams& p, uint32_t* cnt, uint32_t* cursor, uint32_t* lo, uint32_t* list,
                          uint32_t n_cells, cudaStream_t s) {
    cudaMemsetAsync(cnt, 0, ((size_t)n_cells + 1) * 4, s);
    cudaMemsetAsync(cursor, 0, ((size_t)n_cells + 1) * 4, s);
    k_soma_count<<<grid_for(p.n_cones), G_THREADS, 0, s>>>(p, cnt);
    k_scan_small<<<1, 1024, 0, s>>>(cnt, lo, n_cells);
    k_soma_fill<<<grid_for(p.n_cones), G_THREADS, 0, s>>>(p, cursor, list);
}
void axg_launch_connect(const AxgParams& p, cudaStream_t s) { k_connect<<<grid_for(p.n_cones), G_THREADS, 0, s>>>(p); }
void axg_launch_fill_u32(uint32_t* a, uint32_t v, uint32_t n, cudaStream_t s) {
    if (n) k_fill_u32<<<grid_for(n), G_THREADS, 0, s>>>(a, v, n);
}
void axg_launch_graph_build(const AxgGraph& g, cudaStream_t s) {
    const int grid = grid_for(g.n);
    if (!g.directed) {
        cudaMemsetAsync(g.cnt, 0, ((size_t)g.n + 1) * 4, s);
        cudaMemsetAsync(g.cursor, 0, ((size_t)g.n + 1) * 4, s);
        cudaMemsetAsync(g.n_big, 0, 4, s);
        k_g_indeg<<<grid, G_THREADS, 0, s>>>(g);
        k_scan_small<<<1, 1024, 0, s>>>(g.cnt, g.in_lo, g.n);
        k_g_fill<<<grid, G_THREADS, 0, s>>>(g);
        k_g_sort<<<grid, G_THREADS, 0, s>>>(g);
        k_g_sort_big<<<148, G_THREADS, 0, s>>>(g);
    }
    k_g_degree<<<grid, G_THREADS, 0, s>>>(g);
    k_scan_small<<<1, 1024, 0, s>>>(g.cnt, g.Va, g.n);
    k_g_write<<<grid, G_THREADS, 0, s>>>(g);
}
void axg_launch_bfs_init(const AxgGraph& g, uint32_t root, cudaStream_t s) {
    k_bfs_init<<<grid_for(g.n), G_THREADS, 0, s>>>(g, root);
}
void axg_launch_bfs_level(const AxgGraph& g, cudaStream_t s) {
    k_bfs_expand<<<grid_for(g.n), G_THREADS, 0, s>>>(g);
    k_bfs_advance<<<grid_for(g.n), G_THREADS, 0, s>>>(g);
}

// ---- the BFS for callers that may not allocate (include/axg.h axg_bfs_noalloc) ---------------------------------------------
// Same kernels, same algorithm (reading A-30) as axg_bfs; what differs is where the scratch lives: the frontier, the
// updating frontier, the visited flags (one byte per vertex each) and the "frontier not empty" word sit in ONE file-scope
// device array of fixed size instead of buffers taken from the allocator.  Every GPU that loads the library holds these
// 3 MB + 256 B until exit.  All calls share the array and it keeps the last call's contents: k_bfs_init rewrites all four
// regions for the vertices of THIS call before anything reads them, and two calls that overlap on the GPU (different
// streams, or two host threads) race on it.
#include "../../include/axg.h"

void axg_set_global_error(const char* msg);  // axg_api.cu: the message axg_last_error(NULL) returns

namespace {

constexpr uint32_t NOALLOC_MAX_VERTICES = AXG_BFS_NOALLOC_MAX_VERTICES;
constexpr size_t NOALLOC_FLAG_AT = 3 * (size_t)NOALLOC_MAX_VERTICES;  // a multiple of 256
static __device__ __align__(256) unsigned char g_bfs_scratch[NOALLOC_FLAG_AT + 256];

// In host code `g_bfs_scratch` is a host-side stand-in for the symbol, not a device address: the address is asked of the
// runtime once per device, with that device current, and cached.
constexpr int NOALLOC_MAX_DEVICES = 64;
unsigned char* g_bfs_scratch_dev[NOALLOC_MAX_DEVICES] = {nullptr};

int noalloc_fail(int code, const char* msg) {
    axg_set_global_error(msg);
    return code;
}

}  // namespace

extern "C" __attribute__((visibility("default"))) int axg_bfs_noalloc(const uint32_t* va, const uint32_t* ea,
                                                                      uint32_t n_vertices, uint32_t root, int32_t* level,
                                                                      void* stream) {
    if (!va || !ea || !level) return noalloc_fail(AXG_EINVAL, "axg_bfs_noalloc: null argument");
    if (n_vertices == 0) return noalloc_fail(AXG_EINVAL, "axg_bfs_noalloc: empty graph");
    if (n_vertices > NOALLOC_MAX_VERTICES)
        return noalloc_fail(AXG_EINVAL, "axg_bfs_noalloc: more vertices than AXG_BFS_NOALLOC_MAX_VERTICES (2^20): the "
                                        "scratch array is fixed; use axg_bfs");
    if (root >= n_vertices) return noalloc_fail(AXG_EINVAL, "axg_bfs_noalloc: root out of range");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NOALLOC_MAX_DEVICES) {
        cudaGetLastError();
        return noalloc_fail(AXG_ECUDA, "axg_bfs_noalloc: no current CUDA device");
    }
    if (!g_bfs_scratch_dev[dev]) {
        void* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, g_bfs_scratch);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            return noalloc_fail(AXG_ECUDA, "axg_bfs_noalloc: cudaGetSymbolAddress failed");
        }
        g_bfs_scratch_dev[dev] = static_cast<unsigned char*>(ptr);
    }
    unsigned char* const scratch = g_bfs_scratch_dev[dev];
    cudaStream_t s = (cudaStream_t)stream;
    AxgGraph g = {};
    g.n = n_vertices;
    g.Va = const_cast<uint32_t*>(va);  // read only by the BFS kernels
    g.Ea = const_cast<uint32_t*>(ea);
    g.C = level;
    g.F = scratch;
    g.Fu = scratch + NOALLOC_MAX_VERTICES;
    g.X = scratch + 2 * (size_t)NOALLOC_MAX_VERTICES;
    g.flag = reinterpret_cast<uint32_t*>(scratch + NOALLOC_FLAG_AT);
    k_bfs_init<<<grid_for(n_vertices), G_THREADS, 0, s>>>(g, root);  // clears F / Fu / X / C of this call's vertices
    for (uint32_t lv = 0; lv <= n_vertices; ++lv) {  // "repeated until frontier is empty"
        uint32_t more = 0;
        cudaError_t e = cudaMemsetAsync(g.flag, 0, 4, s);
        k_bfs_expand<<<grid_for(n_vertices), G_THREADS, 0, s>>>(g);
        k_bfs_advance<<<grid_for(n_vertices), G_THREADS, 0, s>>>(g);
        if (e == cudaSuccess) e = cudaMemcpyAsync(&more, g.flag, 4, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) return noalloc_fail(AXG_ECUDA, cudaGetErrorString(e));
        if (!more) break;
    }
    return AXG_OK;
}
