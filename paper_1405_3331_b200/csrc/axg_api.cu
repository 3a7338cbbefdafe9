// axg_api.cu -- the C-ABI of include/axg.h: context, device memory, and the per-step kernel sequence.
// Host orchestration only: every step of the path (P1..P5) runs in the kernels of axg_k_*.cu; there is no CPU
// fallback (axg_create fails with AXG_ECUDA without a device).
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/axg.h"
#include "axg_dev.cuh"

#define AXG_API extern "C" __attribute__((visibility("default")))

namespace {

axg_alloc_fn g_alloc = nullptr;
axg_free_fn g_free = nullptr;
void* g_alloc_user = nullptr;
thread_local std::string g_create_err;

struct Source {
    float x, y, z;
    uint8_t species;
    int8_t polarity;
    uint32_t rate;
};

constexpr int N_SM = 148;
// k_reorder variant: four slots per thread when the particle streams cannot live in the L2 (see axg_k_bin.cu)
constexpr uint64_t AXG_REORDER_WIDE_ABOVE = 32ull << 20;

}  // namespace

// the message of a failing call that has no context (axg_create, axg_bfs_noalloc): what axg_last_error(NULL) returns
void axg_set_global_error(const char* msg) { g_create_err = msg ? msg : ""; }

struct axg_ctx {
    axg_grid grid;
    float D, radius, speed, noise;
    uint32_t emission;
    uint64_t seed;
    uint64_t max_particles = 1ull << 20;
    uint32_t max_segments = 1024;
    uint32_t shard_rank = 0, shard_world = 1;
    long long s2_cells = 0;  // S2(R) of the per-cell stencil (alloc_fixed)
    std::vector<Source> sources;
    int8_t species_polarity[AXG_MAX_SPECIES] = {0, 0, 0, 0};
    uint32_t n_cones = 0;
    bool stepped = false;
    cudaStream_t stream = nullptr;
    // P3..P5 of step t run on a side stream while k_diffuse of step t+1 runs on `stream` (axg_step only)
    cudaStream_t side = nullptr;
    cudaEvent_t ev_bin = nullptr, ev_adv = nullptr;
    bool adv_pending = false;
    // one step of axg_step(n >= AXG_GRAPH_MIN_STEPS) as a CUDA graph (enqueue_unit), re-captured when anything it bakes in
    // -- the parameter block, the stream -- has changed
    cudaStream_t gstream = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    cudaGraphExec_t graph_exec = nullptr;
    AxgParams graph_P;
    cudaStream_t graph_stream = nullptr;
    bool graph_cones = false;
    std::string err;

    // device memory
    bool particles_allocated = false;
    std::vector<void*> particle_bufs;  // everything sized by max_particles
    void* d_dev = nullptr;
    void* d_cell_lo = nullptr;
    void* d_cnt = nullptr;
    void* d_scan_state = nullptr;
    int bin_request = AXG_BIN_AUTO;
    bool b_chunked = false;   // the pre-sort array is in the chunked layout of k_diffuse_chunked (count binning)
    bool kp_pending = false;  // count binning: the last P2 left sorted keys / permutation to be derived on read (k_settle<true>)
    bool cnt_dirty = false;   // P1 has counted into cnt and P2 has not consumed (and re-zeroed) it yet
    bool p1_pending = false;  // a P1 has run and its output has not been binned yet: the next AXG_PHASE_BIN bins IT
                              // (the sharded loop enqueues P1 and P2 in separate calls), not a re-keyed copy of A
    void* d_src = nullptr;
    void* d_src_id_prefix = nullptr;
    void* d_src_emit_prefix = nullptr;
    void* d_stencil = nullptr;
    std::vector<void*> cone_bufs;
    void* d_poly = nullptr;
    AxgParams P;
    uint32_t loaded_species_mask = 0;  // species seen by axg_load_particles
    uint32_t n_A = 0, n_B = 0;  // element counts of the sorted / pre-sort arrays as of the last synchronised call

    // stats of the last axg_step
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    float last_ms = 0.f;
    uint64_t last_launches = 0, last_particle_steps = 0, ps0 = 0;
    bool profile_next = false;
    float ktimes[AXG_KERNEL_COUNT] = {0};
    std::vector<cudaEvent_t> prof_events;

    // connection formation / graph (axg_set_connect, axg_build_graph, axg_bfs)
    float r_cone = 0.f, r_soma = 0.f;
    bool soma_grid_built = false;
    std::vector<void*> connect_bufs;   // soma grid
    void* d_target = nullptr;
    std::vector<void*> graph_bufs;
    AxgGraph G;
    bool graph_built = false;
    uint32_t graph_edges = 0;
    bool bfs_done = false;

    int key_order = AXG_KEY_LINEAR;  // axg_set_key_order: AXG_KEY_BRICK pads the key space to whole 8 x 4 x 4 bricks
    size_t nbx() const { return (grid.nx + 7) / 8; }
    size_t nby() const { return (grid.ny + 3) / 4; }
    static int axis_bits(uint32_t n) {
        int b = 0;
        while ((1u << b) < n) ++b;
        return b;
    }
    size_t cells() const {  // size of the key space
        if (key_order == AXG_KEY_LINEAR) return (size_t)grid.nx * grid.ny * grid.nz;
        if (key_order == AXG_KEY_MORTON) return (size_t)1 << (axis_bits(grid.nx) + axis_bits(grid.ny) + axis_bits(grid.nz));
        return nbx() * nby() * ((grid.nz + 3) / 4) * 128;
    }
    // cell arrays are padded to whole scan tiles so that 128-bit accesses of the last tile stay inside
    size_t cells_padded() const { return ((cells() + 1 + AXG_SCAN_TILE - 1) / AXG_SCAN_TILE + 1) * AXG_SCAN_TILE; }
    // look-back words of k_cell_scan (one per tile) / block sums of k_cell_scan2 (one per block, at most 148 x 2)
    size_t scan_tiles() const { return std::max<size_t>(cells_padded() / AXG_SCAN_TILE + 2, 512); }
};

namespace {

int ensure_soma_grid(axg_ctx* c);  // connection formation, defined with the graph calls below

int fail(axg_ctx* c, int code, const std::string& msg) {
    if (c) c->err = msg; else g_create_err = msg;
    return code;
}

int cuda_fail(axg_ctx* c, cudaError_t e, const char* what) {
    return fail(c, AXG_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define CU(c, call)                                            \
    do {                                                       \
        cudaError_t e_ = (call);                               \
        if (e_ != cudaSuccess) return cuda_fail(c, e_, #call); \
    } while (0)

void* dev_alloc(axg_ctx* c, size_t bytes) {
    if (bytes == 0) bytes = 16;
    bytes = (bytes + 255) & ~(size_t)255;
    void* p = nullptr;
    if (g_alloc) {
        p = g_alloc(bytes, (void*)c->stream, g_alloc_user);
    } else if (cudaMalloc(&p, bytes) != cudaSuccess) {
        p = nullptr;
    }
    return p;
}

void dev_free(void* p) {
    if (!p) return;
    if (g_free) g_free(p, g_alloc_user); else cudaFree(p);
}

bool inside(const axg_ctx* c, float x, float y, float z) {
    return x >= 0.0f && x < (float)c->grid.nx && y >= 0.0f && y < (float)c->grid.ny && z >= 0.0f &&
           z < (float)c->grid.nz;
}

uint64_t owned_rate(const axg_ctx* c) {
    uint64_t e = 0;
    for (size_t s = 0; s < c->sources.size(); ++s)
        if (s % c->shard_world == c->shard_rank) e += c->sources[s].rate;
    return e;
}

int key_bits(size_t cells) {
    int bits = 1;
    while (bits < 32 && ((size_t)1 << bits) < cells) ++bits;
    return bits;
}
// 9-bit digits where they save a pass (27-bit keys: C4), 8-bit otherwise (one ballot less per key)
int digit_bits_for(size_t cells) {
    const int b = key_bits(cells);
    return (b + 8) / 9 < (b + 7) / 8 ? 9 : 8;
}

// ---- allocation ------------------------------------------------------------------------------------------
int alloc_fixed(axg_ctx* c) {
    if (c->d_dev) return AXG_OK;
    c->d_dev = dev_alloc(c, sizeof(AxgDev));
    c->d_cell_lo = dev_alloc(c, c->cells_padded() * sizeof(uint32_t));
    c->d_src = dev_alloc(c, AXG_MAX_SOURCES * sizeof(AxgSourceDev));
    c->d_src_id_prefix = dev_alloc(c, (AXG_MAX_SOURCES + 1) * sizeof(uint32_t));
    c->d_src_emit_prefix = dev_alloc(c, (AXG_MAX_SOURCES + 1) * sizeof(uint32_t));
    // stencil {d : |d|^2 <= floor(R^2)} (reading A-11) and S2(R) = sum dx^2 (reading A-12)
    const int r2 = (int)std::floor((double)c->radius * (double)c->radius);
    const int R = (int)std::floor((double)c->radius);
    std::vector<int32_t> st;
    long long s2 = 0;
    for (int dz = -R; dz <= R; ++dz)
        for (int dy = -R; dy <= R; ++dy)
            for (int dx = -R; dx <= R; ++dx)
                if (dx * dx + dy * dy + dz * dz <= r2) {
                    st.push_back((dx & 0xff) | ((dy & 0xff) << 8) | ((dz & 0xff) << 16));
                    s2 += dx * dx;
                }
    c->d_stencil = dev_alloc(c, st.size() * sizeof(int32_t));
    if (!c->d_dev || !c->d_cell_lo || !c->d_src || !c->d_src_id_prefix || !c->d_src_emit_prefix || !c->d_stencil)
        return fail(c, AXG_ECUDA, "device allocation failed");
    CU(c, cudaMemsetAsync(c->d_dev, 0, sizeof(AxgDev), c->stream));
    CU(c, cudaMemsetAsync(c->d_cell_lo, 0, c->cells_padded() * sizeof(uint32_t), c->stream));
    CU(c, cudaMemcpyAsync(c->d_stencil, st.data(), st.size() * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    AxgParams& P = c->P;
    P.dev = (AxgDev*)c->d_dev;
    P.cell_lo = (uint32_t*)c->d_cell_lo;
    P.nx = c->grid.nx; P.ny = c->grid.ny; P.nz = c->grid.nz; P.cells = (uint32_t)c->cells();
    P.key_order = c->key_order; P.nbx = (uint32_t)c->nbx(); P.nby = (uint32_t)c->nby();
    {   // streaming hints where the per-cell arrays (4 B x cells each) are beyond the L2 (126 MB): C4, C5; not C1..C3
        const char* e = std::getenv("AXG_STREAM_HINT");  // 0 / 1 overrides (measurements)
        P.cs = e ? (e[0] == '1') : (c->cells() * sizeof(uint32_t) > (size_t)256 << 20);
    }
    {   // the phases of the Z-order bit rotation (reading A-31)
        const int nb[3] = {axg_ctx::axis_bits(c->grid.nx), axg_ctx::axis_bits(c->grid.ny), axg_ctx::axis_bits(c->grid.nz)};
        const int m3 = std::min(nb[0], std::min(nb[1], nb[2]));
        int rem[3], left[3], n_left = 0;
        for (int a = 0; a < 3; ++a) {
            rem[a] = nb[a] - m3;
            if (rem[a] > 0) left[n_left++] = a;
        }
        P.mo_m3 = (uint32_t)m3; P.mo_m2 = 0; P.mo_p = 0; P.mo_q = 1; P.mo_r = 0; P.mo_rshift = 0; P.mo_rbits = 0;
        if (n_left == 2) {
            const int pa = left[0], qa = left[1], m2 = std::min(rem[pa], rem[qa]);
            P.mo_p = (uint32_t)pa; P.mo_q = (uint32_t)qa; P.mo_m2 = (uint32_t)m2;
            P.mo_r = (uint32_t)(rem[pa] >= rem[qa] ? pa : qa);
            P.mo_rshift = (uint32_t)(m3 + m2);
            P.mo_rbits = (uint32_t)std::abs(rem[pa] - rem[qa]);
        } else if (n_left == 1) {
            P.mo_r = (uint32_t)left[0]; P.mo_rshift = (uint32_t)m3; P.mo_rbits = (uint32_t)rem[left[0]];
        }
    }
    P.fnx = (float)c->grid.nx; P.fny = (float)c->grid.ny; P.fnz = (float)c->grid.nz;
    P.sigma = (float)std::sqrt(2.0 * (double)c->D);  // O0
    P.seed_lo = (uint32_t)(c->seed & 0xffffffffull);
    P.seed_hi = (uint32_t)(c->seed >> 32);
    P.digit_bits = digit_bits_for(c->cells());
    P.n_pass = (key_bits(c->cells()) + P.digit_bits - 1) / P.digit_bits;
    P.final_buf = (P.n_pass - 1) & 1;
    P.src = (const AxgSourceDev*)c->d_src;
    P.src_id_prefix = (const uint32_t*)c->d_src_id_prefix;
    P.src_emit_prefix = (const uint32_t*)c->d_src_emit_prefix;
    P.stencil = (const int32_t*)c->d_stencil;
    P.n_stencil = (uint32_t)st.size();
    c->s2_cells = s2;
    P.s2 = (float)(s2 * (P.sense_mode ? 256 : 1));
    P.radius = c->radius;
    P.r2f = c->radius * c->radius;
    P.speed = c->speed; P.noise = c->noise;
    return AXG_OK;
}

void free_particles(axg_ctx* c) {
    for (void* p : c->particle_bufs) dev_free(p);
    c->particle_bufs.clear();
    c->particles_allocated = false;
}

// fills P.A, P.B, keys, look-back words for `cap` particles
int alloc_particles(axg_ctx* c, uint64_t cap, AxgParams& P, std::vector<void*>& bufs) {
    const size_t pad = 256;  // tail padding: ragged tiles may over-read harmlessly; the chunked layout rounds up to 128
    const size_t n = (size_t)cap + pad;
    const size_t diff_tiles = n / axg_diffuse_tile() + 2, sort_tiles = n / axg_sort_tile() + 2;
    const size_t sizes[] = {n * 4, n * 4, n * 4, n, n * 4,  // A (SoA)
                            n * 16, n,                      // Brec, Bsp
                            n * 8, n * 4, n * 4, n * 4, n * 4,  // key_pre (radix) = kw (count: key + arrival rank), skey[2], sidx[2]
                            diff_tiles * 8, sort_tiles * ((size_t)1 << P.digit_bits) * 8,
                            (n / AXG_CHUNK + 4) * 4, (n / AXG_CHUNK + 4) * 4,   // chunk_cnt, chunk_base
                            (n / 33 + 64) * 4, AXG_MAX_SOURCES * 4};            // big_list, src_arr
    constexpr int NB = 18;
    void* ptr[NB];
    for (int i = 0; i < NB; ++i) {
        ptr[i] = dev_alloc(c, sizes[i]);
        if (!ptr[i]) {
            for (int k = 0; k < i; ++k) dev_free(ptr[k]);
            bufs.resize(bufs.size() - (size_t)i);
            return fail(c, AXG_ECUDA, "device allocation failed (particle arrays)");
        }
        bufs.push_back(ptr[i]);
    }
    P.A = AxgSoA{(float*)ptr[0], (float*)ptr[1], (float*)ptr[2], (uint8_t*)ptr[3], (uint32_t*)ptr[4]};
    P.Brec = (float4*)ptr[5];
    P.Bsp = (uint8_t*)ptr[6];
    P.key_pre = (uint32_t*)ptr[7];
    P.skey[0] = (uint32_t*)ptr[8]; P.skey[1] = (uint32_t*)ptr[9];
    P.sidx[0] = (uint32_t*)ptr[10]; P.sidx[1] = (uint32_t*)ptr[11];
    P.tile_state = (unsigned long long*)ptr[12];
    P.sort_state = (unsigned long long*)ptr[13];
    P.chunk_cnt = (uint32_t*)ptr[14];
    P.chunk_base = (uint32_t*)ptr[15];
    P.kw = (uint2*)ptr[7];
    P.big_list = (uint32_t*)ptr[16];
    P.src_arr = (uint32_t*)ptr[17];
    P.capacity = (uint32_t)cap;
    // look-back words must not alias a live epoch: zero them (epoch 0 words with flag 0 = not ready)
    CU(c, cudaMemsetAsync(ptr[12], 0, sizes[12], c->stream));
    CU(c, cudaMemsetAsync(ptr[13], 0, sizes[13], c->stream));
    return AXG_OK;
}

// AXG_BIN_AUTO -> a concrete mode; the count array exists (all-zero) whenever the mode is COUNT
int resolve_binning(axg_ctx* c) {
    int mode = c->bin_request;
    // count mode pays per cell (scan + 8 B x cells of memory) and per particle; measured faster than radix on C1..C5,
    // also where the count array (C4: 0.5 GB, C5: 1 GB) is far larger than the L2
    if (mode == AXG_BIN_AUTO)
        mode = (c->cells() <= AXG_AUTO_COUNT_MAX_CELLS && c->cells() <= 4 * (size_t)c->max_particles) ? AXG_BIN_COUNT
                                                                                                      : AXG_BIN_RADIX;
    if (mode == AXG_BIN_COUNT && !c->d_cnt) {
        c->d_cnt = dev_alloc(c, c->cells_padded() * sizeof(uint32_t));
        c->d_scan_state = dev_alloc(c, c->scan_tiles() * sizeof(unsigned long long));
        if (!c->d_cnt || !c->d_scan_state) return fail(c, AXG_ECUDA, "device allocation failed (cell counts)");
        CU(c, cudaMemsetAsync(c->d_cnt, 0, c->cells_padded() * sizeof(uint32_t), c->stream));
        CU(c, cudaMemsetAsync(c->d_scan_state, 0, c->scan_tiles() * sizeof(unsigned long long), c->stream));
        c->P.cnt = (uint32_t*)c->d_cnt;
        c->P.scan_state = (unsigned long long*)c->d_scan_state;
    }
    c->P.bin_mode = mode == AXG_BIN_COUNT ? AXG_BIN_COUNT_D : AXG_BIN_RADIX_D;
    return AXG_OK;
}

int ensure_particles(axg_ctx* c) {
    int rc = alloc_fixed(c);
    if (rc) return rc;
    if (!c->particles_allocated) {
        rc = alloc_particles(c, c->max_particles, c->P, c->particle_bufs);
        if (rc) return rc;
        c->particles_allocated = true;
    }
    return resolve_binning(c);
}

void free_graph(axg_ctx* c) {
    for (void* p : c->graph_bufs) dev_free(p);
    c->graph_bufs.clear();
    c->graph_built = c->bfs_done = false;
    c->graph_edges = 0;
}

void free_connect(axg_ctx* c) {
    for (void* p : c->connect_bufs) dev_free(p);
    c->connect_bufs.clear();
    c->soma_grid_built = false;
    c->P.ng_lo = nullptr;
    c->P.ng_list = nullptr;
}

void free_cones(axg_ctx* c) {
    free_graph(c);
    free_connect(c);
    dev_free(c->d_target);
    c->d_target = nullptr;
    for (void* p : c->cone_bufs) dev_free(p);
    c->cone_bufs.clear();
    dev_free(c->d_poly);
    c->d_poly = nullptr;
}

size_t poly_bytes(const axg_ctx* c, uint32_t max_segments) {
    return ((size_t)max_segments + 1) * 3 * (size_t)c->n_cones * sizeof(float);
}

int alloc_cones(axg_ctx* c, uint32_t n) {
    free_cones(c);
    c->n_cones = n;
    AxgParams& P = c->P;
    P.n_cones = n;
    P.max_segments = c->max_segments;
    if (n == 0) return AXG_OK;
    const size_t sizes[] = {(size_t)n * 12, (size_t)n * 12, (size_t)n, (size_t)n * 64, (size_t)n * 12, (size_t)n * 4};
    void* ptr[6];
    for (int i = 0; i < 6; ++i) {
        ptr[i] = dev_alloc(c, sizes[i]);
        if (!ptr[i]) return fail(c, AXG_ECUDA, "device allocation failed (cones)");
        c->cone_bufs.push_back(ptr[i]);
        CU(c, cudaMemsetAsync(ptr[i], 0, sizes[i], c->stream));
    }
    c->d_poly = dev_alloc(c, poly_bytes(c, c->max_segments));
    if (!c->d_poly) return fail(c, AXG_ECUDA, "device allocation failed (polylines)");
    CU(c, cudaMemsetAsync(c->d_poly, 0, poly_bytes(c, c->max_segments), c->stream));
    c->d_target = dev_alloc(c, (size_t)n * 4);
    if (!c->d_target) return fail(c, AXG_ECUDA, "device allocation failed (cone targets)");
    CU(c, cudaMemsetAsync(c->d_target, 0xff, (size_t)n * 4, c->stream));  // 0xffffffff = no connection
    P.cone_target = (uint32_t*)c->d_target;
    P.cone_pos = (float*)ptr[0]; P.cone_heading = (float*)ptr[1]; P.cone_state = (uint8_t*)ptr[2];
    P.sense = (int32_t*)ptr[3]; P.cone_gradient = (float*)ptr[4]; P.poly_len = (uint32_t*)ptr[5];
    P.poly = (float*)c->d_poly;
    return AXG_OK;
}

// upload sources + the two rate prefixes, refresh the source-derived parameters
int upload_sources(axg_ctx* c) {
    int rc = alloc_fixed(c);
    if (rc) return rc;
    const size_t S = c->sources.size();
    std::vector<AxgSourceDev> sd(S);
    std::vector<uint32_t> idp(S + 1, 0u), emp(S + 1, 0u);
    int n_species_used = 0, only = -1;
    for (int s = 0; s < (int)AXG_MAX_SPECIES; ++s) {
        c->P.polarity[s] = c->species_polarity[s];
        if (c->species_polarity[s] != 0 || ((c->loaded_species_mask >> s) & 1u)) { ++n_species_used; only = s; }
    }
    for (size_t s = 0; s < S; ++s) {
        const Source& q = c->sources[s];
        sd[s] = AxgSourceDev{q.x, q.y, q.z, (uint32_t)q.species | (q.polarity == 1 ? 0x100u : 0u)};
        const bool owned = (s % c->shard_world) == c->shard_rank;
        idp[s + 1] = idp[s] + q.rate;
        emp[s + 1] = emp[s] + (owned ? q.rate : 0u);
    }
    if (S) {
        CU(c, cudaMemcpyAsync(c->d_src, sd.data(), S * sizeof(AxgSourceDev), cudaMemcpyHostToDevice, c->stream));
    }
    CU(c, cudaMemcpyAsync(c->d_src_id_prefix, idp.data(), (S + 1) * 4, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(c->d_src_emit_prefix, emp.data(), (S + 1) * 4, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    c->P.n_src = (uint32_t)S;
    c->P.e_total = idp[S];
    c->P.e_owned = emp[S];
    // with one species in use (by sources and by loaded particles) every particle in a cell has it: counts come
    // from cell_lo alone and the species bytes are not walked.
    c->P.single_species = (n_species_used == 1) ? only : -1;
    return AXG_OK;
}

int read_dev(axg_ctx* c, AxgDev* h) {
    CU(c, cudaMemcpyAsync(h, c->d_dev, sizeof(AxgDev), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    return AXG_OK;
}

}  // namespace

// ============================================ step sequence ==================================================
namespace {

struct Prof {
    axg_ctx* c;
    bool on;
    size_t used = 0;
    std::vector<int> tags;
    void mark(int tag) {  // event BEFORE the kernel(s) of `tag`; a final mark(-1) closes the last one
        if (!on) return;
        if (used == c->prof_events.size()) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            c->prof_events.push_back(e);
        }
        cudaEventRecord(c->prof_events[used++], c->stream);
        tags.push_back(tag);
    }
};

// enqueue the selected phases of one step; returns the number of kernel launches
// on / no_realign: the sharded loop's form (axg_enqueue_phase_on) -- the phases go to the stream `on`, and a commit that
// runs beside the next step's P1 must not re-align P1's step index (P1 has already bumped it)
int enqueue_phases(axg_ctx* c, uint32_t mask, Prof& prof, bool overlap = false, cudaStream_t on = nullptr,
                   bool use_on = false, bool no_realign = false) {
    const AxgParams& P = c->P;
    cudaStream_t s = use_on ? on : c->stream;
    int launches = 0;
    const bool count_mode = P.bin_mode == AXG_BIN_COUNT_D;
    auto zero_cnt_if_dirty = [&]() {  // harness orders only (P1 twice, or P2 on given positions after a P1)
        if (count_mode && c->cnt_dirty) cudaMemsetAsync(c->d_cnt, 0, c->cells_padded() * sizeof(uint32_t), s);
    };
    if (mask & AXG_PHASE_DIFFUSE) {
        zero_cnt_if_dirty();
        prof.mark(AXG_K_DIFFUSE);
        axg_launch_diffuse(P, N_SM * 4, s);  // its last block emits and closes P1
        launches += 1;
        c->cnt_dirty = count_mode;
        c->b_chunked = count_mode;
        c->kp_pending = false;  // the records that a replay of k_settle would gather are gone
        c->p1_pending = true;
    }
    if (mask & AXG_PHASE_BIN) {
        // the previous step's P3 (side stream) still reads cell_lo and the species column that P2 rewrites
        if (overlap && c->adv_pending) cudaStreamWaitEvent(s, c->ev_adv, 0);
        if (!c->p1_pending) {  // no P1 of this step: bin the current array as it stands (harness: given positions)
            zero_cnt_if_dirty();
            prof.mark(AXG_K_EMIT);
            axg_launch_rekey(P, N_SM * 8, s);
            axg_launch_emit(P, 0, s);
            launches += 2;
            c->b_chunked = count_mode;
        }
        if (count_mode) {
            prof.mark(AXG_K_SCAN);
            axg_launch_cell_scan(P, N_SM * 4, s);
            prof.mark(AXG_K_PLACE);
            axg_launch_place(P, N_SM * 8, s);
            prof.mark(AXG_K_SETTLE);
            axg_launch_settle(P, N_SM * 8, 0, s);
            launches += 3;
            c->cnt_dirty = false;
            c->kp_pending = true;
        } else {
            c->kp_pending = false;
            prof.mark(AXG_K_SORT);
            for (int q = 0; q < P.n_pass; ++q) axg_launch_sort_pass(P, q, N_SM * 2, s);
            prof.mark(AXG_K_REORDER);
            axg_launch_reorder(P, N_SM * 8, c->max_particles > AXG_REORDER_WIDE_ABOVE ? 1 : 0, s);
            launches += P.n_pass + 1;
        }
        c->p1_pending = false;
    }
    cudaStream_t sc = s;  // stream of the cone kernels
    if (overlap) {
        cudaEventRecord(c->ev_bin, s);
        cudaStreamWaitEvent(c->side, c->ev_bin, 0);
        sc = c->side;
    }
    if ((mask & AXG_PHASE_SENSE) && P.n_cones) {
        prof.mark(AXG_K_SENSE);
        axg_launch_sense(P, sc);
        launches += 1;
    }
    bool committed = false;
    if ((mask & AXG_PHASE_ADVANCE) && P.n_cones) {
        prof.mark(AXG_K_ADVANCE);
        committed = (mask & AXG_PHASE_COMMIT) != 0;  // O10 rides in the last block of k_advance
        axg_launch_advance(P, committed ? 1 : 0, sc);
        launches += 1;
    }
    if ((mask & AXG_PHASE_CONNECT) && P.n_cones && P.conn_thr > 0.0f) {  // reading A-28: after O9, before the next step
        axg_launch_connect(P, sc);
        launches += 1;
    }
    if (overlap) {
        cudaEventRecord(c->ev_adv, c->side);
        c->adv_pending = true;
    }
    if ((mask & AXG_PHASE_COMMIT) && !committed) {
        prof.mark(AXG_K_COMMIT);
        axg_launch_commit(P, 1, s);
        launches += 1;
    } else if (committed && !(mask & AXG_PHASE_DIFFUSE) && !no_realign) {  // phase calls: keep P1's step index aligned
        axg_launch_commit(P, 0, sc);
        launches += 1;
    }
    return launches;
}

// One step as axg_step(n > 1) orders it: [P3..P5 of the PREVIOUS step on the side stream || P1 of this step] -> P2 of this
// step (which rewrites what P3 reads, hence the join before it).  Without cones: P1 -> P2 -> commit.  Everything a step
// needs beyond the parameter block lives in device memory (AxgDev), so the unit is the same for every step and can be
// replayed as a CUDA graph.
int enqueue_unit(axg_ctx* c, cudaStream_t s, bool prev_cones) {
    const AxgParams& P = c->P;
    const bool count_mode = P.bin_mode == AXG_BIN_COUNT_D;
    int launches = 0;
    if (prev_cones) {
        cudaEventRecord(c->ev_bin, s);
        cudaStreamWaitEvent(c->side, c->ev_bin, 0);
        axg_launch_sense(P, c->side);
        axg_launch_advance(P, 1, c->side);  // O10 rides in its last block
        launches += 2;
        if (P.conn_thr > 0.0f) {
            axg_launch_connect(P, c->side);
            launches += 1;
        }
        cudaEventRecord(c->ev_adv, c->side);
    }
    axg_launch_diffuse(P, N_SM * 4, s);
    if (prev_cones) cudaStreamWaitEvent(s, c->ev_adv, 0);
    if (count_mode) {
        axg_launch_cell_scan(P, N_SM * 4, s);
        axg_launch_place(P, N_SM * 8, s);
        axg_launch_settle(P, N_SM * 8, 0, s);
        launches += 4;
    } else {
        for (int q = 0; q < P.n_pass; ++q) axg_launch_sort_pass(P, q, N_SM * 2, s);
        axg_launch_reorder(P, N_SM * 8, c->max_particles > AXG_REORDER_WIDE_ABOVE ? 1 : 0, s);
        launches += P.n_pass + 2;
    }
    if (!P.n_cones) {
        axg_launch_commit(P, 1, s);
        launches += 1;
    }
    return launches;
}

// n whole steps through the graph of one unit.  Returns the number of kernel launches, or -1 when capture failed (the
// caller then falls back to plain enqueueing; the stream is left unharmed).
constexpr uint32_t AXG_GRAPH_MIN_STEPS = 4;
long long enqueue_steps_graph(axg_ctx* c, uint32_t n) {
    const bool cones = c->P.n_cones > 0;
    // the legacy default stream (torch's default) cannot be captured: the steps then run on a stream of the ctx's own,
    // forked from and joined back into the caller's stream with two events
    cudaStream_t s = c->stream;
    const bool detour = s == nullptr || s == cudaStreamLegacy;
    if (detour) {
        if (!c->gstream) {
            if (cudaStreamCreateWithFlags(&c->gstream, cudaStreamNonBlocking) != cudaSuccess ||
                cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) {
                cudaGetLastError();
                return -1;
            }
        }
        s = c->gstream;
    }
    if (c->graph_exec && (std::memcmp(&c->graph_P, &c->P, sizeof(AxgParams)) != 0 || c->graph_stream != s ||
                          c->graph_cones != cones)) {
        cudaGraphExecDestroy(c->graph_exec);
        c->graph_exec = nullptr;
    }
    int unit_launches = 0;
    if (!c->graph_exec) {
        cudaGraph_t g = nullptr;
        if (cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return -1; }
        unit_launches = enqueue_unit(c, s, cones);
        if (cudaStreamEndCapture(s, &g) != cudaSuccess || !g) { cudaGetLastError(); return -1; }
        const cudaError_t e = cudaGraphInstantiate(&c->graph_exec, g, 0);
        cudaGraphDestroy(g);
        if (e != cudaSuccess) { cudaGetLastError(); c->graph_exec = nullptr; return -1; }
        std::memcpy(&c->graph_P, &c->P, sizeof(AxgParams));
        c->graph_stream = s;
        c->graph_cones = cones;
    } else {
        unit_launches = (c->P.bin_mode == AXG_BIN_COUNT_D ? 4 : c->P.n_pass + 2) +
                        (cones ? 2 + (c->P.conn_thr > 0.0f ? 1 : 0) : 1);
    }
    if (detour) {
        cudaEventRecord(c->ev_fork, c->stream);
        cudaStreamWaitEvent(s, c->ev_fork, 0);
    }
    if (c->cnt_dirty) cudaMemsetAsync(c->d_cnt, 0, c->cells_padded() * sizeof(uint32_t), s);
    long long launches = 0;
    uint32_t first_graph_step = 0;
    if (cones) {  // the first step has no previous cones to run beside its P1
        launches += enqueue_unit(c, s, false);
        first_graph_step = 1;
    }
    for (uint32_t i = first_graph_step; i < n; ++i) cudaGraphLaunch(c->graph_exec, s);
    launches += (long long)(n - first_graph_step) * unit_launches;
    if (cones) {  // P3..P5 of the last step
        axg_launch_sense(c->P, s);
        axg_launch_advance(c->P, 1, s);
        launches += 2;
        if (c->P.conn_thr > 0.0f) {
            axg_launch_connect(c->P, s);
            launches += 1;
        }
    }
    if (detour) {
        cudaEventRecord(c->ev_join, s);
        cudaStreamWaitEvent(c->stream, c->ev_join, 0);
    }
    c->cnt_dirty = false;
    c->p1_pending = false;
    c->b_chunked = c->P.bin_mode == AXG_BIN_COUNT_D;
    c->kp_pending = c->b_chunked;
    return launches;
}

void finish_prof(axg_ctx* c, Prof& prof) {
    if (!prof.on) return;
    for (int k = 0; k < AXG_KERNEL_COUNT; ++k) c->ktimes[k] = 0.f;
    for (size_t i = 0; i + 1 < prof.used; ++i) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, c->prof_events[i], c->prof_events[i + 1]);
        if (prof.tags[i] >= 0) c->ktimes[prof.tags[i]] += ms;
    }
}

// host-side pre-checks from device counters: nothing is enqueued when they fail
int capacity_check(axg_ctx* c, uint32_t n, bool diffuse, bool advance, AxgDev* h) {
    const bool census = advance && c->n_cones;
    if (census) {  // longest active polyline, on the stream ahead of the one read below: one synchronisation, not two
        CU(c, cudaMemsetAsync(&((AxgDev*)c->d_dev)->cone_census[0], 0, 5 * sizeof(uint32_t), c->stream));
        axg_launch_census(c->P, c->stream);
    }
    int rc = read_dev(c, h);
    if (rc) return rc;
    if (diffuse && (uint64_t)h->n_live + (uint64_t)n * owned_rate(c) > c->max_particles)
        return fail(c, AXG_ECAPACITY, "particle capacity would overflow");
    if (census && h->cone_census[0] && (uint64_t)h->cone_census[3] + n > (uint64_t)c->max_segments + 1)
        return fail(c, AXG_ECAPACITY, "polyline capacity would overflow");
    return AXG_OK;
}

// The device error word, read after a synchronisation: report it ONCE and clear it, so that a context whose capacity
// has been raised (or whose particles have been replaced) works again.  Bits: 1 particle capacity, 2 polyline
// capacity (both: the step that hit them dropped its emission / its append -- the state is no longer the one an
// unbounded run would have), 4 a loaded particle outside the domain reached AXG_PHASE_BIN (k_rekey).
int report_dev_err(axg_ctx* c, const AxgDev& h) {
    if (!h.err) return AXG_OK;
    cudaMemsetAsync(&((AxgDev*)c->d_dev)->err, 0, sizeof(uint32_t), c->stream);
    cudaStreamSynchronize(c->stream);
    char msg[160];
    std::snprintf(msg, sizeof msg,
                  "device error word 0x%x (1 = particle capacity, 2 = polyline capacity, 4 = particle outside the domain); "
                  "the state is undefined: reload it", h.err);
    return fail(c, (h.err & 3u) ? AXG_ECAPACITY : AXG_EINVAL, msg);
}

int after_sync(axg_ctx* c, const char* what) {
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, what);
    return AXG_OK;
}

}  // namespace

// ============================================ exported ABI ===================================================

AXG_API int axg_set_allocator(axg_alloc_fn alloc, axg_free_fn free_, void* user) {
    if ((alloc == nullptr) != (free_ == nullptr)) return AXG_EINVAL;
    g_alloc = alloc; g_free = free_; g_alloc_user = user;
    return AXG_OK;
}

AXG_API int axg_create(const axg_grid* grid, float D, uint32_t emission, float radius, float speed, float noise,
                       uint64_t seed, axg_ctx** out) {
    if (!grid || !out) return fail(nullptr, AXG_EINVAL, "null argument");
    if (grid->nx == 0 || grid->ny == 0 || grid->nz == 0) return fail(nullptr, AXG_EINVAL, "empty grid");
    if ((double)grid->nx * grid->ny * grid->nz >= 4294967296.0) return fail(nullptr, AXG_EINVAL, "cells >= 2^32");
    if (!(D >= 0.0f) || !(radius >= 1.0f && radius <= 8.0f) || !(speed > 0.0f) || !(noise >= 0.0f) ||
        !std::isfinite(D) || !std::isfinite(speed) || !std::isfinite(noise))
        return fail(nullptr, AXG_EINVAL, "bad D / radius / speed / noise");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, AXG_ECUDA, "no CUDA device: this library has no CPU fallback");
    }
    axg_ctx* c = new axg_ctx();
    c->grid = *grid;
    c->D = D; c->emission = emission; c->radius = radius; c->speed = speed; c->noise = noise; c->seed = seed;
    std::memset(&c->P, 0, sizeof(c->P));
    c->P.single_species = -1;
    *out = c;
    return AXG_OK;
}

AXG_API void axg_destroy(axg_ctx* c) {
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    free_particles(c);
    free_cones(c);
    dev_free(c->d_cnt); dev_free(c->d_scan_state);
    dev_free(c->d_dev); dev_free(c->d_cell_lo); dev_free(c->d_src); dev_free(c->d_src_id_prefix);
    dev_free(c->d_src_emit_prefix); dev_free(c->d_stencil);
    for (cudaEvent_t e : c->prof_events) cudaEventDestroy(e);
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->gstream) cudaStreamDestroy(c->gstream);
    if (c->ev_bin) cudaEventDestroy(c->ev_bin);
    if (c->ev_adv) cudaEventDestroy(c->ev_adv);
    if (c->side) cudaStreamDestroy(c->side);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    delete c;
}

AXG_API const char* axg_last_error(const axg_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }

AXG_API int axg_set_stream(axg_ctx* c, void* stream) {
    if (!c) return AXG_EINVAL;
    cudaStreamSynchronize(c->stream);
    c->stream = (cudaStream_t)stream;
    return AXG_OK;
}

AXG_API int axg_set_shard(axg_ctx* c, uint32_t rank, uint32_t world) {
    if (!c || world == 0 || rank >= world) return fail(c, AXG_EINVAL, "bad shard");
    c->shard_rank = rank; c->shard_world = world;
    c->P.sharded = world > 1 ? 1 : 0;
    return upload_sources(c);
}

AXG_API int axg_set_binning(axg_ctx* c, int mode) {
    if (!c || (mode != AXG_BIN_AUTO && mode != AXG_BIN_RADIX && mode != AXG_BIN_COUNT)) return fail(c, AXG_EINVAL, "bad binning mode");
    if (c->cnt_dirty) return fail(c, AXG_ESTATE, "a step is half done (P1 without P2)");
    c->bin_request = mode;
    return c->particles_allocated ? resolve_binning(c) : AXG_OK;
}

AXG_API int axg_get_binning(axg_ctx* c, int* mode) {
    if (!c || !mode) return fail(c, AXG_EINVAL, "null argument");
    const int rc = ensure_particles(c);
    if (rc) return rc;
    *mode = c->P.bin_mode == AXG_BIN_COUNT_D ? AXG_BIN_COUNT : AXG_BIN_RADIX;
    return AXG_OK;
}

AXG_API int axg_set_steering(axg_ctx* c, int mode, float gain, float turn) {
    if (!c || (mode != AXG_STEER_VECTOR && mode != AXG_STEER_SNR) || !(gain >= 0.0f) || !std::isfinite(gain) ||
        !(turn > 0.0f) || !(turn < 3.14159265f))
        return fail(c, AXG_EINVAL, "bad steering mode / gain / turn");
    c->P.steer_mode = mode;
    c->P.snr_gain = gain;
    c->P.cos_turn = (float)std::cos((double)turn);
    c->P.sin_turn = (float)std::sin((double)turn);
    return AXG_OK;
}

AXG_API int axg_set_key_order(axg_ctx* c, int order) {
    if (!c || (order != AXG_KEY_LINEAR && order != AXG_KEY_BRICK && order != AXG_KEY_MORTON))
        return fail(c, AXG_EINVAL, "bad key order");
    if (order == c->key_order) return AXG_OK;
    if (c->d_dev) return fail(c, AXG_ESTATE, "the key order must be set directly after axg_create");
    const size_t brick_cells = c->nbx() * c->nby() * ((c->grid.nz + 3) / 4) * 128;
    if (order == AXG_KEY_BRICK && brick_cells >= (1ull << 32)) return fail(c, AXG_EINVAL, "padded key space >= 2^32");
    if (order == AXG_KEY_MORTON && axg_ctx::axis_bits(c->grid.nx) + axg_ctx::axis_bits(c->grid.ny) +
                                       axg_ctx::axis_bits(c->grid.nz) > 31)
        return fail(c, AXG_EINVAL, "padded key space >= 2^32");
    c->key_order = order;
    return AXG_OK;
}

AXG_API int axg_set_sensing(axg_ctx* c, int mode) {
    if (!c || (mode != AXG_SENSE_CELL && mode != AXG_SENSE_PARTICLE && mode != AXG_SENSE_PARTICLE_WEIGHTED))
        return fail(c, AXG_EINVAL, "bad sensing mode");
    c->P.sense_mode = mode;
    c->P.s2 = (float)(c->s2_cells * (mode ? 256 : 1));
    return AXG_OK;
}

AXG_API int axg_add_source(axg_ctx* c, float x, float y, float z, uint8_t species, int8_t polarity, uint32_t rate) {
    if (!c) return AXG_EINVAL;
    if (!inside(c, x, y, z)) return fail(c, AXG_EINVAL, "source outside the domain");
    if (species >= AXG_MAX_SPECIES) return fail(c, AXG_EINVAL, "species >= 4");
    if (polarity != 1 && polarity != -1) return fail(c, AXG_EINVAL, "polarity must be +1 or -1");
    if (c->species_polarity[species] != 0 && c->species_polarity[species] != polarity)
        return fail(c, AXG_EINVAL, "polarity conflict within a species");
    if (c->sources.size() >= AXG_MAX_SOURCES) return fail(c, AXG_EINVAL, "too many sources");
    c->species_polarity[species] = polarity;
    c->sources.push_back(Source{x, y, z, species, polarity, rate ? rate : c->emission});
    return upload_sources(c);
}

AXG_API int axg_place_neurons(axg_ctx* c, const float* xyz, const float* heading, uint32_t n) {
    if (!c || (!xyz && n)) return fail(c, AXG_EINVAL, "null argument");
    if (c->stepped) return fail(c, AXG_ESTATE, "neurons cannot be placed after the first step");
    std::vector<float> hd((size_t)n * 3);
    for (uint32_t i = 0; i < n; ++i) {
        if (!inside(c, xyz[i * 3], xyz[i * 3 + 1], xyz[i * 3 + 2])) return fail(c, AXG_EINVAL, "neuron outside the domain");
        if (heading) {
            const float* h = &heading[i * 3];
            const float l = std::sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
            if (!(l > 0.0f) || !std::isfinite(l)) return fail(c, AXG_EINVAL, "bad heading");
            for (int a = 0; a < 3; ++a) hd[(size_t)i * 3 + a] = h[a] / l;
        } else {  // reading A-20: default +z
            hd[(size_t)i * 3 + 0] = 0.0f; hd[(size_t)i * 3 + 1] = 0.0f; hd[(size_t)i * 3 + 2] = 1.0f;
        }
    }
    int rc = alloc_fixed(c);
    if (rc) return rc;
    rc = alloc_cones(c, n);
    if (rc) return rc;
    if (n == 0) return AXG_OK;
    std::vector<uint32_t> ones(n, 1u);
    CU(c, cudaMemcpyAsync(c->P.cone_pos, xyz, (size_t)n * 12, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(c->P.cone_heading, hd.data(), (size_t)n * 12, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(c->P.poly_len, ones.data(), (size_t)n * 4, cudaMemcpyHostToDevice, c->stream));
    axg_launch_poly_init(c->P, c->stream);
    rc = after_sync(c, "axg_place_neurons");
    return rc ? rc : ensure_soma_grid(c);
}

AXG_API int axg_set_capacity(axg_ctx* c, uint64_t max_particles, uint32_t max_segments) {
    if (!c || max_particles == 0 || max_particles >= 0x3fffff00ull) return fail(c, AXG_EINVAL, "bad capacity");
    int rc = alloc_fixed(c);
    if (rc) return rc;
    AxgDev h;
    rc = read_dev(c, &h);
    if (rc) return rc;
    if (h.n_live > max_particles) return fail(c, AXG_ECAPACITY, "live particles exceed the new capacity");
    if (c->n_cones && max_segments != c->max_segments) {
        std::vector<uint32_t> len(c->n_cones);
        CU(c, cudaMemcpy(len.data(), c->P.poly_len, (size_t)c->n_cones * 4, cudaMemcpyDeviceToHost));
        uint32_t longest = *std::max_element(len.begin(), len.end());
        if (longest > (uint64_t)max_segments + 1) return fail(c, AXG_ECAPACITY, "polylines exceed the new capacity");
        // step-major planes: a different capacity only changes the number of rows
        void* np = dev_alloc(c, poly_bytes(c, max_segments));
        if (!np) return fail(c, AXG_ECUDA, "device allocation failed (polylines)");
        CU(c, cudaMemsetAsync(np, 0, poly_bytes(c, max_segments), c->stream));
        CU(c, cudaMemcpyAsync(np, c->d_poly, std::min(poly_bytes(c, max_segments), poly_bytes(c, c->max_segments)),
                              cudaMemcpyDeviceToDevice, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
        dev_free(c->d_poly);
        c->d_poly = np;
        c->P.poly = (float*)np;
    }
    c->max_segments = max_segments;
    c->P.max_segments = max_segments;
    if (c->particles_allocated && max_particles != c->max_particles) {
        AxgParams NP = c->P;
        std::vector<void*> nb;
        rc = alloc_particles(c, max_particles, NP, nb);
        if (rc) return rc;
        const size_t n = h.n_live;
        if (n) {
            CU(c, cudaMemcpyAsync(NP.A.x, c->P.A.x, n * 4, cudaMemcpyDeviceToDevice, c->stream));
            CU(c, cudaMemcpyAsync(NP.A.y, c->P.A.y, n * 4, cudaMemcpyDeviceToDevice, c->stream));
            CU(c, cudaMemcpyAsync(NP.A.z, c->P.A.z, n * 4, cudaMemcpyDeviceToDevice, c->stream));
            CU(c, cudaMemcpyAsync(NP.A.id, c->P.A.id, n * 4, cudaMemcpyDeviceToDevice, c->stream));
            CU(c, cudaMemcpyAsync(NP.A.species, c->P.A.species, n, cudaMemcpyDeviceToDevice, c->stream));
        }
        CU(c, cudaStreamSynchronize(c->stream));
        free_particles(c);
        c->P = NP;
        c->particle_bufs = nb;
        c->particles_allocated = true;
        c->n_B = 0;
        c->kp_pending = false;
        c->p1_pending = false;
    }
    c->max_particles = max_particles;
    CU(c, cudaMemsetAsync(&((AxgDev*)c->d_dev)->err, 0, sizeof(uint32_t), c->stream));
    return c->particles_allocated ? resolve_binning(c) : AXG_OK;  // AXG_BIN_AUTO depends on the capacity
}

AXG_API int axg_load_particles(axg_ctx* c, const float* x, const float* y, const float* z, const uint8_t* species,
                               const uint32_t* id, uint64_t n, uint32_t next_id, uint32_t step) {
    if (!c || (n && (!x || !y || !z || !species || !id))) return fail(c, AXG_EINVAL, "null argument");
    if (n > c->max_particles) return fail(c, AXG_ECAPACITY, "more particles than capacity");
    // which species occur, and that none is out of range: branch-free so that the host compiler vectorises it (this loop
    // runs over every particle of every axg_load_particles call: 16.6 M bytes at C3)
    uint8_t any = 0, has[AXG_MAX_SPECIES] = {0, 0, 0, 0};
    for (uint64_t i = 0; i < n; ++i) {
        const uint8_t sp = species[i];
        any |= sp;
        has[0] |= (uint8_t)(sp == 0); has[1] |= (uint8_t)(sp == 1); has[2] |= (uint8_t)(sp == 2); has[3] |= (uint8_t)(sp == 3);
    }
    if (any >= AXG_MAX_SPECIES) return fail(c, AXG_EINVAL, "species >= 4");
    uint32_t mask = 0;
    for (int sp = 0; sp < (int)AXG_MAX_SPECIES; ++sp) mask |= has[sp] ? (1u << sp) : 0u;
    int rc = ensure_particles(c);
    if (rc) return rc;
    if (n) {
        CU(c, cudaMemcpyAsync(c->P.A.x, x, n * 4, cudaMemcpyHostToDevice, c->stream));
        CU(c, cudaMemcpyAsync(c->P.A.y, y, n * 4, cudaMemcpyHostToDevice, c->stream));
        CU(c, cudaMemcpyAsync(c->P.A.z, z, n * 4, cudaMemcpyHostToDevice, c->stream));
        CU(c, cudaMemcpyAsync(c->P.A.id, id, n * 4, cudaMemcpyHostToDevice, c->stream));
        CU(c, cudaMemcpyAsync(c->P.A.species, species, n, cudaMemcpyHostToDevice, c->stream));
    }
    AxgDev* d = (AxgDev*)c->d_dev;
    const uint32_t n32 = (uint32_t)n;
    CU(c, cudaMemcpyAsync(&d->n_live, &n32, 4, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(&d->next_id, &next_id, 4, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(&d->step, &step, 4, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(&d->pstep, &step, 4, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemsetAsync(&d->err, 0, sizeof(uint32_t), c->stream));  // a new state: an old capacity hit is history
    CU(c, cudaStreamSynchronize(c->stream));
    c->n_A = n32;
    c->p1_pending = false;  // ... and an unbinned P1 output belongs to the old state
    c->kp_pending = false;  // A is new: nothing of the last P2 may be replayed
    c->loaded_species_mask = mask;
    return upload_sources(c);
}

AXG_API int axg_load_cones(axg_ctx* c, const float* pos, const float* heading, const uint8_t* state,
                           const uint32_t* poly_len, uint32_t n) {
    if (!c || !pos || !heading || !state || !poly_len) return fail(c, AXG_EINVAL, "null argument");
    if (n != c->n_cones) return fail(c, AXG_EINVAL, "cone count differs from the placed count");
    for (uint32_t i = 0; i < n; ++i)
        if (poly_len[i] == 0 || poly_len[i] > c->max_segments + 1) return fail(c, AXG_EINVAL, "bad poly_len");
    if (n == 0) return AXG_OK;
    CU(c, cudaMemcpyAsync(c->P.cone_pos, pos, (size_t)n * 12, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(c->P.cone_heading, heading, (size_t)n * 12, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(c->P.cone_state, state, (size_t)n, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(c->P.poly_len, poly_len, (size_t)n * 4, cudaMemcpyHostToDevice, c->stream));
    axg_launch_poly_init(c->P, c->stream);
    return after_sync(c, "axg_load_cones");
}

AXG_API int axg_step(axg_ctx* c, uint32_t n) {
    if (!c) return AXG_EINVAL;
    int rc = ensure_particles(c);
    if (rc) return rc;
    AxgDev h;
    rc = capacity_check(c, n, true, true, &h);
    if (rc) return rc;
    if (!c->ev0) {
        CU(c, cudaEventCreate(&c->ev0));
        CU(c, cudaEventCreate(&c->ev1));
    }
    const unsigned long long ps0 = h.particle_steps;
    Prof prof{c, c->profile_next};
    c->profile_next = false;
    uint64_t launches = 0;
    // With cones and no per-kernel profiling, P3..P5 of step t overlap k_diffuse of step t+1 (they share nothing:
    // P1 draws its step index from AxgDev::pstep, P3..P5 commit AxgDev::step).
    const bool overlap = c->n_cones > 0 && !prof.on && n > 1;
    if (overlap && !c->side) {
        CU(c, cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking));
        CU(c, cudaEventCreateWithFlags(&c->ev_bin, cudaEventDisableTiming));
        CU(c, cudaEventCreateWithFlags(&c->ev_adv, cudaEventDisableTiming));
    }
    CU(c, cudaEventRecord(c->ev0, c->stream));
    long long graphed = -1;
    if (!prof.on && n >= AXG_GRAPH_MIN_STEPS && (overlap || c->n_cones == 0))
        graphed = enqueue_steps_graph(c, n);
    if (graphed >= 0) launches = (uint64_t)graphed;
    else
        for (uint32_t i = 0; i < n; ++i) launches += enqueue_phases(c, AXG_PHASE_ALL | AXG_PHASE_CONNECT, prof, overlap);
    if (c->adv_pending) {  // join: the ctx stream waits for the last step's cones
        CU(c, cudaStreamWaitEvent(c->stream, c->ev_adv, 0));
        c->adv_pending = false;
    }
    prof.mark(-1);
    CU(c, cudaEventRecord(c->ev1, c->stream));
    c->stepped = true;
    rc = read_dev(c, &h);  // the one synchronisation of the call: the copy is queued behind the last kernel
    if (rc) return rc;
    {
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(c, e, "axg_step");
    }
    finish_prof(c, prof);
    cudaEventElapsedTime(&c->last_ms, c->ev0, c->ev1);
    c->last_launches = launches;
    c->last_particle_steps = h.particle_steps - ps0;
    c->n_A = c->n_B = h.n_live;
    return report_dev_err(c, h);
}

AXG_API int axg_check_capacity(axg_ctx* c, uint32_t n) {
    if (!c) return AXG_EINVAL;
    int rc = ensure_particles(c);
    if (rc) return rc;
    AxgDev h;
    rc = capacity_check(c, n, true, true, &h);
    if (rc) return rc;
    c->last_launches = 0;            // the enqueue loop that follows is accounted like one axg_step call
    c->ps0 = h.particle_steps;
    return AXG_OK;
}

AXG_API int axg_enqueue_phase(axg_ctx* c, uint32_t mask) {
    if (!c || (mask & ~(uint32_t)(AXG_PHASE_ALL | AXG_PHASE_CONNECT))) return fail(c, AXG_EINVAL, "bad phase mask");
    int rc = ensure_particles(c);
    if (rc) return rc;
    Prof prof{c, false};
    c->last_launches += (uint64_t)enqueue_phases(c, mask, prof);
    c->stepped = true;
    return AXG_OK;
}

AXG_API int axg_enqueue_phase_on(axg_ctx* c, uint32_t mask, void* stream, int overlapped) {
    if (!c || (mask & ~(uint32_t)(AXG_PHASE_ALL | AXG_PHASE_CONNECT))) return fail(c, AXG_EINVAL, "bad phase mask");
    int rc = ensure_particles(c);
    if (rc) return rc;
    Prof prof{c, false};
    c->last_launches += (uint64_t)enqueue_phases(c, mask, prof, false, (cudaStream_t)stream, true, overlapped != 0);
    c->stepped = true;
    return AXG_OK;
}

// FNV-1a over the kernel parameter block: everything a captured launch bakes in (pointers, sizes, modes)
AXG_API int axg_params_fingerprint(axg_ctx* c, uint64_t* fp) {
    if (!c || !fp) return AXG_EINVAL;
    const int rc = ensure_particles(c);
    if (rc) return rc;
    uint64_t h = 1469598103934665603ull;
    const unsigned char* b = reinterpret_cast<const unsigned char*>(&c->P);
    for (size_t i = 0; i < sizeof(AxgParams); ++i) h = (h ^ b[i]) * 1099511628211ull;
    *fp = h;
    return AXG_OK;
}

AXG_API int axg_sync(axg_ctx* c) {
    if (!c) return AXG_EINVAL;
    int rc = after_sync(c, "axg_sync");
    if (rc) return rc;
    if (!c->d_dev) return AXG_OK;
    AxgDev h;
    rc = read_dev(c, &h);
    if (rc) return rc;
    c->n_A = c->n_B = h.n_live;
    c->last_particle_steps = h.particle_steps - c->ps0;
    return report_dev_err(c, h);
}

AXG_API int axg_step_phase(axg_ctx* c, uint32_t mask) {
    if (!c || (mask & ~(uint32_t)(AXG_PHASE_ALL | AXG_PHASE_CONNECT))) return fail(c, AXG_EINVAL, "bad phase mask");
    int rc = ensure_particles(c);
    if (rc) return rc;
    AxgDev h;
    rc = capacity_check(c, 1, (mask & AXG_PHASE_DIFFUSE) != 0, (mask & AXG_PHASE_ADVANCE) != 0, &h);
    if (rc) return rc;
    Prof prof{c, false};
    enqueue_phases(c, mask, prof);
    c->stepped = true;
    rc = after_sync(c, "axg_step_phase");
    if (rc) return rc;
    rc = read_dev(c, &h);
    if (rc) return rc;
    if (mask & AXG_PHASE_DIFFUSE) c->n_B = h.n_live;
    if (mask & AXG_PHASE_BIN) c->n_A = c->n_B = h.n_live;
    return report_dev_err(c, h);
}

namespace {

// copy `n` elements of `elem` bytes from device memory to dst, with the ESMALL protocol of axg_read_state
int copy_out(axg_ctx* c, const void* dsrc, size_t n, size_t elem, void* dst, size_t dst_bytes, size_t* n_elems) {
    if (n_elems) *n_elems = n;
    if (dst == nullptr && dst_bytes == 0) return AXG_OK;
    if (dst == nullptr || dst_bytes < n * elem) return fail(c, AXG_ESMALL, "destination too small");
    if (n) {
        CU(c, cudaMemcpyAsync(dst, dsrc, n * elem, cudaMemcpyDeviceToHost, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
    }
    return AXG_OK;
}

// fields that are produced by a small export kernel into a scratch buffer first
template <class Launch>
int export_out(axg_ctx* c, size_t n, size_t elem, void* dst, size_t dst_bytes, size_t* n_elems, Launch launch) {
    if (n_elems) *n_elems = n;
    if (dst == nullptr && dst_bytes == 0) return AXG_OK;
    if (dst == nullptr || dst_bytes < n * elem) return fail(c, AXG_ESMALL, "destination too small");
    if (n == 0) return AXG_OK;
    void* tmp = dev_alloc(c, n * elem);
    if (!tmp) return fail(c, AXG_ECUDA, "device allocation failed (export scratch)");
    launch(tmp);
    cudaError_t e = cudaMemcpyAsync(dst, tmp, n * elem, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    dev_free(tmp);
    if (e != cudaSuccess) return cuda_fail(c, e, "export");
    return AXG_OK;
}

}  // namespace

AXG_API int axg_read_state(axg_ctx* c, uint32_t field, void* dst, size_t dst_bytes, size_t* n_elems) {
    if (!c) return AXG_EINVAL;
    if (field >= AXG_FIELD_COUNT) return fail(c, AXG_EINVAL, "unknown field");
    int rc = alloc_fixed(c);
    if (rc) return rc;
    const AxgParams& P = c->P;
    const bool have_p = c->particles_allocated;
    const size_t nA = have_p ? c->n_A : 0, nB = have_p ? c->n_B : 0, C = c->n_cones;
    switch (field) {
        case AXG_COUNTERS: {
            if (n_elems) *n_elems = 9;
            if (dst == nullptr && dst_bytes == 0) return AXG_OK;
            if (dst == nullptr || dst_bytes < 72) return fail(c, AXG_ESMALL, "destination too small");
            CU(c, cudaMemsetAsync(&((AxgDev*)c->d_dev)->cone_census[0], 0, 5 * sizeof(uint32_t), c->stream));
            axg_launch_census(P, c->stream);
            AxgDev h;
            rc = read_dev(c, &h);
            if (rc) return rc;
            const uint64_t v[9] = {h.step, h.n_live, h.next_id, h.emitted, h.absorbed,
                                   h.cone_census[0], h.cone_census[1], h.cone_census[2], h.n_connected};
            std::memcpy(dst, v, 72);
            return AXG_OK;
        }
        case AXG_PART_X: return copy_out(c, P.A.x, nA, 4, dst, dst_bytes, n_elems);
        case AXG_PART_Y: return copy_out(c, P.A.y, nA, 4, dst, dst_bytes, n_elems);
        case AXG_PART_Z: return copy_out(c, P.A.z, nA, 4, dst, dst_bytes, n_elems);
        case AXG_PART_SPECIES: return copy_out(c, P.A.species, nA, 1, dst, dst_bytes, n_elems);
        case AXG_PART_ID: return copy_out(c, P.A.id, nA, 4, dst, dst_bytes, n_elems);
        case AXG_KEYS_SORTED:
        case AXG_PERM:
            if (c->kp_pending) {  // count binning stores neither on the path: derive them now (see k_settle)
                axg_launch_settle(P, N_SM * 8, 1, c->stream);
                c->kp_pending = false;
            }
            if (field == AXG_PERM)
                return export_out(c, nB, 4, dst, dst_bytes, n_elems,
                                  [&](void* t) { axg_launch_perm_export(P, c->b_chunked ? 1 : 0, (uint32_t*)t, c->stream); });
            return copy_out(c, have_p ? P.skey[P.final_buf] : nullptr, nB, 4, dst, dst_bytes, n_elems);
        case AXG_CELL_START:
            return export_out(c, c->cells(), 4, dst, dst_bytes, n_elems,
                              [&](void* t) { axg_launch_cell_export(P, (uint32_t*)t, nullptr, c->stream); });
        case AXG_CELL_END:
            return export_out(c, c->cells(), 4, dst, dst_bytes, n_elems,
                              [&](void* t) { axg_launch_cell_export(P, nullptr, (uint32_t*)t, c->stream); });
        case AXG_CONE_POS: return copy_out(c, P.cone_pos, C * 3, 4, dst, dst_bytes, n_elems);
        case AXG_CONE_HEADING: return copy_out(c, P.cone_heading, C * 3, 4, dst, dst_bytes, n_elems);
        case AXG_CONE_STATE: return copy_out(c, P.cone_state, C, 1, dst, dst_bytes, n_elems);
        case AXG_CONE_COUNTS:
            return export_out(c, C * AXG_MAX_SPECIES, 8, dst, dst_bytes, n_elems,
                              [&](void* t) { axg_launch_sense_export(P, (long long*)t, nullptr, c->stream); });
        case AXG_CONE_MOMENT:
            return export_out(c, C * AXG_MAX_SPECIES * 3, 8, dst, dst_bytes, n_elems,
                              [&](void* t) { axg_launch_sense_export(P, nullptr, (long long*)t, c->stream); });
        case AXG_CONE_GRADIENT: return copy_out(c, P.cone_gradient, C * 3, 4, dst, dst_bytes, n_elems);
        case AXG_POLY_LEN: return copy_out(c, P.poly_len, C, 4, dst, dst_bytes, n_elems);
        case AXG_POLYLINE:
            return export_out(c, C * ((size_t)c->max_segments + 1) * 3, 4, dst, dst_bytes, n_elems,
                              [&](void* t) { axg_launch_poly_export(P, (float*)t, c->stream); });
        case AXG_PRE_X:
        case AXG_PRE_Y:
        case AXG_PRE_Z:
        case AXG_PRE_ID: {
            const int comp = field == AXG_PRE_ID ? 3 : (int)(field - AXG_PRE_X);
            return export_out(c, nB, 4, dst, dst_bytes, n_elems,
                              [&](void* t) { axg_launch_pre_export(P, comp, c->b_chunked ? 1 : 0, t, c->stream); });
        }
        case AXG_PRE_SPECIES:
            return export_out(c, nB, 1, dst, dst_bytes, n_elems,
                              [&](void* t) { axg_launch_pre_export(P, 5, c->b_chunked ? 1 : 0, t, c->stream); });
        case AXG_PRE_KEY:
            return export_out(c, nB, 4, dst, dst_bytes, n_elems,
                              [&](void* t) { axg_launch_pre_export(P, 4, c->b_chunked ? 1 : 0, t, c->stream); });
        case AXG_CONE_TARGET: return copy_out(c, P.cone_target, C, 4, dst, dst_bytes, n_elems);
        case AXG_GRAPH_VA:
            return copy_out(c, c->G.Va, c->graph_built ? C + 1 : 0, 4, dst, dst_bytes, n_elems);
        case AXG_GRAPH_EA:
            return copy_out(c, c->G.Ea, c->graph_built ? c->graph_edges : 0, 4, dst, dst_bytes, n_elems);
        case AXG_BFS_LEVEL:
            return copy_out(c, c->G.C, c->bfs_done ? C : 0, 4, dst, dst_bytes, n_elems);
        default: return fail(c, AXG_EINVAL, "unknown field");
    }
}

// ---- connection formation, adjacency list, BFS (readings A-28..A-30) -------------------
namespace {

// the soma grid: cubic cells of 2^shift unit cells, edge >= reach, at most 2^21 cells; built once (somata do not move)
int ensure_soma_grid(axg_ctx* c) {
    if (c->soma_grid_built || c->n_cones == 0 || !(c->P.conn_thr > 0.0f)) return AXG_OK;
    const float reach = c->r_cone + c->r_soma;
    uint32_t shift = 0;
    while ((float)(1u << shift) < reach) ++shift;
    auto dim = [&](uint32_t n) { return (n + (1u << shift) - 1u) >> shift; };
    while ((uint64_t)dim(c->grid.nx) * dim(c->grid.ny) * dim(c->grid.nz) > (1ull << 21)) ++shift;
    const uint32_t gx = dim(c->grid.nx), gy = dim(c->grid.ny), gz = dim(c->grid.nz), cells = gx * gy * gz;
    free_connect(c);
    void* ptr[4];
    const size_t sizes[4] = {((size_t)cells + 1) * 4, ((size_t)cells + 1) * 4, ((size_t)cells + 1) * 4, (size_t)c->n_cones * 4};
    for (int i = 0; i < 4; ++i) {
        ptr[i] = dev_alloc(c, sizes[i]);
        if (!ptr[i]) return fail(c, AXG_ECUDA, "device allocation failed (soma grid)");
        c->connect_bufs.push_back(ptr[i]);
    }
    c->P.ng_shift = shift; c->P.ngx = gx; c->P.ngy = gy; c->P.ngz = gz;
    c->P.ng_lo = (const uint32_t*)ptr[2];
    c->P.ng_list = (const uint32_t*)ptr[3];
    axg_launch_soma_grid(c->P, (uint32_t*)ptr[0], (uint32_t*)ptr[1], (uint32_t*)ptr[2], (uint32_t*)ptr[3], cells, c->stream);
    c->soma_grid_built = true;
    return after_sync(c, "soma grid");
}

int ensure_graph_bufs(axg_ctx* c) {
    if (!c->graph_bufs.empty()) return AXG_OK;
    const size_t n = c->n_cones;
    const size_t sizes[] = {(n + 1) * 4, (n + 1) * 4, (n + 1) * 4, n * 4 + 4, n * 4 + 4, (n / 33 + 2) * 4, 4, (n + 1) * 4,
                            2 * n * 4 + 4, n * 4 + 4, n + 4, n + 4, n + 4, 4};
    constexpr int NB = 14;
    void* ptr[NB];
    for (int i = 0; i < NB; ++i) {
        ptr[i] = dev_alloc(c, sizes[i]);
        if (!ptr[i]) return fail(c, AXG_ECUDA, "device allocation failed (graph)");
        c->graph_bufs.push_back(ptr[i]);
    }
    AxgGraph& g = c->G;
    g.n = (uint32_t)n;
    g.cnt = (uint32_t*)ptr[0]; g.cursor = (uint32_t*)ptr[1]; g.in_lo = (uint32_t*)ptr[2]; g.in_list = (uint32_t*)ptr[3];
    g.scratch = (uint32_t*)ptr[4]; g.big = (uint32_t*)ptr[5]; g.n_big = (uint32_t*)ptr[6]; g.Va = (uint32_t*)ptr[7];
    g.Ea = (uint32_t*)ptr[8]; g.C = (int32_t*)ptr[9]; g.F = (uint8_t*)ptr[10]; g.Fu = (uint8_t*)ptr[11];
    g.X = (uint8_t*)ptr[12]; g.flag = (uint32_t*)ptr[13];
    return AXG_OK;
}

}  // namespace

AXG_API int axg_set_connect(axg_ctx* c, float r_cone, float r_soma) {
    if (!c || !(r_cone >= 0.0f) || !(r_soma >= 0.0f) || !std::isfinite(r_cone) || !std::isfinite(r_soma) ||
        r_cone + r_soma > 64.0f)
        return fail(c, AXG_EINVAL, "bad radii");
    const float reach = r_cone + r_soma;
    c->r_cone = r_cone; c->r_soma = r_soma;
    c->P.conn_thr = reach > 0.0f ? reach * reach : 0.0f;
    free_connect(c);  // the soma grid depends on the reach
    return ensure_soma_grid(c);
}

AXG_API int axg_load_targets(axg_ctx* c, const uint32_t* target, uint32_t n) {
    if (!c || (!target && n)) return fail(c, AXG_EINVAL, "null argument");
    if (n != c->n_cones) return fail(c, AXG_EINVAL, "cone count differs from the placed count");
    for (uint32_t i = 0; i < n; ++i)
        if (target[i] != 0xffffffffu && (target[i] >= n || target[i] == i)) return fail(c, AXG_EINVAL, "bad target");
    if (n) CU(c, cudaMemcpyAsync(c->P.cone_target, target, (size_t)n * 4, cudaMemcpyHostToDevice, c->stream));
    c->graph_built = c->bfs_done = false;
    return after_sync(c, "axg_load_targets");
}

AXG_API int axg_build_graph(axg_ctx* c, int directed) {
    if (!c) return AXG_EINVAL;
    c->graph_built = c->bfs_done = false;
    c->graph_edges = 0;
    if (c->n_cones == 0) return fail(c, AXG_ESTATE, "no neurons placed");
    int rc = ensure_graph_bufs(c);
    if (rc) return rc;
    c->G.directed = directed ? 1 : 0;
    c->G.target = c->P.cone_target;
    axg_launch_graph_build(c->G, c->stream);
    CU(c, cudaMemcpyAsync(&c->graph_edges, c->G.Va + c->n_cones, 4, cudaMemcpyDeviceToHost, c->stream));
    rc = after_sync(c, "axg_build_graph");
    if (rc) return rc;
    c->graph_built = true;
    return AXG_OK;
}

AXG_API int axg_bfs(axg_ctx* c, uint32_t root) {
    if (!c) return AXG_EINVAL;
    if (!c->graph_built) return fail(c, AXG_ESTATE, "no graph: call axg_build_graph first");
    if (root >= c->n_cones) return fail(c, AXG_EINVAL, "root out of range");
    c->bfs_done = false;
    axg_launch_bfs_init(c->G, root, c->stream);
    for (uint32_t level = 0; level <= c->n_cones; ++level) {   // "repeated until frontier is empty"
        uint32_t more = 0;
        CU(c, cudaMemsetAsync(c->G.flag, 0, 4, c->stream));
        axg_launch_bfs_level(c->G, c->stream);
        CU(c, cudaMemcpyAsync(&more, c->G.flag, 4, cudaMemcpyDeviceToHost, c->stream));
        const int rc = after_sync(c, "axg_bfs");
        if (rc) return rc;
        if (!more) break;
    }
    c->bfs_done = true;
    return AXG_OK;
}

AXG_API int axg_sense_buffer(axg_ctx* c, void** device_ptr, size_t* bytes) {
    if (!c || !device_ptr || !bytes) return AXG_EINVAL;
    *device_ptr = c->n_cones ? (void*)c->P.sense : nullptr;
    *bytes = (size_t)c->n_cones * 16 * sizeof(int32_t);
    return AXG_OK;
}

AXG_API int axg_last_step_stats(axg_ctx* c, float* device_ms, uint64_t* launches, uint64_t* particle_steps) {
    if (!c) return AXG_EINVAL;
    if (device_ms) *device_ms = c->last_ms;
    if (launches) *launches = c->last_launches;
    if (particle_steps) *particle_steps = c->last_particle_steps;
    return AXG_OK;
}

AXG_API int axg_profile_next_step(axg_ctx* c, int enable) {
    if (!c) return AXG_EINVAL;
    c->profile_next = enable != 0;
    return AXG_OK;
}

AXG_API int axg_kernel_times(axg_ctx* c, float* times_ms) {
    if (!c || !times_ms) return AXG_EINVAL;
    std::memcpy(times_ms, c->ktimes, sizeof(c->ktimes));
    return AXG_OK;
}
