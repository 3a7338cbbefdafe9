// axo_oracle.cpp -- the ORACLE: a plain, slow, single-threaded CPU statement of one axon-guidance time step.
//
// TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_1405_3331_b200/, include/) may import, link or
// execute this file; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs do.
// It shares no code, header, table or helper with the CUDA path: its own Philox, std::stable_sort binning,
// grid sensing AND brute-force all-pairs sensing.
//
// What it follows: /root/reference/PAPER.md (P:NNN = line) as completed by BASELINE.json north_star (NS) and the
// readings A-1..A-22 listed in DESIGN.md §3.  The algorithm is written in the order and
// notation of DESIGN.md §3 "O0..O10"; there is no blocking, fusion or reordering.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): T1 Philox known-answer vectors; T1b worked examples;
// T2 moments of the normals; T3 conservation; T4 MSD = 6 D t; T5/T6 closed-form steady state of a point source
// in an absorbing box; T7 Table 1 of the paper; T8 binning invariants vs numpy stable argsort; T9 grid sensing ==
// brute force + planted linear gradient; T10 advance geometry and E[theta^2] = 2 noise^2; T11 append; T13 the
// fixed-turn steering rule (A-25); T14 per-particle sensing (A-26): worked example, reduction to the per-cell rule,
// closed forms for a planted linear density, mirror / translation / order invariants.
// PARITY UNPINNED: the absolute arrival fraction (T12) has no closed form; only GPU-vs-oracle agreement is tested.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC  (oracle/build.py)

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <string>
#include <vector>

#define AXO_API extern "C" __attribute__((visibility("default")))

namespace {

// ---- error codes / enums: restated here on purpose (no shared header with the CUDA path) -------------------
enum { OK = 0, EINVAL_ = -1, ECAPACITY = -2, ESTATE = -3, ESMALL = -5 };
enum { MAX_SPECIES = 4 };
enum { CONE_ACTIVE = 0, CONE_ARRIVED = 1, CONE_EXITED = 2, CONE_CONNECTED = 3 };
enum { PH_DIFFUSE = 1, PH_BIN = 2, PH_SENSE = 4, PH_ADVANCE = 8, PH_COMMIT = 16, PH_CONNECT = 32 };
const uint32_t NO_TARGET = 0xffffffffu;
enum Field {
    F_COUNTERS = 0, F_PART_X, F_PART_Y, F_PART_Z, F_PART_SPECIES, F_PART_ID, F_KEYS_SORTED, F_PERM, F_CELL_START,
    F_CELL_END, F_CONE_POS, F_CONE_HEADING, F_CONE_STATE, F_CONE_COUNTS, F_CONE_MOMENT, F_CONE_GRADIENT,
    F_POLY_LEN, F_POLYLINE, F_PRE_X, F_PRE_Y, F_PRE_Z, F_PRE_SPECIES, F_PRE_ID, F_PRE_KEY, F_CONE_TARGET, F_GRAPH_VA,
    F_GRAPH_EA, F_BFS_LEVEL, F_COUNT
};

// ---- Philox4x32-10 (reading A-2; rationale for a stateless per-thread generator: §5.1) ------------
// Salmon et al. round function: two 32x32->64 multiplies, xor with the neighbouring counter word and the key,
// key bumped by the Weyl constants between rounds.
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {
            k0 += W0;
            k1 += W1;
        }
        const uint64_t p0 = (uint64_t)M0 * c0;
        const uint64_t p1 = (uint64_t)M1 * c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// u32 -> uniform in (0,1), reading A-3: odd integer below 2^24 times 2^-24, exact in fp32, never 0 or 1.
float uniform_from_bits(uint32_t r) { return (float)(((r >> 9) << 1) | 1u) * 0x1p-24f; }

// Three standard normals from one Philox block, reading A-4 (O1): basic Box-Muller evaluated in double,
// each result rounded once to fp32.  z0,z1 share (u0,u1); z2 uses (u2,u3) and only the cosine branch.
void normals3(uint64_t seed, uint32_t entity, uint32_t t, uint32_t stream, float z[3], uint32_t r_out[4]) {
    const uint32_t ctr[4] = {entity, t, stream, 0u};
    const uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
    uint32_t r[4];
    philox4x32_10(ctr, key, r);
    const double u0 = uniform_from_bits(r[0]), u1 = uniform_from_bits(r[1]);
    const double u2 = uniform_from_bits(r[2]), u3 = uniform_from_bits(r[3]);
    const double two_pi = 6.283185307179586476925286766559;
    const double rho1 = std::sqrt(-2.0 * std::log(u0));
    const double rho2 = std::sqrt(-2.0 * std::log(u2));
    z[0] = (float)(rho1 * std::cos(two_pi * u1));
    z[1] = (float)(rho1 * std::sin(two_pi * u1));
    z[2] = (float)(rho2 * std::cos(two_pi * u3));
    if (r_out) std::memcpy(r_out, r, sizeof(r));
}

struct Source {
    float x, y, z;
    uint8_t species;
    int8_t polarity;
    uint32_t rate;
};

struct SoA {
    std::vector<float> x, y, z;
    std::vector<uint8_t> species;
    std::vector<uint32_t> id;
    size_t size() const { return x.size(); }
    void clear() { x.clear(); y.clear(); z.clear(); species.clear(); id.clear(); }
    void push(float px, float py, float pz, uint8_t s, uint32_t i) {
        x.push_back(px); y.push_back(py); z.push_back(pz); species.push_back(s); id.push_back(i);
    }
};

}  // namespace

struct axo_ctx {
    uint32_t nx, ny, nz;
    float D, radius, speed, noise;
    uint32_t emission;
    uint64_t seed;
    uint64_t max_particles = 1ull << 20;
    uint32_t max_segments = 1024;
    uint32_t shard_rank = 0, shard_world = 1;
    // steering rule of P4: 0 = vector addition (north_star), 1 = fixed turn by the sign of N(SNR, 1) (Eq. 5)
    int steer_mode = 0;
    float snr_gain = 1.0f, cos_turn = 1.0f, sin_turn = 0.0f;
    uint32_t n_stencil = 0;  // |N_R|, filled by axo_set_steering
    // sensing rule of P3: 0 = per cell (north_star, O7), 1 = per particle, 2 = per particle with distance weighting
    // (section 5.3; reading A-26)
    int sense_mode = 0;
    int64_t moment_scale() const { return sense_mode == 0 ? 1 : 256; }  // units of M: cells (mode 0), 1/256 cell

    std::vector<Source> sources;
    int8_t species_polarity[MAX_SPECIES] = {0, 0, 0, 0};

    SoA A;  // "sorted order" array: input of P1, output of P2
    SoA B;  // pre-sort array: output of P1
    std::vector<uint32_t> key, keys_sorted, perm, cell_start, cell_end;

    uint32_t step = 0, next_id = 0;
    uint64_t n_live = 0;  // size of the live array (B between P1 and P2, else A)
    uint64_t emitted = 0, absorbed = 0;
    bool stepped = false;

    // cones
    std::vector<float> cone_pos, cone_heading, cone_gradient;  // C*3
    std::vector<uint8_t> cone_state;
    std::vector<int64_t> cone_counts;  // C*MAX_SPECIES
    std::vector<int64_t> cone_moment;  // C*MAX_SPECIES*3
    std::vector<uint32_t> poly_len;
    std::vector<float> poly;  // C*(max_segments+1)*3 neuron-major

    // connection formation (section 3.3, section 3.4; DESIGN.md readings
    // A-28..A-30): target[c] = the neuron whose soma cone c has connected to (NO_TARGET: none), the adjacency list in
    // the paper's compact form (Va = heads, Ea = edges) and the BFS levels of Fig. 5
    bool connect_on = false;
    float r_cone = 0.0f, r_soma = 0.0f;
    std::vector<uint32_t> target;
    std::vector<uint32_t> Va, Ea;
    std::vector<int32_t> bfs_level;

    std::string err;
    // cell order ("a Z-order curve ... potential optimization"; reading A-27):
    // 0 = linear, x fastest (north_star); 1 = bricks of 8 x 4 x 4 cells, bricks in linear order (x fastest), cells inside
    // a brick in linear order (x fastest): key = brick * 128 + (z & 3) * 32 + (y & 3) * 8 + (x & 7).  The key space covers
    // the grid padded to whole bricks.
    // 2 = Z-order (Morton) curve, the order P:263 names (reading A-31): the bits of ix, iy, iz interleaved from
    // the least significant up, x first; a coordinate that has run out of bits (its axis needs fewer than the others)
    // drops out of the rotation.  The key space is the grid padded to powers of two.
    int key_order = 0;
    static int axis_bits(uint32_t n) {
        int b = 0;
        while ((1u << b) < n) ++b;
        return b;
    }
    size_t cells() const {
        if (key_order == 0) return (size_t)nx * ny * nz;
        if (key_order == 2) return (size_t)1 << (axis_bits(nx) + axis_bits(ny) + axis_bits(nz));
        return (size_t)((nx + 7) / 8) * ((ny + 3) / 4) * ((nz + 3) / 4) * 128;
    }
    uint32_t key_of_cell(uint32_t ix, uint32_t iy, uint32_t iz) const {
        if (key_order == 0) return (iz * ny + iy) * nx + ix;
        if (key_order == 2) {
            const int nb[3] = {axis_bits(nx), axis_bits(ny), axis_bits(nz)};
            const uint32_t v[3] = {ix, iy, iz};
            uint32_t key = 0;
            int out = 0;
            for (int bit = 0; bit < 32; ++bit)          // bit `bit` of x, then of y, then of z, for the axes that have it
                for (int a = 0; a < 3; ++a)
                    if (bit < nb[a]) key |= ((v[a] >> bit) & 1u) << out++;
            return key;
        }
        const uint32_t nbx = (nx + 7) / 8, nby = (ny + 3) / 4;
        const uint32_t brick = ((iz / 4) * nby + (iy / 4)) * nbx + (ix / 8);
        return brick * 128 + (iz % 4) * 32 + (iy % 4) * 8 + (ix % 8);
    }
    size_t n_cones() const { return cone_state.size(); }
};

namespace {

thread_local std::string g_create_err;

int fail(axo_ctx* c, int code, const std::string& msg) {
    if (c) c->err = msg; else g_create_err = msg;
    return code;
}

bool inside(const axo_ctx* c, float x, float y, float z) {
    // reading A-7: half-open box, fp32 compares against (float)n
    return x >= 0.0f && x < (float)c->nx && y >= 0.0f && y < (float)c->ny && z >= 0.0f && z < (float)c->nz;
}

// O3 (reading A-8; "calculateHash", linear id): truncation of non-negative fp32, x fastest.
uint32_t cell_key(const axo_ctx* c, float x, float y, float z) {
    return c->key_of_cell((uint32_t)x, (uint32_t)y, (uint32_t)z);  // linear unless axo_set_key_order (A-27)
}

uint64_t owned_rate(const axo_ctx* c) {
    uint64_t e = 0;
    for (size_t s = 0; s < c->sources.size(); ++s)
        if (s % c->shard_world == c->shard_rank) e += c->sources[s].rate;
    return e;
}

// ---- P1: O0, O1, O2, O3 -----------------------------------------------------------------------------------
void phase_diffuse(axo_ctx* c) {
    const float sigma = (float)std::sqrt(2.0 * (double)c->D);  // O0, reading A-1
    const uint32_t t = c->step;
    c->B.clear();
    const size_t N = c->A.size();
    size_t survivors = 0;
    for (size_t i = 0; i < N; ++i) {  // O1, array order
        float zn[3];
        normals3(c->seed, c->A.id[i], t, 0u, zn, nullptr);
        const float x1 = std::fmaf(sigma, zn[0], c->A.x[i]);
        const float y1 = std::fmaf(sigma, zn[1], c->A.y[i]);
        const float z1 = std::fmaf(sigma, zn[2], c->A.z[i]);
        if (inside(c, x1, y1, z1)) {  // P1b absorbing boundary, end-point test only (A-7)
            c->B.push(x1, y1, z1, c->A.species[i], c->A.id[i]);
            ++survivors;
        }
    }
    // O2 emission (A-5: newborns sit exactly at the source and do not move in their birth step; A-6: survivors in
    // input order, then newborns in (source, j) order).  Sharding: a source that is not owned by
    // this rank consumes its ids but emits nothing.
    uint64_t emitted_here = 0;
    for (size_t s = 0; s < c->sources.size(); ++s) {
        const Source& src = c->sources[s];
        const bool owned = (s % c->shard_world) == c->shard_rank;
        for (uint32_t j = 0; j < src.rate; ++j) {
            const uint32_t id = c->next_id++;  // u32 wrap (A-21)
            if (owned) {
                c->B.push(src.x, src.y, src.z, src.species, id);
                ++emitted_here;
            }
        }
    }
    c->emitted += emitted_here;
    c->absorbed += N - survivors;
    // O3 keys
    const size_t N1 = c->B.size();
    c->key.resize(N1);
    for (size_t i = 0; i < N1; ++i) c->key[i] = cell_key(c, c->B.x[i], c->B.y[i], c->B.z[i]);
    c->n_live = N1;
}

// harness path: take A as the pre-sort array (BIN without DIFFUSE)
void adopt_A_as_presort(axo_ctx* c) {
    c->B = c->A;
    const size_t N1 = c->B.size();
    c->key.resize(N1);
    for (size_t i = 0; i < N1; ++i) c->key[i] = cell_key(c, c->B.x[i], c->B.y[i], c->B.z[i]);
}

// ---- P2: O4, O5, O6 ---------------------------------------------------------------------------------------
void phase_bin(axo_ctx* c) {
    const size_t N1 = c->B.size();
    // O4 (A-9): value = pre-sort index, ties keep pre-sort order.  P:263-265: sort of (cell hash, particle id).
    c->perm.resize(N1);
    std::iota(c->perm.begin(), c->perm.end(), 0u);
    const std::vector<uint32_t>& key = c->key;
    std::stable_sort(c->perm.begin(), c->perm.end(), [&key](uint32_t a, uint32_t b) { return key[a] < key[b]; });
    // O5 reorder ("position and velocity arrays were also sorted")
    c->A.clear();
    c->keys_sorted.resize(N1);
    for (size_t j = 0; j < N1; ++j) {
        const uint32_t p = c->perm[j];
        c->A.push(c->B.x[p], c->B.y[p], c->B.z[p], c->B.species[p], c->B.id[p]);
        c->keys_sorted[j] = key[p];
    }
    c->n_live = N1;
    // O6 (P:265 identifyCellStart and its reverse; A-10: empty cells have start = end = 0)
    c->cell_start.assign(c->cells(), 0u);
    c->cell_end.assign(c->cells(), 0u);
    for (size_t j = 0; j < N1; ++j) {
        const uint32_t k = c->keys_sorted[j];
        if (j == 0 || c->keys_sorted[j - 1] != k) c->cell_start[k] = (uint32_t)j;
        if (j + 1 == N1 || c->keys_sorted[j + 1] != k) c->cell_end[k] = (uint32_t)j + 1u;
    }
}

// ---- P3: O7 (grid form) -----------------------------------------------------------------------------------
int64_t stencil_S2(int r2) {  // S2(R) = sum over the stencil of dx^2 (A-12)
    const int R = 8;
    int64_t s2 = 0;
    for (int dz = -R; dz <= R; ++dz)
        for (int dy = -R; dy <= R; ++dy)
            for (int dx = -R; dx <= R; ++dx)
                if (dx * dx + dy * dy + dz * dz <= r2) s2 += dx * dx;
    return s2;
}

void finish_gradient(axo_ctx* c, size_t cone, int64_t G[3]) {
    G[0] = G[1] = G[2] = 0;
    for (int s = 0; s < MAX_SPECIES; ++s)  // A-13: G = sum_s polarity_s * M_s, int64
        for (int a = 0; a < 3; ++a)
            G[a] += (int64_t)c->species_polarity[s] * c->cone_moment[(cone * MAX_SPECIES + s) * 3 + a];
    const int r2 = (int)std::floor((double)c->radius * (double)c->radius);
    const float s2 = (float)(stencil_S2(r2) * c->moment_scale());
    for (int a = 0; a < 3; ++a) c->cone_gradient[cone * 3 + a] = (float)G[a] / s2;
}

// ---- P3, per-particle rule (section 5.3: "each individual particle that the axon's growth cone detects
// would influence the axon's path"; reading A-26).  The plain definition: every active cone against every
// particle, no grid.  A particle at x is detected by the cone at p iff |x - p|^2 <= R^2, the test taken in fp32 in
// the order written here (a floating-point number decides an integer, so both implementations take the decision in
// the same precision); a detected particle adds its offset from the cone, in fixed point, to the first moment of its
// species:
//    mode 1:  M_s += rint(256 * (x - p))                                  (units of 1/256 cell)
//    mode 2:  M_s += rint(16 * w) * rint(16 * (x - p)),  w = 1 - d^2/R^2  (weight falling with the distance; same units)
// rint = round to nearest, ties to even.  The sums are integers, hence independent of the summation order and
// additive over disjoint particle sets (the sharded loop's all-reduce applies unchanged).
void phase_sense_particles(axo_ctx* c) {
    const float R2 = c->radius * c->radius;
    for (size_t cone = 0; cone < c->n_cones(); ++cone) {
        if (c->cone_state[cone] != CONE_ACTIVE) continue;  // A-16
        const float px = c->cone_pos[cone * 3 + 0], py = c->cone_pos[cone * 3 + 1], pz = c->cone_pos[cone * 3 + 2];
        int64_t* n = &c->cone_counts[cone * MAX_SPECIES];
        int64_t* M = &c->cone_moment[cone * MAX_SPECIES * 3];
        std::fill(n, n + MAX_SPECIES, 0);
        std::fill(M, M + MAX_SPECIES * 3, 0);
        for (size_t j = 0; j < c->A.size(); ++j) {
            const float dx = c->A.x[j] - px, dy = c->A.y[j] - py, dz = c->A.z[j] - pz;
            const float d2 = (dx * dx + dy * dy) + dz * dz;
            if (!(d2 <= R2)) continue;
            const int s = c->A.species[j];
            n[s] += 1;
            if (c->sense_mode == 1) {
                M[s * 3 + 0] += (int64_t)std::nearbyint(dx * 256.0f);
                M[s * 3 + 1] += (int64_t)std::nearbyint(dy * 256.0f);
                M[s * 3 + 2] += (int64_t)std::nearbyint(dz * 256.0f);
            } else {
                const float w = 1.0f - d2 / R2;
                const int64_t wq = (int64_t)std::nearbyint(w * 16.0f);
                M[s * 3 + 0] += wq * (int64_t)std::nearbyint(dx * 16.0f);
                M[s * 3 + 1] += wq * (int64_t)std::nearbyint(dy * 16.0f);
                M[s * 3 + 2] += wq * (int64_t)std::nearbyint(dz * 16.0f);
            }
        }
        int64_t G[3];
        finish_gradient(c, cone, G);
    }
}

void phase_sense(axo_ctx* c) {
    if (c->sense_mode != 0) { phase_sense_particles(c); return; }
    if (c->cell_start.size() != c->cells()) {  // nothing binned yet: all cells empty
        c->cell_start.assign(c->cells(), 0u);
        c->cell_end.assign(c->cells(), 0u);
    }
    const int r2 = (int)std::floor((double)c->radius * (double)c->radius);  // floor(R^2), A-11
    const int R = (int)std::floor((double)c->radius);
    for (size_t cone = 0; cone < c->n_cones(); ++cone) {
        if (c->cone_state[cone] != CONE_ACTIVE) continue;  // A-16: frozen cones skip P3..P5
        const int ci = (int)c->cone_pos[cone * 3 + 0], cj = (int)c->cone_pos[cone * 3 + 1],
                  ck = (int)c->cone_pos[cone * 3 + 2];
        int64_t* n = &c->cone_counts[cone * MAX_SPECIES];
        int64_t* M = &c->cone_moment[cone * MAX_SPECIES * 3];
        std::fill(n, n + MAX_SPECIES, 0);
        std::fill(M, M + MAX_SPECIES * 3, 0);
        for (int dz = -R; dz <= R; ++dz)
            for (int dy = -R; dy <= R; ++dy)
                for (int dx = -R; dx <= R; ++dx) {
                    if (dx * dx + dy * dy + dz * dz > r2) continue;
                    const int x = ci + dx, y = cj + dy, z = ck + dz;
                    if (x < 0 || y < 0 || z < 0 || x >= (int)c->nx || y >= (int)c->ny || z >= (int)c->nz) continue;
                    const size_t cell = c->key_of_cell((uint32_t)x, (uint32_t)y, (uint32_t)z);
                    for (uint32_t j = c->cell_start[cell]; j < c->cell_end[cell]; ++j) {
                        const int s = c->A.species[j];
                        n[s] += 1;
                        M[s * 3 + 0] += dx;
                        M[s * 3 + 1] += dy;
                        M[s * 3 + 2] += dz;
                    }
                }
        int64_t G[3];
        finish_gradient(c, cone, G);
    }
}

// ---- P4 + P5: O8, O9 --------------------------------------------------------------------------------------
void phase_advance(axo_ctx* c) {
    const uint32_t t = c->step;
    const size_t stride = (size_t)(c->max_segments + 1) * 3;
    for (size_t cone = 0; cone < c->n_cones(); ++cone) {
        if (c->cone_state[cone] != CONE_ACTIVE) continue;
        int64_t G[3] = {0, 0, 0};
        for (int s = 0; s < MAX_SPECIES; ++s)
            for (int a = 0; a < 3; ++a)
                G[a] += (int64_t)c->species_polarity[s] * c->cone_moment[(cone * MAX_SPECIES + s) * 3 + a];
        float* h = &c->cone_heading[cone * 3];
        float* p = &c->cone_pos[cone * 3];
        float g[3];
        if (G[0] == 0 && G[1] == 0 && G[2] == 0) {  // A-14 (keep the current direction)
            g[0] = h[0]; g[1] = h[1]; g[2] = h[2];
        } else {
            const float gx = (float)G[0], gy = (float)G[1], gz = (float)G[2];
            const float len = std::sqrt(gx * gx + gy * gy + gz * gz);
            g[0] = gx / len; g[1] = gy / len; g[2] = gz / len;
        }
        float xi[3];
        normals3(c->seed, (uint32_t)cone, t, 1u, xi, nullptr);  // stream 1 = cone noise (A-2)
        if (c->steer_mode == 1) {
            // The paper's first steering rule (Eq. 5; reading A-25): a turn of fixed size delta
            // towards ("right") or away from ("left") the gradient direction, by the sign of a draw from N(SNR, 1),
            //   SNR = gain * mu * sqrt(gamma / (1 + gamma)^3) * sin(phi),
            // gamma = particles per cell in range (background concentration), mu = |g| / gamma (relative gradient per
            // cell, g = G / S2), phi = angle between the heading and the gradient direction.  In 3-D the turn is the
            // rotation of the heading by delta in the plane spanned by heading and gradient.  Nothing in range, G = 0
            // or heading parallel to the gradient: keep the direction.
            int64_t n_all = 0;
            for (int s = 0; s < MAX_SPECIES; ++s) n_all += c->cone_counts[cone * MAX_SPECIES + s];
            const float dot = h[0] * g[0] + h[1] * g[1] + h[2] * g[2];
            float w[3];
            for (int a = 0; a < 3; ++a) w[a] = g[a] - dot * h[a];  // part of the gradient direction orthogonal to h
            const float sinphi = std::sqrt(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
            const bool have_g = !(G[0] == 0 && G[1] == 0 && G[2] == 0);
            if (have_g && n_all > 0 && sinphi > 0.0f) {
                const float gx = (float)G[0], gy = (float)G[1], gz = (float)G[2];
                const float glen = std::sqrt(gx * gx + gy * gy + gz * gz) / (float)(c->moment_scale() * stencil_S2(
                                       (int)std::floor((double)c->radius * (double)c->radius)));
                const float gamma = (float)n_all / (float)c->n_stencil;
                const float mu = glen / gamma;
                const float one = 1.0f + gamma;
                const float snr = c->snr_gain * mu * std::sqrt(gamma / (one * one * one)) * sinphi;
                const float sgn = (snr + xi[0] > 0.0f) ? 1.0f : -1.0f;
                float v[3];
                for (int a = 0; a < 3; ++a) v[a] = c->cos_turn * h[a] + (sgn * c->sin_turn) * (w[a] / sinphi);
                const float vlen = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
                for (int a = 0; a < 3; ++a) h[a] = v[a] / vlen;
            }
        } else {
            float v[3];
            for (int a = 0; a < 3; ++a) v[a] = g[a] + c->noise * xi[a];  // A-15
            const float vlen = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
            if (vlen > 0.0f) {
                for (int a = 0; a < 3; ++a) h[a] = v[a] / vlen;
            } else {
                for (int a = 0; a < 3; ++a) h[a] = g[a];
            }
        }
        for (int a = 0; a < 3; ++a) p[a] = p[a] + c->speed * h[a];  // P:282 fixed distance per step
        // O9 append (a capsule is added at the end of the previous one)
        const uint32_t len = c->poly_len[cone];
        float* dst = &c->poly[cone * stride + (size_t)len * 3];
        dst[0] = p[0]; dst[1] = p[1]; dst[2] = p[2];
        c->poly_len[cone] = len + 1;
        if (!inside(c, p[0], p[1], p[2])) {
            c->cone_state[cone] = CONE_EXITED;  // P:239 "out of the simulation bounds"
        } else {
            for (const Source& s : c->sources) {  // A-16: targets = attractive sources, squared distance
                if (s.polarity != 1) continue;
                const float dx = p[0] - s.x, dy = p[1] - s.y, dz = p[2] - s.z;
                const float d2 = dx * dx + dy * dy + dz * dz;
                if (d2 <= 1.0f * 1.0f) {
                    c->cone_state[cone] = CONE_ARRIVED;
                    break;
                }
            }
        }
    }
}

// Connection formation (reading A-28).  P:223-233: "A collision takes place if the distance between the centres
// of the two spheres is less than the sum of the radii ... the algorithm will compare d^2 and the square of the sum of
// the radii"; the axon grows "until the end pivot of the capsule is in 0.05 units of another neuron".  Plain
// definition, all pairs: every cone that is still ACTIVE after O9 is tested against the soma (= first polyline point)
// of every OTHER neuron; of the somata it touches it connects to the nearest (ties: the lowest index) and stops growing.
// fp32 decides an integer here, so the precision and order are part of the reading: d = tip - soma per axis,
// d2 = (dx dx + dy dy) + dz dz, each operation rounded once, compared (strictly) with fl(fl(r_cone + r_soma)^2).
void phase_connect(axo_ctx* c) {
    if (!c->connect_on) return;
    const size_t stride = (size_t)(c->max_segments + 1) * 3;
    const float reach = c->r_cone + c->r_soma;
    const float thr = reach * reach;
    if (c->target.size() != c->n_cones()) c->target.assign(c->n_cones(), NO_TARGET);
    for (size_t cone = 0; cone < c->n_cones(); ++cone) {
        if (c->cone_state[cone] != CONE_ACTIVE) continue;
        const float* p = &c->cone_pos[cone * 3];
        float best = 0.0f;
        uint32_t who = NO_TARGET;
        for (size_t n = 0; n < c->n_cones(); ++n) {
            if (n == cone) continue;  // not its own neuron
            const float* s = &c->poly[n * stride];
            const float dx = p[0] - s[0], dy = p[1] - s[1], dz = p[2] - s[2];
            const float d2 = (dx * dx + dy * dy) + dz * dz;
            if (d2 < thr && (who == NO_TARGET || d2 < best)) {
                best = d2;
                who = (uint32_t)n;
            }
        }
        if (who != NO_TARGET) {
            c->target[cone] = who;
            c->cone_state[cone] = CONE_CONNECTED;
        }
    }
}

// The adjacency list of the network in the paper's compact form (Fig. 4; reading A-29): vertex = neuron,
// Va[i] = head of vertex i's list in Ea, "edges of vertex i+1 following the edges of vertex i", Va[N] = |Ea|.  Every
// connected cone c gives the edge c -> target[c]; undirected (the adjacency MATRIX of Figs. 10/11 is what the paper
// exports): i and j are neighbours if either has connected to the other.  Lists ascending, no duplicates.
void build_graph(axo_ctx* c, bool directed) {
    const size_t N = c->n_cones();
    if (c->target.size() != N) c->target.assign(N, NO_TARGET);
    std::vector<std::vector<uint32_t>> adj(N);
    for (size_t i = 0; i < N; ++i) {
        const uint32_t t = c->target[i];
        if (t == NO_TARGET) continue;
        adj[i].push_back(t);
        if (!directed) adj[t].push_back((uint32_t)i);
    }
    c->Va.assign(N + 1, 0u);
    c->Ea.clear();
    for (size_t i = 0; i < N; ++i) {
        std::sort(adj[i].begin(), adj[i].end());
        adj[i].erase(std::unique(adj[i].begin(), adj[i].end()), adj[i].end());
        c->Va[i] = (uint32_t)c->Ea.size();
        c->Ea.insert(c->Ea.end(), adj[i].begin(), adj[i].end());
    }
    c->Va[N] = (uint32_t)c->Ea.size();
}

// Breadth-first levels from `root` over (Va, Ea): what Fig. 5's CUDA_BFS_KERNEL computes level by level (C_a = cost =
// number of edges from the root), written here as the textbook queue BFS the paper contrasts it with.
// Unreached vertices: -1.
void bfs(axo_ctx* c, uint32_t root) {
    const size_t N = c->n_cones();
    c->bfs_level.assign(N, -1);
    std::vector<uint32_t> queue;
    queue.push_back(root);
    c->bfs_level[root] = 0;
    for (size_t head = 0; head < queue.size(); ++head) {
        const uint32_t v = queue[head];
        for (uint32_t e = c->Va[v]; e < c->Va[v + 1]; ++e) {
            const uint32_t w = c->Ea[e];
            if (c->bfs_level[w] < 0) {
                c->bfs_level[w] = c->bfs_level[v] + 1;
                queue.push_back(w);
            }
        }
    }
}

int run_phases(axo_ctx* c, uint32_t mask) {
    if (mask & PH_DIFFUSE) phase_diffuse(c);
    if (mask & PH_BIN) {
        if (!(mask & PH_DIFFUSE)) adopt_A_as_presort(c);
        phase_bin(c);
    }
    if (mask & PH_SENSE) phase_sense(c);
    if (mask & PH_ADVANCE) phase_advance(c);
    if (mask & PH_CONNECT) phase_connect(c);
    if (mask & PH_COMMIT) c->step += 1;  // O10
    c->stepped = true;
    return OK;
}

int capacity_check(axo_ctx* c, uint32_t n, bool diffuse, bool advance) {
    if (diffuse && c->A.size() + (uint64_t)n * owned_rate(c) > c->max_particles)
        return fail(c, ECAPACITY, "particle capacity would overflow");
    if (advance) {
        uint32_t longest = 0;
        for (size_t i = 0; i < c->n_cones(); ++i)
            if (c->cone_state[i] == CONE_ACTIVE) longest = std::max(longest, c->poly_len[i]);
        if (c->n_cones() && (uint64_t)longest + n > (uint64_t)c->max_segments + 1)
            return fail(c, ECAPACITY, "polyline capacity would overflow");
    }
    return OK;
}

template <class T>
int copy_out(axo_ctx* c, const T* src, size_t n, void* dst, size_t dst_bytes, size_t* n_elems) {
    if (n_elems) *n_elems = n;
    if (dst == nullptr && dst_bytes == 0) return OK;
    if (dst == nullptr || dst_bytes < n * sizeof(T)) return fail(c, ESMALL, "destination too small");
    if (n) std::memcpy(dst, src, n * sizeof(T));
    return OK;
}

}  // namespace

// ============================================ exported ABI ==================================================
// Mirrors include/axg.h call for call (names axo_*), so that one ctypes harness drives both.

AXO_API int axo_create(const uint32_t grid[3], float D, uint32_t emission, float radius, float speed, float noise,
                       uint64_t seed, axo_ctx** out) {
    if (!grid || !out) return fail(nullptr, EINVAL_, "null argument");
    if (grid[0] == 0 || grid[1] == 0 || grid[2] == 0) return fail(nullptr, EINVAL_, "empty grid");
    if ((double)grid[0] * grid[1] * grid[2] >= 4294967296.0) return fail(nullptr, EINVAL_, "cells >= 2^32");
    if (!(D >= 0.0f) || !(radius >= 1.0f && radius <= 8.0f) || !(speed > 0.0f) || !(noise >= 0.0f) ||
        !std::isfinite(D) || !std::isfinite(speed) || !std::isfinite(noise))
        return fail(nullptr, EINVAL_, "bad D / radius / speed / noise");
    axo_ctx* c = new axo_ctx();
    c->nx = grid[0]; c->ny = grid[1]; c->nz = grid[2];
    c->D = D; c->emission = emission; c->radius = radius; c->speed = speed; c->noise = noise; c->seed = seed;
    *out = c;
    return OK;
}

AXO_API void axo_destroy(axo_ctx* c) { delete c; }

AXO_API const char* axo_last_error(const axo_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }

AXO_API int axo_set_capacity(axo_ctx* c, uint64_t max_particles, uint32_t max_segments) {
    if (!c || max_particles == 0) return fail(c, EINVAL_, "bad capacity");
    if (c->A.size() > max_particles) return fail(c, ECAPACITY, "live particles exceed the new capacity");
    for (size_t i = 0; i < c->n_cones(); ++i)
        if (c->poly_len[i] > (uint64_t)max_segments + 1) return fail(c, ECAPACITY, "polylines exceed new capacity");
    // re-stride polylines
    const size_t old_stride = (size_t)(c->max_segments + 1) * 3, new_stride = (size_t)(max_segments + 1) * 3;
    std::vector<float> np(c->n_cones() * new_stride, 0.0f);
    for (size_t i = 0; i < c->n_cones(); ++i)
        std::memcpy(&np[i * new_stride], &c->poly[i * old_stride], (size_t)c->poly_len[i] * 3 * sizeof(float));
    c->poly.swap(np);
    c->max_particles = max_particles;
    c->max_segments = max_segments;
    return OK;
}

AXO_API int axo_place_neurons(axo_ctx* c, const float* xyz, const float* heading, uint32_t n) {
    if (!c || (!xyz && n)) return fail(c, EINVAL_, "null argument");
    if (c->stepped) return fail(c, ESTATE, "neurons cannot be placed after the first step");
    for (uint32_t i = 0; i < n; ++i) {
        if (!inside(c, xyz[i * 3], xyz[i * 3 + 1], xyz[i * 3 + 2])) return fail(c, EINVAL_, "neuron outside the domain");
        if (heading) {
            const float* h = &heading[i * 3];
            const float l = std::sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
            if (!(l > 0.0f) || !std::isfinite(l)) return fail(c, EINVAL_, "bad heading");
        }
    }
    const size_t stride = (size_t)(c->max_segments + 1) * 3;
    c->cone_pos.assign(xyz, xyz + (size_t)n * 3);
    c->cone_heading.resize((size_t)n * 3);
    for (uint32_t i = 0; i < n; ++i) {
        if (heading) {
            const float* h = &heading[i * 3];
            const float l = std::sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
            for (int a = 0; a < 3; ++a) c->cone_heading[i * 3 + a] = h[a] / l;
        } else {  // A-20 default +z
            c->cone_heading[i * 3 + 0] = 0.0f; c->cone_heading[i * 3 + 1] = 0.0f; c->cone_heading[i * 3 + 2] = 1.0f;
        }
    }
    c->cone_state.assign(n, (uint8_t)CONE_ACTIVE);
    c->cone_counts.assign((size_t)n * MAX_SPECIES, 0);
    c->cone_moment.assign((size_t)n * MAX_SPECIES * 3, 0);
    c->cone_gradient.assign((size_t)n * 3, 0.0f);
    c->poly_len.assign(n, 1u);
    c->poly.assign((size_t)n * stride, 0.0f);
    for (uint32_t i = 0; i < n; ++i)
        for (int a = 0; a < 3; ++a) c->poly[i * stride + a] = xyz[i * 3 + a];
    c->target.assign(n, NO_TARGET);
    c->Va.clear(); c->Ea.clear(); c->bfs_level.clear();
    return OK;
}

AXO_API int axo_add_source(axo_ctx* c, float x, float y, float z, uint8_t species, int8_t polarity, uint32_t rate) {
    if (!c) return EINVAL_;
    if (!inside(c, x, y, z)) return fail(c, EINVAL_, "source outside the domain");
    if (species >= MAX_SPECIES) return fail(c, EINVAL_, "species >= 4");
    if (polarity != 1 && polarity != -1) return fail(c, EINVAL_, "polarity must be +1 or -1");
    if (c->species_polarity[species] != 0 && c->species_polarity[species] != polarity)
        return fail(c, EINVAL_, "polarity conflict within a species");
    if (c->sources.size() >= 4096) return fail(c, EINVAL_, "too many sources");
    c->species_polarity[species] = polarity;
    c->sources.push_back(Source{x, y, z, species, polarity, rate ? rate : c->emission});
    return OK;
}

AXO_API int axo_set_shard(axo_ctx* c, uint32_t rank, uint32_t world) {
    if (!c || world == 0 || rank >= world) return fail(c, EINVAL_, "bad shard");
    c->shard_rank = rank; c->shard_world = world;
    return OK;
}

// 0 = linear cell order (default), 1 = bricks of 8 x 4 x 4 cells (reading A-27); only before any particle exists
AXO_API int axo_set_key_order(axo_ctx* c, int order) {
    if (!c || (order < 0 || order > 2)) return fail(c, EINVAL_, "bad key order");
    if (c->stepped || c->A.size() || c->B.size()) return fail(c, ESTATE, "key order must be set before particles exist");
    c->key_order = order;
    c->cell_start.clear(); c->cell_end.clear();
    return OK;
}

// mode 0 = per cell (default), 1 = per particle, 2 = per particle, weighted by 1 - d^2/R^2 (reading A-26)
AXO_API int axo_set_sensing(axo_ctx* c, int mode) {
    if (!c || mode < 0 || mode > 2) return fail(c, EINVAL_, "bad sensing mode");
    c->sense_mode = mode;
    return OK;
}

// mode 0 = vector addition (default), 1 = fixed turn by the sign of N(SNR, 1); gain >= 0; 0 < turn < pi (radians)
AXO_API int axo_set_steering(axo_ctx* c, int mode, float gain, float turn) {
    if (!c || (mode != 0 && mode != 1) || !(gain >= 0.0f) || !std::isfinite(gain) || !(turn > 0.0f) ||
        !(turn < 3.14159265f))
        return fail(c, EINVAL_, "bad steering mode / gain / turn");
    c->steer_mode = mode;
    c->snr_gain = gain;
    c->cos_turn = (float)std::cos((double)turn);
    c->sin_turn = (float)std::sin((double)turn);
    const int r2 = (int)std::floor((double)c->radius * (double)c->radius), R = (int)std::floor((double)c->radius);
    uint32_t cells = 0;
    for (int dz = -R; dz <= R; ++dz)
        for (int dy = -R; dy <= R; ++dy)
            for (int dx = -R; dx <= R; ++dx)
                if (dx * dx + dy * dy + dz * dz <= r2) ++cells;
    c->n_stencil = cells;
    return OK;
}

AXO_API int axo_step(axo_ctx* c, uint32_t n) {
    if (!c) return EINVAL_;
    const int rc = capacity_check(c, n, true, true);
    if (rc) return rc;
    for (uint32_t i = 0; i < n; ++i)
        run_phases(c, PH_DIFFUSE | PH_BIN | PH_SENSE | PH_ADVANCE | PH_COMMIT | (c->connect_on ? PH_CONNECT : 0));
    return OK;
}

AXO_API int axo_step_phase(axo_ctx* c, uint32_t mask) {
    if (!c || (mask & ~63u)) return fail(c, EINVAL_, "bad phase mask");
    const int rc = capacity_check(c, 1, mask & PH_DIFFUSE, mask & PH_ADVANCE);
    if (rc) return rc;
    return run_phases(c, mask);
}

AXO_API int axo_load_particles(axo_ctx* c, const float* x, const float* y, const float* z, const uint8_t* species,
                               const uint32_t* id, uint64_t n, uint32_t next_id, uint32_t step) {
    if (!c || (n && (!x || !y || !z || !species || !id))) return fail(c, EINVAL_, "null argument");
    if (n > c->max_particles) return fail(c, ECAPACITY, "more particles than capacity");
    c->A.x.assign(x, x + n); c->A.y.assign(y, y + n); c->A.z.assign(z, z + n);
    c->A.species.assign(species, species + n); c->A.id.assign(id, id + n);
    c->next_id = next_id; c->step = step; c->n_live = n;
    return OK;
}

AXO_API int axo_load_cones(axo_ctx* c, const float* pos, const float* heading, const uint8_t* state,
                           const uint32_t* poly_len, uint32_t n) {
    if (!c || !pos || !heading || !state || !poly_len) return fail(c, EINVAL_, "null argument");
    if (n != c->n_cones()) return fail(c, EINVAL_, "cone count differs from the placed count");
    for (uint32_t i = 0; i < n; ++i)
        if (poly_len[i] == 0 || poly_len[i] > c->max_segments + 1) return fail(c, EINVAL_, "bad poly_len");
    const size_t stride = (size_t)(c->max_segments + 1) * 3;
    c->cone_pos.assign(pos, pos + (size_t)n * 3);
    c->cone_heading.assign(heading, heading + (size_t)n * 3);
    c->cone_state.assign(state, state + n);
    c->poly_len.assign(poly_len, poly_len + n);
    for (uint32_t i = 0; i < n; ++i)
        for (int a = 0; a < 3; ++a) c->poly[i * stride + (size_t)(poly_len[i] - 1) * 3 + a] = pos[i * 3 + a];
    return OK;
}

AXO_API int axo_read_state(axo_ctx* c, uint32_t field, void* dst, size_t dst_bytes, size_t* n_elems) {
    if (!c) return EINVAL_;
    switch (field) {
        case F_COUNTERS: {
            uint64_t v[9] = {c->step, c->n_live, c->next_id, c->emitted, c->absorbed, 0, 0, 0, 0};
            for (size_t i = 0; i < c->n_cones(); ++i) v[5 + c->cone_state[i]] += 1;  // active, arrived, exited, connected
            return copy_out(c, v, 9, dst, dst_bytes, n_elems);
        }
        case F_PART_X: return copy_out(c, c->A.x.data(), c->A.size(), dst, dst_bytes, n_elems);
        case F_PART_Y: return copy_out(c, c->A.y.data(), c->A.size(), dst, dst_bytes, n_elems);
        case F_PART_Z: return copy_out(c, c->A.z.data(), c->A.size(), dst, dst_bytes, n_elems);
        case F_PART_SPECIES: return copy_out(c, c->A.species.data(), c->A.size(), dst, dst_bytes, n_elems);
        case F_PART_ID: return copy_out(c, c->A.id.data(), c->A.size(), dst, dst_bytes, n_elems);
        case F_KEYS_SORTED: return copy_out(c, c->keys_sorted.data(), c->keys_sorted.size(), dst, dst_bytes, n_elems);
        case F_PERM: return copy_out(c, c->perm.data(), c->perm.size(), dst, dst_bytes, n_elems);
        case F_CELL_START:
        case F_CELL_END: {
            if (c->cell_start.size() != c->cells()) {
                c->cell_start.assign(c->cells(), 0u);
                c->cell_end.assign(c->cells(), 0u);
            }
            const std::vector<uint32_t>& v = field == F_CELL_START ? c->cell_start : c->cell_end;
            return copy_out(c, v.data(), v.size(), dst, dst_bytes, n_elems);
        }
        case F_CONE_POS: return copy_out(c, c->cone_pos.data(), c->cone_pos.size(), dst, dst_bytes, n_elems);
        case F_CONE_HEADING: return copy_out(c, c->cone_heading.data(), c->cone_heading.size(), dst, dst_bytes, n_elems);
        case F_CONE_STATE: return copy_out(c, c->cone_state.data(), c->cone_state.size(), dst, dst_bytes, n_elems);
        case F_CONE_COUNTS: return copy_out(c, c->cone_counts.data(), c->cone_counts.size(), dst, dst_bytes, n_elems);
        case F_CONE_MOMENT: return copy_out(c, c->cone_moment.data(), c->cone_moment.size(), dst, dst_bytes, n_elems);
        case F_CONE_GRADIENT: return copy_out(c, c->cone_gradient.data(), c->cone_gradient.size(), dst, dst_bytes, n_elems);
        case F_POLY_LEN: return copy_out(c, c->poly_len.data(), c->poly_len.size(), dst, dst_bytes, n_elems);
        case F_POLYLINE: return copy_out(c, c->poly.data(), c->poly.size(), dst, dst_bytes, n_elems);
        case F_PRE_X: return copy_out(c, c->B.x.data(), c->B.size(), dst, dst_bytes, n_elems);
        case F_PRE_Y: return copy_out(c, c->B.y.data(), c->B.size(), dst, dst_bytes, n_elems);
        case F_PRE_Z: return copy_out(c, c->B.z.data(), c->B.size(), dst, dst_bytes, n_elems);
        case F_PRE_SPECIES: return copy_out(c, c->B.species.data(), c->B.size(), dst, dst_bytes, n_elems);
        case F_PRE_ID: return copy_out(c, c->B.id.data(), c->B.size(), dst, dst_bytes, n_elems);
        case F_PRE_KEY: return copy_out(c, c->key.data(), c->key.size(), dst, dst_bytes, n_elems);
        case F_CONE_TARGET:
            if (c->target.size() != c->n_cones()) c->target.assign(c->n_cones(), NO_TARGET);
            return copy_out(c, c->target.data(), c->target.size(), dst, dst_bytes, n_elems);
        case F_GRAPH_VA: return copy_out(c, c->Va.data(), c->Va.size(), dst, dst_bytes, n_elems);
        case F_GRAPH_EA: return copy_out(c, c->Ea.data(), c->Ea.size(), dst, dst_bytes, n_elems);
        case F_BFS_LEVEL: return copy_out(c, c->bfs_level.data(), c->bfs_level.size(), dst, dst_bytes, n_elems);
        default: return fail(c, EINVAL_, "unknown field");
    }
}

AXO_API int axo_set_connect(axo_ctx* c, float r_cone, float r_soma) {
    if (!c || !(r_cone >= 0.0f) || !(r_soma >= 0.0f) || !std::isfinite(r_cone) || !std::isfinite(r_soma))
        return fail(c, EINVAL_, "bad radii");
    c->connect_on = (r_cone + r_soma) > 0.0f;
    c->r_cone = r_cone;
    c->r_soma = r_soma;
    return OK;
}

// harness hook: replace the connection targets (graph / BFS checked on given graphs)
AXO_API int axo_load_targets(axo_ctx* c, const uint32_t* target, uint32_t n) {
    if (!c || (!target && n)) return fail(c, EINVAL_, "null argument");
    if (n != c->n_cones()) return fail(c, EINVAL_, "cone count differs from the placed count");
    for (uint32_t i = 0; i < n; ++i)
        if (target[i] != NO_TARGET && (target[i] >= n || target[i] == i)) return fail(c, EINVAL_, "bad target");
    c->target.assign(target, target + n);
    return OK;
}

AXO_API int axo_build_graph(axo_ctx* c, int directed) {
    if (!c) return EINVAL_;
    build_graph(c, directed != 0);
    return OK;
}

AXO_API int axo_bfs(axo_ctx* c, uint32_t root) {
    if (!c) return EINVAL_;
    if (c->Va.size() != c->n_cones() + 1) return fail(c, ESTATE, "no graph: call axo_build_graph first");
    if (root >= c->n_cones()) return fail(c, EINVAL_, "root out of range");
    bfs(c, root);
    return OK;
}

// Harness-only load hook for the sharded loop (world_size-2 gloo tests): replace the per-cone sums of the last P3
// (e.g. by their sum over ranks) before P4 reads them.  No arithmetic: P4 recomputes G from these.
AXO_API int axo_load_sense(axo_ctx* c, const int64_t* counts, const int64_t* moment, uint32_t n) {
    if (!c || !counts || !moment) return fail(c, EINVAL_, "null argument");
    if (n != c->n_cones()) return fail(c, EINVAL_, "cone count differs from the placed count");
    c->cone_counts.assign(counts, counts + (size_t)n * MAX_SPECIES);
    c->cone_moment.assign(moment, moment + (size_t)n * MAX_SPECIES * 3);
    return OK;
}

// ---- oracle-only entry points used by the pins --------------------------------------------------------------

// T1: the raw block function.
AXO_API void axo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    philox4x32_10(ctr, key, out);
}

// T1b/T2: n blocks for entities id0..id0+n-1 at (seed, t, stream): r = 4n raw words, u = 4n uniforms, z = 3n normals.
AXO_API void axo_normals(uint64_t seed, uint32_t id0, uint32_t n, uint32_t t, uint32_t stream, uint32_t* r, float* u,
                         float* z) {
    for (uint32_t i = 0; i < n; ++i) {
        uint32_t rr[4];
        float zz[3];
        normals3(seed, id0 + i, t, stream, zz, rr);
        if (r) std::memcpy(r + 4 * (size_t)i, rr, sizeof(rr));
        if (u) for (int k = 0; k < 4; ++k) u[4 * (size_t)i + k] = uniform_from_bits(rr[k]);
        if (z) std::memcpy(z + 3 * (size_t)i, zz, sizeof(zz));
    }
}

// T9: O7 "brute form": all particles x all cones, independent of the sort and of cellStart/cellEnd.  Works on the
// current particle array (sorted or not).  counts: C*4 int64, moment: C*4*3 int64 (frozen cones are computed too).
AXO_API int axo_sense_brute(axo_ctx* c, int64_t* counts, int64_t* moment) {
    if (!c || !counts || !moment) return EINVAL_;
    const int r2 = (int)std::floor((double)c->radius * (double)c->radius);
    for (size_t cone = 0; cone < c->n_cones(); ++cone) {
        const int ci = (int)c->cone_pos[cone * 3 + 0], cj = (int)c->cone_pos[cone * 3 + 1],
                  ck = (int)c->cone_pos[cone * 3 + 2];
        int64_t* n = &counts[cone * MAX_SPECIES];
        int64_t* M = &moment[cone * MAX_SPECIES * 3];
        std::fill(n, n + MAX_SPECIES, 0);
        std::fill(M, M + MAX_SPECIES * 3, 0);
        for (size_t p = 0; p < c->A.size(); ++p) {
            const int dx = (int)c->A.x[p] - ci, dy = (int)c->A.y[p] - cj, dz = (int)c->A.z[p] - ck;
            if (dx * dx + dy * dy + dz * dz <= r2) {
                const int s = c->A.species[p];
                n[s] += 1;
                M[s * 3 + 0] += dx; M[s * 3 + 1] += dy; M[s * 3 + 2] += dz;
            }
        }
    }
    return OK;
}

// T7 / T8: bin arbitrary keys (no positions): perm, keys_sorted, cell_start, cell_end for n keys over `cells` cells,
// using exactly phase_bin's code path (O4..O6) on a scratch ctx.
AXO_API int axo_bin_keys(const uint32_t* keys, uint32_t n, uint32_t cells, uint32_t* perm, uint32_t* keys_sorted,
                         uint32_t* cell_start, uint32_t* cell_end) {
    axo_ctx c;
    c.nx = cells; c.ny = 1; c.nz = 1;
    for (uint32_t i = 0; i < n; ++i) {
        if (keys[i] >= cells) return EINVAL_;
        c.B.push((float)keys[i], 0.0f, 0.0f, 0, i);
    }
    c.key.assign(keys, keys + n);
    phase_bin(&c);
    std::memcpy(perm, c.perm.data(), n * sizeof(uint32_t));
    std::memcpy(keys_sorted, c.keys_sorted.data(), n * sizeof(uint32_t));
    std::memcpy(cell_start, c.cell_start.data(), cells * sizeof(uint32_t));
    std::memcpy(cell_end, c.cell_end.data(), cells * sizeof(uint32_t));
    return OK;
}

AXO_API int64_t axo_stencil_S2(float radius) {
    return stencil_S2((int)std::floor((double)radius * (double)radius));
}
