/* axg.h -- C-ABI boundary of the B200-native axon-guidance time step.
 *
 * One `axg_step` = one pass of the per-timestep hot path of the cue-diffusion guidance model of
 * arxiv/paper_1405_3331, as fixed by BASELINE.json `north_star` (NS) and SURVEY.md §8:
 *   P1 Brownian diffusion of cue particles + emission at sources + absorbing-boundary removal, compacted
 *      in order                                     (§3.5 "integration"; NS (1))
 *   P2 uniform-grid binning: linear cell key, stable LSD radix sort of (key, index), SoA reorder,
 *      cellStart / cellEnd                           (§3.5, Table 1; NS (2))
 *   P3 growth-cone sensing: per-species counts and integer first moments over the cells within the
 *      sensing radius                                (§3.5; NS (3))
 *   P4 cone advance along the normalised gradient + seeded angular noise at fixed speed
 *                                                    (NS (4))
 *   P5 append of the new segment to the axon polyline, arrival / exit test
 *                                                    (§3.4, §3.3; NS (5))
 * The exact arithmetic (Philox keying, uniform mapping, Box-Muller pairing, stencil, tie order ...) is the
 * list of readings in DESIGN.md §3; every kernel follows it and tests/ checks it against oracle/.
 *
 * Conventions
 *  - Every pointer argument is a HOST pointer owned by the caller unless it says "device".  The library copies;
 *    it never keeps a caller pointer after the call returns.
 *  - The ctx owns all device memory.  One ctx is used from one host thread at a time.  No global state.
 *  - All work is enqueued on the ctx stream (default: the legacy default stream; see axg_set_stream).
 *  - Every call returns 0 (AXG_OK) or a negative error code; axg_last_error() gives a message.  A call that
 *    fails with AXG_EINVAL / AXG_ECAPACITY / AXG_ESTATE / AXG_ESMALL has changed nothing.
 *  - There is NO CPU fallback: without a CUDA device axg_create fails with AXG_ECUDA.
 */
#ifndef AXG_H
#define AXG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct axg_ctx axg_ctx; /* opaque */

/* Unit cells; the domain is [0,nx) x [0,ny) x [0,nz) in cell units ("uniform grid", cell size 1). */
typedef struct axg_grid {
    uint32_t nx, ny, nz;
} axg_grid;

enum {
    AXG_OK = 0,
    AXG_EINVAL = -1,    /* bad argument (null, NaN, out of the domain, radius not in [1,8], cells >= 2^32 ...)   */
    AXG_ECAPACITY = -2, /* particle or polyline capacity would overflow (checked on host bounds before launch); or the
                           device error word was found set after a synchronisation (only reachable through
                           axg_enqueue_phase, which checks nothing): the step that hit the capacity dropped its emission
                           or its append, so the state is UNDEFINED from there on.  The word is cleared when it is
                           reported, by axg_set_capacity and by axg_load_particles: raise the capacity, reload the
                           state, go on.                                                                           */
    AXG_ESTATE = -3,    /* call not allowed in this state (neurons placed after the first step)                */
    AXG_ECUDA = -4,     /* CUDA runtime error, or no device                                                    */
    AXG_ESMALL = -5     /* dst_bytes too small; *n_elems holds the element count required                      */
};

#define AXG_MAX_SPECIES 4u
#define AXG_MAX_SOURCES 4096u
#define AXG_R_CAPTURE 1.0f /* arrival radius in cells (reading A-16) */

/* cone state */
enum { AXG_CONE_ACTIVE = 0, AXG_CONE_ARRIVED = 1, AXG_CONE_EXITED = 2, AXG_CONE_CONNECTED = 3 /* axg_set_connect */ };

/* phases for axg_step_phase */
enum {
    AXG_PHASE_DIFFUSE = 1, /* P1: diffuse, absorb, compact, emit, key (+ digit histograms)           */
    AXG_PHASE_BIN = 2,     /* P2: sort, reorder, cellStart/cellEnd                                   */
    AXG_PHASE_SENSE = 4,   /* P3                                                                     */
    AXG_PHASE_ADVANCE = 8, /* P4 + P5                                                                */
    AXG_PHASE_COMMIT = 16, /* step counter t += 1                                                    */
    AXG_PHASE_ALL = 31,
    AXG_PHASE_CONNECT = 32 /* connection formation after P5 (axg_set_connect; a no-op while it is off); part of every
                              whole step of axg_step once enabled, not of AXG_PHASE_ALL                              */
};

/* fields for axg_read_state.  "sorted order" = the particle array left by P2 (input of the next P1).
 * "pre-sort" = the array written by P1 (survivors in input order, then newborns), input of P2.         */
enum {
    AXG_COUNTERS = 0,     /* u64[9]: step, n_live, next_id, emitted, absorbed, active, arrived, exited, connected */
    AXG_PART_X = 1,       /* f32[n_live]  sorted order                                                  */
    AXG_PART_Y = 2,
    AXG_PART_Z = 3,
    AXG_PART_SPECIES = 4, /* u8[n_live]                                                                 */
    AXG_PART_ID = 5,      /* u32[n_live]                                                                */
    AXG_KEYS_SORTED = 6,  /* u32[n_live]                                                                */
    AXG_PERM = 7,         /* u32[n_live]  sorted j -> pre-sort index                                    */
                          /* (6, 7: those of the last completed P2; under count binning they are not stored on the path
                           *  but derived here, on read, from the intact inputs of that P2; undefined between a P1 and its P2) */
    AXG_CELL_START = 8,   /* u32[cells]   first sorted j of the cell, 0 if empty                        */
    AXG_CELL_END = 9,     /* u32[cells]   one past the last sorted j, 0 if empty                        */
    AXG_CONE_POS = 10,    /* f32[C*3] AoS                                                               */
    AXG_CONE_HEADING = 11,/* f32[C*3] AoS                                                               */
    AXG_CONE_STATE = 12,  /* u8[C]                                                                      */
    AXG_CONE_COUNTS = 13, /* i64[C*AXG_MAX_SPECIES]      n_s of the last P3 in which the cone was active */
    AXG_CONE_MOMENT = 14, /* i64[C*AXG_MAX_SPECIES*3]    M_s                                            */
    AXG_CONE_GRADIENT = 15,/* f32[C*3]  g = G / S2(R)                                                   */
    AXG_POLY_LEN = 16,    /* u32[C]                                                                     */
    AXG_POLYLINE = 17,    /* f32[C*(max_segments+1)*3] neuron-major; entries >= poly_len are 0          */
    AXG_PRE_X = 18,       /* f32[n_live]  pre-sort array (valid after P1 of the current step)           */
    AXG_PRE_Y = 19,
    AXG_PRE_Z = 20,
    AXG_PRE_SPECIES = 21,
    AXG_PRE_ID = 22,
    AXG_PRE_KEY = 23,     /* u32[n_live]  cell key of the pre-sort array                                */
    AXG_CONE_TARGET = 24, /* u32[C]  neuron the cone has connected to, 0xffffffff = none (axg_set_connect)      */
    AXG_GRAPH_VA = 25,    /* u32[C+1] heads of the adjacency lists (axg_build_graph); empty before              */
    AXG_GRAPH_EA = 26,    /* u32[E]   edges: neighbours of vertex i at Ea[Va[i] .. Va[i+1]), ascending          */
    AXG_BFS_LEVEL = 27,   /* i32[C]   BFS level from the root of the last axg_bfs, -1 = not reached             */
    AXG_FIELD_COUNT = 28
};

/* Create a context on the current CUDA device.
 *  grid      unit-cell grid, nx*ny*nz < 2^32, each >= 1
 *  D         diffusion coefficient in cell^2/step; per-axis Gaussian step sigma = sqrt(2 D) (NS (1), config C1/C4)
 *  emission  default particles per step per source (used when axg_add_source rate == 0)
 *  radius    sensing radius R in cells, 1 <= R <= 8; stencil = {d in Z^3 : |d|^2 <= floor(R^2)} (A-11)
 *  speed     cone advance per step in cells, > 0 ("a predefined distance is traversed")
 *  noise     standard deviation (rad, small-angle) of the Gaussian heading noise, >= 0 (NS (4))
 *  seed      Philox key = (seed low 32 bits, seed high 32 bits)
 * Default capacities: 2^20 particles, 1024 polyline segments per cone (axg_set_capacity changes them).     */
int axg_create(const axg_grid* grid, float D, uint32_t emission, float radius, float speed, float noise,
               uint64_t seed, axg_ctx** out);

/* Place n neurons, i.e. their growth cones (one axon per neuron, growing from the neuron).
 *  xyz      n*3 floats AoS, each inside the domain
 *  heading  n*3 floats AoS (normalised by the library) or NULL => (0,0,1)
 * Replaces any neurons placed before.  Sets poly[c][0] = xyz[c], poly_len = 1, state ACTIVE.
 * AXG_ESTATE after the first step.                                                                       */
int axg_place_neurons(axg_ctx* ctx, const float* xyz, const float* heading, uint32_t n);

/* Add a cue source ("particle systems ... placed", "particles are generated").
 *  (x,y,z) inside the domain; species < AXG_MAX_SPECIES; polarity +1 attract / -1 repel, fixed
 *  per species by the first source of that species (conflict => AXG_EINVAL); rate particles/step, 0 => default.
 * Attractive sources are the arrival targets.  Allowed at any time; emits from the next step on.         */
int axg_add_source(axg_ctx* ctx, float x, float y, float z, uint8_t species, int8_t polarity, uint32_t rate);

/* Run n whole time steps (P1..P5 + commit each) on the device without host synchronisation in between;
 * returns after the stream has been synchronised and the device error word read.  With cones placed, P3..P5 of
 * step t run on a ctx-owned side stream concurrently with P1 of step t+1 (they share no data; joined by events
 * before P2 of step t+1 and before the call returns).  For n >= 4 one step is captured once as a CUDA graph and
 * replayed (re-captured when a setting or an allocation has changed); when the ctx stream is the legacy default
 * stream, which cannot be captured, the steps run on a ctx-owned stream forked from and joined back into it.  */
int axg_step(axg_ctx* ctx, uint32_t n);

/* Copy one field to host memory.  If dst == NULL or dst_bytes is too small: returns AXG_ESMALL (or AXG_OK when
 * dst == NULL and dst_bytes == 0) with *n_elems = number of elements of the field.  Synchronises the stream. */
int axg_read_state(axg_ctx* ctx, uint32_t field, void* dst, size_t dst_bytes, size_t* n_elems);

void axg_destroy(axg_ctx* ctx);

/* Message of the last failing call on this ctx (ctx-owned, valid until the next call); with ctx == NULL the
 * message of the last failing axg_create of this thread.                                                 */
const char* axg_last_error(const axg_ctx* ctx);

/* ---- harness / plumbing calls (not part of the paper's problem statement) ------------------------------- */

/* Re-allocate for at most max_particles live particles and max_segments appended segments per cone.
 * Keeps sources and neurons; live particles are kept if they fit, else AXG_ECAPACITY.  max_particles < 2^30 - 256
 * (the sort value carries the species in its top two bits), else AXG_EINVAL.                              */
int axg_set_capacity(axg_ctx* ctx, uint64_t max_particles, uint32_t max_segments);

/* Replace the particle array (taken as the "sorted order" array, i.e. the input of the next P1) and the id /
 * step counters, and clear the device error word.  Positions are not validated here (n <= capacity and species < 4
 * are): P1 absorbs a row that is outside the domain after its move like any other; AXG_PHASE_BIN without
 * AXG_PHASE_DIFFUSE on a row outside the domain fails with AXG_EINVAL (device error word bit 4; the row is binned into
 * cell 0, nothing is written out of bounds, the state is undefined).                                        */
int axg_load_particles(axg_ctx* ctx, const float* x, const float* y, const float* z, const uint8_t* species,
                       const uint32_t* id, uint64_t n, uint32_t next_id, uint32_t step);

/* Replace cone position / heading / state / polyline length of the n placed cones (n must equal the placed
 * count).  Polyline contents are kept; entry poly_len-1 is set to pos.                                    */
int axg_load_cones(axg_ctx* ctx, const float* pos, const float* heading, const uint8_t* state,
                   const uint32_t* poly_len, uint32_t n);

/* Run the selected phases of ONE step (for per-phase parity).  AXG_PHASE_BIN bins the output of the step's P1 if one has
 * run and is still unbinned (in this call or an earlier one); otherwise it takes the current particle array as the
 * pre-sort array (copy + re-key), so that binning can be checked on positions produced elsewhere.  Synchronises. */
int axg_step_phase(axg_ctx* ctx, uint32_t phase_mask);

/* Multi-GPU sharding by source: this rank emits only sources with index % world == rank; the
 * others still consume their particle ids, so trajectories equal the 1-GPU run.  Default (0,1).  With world > 1
 * P3 writes zeros for frozen cones (so that the all-reduced buffer stays meaningful); their AXG_CONE_COUNTS /
 * AXG_CONE_MOMENT then read 0 instead of the last active value.                                           */
int axg_set_shard(axg_ctx* ctx, uint32_t rank, uint32_t world);

/* How P2 (binning) is computed; the results are identical bit for bit.
 *  AXG_BIN_RADIX  stable LSD radix sort of (key, index), 8-bit digits, one onesweep pass per digit, then the
 *                 reorder + cell-range kernel.  Cost ~ passes x N; independent of the number of cells.
 *  AXG_BIN_COUNT  counting sort over the cells: P1 counts particles per cell (one atomic each, which also returns the
 *                 particle's arrival rank inside its cell), a single-pass scan over the cells gives the cell ranges,
 *                 and a rank-inside-the-cell kernel restores the stable order.  Cost ~ N + cells; 4 B x cells of
 *                 extra device memory.  Measured faster than RADIX on every config of BASELINE.json.
 *  AXG_BIN_AUTO   (default) COUNT when cells <= 4 x particle capacity (a sparse population in a huge grid pays
 *                 per cell) and cells <= AXG_AUTO_COUNT_MAX_CELLS, else RADIX.
 * Allowed whenever no step is half done (not between AXG_PHASE_DIFFUSE and AXG_PHASE_BIN): AXG_ESTATE.    */
enum { AXG_BIN_AUTO = 0, AXG_BIN_RADIX = 1, AXG_BIN_COUNT = 2 };
#define AXG_AUTO_COUNT_MAX_CELLS 2147483648u
int axg_set_binning(axg_ctx* ctx, int mode);
/* *mode = AXG_BIN_RADIX or AXG_BIN_COUNT: what the requested mode resolves to for the current grid, key order and
 * capacity (allocates the particle arrays if they do not exist yet).                                         */
int axg_get_binning(axg_ctx* ctx, int* mode);

/* Steering rule of P4.
 *  AXG_STEER_VECTOR (default)  north_star's rule: heading = normalise(gradient direction + noise x N(0, I)).
 *  AXG_STEER_SNR    the paper's first rule (Eq. 5; reading A-25): the heading turns by the
 *                   fixed angle `turn` (radians; the paper's pi/30) in the plane of heading and gradient, TOWARDS the
 *                   gradient direction if a draw from N(SNR, 1) is positive, away from it otherwise, with
 *                   SNR = gain x mu x sqrt(gamma / (1 + gamma)^3) x sin(phi); gamma = particles per cell over the
 *                   sensing stencil, mu = |g| / gamma (g = the gradient estimate of P3), phi = angle between heading
 *                   and gradient.  Nothing in range, zero gradient or heading parallel to it: direction kept.  The
 *                   draw is the first normal of the cone's Philox block (stream 1); `noise` is not used.
 * gain >= 0, 0 < turn < pi, else AXG_EINVAL.  May be called between any two steps.                         */
enum { AXG_STEER_VECTOR = 0, AXG_STEER_SNR = 1 };
int axg_set_steering(axg_ctx* ctx, int mode, float gain, float turn);

/* Cell order = what the cell key of P2a is ("a Z-order curve ... potential
 * optimization"; reading A-27).
 *  AXG_KEY_LINEAR (default)  north_star's key: (z * ny + y) * nx + x.
 *  AXG_KEY_BRICK   bricks of 8 x 4 x 4 cells; bricks in linear order (x fastest), the cells of a brick in linear order:
 *                  key = (((z/4) * ceil(ny/4) + y/4) * ceil(nx/8) + x/8) * 128 + (z%4) * 32 + (y%4) * 8 + x%8.
 *                  A particle that moves one cell stays inside, or next to, 512 contiguous bytes of the per-cell
 *                  arrays.  The key space is the grid padded to whole bricks: AXG_CELL_START / AXG_CELL_END then have
 *                  ceil(nx/8) * ceil(ny/4) * ceil(nz/4) * 128 entries, indexed by key; AXG_KEYS_SORTED, AXG_PERM and the
 *                  order of the AXG_PART_* rows follow this key.  Trajectories, cones and all sums are unchanged.
 *  AXG_KEY_MORTON  the Z-order curve the paper names (reading A-31): bit b of x, of y and of z in turn, b = 0,
 *                  1, ..., from the least significant key bit up; an axis that needs fewer bits than the others drops out
 *                  of the rotation once its bits are used.  Key space = the grid padded to powers of two; indexing of
 *                  AXG_CELL_START / AXG_CELL_END etc. as under AXG_KEY_BRICK.
 * Only directly after axg_create (before neurons, sources or particles exist): AXG_ESTATE otherwise.
 * AXG_EINVAL: bad value, or a padded key space of 2^32 or more.                                             */
enum { AXG_KEY_LINEAR = 0, AXG_KEY_BRICK = 1, AXG_KEY_MORTON = 2 };
int axg_set_key_order(axg_ctx* ctx, int order);

/* Sensing rule of P3 (section 5.3: "each individual particle that the axon's
 * growth cone detects would influence the axon's path"; reading A-26).
 *  AXG_SENSE_CELL (default)  north_star's rule: counts and first moments over the CELLS of the index-space ball.
 *  AXG_SENSE_PARTICLE        every particle at x with |x - p|^2 <= R^2 of the cone at p (fp32: d = x - p per axis,
 *                            d2 = (dx*dx + dy*dy) + dz*dz, each operation rounded once, compared with fl(R*R)) counts 1
 *                            and adds rint(256 d) per axis to the first moment of its species.
 *  AXG_SENSE_PARTICLE_WEIGHTED  the same test; the particle adds rint(16 w) * rint(16 d) with w = 1 - d2 / fl(R*R):
 *                            near particles weigh more.
 * rint = round to nearest even.  Under both particle rules AXG_CONE_MOMENT is in units of 1/256 cell and
 * AXG_CONE_GRADIENT = G / (256 S2(R)); the sums stay integers (bit-exact, additive over shards, same sense buffer and
 * all-reduce), and P4 / P5 are unchanged.  Per cone the sums are int32 on the device and are not checked for overflow: a
 * moment component is bounded by n R (cell rule) or 256 n R (particle rules) for n particles in range, i.e. n must stay
 * below 2^31 / R resp. 2^31 / (256 R) = 2.7 M at R = 3, 1.05 M at R = 8 (C1..C5: at most a few thousand).  Needs the binned state of P2 like the cell rule.  May be called between any two steps; bad mode: AXG_EINVAL. */
enum { AXG_SENSE_CELL = 0, AXG_SENSE_PARTICLE = 1, AXG_SENSE_PARTICLE_WEIGHTED = 2 };
int axg_set_sensing(axg_ctx* ctx, int mode);

/* Connection formation (reading A-28).  PAPER.md:223-233 (section 3.3): "A collision
 * takes place if the distance between the centres of the two spheres is less than the sum of the radii ... the algorithm
 * will compare d^2 and the square of the sum of the radii"; the axon grows "until the end pivot of the
 * capsule is in 0.05 units of another neuron"; the neurons "stored in a grid data structure entirely
 * computed on the GPU" as the broadphase.
 *  r_cone, r_soma   radii (cells) of the sphere around a growth-cone tip and around a soma (= the point where
 *                   axg_place_neurons put the neuron); both >= 0, sum <= 64; sum 0 switches the rule off (default).
 * Once on, every whole step ends with AXG_PHASE_CONNECT: each cone still ACTIVE after P5 is tested against the somata of
 * all OTHER neurons, d2 = (dx dx + dy dy) + dz dz in fp32 (each operation rounded once), a hit iff d2 < fl(fl(r_cone +
 * r_soma)^2); it connects to the nearest soma it hits (equal distances: the lowest index): AXG_CONE_TARGET[c] = that
 * neuron, state AXG_CONE_CONNECTED, and it stops growing.  The somata are binned into a uniform grid of cubic cells whose
 * edge is a power of two >= r_cone + r_soma, so a tip meets the somata of 27 cells only.  Sharded runs: replicated on
 * every rank (same cones, same result).                                                                           */
int axg_set_connect(axg_ctx* ctx, float r_cone, float r_soma);

/* Harness hook: replace AXG_CONE_TARGET (n = the placed count; entries 0xffffffff or a neuron index other than the
 * cone's own: AXG_EINVAL otherwise) so that the graph calls can be checked on given graphs.                         */
int axg_load_targets(axg_ctx* ctx, const uint32_t* target, uint32_t n);

/* The network as the paper's compact adjacency list (Fig. 4; reading A-29): vertex = neuron,
 * every connected cone c is the edge c -> AXG_CONE_TARGET[c].  AXG_GRAPH_VA[i] is the head of vertex i's list in
 * AXG_GRAPH_EA, the lists follow one another, AXG_GRAPH_VA[C] = E.  directed == 0: neighbours in either direction (the 0/1
 * adjacency MATRIX the paper exports, Figs. 10-11, is symmetric); directed != 0: out-neighbours only.  Lists ascending,
 * no duplicates.  AXG_ESTATE without neurons.  Synchronises.                                                       */
int axg_build_graph(axg_ctx* ctx, int directed);

/* Level-synchronous breadth-first search over the list of the last axg_build_graph (Fig. 5
 * CUDA_BFS_KERNEL: one thread per vertex, frontier F_a, visited X_a, cost C_a, "repeated until frontier is empty";
 * DESIGN.md reading A-30: with the second, updating frontier array of the algorithm the paper cites).  AXG_BFS_LEVEL[v] =
 * number of edges from root, -1 if v is not reached.  AXG_ESTATE without a graph, AXG_EINVAL for a bad root.        */
int axg_bfs(axg_ctx* ctx, uint32_t root);

/* The same BFS for callers that may not allocate device memory (code under CUDA graph capture around it, tight serving
 * loops, harnesses that forbid cudaMalloc): no context, no cudaMalloc / cudaFree / allocating library call -- the scratch
 * (frontier, updating frontier, visited: one byte per vertex each, and the "frontier not empty" word) is a file-scope
 * device array of the library, 3 x AXG_BFS_NOALLOC_MAX_VERTICES + 256 bytes (3 MB), which every GPU that loads the library
 * holds until the process exits.
 *  va, ea   DEVICE pointers: the adjacency list as AXG_GRAPH_VA / AXG_GRAPH_EA describe it (va[n_vertices + 1] heads,
 *           ea[va[n_vertices]] neighbours); read only
 *  level    DEVICE pointer, int32[n_vertices]: written, level from root or -1 (= AXG_BFS_LEVEL)
 *  stream   a cudaStream_t (NULL: the default stream); the call returns after the stream has been synchronised
 * All four are owned by the caller.  AXG_EINVAL: a null pointer, n_vertices == 0 or > AXG_BFS_NOALLOC_MAX_VERTICES (use
 * axg_bfs then), root >= n_vertices; AXG_ECUDA: no current device or a CUDA error; the message is axg_last_error(NULL).
 * Every call shares the one scratch array, which keeps the last call's contents (each call re-initialises the part it
 * uses before reading it): calls that overlap on the GPU -- different streams, several host threads -- RACE; serialise
 * them.  The current CUDA device at the time of the call is the one used.                                          */
#define AXG_BFS_NOALLOC_MAX_VERTICES 1048576u
int axg_bfs_noalloc(const uint32_t* va, const uint32_t* ea, uint32_t n_vertices, uint32_t root, int32_t* level,
                    void* stream);

/* Device pointer (int32[C][AXG_MAX_SPECIES][4] = n,Mx,My,Mz) of the per-cone sensing sums, for the NCCL
 * all-reduce between P3 and P4 when sharded.  *bytes = its size.  Owned by ctx.                           */
int axg_sense_buffer(axg_ctx* ctx, void** device_ptr, size_t* bytes);

/* The sharded step loop without a host synchronisation per step:
 *     axg_check_capacity(ctx, n);
 *     n times { axg_enqueue_phase(ctx, DIFFUSE|BIN|SENSE);  all-reduce of axg_sense_buffer on the ctx stream;
 *               axg_enqueue_phase(ctx, ADVANCE|COMMIT); }
 *     axg_sync(ctx);
 * axg_check_capacity is the host-side pre-check that axg_step does for n further steps (AXG_ECAPACITY, nothing
 * changed).  axg_enqueue_phase launches the kernels of the selected phases of ONE step on the ctx stream and returns
 * at once; it checks nothing.  axg_sync waits for the stream, reads the device error word (AXG_ECAPACITY if set,
 * AXG_ECUDA on a CUDA error) and refreshes the element counts that axg_read_state reports.                */
int axg_check_capacity(axg_ctx* ctx, uint32_t n);
int axg_enqueue_phase(axg_ctx* ctx, uint32_t phase_mask);
int axg_sync(axg_ctx* ctx);

/* The same, on a stream of the caller's choice (a cudaStream_t; the ctx stream is not touched), for the OVERLAPPED sharded
 * step: P3, the all-reduce and P4 / P5 of step t on a side stream beside P1 of step t+1 on the main stream -- they share no
 * data (P1 takes its step index from a counter of its own) -- joined by the caller's events before P2 of step t+1, exactly
 * as axg_step orders one GPU's work.  overlapped != 0: the commit of these phases may run beside the NEXT step's P1 and must
 * not re-align P1's step index (pass it for ADVANCE | COMMIT in that loop).  Capturable into a CUDA graph together with the
 * NCCL all-reduce; axg_params_fingerprint changes whenever a captured launch would be stale (an allocation, a mode or a
 * parameter changed).  paper_1405_3331_b200/sharded.py is the loop.                                                */
int axg_enqueue_phase_on(axg_ctx* ctx, uint32_t phase_mask, void* stream, int overlapped);
int axg_params_fingerprint(axg_ctx* ctx, uint64_t* fingerprint);

/* Use `stream` (a cudaStream_t) for all later work of this ctx.                                          */
int axg_set_stream(axg_ctx* ctx, void* stream);

/* Device-memory hooks: alloc(bytes, stream, user) -> device pointer or NULL, free(ptr, user).  Process-wide,
 * must be set before axg_create; NULL restores cudaMalloc / cudaFree.  The Python binding routes these to the
 * PyTorch caching allocator (NS: "PyTorch is used only for device memory and streams").                  */
typedef void* (*axg_alloc_fn)(size_t bytes, void* stream, void* user);
typedef void (*axg_free_fn)(void* ptr, void* user);
int axg_set_allocator(axg_alloc_fn alloc, axg_free_fn free_, void* user);

/* Timing of the last axg_step call: device milliseconds between the first and last kernel (CUDA events on the
 * ctx stream), kernels launched, and the sum over its steps of the live particle count entering each step.  */
int axg_last_step_stats(axg_ctx* ctx, float* device_ms, uint64_t* launches, uint64_t* particle_steps);

/* Per-kernel device time of the NEXT axg_step call (debug; inserts events between kernels).  times_ms must
 * hold AXG_KERNEL_COUNT floats after the call via axg_kernel_times.                                      */
enum {
    AXG_K_CLEAR = 0, AXG_K_DIFFUSE = 1, AXG_K_EMIT = 2, AXG_K_SORT = 3, AXG_K_REORDER = 4, AXG_K_SENSE = 5,
    AXG_K_ADVANCE = 6, AXG_K_COMMIT = 7, AXG_K_SCAN = 8, AXG_K_PLACE = 9, AXG_K_SETTLE = 10, AXG_KERNEL_COUNT = 11
};
int axg_profile_next_step(axg_ctx* ctx, int enable);
int axg_kernel_times(axg_ctx* ctx, float* times_ms /* AXG_KERNEL_COUNT */);

#ifdef __cplusplus
}
#endif
#endif /* AXG_H */
