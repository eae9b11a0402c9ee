/*
 * manta.h -- C ABI of the B200-native MANTA vehicle-update hot path (libmanta.so).
 *
 * What the library computes: the per-timestep (dt = 0.5 s) update of every active vehicle of a
 * metropolitan traffic microsimulation over the "traffic atlas": leader look-ahead, IDM car
 * following (Eq. 1), lane change with gap acceptance (Eq. 2-4), integration, edge /
 * intersection transfer along precomputed routes, departure release, and
 * the per-edge counts / travel times the paper reports.  The exact rules (R0-R9) and the
 * readings taken where the paper is silent are in DESIGN.md sections 2-3.  Routing and initialisation are outside
 * the timed path: manta_create / manta_load_trips are initialisation, manta_step is the hot path.
 *
 * Conventions
 *   - Every pointer argument is a HOST pointer unless its name ends in _dev.  Input arrays are copied during the
 *     call; the caller may free them on return.  Output arrays are caller-allocated.
 *   - Every call returns 0 (MANTA_OK) or a negative MANTA_ERR_* code; no exceptions, no abort.  After an error
 *     manta_last_error() gives a text; a failed call leaves the simulation state as it was (manta_step excepted:
 *     a CUDA fault is sticky and every later call returns MANTA_ERR_CUDA).
 *   - All kernels run on one CUDA device and on the stream given by manta_set_stream (default: the legacy
 *     default stream).  Device memory comes from cudaMalloc unless manta_set_allocator installed callbacks
 *     (the Python binding hands out PyTorch caching-allocator blocks that way).
 *   - There is no CPU fallback: without a CUDA device manta_create returns MANTA_ERR_CUDA.
 */
#ifndef MANTA_H
#define MANTA_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MANTA_OK 0
#define MANTA_ERR_INVALID_ARG (-1)
#define MANTA_ERR_BAD_NETWORK (-2)
#define MANTA_ERR_BAD_ROUTE (-3)
#define MANTA_ERR_OOM (-4)
#define MANTA_ERR_CUDA (-5)
#define MANTA_ERR_STATE (-6)

#define MANTA_GREEN 0    /* case 2: every vehicle passes; conflicts per (edge, lane) entry  */
#define MANTA_PRIORITY 1 /* case 1 exclusivity: one vehicle per node per step, smallest vehicle id first */
#define MANTA_STOP 2     /* case 1 in full: every vehicle stands stop_time_s at the stop line, then
                            one vehicle per node per step, the (inbound, outbound) edge combinations taking turns
                            (round-robin), equal combinations by smallest vehicle id -- rule R8s of DESIGN.md.
                            Limits that apply only to networks with STOP nodes: in-degree x out-degree <= 256 per
                            STOP node, n_trips < 2^24, ceil(stop_time_s / dt) <= 7 (else stop_time_s is unused) */

#define MANTA_WAITING 0
#define MANTA_ACTIVE 1
#define MANTA_DONE 2

#define MANTA_NONE 0xFFFFFFFFu
#define MANTA_MAX_LANES 8
#define MANTA_MAX_EDGE_CELLS 65535u

/* manta_params.flags */
#define MANTA_FLAG_MULTI_KERNEL 2u     /* three launches per timestep instead of the persistent cooperative kernel */
#define MANTA_FLAG_RECORD_ACC 4u       /* keep each vehicle's last acceleration for manta_state.acc (tests)  */
#define MANTA_FLAG_NO_FUSE 16u         /* admission of step t + 1 as a phase of its own (three grid barriers per step)
                                          instead of inside the second phase of step t (A/B switch)              */
#define MANTA_FLAG_NO_L2_PIN 8u        /* never pin the occupancy planes in L2 (A/B switch).  By default the planes get a
                                          persisting L2 access-policy window while at least 400,000 vehicle slots are in
                                          use (counted at manta_sync) and the planes fit the device's carve-out; the
                                          device-wide cudaLimitPersistingL2CacheSize is raised for that and put back     */

#define MANTA_FLAG_FEW_SEGMENTS 64u    /* test switch: the vehicles are kept in TWO segments (two thread blocks per
                                          phase) instead of one per resident block, so that small cases put thousands
                                          of slots into one segment and run the multi-chunk software pipeline of the
                                          update pass and the real overflow of the deferred queue                    */
#define MANTA_FLAG_TINY_QUEUES 32u     /* test switch: a block keeps only 2 deferred-list entries in shared memory, so
                                          that the overflow path through device memory runs in small cases       */

typedef struct manta_sim manta_sim; /* opaque; owned by the library; one simulation on one device */

/* Street network (per edge lanes, length in metres, free-flow speed).  Edges are numbered in
 * CSR order by TAIL node: edges row_ptr[u] .. row_ptr[u+1]-1 leave node u. */
typedef struct {
    uint32_t n_nodes, n_edges;
    const uint32_t *row_ptr;     /* [n_nodes+1]                                                         */
    const uint32_t *head;        /* [n_edges]  head node of each edge                                   */
    const float *length_m;       /* [n_edges]  > 0; rounded to whole 1 m cells; >= LEN_MIN (R0) */
    const uint8_t *lanes;        /* [n_edges]  1..8                                                     */
    const float *speed_limit;    /* [n_edges]  m/s, > 0; used as IDM v0                   */
    const uint8_t *node_ctrl;    /* [n_nodes] MANTA_GREEN / MANTA_PRIORITY / MANTA_STOP, or NULL = all GREEN */
} manta_network;

/* Model parameters; one set shared by all vehicles.  delta of Eq. 1 is fixed at 4. */
typedef struct {
    uint32_t size;             /* = sizeof(manta_params): versioning                                     */
    float dt;                  /* timestep, s                                                            */
    float a, b, T, s0;         /* IDM: acceleration, braking, headway, standstill gap (Eq. 1, Table I)   */
    float veh_len;             /* vehicle length L, m                                                    */
    uint32_t lookahead_cells;  /* H of R2                                                                */
    uint32_t lookback_cells;   /* lag search range of R5; must be >= ceil(L) + Z_out                     */
    float mlc_scale_m;         /* Lambda: unit of x_i, x_0 in Eq. 2 (reading G6)                         */
    float dlc_gain_thr;        /* discretionary gain threshold, m/s^2 (reading G9)                       */
    float lc_alpha;            /* anticipation time alpha, s (Eq. 3, 4)                                  */
    float lc_gap_low;          /* desired gap below 25 mph, m                             */
    float lc_gap_high;         /* desired gap above 25 mph, m                                            */
    float lc_eps_sigma;        /* standard deviation of epsilon, m (Eq. 3, 4)                            */
    uint64_t seed;             /* counter-based generator seed (G22)                                     */
    uint32_t flags;            /* MANTA_FLAG_*                                                           */
    float stop_time_s;         /* MANTA_STOP nodes: standing time at the stop line, s (2)  */
    float v0_sigma_rel;        /* per-driver desired speed (reading G27): on every edge of its route
                                  a vehicle's v0 = limit * clamp(1 + v0_sigma_rel * z, 1/2, 3/2), z ~ N(0, 1) from the
                                  counter-based generator; 0 = v0 is the limit                             */
    uint32_t stat_period_steps; /* per-edge speed statistics (inputs of Eq. 5): every this many
                                   steps each ACTIVE vehicle adds its speed to its edge's accumulators; 0 = off    */
    uint32_t stat_slice_steps;  /* steps per time slice of the statistics (e.g. 7200 = one hour)                   */
    uint32_t stat_n_slices;     /* time slices kept; samples of later steps are dropped                            */
} manta_params;

/* Per-trip state snapshot, indexed by the CALLER's trip index.  Any member may be NULL (skipped). */
typedef struct {
    uint8_t *status;           /* MANTA_WAITING / ACTIVE / DONE                                          */
    uint32_t *route_pos;       /* index into the trip's route (ACTIVE only, else 0)                      */
    uint8_t *lane;             /* ACTIVE only                                                            */
    uint8_t *tag;              /* mandatory-lane-change tag of Eq. 2 (ACTIVE only)                       */
    uint32_t *x_fx;            /* position on the edge, Q22.10 metres (ACTIVE only)                      */
    float *v;                  /* speed m/s (ACTIVE only)                                                */
    float *acc;                /* acceleration applied in the last step (ACTIVE only)                    */
    uint8_t *wait;             /* steps already stood at the stop line of a MANTA_STOP node (ACTIVE only) */
} manta_state;

typedef struct {
    uint32_t admit_step;       /* step at which the trip entered the network, MANTA_NONE if still waiting */
    uint32_t arrive_step;      /* step count at arrival (travel steps = arrive - admit), MANTA_NONE if not done */
} manta_trip_result;

typedef struct {
    uint64_t t;                /* steps simulated so far                                                 */
    uint64_t n_waiting, n_active, n_done;
    uint64_t sum_travel_steps; /* sum over DONE trips of arrive_step - admit_step                        */
    uint64_t vehicle_updates;  /* ACTIVE vehicles processed by the update, summed over steps (the metric's unit) */
    uint64_t lane_changes;     /* executed lane changes                                                  */
    uint64_t cells_examined;   /* atlas cells examined by the own-lane look-ahead (R2), summed           */
    uint64_t lc_evals;         /* updates that evaluated the adjacent lane (R5)                          */
    uint64_t n_stopped;        /* ACTIVE vehicles standing still (v = 0) now: the stuck count of a gridlocked network;
                                  n_stopped == n_active > 0 over many steps = gridlock       */
} manta_summary;

/* Optional device-memory callbacks (process-wide; install before manta_create).  alloc returns a device pointer
 * valid on `device` or NULL; free receives that pointer.  NULL, NULL restores cudaMalloc / cudaFree. */
typedef void *(*manta_alloc_fn)(uint64_t bytes, int device, void *ctx);
typedef void (*manta_free_fn)(void *ptr_dev, int device, void *ctx);
int manta_set_allocator(manta_alloc_fn alloc, manta_free_fn free_, void *ctx);

/* Builds the atlas (one row of 1 m cells per (edge, lane)) and the static tables of R0 on
 * `cuda_device`.  Errors: INVALID_ARG (NULL, params->size mismatch, non-positive dt/a/b/...), BAD_NETWORK (lanes
 * outside 1..8, length < LEN_MIN or > 65535 cells, non-finite values, head out of range, out-degree > 255,
 * more than 2^32 - 1 atlas cells, n_nodes >= 2^27, 8 n_edges + n_nodes >= 2^32), OOM, CUDA. */
int manta_create(const manta_network *net, const manta_params *params, int cuda_device, manta_sim **out);

/* Loads the demand: trip i follows route_edges[route_ptr[i] .. route_ptr[i+1]-1] ("routes are
 * fixed") and is released at depart_time_s[i].  init_pos_m / init_speed may be NULL; a trip with
 * init_pos_m[i] >= 0 is pre-placed at that position on its first edge, lane 0, with speed init_speed[i], active from
 * step 0 (R1).  Vehicle ids are ranks in the stable (depart_step, trip index) order.  May be called once per
 * simulation.  Errors: BAD_ROUTE (empty route, edge id out of range, head(e_k) != tail(e_k+1), negative departure,
 * negative / non-finite init_speed, pre-placed vehicles closer than L in one row or beyond the edge), INVALID_ARG
 * (lookback_cells too small for R5), STATE (already loaded), OOM, CUDA. */
int manta_load_trips(manta_sim *sim, uint32_t n_trips, const uint64_t *route_ptr, const uint32_t *route_edges,
                     const float *depart_time_s, const float *init_pos_m, const float *init_speed);

/* THE HOT PATH.  Advances the simulation by n_steps timesteps (rules R1-R9) and returns when they completed.
 * manta_step_async only enqueues the work on the simulation's stream; manta_sync waits for it. */
int manta_step(manta_sim *sim, uint32_t n_steps);
int manta_step_async(manta_sim *sim, uint32_t n_steps);
int manta_sync(manta_sim *sim);

/* Replica batching (the calibration runs several parameter sets per iteration): advances 2..4
 * independent simulations -- each created and loaded on its own, typically the same network and demand with
 * different model parameters -- by n_steps in ONE cooperative launch per 8,192 steps; every phase works through all
 * replicas between the same two grid barriers, so the per-step synchronisation is paid once for the batch.  Results
 * of every replica are exactly those of stepping it alone.  All simulations must be on the same device and stream, at
 * the same step counter, with the same launch geometry (n_sims = 1: plain manta_step).  Errors: INVALID_ARG, STATE
 * (the batch does not fit the device's shared memory), CUDA.  Returns after the steps completed.
 * MEASURED (profiles/r02_final.md, B200, configs[2] at 07:30): as built this is SLOWER than stepping the replicas in
 * separate manta_step calls -- 31.4 us per replica-step with 2 replicas, 40 us with 4, against 26.7 us alone --
 * because each block walks its replicas one after the other inside a phase.  Use it for its exactness guarantee
 * (one launch, identical results), not for throughput; for a parameter sweep call manta_step per replica. */
int manta_step_batch(manta_sim **sims, uint32_t n_sims, uint32_t n_steps);

/* Same as manta_step, with CUDA events recorded on the simulation's stream around every phase; adds the device
 * time of the admission, update and second (claim resolution) phases (ms, summed over the n_steps) to phase_ms[0..2].
 * For measurement only (the events cost a little); results are identical to manta_step. */
int manta_step_timed(manta_sim *sim, uint32_t n_steps, double phase_ms[3]);

/* Copies results to host buffers (each may be NULL): per-trip state, cumulative per-edge entry counts
 * ([n_edges]), per-trip admit/arrive steps ([n_trips]), and the summary counters. */
int manta_readback(manta_sim *sim, manta_state *state, uint32_t *edge_entries, manta_trip_result *trips,
                   manta_summary *summary);

/* manta_readback for callers that must not allocate device memory.  manta_readback takes a temporary staging block
 * (28 bytes per trip) from cudaMalloc or the manta_set_allocator callback on every call and frees it again.  Two kinds
 * of caller cannot afford that: a host program that has already given all free device memory to a pool of its own (a
 * training framework's caching allocator, a fixed memory partition) -- there a fresh cudaMalloc simply fails -- and a
 * loop that reads results while other streams are busy, because cudaMalloc / cudaFree may wait for the whole device
 * and stall that work.  This variant runs the same two gather kernels with their staging arrays inside a fixed
 * array that is part of the library image itself (static __device__, 7 MiB: MANTA_NOALLOC_MAX_TRIPS x 28 B; every
 * device that loads libmanta.so holds it until the process exits).  It calls no cudaMalloc, cudaFree, allocator
 * callback or other routine that allocates device memory (host side: two small std::vector temporaries for the
 * summary).  Arguments, outputs and results are exactly those of manta_readback.
 *   - Limit: simulations with more than MANTA_NOALLOC_MAX_TRIPS trips are refused with MANTA_ERR_INVALID_ARG and a
 *     text that names the limit; nothing is read in that case.  Use manta_readback for those.
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, once per device, with
 *     that device current).  Make that first call before any stream capture begins.
 *   - All calls on a device share the one array and it keeps the previous call's contents; each call clears the part
 *     it reads before its kernels run.  Two calls that overlapped on the GPU would race on it; inside one process the
 *     library therefore holds a lock from the first kernel until the results are on the host, so calls from several
 *     threads (or for several simulations) simply run one after the other. */
#define MANTA_NOALLOC_MAX_TRIPS 262144u
int manta_readback_noalloc(manta_sim *sim, manta_state *state, uint32_t *edge_entries, manta_trip_result *trips,
                           manta_summary *summary);

/* Checkpoint / resume (and tests): replaces the dynamic state by the caller's -- the arrays manta_readback returns
 * (caller trip order; status, route_pos, lane, tag, x_fx, v required, wait optional, acc ignored), the per-trip
 * admit / arrive steps, the cumulative per-edge entries (NULL: kept) and the step counter t -- and rebuilds the
 * atlas, the vehicle slots and the admission queues from it.  Summary counters that are not functions of the state
 * (vehicle_updates, lane_changes, cells_examined, lc_evals) and the speed statistics are left to restart / continue.
 * Errors: INVALID_ARG (missing array; status > 2; route position, lane, position or counter out of range; a speed
 * that is negative, not finite or above the fastest possible one = max(largest desired speed, largest init_speed)
 * + a dt; admit / arrive steps that contradict the status or lie after t; an admitted trip queued behind a waiting
 * one; two vehicles in one cell -- the last is found while rebuilding and leaves the handle unusable), STATE (no
 * trips loaded), OOM, CUDA.  Otherwise a failed call changes nothing.  NOT checked: that vehicles of one lane are at
 * least veh_len apart (a state that a run of this library or of the rules R1-R8 produced always is). */
int manta_load_state(manta_sim *sim, uint32_t t, const manta_state *state, const manta_trip_result *trips,
                     const uint32_t *edge_entries);

/* Per-edge speed statistics (manta_params.stat_*): sum_q8[slice * n_edges + e] = sum over the samples of
 * rint(v * 256) (v in m/s), samples[slice * n_edges + e] = their number; mean speed = sum / (256 * samples): the
 * per-edge average the paper's calibration compares with measured speeds (Eq. 5).  Either array
 * may be NULL.  Error STATE if the statistics are off. */
int manta_readback_edge_speeds(manta_sim *sim, uint64_t *sum_q8, uint32_t *samples);

/* Logical atlas of the current step for tests: occ[i] = 0 (empty) or 1 + frac10 per padded cell, spd[i] the
 * occupant's speed; row (e, lane) starts at cell_off[e] + lane * pitch[e].  Sizes via manta_atlas_cells.  (On the
 * device the atlas is a 1-bit occupancy plane plus an 8-byte payload plane; this call expands it.) */
uint64_t manta_atlas_cells(const manta_sim *sim);
int manta_readback_atlas(manta_sim *sim, uint16_t *occ, float *spd, uint32_t *cell_off, uint32_t *pitch);

/* Bounds-checking build (libmanta_check.so, compiled with -DMANTA_CHECK): every index the kernels compute is compared
 * with its array's size; returns the largest failure code seen since manta_load_trips (0 = none).  The product
 * build has no checks compiled in and returns -1. */
int manta_check_failures(manta_sim *sim);

/* Self-test of the software grid barrier that separates the phases of a step inside the persistent kernel (tests).
 * One cooperative launch in the step kernel's geometry (blocks of 512 threads, two per SM) runs n_rounds rounds of:
 * every block writes the round number to its own 32 words (plain stores), barrier, every block reads all blocks'
 * words (plain loads), barrier.  *n_stale = words read with another round's value (must be 0), *n_blocks (may be
 * NULL) = blocks launched.  Uses cudaMalloc / the default stream of `cuda_device`; needs no simulation.  Errors:
 * INVALID_ARG (NULL, 0 or more than 2^22 rounds), STATE (no cooperative launch), CUDA (time-out, lost arrivals). */
int manta_selftest_grid_barrier(int cuda_device, uint32_t n_rounds, uint64_t *n_stale, uint32_t *n_blocks);

int manta_set_stream(manta_sim *sim, void *cuda_stream);   /* cudaStream_t; work already enqueued is not moved */
/* Process-wide: the stream (cudaStream_t, NULL = legacy default stream) that simulations created AFTERWARDS use from
 * manta_create on (its uploads and memsets included).  All work of a simulation and the frees of manta_destroy
 * (after a synchronize) are ordered on its one stream; an allocator callback that hands out stream-ordered memory
 * (PyTorch's caching allocator) must allocate for that stream. */
int manta_set_default_stream(void *cuda_stream);
/* Switches between the persistent kernel and kernel-per-phase stepping for the following manta_step calls
 * (on != 0: as if MANTA_FLAG_MULTI_KERNEL had been given).  Results are identical either way; profilers use it to
 * advance a simulation in one launch and then look at single phases. */
int manta_set_multi_kernel(manta_sim *sim, int on);
uint64_t manta_launch_count(const manta_sim *sim);         /* kernels launched by this simulation so far   */
uint64_t manta_device_bytes(const manta_sim *sim);         /* device memory held                           */
void manta_destroy(manta_sim *sim);
const char *manta_last_error(const manta_sim *sim);        /* sim may be NULL: error of the last failed create */

#ifdef __cplusplus
}
#endif
#endif
