// manta_device.cuh -- device-side data layout and per-vehicle arithmetic of the MANTA step (sm_100a).
//
// Rules R0-R9 and readings G1-G25 are in DESIGN.md sections 2-3; the paper passages are cited per function.
// Deterministic mode: this translation unit is compiled with -fmad=false and IEEE division, and every
// floating-point expression below is written one operation per statement in the order DESIGN.md gives.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace manta {

typedef unsigned long long u64;

// ---------------------------------------------------------------------------------------------------------
// Layout in HBM
//
// Traffic atlas (one cell per metre of lane, at most one vehicle per cell, the cell records the
// occupant's velocity), stored as two SoA planes over the same cell index:
//   bits[2]  OCCUPANCY plane, 1 bit per 1 m cell, packed 64 cells per u64 word.  Buffer t & 1 holds the marks of
//            time t.  Step t reads buffer t & 1 and turns buffer (t+1) & 1 -- which still holds the marks of time
//            t-1 -- into the marks of time t+1 with XOR toggles: every vehicle toggles its own time-(t-1) mark off
//            and its time-(t+1) mark on.  XOR commutes, so a cell that one vehicle leaves and another enters in
//            the same step ends up set whatever the order, and a vehicle whose old and new mark share a word
//            issues ONE atomic (none at all if it did not change cell).  No phase reads and writes one buffer.
//            A 256-cell look-ahead is 4-5 words (one or two sectors).
//   pay[2]   PAYLOAD plane: one 8-byte entry { frac10 of the occupant's Q22.10 position, its fp32 speed bits } per
//            aligned group of FOUR cells when vehicles are at least 4 m long (pay_shift = 2: such a group never holds
//            two vehicles, and the occupant's cell is known from the occupancy bit), one entry per cell otherwise
//            (pay_shift = 0).  Buffer t & 1 is valid where a bit is set in bits[t & 1]; never cleared.
// Row (edge e, lane l) starts at cell  cell_off[e] + l * pitch(e),  pitch = len_c rounded up to 64 cells, so every
// row starts on a word boundary and no word is shared by two rows.
//
// Route store: one 16-byte RouteRec per route entry (edge attributes inlined, so following a route costs one
// gather instead of route -> edge table); consecutive entries of a trip are consecutive in memory:
//   w0 cell_off   w1 geom   w2 edge id   w3 speed limit v0 (fp32 bits)
// geom bits: 0-15 len_c | 16-19 lanes | 20-22 lo | 23-25 hi | 26 last | 27 head-node PRIORITY | 28-30 lane | 31 tag
// (lane / tag are only meaningful in a vehicle's private copy).  The route store is read only when a vehicle
// enters an edge or changes lane (admission, cross phase, second pass of the update), never by the per-step
// look-ahead: what the look-ahead needs of the next four route edges is cached in the vehicle's state (S2, S3).
//
// Active vehicles: n_seg SEGMENTS of seg_cap slots, four uint4 per vehicle (64 bytes), updated IN PLACE.
// A segment is processed by one thread block per phase.  Every MANTA_SORT_EVERY timesteps all live slots are
// re-sorted by atlas position (counting sort on absolute cell >> MANTA_BUCKET_SHIFT, into the second state buffer)
// and dealt out in equal shares: segment s then holds the vehicles of one contiguous stretch of the atlas, so a
// block's look-ahead, payload and mark traffic stays inside a few hundred KB that its SM's L1 and one L2 partition
// can hold, and DRAM sees runs of neighbouring sectors instead of single random ones.  Dead slots (arrived
// vehicles, id = NONE) are dropped by the same pass.  Between two sorts a vehicle keeps its slot; admission
// appends to the segment that currently covers the origin edge's stretch.
//   S0 = { x_fx | stop-line counter << 28 (R8s), v bits, absolute cell of the time-(t-1) mark or NONE, vehicle id or NONE (dead slot) }
//   S1 = { row0 = absolute cell at which the row of the vehicle's own lane starts, geom (+ lane, tag),
//          route cursor (absolute RouteRec index), v0 bits }
//   S2 = { word index (cell >> 6) of the row the look-ahead continues in on route edges +1, +2, +3, +4
//          (lane clamped hop by hop, R2) }
//   S3 = { len_c of edges +1 | +2 << 16, len_c of edges +3 | +4 << 16 (0 = the route ended before),
//          bit 0: the route goes on past edge +4, bits 1-3: the (clamped) lane the look-ahead is in on edge +4,
//          bits 4-30: head node of this edge if it is a PRIORITY or STOP node (its claim word of R8), bit 31: STOP node,
//          lane entry (e+ * 8 + lanes(e+) - 1) the vehicle heads for at this edge's end }
// A stayer rewrites S0 only (S1 when its tag or lane changed, S2/S3 when its lane changed).  A vehicle that
// arrives leaves a GHOST in its slot for one step, which toggles the vehicle's last mark off (that mark is in the
// plane everybody reads during the arrival step, so it cannot be cleared earlier) and then frees the slot.
// Two per-segment lists of 16-byte entries carry the few vehicles that need the second phase: the CROSS list
// (edge-end candidates, whose claim must be resolved) and the DEFERRED list (vehicles that must look at the
// adjacent lane, R5, or whose look-ahead window does not fit the fast search; neither can reach its edge end in
// this step nor mark an entry window, so nothing they do can matter to a claim or to the fused admission: both
// lists are worked off in the same phase, by different warps).
// ---------------------------------------------------------------------------------------------------------

#define GEOM_LEN(g) ((g) & 0xFFFFu)
#define GEOM_LANES(g) (((g) >> 16) & 15u)
#define GEOM_LO(g) (((g) >> 20) & 7u)
#define GEOM_HI(g) (((g) >> 23) & 7u)
#define GEOM_LAST(g) (((g) >> 26) & 1u)
#define GEOM_PRIO(g) (((g) >> 27) & 1u)
#define GEOM_LANE(g) (((g) >> 28) & 7u)
#define GEOM_TAG(g) ((g) >> 31)
#define GEOM_STATIC_MASK 0x0FFFFFFFu
#define X_MASK 0x0FFFFFFFu     // S0.x: bits 0-27 position (Q22.10, edges have at most 65,535 cells), bits 28-30 stop-line counter of R8s
#define WAIT_SHIFT 28
#define NODE_MASK 0x07FFFFFFu  // head-node field of edge_tab / S3.z >> 4: bits 0-26 node id, bit 27 the node is a STOP node
#define CELL_NONE 0xFFFFFFFFu
#define ID_GHOST 0xFFFFFFFEu   // slot of a vehicle that arrived in the previous step: clears its last mark, then dies
#ifndef MANTA_SORT_EVERY
#define MANTA_SORT_EVERY 64u      // timesteps between two spatial re-sorts of the vehicle slots
#endif
#ifndef MANTA_BUCKET_SHIFT
#define MANTA_BUCKET_SHIFT 8      // sort key = absolute atlas cell >> this
#endif

enum { KIND_STAY = 0, KIND_DONE = 1, KIND_CAND = 2 };

// ---------------------------------------------------------------------------------------------------------
// Bounds checks of the MANTA_CHECK build (libmanta_check.so; compute-sanitizer is closed on the GPU pool this was
// developed on, so the library checks its own indices): every computed index into the atlas planes, the payload
// planes, the vehicle arrays and lists, the claim words, the route store and the per-edge arrays is compared with
// the size of its array; the largest failure code is kept in g_check.fail and read by manta_check_failures().
// Compiled out of the product build.
struct CheckCtx {
    unsigned long long plane_words, pay_entries, n_cells, n_claims, route_total, slots, n_edges, n_trips;
    unsigned int fail;
};
#ifdef MANTA_CHECK
__device__ CheckCtx g_check;
#define MANTA_ASSERT(cond, code) do { if (!(cond)) atomicMax(&g_check.fail, (unsigned int)(code)); } while (0)
#else
#define MANTA_ASSERT(cond, code) do { } while (0)
#endif
enum { CHK_PLANE = 1, CHK_PAY = 2, CHK_CELL = 3, CHK_CLAIM = 4, CHK_ROUTE = 5, CHK_SLOT = 6, CHK_EDGE = 7, CHK_ID = 8, CHK_LIST = 9 };

struct Counters {                        // grid barrier of the persistent kernel; one 128-byte line per word, so
    unsigned int bar_count, pad0[31];    // the arrival atomics, the generation polls and the abort flag do not
    unsigned int bar_gen, pad1[31];      // queue up on one L2 sector
    unsigned int abort, pad2[31];
};

// per-block private statistics and result counters (no global atomics on the hot path; summed at readback)
struct BlockStats {
    u64 lane_changes, cells_examined, lc_evals, n_updates, n_done, sum_travel, pad0, pad1;
};

// one buffer of vehicle state (see the layout comment); acc is optional (MANTA_FLAG_RECORD_ACC)
struct StBuf {
    uint4 *S0, *S1, *S2, *S3;
    float *acc;
};

struct DevP {
    // model constants (R0), rounded once on the host from double
    float dt, a, T, s0, veh_len, C1, HALF_DT, VSCALE, ADT;
    float dlc_thr, alpha, gap_low, gap_high, eps_sigma;
    float vcap;                  // R0: no vehicle is ever faster (largest desired or initial speed + a dt, rounded up); Z_out is built on it
    uint32_t H, lookback, L_c, Z_out, Z_in, Lam;
    int32_t L_fx;
    uint32_t seed_lo, seed_hi;
    uint32_t n_edges, n_queues, flags;
    uint32_t n_seg, seg_cap;     // active-vehicle segments
    // STOP control (R8s), per-driver desired speed (R3s), per-edge speed statistics (R9s)
    uint32_t W_stop;             // steps a vehicle stands at the stop line of a STOP node
    uint32_t id_mask;            // low bits of a claim key that hold the vehicle id: 2^24 - 1 if the network has STOP nodes (the turn rank sits above), else all ones
    float v0_sigma_rel;
    uint32_t stat_period, stat_slice, stat_n_slices;
    u64 *stat_sum;               // [stat_n_slices * n_edges]
    uint32_t *stat_cnt;
    const uint4 *edge_stop;      // per edge whose head is a STOP node: {n_in * n_out of the node, in_idx * n_out, first out-edge of the node, 0}
    // network
    const uint4 *edge_tab;       // per edge: {cell_off, geom (len | lanes | PRIORITY bit), head node | STOP << 27, v0 bits}
    // atlas
    u64 *bits[2];
    uint2 *pay[2];
    uint32_t pay_shift;          // payload entry of a cell = pay[cell >> pay_shift]: 2 (one entry per aligned group of four cells) if L >= 4 m, else 0
    // routes
    const uint4 *route;
    // vehicles: segment s occupies slots [s * seg_cap, s * seg_cap + seg_cnt[s]) (live and dead slots)
    StBuf st[2];                 // step t uses buffer sbuf_of(t); the periodic spatial re-sort copies into the other one
    uint32_t *seg_cnt;
    uint4 *xlist;                // cross list of segment s at [s * seg_cap, ...): {slot, claim word, cursor, id}
    uint4 *dlist;                // deferred list of segment s, same place: {slot, lead_abs, v_lead bits, 0 | 1 found | 2 search to do}
    uint32_t *seg_xn, *seg_qn;   // entries of the two lists of each segment (written by the update phase)
    // spatial re-sort (every MANTA_SORT_EVERY steps): counting sort of the live slots by atlas bucket
    uint32_t n_buckets;          // buckets of 2^MANTA_BUCKET_SHIFT atlas cells
    uint32_t *sort_hist;         // [n_buckets + 1] counts, then exclusive offsets
    uint32_t *sort_part;         // [n_seg] per-block partial sums of the scan; [n_seg] = live total
    uint32_t *sort_rank;         // [n_seg * seg_cap] rank of each slot inside its bucket (NONE = dead)
    uint32_t *bucket_seg;        // [n_buckets] segment that holds the bucket's vehicles: where admission appends
    // per vehicle id
    const uint32_t *route_start;
    const uint32_t *route_len;   // entries of the trip's route (manta_load_state validates route positions against it)
    const uint32_t *q_begin;     // [n_queues] index in q_ent of the queue's first entry (q_state moves on; this does not)
    uint32_t *admit_step;
    uint32_t *arrive_step;
    // admission queues: one FIFO per origin edge (reading G25), entries in vehicle-id order
    const uint4 *q_row;          // [n_queues] {cell_off, len_c | lanes << 16, claim word of the tail node if it is PRIORITY else NONE, edge id}
    const uint4 *q_ent;          // [waiting trips + 1] {vehicle id, depart_step, route cursor, depart_step of the next entry}
    const uint32_t *q_end;       // [n_queues] index in q_ent one past the queue's last entry
    uint4 *q_state;              // [n_queues] head of the FIFO: {its depart_step (NONE: exhausted), index in q_ent, vehicle id, route cursor}
    uint2 *cand_info;            // [n_trips] written by an edge-end candidate: {lane entry e+ * 8 + l+ it heads for, cell it would land in}
    // claims, counters, tables
    u64 *claim;                  // [n_edges * 8 + n_nodes]
    uint32_t *edge_entries;
    const uint32_t *P_mlc;       // [5 * Lam + 1]
    Counters *ctr;
    u64 *dbg_buf;               // [n_seg * 8] timestamps (MANTA_DBG builds only)
    BlockStats *blk;
};

__device__ __forceinline__ int sbuf_of(uint32_t t) { return (int)((t / MANTA_SORT_EVERY) & 1u); }
__device__ __forceinline__ uint32_t pitch_of(uint32_t len_c) { return (len_c + 63u) & ~63u; }

// ------------------------------------------------------------------------------------------- G22: rng(id, t, k)
__device__ __forceinline__ uint32_t mix32(uint32_t h)
{
    h ^= h >> 16;
    h *= 0x7feb352du;
    h ^= h >> 15;
    h *= 0x846ca68bu;
    h ^= h >> 16;
    return h;
}
__device__ __forceinline__ uint32_t rng32(const DevP &P, uint32_t id, uint32_t t, uint32_t k)
{
    uint32_t h = mix32(P.seed_lo + 0x9E3779B9u * (id + 1u));
    h = mix32((h ^ P.seed_hi) + 0x85EBCA6Bu * (t + 1u));
    h = mix32(h + 0xC2B2AE35u * (k + 1u));
    return h;
}
// R6: epsilon of Eq. (3), (4) as an integer Irwin-Hall sum of 12 bytes
__device__ __forceinline__ float eps_draw(const DevP &P, uint32_t id, uint32_t t, uint32_t k0)
{
    int sum = 0;
#pragma unroll
    for (uint32_t k = 0; k < 3; k++) {
        uint32_t w = rng32(P, id, t, k0 + k);
        sum += (int)(w & 255u) + (int)((w >> 8) & 255u) + (int)((w >> 16) & 255u) + (int)(w >> 24);
    }
    float e = (float)(sum - 1530);
    e = e * 0.00390625f;
    e = P.eps_sigma * e;
    return e;
}

// ------------------------------------------------------------------------------------------- R3s: per-driver v0
// every driver's desired speed on an edge is drawn around the edge's limit (reading G27):
// v0 = limit * clamp(1 + sigma z, 1/2, 3/2), z the Irwin-Hall normal of generator words 7..9 at counter 0xFFFFFFFF - r.
// Evaluated when a vehicle enters an edge (admission, claim winner, pre-placement) and kept in S1.w.
__device__ __forceinline__ uint32_t desired_speed_bits(const DevP &P, uint32_t id, uint32_t r, uint32_t limit_bits)
{
    if (!(P.v0_sigma_rel > 0.0f)) return limit_bits;
    int sum = 0;
#pragma unroll
    for (uint32_t k = 7u; k < 10u; k++) {
        uint32_t w = rng32(P, id, 0xFFFFFFFFu - r, k);
        sum += (int)(w & 255u) + (int)((w >> 8) & 255u) + (int)((w >> 16) & 255u) + (int)(w >> 24);
    }
    float z = (float)(sum - 1530);
    z = z * 0.00390625f;
    float f = P.v0_sigma_rel * z;
    f = 1.0f + f;
    f = fmaxf(f, 0.5f);
    f = fminf(f, 1.5f);
    return __float_as_uint(__uint_as_float(limit_bits) * f);
}

// ------------------------------------------------------------------------------------------- R3: IDM, Eq. (1)
// PAPER.md:84, delta = 4, guard G5.  One IEEE operation per statement.
__device__ __forceinline__ float idm_acc(const DevP &P, float v, float v0, bool has_leader, float s, float v_lead)
{
    float r = v / v0;
    float r2 = r * r;
    float fr = r2 * r2;
    float inter = 0.0f;
    if (has_leader) {
        float dv = v - v_lead;
        float q = v * dv;
        q = q * P.C1;
        float ss = P.T * v;
        ss = ss + q;
        ss = fmaxf(0.0f, ss);
        ss = P.s0 + ss;
        float se = fmaxf(s, 0.01f);
        float z = ss / se;
        inter = z * z;
    }
    float acc = 1.0f - fr;
    acc = acc - inter;
    acc = P.a * acc;
    return acc;
}

// ------------------------------------------------------------------------------------------- atlas row scans
// "Looking up the status of neighboring cells" on the occupancy plane: 64 cells per load, the word
// after the current one is requested before the current one is examined.
__device__ __forceinline__ u64 bits_below(uint32_t n) { return n >= 64u ? ~0ull : ((1ull << n) - 1ull); }  // n in 1..64

// first occupied cell j in [start, end) of the row whose cell 0 is absolute cell `row`; requires start < end
__device__ __forceinline__ bool first_set(const u64 *B, uint32_t row, uint32_t start, uint32_t end, uint32_t &j)
{
    const u64 *p = B + (row >> 6);
    uint32_t w = start >> 6;
    const uint32_t wl = (end - 1u) >> 6;
    MANTA_ASSERT((u64)(row >> 6) + wl < g_check.plane_words, CHK_PLANE);
    u64 m = p[w];
    u64 m_next = (w < wl) ? p[w + 1u] : 0ull;
    m &= ~0ull << (start & 63u);
    for (;;) {
        if (w == wl) m &= bits_below(end - (w << 6));
        if (m) {
            j = (w << 6) + (uint32_t)__ffsll((long long)m) - 1u;
            return true;
        }
        if (w == wl) return false;
        ++w;
        m = m_next;
        m_next = (w < wl) ? p[w + 1u] : 0ull;
    }
}
// last occupied cell j in [start, end); requires start < end
__device__ __forceinline__ bool last_set(const u64 *B, uint32_t row, uint32_t start, uint32_t end, uint32_t &j)
{
    const u64 *p = B + (row >> 6);
    uint32_t w = (end - 1u) >> 6;
    const uint32_t w0 = start >> 6;
    MANTA_ASSERT((u64)(row >> 6) + w < g_check.plane_words, CHK_PLANE);
    u64 m = p[w];
    u64 m_next = (w > w0) ? p[w - 1u] : 0ull;
    m &= bits_below(end - (w << 6));
    for (;;) {
        if (w == w0) m &= ~0ull << (start & 63u);
        if (m) {
            j = (w << 6) + 63u - (uint32_t)__clzll((long long)m);
            return true;
        }
        if (w == w0) return false;
        --w;
        m = m_next;
        m_next = (w > w0) ? p[w - 1u] : 0ull;
    }
}
// Marks are XOR toggles (see the layout comment): setting a clear bit and clearing a set bit are the same operation.
__device__ __forceinline__ void mark_toggle(u64 *B, uint32_t cell)
{
    MANTA_ASSERT(cell < g_check.n_cells, CHK_CELL);
    atomicXor(&B[cell >> 6], 1ull << (cell & 63u));
}
// a vehicle's old mark off and new mark on, merged into one atomic when both fall in one word
__device__ __forceinline__ void mark_move(u64 *B, uint32_t cell_old, uint32_t cell_new)
{
    MANTA_ASSERT(cell_old < g_check.n_cells && cell_new < g_check.n_cells, CHK_CELL);
    const u64 m_old = 1ull << (cell_old & 63u), m_new = 1ull << (cell_new & 63u);
    if ((cell_old >> 6) == (cell_new >> 6)) {
        const u64 m = m_old ^ m_new;
        if (m) atomicXor(&B[cell_new >> 6], m);
    } else {
        atomicXor(&B[cell_old >> 6], m_old);
        atomicXor(&B[cell_new >> 6], m_new);
    }
}

// Payload of the vehicle in `cell`.  Vehicles in one row are at least L apart; for L >= 4 m an aligned group of
// four cells never holds two of them at the same time, so the plane keeps ONE 8-byte entry per group (pay_shift = 2:
// 2 bytes per cell instead of 8; the reader knows the occupant's cell from the occupancy bit).  Shorter vehicles get
// one entry per cell (pay_shift = 0).
__device__ __forceinline__ void pay_store(const DevP &P, uint2 *pay, uint32_t cell, uint32_t frac, uint32_t vbits)
{
    MANTA_ASSERT((cell >> P.pay_shift) < g_check.pay_entries, CHK_PAY);
    pay[cell >> P.pay_shift] = make_uint2(frac, vbits);
}

// first occupied cell j in [start, end) of a row, for windows of at most 256 cells (H <= 256): the up-to-five words
// are requested together, then examined.  Requires start < end <= start + 256.
__device__ __forceinline__ bool first_set_w(const u64 *B, uint32_t row, uint32_t start, uint32_t end, uint32_t &j)
{
    const u64 *p = B + (row >> 6);
    const uint32_t w0 = start >> 6, wl = (end - 1u) >> 6;
    u64 m[5];
#pragma unroll
    for (uint32_t i = 0; i < 5u; i++) m[i] = (w0 + i <= wl) ? p[w0 + i] : 0ull;
    m[0] &= ~0ull << (start & 63u);
    const u64 tail = bits_below(end - (wl << 6));
#pragma unroll
    for (uint32_t i = 0; i < 5u; i++) {
        if (w0 + i == wl) m[i] &= tail;
        if (m[i]) {
            j = ((w0 + i) << 6) + (uint32_t)__ffsll((long long)m[i]) - 1u;
            return true;
        }
    }
    return false;
}
// last occupied cell j in [start, end), windows of at most 128 cells (lookback <= 128): up to three words at once
__device__ __forceinline__ bool last_set_w(const u64 *B, uint32_t row, uint32_t start, uint32_t end, uint32_t &j)
{
    const u64 *p = B + (row >> 6);
    const uint32_t w0 = start >> 6, wl = (end - 1u) >> 6;
    u64 m[3];
#pragma unroll
    for (uint32_t i = 0; i < 3u; i++) m[i] = (wl >= w0 + i) ? p[wl - i] : 0ull;
    m[0] &= bits_below(end - (wl << 6));
    const u64 head = ~0ull << (start & 63u);
#pragma unroll
    for (uint32_t i = 0; i < 3u; i++) {
        if (wl - i == w0) m[i] &= head;
        if (m[i]) {
            j = ((wl - i) << 6) + 63u - (uint32_t)__clzll((long long)m[i]);
            return true;
        }
        if (wl - i == w0) return false;
    }
    return false;
}

// R5 in one round of loads (H <= 256, lookback <= 128): lead = first occupied cell in [c, end) and lag = last occupied
// cell in [b0, c) of the row; the up-to-five words ahead and up-to-three words behind are requested together.
__device__ __forceinline__ void lead_lag_w(const u64 *B, uint32_t row, uint32_t c, uint32_t end, uint32_t b0, bool &has_a, uint32_t &ja,
                                           bool &has_b, uint32_t &jb)
{
    const u64 *p = B + (row >> 6);
    MANTA_ASSERT((u64)(row >> 6) + ((end - 1u) >> 6) < g_check.plane_words && c < end, CHK_PLANE);
    const uint32_t w0 = c >> 6, wl = (end - 1u) >> 6;        // c < end: R4 allows lane changes only before len_c - Z_out
    const uint32_t v0 = b0 >> 6, vl = (c - 1u) >> 6;         // used only when c > b0
    const bool back = c > b0;
    u64 m[5], k[3];
#pragma unroll
    for (uint32_t i = 0; i < 5u; i++) m[i] = (w0 + i <= wl) ? p[w0 + i] : 0ull;
#pragma unroll
    for (uint32_t i = 0; i < 3u; i++) k[i] = (back && vl >= v0 + i) ? p[vl - i] : 0ull;
    m[0] &= ~0ull << (c & 63u);
    const u64 tail = bits_below(end - (wl << 6));
    has_a = false;
#pragma unroll
    for (int i = 4; i >= 0; i--) {
        if (w0 + (uint32_t)i == wl) m[i] &= tail;
        if (m[i]) {
            ja = ((w0 + (uint32_t)i) << 6) + (uint32_t)__ffsll((long long)m[i]) - 1u;
            has_a = true;
        }
    }
    has_b = false;
    if (back) {
        k[0] &= bits_below(c - (vl << 6));
        const u64 head = ~0ull << (b0 & 63u);
#pragma unroll
        for (int i = 2; i >= 0; i--) {
            if (vl >= v0 + (uint32_t)i) {
                if (vl - (uint32_t)i == v0) k[i] &= head;
                if (k[i]) {
                    jb = ((vl - (uint32_t)i) << 6) + 63u - (uint32_t)__clzll((long long)k[i]);
                    has_b = true;
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------- look-ahead cache
// What R2 needs of the four route edges after the current one, for a vehicle at RouteRec `cursor` in lane l:
// the word index of the row it would continue in (lane clamped hop by hop: "the lane index carried on is the
// clamped one") and the edge lengths.  Built when a vehicle enters an edge or changes lane; off the per-step path.
// The route store is padded with 8 zero records, so the four loads are always in bounds; records past the trip's
// last one belong to another trip and are ignored (len 0).
struct Hops {
    uint4 s2, s3;
};
struct HopRecs {
    uint2 r[4];   // {cell_off, geom} of RouteRecs cursor + 1 .. cursor + 4
    uint32_t e1;  // edge id of RouteRec cursor + 1
};
// the loads, separated from the arithmetic so that callers can issue them together with their other gathers
__device__ __forceinline__ HopRecs load_hop_recs(const DevP &P, uint32_t cursor)
{
    HopRecs R;
    MANTA_ASSERT((u64)cursor + 4u < g_check.route_total + 8u, CHK_ROUTE);
    const uint4 *rp = P.route + cursor;
#pragma unroll
    for (int k = 0; k < 4; k++) R.r[k] = *reinterpret_cast<const uint2 *>(rp + k + 1);
    R.e1 = rp[1].z;
    return R;
}
// node: head node of the current edge if it is a PRIORITY node (GEOM_PRIO(geom_cur)), else ignored
__device__ __forceinline__ Hops make_hops(const HopRecs &R, uint32_t geom_cur, uint32_t l, uint32_t node)
{
    bool ended = GEOM_LAST(geom_cur) != 0u;
    uint32_t roww[4], len[4];
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const uint32_t g = R.r[k].y;
        const uint32_t lk = min(l, GEOM_LANES(g) - 1u);
        roww[k] = ended ? 0u : (R.r[k].x + lk * pitch_of(GEOM_LEN(g))) >> 6;
        len[k] = ended ? 0u : GEOM_LEN(g);
        l = ended ? l : lk;
        ended = ended || GEOM_LAST(g) != 0u;
    }
    // lane entry (e+, l+) the vehicle heads for at the end of this edge; the low 3 bits hold lanes(e+) - 1 until l'
    // is known.  Behind a PRIORITY node the claim word of R8 is the node instead: its id goes into S3.z.
    uint32_t word = 0u;
    if (!GEOM_LAST(geom_cur)) word = R.e1 * 8u + (GEOM_LANES(R.r[0].y) - 1u);
    if (GEOM_LAST(geom_cur) || !GEOM_PRIO(geom_cur)) node = 0u;
    Hops h;
    h.s2 = make_uint4(roww[0], roww[1], roww[2], roww[3]);
    h.s3 = make_uint4(len[0] | (len[1] << 16), len[2] | (len[3] << 16), (ended ? 0u : 1u) | (l << 1) | (node << 4), word);
    return h;
}
__device__ __forceinline__ Hops build_hops(const DevP &P, uint32_t cursor, uint32_t geom_cur, uint32_t l)
{
    const HopRecs R = load_hop_recs(P, cursor);
    uint32_t node = 0u;
    if (!GEOM_LAST(geom_cur) && GEOM_PRIO(geom_cur)) node = P.edge_tab[P.route[cursor].z].z;   // (with its STOP bit)
    return make_hops(R, geom_cur, l, node);
}

}  // namespace manta
