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
//   bits[3]  OCCUPANCY plane, 1 bit per 1 m cell, packed 64 cells per u64 word.  Buffer t % 3 holds the marks of
//            time t: step t reads buffer t % 3, sets the time-(t+1) marks in buffer (t+1) % 3 and clears its own
//            time-(t-1) marks in buffer (t+2) % 3, so a buffer is all-zero again when it is next written and no
//            phase both reads and writes one buffer.  A 256-cell look-ahead is 4-5 words (one or two sectors).
//   pay[2]   PAYLOAD plane, 8 bytes per cell: { frac10 of the occupant's Q22.10 position, its fp32 speed bits }.
//            Buffer t & 1 is valid for the cells whose bit is set in bits[t % 3]; never cleared.
// Row (edge e, lane l) starts at cell  cell_off[e] + l * pitch(e),  pitch = len_c rounded up to 64 cells, so every
// row starts on a word boundary and no word is shared by two rows.
//
// Route store: one 16-byte RouteRec per route entry (edge attributes inlined, so following a route costs one
// gather instead of route -> edge table); consecutive entries of a trip are consecutive in memory:
//   w0 cell_off   w1 geom   w2 edge id   w3 speed limit v0 (fp32 bits)
// geom bits: 0-15 len_c | 16-19 lanes | 20-22 lo | 23-25 hi | 26 last | 27 head-node PRIORITY | 28-30 lane | 31 tag
// (lane / tag are only meaningful in a vehicle's private copy).
//
// Active vehicles: compact double-buffered arrays of two uint4 per vehicle (32 bytes, one sector); the update
// phase reads buffer t & 1 and writes the survivors, compacted, to buffer (t+1) & 1:
//   S0 = { x_fx, v bits, vehicle id, route cursor (absolute RouteRec index) }
//   S1 = { cell_off, geom (+ lane, tag), absolute cell of the time-(t-1) mark or NONE, v0 bits }
// Cross list: 8-byte entries made by the update phase for the few vehicles that need the second phase
// (edge-end candidates, whose claim must be resolved, and arrivals, whose time-t mark must be cleared).
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
#define CELL_NONE 0xFFFFFFFFu
#define XL_DONE 0x80000000u

enum { KIND_STAY = 0, KIND_DONE = 1, KIND_CAND = 2 };

struct Counters {
    u64 fill[2];                         // low 32 bits: fill of active buffer k; high 32: cross-list entries made while filling it
    u64 n_done, sum_travel, n_updates;
    unsigned int bar_count, bar_gen;     // grid barrier of the persistent kernel
    unsigned int abort, pad;
};

// per-block private statistics (no atomics on the hot path; summed at readback)
struct BlockStats {
    u64 lane_changes, cells_examined, lc_evals, pad;
};

struct DevP {
    // model constants (R0), rounded once on the host from double
    float dt, a, T, s0, veh_len, C1, HALF_DT, VSCALE, ADT;
    float dlc_thr, alpha, gap_low, gap_high, eps_sigma;
    uint32_t H, lookback, L_c, Z_out, Z_in, Lam;
    int32_t L_fx;
    uint32_t seed_lo, seed_hi;
    uint32_t n_edges, n_queues, flags, cap;
    // network
    const uint4 *edge_tab;       // per edge: {cell_off, geom (len | lanes | PRIORITY bit), head node, v0 bits}
    const uint32_t *head;        // head node per edge (PRIORITY claims only)
    // atlas
    u64 *bits[3];
    uint2 *pay[2];
    // routes
    const uint4 *route;
    // vehicles
    uint4 *S0[2];
    uint4 *S1[2];
    uint2 *xlist;                // cross list: {XL_DONE, cell to clear} or {position in the next buffer, claim word}
    float *acc[2];               // optional (MANTA_FLAG_RECORD_ACC): acceleration applied in the last step
    // per vehicle id
    const uint32_t *depart_step;
    const uint32_t *route_start;
    uint32_t *admit_step;
    uint32_t *arrive_step;
    // admission queues: one FIFO per origin edge (reading G25)
    const uint32_t *q_edge;
    const uint32_t *q_ptr;
    const uint32_t *q_ids;
    uint32_t *q_head;
    // claims, counters, tables
    u64 *claim;                  // [n_edges * 8 + n_nodes]
    uint32_t *edge_entries;
    const uint32_t *P_mlc;       // [5 * Lam + 1]
    Counters *ctr;
    BlockStats *blk;
};

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
__device__ __forceinline__ void mark_set(u64 *B, uint32_t cell) { atomicOr(&B[cell >> 6], 1ull << (cell & 63u)); }
__device__ __forceinline__ void mark_clear(u64 *B, uint32_t cell) { atomicAnd(&B[cell >> 6], ~(1ull << (cell & 63u))); }

}  // namespace manta
