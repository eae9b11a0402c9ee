// manta_device.cuh -- device-side data layout and per-vehicle arithmetic of the MANTA step (sm_100a).
//
// Rules R0-R9 and readings G1-G25 are in DESIGN.md sections 2-3; the paper passages are cited per function.
// Deterministic mode: this translation unit is compiled with -fmad=false and IEEE division, and every
// floating-point expression below is written one operation per statement in the order DESIGN.md gives.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace manta {

// ---------------------------------------------------------------------------------------------------------
// Layout in HBM
//
// Atlas: plane occ[2] of u16 per 1 m cell (0 = empty, 1 + frac10 of the occupant's Q22.10
// position) and plane spd[2] of fp32 (occupant's speed); buffer t&1 is read in step t, buffer (t+1)&1 written.
// Row (edge e, lane l) starts at cell  cell_off[e] + l * pitch(e),  pitch = len_c rounded up to 16 cells, so
// every row starts on a 32-byte sector and 16-byte vector loads never straddle rows.
//
// Route store: one 16-byte RouteRec per route entry (edge attributes inlined, so following a route costs one
// gather instead of route -> edge table):
//   w0 cell_off   w1 geom   w2 edge id   w3 speed limit v0 (fp32 bits)
// geom bits: 0-15 len_c | 16-19 lanes | 20-22 lo | 23-25 hi | 26 last | 27 head-node PRIORITY | 28-30 lane | 31 tag
// (lane / tag are only meaningful in a vehicle's private copy of its current RouteRec).
//
// Active vehicles: compact double-buffered arrays of two uint4 per vehicle (32 bytes, one sector):
//   A0 = { x_fx, v bits, vehicle id, route cursor (absolute RouteRec index) }     A1 = current RouteRec copy
// plus a 16-byte tentative next state N written by the update phase and consumed by the commit phase:
//   N  = { x', v' bits, meta (kind | lane' << 2 | tag' << 5), claim word index }
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

enum { KIND_STAY = 0, KIND_DONE = 1, KIND_CAND = 2 };

struct Counters {
    unsigned int n_act[2];               // active-array fill of buffer 0 / 1
    unsigned int pad[2];
    unsigned long long n_done, sum_travel, n_updates;
    unsigned int bar_count, bar_gen;     // grid barrier of the persistent kernel
    unsigned int t_dev, pad2;
};

// per-block private statistics (no atomics on the hot path; summed at readback)
struct BlockStats {
    unsigned long long lane_changes, cells_examined, lc_evals, pad;
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
    uint16_t *occ[2];
    float *spd[2];
    // routes
    const uint4 *route;
    // vehicles
    uint4 *A0[2];
    uint4 *A1[2];
    uint4 *N;
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
    unsigned long long *claim;   // [n_edges * 8 + n_nodes]
    uint32_t *edge_entries;
    const uint32_t *P_mlc;       // [5 * Lam + 1]
    Counters *ctr;
    BlockStats *blk;
};

__device__ __forceinline__ uint32_t pitch_of(uint32_t len_c) { return (len_c + 15u) & ~15u; }

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
// 8 cells (16 bytes) per load; rows are 16-cell aligned so an 8-aligned group never leaves the row's padding.
__device__ __forceinline__ uint32_t nzmask8(const uint4 &w)
{
    uint32_t m = 0;
    m |= (w.x & 0xFFFFu) ? 1u : 0u;
    m |= (w.x >> 16) ? 2u : 0u;
    m |= (w.y & 0xFFFFu) ? 4u : 0u;
    m |= (w.y >> 16) ? 8u : 0u;
    m |= (w.z & 0xFFFFu) ? 16u : 0u;
    m |= (w.z >> 16) ? 32u : 0u;
    m |= (w.w & 0xFFFFu) ? 64u : 0u;
    m |= (w.w >> 16) ? 128u : 0u;
    return m;
}
__device__ __forceinline__ uint32_t code_at(const uint4 &w, uint32_t i)
{
    uint32_t word = (i & 4u) ? ((i & 2u) ? w.w : w.z) : ((i & 2u) ? w.y : w.x);
    return (i & 1u) ? (word >> 16) : (word & 0xFFFFu);
}
// first occupied cell j in [start, end) of the row starting at absolute cell `row`; returns false if none
__device__ __forceinline__ bool scan_fwd(const uint16_t *occ, uint32_t row, uint32_t start, uint32_t end, uint32_t &j,
                                         uint32_t &code)
{
    for (uint32_t base = start & ~7u; base < end; base += 8u) {
        uint4 w = *reinterpret_cast<const uint4 *>(occ + (size_t)row + base);
        uint32_t m = nzmask8(w);
        if (start > base) m &= 0xFFu << (start - base);
        if (end - base < 8u) m &= (1u << (end - base)) - 1u;
        if (m) {
            uint32_t i = (uint32_t)__ffs((int)m) - 1u;
            j = base + i;
            code = code_at(w, i);
            return true;
        }
    }
    return false;
}
// last occupied cell j in [start, end)
__device__ __forceinline__ bool scan_bwd(const uint16_t *occ, uint32_t row, uint32_t start, uint32_t end, uint32_t &j,
                                         uint32_t &code)
{
    if (end <= start) return false;
    for (int base = (int)((end - 1u) & ~7u); base + 8 > (int)start; base -= 8) {
        uint4 w = *reinterpret_cast<const uint4 *>(occ + (size_t)row + (uint32_t)base);
        uint32_t m = nzmask8(w);
        if ((int)start > base) m &= 0xFFu << (start - (uint32_t)base);
        if (end - (uint32_t)base < 8u) m &= (1u << (end - (uint32_t)base)) - 1u;
        if (m) {
            uint32_t i = 31u - (uint32_t)__clz((int)m);
            j = (uint32_t)base + i;
            code = code_at(w, i);
            return true;
        }
    }
    return false;
}

}  // namespace manta
