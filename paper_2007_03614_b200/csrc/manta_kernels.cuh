// manta_kernels.cuh -- the three phases of one MANTA timestep as device functions, plus their kernels.
//
//   A admit   (R1)      : one thread per origin-edge FIFO; idle queues cost one coalesced load (q_next); a due head
//                         trip is released if its entry window is free
//   U update  (R2-R9)   : one thread block per vehicle segment, one thread per active vehicle, state updated in
//                         place, no block barrier inside.  Branch-free for nearly every vehicle: the (at most
//                         eight) occupancy words of the whole look-ahead window -- own row and the rows it continues
//                         in on the next route edges, whose addresses come from the vehicle's own state -- are
//                         requested together, searched with selects and one find-first-set, then the leader's
//                         payload is fetched; IDM, lane-change pre-tests, integration, classification.  Vehicles
//                         that stay on their edge finish the step here: next state, time-(t+1) mark and payload,
//                         time-(t-1) mark toggled off.  Edge-end candidates post a min-id claim and a cross-list
//                         entry.  Vehicles that must look at the adjacent lane (~6 %) or whose window does not fit
//                         the fast search are put on the deferred list: they cannot reach their edge end in this
//                         step, so they do not hold their warps here.
//   X second  (R5-R9)   : one thread per list entry, densely packed: cross-list entries resolve their claim (winner
//                         moves to its next route edge and rebuilds its look-ahead cache, loser holds at the stop
//                         line) and write their mark; deferred entries run the adjacent-lane search, gap acceptance
//                         and the rest of the update.
//
// A grid-wide barrier separates the phases: the software barrier of k_persistent (one cooperative launch runs
// many timesteps), or kernel boundaries (k_admit / k_update / k_second: MANTA_FLAG_MULTI_KERNEL, manta_step_timed).
#pragma once
#include "manta_device.cuh"

namespace manta {

#ifndef MANTA_NT
#define MANTA_NT 512      // threads per block of the step kernels
#endif
#ifndef MANTA_MINB
#define MANTA_MINB 2      // blocks per SM the step kernels are compiled for
#endif
#ifndef MANTA_TWO_STAGE
#define MANTA_TWO_STAGE 1  // update pass as two software-pipelined stages per chunk through shared memory (needs MANTA_REC_BYTES of dynamic shared memory)
#endif
#define MANTA_REC_BYTES (MANTA_TWO_STAGE ? 2 * 3 * 16 * MANTA_NT : 0)   // two buffers of three uint4 per thread
#ifndef MANTA_BAR
#define MANTA_BAR 3       // grid barrier: 3 = release reduction + relaxed polling of the arrival counter + one acquire load, 1 = acquire polling, 0 = atomicAdd + generation word + fences
#endif
#ifndef MANTA_DQ
#define MANTA_DQ 256      // deferred-list entries (with their vehicle records) a block keeps in shared memory; the overflow goes to P.dlist (0: all there)
#endif
#ifndef MANTA_PF
#define MANTA_PF 3        // state records requested ahead: 1 = next chunk into L2, 2 = into L1, 3 = 1 + the first chunks of step t + 1 before the grid barrier
#endif
#define MANTA_NW (MANTA_NT / 32)
#define MANTA_NS 8        // occupancy words the fast look-ahead search requests per vehicle
#define MANTA_MAX_LANES_DEV 8u

// MANTA_DBG builds stamp %globaltimer per block at the phase boundaries of one step in 32 (manta_debug_read): the
// per-block timeline that the phase structure was tuned with.  Compiled out of the product build.
#ifdef MANTA_DBG
__device__ __forceinline__ u64 gtimer() { u64 v; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(v)); return v; }
#define DBG_STAMP(k) do { if (threadIdx.x == 0u && (t & 31u) == 7u) P.dbg_buf[blockIdx.x * 8u + (k)] = gtimer(); } while (0)
#else
#define DBG_STAMP(k) do { } while (0)
#endif
__device__ __forceinline__ void prefetch_line(const void *p)
{
#if MANTA_PF == 2
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
#else
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
#endif
}
struct Lead {
    bool found;
    int32_t lead_abs;   // leader position in the follower's frame, Q22.10 (R2)
    float v_lead;
};

// Per-vehicle context carried from the leader search to the end of the update.
struct Veh {
    int32_t x;
    float v, v0;
    uint32_t id, cursor, row0, geom, prev;
    uint32_t len_c, n, l, c, pitch, wait;
    bool last;
    uint32_t claim;     // S3.w
    uint32_t hopz;      // S3.z
    // after pre_lc
    float acc_cur;
    int32_t bound;
    uint32_t tag, lt;
    bool mand, disc_pre, need_lc;
};

struct Outcome {
    uint32_t kind, nx, l_new;
    float vn, acc;
};

// shared memory of the step kernels
struct UpdateSmem {
    u64 ev[4];                    // event counters of this launch (up to 8,192 timesteps): lane changes, lane-change evaluations, arrivals, travel steps
    u64 wcnt[MANTA_NT / 32][2];   // replica batching only: cells examined, vehicle-updates per warp (its lane 0 adds, no atomics; per-thread registers in the single-simulation kernels)
    uint32_t xn, qn, flag, next;  // per segment: cross-list / deferred-list entries, next unclaimed chunk; barrier flag
    uint32_t wsum[MANTA_NW];      // re-sort: per-warp partial sums
#if MANTA_DQ
    uint4 dq[MANTA_DQ][3];        // deferred entries with their vehicle records {S0, S1, entry}; the overflow goes to P.dlist
#endif
};
enum { EV_LC = 0, EV_EVAL = 1, EV_DONE = 2, EV_TRAVEL = 3 };

__device__ __forceinline__ void veh_load(Veh &V, const uint4 &s0v, const uint4 &s1v)
{
    V.x = (int32_t)(s0v.x & X_MASK);
    V.wait = s0v.x >> WAIT_SHIFT;
    V.v = __uint_as_float(s0v.y);
    V.prev = s0v.z;
    V.id = s0v.w;
    V.row0 = s1v.x;
    V.geom = s1v.y;
    V.cursor = s1v.z;
    V.v0 = __uint_as_float(s1v.w);
    V.len_c = GEOM_LEN(V.geom);
    V.n = GEOM_LANES(V.geom);
    V.l = GEOM_LANE(V.geom);
    V.last = GEOM_LAST(V.geom) != 0u;
    V.c = (uint32_t)V.x >> 10;
    V.pitch = pitch_of(V.len_c);
}

template <bool W256>
__device__ __forceinline__ bool scan_fwd(const u64 *B, uint32_t row, uint32_t start, uint32_t end, uint32_t &j)
{
    if (W256) return first_set_w(B, row, start, end, j);
    return first_set(B, row, start, end, j);
}
template <bool W256>
__device__ __forceinline__ bool scan_bwd(const u64 *B, uint32_t row, uint32_t start, uint32_t end, uint32_t &j)
{
    if (W256) return last_set_w(B, row, start, end, j);
    return last_set(B, row, start, end, j);
}

// ------------------------------------------------------------------------------------------------ R2
// Leader search along the own lane and on along the route ("looking up the status of neighboring
// cells"; G16).  Result: the leader's absolute atlas cell and its distance in cells from the tail of the
// follower's edge.
struct Hit {
    bool found;
    uint32_t cell, dist;
};

// Generic walk (any H, any number of hops): one row after the other, route records fetched as the walk reaches
// them.  Used by the second pass for the few vehicles whose window does not fit the fast search, and by every
// vehicle when H > 256.
__device__ __forceinline__ Hit walk_rows(const DevP &P, const u64 *B, const Veh &V, uint32_t &examined)
{
    Hit h;
    h.found = false;
    h.cell = 0u;
    h.dist = 0u;
    const uint4 *rp = P.route + V.cursor;
    uint32_t hop = 0u, row = V.row0, len = V.len_c, start = V.c + 1u, l = V.l, rem = P.H, dist_base = 0u;
    bool last = V.last;
    for (;;) {
        const uint32_t end = min(len, start + rem);
        if (start < end) {
            uint32_t j;
            if (first_set(B, row, start, end, j)) {
                examined += j - start + 1u;
                h.found = true;
                h.cell = row + j;
                h.dist = dist_base + j;
                return h;
            }
            examined += end - start;
            rem -= end - start;
        }
        if (rem == 0u || last) return h;
        hop += 1u;
        const uint2 rn = *reinterpret_cast<const uint2 *>(rp + hop);
        dist_base += len;
        len = GEOM_LEN(rn.y);
        l = min(l, GEOM_LANES(rn.y) - 1u);
        row = rn.x + l * pitch_of(len);
        start = 0u;
        last = GEOM_LAST(rn.y) != 0u;
    }
}

__device__ __forceinline__ uint32_t ffs64(u64 m)   // index of the lowest set bit; m != 0
{
    return (uint32_t)__ffsll((long long)m) - 1u;
}

// Fast search (H <= 256).  The window is a sequence of at most five segments -- the rest of the own row, then
// the first cells of the rows cached in S2 / S3 -- of n_0 .. n_4 occupancy words; word slot s of the sequence
// lives at word address s + A_j, j the segment it falls in.  All MANTA_NS word loads are issued before any is
// examined.  Bits past the end of a segment can only be padding (never set) or lie beyond the H-th examined cell,
// which the final distance test rejects, so no tail masks are needed.
//   own-row part : `own` cells starting at cell `start` of the row whose cell 0 is absolute cell row0 (own = 0: none)
//   hops         : rows s2, lengths s3.x / s3.y; the first hop row starts dist_hops cells from the tail of the
//                  vehicle's edge; at most `budget` cells are examined in total
// Returns WIN_DONE (h valid: leader found, or the window is exhausted / the route ends), WIN_MORE (nothing found
// and the look-ahead goes on past the four cached hops: budget_left cells remain, starting dist_next cells from
// the tail) or WIN_NOFIT (more than MANTA_NS words and nothing in the first MANTA_NS of them: use walk_rows).
enum { WIN_DONE = 0, WIN_MORE = 1, WIN_NOFIT = 2 };
__device__ __forceinline__ int leader_window(const DevP &P, const u64 *B, uint32_t c, uint32_t row0, uint32_t start, uint32_t own,
                                             uint32_t dist_hops, uint32_t budget, const uint4 &s2, const uint4 &s3, Hit &h,
                                             uint32_t &budget_left, uint32_t &dist_next)
{
    uint32_t rem = budget - own;
    const uint32_t len1 = s3.x & 0xFFFFu, len2 = s3.x >> 16, len3 = s3.y & 0xFFFFu, len4 = s3.y >> 16;
    const uint32_t k1 = min(len1, rem);
    rem -= k1;
    const uint32_t k2 = min(len2, rem);
    rem -= k2;
    const uint32_t k3 = min(len3, rem);
    rem -= k3;
    const uint32_t k4 = min(len4, rem);
    rem -= k4;
    const uint32_t w0 = start >> 6;
    const uint32_t n0 = own ? ((start + own - 1u) >> 6) - w0 + 1u : 0u;
    const uint32_t c0 = n0, c1 = c0 + ((k1 + 63u) >> 6), c2 = c1 + ((k2 + 63u) >> 6), c3 = c2 + ((k3 + 63u) >> 6),
                   c4 = c3 + ((k4 + 63u) >> 6);
    h.found = false;
    h.cell = 0u;
    h.dist = 0u;
    budget_left = rem;
    const uint32_t d1 = dist_hops, d2 = d1 + len1, d3 = d2 + len2, d4 = d3 + len3;
    dist_next = d4 + len4;
    // A window of more than MANTA_NS words: its first MANTA_NS words are searched all the same -- slots are in order
    // of distance, so a leader found there is the leader; only if they are empty the caller must walk the rows.
    const bool nofit = c4 > (uint32_t)MANTA_NS;
    // word address of slot s = s + A_j; distance (cells from the tail of the own edge) of bit b of slot s = 64 s + b + D_j
    const uint32_t A0 = (row0 >> 6) + w0, A1 = s2.x - c0, A2 = s2.y - c1, A3 = s2.z - c2, A4 = s2.w - c3;
    u64 m[MANTA_NS];
#pragma unroll
    for (uint32_t s = 0; s < (uint32_t)MANTA_NS; s++) {
        const uint32_t A = s < c0 ? A0 : (s < c1 ? A1 : (s < c2 ? A2 : (s < c3 ? A3 : A4)));
        MANTA_ASSERT(!(s < c4) || (u64)(uint32_t)(A + s) < g_check.plane_words, CHK_PLANE);   // (A_j = row word - c_j may wrap; A_j + s does not)
        m[s] = s < c4 ? B[A + s] : 0ull;
    }
    if (n0) m[0] &= ~0ull << (start & 63u);
    u64 sel = 0ull;
    uint32_t si = 0u;
#pragma unroll
    for (int s = MANTA_NS - 1; s >= 0; s--)
        if (m[s]) {
            sel = m[s];
            si = (uint32_t)s;
        }
    if (sel) {
        const uint32_t b = ffs64(sel);
        uint32_t A = A4, D = d4 - (c3 << 6);
        if (si < c3) { A = A3; D = d3 - (c2 << 6); }
        if (si < c2) { A = A2; D = d2 - (c1 << 6); }
        if (si < c1) { A = A1; D = d1 - (c0 << 6); }
        if (si < c0) { A = A0; D = w0 << 6; }
        const uint32_t dist = (si << 6) + b + D;
        if (dist - c <= P.H) {
            h.found = true;
            h.dist = dist;
            h.cell = ((A + si) << 6) + b;
            return WIN_DONE;
        }
    }
    if (nofit) return WIN_NOFIT;
    return (rem > 0u && (s3.z & 1u)) ? WIN_MORE : WIN_DONE;
}

template <bool W256>
__device__ __forceinline__ Lead lead_from_hit(const uint2 *pay, uint32_t pay_shift, const Hit &h)
{
    Lead L;
    L.found = h.found;
    L.lead_abs = 0;
    L.v_lead = 0.0f;
    if (h.found) {
        MANTA_ASSERT((h.cell >> pay_shift) < g_check.pay_entries, CHK_PAY);
        const uint2 pc = pay[h.cell >> pay_shift];
        L.lead_abs = (int32_t)((h.dist << 10) | pc.x);
        L.v_lead = __uint_as_float(pc.y);
    }
    return L;
}

// R3 against the own-lane leader, R4 (mandatory tag of Eq. 2, lane-change desire pre-tests).
__device__ __forceinline__ void pre_lc(const DevP &P, uint32_t t, Veh &V, const Lead &ld)
{
    float s = 0.0f;
    V.bound = 0x7FFFFFFF;
    if (ld.found) {
        float sf = (float)(ld.lead_abs - V.x);
        sf = sf * 0.0009765625f;
        s = sf - P.veh_len;
        V.bound = ld.lead_abs - P.L_fx;
    }
    // R3, Eq. (1); the free-road term is kept for the discretionary pre-test of R4
    float r = V.v / V.v0;
    float r2 = r * r;
    float fr = r2 * r2;
    float inter = 0.0f;
    if (ld.found) {
        float dv = V.v - ld.v_lead;
        float q = V.v * dv;
        q = q * P.C1;
        float ss = P.T * V.v;
        ss = ss + q;
        ss = fmaxf(0.0f, ss);
        ss = P.s0 + ss;
        float se = fmaxf(s, 0.01f);
        float z = ss / se;
        inter = z * z;
    }
    const float one_m_fr = 1.0f - fr;
    float acc = one_m_fr - inter;
    acc = P.a * acc;
    V.acc_cur = acc;
    // R4: mandatory tag, Eq. (2)
    uint32_t tag = GEOM_TAG(V.geom);
    if (tag == 0u && !V.last && V.n >= 2u) {
        const uint32_t dcell = V.len_c - V.c;
        if (dcell <= P.Lam)
            tag = 1u;
        else if (dcell <= 5u * P.Lam) {
            const uint32_t u0 = rng32(P, V.id, t, 0u);
            if (u0 < P.P_mlc[dcell]) tag = 1u;
        }
    }
    V.tag = tag;
    const uint32_t lo = GEOM_LO(V.geom), hi = GEOM_HI(V.geom);
    const int dir = (t & 1u) ? -1 : 1;  // G11
    const int lt_s = (int)V.l + dir;
    V.mand = false;
    V.disc_pre = false;
    V.lt = 0u;
    const bool possible = lt_s >= 0 && lt_s < (int)V.n && V.c >= P.Z_in && V.c + P.Z_out < V.len_c;
    if (possible) {
        const uint32_t lt = (uint32_t)lt_s;
        V.lt = lt;
        const bool l_in = (V.l >= lo && V.l <= hi), lt_in = (lt >= lo && lt <= hi);
        V.mand = tag == 1u && !l_in && ((V.l < lo && dir > 0) || (V.l > hi && dir < 0));
        if (!(tag == 1u && !lt_in) && ld.found) {  // G9: impeded in the own lane
            float af = P.a * one_m_fr;
            float g = af - V.acc_cur;
            V.disc_pre = g > P.dlc_thr;
        }
    }
    V.need_lc = V.mand || V.disc_pre;
}

// R5 gaps, R6 gap acceptance (Eq. 3, 4), R7 integration and clamp, R8 edge-end classification and claim.
// (has_a, x_a, v_a) / (has_b, x_b, v_b): lead / lag found in the target lane (Q22.10 position, speed); ignored
// unless V.need_lc.
__device__ __forceinline__ Outcome post_lc(const DevP &P, uint32_t t, const Veh &V, bool has_a, int32_t x_a, float v_a,
                                           bool has_b, int32_t x_b, float v_b)
{
    const int32_t x = V.x;
    const float v = V.v;
    uint32_t l_new = V.l;
    float acc = V.acc_cur;
    int32_t bound = V.bound;
    if (V.need_lc) {
        float gap_lead = 0.0f, gap_lag = 0.0f;
        if (has_a) {
            float gf = (float)(x_a - x);
            gf = gf * 0.0009765625f;
            gap_lead = gf - P.veh_len;
        }
        if (has_b) {
            float gf = (float)(x - x_b);
            gf = gf * 0.0009765625f;
            gap_lag = gf - P.veh_len;
        }
        const float acc_tgt = idm_acc(P, v, V.v0, has_a, gap_lead, v_a);
        const float gain = acc_tgt - V.acc_cur;
        const bool want = V.mand || (V.disc_pre && gain > P.dlc_thr);
        if (want) {
            // R6: gap acceptance, Eq. (3), (4)
            const float g0 = (v < 11.176f) ? P.gap_low : P.gap_high;
            bool ok = true;
            if (has_a) {
                float t1 = P.alpha * v;
                float t2 = v - v_a;
                t2 = P.alpha * t2;
                float g = g0 + t1;
                g = g + t2;
                g = fmaxf(g0, g);
                g = g + eps_draw(P, V.id, t, 1u);
                g = fmaxf(g, 0.0f);
                if (!(gap_lead >= g)) ok = false;
            }
            if (has_b) {
                float t1 = P.alpha * v;
                float t2 = v - v_b;
                t2 = P.alpha * t2;
                float g = g0 + t1;
                g = g + t2;
                g = fmaxf(g0, g);
                g = g + eps_draw(P, V.id, t, 4u);
                float fl = v_b + P.ADT;  // hard safety floor
                fl = fl * P.dt;
                fl = fl + 0.01f;
                g = fmaxf(g, fl);
                if (!(gap_lag >= g)) ok = false;
            }
            if (ok) {
                l_new = V.lt;
                acc = fminf(V.acc_cur, acc_tgt);
                if (has_a) bound = min(bound, x_a - P.L_fx);
            }
        }
    }
    // R7: ballistic update (G4) and hard clamp
    float vn = acc * P.dt;
    vn = v + vn;
    vn = fmaxf(0.0f, vn);
    float m = v + vn;
    m = m * P.HALF_DT;
    const int32_t dx = __float2int_rn(m * 1024.0f);
    int32_t xn = x + dx;
    if (xn > bound) {
        xn = bound > x ? bound : x;
        float vc = (float)(xn - x);
        vc = vc * P.VSCALE;
        vn = fminf(vn, vc);
    }
    // R8
    Outcome O;
    O.acc = acc;
    O.vn = vn;
    O.l_new = l_new;
    const int32_t len_fx = (int32_t)(V.len_c << 10);
    if (xn < len_fx) {
        O.kind = KIND_STAY;
        O.nx = (uint32_t)xn;
    } else if (V.last) {
        O.kind = KIND_DONE;  // G18
        O.nx = 0u;
    } else {
        O.kind = KIND_CAND;
        O.nx = (uint32_t)(xn - len_fx);
    }
    return O;
}

// R9 for one vehicle, in place: next state, time-(t+1) mark and payload for stayers, time-(t-1) mark toggled
// off, claim + cross-list entry for edge-end candidates, cross-list entry + freed slot for arrivals.
__device__ __forceinline__ void write_out(const DevP &P, uint32_t t, UpdateSmem &sm, uint32_t seg_base, uint32_t slot, const Veh &V,
                                          const Outcome &O)
{
    const int nxt = (int)((t & 1u) ^ 1u);
    const StBuf &S = P.st[sbuf_of(t)];
    u64 *Bn = P.bits[nxt];
    const uint32_t cur_abs = V.row0 + V.c;
    const uint32_t at = seg_base + slot;
    MANTA_ASSERT(at < g_check.slots && V.id < g_check.n_trips && (V.prev == CELL_NONE || V.prev < g_check.n_cells), CHK_SLOT);
    const bool changed = O.l_new != V.l;
    const uint32_t row_n = changed ? (O.l_new > V.l ? V.row0 + V.pitch : V.row0 - V.pitch) : V.row0;
    const uint32_t geom_n = (V.geom & GEOM_STATIC_MASK) | (O.l_new << 28) | (V.tag << 31);
    if (O.kind == KIND_STAY) {
        const uint32_t cell = row_n + (O.nx >> 10);
        if (V.prev != CELL_NONE)
            mark_move(Bn, V.prev, cell);
        else
            mark_toggle(Bn, cell);
        pay_store(P, P.pay[nxt], cell, O.nx & 1023u, __float_as_uint(O.vn));
        S.S0[at] = make_uint4(O.nx | (V.wait << WAIT_SHIFT), __float_as_uint(O.vn), cur_abs, V.id);
    } else {
        if (V.prev != CELL_NONE) mark_toggle(Bn, V.prev);
        const bool stop = GEOM_PRIO(V.geom) && (V.hopz >> 31) != 0u;   // the head node is a STOP node (R8s)
        if (O.kind == KIND_DONE) {
            P.arrive_step[V.id] = t + 1u;
            atomicAdd(&sm.ev[EV_DONE], 1ull);
            atomicAdd(&sm.ev[EV_TRAVEL], (u64)(t + 1u - P.admit_step[V.id]));
            S.S0[at] = make_uint4(0u, 0u, cur_abs, ID_GHOST);   // the ghost clears the time-t mark in the next step
        } else if (stop && V.wait < P.W_stop) {
            // R8s: it stands at the stop line (the place claim losers hold at, G15) one more step;
            // no claim, nothing for the second phase
            const uint32_t x_line = (V.len_c << 10) - 1u;
            const uint32_t cell = V.row0 + V.len_c - 1u;       // (no lane change this close to the edge end)
            mark_toggle(Bn, cell);
            pay_store(P, P.pay[nxt], cell, x_line & 1023u, 0u);
            S.S0[at] = make_uint4(x_line | ((V.wait + 1u) << WAIT_SHIFT), 0u, cur_abs, V.id);
        } else {
            // smallest key wins; the key carries ~t in the high word so claim words never need a reset
            const uint32_t target = (V.claim & ~7u) + min(O.l_new, V.claim & 7u);   // lane entry (e+, l+)
            const uint32_t word = GEOM_PRIO(V.geom) ? P.n_edges * 8u + ((V.hopz >> 4) & NODE_MASK) : target;
            uint32_t key_lo = V.id;
            if (stop) {
                // R8s: the n x m (inbound, outbound) combinations of the node take turns; at step t
                // combination c has rank (c - t) mod nm, the smallest rank enters, equal ranks by smallest id
                const uint4 es = P.edge_stop[P.route[V.cursor].z];   // {nm, in_idx * m, first out-edge of the node, 0}
                const uint32_t c = es.y + ((V.claim >> 3) - es.z);
                const uint32_t rank = (c + es.x - t % es.x) % es.x;
                key_lo = (rank << 24) | V.id;
            }
            P.cand_info[V.id] = make_uint2(target, O.nx >> 10);
            const u64 key = ((u64)(0xFFFFFFFFu - t) << 32) | (u64)key_lo;
            MANTA_ASSERT(word < g_check.n_claims && sm.xn < P.seg_cap, CHK_CLAIM);
            atomicMin(&P.claim[word], key);
            P.xlist[seg_base + atomicAdd(&sm.xn, 1u)] = make_uint4(slot | (V.wait << WAIT_SHIFT), word, V.cursor, key_lo);
            S.S0[at] = make_uint4(O.nx, __float_as_uint(O.vn), cur_abs, V.id);   // tentative winner state (counter 0); the second phase decides
        }
    }
    if (geom_n != V.geom) S.S1[at] = make_uint4(row_n, geom_n, V.cursor, __float_as_uint(V.v0));
    if (changed) {   // executed lane change: the look-ahead continues in other rows now
        atomicAdd(&sm.ev[EV_LC], 1ull);
        const Hops hp = build_hops(P, V.cursor, V.geom, O.l_new);
        S.S2[at] = hp.s2;
        S.S3[at] = hp.s3;
    }
    if (S.acc) S.acc[at] = O.acc;
}

// R5: lead (first occupied cell >= c, within the edge) and lag (last occupied cell < c) in the target lane, then
// the rest of the update.
template <bool W256>
__device__ __forceinline__ Outcome lane_change_and_finish(const DevP &P, uint32_t t, const u64 *B, const uint2 *pay, const Veh &V)
{
    const uint32_t rowt = V.lt > V.l ? V.row0 + V.pitch : V.row0 - V.pitch;
    uint32_t ja = 0u, jb = 0u;
    const uint32_t b0 = V.c > P.lookback ? V.c - P.lookback : 0u;
    bool has_a, has_b;
    if (W256) {
        lead_lag_w(B, rowt, V.c, min(V.len_c, V.c + P.H), b0, has_a, ja, has_b, jb);
    } else {
        has_a = scan_fwd<W256>(B, rowt, V.c, min(V.len_c, V.c + P.H), ja);
        has_b = V.c > b0 && scan_bwd<W256>(B, rowt, b0, V.c, jb);
    }
    int32_t x_a = 0, x_b = 0;
    float v_a = 0.0f, v_b = 0.0f;
    uint2 pa = make_uint2(0u, 0u), pb = pa;
    MANTA_ASSERT((!has_a || ((rowt + ja) >> P.pay_shift) < g_check.pay_entries) && (!has_b || ((rowt + jb) >> P.pay_shift) < g_check.pay_entries), CHK_PAY);
    if (has_a) pa = pay[(rowt + ja) >> P.pay_shift];
    if (has_b) pb = pay[(rowt + jb) >> P.pay_shift];
    if (has_a) {
        x_a = (int32_t)((ja << 10) | pa.x);
        v_a = __uint_as_float(pa.y);
    }
    if (has_b) {
        x_b = (int32_t)((jb << 10) | pb.x);
        v_b = __uint_as_float(pb.y);
    }
    return post_lc(P, t, V, has_a, x_a, v_a, has_b, x_b, v_b);
}

// ------------------------------------------------------------------------------------------------ A: R1
// Departure admission (G17, G25) for step t.  Thread k owns the FIFO of one origin edge; trips in it
// are in vehicle-id (= departure) order, so the head is the smallest waiting id on that edge.  New vehicles go
// into state buffer sb.
// FUSED = false: runs between two grid barriers; atlas_t is complete.
// FUSED = true : runs in the same phase as second_phase(t - 1), whose winners may be writing their marks into the
// entry windows tested here.  The only marks of that phase that can fall into a window [0, L_c] are those of claim
// winners (losers hold in the last cell of a row, which lies beyond the window: the host fuses only if every edge
// has at least L_c + 2 cells), at most one per lane entry, and which vehicle wins and where it lands can be read
// from the claim word and cand_info: the winner's bit is ORed into the word, whether its toggle has landed or not.
template <bool FUSED>
__device__ __forceinline__ void admit_phase(const DevP &P, uint32_t t, int sb)
{
    // queue k is served by block k % gridDim, counted down from the block's LAST thread: the queues are spread over
    // all blocks, away from the low threads that carry the cross-list entries of the same phase
    const uint32_t gsize = gridDim.x * blockDim.x;
    const uint32_t gtid = blockIdx.x + gridDim.x * (blockDim.x - 1u - threadIdx.x);
    const int cur = (int)(t & 1u);
    const StBuf &S = P.st[sb];
    u64 *B = P.bits[cur];
    uint2 *pay = P.pay[cur];
    const u64 window = bits_below(P.L_c + 1u);
    for (uint32_t k = gtid; k < P.n_queues; k += gsize) {
        const uint4 qs = P.q_state[k];                 // {depart_step, index in q_ent, vehicle id, route cursor} of the head
        if (qs.x > t) continue;                        // idle (or exhausted: NONE) queue
        const uint4 er = P.q_row[k];
        const uint32_t q_end = P.q_end[k];
        const uint4 nx = P.q_ent[qs.y + 1u];           // the entry that becomes the head (padding entry after the last)
        const uint32_t id = qs.z, cursor = qs.w;
        const uint4 rr = P.route[cursor];
        const HopRecs hr = load_hop_recs(P, cursor);   // all gathers of this admission are requested here, together
        const uint32_t head_node = P.edge_tab[er.w].z;
        const uint32_t len = GEOM_LEN(er.y), lanes = GEOM_LANES(er.y), pitch = pitch_of(len);
        uint32_t seg = P.bucket_seg[er.x >> MANTA_BUCKET_SHIFT];   // the segment whose vehicles are in this stretch of the atlas
        u64 w[MANTA_MAX_LANES_DEV];
#pragma unroll
        for (uint32_t l = 0; l < MANTA_MAX_LANES_DEV; l++) w[l] = l < lanes ? B[(er.x + l * pitch) >> 6] : ~0ull;
        if (FUSED) {
            const uint32_t stamp = 0xFFFFFFFFu - (t - 1u);   // claims of the step whose second phase is running
            u64 key[MANTA_MAX_LANES_DEV];
#pragma unroll
            for (uint32_t l = 0; l < MANTA_MAX_LANES_DEV; l++) {
                key[l] = ~0ull;
                if (er.z != CELL_NONE) {               // PRIORITY tail node: one claim word for all entries
                    if (l == 0u) key[l] = P.claim[er.z];
                } else if (l < lanes) {
                    key[l] = P.claim[er.w * 8u + l];
                }
            }
#pragma unroll
            for (uint32_t l = 0; l < MANTA_MAX_LANES_DEV; l++)
                if ((uint32_t)(key[l] >> 32) == stamp && (uint32_t)key[l] != CELL_NONE) {   // (never-claimed words are all ones)
                    const uint2 ci = P.cand_info[(uint32_t)key[l] & P.id_mask];   // {lane entry it heads for, landing cell}
#pragma unroll
                    for (uint32_t m = 0; m < MANTA_MAX_LANES_DEV; m++)
                        if (ci.x == er.w * 8u + m) w[m] |= 1ull << (ci.y & 63u);
                }
        }
        uint32_t l_sel = 0xFFFFFFFFu;
#pragma unroll
        for (uint32_t l = 0; l < MANTA_MAX_LANES_DEV; l++)
            if (l_sel == 0xFFFFFFFFu && !(w[l] & window)) l_sel = l;   // first lane whose window [0, L_c] is free
        if (l_sel == 0xFFFFFFFFu) continue;
        const uint32_t geom = (rr.y & GEOM_STATIC_MASK) | (l_sel << 28);
        const Hops hp = make_hops(hr, geom, l_sel, head_node);
        uint32_t slot;
        for (;;) {
            slot = atomicAdd(&P.seg_cnt[seg], 1u);
            if (slot < P.seg_cap) break;
            atomicSub(&P.seg_cnt[seg], 1u);            // full: the total capacity covers every trip, so another has room
            seg = seg + 1u == P.n_seg ? 0u : seg + 1u;
        }
        const uint32_t row = er.x + l_sel * pitch;
        const size_t at = (size_t)seg * P.seg_cap + slot;
        MANTA_ASSERT(at < g_check.slots && id < g_check.n_trips && cursor < g_check.route_total && rr.z < g_check.n_edges, CHK_SLOT);
        S.S0[at] = make_uint4(0u, 0u, CELL_NONE, id);
        S.S1[at] = make_uint4(row, geom, cursor, desired_speed_bits(P, id, 0u, rr.w));
        S.S2[at] = hp.s2;
        S.S3[at] = hp.s3;
        if (S.acc) S.acc[at] = 0.0f;
        mark_toggle(B, row);                           // cell 0, frac10 = 0, v = 0: visible to this step's update
        pay_store(P, pay, row, 0u, 0u);
        P.admit_step[id] = t;
        atomicAdd(&P.edge_entries[rr.z], 1u);
        P.q_state[k] = make_uint4(qs.y + 1u < q_end ? nx.y : CELL_NONE, qs.y + 1u, nx.x, nx.z);
    }
}

// ------------------------------------------------------------------------------------------------ A8: re-sort
// Spatial re-sort of the vehicle slots (before step t, t a multiple of MANTA_SORT_EVERY): counting sort of all
// live slots of buffer `from` by atlas bucket into buffer `from ^ 1`, dealt out in equal shares of per_seg slots.
// Five grid-wide stages: zero the histogram | count (each slot gets its rank inside its bucket) | per-block sums
// of the histogram | exclusive scan (offsets, and the bucket -> segment map admission uses) | scatter.
// Results do not depend on slot order (every rule reads time-t state only), so any order inside a bucket will do.
__device__ __forceinline__ uint32_t sort_key(const uint4 &s0v, uint32_t row0)
{
    const uint32_t cell = s0v.w == ID_GHOST ? s0v.z : row0 + ((s0v.x & X_MASK) >> 10);   // a ghost sorts by the mark it has to clear
    return cell >> MANTA_BUCKET_SHIFT;
}
__device__ __forceinline__ void sort_zero(const DevP &P)
{
    for (uint32_t b = blockIdx.x * blockDim.x + threadIdx.x; b <= P.n_buckets; b += gridDim.x * blockDim.x) P.sort_hist[b] = 0u;
}
__device__ __forceinline__ void sort_count(const DevP &P, int from)
{
    const StBuf &S = P.st[from];
    for (uint32_t seg = blockIdx.x; seg < P.n_seg; seg += gridDim.x) {
        const uint32_t n = P.seg_cnt[seg];
        const size_t seg_base = (size_t)seg * P.seg_cap;
        for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
            const uint4 s0v = S.S0[seg_base + i];
            uint32_t r = CELL_NONE;
            if (s0v.w != CELL_NONE) r = atomicAdd(&P.sort_hist[sort_key(s0v, S.S1[seg_base + i].x)], 1u);
            P.sort_rank[seg_base + i] = r;
        }
    }
}
// slice of the histogram that block j scans
__device__ __forceinline__ void sort_slice(const DevP &P, uint32_t j, uint32_t &b0, uint32_t &b1)
{
    const uint32_t per = (P.n_buckets + gridDim.x - 1u) / gridDim.x;
    b0 = min(j * per, P.n_buckets);
    b1 = min(b0 + per, P.n_buckets);
}
__device__ __forceinline__ uint32_t block_sum(uint32_t v, uint32_t *wsum)   // all threads; result valid in every thread
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, d);
    __syncthreads();
    if ((threadIdx.x & 31u) == 0u) wsum[threadIdx.x >> 5] = v;
    __syncthreads();
    uint32_t tot = 0u;
    for (uint32_t w = 0; w < (blockDim.x >> 5); w++) tot += wsum[w];
    return tot;
}
__device__ __forceinline__ void sort_partial(const DevP &P, UpdateSmem &sm)
{
    uint32_t b0, b1;
    sort_slice(P, blockIdx.x, b0, b1);
    uint32_t v = 0u;
    for (uint32_t b = b0 + threadIdx.x; b < b1; b += blockDim.x) v += P.sort_hist[b];
    const uint32_t tot = block_sum(v, sm.wsum);
    if (threadIdx.x == 0u) P.sort_part[blockIdx.x] = tot;
}
__device__ __forceinline__ void sort_scan(const DevP &P, UpdateSmem &sm, uint32_t &n_live, uint32_t &per_seg)
{
    // offset of this block's slice and the live total, from the per-block sums
    uint32_t before = 0u, all = 0u;
    for (uint32_t k = threadIdx.x; k < gridDim.x; k += blockDim.x) {
        const uint32_t c = P.sort_part[k];
        all += c;
        before += k < blockIdx.x ? c : 0u;
    }
    all = block_sum(all, sm.wsum);
    before = block_sum(before, sm.wsum);
    n_live = all;
    per_seg = max(1u, (all + P.n_seg - 1u) / P.n_seg);
    uint32_t b0, b1;
    sort_slice(P, blockIdx.x, b0, b1);
    const uint32_t lane_id = threadIdx.x & 31u, warp_id = threadIdx.x >> 5;
    uint32_t run = before;
    for (uint32_t base = b0; base < b1; base += blockDim.x) {
        const uint32_t b = base + threadIdx.x;
        const uint32_t c = b < b1 ? P.sort_hist[b] : 0u;
        uint32_t inc = c;   // inclusive scan inside the warp
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, inc, d);
            if (lane_id >= (uint32_t)d) inc += o;
        }
        __syncthreads();
        if (lane_id == 31u) sm.wsum[warp_id] = inc;
        __syncthreads();
        uint32_t wpre = 0u, tot = 0u;
        for (uint32_t w = 0; w < (blockDim.x >> 5); w++) {
            const uint32_t x = sm.wsum[w];
            wpre += w < warp_id ? x : 0u;
            tot += x;
        }
        if (b < b1) {
            const uint32_t off = run + wpre + inc - c;
            P.sort_hist[b] = off;
            P.bucket_seg[b] = (off >> 5) % P.n_seg;   // segment of the chunk the bucket's first vehicle goes to
        }
        run += tot;
    }
}
__device__ __forceinline__ void sort_scatter(const DevP &P, int from, uint32_t n_live, uint32_t per_seg)
{
    const StBuf &S = P.st[from];
    const StBuf &D = P.st[from ^ 1];
    for (uint32_t seg = blockIdx.x; seg < P.n_seg; seg += gridDim.x) {
        const uint32_t n = P.seg_cnt[seg];
        const size_t seg_base = (size_t)seg * P.seg_cap;
        for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
            const uint32_t r = P.sort_rank[seg_base + i];
            if (r == CELL_NONE) continue;
            const uint4 a0 = S.S0[seg_base + i], a1 = S.S1[seg_base + i], a2 = S.S2[seg_base + i], a3 = S.S3[seg_base + i];
            const uint32_t g = P.sort_hist[sort_key(a0, a1.x)] + r;
            // chunks of 32 consecutive vehicles are dealt round-robin: chunk j goes to segment j % n_seg
            const uint32_t chunk = g >> 5, sd = chunk % P.n_seg;
            const size_t at = (size_t)sd * P.seg_cap + ((chunk / P.n_seg) << 5) + (g & 31u);
            MANTA_ASSERT(at < g_check.slots && ((chunk / P.n_seg) << 5) + (g & 31u) < P.seg_cap, CHK_SLOT);
            D.S0[at] = a0;
            D.S1[at] = a1;
            D.S2[at] = a2;
            D.S3[at] = a3;
            if (S.acc) D.acc[at] = S.acc[seg_base + i];
        }
    }
    __syncthreads();   // this block has read the old counts of all its segments
    const uint32_t n_chunks = (n_live + 31u) >> 5;
    for (uint32_t seg = blockIdx.x; seg < P.n_seg; seg += gridDim.x)
        if (threadIdx.x == 0u) {
            uint32_t cnt = 0u;
            if (seg < n_chunks) {
                const uint32_t mine = (n_chunks - 1u - seg) / P.n_seg + 1u;          // chunks seg, seg + n_seg, ...
                const bool has_last = (n_chunks - 1u) % P.n_seg == seg;              // only the last chunk can be partial
                cnt = has_last ? ((mine - 1u) << 5) + (n_live - ((n_chunks - 1u) << 5)) : mine << 5;
            }
            P.seg_cnt[seg] = cnt;
        }
}
__device__ __forceinline__ bool sort_due(uint32_t t) { return t != 0u && t % MANTA_SORT_EVERY == 0u; }

// ------------------------------------------------------------------------------------------------ U: R2-R9
// A vehicle further than Z_out cells from its edge end cannot reach it in this step (R0: Z_out > vcap dt), so it
// can be neither an edge-end candidate nor an arrival, whatever its leader.  (R4 allows lane changes only there.)
__device__ __forceinline__ bool cannot_cross(const DevP &P, const Veh &V) { return V.c + P.Z_out < V.len_c; }
// A vehicle may be handed to the deferred stage -- which runs in the same phase as the claim resolution of this step and
// the (fused) admission of the next -- only if nothing it does can matter there: it cannot reach its edge end (no
// claim), and its time-(t+1) mark cannot fall into an entry window [0, L_c] that admission is testing (vehicles do
// not move backwards, so c > L_c is enough; lane changes start at c >= Z_in > L_c anyway).
__device__ __forceinline__ bool may_defer(const DevP &P, const Veh &V) { return cannot_cross(P, V) && V.c > P.L_c; }

// Look-ahead past the four cached hops (rare: a run of short edges): the cache the vehicle would have four route
// edges further on is rebuilt from the route store and searched the same way, until the budget of H cells is used
// up, the route ends or a leader is found.
__device__ __forceinline__ Hit leader_continue(const DevP &P, const u64 *B, const Veh &V, uint32_t s3z, uint32_t budget_left,
                                              uint32_t dist_next, uint32_t &n_cells)
{
    Hit h;
    uint32_t cursor = V.cursor, lane = (s3z >> 1) & 7u;
    HopRecs R = load_hop_recs(P, cursor + 4u);
    for (int rounds = 0; rounds < 16; rounds++) {
        cursor += 4u;
        const HopRecs Rn = load_hop_recs(P, cursor + 4u);   // the next round's records travel while this round is searched (the store is padded; a route that ended is never followed)
        const Hops hp = make_hops(R, 0u, lane, 0u);
        R = Rn;
        const int r = leader_window(P, B, V.c, 0u, 0u, 0u, dist_next, budget_left, hp.s2, hp.s3, h, budget_left, dist_next);
        if (r == WIN_DONE) {
            n_cells += h.found ? h.dist - V.c : P.H - budget_left;
            return h;
        }
        if (r == WIN_NOFIT) break;
        lane = (hp.s3.z >> 1) & 7u;
    }
    return walk_rows(P, B, V, n_cells);
}

// Deferred-list entry kinds: 0 / 1 = adjacent-lane evaluation (own-lane leader not found / found, carried in the
// entry); 2 = look-ahead to be continued past the cached hops (budget_left, dist_next carried); 3 = walk_rows.
template <bool W256>
__device__ __forceinline__ void finish_deferred(const DevP &P, uint32_t t, UpdateSmem &sm, uint32_t seg_base, const uint4 &e, const uint4 &s0v, const uint4 &s1v,
                                                uint32_t &n_cells)
{
    const int cur = (int)(t & 1u);
    const StBuf &S = P.st[sbuf_of(t)];
    const u64 *B = P.bits[cur];
    const uint2 *pay = P.pay[cur];
    const uint32_t slot = e.x & 0x3FFFFFFFu, kind = e.x >> 30;
    Veh V;
    veh_load(V, s0v, s1v);
    if (kind < 2u) {   // a lane change rebuilds the look-ahead cache from these route records: on their way now
        prefetch_line(P.route + V.cursor + 1u);
        prefetch_line(P.route + V.cursor + 4u);
    }
    V.claim = 0u;   // a deferred vehicle cannot reach its edge end
    V.hopz = 0u;
    Lead ld;
    if (kind >= 2u) {
        const Hit h = kind == 2u ? leader_continue(P, B, V, e.w, e.y, e.z, n_cells) : walk_rows(P, B, V, n_cells);
        ld = lead_from_hit<W256>(pay, P.pay_shift, h);
    } else {
        ld.found = kind != 0u;
        ld.lead_abs = (int32_t)e.y;
        ld.v_lead = __uint_as_float(e.z);
    }
    pre_lc(P, t, V, ld);
    Outcome O;
    if (V.need_lc) {
        atomicAdd(&sm.ev[EV_EVAL], 1ull);
        O = lane_change_and_finish<W256>(P, t, B, pay, V);
    } else {
        O = post_lc(P, t, V, false, 0, 0.0f, false, 0, 0.0f);
    }
    write_out(P, t, sm, seg_base, slot, V, O);
}

// R9s: per-edge speed statistics (inputs of Eq. 5).  In a sampling step every live vehicle adds
// rint(v * 256) of its time-t speed to the accumulators of (time slice, its edge).  The edge id is not part of the
// vehicle state: one gather from the route store, in sampling steps only.
__device__ __forceinline__ void sample_speed(const DevP &P, uint32_t t, const Veh &V)
{
    const uint32_t slice = t / P.stat_slice;
    if (slice >= P.stat_n_slices) return;
    const uint32_t e = P.route[V.cursor].z;
    MANTA_ASSERT(e < g_check.n_edges && V.cursor < g_check.route_total, CHK_EDGE);
    const size_t k = (size_t)slice * P.n_edges + e;
    atomicAdd(&P.stat_sum[k], (u64)__float2int_rn(V.v * 256.0f));
    atomicAdd(&P.stat_cnt[k], 1u);
}
__device__ __forceinline__ bool sampling_step(const DevP &P, uint32_t t) { return P.stat_period != 0u && t % P.stat_period == 0u; }

// Puts the vehicle of slot i on the deferred list of its block.  Its time-(t-1) mark is toggled off HERE, in the pass:
// that mark may lie in an entry window the fused admission reads while the deferred stage runs (the time-(t+1) mark
// cannot: may_defer), so the deferred stage must only ever set marks beyond the windows.
__device__ __forceinline__ void defer_entry(const DevP &P, uint32_t t, UpdateSmem &sm, const StBuf &S, uint32_t seg_base, uint32_t i,
                                            uint32_t dq_cap, uint4 s0v, const uint4 &s1v, const uint4 &e)
{
    if (s0v.z != CELL_NONE) {
        mark_toggle(P.bits[(t & 1u) ^ 1u], s0v.z);
        s0v.z = CELL_NONE;
    }
    const uint32_t k = atomicAdd(&sm.qn, 1u);
    MANTA_ASSERT(k < P.seg_cap, CHK_LIST);
#if MANTA_DQ
    if (k < dq_cap) {
        sm.dq[k][0] = s0v;
        sm.dq[k][1] = s1v;
        sm.dq[k][2] = e;
    } else
#endif
    {
        P.dlist[seg_base + k] = e;
        reinterpret_cast<uint32_t *>(&S.S0[seg_base + i])[2] = CELL_NONE;   // the stage re-reads S0 from the state array
    }
}

#if MANTA_TWO_STAGE
// ---- the pass in two stages per chunk, software-pipelined per warp through shared memory (H <= 256 only) --------
// Stage A of chunk k + 1 (state records, occupancy words, search; the leader's payload entry is requested with
// cp.async straight into the thread's record) runs BEFORE stage B of chunk k (payload -> IDM -> integration ->
// writes), so the payload gather of a chunk has a whole stage A to land and only the occupancy-word gather is
// waited for.  A thread's record lives in its own shared-memory words (two buffers): no cross-thread traffic.
#define REC(buf, f) rec[((buf) * 3 + (f)) * MANTA_NT + threadIdx.x]   // per thread and buffer: S0 | S1 | {dist + flags, claim word, payload}
__device__ __forceinline__ void cp_async8(void *smem_dst, const void *gsrc)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void stage_search(const DevP &P, uint32_t t, UpdateSmem &sm, uint4 *rec, int buf, const StBuf &S, const u64 *B,
                                             const uint2 *pay, uint32_t seg_base, uint32_t n, uint32_t i, uint32_t dq_cap,
                                             uint32_t &n_cells, uint32_t &n_upd)
{
    uint4 s0v = make_uint4(0u, 0u, 0u, CELL_NONE), s1v = s0v, s2v = s0v, s3v = s0v;
    if (i < n) {
        s0v = S.S0[seg_base + i];
        s1v = S.S1[seg_base + i];
        s2v = S.S2[seg_base + i];
        s3v = S.S3[seg_base + i];
    }
    if (s0v.w == ID_GHOST) {   // the ghost of last step's arrival clears that vehicle's last mark
        mark_toggle(P.bits[(t & 1u) ^ 1u], s0v.z);
        S.S0[seg_base + i] = make_uint4(0u, 0u, CELL_NONE, CELL_NONE);
    }
    const bool live = s0v.w < ID_GHOST;
    Veh V;
    veh_load(V, s0v, s1v);
    Hit h;
    h.found = false;
    h.cell = 0u;
    h.dist = 0u;
    uint32_t budget_left = 0u, dist_next = 0u;
    int r = WIN_DONE;
    if (live) {
        n_upd += 1u;
        if (sampling_step(P, t)) sample_speed(P, t, V);
        const uint32_t start = V.c + 1u;
        const uint32_t own = start < V.len_c ? min(V.len_c - start, P.H) : 0u;
        r = leader_window(P, B, V.c, V.row0, start, own, V.len_c, P.H, s2v, s3v, h, budget_left, dist_next);
        if (r == WIN_DONE) {
            n_cells += h.found ? h.dist - V.c : P.H - budget_left;
        } else if (!may_defer(P, V)) {   // rare: near an edge end and the window does not fit
            h = r == WIN_MORE ? leader_continue(P, B, V, s3v.z, budget_left, dist_next, n_cells) : walk_rows(P, B, V, n_cells);
            r = WIN_DONE;
        }
    }
    const bool searched = live && r == WIN_DONE;
    if (live && !searched) {   // look-ahead to be continued (2) or walked (3) by the deferred stage
        const uint32_t kind = r == WIN_MORE ? 2u : 3u;
        const uint4 e = make_uint4(i | (kind << 30), budget_left, dist_next, s3v.z);
        // the deferred stage continues with RouteRecs cursor + 5 .. cursor + 8 (kind 2) or walks on from cursor + 1
        // (kind 3): out of the route store into L2 now
        prefetch_line(P.route + V.cursor + (kind == 2u ? 5u : 1u));
        prefetch_line(P.route + V.cursor + (kind == 2u ? 8u : 4u));
        defer_entry(P, t, sm, S, seg_base, i, dq_cap, s0v, s1v, e);
    }
    REC(buf, 0) = s0v;
    REC(buf, 1) = s1v;
    REC(buf, 2).x = h.dist | (searched ? 1u << 30 : 0u) | ((searched && h.found) ? 1u << 31 : 0u);
    REC(buf, 2).y = s3v.w;   // claim word of R8
    if (searched && h.found) cp_async8(&REC(buf, 2).z, &pay[h.cell >> P.pay_shift]);
    cp_async_commit();
}

__device__ __forceinline__ void stage_finish(const DevP &P, uint32_t t, UpdateSmem &sm, uint4 *rec, int buf, uint32_t seg_base, uint32_t i,
                                             uint32_t dq_cap)
{
    const uint4 m = REC(buf, 2);
    const bool searched = (m.x >> 30) & 1u;
    const uint4 s0v = REC(buf, 0), s1v = REC(buf, 1);
    Veh V;
    veh_load(V, s0v, s1v);
    V.hopz = 0u;
    V.claim = m.y;
    Lead ld;
    ld.found = (m.x >> 31) != 0u;
    ld.lead_abs = 0;
    ld.v_lead = 0.0f;
    V.need_lc = false;
    if (searched) {
        if (ld.found) {
            ld.lead_abs = (int32_t)(((m.x & 0x3FFFFFFFu) << 10) | m.z);
            ld.v_lead = __uint_as_float(m.w);
        }
        pre_lc(P, t, V, ld);
    }
    __syncwarp();
    if (searched && !V.need_lc) {
        const Outcome O = post_lc(P, t, V, false, 0, 0.0f, false, 0, 0.0f);
        if (O.kind == KIND_CAND && GEOM_PRIO(V.geom))   // behind a PRIORITY node the claim word is the node: its id is in S3.z
            V.hopz = P.st[sbuf_of(t)].S3[seg_base + i].z;
        write_out(P, t, sm, seg_base, i, V, O);
    } else if (searched) {   // must look at the adjacent lane (R5): deferred, kinds 0 / 1
        const uint4 e = make_uint4(i | ((ld.found ? 1u : 0u) << 30), (uint32_t)ld.lead_abs, __float_as_uint(ld.v_lead), 0u);
        defer_entry(P, t, sm, P.st[sbuf_of(t)], seg_base, i, dq_cap, s0v, s1v, e);
    }
    __syncwarp();
}

// the chunk loop of one segment; all warps of the block
__device__ __forceinline__ void pass_two_stage(const DevP &P, uint32_t t, UpdateSmem &sm, uint4 *rec, const StBuf &S, const u64 *B,
                                               const uint2 *pay, uint32_t seg_base, uint32_t n, uint32_t dq_cap, uint32_t &n_cells,
                                               uint32_t &n_upd)
{
    const uint32_t lane_id = threadIdx.x & 31u;
    uint32_t base = threadIdx.x & ~31u;
    if (base >= n) return;
    int buf = 0;
    stage_search(P, t, sm, rec, buf, S, B, pay, seg_base, n, base + lane_id, dq_cap, n_cells, n_upd);
    for (;;) {
        uint32_t next_base = 0u;
        if (lane_id == 0u) next_base = atomicAdd(&sm.next, 32u);
        next_base = __shfl_sync(0xFFFFFFFFu, next_base, 0);
        const bool more = next_base < n;
        if (more) {
            stage_search(P, t, sm, rec, buf ^ 1, S, B, pay, seg_base, n, next_base + lane_id, dq_cap, n_cells, n_upd);
            cp_async_wait<1>();   // everything but the group just committed: this chunk's payload entries are in
        } else {
            cp_async_wait<0>();
        }
        __syncwarp();
        stage_finish(P, t, sm, rec, buf, seg_base, base + lane_id, dq_cap);
        if (!more) break;
        base = next_base;
        buf ^= 1;
    }
}
#undef REC
#endif

// Must be called by ALL threads of the block (contains __syncthreads).  Warps take chunks of 32 slots from a
// shared counter, so a warp that met slow vehicles simply takes fewer chunks.
// how many deferred entries of a block stay in shared memory (with their S0 / S1 records); the rest go through P.dlist.
// Kernel-per-phase stepping keeps none: there the deferred stage runs in the next launch.
__device__ __forceinline__ uint32_t dq_capacity(const DevP &P, bool persistent)
{
    if (!MANTA_DQ || !persistent) return 0u;
    return (P.flags & MANTA_FLAG_TINY_QUEUES) ? 2u : (uint32_t)MANTA_DQ;
}

// The update pass over the block's segment.  Vehicles that must look at the adjacent lane (or continue their
// look-ahead past the cached hops) are only QUEUED here (deferred list); they are finished by second_phase, after
// the grid barrier, next to the claim resolution -- two dependent chains that used to run one after the other.
template <bool W256>
__device__ __forceinline__ void update_phase(const DevP &P, uint32_t t, UpdateSmem &sm, uint32_t &n_cells, uint32_t &n_upd, uint4 *rec, bool persistent)
{
    const int cur = (int)(t & 1u), nxt = cur ^ 1;
    const StBuf &S = P.st[sbuf_of(t)];
    const u64 *B = P.bits[cur];
    const uint2 *pay = P.pay[cur];
    const uint32_t lane_id = threadIdx.x & 31u;
    const uint32_t dq_cap = dq_capacity(P, persistent);
    for (uint32_t seg = blockIdx.x; seg < P.n_seg; seg += gridDim.x) {
        const uint32_t n = P.seg_cnt[seg];
        const uint32_t seg_base = seg * P.seg_cap;
        if (threadIdx.x == 0u) {
            sm.xn = 0u;
            sm.qn = 0u;
            sm.next = blockDim.x;
        }
        DBG_STAMP(1);
        __syncthreads();
#if MANTA_TWO_STAGE
        if (W256) {
            pass_two_stage(P, t, sm, rec, S, B, pay, seg_base, n, dq_cap, n_cells, n_upd);
        } else
#endif
        for (uint32_t base = threadIdx.x & ~31u; base < n;) {
            const uint32_t i = base + lane_id;
            uint4 s0v = make_uint4(0u, 0u, 0u, CELL_NONE), s1v = s0v, s2v = s0v, s3v = s0v;
            if (i < n) {
                s0v = S.S0[seg_base + i];
                s1v = S.S1[seg_base + i];
                s2v = S.S2[seg_base + i];
                s3v = S.S3[seg_base + i];
            }
            // the next chunk of this warp (requested now, needed after this one)
            uint32_t next_base = 0u;
            if (lane_id == 0u) next_base = atomicAdd(&sm.next, 32u);
#if MANTA_PF
            next_base = __shfl_sync(0xFFFFFFFFu, next_base, 0);
            if (next_base + lane_id < n) {   // its state records, requested a whole chunk ahead
                const uint32_t at = seg_base + next_base + lane_id;
                prefetch_line(&S.S0[at]);
                prefetch_line(&S.S1[at]);
                prefetch_line(&S.S2[at]);
                prefetch_line(&S.S3[at]);
            }
#endif
            if (s0v.w == ID_GHOST) {   // the ghost of last step's arrival clears that vehicle's last mark
                mark_toggle(P.bits[nxt], s0v.z);
                S.S0[seg_base + i] = make_uint4(0u, 0u, CELL_NONE, CELL_NONE);
            }
            // The stages below are separated by __syncwarp() so that the warp runs each of them once, with all its
            // live lanes, whatever rare side paths single lanes took in the stage before.
            const bool live = s0v.w < ID_GHOST;
            Veh V;
            veh_load(V, s0v, s1v);
            V.claim = s3v.w;
            V.hopz = s3v.z;
            Hit h;
            h.found = false;
            h.cell = 0u;
            h.dist = 0u;
            uint32_t budget_left = 0u, dist_next = 0u;
            int r = WIN_DONE;
            // ---- stage 1: look-ahead (R2)
            if (live) {
                n_upd += 1u;
                if (sampling_step(P, t)) sample_speed(P, t, V);
                if (W256) {
                    const uint32_t start = V.c + 1u;
                    const uint32_t own = start < V.len_c ? min(V.len_c - start, P.H) : 0u;
                    r = leader_window(P, B, V.c, V.row0, start, own, V.len_c, P.H, s2v, s3v, h, budget_left, dist_next);
                    if (r == WIN_DONE) {
                        n_cells += h.found ? h.dist - V.c : P.H - budget_left;
                    } else if (!may_defer(P, V)) {   // rare: near an edge end and the window does not fit
                        h = r == WIN_MORE ? leader_continue(P, B, V, s3v.z, budget_left, dist_next, n_cells) : walk_rows(P, B, V, n_cells);
                        r = WIN_DONE;
                    }
                } else {
                    h = walk_rows(P, B, V, n_cells);
                }
            }
            __syncwarp();
            // ---- stage 2: leader payload, IDM, lane-change pre-tests (R3, R4)
            const bool searched = live && r == WIN_DONE;
            Lead ld;
            ld.found = false;
            ld.lead_abs = 0;
            ld.v_lead = 0.0f;
            V.need_lc = false;
            if (searched) {
                ld = lead_from_hit<W256>(pay, P.pay_shift, h);
                pre_lc(P, t, V, ld);
            }
            __syncwarp();
            // ---- stage 3: integrate, classify (R7, R8), next state and marks (R9); or defer
            if (searched && !V.need_lc) {
                const Outcome O = post_lc(P, t, V, false, 0, 0.0f, false, 0, 0.0f);
                write_out(P, t, sm, seg_base, i, V, O);
            } else if (live) {
                // deferred: must look at the adjacent lane (kinds 0 / 1, R5), or look-ahead to be continued (2) or walked (3)
                const uint32_t kind = searched ? (ld.found ? 1u : 0u) : (r == WIN_MORE ? 2u : 3u);
                const uint4 e = searched ? make_uint4(i | (kind << 30), (uint32_t)ld.lead_abs, __float_as_uint(ld.v_lead), 0u)
                                         : make_uint4(i | (kind << 30), budget_left, dist_next, s3v.z);
                defer_entry(P, t, sm, S, seg_base, i, dq_cap, s0v, s1v, e);
            }
            __syncwarp();
#if MANTA_PF
            base = next_base;
#else
            base = __shfl_sync(0xFFFFFFFFu, next_base, 0);
#endif
        }
        __syncthreads();   // the cross list and the deferred list of this segment are complete
        DBG_STAMP(2);
        if (threadIdx.x == 0u) {
            P.seg_xn[seg] = sm.xn;
            P.seg_qn[seg] = sm.qn;
        }
    }
}

// ------------------------------------------------------------------------------------------------ X: R8
// One thread per cross-list entry: resolve the claim; the winner moves to its next route edge and rebuilds its
// look-ahead cache, the loser holds at the stop line; both write their time-(t+1) mark and payload.
// Then the deferred list of the same segment (R5-R7 for the vehicles that look at the adjacent lane, R2 for look-aheads
// that run past the cached hops): they read atlas_t only, cannot be edge-end candidates and do not mark entry windows
// (may_defer), so nothing they do interacts with the claims or with the fused admission.  Cross-list entries go to
// the first MANTA_XT threads of the block, deferred entries to the others: the two chains run in different warps.
#ifndef MANTA_XT
#define MANTA_XT 128u   // threads of a block that take cross-list entries in the second phase; the others take deferred entries
#endif
// Replica batching (k_persistent_batch): replica r of n gets its own share of both thread ranges, so that the chains of
// the replicas run side by side as well.
template <bool W256>
__device__ __forceinline__ void second_phase(const DevP &P, uint32_t t, UpdateSmem &sm, uint32_t &n_cells, bool persistent,
                                             uint32_t r = 0u, uint32_t n = 1u)
{
    const int nxt = (int)((t & 1u) ^ 1u);
    const StBuf &S = P.st[sbuf_of(t)];
    u64 *Bn = P.bits[nxt];
    uint2 *payn = P.pay[nxt];
    const uint32_t dq_cap = dq_capacity(P, persistent);
    const bool split = blockDim.x > MANTA_XT;
    const uint32_t xw = split ? max(32u, (MANTA_XT / n) & ~31u) : blockDim.x, x_lo = split ? xw * r : 0u;
    const uint32_t dw = split ? max(32u, ((blockDim.x - MANTA_XT) / n) & ~31u) : blockDim.x, d_lo = split ? MANTA_XT + dw * r : 0u;
    for (uint32_t seg = blockIdx.x; seg < P.n_seg; seg += gridDim.x) {
        const uint32_t xn = persistent ? sm.xn : P.seg_xn[seg];
        const uint32_t qn = persistent ? sm.qn : P.seg_qn[seg];
        const uint32_t seg_base = seg * P.seg_cap;
        if (threadIdx.x >= d_lo && threadIdx.x < d_lo + dw)
            for (uint32_t k = threadIdx.x - d_lo; k < qn; k += dw) {
                uint4 e, a0, a1;   // one call site: finish_deferred is ~2 k instructions
#if MANTA_DQ
                if (k < dq_cap) {
                    e = sm.dq[k][2];
                    a0 = sm.dq[k][0];
                    a1 = sm.dq[k][1];
                } else
#endif
                {
                    e = P.dlist[seg_base + k];
                    const uint32_t slot = e.x & 0x3FFFFFFFu;
                    a0 = S.S0[seg_base + slot];
                    a1 = S.S1[seg_base + slot];
                }
                finish_deferred<W256>(P, t, sm, seg_base, e, a0, a1, n_cells);
            }
        if (threadIdx.x >= x_lo && threadIdx.x < x_lo + xw)
        for (uint32_t k = threadIdx.x - x_lo; k < xn; k += xw) {
            const uint4 xl = P.xlist[seg_base + k];     // {slot | stop-line counter << 28, claim word, cursor, low word of the claim key}
            const size_t at = (size_t)seg_base + (xl.x & X_MASK);
            MANTA_ASSERT(at < g_check.slots && xl.y < g_check.n_claims && (u64)xl.z + 1u < g_check.route_total, CHK_LIST);
            uint4 s0 = S.S0[at];
            const uint4 s1 = S.S1[at];
            const u64 won = P.claim[xl.y];
            const uint4 rn = P.route[xl.z + 1u];
            const HopRecs hr = load_hop_recs(P, xl.z + 1u);   // requested with the other gathers; used by the winner
            const u64 key = ((u64)(0xFFFFFFFFu - t) << 32) | (u64)xl.w;
            uint32_t cell;
            if (won == key) {             // winner crosses
                const uint32_t lplus = min(GEOM_LANE(s1.y), GEOM_LANES(rn.y) - 1u);
                const uint32_t geom = (rn.y & GEOM_STATIC_MASK) | (lplus << 28);
                const uint32_t row = rn.x + lplus * pitch_of(GEOM_LEN(rn.y));
                uint32_t node = 0u;
                if (!GEOM_LAST(geom) && GEOM_PRIO(geom)) node = P.edge_tab[rn.z].z;
                const Hops hp = make_hops(hr, geom, lplus, node);
                uint32_t v0b = rn.w;
                if (P.v0_sigma_rel > 0.0f) {   // R3s: this driver's desired speed on the edge it enters
                    const uint32_t id = xl.w & P.id_mask;
                    v0b = desired_speed_bits(P, id, xl.z + 1u - P.route_start[id], rn.w);
                }
                S.S1[at] = make_uint4(row, geom, xl.z + 1u, v0b);
                S.S2[at] = hp.s2;
                S.S3[at] = hp.s3;
                MANTA_ASSERT(rn.z < g_check.n_edges, CHK_EDGE);
                atomicAdd(&P.edge_entries[rn.z], 1u);
                cell = row + (s0.x >> 10);
            } else {                      // loser holds at the stop line (G15)
                const uint32_t x_line = (GEOM_LEN(s1.y) << 10) - 1u;
                s0.x = x_line | (xl.x & ~X_MASK);      // keeps its stop-line counter (R8s)
                s0.y = 0u;
                S.S0[at] = s0;
                cell = s1.x + (x_line >> 10);
            }
            mark_toggle(Bn, cell);
            pay_store(P, payn, cell, s0.x & 1023u, s0.y);
        }
    }
}

// per-thread and per-block counters of this kernel -> this block's record
__device__ __forceinline__ void flush_stats(const DevP &P, UpdateSmem &sm, uint32_t n_cells32, uint32_t n_upd32)
{
    u64 n_cells = n_cells32, n_upd = n_upd32;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        n_cells += __shfl_down_sync(0xFFFFFFFFu, n_cells, d);
        n_upd += __shfl_down_sync(0xFFFFFFFFu, n_upd, d);
    }
    BlockStats *b = &P.blk[blockIdx.x];
    if ((threadIdx.x & 31u) == 0u) {
        if (n_cells) atomicAdd(&b->cells_examined, n_cells);
        if (n_upd) atomicAdd(&b->n_updates, n_upd);
    }
    __syncthreads();
    if (threadIdx.x == 0u) {
        if (sm.ev[EV_LC]) atomicAdd(&b->lane_changes, sm.ev[EV_LC]);
        if (sm.ev[EV_EVAL]) atomicAdd(&b->lc_evals, sm.ev[EV_EVAL]);
        if (sm.ev[EV_DONE]) atomicAdd(&b->n_done, sm.ev[EV_DONE]);
        if (sm.ev[EV_TRAVEL]) atomicAdd(&b->sum_travel, sm.ev[EV_TRAVEL]);
    }
}

// ------------------------------------------------------------------------------------------------ kernels
extern __shared__ uint4 dyn_rec[];   // MANTA_REC_BYTES: per-thread records of the two-stage pass (k_update, k_persistent)
__global__ void __launch_bounds__(256) k_admit(const DevP P, uint32_t t)
{
    admit_phase<false>(P, t, sbuf_of(t));
}

template <bool W256>
__global__ void __launch_bounds__(MANTA_NT, MANTA_MINB) k_update(const DevP P, uint32_t t)
{
    __shared__ UpdateSmem sm;
    if (threadIdx.x < 4u) sm.ev[threadIdx.x] = 0ull;
    __syncthreads();
    uint32_t n_cells = 0u, n_upd = 0u;
    update_phase<W256>(P, t, sm, n_cells, n_upd, dyn_rec, false);
    flush_stats(P, sm, n_cells, n_upd);
}

// second phase of step t (claim resolution + deferred list); with admit_next, the admission of step t + 1 runs in the
// same launch (fused, see admit_phase)
template <bool W256>
__global__ void __launch_bounds__(MANTA_NT, MANTA_MINB) k_second(const DevP P, uint32_t t, int admit_next)
{
    __shared__ UpdateSmem sm;
    if (threadIdx.x < 4u) sm.ev[threadIdx.x] = 0ull;
    __syncthreads();
    uint32_t n_cells = 0u;
    if (admit_next) admit_phase<true>(P, t + 1u, sbuf_of(t));
    second_phase<W256>(P, t, sm, n_cells, false);
    flush_stats(P, sm, n_cells, 0u);
}

// the five stages of the re-sort as kernels (multi-kernel mode); n_live / per_seg travel through sort_part[n_seg..]
__global__ void __launch_bounds__(MANTA_NT) k_sort_zero(const DevP P) { sort_zero(P); }
__global__ void __launch_bounds__(MANTA_NT) k_sort_count(const DevP P, int from) { sort_count(P, from); }
__global__ void __launch_bounds__(MANTA_NT) k_sort_partial(const DevP P)
{
    __shared__ UpdateSmem sm;
    sort_partial(P, sm);
}
__global__ void __launch_bounds__(MANTA_NT) k_sort_scan(const DevP P)
{
    __shared__ UpdateSmem sm;
    uint32_t n_live, per_seg;
    sort_scan(P, sm, n_live, per_seg);
}
__global__ void __launch_bounds__(MANTA_NT) k_sort_scatter(const DevP P, int from)
{
    __shared__ UpdateSmem sm;
    uint32_t all = 0u;   // recompute the live total from the per-block sums
    for (uint32_t k = threadIdx.x; k < gridDim.x; k += blockDim.x) all += P.sort_part[k];
    all = block_sum(all, sm.wsum);
    sort_scatter(P, from, all, max(1u, (all + P.n_seg - 1u) / P.n_seg));
}

// Grid-wide barrier of the persistent kernel.  Arrival: bar.sync, then thread 0 adds 1 to the arrival counter with
// red.release.gpu (MEMBAR.ALL.GPU + REDG: the block's writes are performed before the count moves; no round trip).
// Departure: thread 0 polls the counter with ld.relaxed.gpu until it reaches generation x grid size, then reads it
// once more with ld.acquire.gpu (LDG.STRONG.GPU + CCTL.IVALL: it observes a value at the end of the chain of
// release reductions, so it synchronises with every arrival, and the SM's L1 holds nothing stale when the other
// threads are let through bar.sync and read the other SMs' writes with plain loads).  The counter is never reset inside a launch.  A spin
// that lasts longer than ~4 s sets the abort flag; every block then leaves the kernel and manta_step reports it.
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ bool grid_barrier(Counters *c, unsigned &gen, uint32_t *s_flag)
{
    __syncthreads();
    if (threadIdx.x == 0u) {
        gen += 1u;
        unsigned ab = 0u;
#if MANTA_BAR >= 1
        // arrival = one release reduction (no round trip); everybody polls the arrival counter itself
        const unsigned target = gen * gridDim.x;
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(&c->bar_count) : "memory");
        {
            const long long t0 = clock64();
            unsigned spins = 0u;
#if MANTA_BAR == 3
            while (ld_relaxed_u32(&c->bar_count) < target) {
#else
            while (ld_acquire_u32(&c->bar_count) < target) {
#endif
#else
        __threadfence();
        const unsigned prev = atomicAdd(&c->bar_count, 1u);
        if (prev + 1u == gen * gridDim.x) {
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(&c->bar_gen), "r"(gen) : "memory");
        } else {
            const long long t0 = clock64();
            unsigned spins = 0u;
            while (ld_acquire_u32(&c->bar_gen) < gen) {
#endif
                if ((++spins & 1023u) == 0u) {   // now and then: has another block given up, or is this taking seconds?
                    if (ld_acquire_u32(&c->abort)) {
                        ab = 1u;
                        break;
                    }
                    if (clock64() - t0 > 8000000000ll) {
                        atomicExch(&c->abort, 1u);
                        ab = 1u;
                        break;
                    }
                }
            }
        }
#if MANTA_BAR == 0
        __threadfence();
#elif MANTA_BAR == 3
        (void)ld_acquire_u32(&c->bar_count);   // the acquire (and the L1 invalidation) once, after the relaxed polling
#endif
        *s_flag = ab;
    }
    __syncthreads();
    return *s_flag == 0u;
}

// Litmus test of grid_barrier (manta_selftest_grid_barrier): in every round each block writes the round number into
// its own 32 words with PLAIN stores, passes the barrier, and every block reads ALL blocks' words with PLAIN loads --
// the very pattern the step phases rely on (writes before the arrival are visible after the departure, through each
// SM's L1) -- then a second barrier keeps the next round's writes behind everybody's reads.  Counts stale words.
__global__ void __launch_bounds__(MANTA_NT, MANTA_MINB) k_barrier_litmus(Counters *c, uint32_t *words, uint32_t n_rounds, unsigned long long *n_stale)
{
    __shared__ uint32_t flag;
    unsigned gen = 0u;
    unsigned long long bad = 0ull;
    for (uint32_t r = 1u; r <= n_rounds; r++) {
        for (uint32_t k = threadIdx.x; k < 32u; k += blockDim.x) words[blockIdx.x * 32u + k] = r;
        if (!grid_barrier(c, gen, &flag)) return;
        for (uint32_t k = threadIdx.x; k < gridDim.x * 32u; k += blockDim.x) bad += words[k] != r ? 1ull : 0ull;
        if (!grid_barrier(c, gen, &flag)) return;
    }
    if (bad) atomicAdd(n_stale, bad);
}

__device__ __forceinline__ bool sort_all(const DevP &P, UpdateSmem &sm, int from, unsigned &gen, Counters *ctr)
{
    uint32_t n_live, per_seg;
    sort_zero(P);
    if (!grid_barrier(ctr, gen, &sm.flag)) return false;
    sort_count(P, from);
    if (!grid_barrier(ctr, gen, &sm.flag)) return false;
    sort_partial(P, sm);
    if (!grid_barrier(ctr, gen, &sm.flag)) return false;
    sort_scan(P, sm, n_live, per_seg);
    if (!grid_barrier(ctr, gen, &sm.flag)) return false;
    sort_scatter(P, from, n_live, per_seg);
    return grid_barrier(ctr, gen, &sm.flag);
}

// One cooperative launch = n_steps timesteps; the host is not involved between steps.  Two grid barriers per
// timestep when the admission of step t + 1 is fused into the second phase of step t (fuse != 0), else three.
template <bool W256>
__global__ void __launch_bounds__(MANTA_NT, MANTA_MINB) k_persistent(const DevP P, uint32_t t0, uint32_t n_steps, int fuse)
{
    __shared__ UpdateSmem sm;
    if (threadIdx.x < 4u) sm.ev[threadIdx.x] = 0ull;
    unsigned gen = 0u;
    uint32_t n_cells = 0u, n_upd = 0u;
    const uint32_t t_end = t0 + n_steps;
    // the first step of a launch: re-sort if due, admission on its own
    if (sort_due(t0) && !sort_all(P, sm, sbuf_of(t0 - 1u), gen, P.ctr)) return;
    admit_phase<false>(P, t0, sbuf_of(t0));
    if (!grid_barrier(P.ctr, gen, &sm.flag)) return;
    for (uint32_t t = t0; t < t_end; t++) {
        DBG_STAMP(0);
        update_phase<W256>(P, t, sm, n_cells, n_upd, dyn_rec, true);
        if (!grid_barrier(P.ctr, gen, &sm.flag)) return;
        DBG_STAMP(4);
        const bool more = t + 1u < t_end;
        if (more && fuse) admit_phase<true>(P, t + 1u, sbuf_of(t));   // the longer dependent chain first
        DBG_STAMP(3);
        second_phase<W256>(P, t, sm, n_cells, true);
#ifdef MANTA_DBG
        if (threadIdx.x == MANTA_XT && (t & 31u) == 7u) P.dbg_buf[blockIdx.x * 8u + 7u] = gtimer();
#endif
#if MANTA_PF >= 3
        if (more) {   // the state records of this block's first chunks of step t + 1: on their way while the barrier completes
            const StBuf &Sn = P.st[sbuf_of(t + 1u)];
            for (uint32_t seg = blockIdx.x; seg < P.n_seg; seg += gridDim.x) {
                const uint32_t at = seg * P.seg_cap + threadIdx.x;
                if (threadIdx.x < P.seg_cnt[seg]) {
                    prefetch_line(&Sn.S0[at]);
                    prefetch_line(&Sn.S1[at]);
                    prefetch_line(&Sn.S2[at]);
                    prefetch_line(&Sn.S3[at]);
                }
            }
        }
#endif
        DBG_STAMP(5);
        if (!grid_barrier(P.ctr, gen, &sm.flag)) return;
        DBG_STAMP(6);
        if (more) {
            if (sort_due(t + 1u) && !sort_all(P, sm, sbuf_of(t), gen, P.ctr)) return;
            if (!fuse) {
                admit_phase<false>(P, t + 1u, sbuf_of(t + 1u));
                if (!grid_barrier(P.ctr, gen, &sm.flag)) return;
            }
        }
    }
    flush_stats(P, sm, n_cells, n_upd);
}

// ------------------------------------------------------------------------------------------------ replica batching
// SURVEY 8(f) N4 (the calibration runs several parameter sets per iteration): up to NB independent
// simulations -- own parameters, atlas, vehicles, results; same launch geometry and step counter -- advance in ONE
// cooperative launch.  Every phase loops over the replicas between the same two grid barriers per timestep, so the
// barriers, their fences and the wait for the slowest block are paid once per step instead of once per replica and
// step, and the SMs that a single simulation leaves idle ~ 40 % of a step have the other replicas' chunks to run.
// The barrier words are replica 0's.  Shared memory: the records of the two-stage pass (used by one replica's pass
// at a time), then one UpdateSmem per replica (its lists must survive the barrier between pass and second phase).
template <int NB>
struct BatchP {
    DevP p[NB];
};
#define MANTA_BATCH_SMEM(nb) (MANTA_REC_BYTES + (nb) * sizeof(UpdateSmem))
// per-thread counters of one pass -> the replica's shared counters (one shared atomic per warp and counter)
__device__ __forceinline__ void add_counts(UpdateSmem &sm, uint32_t n_cells, uint32_t n_upd)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        n_cells += __shfl_down_sync(0xFFFFFFFFu, n_cells, d);
        n_upd += __shfl_down_sync(0xFFFFFFFFu, n_upd, d);
    }
    if ((threadIdx.x & 31u) == 0u) {
        sm.wcnt[threadIdx.x >> 5][0] += (u64)n_cells;
        sm.wcnt[threadIdx.x >> 5][1] += (u64)n_upd;
    }
}
template <bool W256, int NB>
__global__ void __launch_bounds__(MANTA_NT, MANTA_MINB) k_persistent_batch(const BatchP<NB> Bp, int n_rep, uint32_t t0, uint32_t n_steps, int fuse)
{
    UpdateSmem *sm = reinterpret_cast<UpdateSmem *>(reinterpret_cast<unsigned char *>(dyn_rec) + MANTA_REC_BYTES);
    for (uint32_t k = threadIdx.x; k < (uint32_t)NB * (4u + 2u * MANTA_NW); k += blockDim.x) {
        UpdateSmem &q = sm[k / (4u + 2u * MANTA_NW)];
        const uint32_t j = k % (4u + 2u * MANTA_NW);
        if (j < 4u) q.ev[j] = 0ull;
        else q.wcnt[(j - 4u) >> 1][(j - 4u) & 1u] = 0ull;
    }
    Counters *ctr = Bp.p[0].ctr;
    unsigned gen = 0u;
    const uint32_t t_end = t0 + n_steps;
    // the replica loops are NOT unrolled: one copy of the phase code, the replica's parameter block addressed by r
    if (sort_due(t0)) {
#pragma unroll 1
        for (int r = 0; r < n_rep; r++)
            if (!sort_all(Bp.p[r], sm[r], sbuf_of(t0 - 1u), gen, ctr)) return;
    }
#pragma unroll 1
    for (int r = 0; r < n_rep; r++) admit_phase<false>(Bp.p[r], t0, sbuf_of(t0));
    if (!grid_barrier(ctr, gen, &sm[0].flag)) return;
    for (uint32_t t = t0; t < t_end; t++) {
#pragma unroll 1
        for (int r = 0; r < n_rep; r++) {
            uint32_t n_cells = 0u, n_upd = 0u;
            update_phase<W256>(Bp.p[r], t, sm[r], n_cells, n_upd, dyn_rec, true);
            add_counts(sm[r], n_cells, n_upd);
        }
        if (!grid_barrier(ctr, gen, &sm[0].flag)) return;
        const bool more = t + 1u < t_end;
#pragma unroll 1
        for (int r = 0; r < n_rep; r++) {
            uint32_t n_cells = 0u;
            if (more && fuse) admit_phase<true>(Bp.p[r], t + 1u, sbuf_of(t));
            second_phase<W256>(Bp.p[r], t, sm[r], n_cells, true, (uint32_t)r, (uint32_t)n_rep);
            add_counts(sm[r], n_cells, 0u);
        }
#if MANTA_PF >= 3
        if (more) {   // the state records of this block's first chunks of step t + 1, every replica's: on their way while the barrier completes
#pragma unroll 1
            for (int r = 0; r < n_rep; r++) {
                const DevP &P = Bp.p[r];
                const StBuf &Sn = P.st[sbuf_of(t + 1u)];
                const uint32_t at = blockIdx.x * P.seg_cap + threadIdx.x;
                if (blockIdx.x < P.n_seg && threadIdx.x < P.seg_cnt[blockIdx.x]) {
                    prefetch_line(&Sn.S0[at]);
                    prefetch_line(&Sn.S1[at]);
                    prefetch_line(&Sn.S2[at]);
                    prefetch_line(&Sn.S3[at]);
                }
            }
        }
#endif
        if (!grid_barrier(ctr, gen, &sm[0].flag)) return;
        if (more) {
            if (sort_due(t + 1u)) {
#pragma unroll 1
                for (int r = 0; r < n_rep; r++)
                    if (!sort_all(Bp.p[r], sm[r], sbuf_of(t), gen, ctr)) return;
            }
            if (!fuse) {
#pragma unroll 1
                for (int r = 0; r < n_rep; r++) admit_phase<false>(Bp.p[r], t + 1u, sbuf_of(t + 1u));
                if (!grid_barrier(ctr, gen, &sm[0].flag)) return;
            }
        }
    }
    __syncthreads();
#pragma unroll 1
    for (int r = 0; r < n_rep; r++) {
        if (threadIdx.x == 0u) {
            BlockStats *b = &Bp.p[r].blk[blockIdx.x];
            u64 c = 0ull, u = 0ull;
            for (uint32_t w = 0; w < (uint32_t)MANTA_NW; w++) {
                c += sm[r].wcnt[w][0];
                u += sm[r].wcnt[w][1];
            }
            if (c) atomicAdd(&b->cells_examined, c);
            if (u) atomicAdd(&b->n_updates, u);
        }
        flush_stats(Bp.p[r], sm[r], 0u, 0u);
    }
}

// ------------------------------------------------------------------------------------------------ set-up kernels
// Route expansion (load time, outside the timed path): RouteRec k from edge id re[k]; lo/hi of R0 from the next
// entry.  Entries that end a trip are fixed up by k_mark_last.
__global__ void k_expand_routes(const uint4 *edge_tab, const uint32_t *row_ptr, const uint32_t *re, uint64_t total,
                                uint4 *route)
{
    for (uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t e = re[k];
        const uint4 er = edge_tab[e];                       // {cell_off, static geom, head node, v0}
        const uint32_t n = GEOM_LANES(er.y);
        const uint32_t head = er.z & NODE_MASK;
        const uint32_t out_base = row_ptr[head], d = row_ptr[head + 1u] - out_base;
        uint32_t lo = 0u, hi = n - 1u;
        if (k + 1u < total) {
            const uint32_t j = re[k + 1u] - out_base;
            if (j < d) {
                lo = (j * n) / d;
                const uint32_t hi1 = ((j + 1u) * n) / d;
                hi = (hi1 >= 1u && hi1 - 1u > lo) ? hi1 - 1u : lo;
            }
        }
        const uint32_t geom = (er.y & 0x080FFFFFu) | (lo << 20) | (hi << 23);
        route[k] = make_uint4(er.x, geom, e, er.w);
    }
}
__global__ void k_mark_last(const uint64_t *route_ptr, uint32_t n_trips, uint4 *route)
{
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_trips; i += gridDim.x * blockDim.x) {
        const uint64_t k = route_ptr[i + 1u] - 1ull;
        uint4 r = route[k];
        const uint32_t n = GEOM_LANES(r.y);
        r.y = (r.y & 0x080FFFFFu) | (0u << 20) | ((n - 1u) << 23) | (1u << 26);
        route[k] = r;
    }
}
// Pre-placed vehicles (R1, last sentence): vehicle i of the list goes to segment i % n_seg; fill the state from the
// route store, mark atlas_0, count the entry.  init = {x_fx, v bits, vehicle id, route cursor}.
__global__ void k_place_initial(const DevP P, const uint4 *init, uint32_t n_init)
{
    const StBuf &S = P.st[0];
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_init; i += gridDim.x * blockDim.x) {
        const uint4 iv = init[i];
        const uint4 rr = P.route[iv.w];
        const size_t at = (size_t)(i % P.n_seg) * P.seg_cap + i / P.n_seg;
        const uint32_t geom = rr.y & GEOM_STATIC_MASK;      // lane 0, tag 0
        const Hops hp = build_hops(P, iv.w, geom, 0u);
        S.S0[at] = make_uint4(iv.x, iv.y, CELL_NONE, iv.z);   // no earlier mark
        S.S1[at] = make_uint4(rr.x, geom, iv.w, desired_speed_bits(P, iv.z, 0u, rr.w));
        S.S2[at] = hp.s2;
        S.S3[at] = hp.s3;
        const uint32_t cell = rr.x + (iv.x >> 10);
        mark_toggle(P.bits[0], cell);
        pay_store(P, P.pay[0], cell, iv.x & 1023u, iv.y);
        P.admit_step[iv.z] = 0u;
        atomicAdd(&P.edge_entries[rr.z], 1u);
    }
}
// manta_load_state, pass 1: nothing is written but the error word (1 bad status, 2 route position beyond the route,
// 3 lane / position beyond the edge, stop counter above 7, speed negative, not finite or above vcap (the layout's
// Z_out, cannot_cross and may_defer rest on v <= vcap: a faster vehicle would be moved outside its row),
// 4 an admitted trip behind a waiting one in its origin queue, 5 admit / arrive steps that contradict the status).
struct StateIn {
    const uint8_t *status, *lane, *tag, *wait;   // caller (trip) order; wait may be null
    const uint32_t *route_pos, *x_fx;
    const float *v;
    const uint2 *steps;                          // {admit_step, arrive_step} per trip
};
__global__ void k_state_validate(const DevP P, StateIn in, const uint32_t *trip_of_id, uint32_t n_trips, uint32_t t, uint32_t *err)
{
    for (uint32_t id = blockIdx.x * blockDim.x + threadIdx.x; id < n_trips; id += gridDim.x * blockDim.x) {
        const uint32_t tr = trip_of_id[id];
        const uint32_t st = in.status[tr];
        if (st > 2u) { atomicMax(err, 1u); continue; }
        const uint2 ab = in.steps[tr];
        // WAITING: neither step; ACTIVE: admitted by now, not arrived; DONE: admitted, then arrived, by now
        const bool steps_ok = st == 0u ? (ab.x == CELL_NONE && ab.y == CELL_NONE)
                            : st == 1u ? (ab.x <= t && ab.y == CELL_NONE)
                                       : (ab.x <= ab.y && ab.y <= t);
        if (!steps_ok) atomicMax(err, 5u);
        if (st != 1u) continue;
        if (in.route_pos[tr] >= P.route_len[id]) { atomicMax(err, 2u); continue; }
        const uint4 rr = P.route[P.route_start[id] + in.route_pos[tr]];
        if (in.lane[tr] >= GEOM_LANES(rr.y) || (in.x_fx[tr] >> 10) >= GEOM_LEN(rr.y) || (in.wait && in.wait[tr] > 7u) || !(in.v[tr] >= 0.0f) || !(in.v[tr] <= P.vcap))
            atomicMax(err, 3u);
    }
    for (uint32_t k = blockIdx.x * blockDim.x + threadIdx.x; k < P.n_queues; k += gridDim.x * blockDim.x) {
        bool waiting_seen = false;
        for (uint32_t i = P.q_begin[k]; i < P.q_end[k]; i++) {
            const bool waiting = in.status[trip_of_id[P.q_ent[i].x]] == 0u;
            if (waiting_seen && !waiting) atomicMax(err, 4u);
            waiting_seen = waiting_seen || waiting;
        }
    }
}
// pass 2: per-id results, vehicle slots (dealt round-robin over the segments through one counter), marks and payload of
// atlas_t (the other plane is empty: no vehicle has an earlier mark), arrival counters, queue heads.
__global__ void k_state_load(const DevP P, StateIn in, const uint32_t *trip_of_id, uint32_t n_trips, uint32_t t, int sb,
                             uint32_t *slot_counter, uint32_t *err)
{
    const StBuf &S = P.st[sb];
    u64 *B = P.bits[t & 1u];
    uint2 *pay = P.pay[t & 1u];
    unsigned long long done = 0ull, travel = 0ull;
    for (uint32_t id = blockIdx.x * blockDim.x + threadIdx.x; id < n_trips; id += gridDim.x * blockDim.x) {
        const uint32_t tr = trip_of_id[id];
        const uint2 steps = in.steps[tr];
        P.admit_step[id] = steps.x;
        P.arrive_step[id] = steps.y;
        const uint32_t st = in.status[tr];
        if (st == 2u) {
            done += 1ull;
            travel += (unsigned long long)(steps.y - steps.x);
        }
        if (st != 1u) continue;
        const uint32_t cursor = P.route_start[id] + in.route_pos[tr];
        const uint4 rr = P.route[cursor];
        const uint32_t l = in.lane[tr];
        const uint32_t geom = (rr.y & GEOM_STATIC_MASK) | (l << 28) | ((uint32_t)(in.tag[tr] != 0u) << 31);
        const uint32_t row = rr.x + l * pitch_of(GEOM_LEN(rr.y));
        const Hops hp = build_hops(P, cursor, geom, l);
        const uint32_t slot = atomicAdd(slot_counter, 1u);
        const size_t at = (size_t)(slot % P.n_seg) * P.seg_cap + slot / P.n_seg;
        const uint32_t x = in.x_fx[tr], vb = __float_as_uint(in.v[tr]);
        S.S0[at] = make_uint4(x | ((in.wait ? (uint32_t)in.wait[tr] : 0u) << WAIT_SHIFT), vb, CELL_NONE, id);
        S.S1[at] = make_uint4(row, geom, cursor, desired_speed_bits(P, id, in.route_pos[tr], rr.w));
        S.S2[at] = hp.s2;
        S.S3[at] = hp.s3;
        if (S.acc) S.acc[at] = 0.0f;
        const uint32_t cell = row + (x >> 10);
        const u64 bit = 1ull << (cell & 63u);
        if (atomicOr(&B[cell >> 6], bit) & bit) atomicMax(err, 5u);   // two vehicles in one cell
        pay_store(P, pay, cell, x & 1023u, vb);
    }
    if (done) {
        atomicAdd(&P.blk[blockIdx.x % 64u].n_done, done);
        atomicAdd(&P.blk[blockIdx.x % 64u].sum_travel, travel);
    }
    for (uint32_t k = blockIdx.x * blockDim.x + threadIdx.x; k < P.n_queues; k += gridDim.x * blockDim.x) {
        uint32_t i = P.q_begin[k];
        const uint32_t end = P.q_end[k];
        while (i < end && in.status[trip_of_id[P.q_ent[i].x]] != 0u) i++;
        const uint4 h = P.q_ent[i];   // (the padding entry after the last queue if i == total)
        P.q_state[k] = i < end ? make_uint4(h.y, i, h.x, h.z) : make_uint4(CELL_NONE, i, CELL_NONE, 0u);
    }
}
__global__ void k_state_counts(const DevP P, const uint32_t *slot_counter)
{
    const uint32_t total = *slot_counter;
    for (uint32_t seg = blockIdx.x * blockDim.x + threadIdx.x; seg < P.n_seg; seg += gridDim.x * blockDim.x)
        P.seg_cnt[seg] = total / P.n_seg + (seg < total % P.n_seg ? 1u : 0u);
}

// Readback: scatter the live slots of the segments into per-trip arrays (caller order).
__global__ void k_gather_state(const DevP P, int sb, const uint32_t *trip_of_id, uint8_t *status, uint32_t *route_pos,
                               uint8_t *lane, uint8_t *tag, uint32_t *x_fx, float *v, float *acc, uint8_t *wait,
                               unsigned long long *n_stopped)
{
    const StBuf &S = P.st[sb];
    for (uint32_t seg = blockIdx.x; seg < P.n_seg; seg += gridDim.x) {
        const uint32_t n = P.seg_cnt[seg];
        const size_t seg_base = (size_t)seg * P.seg_cap;
        for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
            const uint4 s0v = S.S0[seg_base + i];
            if (s0v.w >= ID_GHOST) continue;
            const uint4 s1v = S.S1[seg_base + i];
            const uint32_t tr = trip_of_id[s0v.w];
            status[tr] = 1u;
            route_pos[tr] = s1v.z - P.route_start[s0v.w];
            lane[tr] = (uint8_t)GEOM_LANE(s1v.y);
            tag[tr] = (uint8_t)GEOM_TAG(s1v.y);
            x_fx[tr] = s0v.x & X_MASK;
            wait[tr] = (uint8_t)(s0v.x >> WAIT_SHIFT);
            if (__uint_as_float(s0v.y) == 0.0f) atomicAdd(n_stopped, 1ull);
            v[tr] = __uint_as_float(s0v.y);
            acc[tr] = S.acc ? S.acc[seg_base + i] : 0.0f;
        }
    }
}
__global__ void k_status_from_steps(uint32_t n_trips, const uint32_t *trip_of_id, const uint32_t *admit_step,
                                    const uint32_t *arrive_step, uint8_t *status, uint2 *results)
{
    for (uint32_t id = blockIdx.x * blockDim.x + threadIdx.x; id < n_trips; id += gridDim.x * blockDim.x) {
        const uint32_t tr = trip_of_id[id];
        const uint32_t a = admit_step[id], b = arrive_step[id];
        status[tr] = b != 0xFFFFFFFFu ? 2u : (a != 0xFFFFFFFFu ? 1u : 0u);
        results[tr] = make_uint2(a, b);
    }
}
// Logical atlas of the current step for tests: occ = 0 / 1 + frac10, spd = occupant's speed
__global__ void k_export_atlas(const u64 *B, const uint2 *pay, uint32_t pay_shift, uint64_t n_cells, uint16_t *occ, float *spd)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_cells; i += (uint64_t)gridDim.x * blockDim.x) {
        const bool on = (B[i >> 6] >> (i & 63ull)) & 1ull;
        const uint2 pc = on ? pay[i >> pay_shift] : make_uint2(0u, 0u);
        occ[i] = on ? (uint16_t)(1u + pc.x) : (uint16_t)0u;
        spd[i] = on ? __uint_as_float(pc.y) : 0.0f;
    }
}

}  // namespace manta
