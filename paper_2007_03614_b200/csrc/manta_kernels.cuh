// manta_kernels.cuh -- the three phases of one MANTA timestep as device functions, plus their kernels.
//
//   A admit   (R1)      : one thread per origin-edge FIFO; idle queues cost one coalesced load (q_next); a due head
//                         trip is released if its entry window is free
//   U update  (R2-R9)   : one thread block per vehicle segment, one thread per active vehicle.  First pass: leader
//                         search on the time-t occupancy words (the next four route records are requested up
//                         front, the words of a row are requested together), IDM, lane-change pre-tests.  Vehicles
//                         that must look at the adjacent lane (~6 %) are parked in a shared-memory queue and handled
//                         by a dense second pass, so they do not hold their warps.  Vehicles that stay on their
//                         edge (the great majority) finish the step here: next state to the compacted next buffer
//                         of the segment (warp ballot + one shared-memory atomic per warp), time-(t+1) mark and
//                         payload, time-(t-1) mark toggled off.  Edge-end candidates post a min-id claim and a
//                         cross-list entry; arrivals post a cross-list entry.
//   X cross   (R8, R9)  : one thread per cross-list entry: resolves the claim (winner moves to its next route
//                         edge, loser holds at the stop line), writes its mark; clears the marks of arrivals.
//
// A grid-wide barrier separates the phases: the software barrier of k_persistent (one cooperative launch runs
// many timesteps), or kernel boundaries (k_admit / k_update / k_cross: MANTA_FLAG_MULTI_KERNEL, manta_step_timed).
#pragma once
#include "manta_device.cuh"

namespace manta {

#ifndef MANTA_NT
#define MANTA_NT 512      // threads per block of the step kernels
#endif
#ifndef MANTA_MINB
#define MANTA_MINB 1      // blocks per SM the step kernels are compiled for
#endif
#define MANTA_NW (MANTA_NT / 32)
#define MANTA_QCAP 64     // lane-change queue entries per warp (drained whenever 32 or more are waiting)
#define MANTA_MAX_LANES_DEV 8u

struct Lead {
    bool found;
    int32_t lead_abs;   // leader position in the follower's frame, Q22.10 (R2)
    float v_lead;
};

// Per-vehicle context carried from the leader search to the end of the update.
struct Veh {
    int32_t x;
    float v, v0;
    uint32_t id, cursor, cell_off, geom, prev;
    uint32_t len_c, n, l, c, pitch;
    bool last;
    uint4 rn;           // next route record (valid unless last)
    // after pre_lc
    float acc_cur;
    int32_t bound;
    uint32_t tag, lt;
    bool mand, disc_pre, need_lc;
};

struct Outcome {
    uint32_t kind, nx, l_new, word;
    float vn, acc;
};

// shared memory of the update phase
struct UpdateSmem {
    u64 stats[6];                 // lane_changes, cells_examined, lc_evals, n_updates, n_done, sum_travel (kernel lifetime)
    uint32_t out, xn, flag, pad;  // per segment: survivors written, cross-list entries; barrier flag
    uint4 q[MANTA_NW][MANTA_QCAP]; // per-warp queues of lane-change evaluations: {slot, lead_abs, v_lead bits, found}
};
enum { ST_LC = 0, ST_CELLS = 1, ST_EVAL = 2, ST_UPD = 3, ST_DONE = 4, ST_TRAVEL = 5 };

__device__ __forceinline__ void veh_load(Veh &V, const uint4 &s0v, const uint4 &s1v)
{
    V.x = (int32_t)s0v.x;
    V.v = __uint_as_float(s0v.y);
    V.id = s0v.z;
    V.cursor = s0v.w;
    V.cell_off = s1v.x;
    V.geom = s1v.y;
    V.prev = s1v.z;
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
// follower's edge; the caller fetches the payload once, after the search, for the whole warp.
struct Hit {
    bool found;
    uint32_t cell, dist;
};

// Generic walk (any H): one row after the other, records fetched as the walk reaches them.  Starts at `hop`
// records past the vehicle's cursor, in row `row` of length `len` at cell `start`.
template <bool W256>
__device__ __forceinline__ Hit walk_rows(const DevP &P, const u64 *B, const uint4 *rp, uint32_t hop, uint32_t row, uint32_t len,
                                         uint32_t start, uint32_t l, uint32_t rem, uint32_t dist_base, bool last,
                                         uint32_t &examined)
{
    Hit h;
    h.found = false;
    h.cell = 0u;
    h.dist = 0u;
    for (;;) {
        const uint32_t end = min(len, start + rem);
        if (start < end) {
            uint32_t j;
            if (scan_fwd<W256>(B, row, start, end, j)) {
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

// H <= 256.  Three rounds of loads at most for nearly every vehicle: (1) the words of the own row together with
// the next four route records (consecutive in memory); (2) the first two words of each of the next four rows,
// all requested together; (3) the leader's payload (by the caller).  Longer walks (a row with more than 128
// cells to examine after the own one, more than four hops) continue with dependent loads.  Records past the
// trip's last one belong to another trip: they may be loaded but are never used (the walk stops at `last`).
__device__ __forceinline__ Hit leader_cells_w(const DevP &P, const u64 *B, Veh &V, uint32_t &examined)
{
    Hit h;
    h.found = false;
    h.cell = 0u;
    h.dist = 0u;
    const uint4 *rp = P.route + V.cursor;
    uint2 rr[4];
    V.rn = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
    for (int k = 0; k < 4; k++) rr[k] = make_uint2(0u, 0u);
    if (!V.last) {
        V.rn = rp[1];
        rr[1] = *reinterpret_cast<const uint2 *>(rp + 2);
        rr[2] = *reinterpret_cast<const uint2 *>(rp + 3);
        rr[3] = *reinterpret_cast<const uint2 *>(rp + 4);
    }
    uint32_t rem = P.H;
    const uint32_t row0 = V.cell_off + V.l * V.pitch;
    {   // own row
        const uint32_t start = V.c + 1u, end = min(V.len_c, start + rem);
        if (start < end) {
            uint32_t j;
            if (first_set_w(B, row0, start, end, j)) {
                examined += j - start + 1u;
                h.found = true;
                h.cell = row0 + j;
                h.dist = j;
                return h;
            }
            examined += end - start;
            rem -= end - start;
        }
    }
    if (rem == 0u || V.last) return h;
    rr[0] = make_uint2(V.rn.x, V.rn.y);
    uint32_t rowk[4], nk[4], lenk[4];
    u64 wa[4], wb[4];
    bool valid = true;
    uint32_t lk = V.l;
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const uint32_t g = rr[k].y;
        lenk[k] = GEOM_LEN(g);
        lk = min(lk, GEOM_LANES(g) - 1u);
        rowk[k] = rr[k].x + lk * pitch_of(lenk[k]);
        nk[k] = valid ? min(lenk[k], rem) : 0u;
        wa[k] = nk[k] ? B[rowk[k] >> 6] : 0ull;
        wb[k] = nk[k] > 64u ? B[(rowk[k] >> 6) + 1u] : 0ull;
        rem -= nk[k];
        valid = valid && GEOM_LAST(g) == 0u && rem > 0u;
    }
    uint32_t dist_base = V.len_c;
#pragma unroll
    for (int k = 0; k < 4; k++) {
        if (nk[k] && !h.found) {
            const u64 ma = wa[k] & bits_below(min(nk[k], 64u));
            uint32_t j = 0u;
            bool f = false;
            if (ma) {
                j = (uint32_t)__ffsll((long long)ma) - 1u;
                f = true;
            } else if (nk[k] > 64u) {
                const u64 mb = wb[k] & bits_below(min(nk[k] - 64u, 64u));
                if (mb) {
                    j = 64u + (uint32_t)__ffsll((long long)mb) - 1u;
                    f = true;
                } else if (nk[k] > 128u) {
                    f = first_set_w(B, rowk[k], 128u, nk[k], j);
                }
            }
            if (f) {
                examined += j + 1u;
                h.found = true;
                h.cell = rowk[k] + j;
                h.dist = dist_base + j;
            } else {
                examined += nk[k];
            }
        }
        dist_base += lenk[k];
    }
    if (h.found || !valid) return h;
    // more than four hops: go on from the end of the fourth row (start = len: nothing left to examine in it)
    return walk_rows<true>(P, B, rp, 4u, rowk[3], lenk[3], lenk[3], lk, rem, dist_base - lenk[3], false, examined);
}

template <bool W256>
__device__ __forceinline__ Lead leader_search(const DevP &P, const u64 *B, const uint2 *pay, Veh &V, uint32_t &examined)
{
    Hit h;
    if (W256) {
        h = leader_cells_w(P, B, V, examined);
    } else {
        V.rn = make_uint4(0u, 0u, 0u, 0u);
        if (!V.last) V.rn = P.route[V.cursor + 1u];
        h = walk_rows<false>(P, B, P.route + V.cursor, 0u, V.cell_off + V.l * V.pitch, V.len_c, V.c + 1u, V.l, P.H, 0u, V.last,
                             examined);
    }
    Lead L;
    L.found = h.found;
    L.lead_abs = 0;
    L.v_lead = 0.0f;
    if (h.found) {
        const uint2 pc = pay[h.cell];
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
    V.acc_cur = idm_acc(P, V.v, V.v0, ld.found, s, ld.v_lead);
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
            float rr = V.v / V.v0;
            float rr2 = rr * rr;
            float fr = rr2 * rr2;
            float af = 1.0f - fr;
            af = P.a * af;
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
                                           bool has_b, int32_t x_b, float v_b, uint32_t &n_lc)
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
                n_lc += 1u;
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
    O.word = 0u;
    const int32_t len_fx = (int32_t)(V.len_c << 10);
    if (xn < len_fx) {
        O.kind = KIND_STAY;
        O.nx = (uint32_t)xn;
    } else if (V.last) {
        O.kind = KIND_DONE;  // G18
        O.nx = 0u;
    } else {
        if (GEOM_PRIO(V.geom)) {   // PRIORITY: the claim word is the head node of this edge
            O.word = P.n_edges * 8u + P.edge_tab[P.route[V.cursor].z].z;
        } else {                   // GREEN: the lane entry (e+, l+)
            O.word = V.rn.z * 8u + min(l_new, GEOM_LANES(V.rn.y) - 1u);
        }
        O.kind = KIND_CAND;
        O.nx = (uint32_t)(xn - len_fx);
        // smallest id wins; the key carries ~t in the high word so claim words never need a reset
        const u64 key = ((u64)(0xFFFFFFFFu - t) << 32) | (u64)V.id;
        atomicMin(&P.claim[O.word], key);
    }
    return O;
}

// R5: lead (first occupied cell >= c, within the edge) and lag (last occupied cell < c) in the target lane, then
// the rest of the update.
template <bool W256>
__device__ __forceinline__ Outcome lane_change_and_finish(const DevP &P, uint32_t t, const u64 *B, const uint2 *pay, const Veh &V,
                                                          uint32_t &n_lc)
{
    const uint32_t rowt = V.cell_off + V.lt * V.pitch;
    uint32_t ja = 0u, jb = 0u;
    const uint32_t b0 = V.c > P.lookback ? V.c - P.lookback : 0u;
    const bool has_a = scan_fwd<W256>(B, rowt, V.c, min(V.len_c, V.c + P.H), ja);
    const bool has_b = V.c > b0 && scan_bwd<W256>(B, rowt, b0, V.c, jb);
    int32_t x_a = 0, x_b = 0;
    float v_a = 0.0f, v_b = 0.0f;
    uint2 pa = make_uint2(0u, 0u), pb = pa;
    if (has_a) pa = pay[(size_t)rowt + ja];
    if (has_b) pb = pay[(size_t)rowt + jb];
    if (has_a) {
        x_a = (int32_t)((ja << 10) | pa.x);
        v_a = __uint_as_float(pa.y);
    }
    if (has_b) {
        x_b = (int32_t)((jb << 10) | pb.x);
        v_b = __uint_as_float(pb.y);
    }
    return post_lc(P, t, V, has_a, x_a, v_a, has_b, x_b, v_b, n_lc);
}

// R9 for one warp's vehicles: survivors compacted into the segment's next buffer (warp ballot + one shared-memory
// atomic), time-(t+1) mark and payload for stayers, time-(t-1) mark toggled off, cross-list entries.  Must be
// called by all 32 lanes; `have` says whether this lane carries a vehicle.
__device__ __forceinline__ void write_out(const DevP &P, uint32_t t, UpdateSmem &sm, uint32_t seg_base, bool have, const Veh &V,
                                          const Outcome &O)
{
    const int nxt = (int)((t & 1u) ^ 1u);
    u64 *Bn = P.bits[nxt];
    const uint32_t lane_id = threadIdx.x & 31u;
    const bool alive = have && O.kind != KIND_DONE, listed = have && O.kind != KIND_STAY;
    const uint32_t bal_a = __ballot_sync(0xFFFFFFFFu, alive), bal_x = __ballot_sync(0xFFFFFFFFu, listed);
    uint32_t base_a = 0u, base_x = 0u;
    if (lane_id == 0u) {
        if (bal_a) base_a = atomicAdd(&sm.out, (uint32_t)__popc(bal_a));
        if (bal_x) base_x = atomicAdd(&sm.xn, (uint32_t)__popc(bal_x));
    }
    base_a = __shfl_sync(0xFFFFFFFFu, base_a, 0);
    base_x = __shfl_sync(0xFFFFFFFFu, base_x, 0);
    if (!have) return;
    const uint32_t lt_mask = (1u << lane_id) - 1u;
    const uint32_t pos = base_a + __popc(bal_a & lt_mask);
    const uint32_t xpos = seg_base + base_x + __popc(bal_x & lt_mask);
    const uint32_t cur_abs = V.cell_off + V.l * V.pitch + V.c;
    const uint32_t geom_n = (V.geom & GEOM_STATIC_MASK) | (O.l_new << 28) | (V.tag << 31);
    if (O.kind == KIND_STAY) {
        const uint32_t cell = V.cell_off + O.l_new * V.pitch + (O.nx >> 10);
        if (V.prev != CELL_NONE)
            mark_move(Bn, V.prev, cell);
        else
            mark_toggle(Bn, cell);
        P.pay[nxt][cell] = make_uint2(O.nx & 1023u, __float_as_uint(O.vn));
    } else {
        if (V.prev != CELL_NONE) mark_toggle(Bn, V.prev);
        if (O.kind == KIND_DONE) {
            P.xlist[xpos] = make_uint4(XL_DONE, cur_abs, 0u, 0u);
            P.arrive_step[V.id] = t + 1u;
            atomicAdd(&sm.stats[ST_DONE], 1ull);
            atomicAdd(&sm.stats[ST_TRAVEL], (u64)(t + 1u - P.admit_step[V.id]));
        } else {
            P.xlist[xpos] = make_uint4(pos, O.word, V.cursor, V.id);
        }
    }
    if (alive) {  // candidates: tentative winner state; the cross phase decides
        P.S0[nxt][seg_base + pos] = make_uint4(O.nx, __float_as_uint(O.vn), V.id, V.cursor);
        P.S1[nxt][seg_base + pos] = make_uint4(V.cell_off, geom_n, cur_abs, __float_as_uint(V.v0));
        if (P.acc[nxt]) P.acc[nxt][seg_base + pos] = O.acc;
    }
}

// ------------------------------------------------------------------------------------------------ A: R1
// Departure admission (G17, G25).  Thread k owns the FIFO of one origin edge; trips in it are in
// vehicle-id (= departure) order, so the head is the smallest waiting id on that edge.
__device__ __forceinline__ void admit_phase(const DevP &P, uint32_t t, uint32_t gtid, uint32_t gsize)
{
    const int cur = (int)(t & 1u);
    u64 *B = P.bits[cur];
    uint2 *pay = P.pay[cur];
    const u64 window = bits_below(P.L_c + 1u);
    for (uint32_t k = gtid; k < P.n_queues; k += gsize) {
        if (P.q_next[k] > t) continue;                 // idle (or exhausted: NONE) queue
        const uint32_t h = P.q_head[k];
        const uint4 er = P.q_row[k];
        const uint4 ent = P.q_ent[h];                  // {id, depart_step, route_start, depart_step of the next entry}
        const uint32_t len = GEOM_LEN(er.y), lanes = GEOM_LANES(er.y), pitch = pitch_of(len);
        u64 w[MANTA_MAX_LANES_DEV];
#pragma unroll
        for (uint32_t l = 0; l < MANTA_MAX_LANES_DEV; l++) w[l] = l < lanes ? B[(er.x + l * pitch) >> 6] : ~0ull;
        uint32_t l_sel = 0xFFFFFFFFu;
#pragma unroll
        for (uint32_t l = 0; l < MANTA_MAX_LANES_DEV; l++)
            if (l_sel == 0xFFFFFFFFu && !(w[l] & window)) l_sel = l;   // first lane whose window [0, L_c] is free
        if (l_sel == 0xFFFFFFFFu) continue;
        const uint32_t id = ent.x, cursor = ent.z;
        const uint4 rr = P.route[cursor];
        // the emptier of two pseudo-random segments (keeps the segments balanced as trips come and go)
        uint32_t hsh = mix32(k * 0x9E3779B9u + t);
        uint32_t sa = hsh % P.n_seg, sb = (sa + 1u + (hsh >> 16) % max(P.n_seg - 1u, 1u)) % P.n_seg;
        uint32_t seg = P.seg_cnt[cur][sb] < P.seg_cnt[cur][sa] ? sb : sa;
        uint32_t slot;
        for (;;) {
            slot = atomicAdd(&P.seg_cnt[cur][seg], 1u);
            if (slot < P.seg_cap) break;
            atomicSub(&P.seg_cnt[cur][seg], 1u);       // full: the total capacity covers every trip, so another has room
            seg = seg + 1u == P.n_seg ? 0u : seg + 1u;
        }
        const uint32_t row = er.x + l_sel * pitch;
        const size_t at = (size_t)seg * P.seg_cap + slot;
        P.S0[cur][at] = make_uint4(0u, 0u, id, cursor);
        P.S1[cur][at] = make_uint4(rr.x, (rr.y & GEOM_STATIC_MASK) | (l_sel << 28), CELL_NONE, rr.w);
        if (P.acc[cur]) P.acc[cur][at] = 0.0f;
        mark_toggle(B, row);                           // cell 0, frac10 = 0, v = 0: visible to this step's update
        pay[(size_t)row] = make_uint2(0u, 0u);
        P.admit_step[id] = t;
        atomicAdd(&P.edge_entries[rr.z], 1u);
        P.q_head[k] = h + 1u;
        P.q_next[k] = ent.w;
    }
}

// ------------------------------------------------------------------------------------------------ U: R2-R9
// Second pass of one warp: the lane-change evaluations it has parked, densely packed over its lanes.
template <bool W256>
__device__ __forceinline__ void drain_lc(const DevP &P, uint32_t t, UpdateSmem &sm, uint32_t seg_base, uint32_t &qn, uint32_t &n_cells,
                                         uint32_t &n_lc)
{
    const int cur = (int)(t & 1u);
    const u64 *B = P.bits[cur];
    const uint2 *pay = P.pay[cur];
    const uint32_t lane_id = threadIdx.x & 31u, warp_id = threadIdx.x >> 5;
    __syncwarp();
    while (qn > 0u) {
        const uint32_t take = min(qn, 32u);
        const bool have = lane_id < take;
        Veh V;
        Outcome O;
        O.kind = KIND_STAY;
        if (have) {
            const uint4 e = sm.q[warp_id][qn - take + lane_id];
            veh_load(V, P.S0[cur][seg_base + e.x], P.S1[cur][seg_base + e.x]);
            V.rn = make_uint4(0u, 0u, 0u, 0u);
            if (!V.last) V.rn = P.route[V.cursor + 1u];
            Lead ld;
            ld.found = e.w != 0u;
            ld.lead_abs = (int32_t)e.y;
            ld.v_lead = __uint_as_float(e.z);
            pre_lc(P, t, V, ld);
            O = lane_change_and_finish<W256>(P, t, B, pay, V, n_lc);
        }
        write_out(P, t, sm, seg_base, have, V, O);
        qn -= take;
    }
    __syncwarp();
}

// Must be called by ALL threads of the block (contains __syncthreads).
template <bool W256>
__device__ __forceinline__ void update_phase(const DevP &P, uint32_t t, UpdateSmem &sm)
{
    const int cur = (int)(t & 1u), nxt = cur ^ 1;
    const u64 *B = P.bits[cur];
    const uint2 *pay = P.pay[cur];
    const uint32_t lane_id = threadIdx.x & 31u, warp_id = threadIdx.x >> 5;
    for (uint32_t seg = blockIdx.x; seg < P.n_seg; seg += gridDim.x) {
        const uint32_t n = P.seg_cnt[cur][seg];
        const uint32_t seg_base = seg * P.seg_cap;
        if (threadIdx.x == 0u) {
            sm.out = 0u;
            sm.xn = 0u;
        }
        __syncthreads();
        uint32_t n_cells = 0u, n_lc = 0u, qn = 0u;
        for (uint32_t base = warp_id * 32u; base < n; base += blockDim.x) {
            // ---- first pass: everything but the adjacent-lane look-up
            const uint32_t i = base + lane_id;
            const bool have = i < n;
            Veh V;
            Outcome O;
            O.kind = KIND_STAY;
            Lead ld;
            ld.found = false;
            ld.lead_abs = 0;
            ld.v_lead = 0.0f;
            bool want_q = false;
            if (have) {
                veh_load(V, P.S0[cur][seg_base + i], P.S1[cur][seg_base + i]);
                ld = leader_search<W256>(P, B, pay, V, n_cells);
                pre_lc(P, t, V, ld);
                want_q = V.need_lc;
                if (!want_q) O = post_lc(P, t, V, false, 0, 0.0f, false, 0, 0.0f, n_lc);
            }
            const uint32_t bal_q = __ballot_sync(0xFFFFFFFFu, want_q);
            if (want_q)   // parked: vehicles that must look at the adjacent lane (R5) do not hold the warp
                sm.q[warp_id][qn + __popc(bal_q & ((1u << lane_id) - 1u))] =
                    make_uint4(i, (uint32_t)ld.lead_abs, __float_as_uint(ld.v_lead), ld.found ? 1u : 0u);
            write_out(P, t, sm, seg_base, have && !want_q, V, O);
            if (bal_q) {
                qn += (uint32_t)__popc(bal_q);
                if (lane_id == 0u) atomicAdd(&sm.stats[ST_EVAL], (u64)__popc(bal_q));
                if (qn >= 32u) drain_lc<W256>(P, t, sm, seg_base, qn, n_cells, n_lc);
            }
        }
        drain_lc<W256>(P, t, sm, seg_base, qn, n_cells, n_lc);
        // ---- per-segment bookkeeping
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            n_cells += __shfl_down_sync(0xFFFFFFFFu, n_cells, d);
            n_lc += __shfl_down_sync(0xFFFFFFFFu, n_lc, d);
        }
        if (lane_id == 0u) {
            if (n_cells) atomicAdd(&sm.stats[ST_CELLS], (u64)n_cells);
            if (n_lc) atomicAdd(&sm.stats[ST_LC], (u64)n_lc);
        }
        __syncthreads();
        if (threadIdx.x == 0u) {
            P.seg_cnt[nxt][seg] = sm.out;
            P.seg_xn[seg] = sm.xn;
            sm.stats[ST_UPD] += (u64)n;
        }
    }
}

// ------------------------------------------------------------------------------------------------ X: R8, R9
__device__ __forceinline__ void cross_phase(const DevP &P, uint32_t t)
{
    const int cur = (int)(t & 1u), nxt = cur ^ 1;
    u64 *Bc = P.bits[cur];
    u64 *Bn = P.bits[nxt];
    uint2 *payn = P.pay[nxt];
    for (uint32_t seg = blockIdx.x; seg < P.n_seg; seg += gridDim.x) {
        const uint32_t n = P.seg_xn[seg];
        const size_t seg_base = (size_t)seg * P.seg_cap;
        for (uint32_t k = threadIdx.x; k < n; k += blockDim.x) {
            const uint4 xl = P.xlist[seg_base + k];     // {slot | XL_DONE, claim word | cell, cursor, id}
            if (xl.x == XL_DONE) {
                mark_toggle(Bc, xl.y);    // an arrival leaves no time-(t+1) state to clear its time-t mark later
                continue;
            }
            uint4 s0 = P.S0[nxt][seg_base + xl.x];
            uint4 s1 = P.S1[nxt][seg_base + xl.x];
            const u64 won = P.claim[xl.y];
            const uint4 rn = P.route[xl.z + 1u];
            const u64 key = ((u64)(0xFFFFFFFFu - t) << 32) | (u64)xl.w;
            if (won == key) {             // winner crosses (R8)
                const uint32_t lplus = min(GEOM_LANE(s1.y), GEOM_LANES(rn.y) - 1u);
                s0.w += 1u;
                s1 = make_uint4(rn.x, (rn.y & GEOM_STATIC_MASK) | (lplus << 28), s1.z, rn.w);
                atomicAdd(&P.edge_entries[rn.z], 1u);
            } else {                      // loser holds at the stop line (G15)
                s0.x = (GEOM_LEN(s1.y) << 10) - 1u;
                s0.y = 0u;
            }
            P.S0[nxt][seg_base + xl.x] = s0;
            P.S1[nxt][seg_base + xl.x] = s1;
            const uint32_t cell = s1.x + GEOM_LANE(s1.y) * pitch_of(GEOM_LEN(s1.y)) + (s0.x >> 10);
            mark_toggle(Bn, cell);
            payn[cell] = make_uint2(s0.x & 1023u, s0.y);
        }
    }
}

__device__ __forceinline__ void flush_stats(const DevP &P, UpdateSmem &sm)
{
    __syncthreads();
    if (threadIdx.x == 0u) {
        BlockStats *b = &P.blk[blockIdx.x];
        b->lane_changes += sm.stats[ST_LC];
        b->cells_examined += sm.stats[ST_CELLS];
        b->lc_evals += sm.stats[ST_EVAL];
        b->n_updates += sm.stats[ST_UPD];
        b->n_done += sm.stats[ST_DONE];
        b->sum_travel += sm.stats[ST_TRAVEL];
    }
}

// ------------------------------------------------------------------------------------------------ kernels
__global__ void __launch_bounds__(256) k_admit(const DevP P, uint32_t t)
{
    admit_phase(P, t, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}

template <bool W256>
__global__ void __launch_bounds__(MANTA_NT, MANTA_MINB) k_update(const DevP P, uint32_t t)
{
    __shared__ UpdateSmem sm;
    if (threadIdx.x < 6u) sm.stats[threadIdx.x] = 0ull;
    __syncthreads();
    update_phase<W256>(P, t, sm);
    flush_stats(P, sm);
}

__global__ void __launch_bounds__(256) k_cross(const DevP P, uint32_t t) { cross_phase(P, t); }

// Grid-wide barrier of the persistent kernel: arrival counter + generation word, release / acquire at gpu scope
// (the fences also invalidate L1, so plain loads after the barrier see the other SMs' writes).  A spin that lasts
// longer than ~4 s sets the abort flag; every block then leaves the kernel and manta_step reports the failure.
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ bool grid_barrier(Counters *c, unsigned &gen, uint32_t *s_flag)
{
    __syncthreads();
    if (threadIdx.x == 0u) {
        gen += 1u;
        __threadfence();
        const unsigned prev = atomicAdd(&c->bar_count, 1u);
        if (prev + 1u == gen * gridDim.x) {
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(&c->bar_gen), "r"(gen) : "memory");
        } else {
            const long long t0 = clock64();
            while (ld_acquire_u32(&c->bar_gen) < gen) {
                if (ld_acquire_u32(&c->abort)) break;
                if (clock64() - t0 > 8000000000ll) {
                    atomicExch(&c->abort, 1u);
                    break;
                }
            }
        }
        __threadfence();
        *s_flag = ld_acquire_u32(&c->abort);
    }
    __syncthreads();
    return *s_flag == 0u;
}

// One cooperative launch = n_steps timesteps; the host is not involved between steps.
template <bool W256>
__global__ void __launch_bounds__(MANTA_NT, MANTA_MINB) k_persistent(const DevP P, uint32_t t0, uint32_t n_steps)
{
    __shared__ UpdateSmem sm;
    if (threadIdx.x < 6u) sm.stats[threadIdx.x] = 0ull;
    unsigned gen = 0u;
    const uint32_t gtid = blockIdx.x * blockDim.x + threadIdx.x, gsize = gridDim.x * blockDim.x;
    for (uint32_t t = t0; t < t0 + n_steps; t++) {
        admit_phase(P, t, gtid, gsize);
        if (!grid_barrier(P.ctr, gen, &sm.flag)) return;
        update_phase<W256>(P, t, sm);
        if (!grid_barrier(P.ctr, gen, &sm.flag)) return;
        cross_phase(P, t);
        if (!grid_barrier(P.ctr, gen, &sm.flag)) return;
    }
    flush_stats(P, sm);
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
        const uint32_t out_base = row_ptr[er.z], d = row_ptr[er.z + 1u] - out_base;
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
// Pre-placed vehicles (R1, last sentence): vehicle i of the list goes to segment i % n_seg; fill S1 from the route
// store, mark atlas_0, count the entry.
__global__ void k_place_initial(const DevP P, const uint4 *init, uint32_t n_init)
{
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_init; i += gridDim.x * blockDim.x) {
        const uint4 s0v = init[i];
        const uint4 rr = P.route[s0v.w];
        const size_t at = (size_t)(i % P.n_seg) * P.seg_cap + i / P.n_seg;
        P.S0[0][at] = s0v;
        P.S1[0][at] = make_uint4(rr.x, rr.y & GEOM_STATIC_MASK, CELL_NONE, rr.w);  // lane 0, tag 0, no earlier mark
        const uint32_t cell = rr.x + (s0v.x >> 10);
        mark_toggle(P.bits[0], cell);
        P.pay[0][cell] = make_uint2(s0v.x & 1023u, s0v.y);
        P.admit_step[s0v.z] = 0u;
        atomicAdd(&P.edge_entries[rr.z], 1u);
    }
}
// Readback: scatter the active segments into per-trip arrays (caller order).
__global__ void k_gather_state(const DevP P, int cur, const uint32_t *trip_of_id, uint8_t *status, uint32_t *route_pos,
                               uint8_t *lane, uint8_t *tag, uint32_t *x_fx, float *v, float *acc)
{
    for (uint32_t seg = blockIdx.x; seg < P.n_seg; seg += gridDim.x) {
        const uint32_t n = P.seg_cnt[cur][seg];
        const size_t seg_base = (size_t)seg * P.seg_cap;
        for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
            const uint4 s0v = P.S0[cur][seg_base + i];
            const uint4 s1v = P.S1[cur][seg_base + i];
            const uint32_t tr = trip_of_id[s0v.z];
            status[tr] = 1u;
            route_pos[tr] = s0v.w - P.route_start[s0v.z];
            lane[tr] = (uint8_t)GEOM_LANE(s1v.y);
            tag[tr] = (uint8_t)GEOM_TAG(s1v.y);
            x_fx[tr] = s0v.x;
            v[tr] = __uint_as_float(s0v.y);
            acc[tr] = P.acc[cur] ? P.acc[cur][seg_base + i] : 0.0f;
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
__global__ void k_export_atlas(const u64 *B, const uint2 *pay, uint64_t n_cells, uint16_t *occ, float *spd)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_cells; i += (uint64_t)gridDim.x * blockDim.x) {
        const bool on = (B[i >> 6] >> (i & 63ull)) & 1ull;
        const uint2 pc = on ? pay[i] : make_uint2(0u, 0u);
        occ[i] = on ? (uint16_t)(1u + pc.x) : (uint16_t)0u;
        spd[i] = on ? __uint_as_float(pc.y) : 0.0f;
    }
}

}  // namespace manta
