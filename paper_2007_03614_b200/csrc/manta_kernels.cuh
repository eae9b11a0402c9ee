// manta_kernels.cuh -- the three phases of one MANTA timestep as device functions, plus their kernels.
//
//   A admit   (R1)      : one thread per origin-edge FIFO; releases the head trip if its entry window is free
//   U update  (R2-R9)   : one thread per active vehicle; reads the time-t atlas, and for the vehicles that stay on
//                         their edge (the great majority) finishes the step: next state to the compacted next
//                         buffer, time-(t+1) mark, clearing of the time-(t-1) mark.  Edge-end candidates post a
//                         min-id claim and an entry of the cross list; arrivals post an entry too.
//   X cross   (R8, R9)  : one thread per cross-list entry: resolves the claim (winner moves to its next route
//                         edge, loser holds at the stop line), writes its mark; clears the marks of arrivals.
//
// A grid-wide barrier separates the phases: the software barrier of k_persistent (one cooperative launch runs
// many timesteps), or kernel boundaries (k_admit / k_update / k_cross: MANTA_FLAG_MULTI_KERNEL, manta_step_timed).
#pragma once
#include "manta_device.cuh"

namespace manta {

#define MANTA_NT 512   // threads per block of the step kernels

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

// ------------------------------------------------------------------------------------------------ R2
// Leader search along the own lane and on along the route ("looking up the status of neighboring
// cells"; G16).  The next route record is requested before the current row's words are examined, so the chain of
// dependent loads is: state -> {own-row words, next record} -> next row's words -> leader payload.
__device__ __forceinline__ Lead leader_search(const DevP &P, const u64 *B, const uint2 *pay, const Veh &V, u64 &examined)
{
    Lead L;
    L.found = false;
    L.lead_abs = 0;
    L.v_lead = 0.0f;
    uint32_t len = V.len_c, row = V.cell_off + V.l * V.pitch, start = V.c + 1u, rem = P.H, dist_base = 0u, l = V.l;
    uint32_t cursor = V.cursor;
    bool last = V.last;
    uint4 rn = make_uint4(0u, 0u, 0u, 0u);
    if (!last) rn = P.route[cursor + 1u];
    for (;;) {
        const uint32_t end = min(len, start + rem);
        if (start < end) {
            uint32_t j;
            if (first_set(B, row, start, end, j)) {
                const uint2 pc = pay[(size_t)row + j];
                examined += (u64)(j - start + 1u);
                L.found = true;
                L.lead_abs = (int32_t)(((dist_base + j) << 10) | pc.x);
                L.v_lead = __uint_as_float(pc.y);
                return L;
            }
            examined += (u64)(end - start);
            rem -= end - start;
        }
        if (rem == 0u || last) return L;
        cursor += 1u;
        dist_base += len;
        len = GEOM_LEN(rn.y);
        l = min(l, GEOM_LANES(rn.y) - 1u);
        row = rn.x + l * pitch_of(len);
        start = 0u;
        last = GEOM_LAST(rn.y) != 0u;
        if (!last) rn = P.route[cursor + 1u];
    }
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
                                           bool has_b, int32_t x_b, float v_b, u64 &n_lc)
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
                n_lc += 1ull;
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
        const uint4 rn = P.route[V.cursor + 1u];
        const uint32_t lplus = min(l_new, GEOM_LANES(rn.y) - 1u);
        O.word = GEOM_PRIO(V.geom) ? (P.n_edges * 8u + P.head[P.route[V.cursor].z])  // PRIORITY: the node
                                   : (rn.z * 8u + lplus);                             // GREEN: the lane entry
        O.kind = KIND_CAND;
        O.nx = (uint32_t)(xn - len_fx);
        // smallest id wins; the key carries ~t in the high word so claim words never need a reset
        const u64 key = ((u64)(0xFFFFFFFFu - t) << 32) | (u64)V.id;
        atomicMin(&P.claim[O.word], key);
    }
    return O;
}

// The whole R2-R8 arithmetic of one vehicle (reads only the time-t atlas).
__device__ __forceinline__ Outcome update_vehicle(const DevP &P, uint32_t t, const u64 *B, const uint2 *pay, Veh &V, u64 &n_lc,
                                                  u64 &n_cells, u64 &n_eval)
{
    const Lead ld = leader_search(P, B, pay, V, n_cells);
    pre_lc(P, t, V, ld);
    bool has_a = false, has_b = false;
    int32_t x_a = 0, x_b = 0;
    float v_a = 0.0f, v_b = 0.0f;
    if (V.need_lc) {
        // R5: lead (first occupied cell >= c, within the edge) and lag (last occupied cell < c) in the target lane
        n_eval += 1ull;
        const uint32_t rowt = V.cell_off + V.lt * V.pitch;
        uint32_t ja = 0u, jb = 0u;
        has_a = first_set(B, rowt, V.c, min(V.len_c, V.c + P.H), ja);
        const uint32_t b0 = V.c > P.lookback ? V.c - P.lookback : 0u;
        has_b = V.c > b0 && last_set(B, rowt, b0, V.c, jb);
        if (has_a) {
            const uint2 pc = pay[(size_t)rowt + ja];
            x_a = (int32_t)((ja << 10) | pc.x);
            v_a = __uint_as_float(pc.y);
        }
        if (has_b) {
            const uint2 pc = pay[(size_t)rowt + jb];
            x_b = (int32_t)((jb << 10) | pc.x);
            v_b = __uint_as_float(pc.y);
        }
    }
    return post_lc(P, t, V, has_a, x_a, v_a, has_b, x_b, v_b, n_lc);
}

// ------------------------------------------------------------------------------------------------ A: R1
// Departure admission (G17, G25).  Thread k owns the FIFO of origin edge q_edge[k]; trips in it are
// in vehicle-id (= departure) order, so the head is the smallest waiting id on that edge.
__device__ __forceinline__ void admit_phase(const DevP &P, uint32_t t, uint32_t gtid, uint32_t gsize)
{
    const int cur = (int)(t & 1u);
    u64 *B = P.bits[t % 3u];
    uint2 *pay = P.pay[cur];
    const u64 window = bits_below(P.L_c + 1u);
    for (uint32_t k = gtid; k < P.n_queues; k += gsize) {
        const uint32_t h = P.q_head[k];
        if (h >= P.q_ptr[k + 1u]) continue;
        const uint32_t id = P.q_ids[h];
        if (P.depart_step[id] > t) continue;
        const uint32_t e = P.q_edge[k];
        const uint4 er = P.edge_tab[e];
        const uint32_t len = GEOM_LEN(er.y), lanes = GEOM_LANES(er.y), pitch = pitch_of(len);
        for (uint32_t l = 0; l < lanes; l++) {
            const uint32_t row = er.x + l * pitch;
            if (B[row >> 6] & window) continue;   // window [0, L_c] not free
            const uint32_t slot = (uint32_t)atomicAdd(&P.ctr->fill[cur], 1ull);
            const uint32_t cursor = P.route_start[id];
            const uint4 rr = P.route[cursor];
            P.S0[cur][slot] = make_uint4(0u, 0u, id, cursor);
            P.S1[cur][slot] = make_uint4(rr.x, (rr.y & GEOM_STATIC_MASK) | (l << 28), CELL_NONE, rr.w);
            if (P.acc[cur]) P.acc[cur][slot] = 0.0f;
            mark_set(B, row);                    // cell 0, frac10 = 0, v = 0: visible to this step's update
            pay[(size_t)row] = make_uint2(0u, 0u);
            P.admit_step[id] = t;
            atomicAdd(&P.edge_entries[e], 1u);
            P.q_head[k] = h + 1u;
            break;
        }
    }
}

// ------------------------------------------------------------------------------------------------ U: R2-R9
// Must be called by ALL threads of the block (contains __syncthreads).  s_scan: 2 * 32 + 2 words of shared memory.
__device__ __forceinline__ void update_phase(const DevP &P, uint32_t t, uint32_t *s_scan, u64 &n_lc, u64 &n_cells, u64 &n_eval)
{
    const int cur = (int)(t & 1u), nxt = cur ^ 1;
    const u64 *B = P.bits[t % 3u];
    u64 *Bn = P.bits[(t + 1u) % 3u];
    u64 *Bp = P.bits[(t + 2u) % 3u];
    const uint2 *pay = P.pay[cur];
    uint2 *payn = P.pay[nxt];
    const uint32_t n = (uint32_t)P.ctr->fill[cur];
    const uint32_t lane_id = threadIdx.x & 31u, warp_id = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
    const uint32_t gsize = gridDim.x * blockDim.x;
    for (uint32_t base = blockIdx.x * blockDim.x; base < n; base += gsize) {
        const uint32_t i = base + threadIdx.x;
        bool alive = false, listed = false;
        uint4 o0 = make_uint4(0, 0, 0, 0), o1 = make_uint4(0, 0, 0, 0);
        uint2 xl = make_uint2(0u, 0u);
        float acc_v = 0.0f;
        if (i < n) {
            Veh V;
            veh_load(V, P.S0[cur][i], P.S1[cur][i]);
            if (V.prev != CELL_NONE) mark_clear(Bp, V.prev);          // the time-(t-1) mark
            const uint32_t cur_abs = V.cell_off + V.l * V.pitch + V.c;
            const Outcome O = update_vehicle(P, t, B, pay, V, n_lc, n_cells, n_eval);
            acc_v = O.acc;
            const uint32_t geom_n = (V.geom & GEOM_STATIC_MASK) | (O.l_new << 28) | (V.tag << 31);
            if (O.kind == KIND_STAY) {
                alive = true;
                const uint32_t cell = V.cell_off + O.l_new * V.pitch + (O.nx >> 10);
                mark_set(Bn, cell);                                    // R9: the time-(t+1) mark
                payn[cell] = make_uint2(O.nx & 1023u, __float_as_uint(O.vn));
                o0 = make_uint4(O.nx, __float_as_uint(O.vn), V.id, V.cursor);
                o1 = make_uint4(V.cell_off, geom_n, cur_abs, __float_as_uint(V.v0));
            } else if (O.kind == KIND_DONE) {
                listed = true;
                xl = make_uint2(XL_DONE, cur_abs);
                P.arrive_step[V.id] = t + 1u;
                atomicAdd(&P.ctr->n_done, 1ull);
                atomicAdd(&P.ctr->sum_travel, (u64)(t + 1u - P.admit_step[V.id]));
            } else {  // candidate: tentative winner state; the cross phase decides
                alive = true;
                listed = true;
                xl.y = O.word;
                o0 = make_uint4(O.nx, __float_as_uint(O.vn), V.id, V.cursor);
                o1 = make_uint4(V.cell_off, geom_n, cur_abs, __float_as_uint(V.v0));
            }
        }
        // compaction of the survivors and of the cross list: warp ballots + block prefix sum, one atomic per block
        const uint32_t bal_a = __ballot_sync(0xFFFFFFFFu, alive), bal_x = __ballot_sync(0xFFFFFFFFu, listed);
        if (lane_id == 0u) {
            s_scan[warp_id] = __popc(bal_a);
            s_scan[32u + warp_id] = __popc(bal_x);
        }
        __syncthreads();
        if (warp_id == 0u) {
            const uint32_t ca = lane_id < n_warps ? s_scan[lane_id] : 0u, cx = lane_id < n_warps ? s_scan[32u + lane_id] : 0u;
            uint32_t ia = ca, ix = cx;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t ya = __shfl_up_sync(0xFFFFFFFFu, ia, d), yx = __shfl_up_sync(0xFFFFFFFFu, ix, d);
                if ((int)lane_id >= d) {
                    ia += ya;
                    ix += yx;
                }
            }
            const uint32_t ta = __shfl_sync(0xFFFFFFFFu, ia, 31), tx = __shfl_sync(0xFFFFFFFFu, ix, 31);
            u64 g = 0ull;
            if (lane_id == 0u && (ta | tx)) g = atomicAdd(&P.ctr->fill[nxt], (u64)ta | ((u64)tx << 32));
            g = __shfl_sync(0xFFFFFFFFu, g, 0);
            if (lane_id < n_warps) {
                s_scan[lane_id] = (uint32_t)g + ia - ca;
                s_scan[32u + lane_id] = (uint32_t)(g >> 32) + ix - cx;
            }
        }
        __syncthreads();
        if (alive) {
            const uint32_t pos = s_scan[warp_id] + __popc(bal_a & ((1u << lane_id) - 1u));
            P.S0[nxt][pos] = o0;
            P.S1[nxt][pos] = o1;
            if (P.acc[nxt]) P.acc[nxt][pos] = acc_v;
            xl.x = pos;
        }
        if (listed) P.xlist[s_scan[32u + warp_id] + __popc(bal_x & ((1u << lane_id) - 1u))] = xl;
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------ X: R8, R9
__device__ __forceinline__ void cross_phase(const DevP &P, uint32_t t, uint32_t gtid, uint32_t gsize)
{
    const int nxt = (int)((t & 1u) ^ 1u);
    u64 *Bc = P.bits[t % 3u];
    u64 *Bn = P.bits[(t + 1u) % 3u];
    uint2 *payn = P.pay[nxt];
    const uint32_t n = (uint32_t)(P.ctr->fill[nxt] >> 32);
    for (uint32_t k = gtid; k < n; k += gsize) {
        const uint2 xl = P.xlist[k];
        if (xl.x == XL_DONE) {
            mark_clear(Bc, xl.y);     // an arrival leaves no time-(t+1) state to clear its time-t mark later
            continue;
        }
        uint4 s0 = P.S0[nxt][xl.x];
        uint4 s1 = P.S1[nxt][xl.x];
        const u64 key = ((u64)(0xFFFFFFFFu - t) << 32) | (u64)s0.z;
        if (P.claim[xl.y] == key) {   // winner crosses (R8)
            const uint4 rn = P.route[s0.w + 1u];
            const uint32_t lplus = min(GEOM_LANE(s1.y), GEOM_LANES(rn.y) - 1u);
            s0.w += 1u;
            s1 = make_uint4(rn.x, (rn.y & GEOM_STATIC_MASK) | (lplus << 28), s1.z, rn.w);
            atomicAdd(&P.edge_entries[rn.z], 1u);
        } else {                      // loser holds at the stop line (G15)
            s0.x = (GEOM_LEN(s1.y) << 10) - 1u;
            s0.y = 0u;
        }
        P.S0[nxt][xl.x] = s0;
        P.S1[nxt][xl.x] = s1;
        const uint32_t cell = s1.x + GEOM_LANE(s1.y) * pitch_of(GEOM_LEN(s1.y)) + (s0.x >> 10);
        mark_set(Bn, cell);
        payn[cell] = make_uint2(s0.x & 1023u, s0.y);
    }
}

__device__ __forceinline__ void flush_stats(const DevP &P, u64 n_lc, u64 n_cells, u64 n_eval, u64 *s_stats /*[3]*/)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        n_lc += __shfl_down_sync(0xFFFFFFFFu, n_lc, d);
        n_cells += __shfl_down_sync(0xFFFFFFFFu, n_cells, d);
        n_eval += __shfl_down_sync(0xFFFFFFFFu, n_eval, d);
    }
    if ((threadIdx.x & 31u) == 0u) {
        if (n_lc) atomicAdd(&s_stats[0], n_lc);
        if (n_cells) atomicAdd(&s_stats[1], n_cells);
        if (n_eval) atomicAdd(&s_stats[2], n_eval);
    }
    __syncthreads();
    if (threadIdx.x == 0u) {
        BlockStats *b = &P.blk[blockIdx.x];
        b->lane_changes += s_stats[0];
        b->cells_examined += s_stats[1];
        b->lc_evals += s_stats[2];
    }
}

// ------------------------------------------------------------------------------------------------ kernels
__global__ void __launch_bounds__(256) k_admit(const DevP P, uint32_t t)
{
    const uint32_t gtid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gtid == 0u) P.ctr->fill[(t & 1u) ^ 1u] = 0ull;   // the buffer (and cross list) this step's update will fill
    admit_phase(P, t, gtid, gridDim.x * blockDim.x);
}

__global__ void __launch_bounds__(MANTA_NT, 2) k_update(const DevP P, uint32_t t)
{
    __shared__ u64 s_stats[3];
    __shared__ uint32_t s_scan[64];
    if (threadIdx.x < 3u) s_stats[threadIdx.x] = 0ull;
    __syncthreads();
    u64 n_lc = 0ull, n_cells = 0ull, n_eval = 0ull;
    if (blockIdx.x == 0u && threadIdx.x == 0u) P.ctr->n_updates += P.ctr->fill[t & 1u] & 0xFFFFFFFFull;
    update_phase(P, t, s_scan, n_lc, n_cells, n_eval);
    flush_stats(P, n_lc, n_cells, n_eval, s_stats);
}

__global__ void __launch_bounds__(256) k_cross(const DevP P, uint32_t t)
{
    cross_phase(P, t, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}

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
__global__ void __launch_bounds__(MANTA_NT, 2) k_persistent(const DevP P, uint32_t t0, uint32_t n_steps)
{
    __shared__ u64 s_stats[3];
    __shared__ uint32_t s_scan[64];
    __shared__ uint32_t s_flag;
    if (threadIdx.x < 3u) s_stats[threadIdx.x] = 0ull;
    u64 n_lc = 0ull, n_cells = 0ull, n_eval = 0ull;
    unsigned gen = 0u;
    const uint32_t gtid = blockIdx.x * blockDim.x + threadIdx.x, gsize = gridDim.x * blockDim.x;
    for (uint32_t t = t0; t < t0 + n_steps; t++) {
        if (gtid == 0u) P.ctr->fill[(t & 1u) ^ 1u] = 0ull;
        admit_phase(P, t, gtid, gsize);
        if (!grid_barrier(P.ctr, gen, &s_flag)) return;
        if (gtid == 0u) P.ctr->n_updates += P.ctr->fill[t & 1u] & 0xFFFFFFFFull;
        update_phase(P, t, s_scan, n_lc, n_cells, n_eval);
        if (!grid_barrier(P.ctr, gen, &s_flag)) return;
        cross_phase(P, t, gtid, gsize);
        if (!grid_barrier(P.ctr, gen, &s_flag)) return;
    }
    flush_stats(P, n_lc, n_cells, n_eval, s_stats);
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
// Pre-placed vehicles (R1, last sentence): fill S1 from the route store, mark atlas_0, count the entry.
__global__ void k_place_initial(const DevP P, uint32_t n_init)
{
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_init; i += gridDim.x * blockDim.x) {
        const uint4 s0v = P.S0[0][i];
        const uint4 rr = P.route[s0v.w];
        P.S1[0][i] = make_uint4(rr.x, rr.y & GEOM_STATIC_MASK, CELL_NONE, rr.w);  // lane 0, tag 0, no earlier mark
        const uint32_t cell = rr.x + (s0v.x >> 10);
        mark_set(P.bits[0], cell);
        P.pay[0][cell] = make_uint2(s0v.x & 1023u, s0v.y);
        P.admit_step[s0v.z] = 0u;
        atomicAdd(&P.edge_entries[rr.z], 1u);
    }
}
// Readback: scatter the active array into per-trip arrays (caller order).
__global__ void k_gather_state(const DevP P, int cur, const uint32_t *trip_of_id, uint8_t *status, uint32_t *route_pos,
                               uint8_t *lane, uint8_t *tag, uint32_t *x_fx, float *v, float *acc)
{
    const uint32_t n = (uint32_t)P.ctr->fill[cur];
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const uint4 s0v = P.S0[cur][i];
        const uint4 s1v = P.S1[cur][i];
        const uint32_t tr = trip_of_id[s0v.z];
        status[tr] = 1u;
        route_pos[tr] = s0v.w - P.route_start[s0v.z];
        lane[tr] = (uint8_t)GEOM_LANE(s1v.y);
        tag[tr] = (uint8_t)GEOM_TAG(s1v.y);
        x_fx[tr] = s0v.x;
        v[tr] = __uint_as_float(s0v.y);
        acc[tr] = P.acc[cur] ? P.acc[cur][i] : 0.0f;
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
