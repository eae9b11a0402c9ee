// manta_kernels.cuh -- the three phases of one MANTA timestep as device functions, plus their kernels.
//
//   P0 admit   (R1)      : one thread per origin-edge FIFO; releases the head trip if its entry window is free
//   P1 update  (R2-R8)   : one thread per active vehicle; reads atlas_t, writes the tentative next state N and
//                          min-id claims for edge / node crossings
//   P2 commit  (R8, R9)  : resolves claims, clears atlas_t marks, writes atlas_{t+1}, compacts the active array
//
// A grid-wide barrier separates the phases (kernel boundaries, or the software barrier of k_persistent).
#pragma once
#include "manta_device.cuh"

namespace manta {

struct Lead {
    bool found;
    int32_t lead_abs;   // leader position in the follower's frame, Q22.10 (R2)
    float v_lead;
};

// ------------------------------------------------------------------------------------------------ R2 (scalar)
// Leader search along the own lane and on along the route ("looking up the status of neighboring
// cells"; G16).  Per-thread version: 16-byte loads, early exit.
__device__ __forceinline__ Lead leader_scalar(const DevP &P, const uint16_t *occ, const float *spd, uint32_t cursor,
                                              uint32_t cell_off, uint32_t geom, uint32_t lane, uint32_t c,
                                              unsigned long long &examined)
{
    Lead L;
    L.found = false;
    L.lead_abs = 0;
    L.v_lead = 0.0f;
    uint32_t len = GEOM_LEN(geom);
    uint32_t row = cell_off + lane * pitch_of(len);
    uint32_t start = c + 1u, rem = P.H, dist_base = 0u, l = lane;
    bool last = GEOM_LAST(geom) != 0u;
    for (;;) {
        uint32_t end = min(len, start + rem);
        if (start < end) {
            uint32_t j, code;
            if (scan_fwd(occ, row, start, end, j, code)) {
                examined += (unsigned long long)(j - start + 1u);
                L.found = true;
                L.lead_abs = (int32_t)(((dist_base + j) << 10) | (code - 1u));
                L.v_lead = spd[(size_t)row + j];
                return L;
            }
            examined += (unsigned long long)(end - start);
            rem -= end - start;
        }
        if (rem == 0u || last) return L;
        cursor += 1u;
        uint4 rr = P.route[cursor];
        dist_base += len;
        len = GEOM_LEN(rr.y);
        l = min(l, GEOM_LANES(rr.y) - 1u);
        row = rr.x + l * pitch_of(len);
        start = 0u;
        last = GEOM_LAST(rr.y) != 0u;
    }
}

// ------------------------------------------------------------------------------------------------ R3-R8
// Per-vehicle context carried from the leader search to the end of the update.
struct Veh {
    int32_t x;
    float v, v0;
    uint32_t id, cursor, cell_off, geom, eid;
    uint32_t len_c, n, l, c, pitch;
    bool last;
    // after pre_lc
    float acc_cur;
    int32_t bound;
    uint32_t tag, lt;
    bool mand, disc_pre, need_lc;
};

__device__ __forceinline__ void veh_load(Veh &V, const uint4 &s0v, const uint4 &s1v)
{
    V.x = (int32_t)s0v.x;
    V.v = __uint_as_float(s0v.y);
    V.id = s0v.z;
    V.cursor = s0v.w;
    V.cell_off = s1v.x;
    V.geom = s1v.y;
    V.eid = s1v.z;
    V.v0 = __uint_as_float(s1v.w);
    V.len_c = GEOM_LEN(V.geom);
    V.n = GEOM_LANES(V.geom);
    V.l = GEOM_LANE(V.geom);
    V.last = GEOM_LAST(V.geom) != 0u;
    V.c = (uint32_t)V.x >> 10;
    V.pitch = pitch_of(V.len_c);
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
// (has_a, ja, ca, v_a) / (has_b, jb, cb, v_b): lead / lag found in the target lane (cell index, cell code, speed);
// ignored unless V.need_lc.
__device__ __forceinline__ void post_lc(const DevP &P, uint32_t t, const Veh &V, uint32_t slot, bool has_a, uint32_t ja,
                                        uint32_t ca, float v_a, bool has_b, uint32_t jb, uint32_t cb, float v_b,
                                        float *acc_out, unsigned long long &n_lc)
{
    const int32_t x = V.x;
    const float v = V.v;
    uint32_t l_new = V.l;
    float acc = V.acc_cur;
    int32_t bound = V.bound;
    if (V.need_lc) {
        int32_t x_a = 0, x_b = 0;
        float gap_lead = 0.0f, gap_lag = 0.0f;
        if (has_a) {
            x_a = (int32_t)((ja << 10) | (ca - 1u));
            float gf = (float)(x_a - x);
            gf = gf * 0.0009765625f;
            gap_lead = gf - P.veh_len;
        }
        if (has_b) {
            x_b = (int32_t)((jb << 10) | (cb - 1u));
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
    if (acc_out) acc_out[slot] = acc;
    // R8
    const int32_t len_fx = (int32_t)(V.len_c << 10);
    uint32_t kind, word = 0u, nx;
    if (xn < len_fx) {
        kind = KIND_STAY;
        nx = (uint32_t)xn;
    } else if (V.last) {
        kind = KIND_DONE;  // G18
        nx = 0u;
    } else {
        const uint4 rn = P.route[V.cursor + 1u];
        const uint32_t lplus = min(l_new, GEOM_LANES(rn.y) - 1u);
        word = GEOM_PRIO(V.geom) ? (P.n_edges * 8u + P.head[V.eid])  // PRIORITY: the node
                                 : (rn.z * 8u + lplus);              // GREEN: the lane entry
        kind = KIND_CAND;
        nx = (uint32_t)(xn - len_fx);
        // smallest id wins; the key carries ~t in the high word so claim words never need a reset
        const unsigned long long key = ((unsigned long long)(0xFFFFFFFFu - t) << 32) | (unsigned long long)V.id;
        atomicMin(&P.claim[word], key);
    }
    P.N[slot] = make_uint4(nx, __float_as_uint(vn), kind | (l_new << 2) | (V.tag << 5), word);
}

// Scalar version of the whole update of one vehicle (MANTA_FLAG_SCALAR_SCAN, and the fallback of the cooperative
// path for vehicles whose window does not fit its chunk list).
__device__ __forceinline__ void lc_scans_scalar(const DevP &P, const uint16_t *occ, const float *spd, const Veh &V,
                                                bool &has_a, uint32_t &ja, uint32_t &ca, float &v_a, bool &has_b,
                                                uint32_t &jb, uint32_t &cb, float &v_b)
{
    // R5: lead / lag in the target lane
    const uint32_t rowt = V.cell_off + V.lt * V.pitch;
    has_a = scan_fwd(occ, rowt, V.c, min(V.len_c, V.c + P.H), ja, ca);
    has_b = scan_bwd(occ, rowt, V.c > P.lookback ? V.c - P.lookback : 0u, V.c, jb, cb);
    v_a = has_a ? spd[(size_t)rowt + ja] : 0.0f;
    v_b = has_b ? spd[(size_t)rowt + jb] : 0.0f;
}

// ------------------------------------------------------------------------------------------------ R2/R5 cooperative
// Warp-cooperative look-ahead.  Each lane owns one vehicle and writes the atlas windows it has to search as a list
// of CHUNKS (64 cells = 128 bytes = one cache line, 8-cell aligned inside its row) into the warp's shared-memory
// scratch.  The warp then serves the lists in rounds: in round r, the four 8-lane groups each issue chunk r of up
// to eight owners as one 16-byte load per lane (8 independent, fully coalesced 128-byte requests in flight per
// lane), then find the first (or last) occupied cell with ballot + ffs.  Lanes outside a chunk's valid range are
// predicated off, so no sector outside the window is fetched.
#define MANTA_MAXCH 12
#define MANTA_CH_STRIDE 13
struct WarpScratch {
    uint2 ch[32 * MANTA_CH_STRIDE];  // chunk lists: x = absolute cell index of the chunk, y = rel | lo << 10 | hi << 16
    uint2 res[32];                   // per owner: x = absolute cell index of the hit, y = rel_dist << 16 | cell code
    uint32_t nch[32];
};

// chunks of cells [start, end) of the row at absolute cell `row`, ascending.  `bias` = (distance in cells from the
// owner's reference to the row's cell 0) so that rel = bias + base.  Returns the new list length (ovf on overflow).
__device__ __forceinline__ uint32_t emit_fwd(uint2 *list, uint32_t k, uint32_t row, uint32_t start, uint32_t end, int bias,
                                             bool &ovf)
{
    for (uint32_t base = start & ~7u; base < end; base += 64u) {
        if (k >= MANTA_MAXCH) {
            ovf = true;
            return k;
        }
        const uint32_t lo = start > base ? start - base : 0u;
        const uint32_t hi = min(end - base, 64u);
        list[k++] = make_uint2(row + base, (uint32_t)(bias + (int)base) | (lo << 10) | (hi << 16));
    }
    return k;
}
// chunks of cells [start, end) descending (nearest first) for the backward (lag) search; rel = c - base
__device__ __forceinline__ uint32_t emit_bwd(uint2 *list, uint32_t k, uint32_t row, uint32_t start, uint32_t end, uint32_t c,
                                             bool &ovf)
{
    if (end <= start) return k;
    for (int base = (int)((end - 1u) & ~63u) ; base + 64 > (int)start; base -= 64) {
        if (k >= MANTA_MAXCH) {
            ovf = true;
            return k;
        }
        const uint32_t b = (uint32_t)base;
        const uint32_t lo = (int)start > base ? start - b : 0u;
        const uint32_t hi = min(end - b, 64u);
        list[k++] = make_uint2(row + b, (c - b) | (lo << 10) | (hi << 16));
    }
    return k;
}

template <bool BACKWARD>
__device__ __forceinline__ void coop_scan(const uint16_t *occ, WarpScratch &ws, uint32_t lane)
{
    const uint32_t q = lane >> 3, j = lane & 7u, my = j * 8u;
    uint32_t pend = 0u, maxr = 0u;
#pragma unroll
    for (uint32_t p = 0; p < 8u; p++) {
        const uint32_t nc = ws.nch[p * 4u + q];
        if (nc) pend |= 1u << p;
        maxr = max(maxr, nc);
    }
    maxr = __reduce_max_sync(0xFFFFFFFFu, maxr);
    for (uint32_t r = 0; r < maxr; r++) {
        if (!__any_sync(0xFFFFFFFFu, pend != 0u)) break;
        uint4 w[8];
#pragma unroll
        for (uint32_t p = 0; p < 8u; p++) {
            const uint32_t o = p * 4u + q;
            w[p] = make_uint4(0u, 0u, 0u, 0u);
            if (((pend >> p) & 1u) && r < ws.nch[o]) {
                const uint2 d = ws.ch[o * MANTA_CH_STRIDE + r];
                const uint32_t lo = (d.y >> 10) & 63u, hi = (d.y >> 16) & 127u;
                if (my + 8u > lo && my < hi) w[p] = *reinterpret_cast<const uint4 *>(occ + (size_t)d.x + my);
            }
        }
#pragma unroll
        for (uint32_t p = 0; p < 8u; p++) {
            const uint32_t o = p * 4u + q;
            uint32_t m = nzmask8(w[p]);
            uint2 d = make_uint2(0u, 0u);
            if (m) {
                d = ws.ch[o * MANTA_CH_STRIDE + r];
                const uint32_t lo = (d.y >> 10) & 63u, hi = (d.y >> 16) & 127u;
                if (lo > my) m &= 0xFFu << (lo - my);
                if (hi < my + 8u) m &= (1u << (hi - my)) - 1u;
            }
            const uint32_t bal = __ballot_sync(0xFFFFFFFFu, m != 0u);
            const uint32_t gb = (bal >> (q * 8u)) & 0xFFu;
            if (gb) {
                const uint32_t jj = BACKWARD ? (31u - (uint32_t)__clz((int)gb)) : ((uint32_t)__ffs((int)gb) - 1u);
                if (j == jj) {
                    const uint32_t i = BACKWARD ? (31u - (uint32_t)__clz((int)m)) : ((uint32_t)__ffs((int)m) - 1u);
                    const uint32_t off = my + i, rel = d.y & 1023u;
                    ws.res[o] = make_uint2(d.x + off, ((BACKWARD ? rel - off : rel + off) << 16) | code_at(w[p], i));
                }
                pend &= ~(1u << p);
            } else if (((pend >> p) & 1u) && r + 1u >= ws.nch[o]) {
                pend &= ~(1u << p);
            }
        }
    }
    __syncwarp();
}

// ------------------------------------------------------------------------------------------------ P0: R1
// Departure admission (G17, G25).  Thread k owns the FIFO of origin edge q_edge[k]; trips in it are
// in vehicle-id (= departure) order, so the head is the smallest waiting id on that edge.
__device__ __forceinline__ void admit_phase(const DevP &P, uint32_t t, uint32_t gtid, uint32_t gsize)
{
    const int cur = (int)(t & 1u);
    uint16_t *occ = P.occ[cur];
    float *spd = P.spd[cur];
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
            uint32_t j, code;
            if (scan_fwd(occ, row, 0u, P.L_c + 1u, j, code)) continue;   // window [0, L_c] not free
            const uint32_t slot = atomicAdd(&P.ctr->n_act[cur], 1u);
            const uint32_t cursor = P.route_start[id];
            uint4 rr = P.route[cursor];
            rr.y = (rr.y & GEOM_STATIC_MASK) | (l << 28);
            P.A0[cur][slot] = make_uint4(0u, 0u, id, cursor);
            P.A1[cur][slot] = rr;
            occ[(size_t)row] = 1u;          // frac10 = 0
            spd[(size_t)row] = 0.0f;
            P.admit_step[id] = t;
            atomicAdd(&P.edge_entries[e], 1u);
            P.q_head[k] = h + 1u;
            break;
        }
    }
}

// ------------------------------------------------------------------------------------------------ P1: R2-R8
// Scalar variant: one thread does everything for its vehicle (A/B baseline, MANTA_FLAG_SCALAR_SCAN).
__device__ __forceinline__ void update_phase_scalar(const DevP &P, uint32_t t, uint32_t gtid, uint32_t gsize,
                                                    unsigned long long &n_lc, unsigned long long &n_cells,
                                                    unsigned long long &n_eval)
{
    const int cur = (int)(t & 1u);
    const uint16_t *occ = P.occ[cur];
    const float *spd = P.spd[cur];
    const uint32_t n = P.ctr->n_act[cur];
    float *acc_out = P.acc[cur];
    for (uint32_t i = gtid; i < n; i += gsize) {
        Veh V;
        veh_load(V, P.A0[cur][i], P.A1[cur][i]);
        const Lead ld = leader_scalar(P, occ, spd, V.cursor, V.cell_off, V.geom, V.l, V.c, n_cells);
        pre_lc(P, t, V, ld);
        bool has_a = false, has_b = false;
        uint32_t ja = 0, ca = 0, jb = 0, cb = 0;
        float v_a = 0.0f, v_b = 0.0f;
        if (V.need_lc) {
            n_eval += 1ull;
            lc_scans_scalar(P, occ, spd, V, has_a, ja, ca, v_a, has_b, jb, cb, v_b);
        }
        post_lc(P, t, V, i, has_a, ja, ca, v_a, has_b, jb, cb, v_b, acc_out, n_lc);
    }
}

// Warp-cooperative variant (default): lane = vehicle; the atlas windows of the 32 vehicles of a warp are searched
// by coop_scan.  Must be entered by whole warps.
__device__ __forceinline__ void update_phase_coop(const DevP &P, uint32_t t, WarpScratch &ws, uint32_t warp_gid,
                                                  uint32_t n_warps_total, unsigned long long &n_lc,
                                                  unsigned long long &n_cells, unsigned long long &n_eval)
{
    const int cur = (int)(t & 1u);
    const uint16_t *occ = P.occ[cur];
    const float *spd = P.spd[cur];
    const uint32_t n = P.ctr->n_act[cur];
    float *acc_out = P.acc[cur];
    const uint32_t lane = threadIdx.x & 31u;
    uint2 *mylist = &ws.ch[lane * MANTA_CH_STRIDE];
    for (uint32_t base = warp_gid * 32u; base < n; base += n_warps_total * 32u) {
        const uint32_t i = base + lane;
        const bool valid = i < n;
        Veh V;
        Lead ld;
        ld.found = false;
        ld.lead_abs = 0;
        ld.v_lead = 0.0f;
        bool ovf = false;
        uint32_t k = 0u, win_total = 0u;
        V.need_lc = false;
        if (valid) {
            veh_load(V, P.A0[cur][i], P.A1[cur][i]);
            // R2: the look-ahead window as chunk list: own row from c+1, then on along the route
            uint32_t len = V.len_c, row = V.cell_off + V.l * V.pitch, start = V.c + 1u, rem = P.H, dist0 = 0u, l = V.l;
            uint32_t cursor = V.cursor;
            bool last = V.last;
            for (;;) {
                const uint32_t end = min(len, start + rem);
                if (start < end) {
                    k = emit_fwd(mylist, k, row, start, end, (int)dist0 - (int)V.c + 8, ovf);
                    win_total += end - start;
                    rem -= end - start;
                }
                if (ovf || rem == 0u || last) break;
                cursor += 1u;
                const uint4 rr = P.route[cursor];
                dist0 += len;
                len = GEOM_LEN(rr.y);
                l = min(l, GEOM_LANES(rr.y) - 1u);
                row = rr.x + l * pitch_of(len);
                start = 0u;
                last = GEOM_LAST(rr.y) != 0u;
            }
        }
        ws.nch[lane] = (valid && !ovf) ? k : 0u;
        ws.res[lane] = make_uint2(0u, 0u);
        __syncwarp();
        coop_scan<false>(occ, ws, lane);
        if (valid) {
            if (ovf) {
                ld = leader_scalar(P, occ, spd, V.cursor, V.cell_off, V.geom, V.l, V.c, n_cells);
            } else {
                const uint2 r = ws.res[lane];
                if (r.y & 0xFFFFu) {
                    const uint32_t dist = V.c + (r.y >> 16) - 8u;   // cells from the own edge's tail to the leader
                    ld.found = true;
                    ld.lead_abs = (int32_t)((dist << 10) | ((r.y & 0xFFFFu) - 1u));
                    ld.v_lead = spd[r.x];
                    n_cells += (unsigned long long)(dist - V.c);
                } else {
                    n_cells += (unsigned long long)win_total;
                }
            }
            pre_lc(P, t, V, ld);
        }
        const bool need = valid && V.need_lc;
        bool has_a = false, has_b = false;
        uint32_t ja = 0, ca = 0, jb = 0, cb = 0;
        float v_a = 0.0f, v_b = 0.0f;
        if (__any_sync(0xFFFFFFFFu, need)) {
            // R5: lead (forward from c) and lag (backward from c-1) in the target lane, same machinery
            const uint32_t rowt = V.cell_off + V.lt * V.pitch;
            bool ovf2 = false;
            k = 0u;
            if (need) k = emit_fwd(mylist, 0u, rowt, V.c, min(V.len_c, V.c + P.H), 8 - (int)V.c, ovf2);
            ws.nch[lane] = (need && !ovf2) ? k : 0u;
            ws.res[lane] = make_uint2(0u, 0u);
            __syncwarp();
            coop_scan<false>(occ, ws, lane);
            if (need && !ovf2) {
                const uint2 r = ws.res[lane];
                if (r.y & 0xFFFFu) {
                    has_a = true;
                    ja = V.c + (r.y >> 16) - 8u;
                    ca = r.y & 0xFFFFu;
                    v_a = spd[r.x];
                }
            }
            k = 0u;
            if (need) k = emit_bwd(mylist, 0u, rowt, V.c > P.lookback ? V.c - P.lookback : 0u, V.c, V.c, ovf2);
            ws.nch[lane] = (need && !ovf2) ? k : 0u;
            ws.res[lane] = make_uint2(0u, 0u);
            __syncwarp();
            coop_scan<true>(occ, ws, lane);
            if (need && !ovf2) {
                const uint2 r = ws.res[lane];
                if (r.y & 0xFFFFu) {
                    has_b = true;
                    jb = V.c - (r.y >> 16);
                    cb = r.y & 0xFFFFu;
                    v_b = spd[r.x];
                }
            }
            if (need && ovf2) lc_scans_scalar(P, occ, spd, V, has_a, ja, ca, v_a, has_b, jb, cb, v_b);
        }
        if (valid) {
            if (need) n_eval += 1ull;
            post_lc(P, t, V, i, has_a, ja, ca, v_a, has_b, jb, cb, v_b, acc_out, n_lc);
        }
    }
}

// ------------------------------------------------------------------------------------------------ P2: R8, R9
// Claim resolution, atlas clear / write, compaction (warp ballot + block prefix sum, one atomic per block).
// Must be called by ALL threads of the block (contains __syncthreads).
__device__ __forceinline__ void commit_phase(const DevP &P, uint32_t t, uint32_t *s_warp /*[33]*/)
{
    const int cur = (int)(t & 1u), nxt = cur ^ 1;
    uint16_t *occ_c = P.occ[cur];
    uint16_t *occ_n = P.occ[nxt];
    float *spd_n = P.spd[nxt];
    const uint32_t n = P.ctr->n_act[cur];
    const uint32_t lane_id = threadIdx.x & 31u, warp_id = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
    const uint32_t gsize = gridDim.x * blockDim.x;
    for (uint32_t base = blockIdx.x * blockDim.x; base < n; base += gsize) {
        const uint32_t i = base + threadIdx.x;
        bool alive = false;
        uint4 o0 = make_uint4(0, 0, 0, 0), o1 = make_uint4(0, 0, 0, 0);
        float acc_v = 0.0f;
        if (i < n) {
            const uint4 s0v = P.A0[cur][i];
            const uint4 s1v = P.A1[cur][i];
            const uint4 nv = P.N[i];
            if (P.acc[cur]) acc_v = P.acc[cur][i];
            const uint32_t geom = s1v.y, len_c = GEOM_LEN(geom);
            const uint32_t id = s0v.z;
            // clear the time-t mark (atlas_t becomes the write buffer of step t+1)
            occ_c[(size_t)s1v.x + GEOM_LANE(geom) * pitch_of(len_c) + (s0v.x >> 10)] = 0u;
            const uint32_t kind = nv.z & 3u, l_new = (nv.z >> 2) & 7u, tag = (nv.z >> 5) & 1u;
            if (kind == KIND_STAY) {
                alive = true;
                o0 = make_uint4(nv.x, nv.y, id, s0v.w);
                o1 = make_uint4(s1v.x, (geom & GEOM_STATIC_MASK) | (l_new << 28) | (tag << 31), s1v.z, s1v.w);
            } else if (kind == KIND_DONE) {
                const uint32_t adm = P.admit_step[id];
                P.arrive_step[id] = t + 1u;
                atomicAdd(&P.ctr->n_done, 1ull);
                atomicAdd(&P.ctr->sum_travel, (unsigned long long)(t + 1u - adm));
            } else {
                alive = true;
                const unsigned long long key = ((unsigned long long)(0xFFFFFFFFu - t) << 32) | (unsigned long long)id;
                if (P.claim[nv.w] == key) {  // winner crosses
                    uint4 rn = P.route[s0v.w + 1u];
                    const uint32_t lplus = min(l_new, GEOM_LANES(rn.y) - 1u);
                    rn.y = (rn.y & GEOM_STATIC_MASK) | (lplus << 28);
                    o0 = make_uint4(nv.x, nv.y, id, s0v.w + 1u);
                    o1 = rn;
                    atomicAdd(&P.edge_entries[rn.z], 1u);
                } else {  // loser holds at the stop line (G15)
                    o0 = make_uint4((len_c << 10) - 1u, 0u, id, s0v.w);
                    o1 = make_uint4(s1v.x, (geom & GEOM_STATIC_MASK) | (l_new << 28) | (tag << 31), s1v.z, s1v.w);
                }
            }
            if (alive) {
                const size_t cell = (size_t)o1.x + GEOM_LANE(o1.y) * pitch_of(GEOM_LEN(o1.y)) + (o0.x >> 10);
                occ_n[cell] = (uint16_t)(1u + (o0.x & 1023u));
                spd_n[cell] = __uint_as_float(o0.y);
            }
        }
        // compaction
        const uint32_t bal = __ballot_sync(0xFFFFFFFFu, alive);
        if (lane_id == 0u) s_warp[warp_id] = __popc(bal);
        __syncthreads();
        if (warp_id == 0u) {
            uint32_t cnt = lane_id < n_warps ? s_warp[lane_id] : 0u;
            uint32_t incl = cnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                uint32_t y = __shfl_up_sync(0xFFFFFFFFu, incl, d);
                if ((int)lane_id >= d) incl += y;
            }
            const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
            uint32_t gbase = 0u;
            if (lane_id == 0u && total) gbase = atomicAdd(&P.ctr->n_act[nxt], total);
            gbase = __shfl_sync(0xFFFFFFFFu, gbase, 0);
            if (lane_id < n_warps) s_warp[lane_id] = gbase + incl - cnt;
        }
        __syncthreads();
        if (alive) {
            const uint32_t pos = s_warp[warp_id] + __popc(bal & ((1u << lane_id) - 1u));
            P.A0[nxt][pos] = o0;
            P.A1[nxt][pos] = o1;
            if (P.acc[nxt]) P.acc[nxt][pos] = acc_v;
        }
        __syncthreads();
    }
}

__device__ __forceinline__ void flush_stats(const DevP &P, unsigned long long n_lc, unsigned long long n_cells,
                                            unsigned long long n_eval, unsigned long long *s_stats /*[3]*/)
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
    if (gtid == 0u) P.ctr->n_act[(t & 1u) ^ 1u] = 0u;   // the buffer this step's commit will fill
    admit_phase(P, t, gtid, gridDim.x * blockDim.x);
}

__global__ void __launch_bounds__(256) k_update(const DevP P, uint32_t t)
{
    __shared__ unsigned long long s_stats[3];
    __shared__ WarpScratch s_ws[8];
    if (threadIdx.x < 3u) s_stats[threadIdx.x] = 0ull;
    __syncthreads();
    unsigned long long n_lc = 0ull, n_cells = 0ull, n_eval = 0ull;
    const uint32_t gtid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gtid == 0u) P.ctr->n_updates += (unsigned long long)P.ctr->n_act[t & 1u];
    if (P.flags & 1u)   // MANTA_FLAG_SCALAR_SCAN
        update_phase_scalar(P, t, gtid, gridDim.x * blockDim.x, n_lc, n_cells, n_eval);
    else
        update_phase_coop(P, t, s_ws[threadIdx.x >> 5], gtid >> 5, (gridDim.x * blockDim.x) >> 5, n_lc, n_cells, n_eval);
    flush_stats(P, n_lc, n_cells, n_eval, s_stats);
}

__global__ void __launch_bounds__(256) k_commit(const DevP P, uint32_t t)
{
    __shared__ uint32_t s_warp[33];
    commit_phase(P, t, s_warp);
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
// Pre-placed vehicles (R1, last sentence): fill A1 from the route store, mark atlas_0, count the entry.
__global__ void k_place_initial(const DevP P, uint32_t n_init)
{
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_init; i += gridDim.x * blockDim.x) {
        const uint4 s0v = P.A0[0][i];
        uint4 rr = P.route[s0v.w];
        rr.y = rr.y & GEOM_STATIC_MASK;  // lane 0, tag 0
        P.A1[0][i] = rr;
        const size_t cell = (size_t)rr.x + (s0v.x >> 10);
        P.occ[0][cell] = (uint16_t)(1u + (s0v.x & 1023u));
        P.spd[0][cell] = __uint_as_float(s0v.y);
        P.admit_step[s0v.z] = 0u;
        atomicAdd(&P.edge_entries[rr.z], 1u);
    }
}
// Readback: scatter the active array into per-trip arrays (caller order).
__global__ void k_gather_state(const DevP P, int cur, const uint32_t *trip_of_id, uint8_t *status, uint32_t *route_pos,
                               uint8_t *lane, uint8_t *tag, uint32_t *x_fx, float *v, float *acc)
{
    const uint32_t n = P.ctr->n_act[cur];
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const uint4 s0v = P.A0[cur][i];
        const uint4 s1v = P.A1[cur][i];
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

}  // namespace manta
