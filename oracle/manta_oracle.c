/*
 * oracle/manta_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain single-threaded CPU microsimulator of MANTA's vehicle update
 * (arxiv 2007.03614).  One function per rule of DESIGN.md ("Rules" R0..R9),
 * written in the order of the rule text, no blocking / fusion / reordering.
 * Each function cites the PAPER.md passage it follows.  fp32 arithmetic is
 * IEEE op-by-op: build with  gcc -O2 -ffp-contract=off -fno-fast-math  (x86-64 SSE).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): K1..K12 of DESIGN.md -- closed forms of
 * Eq. (1), invariants, brute force on 2-3 vehicle intersections, reduction to a
 * textbook IDM loop.  Paper-level outputs (mean speeds by limit, Bay-Bridge volume):
 * parity unpinned (they need the real network / demand / calibrated parameters,
 * PAPER.md:115, 160, 198-204).
 *
 * Shares nothing with paper_2007_03614_b200/csrc.
 */
#include "manta_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define NONE32 0xFFFFFFFFu
#define NONE64 0xFFFFFFFFFFFFFFFFull
#define BOUND_INF 0x7FFFFFFF

struct mo_sim {
    /* network (lanes, length, free-flow speed per edge) */
    uint32_t n_nodes, n_edges;
    uint32_t *row_ptr, *head, *tail, *len_c;
    uint32_t *in_idx, *indeg; /* STOP nodes (R8s): index of an edge among its head node's inbound edges; in-degree */
    uint8_t *lanes, *ctrl;
    float *limit;
    double max_limit;
    /* traffic atlas: one row of 1 m cells per (edge, lane) */
    uint32_t n_rows;
    uint64_t n_cells;
    uint32_t *first_row; /* [n_edges]  */
    uint64_t *row_off;   /* [n_rows]   */
    uint8_t *occ[2];     /* logical cell content: occupied?           */
    uint16_t *frac[2];   /*   low 10 bits of the occupant's x_fx (G3) */
    float *spd[2];       /*   occupant's speed          */
    /* parameters and R0 constants */
    mo_params p;
    float C1, HALF_DT, VSCALE, ADT;
    int32_t L_fx;
    uint32_t L_c, Z_out, Z_in, LEN_MIN, Lam;
    uint32_t *P_mlc; /* [5*Lam+1] */
    /* trips, indexed by vehicle id = rank in (depart_step, caller index) order */
    uint32_t n_trips;
    uint64_t *route_ptr;   /* caller order, [n_trips+1] */
    uint32_t *route_edges; /* caller order              */
    uint32_t *trip_of_id, *id_of_trip;
    uint32_t *depart_step;
    uint8_t *status, *lane, *tag, *wait;
    uint32_t *rpos, *x_fx, *admit_step, *arrive_step;
    float *v, *acc_last;
    /* tentative next state of the step in flight */
    uint8_t *nx_kind, *nx_lane, *nx_tag;
    uint32_t *nx_x, *nx_claim;
    float *nx_v;
    uint64_t *claim; /* [n_rows + n_nodes] claim words: smallest key wins (key = vehicle id, or rank << 32 | id at STOP nodes) */
    uint64_t *nx_key;
    uint32_t W_stop; /* steps a vehicle stands at a STOP node's stop line: ceil(stop_time_s / dt) */
    uint64_t *stat_sum; /* [stat_n_slices * n_edges] */
    uint32_t *stat_cnt;
    /* lists */
    uint32_t *active, n_active;
    uint32_t *pending, n_pending, next_dep;
    uint32_t *adm_row; /* per pending entry: chosen row or NONE */
    uint32_t *order_buf;
    /* counters */
    uint32_t t;
    uint32_t *edge_entries;
    uint64_t n_done, sum_travel, n_updates, n_lane_changes, n_cells_examined, n_lc_evals;
    int order_mode;
    uint64_t order_state;
};

/* ---------------------------------------------------------------- G22 */
/* Counter-based generator rng(id, t, k): three rounds of a 32-bit avalanche mixer
 * (multiply-xorshift finaliser) over (seed, id, t, k).  Reading G22. */
static uint32_t mix32(uint32_t h)
{
    h ^= h >> 16;
    h *= 0x7feb352du;
    h ^= h >> 15;
    h *= 0x846ca68bu;
    h ^= h >> 16;
    return h;
}
static uint32_t rng32(uint64_t seed, uint32_t id, uint32_t t, uint32_t k)
{
    uint32_t lo = (uint32_t)seed, hi = (uint32_t)(seed >> 32);
    uint32_t h = mix32(lo + 0x9E3779B9u * (id + 1u));
    h = mix32((h ^ hi) + 0x85EBCA6Bu * (t + 1u));
    h = mix32(h + 0xC2B2AE35u * (k + 1u));
    return h;
}
uint32_t mo_rng(const mo_sim *S, uint32_t id, uint32_t t, uint32_t k) { return rng32(S->p.seed, id, t, k); }

/* R6: epsilon ~ N(0, sigma) as an Irwin-Hall sum of the 12 bytes of rng(id,t,k0..k0+2)
 * (Eq. 3, 4: "normally distributed with mean 0 and standard deviation 1"). */
static float eps_draw(const mo_sim *S, uint32_t id, uint32_t t, uint32_t k0)
{
    int32_t sum = 0;
    for (uint32_t k = k0; k < k0 + 3; k++) {
        uint32_t w = rng32(S->p.seed, id, t, k);
        sum += (int32_t)(w & 255u) + (int32_t)((w >> 8) & 255u) + (int32_t)((w >> 16) & 255u) + (int32_t)(w >> 24);
    }
    float e = (float)(sum - 1530);
    e = e * 0.00390625f; /* 2^-8 */
    e = S->p.lc_eps_sigma * e;
    return e;
}
float mo_eps(const mo_sim *S, uint32_t id, uint32_t t, uint32_t k0) { return eps_draw(S, id, t, k0); }

/* ---------------------------------------------------------------- R3 */
/* IDM acceleration, Eq. (1), delta = 4, guard G5. */
static float idm_acc(const mo_sim *S, float v, float v0, int has_leader, float s, float v_lead)
{
    float r = v / v0;
    float r2 = r * r;
    float fr = r2 * r2; /* (v/v0)^4 */
    float inter = 0.0f;
    if (has_leader) {
        float dv = v - v_lead;
        float q = v * dv;
        q = q * S->C1; /* v dv / (2 sqrt(ab)) */
        float ss = S->p.T * v;
        ss = ss + q;
        ss = fmaxf(0.0f, ss);
        ss = S->p.s0 + ss;
        float se = fmaxf(s, 0.01f);
        float z = ss / se;
        inter = z * z;
    }
    float acc = 1.0f - fr;
    acc = acc - inter;
    acc = S->p.a * acc;
    return acc;
}
float mo_idm_acc(const mo_sim *S, float v, float v0, int has_leader, float s, float v_lead)
{
    return idm_acc(S, v, v0, has_leader, s, v_lead);
}

uint32_t mo_pmlc(const mo_sim *S, uint32_t dcell) { return dcell <= 5u * S->Lam ? S->P_mlc[dcell] : 0u; }

/* ---------------------------------------------------------------- R3s */
/* Desired speed of a driver on an edge ("each driver's maximum possible speed per edge, v0, is
 * sampled from a Gaussian distribution centered around the edge's predetermined speed limit"; reading G27):
 * v0 = limit * clamp(1 + v0_sigma_rel * z, 1/2, 3/2), z the Irwin-Hall normal of generator words 7..9 at the
 * counter 0xFFFFFFFF - r (r = route position), so every (vehicle, route position) has its own draw.  sigma = 0: limit. */
static float desired_speed(const mo_sim *S, uint32_t id, uint32_t r, float limit)
{
    if (!(S->p.v0_sigma_rel > 0.0f)) return limit;
    int32_t sum = 0;
    for (uint32_t k = 7; k < 10; k++) {
        uint32_t w = rng32(S->p.seed, id, 0xFFFFFFFFu - r, k);
        sum += (int32_t)(w & 255u) + (int32_t)((w >> 8) & 255u) + (int32_t)((w >> 16) & 255u) + (int32_t)(w >> 24);
    }
    float z = (float)(sum - 1530);
    z = z * 0.00390625f; /* 2^-8 */
    float f = S->p.v0_sigma_rel * z;
    f = 1.0f + f;
    f = fmaxf(f, 0.5f);
    f = fminf(f, 1.5f);
    return limit * f;
}

/* ---------------------------------------------------------------- R0 */
static void derive_constants(mo_sim *S, double max_init_speed)
{
    const mo_params *p = &S->p;
    /* the fastest possible vehicle: the largest desired speed (limit, times 3/2 at most with per-driver v0, G27) */
    double vmax = S->max_limit * (p->v0_sigma_rel > 0.0f ? 1.5 : 1.0);
    double vcap = (vmax > max_init_speed ? vmax : max_init_speed) + (double)p->a * (double)p->dt;
    S->L_c = (uint32_t)ceil((double)p->veh_len);
    S->L_fx = (int32_t)lround((double)p->veh_len * 1024.0);
    S->Z_out = (uint32_t)ceil(vcap * (double)p->dt) + 1u;
    S->Z_in = S->L_c + S->Z_out;
    S->LEN_MIN = S->Z_out + 1u;
    if (S->LEN_MIN < S->L_c + 1u) S->LEN_MIN = S->L_c + 1u; /* R1 reads cells [0, L_c] of a row */
}

mo_sim *mo_create(uint32_t n_nodes, uint32_t n_edges, const uint32_t *row_ptr, const uint32_t *head,
                  const float *length_m, const uint8_t *lanes, const float *speed_limit,
                  const uint8_t *node_ctrl, const mo_params *p)
{
    mo_sim *S = (mo_sim *)calloc(1, sizeof(mo_sim));
    S->n_nodes = n_nodes;
    S->n_edges = n_edges;
    S->p = *p;
    S->row_ptr = (uint32_t *)malloc(sizeof(uint32_t) * (n_nodes + 1));
    memcpy(S->row_ptr, row_ptr, sizeof(uint32_t) * (n_nodes + 1));
    S->head = (uint32_t *)malloc(sizeof(uint32_t) * n_edges);
    S->tail = (uint32_t *)malloc(sizeof(uint32_t) * n_edges);
    S->len_c = (uint32_t *)malloc(sizeof(uint32_t) * n_edges);
    S->lanes = (uint8_t *)malloc(n_edges);
    S->limit = (float *)malloc(sizeof(float) * n_edges);
    S->ctrl = (uint8_t *)calloc(n_nodes, 1);
    S->first_row = (uint32_t *)malloc(sizeof(uint32_t) * n_edges);
    if (node_ctrl) memcpy(S->ctrl, node_ctrl, n_nodes);
    for (uint32_t u = 0; u < n_nodes; u++)
        for (uint32_t e = row_ptr[u]; e < row_ptr[u + 1]; e++) S->tail[e] = u;
    S->in_idx = (uint32_t *)calloc(n_edges, sizeof(uint32_t));
    S->indeg = (uint32_t *)calloc(n_nodes, sizeof(uint32_t));
    for (uint32_t e = 0; e < n_edges; e++) /* inbound edges of a node in edge-id order */
        if (head[e] < n_nodes) S->in_idx[e] = S->indeg[head[e]]++;
    S->max_limit = 0.0;
    uint32_t rows = 0;
    for (uint32_t e = 0; e < n_edges; e++) {
        if (!(lanes[e] >= 1 && lanes[e] <= 8) || !(length_m[e] > 0.0f) || !(speed_limit[e] > 0.0f) ||
            head[e] >= n_nodes || !isfinite(length_m[e]) || !isfinite(speed_limit[e])) {
            mo_destroy(S);
            return NULL;
        }
        S->head[e] = head[e];
        S->lanes[e] = lanes[e];
        S->limit[e] = speed_limit[e];
        S->len_c[e] = (uint32_t)lround((double)length_m[e]); /* t_m = 1 m cells */
        if ((double)speed_limit[e] > S->max_limit) S->max_limit = (double)speed_limit[e];
        S->first_row[e] = rows;
        rows += lanes[e];
    }
    S->n_rows = rows;
    S->row_off = (uint64_t *)malloc(sizeof(uint64_t) * (rows + 1));
    uint64_t cells = 0;
    for (uint32_t e = 0; e < n_edges; e++)
        for (uint32_t l = 0; l < lanes[e]; l++) {
            S->row_off[S->first_row[e] + l] = cells;
            cells += S->len_c[e];
        }
    S->row_off[rows] = cells;
    S->n_cells = cells;
    for (int k = 0; k < 2; k++) {
        S->occ[k] = (uint8_t *)calloc(cells + 1, 1);
        S->frac[k] = (uint16_t *)calloc(cells + 1, sizeof(uint16_t));
        S->spd[k] = (float *)calloc(cells + 1, sizeof(float));
    }
    /* R0 constants: rounded once from double */
    S->C1 = (float)(1.0 / (2.0 * sqrt((double)p->a * (double)p->b)));
    S->HALF_DT = (float)(0.5 * (double)p->dt);
    S->VSCALE = (float)((1.0 / 1024.0) / (double)p->dt);
    S->ADT = (float)((double)p->a * (double)p->dt);
    derive_constants(S, 0.0);
    for (uint32_t e = 0; e < n_edges; e++)
        if (S->len_c[e] < S->LEN_MIN) { /* G19 */
            mo_destroy(S);
            return NULL;
        }
    /* Eq. (2) table, distances in units of Lambda (G6) */
    S->Lam = (uint32_t)lround((double)p->mlc_scale_m);
    if (S->Lam < 1) S->Lam = 1;
    S->P_mlc = (uint32_t *)malloc(sizeof(uint32_t) * (5 * S->Lam + 1));
    for (uint32_t d = 0; d <= 5 * S->Lam; d++) {
        if (d <= S->Lam)
            S->P_mlc[d] = 0xFFFFFFFFu; /* x_i <= x_0: m_i = 1 */
        else {
            double xi = (double)d / (double)S->Lam;
            S->P_mlc[d] = (uint32_t)floor(4294967296.0 * exp(-(xi - 1.0) * (xi - 1.0)));
        }
    }
    S->claim = (uint64_t *)malloc(sizeof(uint64_t) * ((size_t)rows + n_nodes));
    for (size_t i = 0; i < (size_t)rows + n_nodes; i++) S->claim[i] = NONE64;
    S->W_stop = (uint32_t)ceil((double)p->stop_time_s / (double)p->dt - 1e-9);
    if (p->stat_period_steps && p->stat_n_slices) {
        S->stat_sum = (uint64_t *)calloc((size_t)p->stat_n_slices * n_edges, sizeof(uint64_t));
        S->stat_cnt = (uint32_t *)calloc((size_t)p->stat_n_slices * n_edges, sizeof(uint32_t));
    }
    S->edge_entries = (uint32_t *)calloc(n_edges, sizeof(uint32_t));
    return S;
}

void mo_destroy(mo_sim *S)
{
    if (!S) return;
    free(S->row_ptr); free(S->head); free(S->tail); free(S->len_c); free(S->lanes); free(S->ctrl);
    free(S->in_idx); free(S->indeg); free(S->wait); free(S->nx_key); free(S->stat_sum); free(S->stat_cnt);
    free(S->limit); free(S->first_row); free(S->row_off);
    for (int k = 0; k < 2; k++) { free(S->occ[k]); free(S->frac[k]); free(S->spd[k]); }
    free(S->P_mlc); free(S->route_ptr); free(S->route_edges); free(S->trip_of_id); free(S->id_of_trip);
    free(S->depart_step); free(S->status); free(S->lane); free(S->tag); free(S->rpos); free(S->x_fx);
    free(S->admit_step); free(S->arrive_step); free(S->v); free(S->acc_last);
    free(S->nx_kind); free(S->nx_lane); free(S->nx_tag); free(S->nx_x); free(S->nx_claim); free(S->nx_v);
    free(S->claim); free(S->active); free(S->pending); free(S->adm_row); free(S->order_buf);
    free(S->edge_entries);
    free(S);
}

static void mark_cell(mo_sim *S, int buf, uint32_t e, uint32_t l, uint32_t x_fx, float v)
{
    uint64_t cell = S->row_off[S->first_row[e] + l] + (x_fx >> 10);
    S->occ[buf][cell] = 1;
    S->frac[buf][cell] = (uint16_t)(x_fx & 1023u);
    S->spd[buf][cell] = v;
}
static void clear_cell(mo_sim *S, int buf, uint32_t e, uint32_t l, uint32_t x_fx)
{
    uint64_t cell = S->row_off[S->first_row[e] + l] + (x_fx >> 10);
    S->occ[buf][cell] = 0;
}
static uint32_t route_edge(const mo_sim *S, uint32_t id, uint32_t r)
{
    return S->route_edges[S->route_ptr[S->trip_of_id[id]] + r];
}
static uint32_t route_len(const mo_sim *S, uint32_t id)
{
    uint32_t tr = S->trip_of_id[id];
    return (uint32_t)(S->route_ptr[tr + 1] - S->route_ptr[tr]);
}

typedef struct { uint32_t key, idx; } keyidx;
static int cmp_keyidx(const void *a, const void *b)
{
    const keyidx *x = (const keyidx *)a, *y = (const keyidx *)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    return x->idx < y->idx ? -1 : (x->idx > y->idx);
}

/* R0 (trip part) and R1 (pre-placed vehicles). */
int mo_load_trips(mo_sim *S, uint32_t n_trips, const uint64_t *route_ptr, const uint32_t *route_edges,
                  const float *depart_time_s, const float *init_pos_m, const float *init_speed)
{
    if (S->n_trips) return -6; /* already loaded */
    double max_init = 0.0;
    for (uint32_t i = 0; i < n_trips; i++) {
        uint64_t b = route_ptr[i], e = route_ptr[i + 1];
        if (e <= b) return -3; /* empty route */
        for (uint64_t k = b; k < e; k++) {
            if (route_edges[k] >= S->n_edges) return -3;
            if (k > b && S->head[route_edges[k - 1]] != S->tail[route_edges[k]]) return -3;
        }
        int pre = init_pos_m && init_pos_m[i] >= 0.0f;
        if (!pre && !(depart_time_s[i] >= 0.0f)) return -3;
        if (init_speed) {
            if (!(init_speed[i] >= 0.0f) || !isfinite(init_speed[i])) return -3;
            if (pre && (double)init_speed[i] > max_init) max_init = (double)init_speed[i];
        }
    }
    derive_constants(S, max_init);
    for (uint32_t e = 0; e < S->n_edges; e++)
        if (S->len_c[e] < S->LEN_MIN) return -3;
    if (S->p.lookback_cells < S->L_c + S->Z_out) return -1; /* R5 requirement */

    S->n_trips = n_trips;
    uint64_t total = route_ptr[n_trips];
    S->route_ptr = (uint64_t *)malloc(sizeof(uint64_t) * (n_trips + 1));
    memcpy(S->route_ptr, route_ptr, sizeof(uint64_t) * (n_trips + 1));
    S->route_edges = (uint32_t *)malloc(sizeof(uint32_t) * (total + 1));
    memcpy(S->route_edges, route_edges, sizeof(uint32_t) * total);
    /* vehicle id = rank in stable (depart_step, caller index) order (boundary) */
    keyidx *ki = (keyidx *)malloc(sizeof(keyidx) * (n_trips + 1));
    for (uint32_t i = 0; i < n_trips; i++) {
        int pre = init_pos_m && init_pos_m[i] >= 0.0f;
        ki[i].key = pre ? 0u : (uint32_t)floor((double)depart_time_s[i] / (double)S->p.dt);
        ki[i].idx = i;
    }
    qsort(ki, n_trips, sizeof(keyidx), cmp_keyidx);
    size_t n = (size_t)n_trips + 1;
    S->trip_of_id = (uint32_t *)malloc(4 * n); S->id_of_trip = (uint32_t *)malloc(4 * n);
    S->depart_step = (uint32_t *)malloc(4 * n);
    S->status = (uint8_t *)calloc(n, 1); S->lane = (uint8_t *)calloc(n, 1); S->tag = (uint8_t *)calloc(n, 1);
    S->wait = (uint8_t *)calloc(n, 1); S->nx_key = (uint64_t *)calloc(n, sizeof(uint64_t));
    S->rpos = (uint32_t *)calloc(n, 4); S->x_fx = (uint32_t *)calloc(n, 4);
    S->admit_step = (uint32_t *)malloc(4 * n); S->arrive_step = (uint32_t *)malloc(4 * n);
    S->v = (float *)calloc(n, 4); S->acc_last = (float *)calloc(n, 4);
    S->nx_kind = (uint8_t *)calloc(n, 1); S->nx_lane = (uint8_t *)calloc(n, 1); S->nx_tag = (uint8_t *)calloc(n, 1);
    S->nx_x = (uint32_t *)calloc(n, 4); S->nx_claim = (uint32_t *)calloc(n, 4); S->nx_v = (float *)calloc(n, 4);
    S->active = (uint32_t *)malloc(4 * n); S->pending = (uint32_t *)malloc(4 * n);
    S->adm_row = (uint32_t *)malloc(4 * n); S->order_buf = (uint32_t *)malloc(4 * n);
    for (uint32_t id = 0; id < n_trips; id++) {
        S->trip_of_id[id] = ki[id].idx;
        S->id_of_trip[ki[id].idx] = id;
        S->depart_step[id] = ki[id].key;
        S->admit_step[id] = NONE32;
        S->arrive_step[id] = NONE32;
        S->status[id] = MO_WAITING;
    }
    free(ki);
    /* pre-placed vehicles: ACTIVE at t = 0 on route[0], lane 0 (R1, last sentence) */
    S->n_active = 0;
    for (uint32_t id = 0; id < n_trips; id++) {
        uint32_t tr = S->trip_of_id[id];
        if (!(init_pos_m && init_pos_m[tr] >= 0.0f)) continue;
        uint32_t e = route_edge(S, id, 0);
        uint32_t x = (uint32_t)lround((double)init_pos_m[tr] * 1024.0);
        if (x >= (S->len_c[e] << 10)) return -3;
        S->status[id] = MO_ACTIVE;
        S->x_fx[id] = x;
        S->v[id] = init_speed ? init_speed[tr] : 0.0f;
        S->lane[id] = 0;
        S->rpos[id] = 0;
        S->admit_step[id] = 0;
        S->edge_entries[e] += 1;
        S->active[S->n_active++] = id;
    }
    /* spacing check between pre-placed vehicles of one row: >= L (BAD_ROUTE otherwise) */
    {
        /* sort (row, x) pairs, then compare neighbours */
        keyidx *kx = (keyidx *)malloc(sizeof(keyidx) * (S->n_active + 1));
        for (uint32_t k = 0; k < S->n_active; k++) {
            uint32_t id = S->active[k];
            kx[k].key = S->first_row[route_edge(S, id, 0)];
            kx[k].idx = S->x_fx[id];
        }
        qsort(kx, S->n_active, sizeof(keyidx), cmp_keyidx);
        int bad = 0;
        for (uint32_t k = 1; k < S->n_active; k++)
            if (kx[k].key == kx[k - 1].key && (int64_t)kx[k].idx - (int64_t)kx[k - 1].idx < (int64_t)S->L_fx) bad = 1;
        free(kx);
        if (bad) return -3;
    }
    for (uint32_t k = 0; k < S->n_active; k++) {
        uint32_t id = S->active[k];
        mark_cell(S, 0, route_edge(S, id, 0), 0, S->x_fx[id], S->v[id]);
    }
    /* pre-placed vehicles sort with key 0 among the depart_step-0 trips; R1 skips them by status */
    S->next_dep = 0;
    S->n_pending = 0;
    S->t = 0;
    return 0;
}

void mo_set_order(mo_sim *S, int mode, uint64_t seed)
{
    S->order_mode = mode;
    S->order_state = seed * 0x9E3779B97F4A7C15ull + 1ull;
}

/* processing order of a list (pin K10: the result must not depend on it) */
static const uint32_t *ordered(mo_sim *S, const uint32_t *list, uint32_t n)
{
    if (S->order_mode == 0) return list;
    for (uint32_t i = 0; i < n; i++) S->order_buf[i] = list[i];
    if (S->order_mode == 1) {
        for (uint32_t i = 0; i < n / 2; i++) {
            uint32_t tmp = S->order_buf[i];
            S->order_buf[i] = S->order_buf[n - 1 - i];
            S->order_buf[n - 1 - i] = tmp;
        }
    } else {
        for (uint32_t i = n; i > 1; i--) {
            S->order_state = S->order_state * 6364136223846793005ull + 1442695040888963407ull;
            uint32_t j = (uint32_t)((S->order_state >> 33) % i);
            uint32_t tmp = S->order_buf[i - 1];
            S->order_buf[i - 1] = S->order_buf[j];
            S->order_buf[j] = tmp;
        }
    }
    return S->order_buf;
}

/* ---------------------------------------------------------------- R1 */
/* Departure admission (every trip starts at its departure time; G17). */
static void admission(mo_sim *S)
{
    int A = (int)(S->t & 1u);
    /* release trips whose depart_step <= t */
    while (S->next_dep < S->n_trips && S->depart_step[S->next_dep] <= S->t) {
        if (S->status[S->next_dep] == MO_WAITING) S->pending[S->n_pending++] = S->next_dep;
        S->next_dep++;
    }
    const uint32_t *ord = ordered(S, S->pending, S->n_pending);
    uint32_t *ordcopy = (uint32_t *)malloc(sizeof(uint32_t) * (S->n_pending + 1));
    memcpy(ordcopy, ord, sizeof(uint32_t) * S->n_pending);
    /* every decision is taken against atlas_t BEFORE any admission of this step */
    for (uint32_t k = 0; k < S->n_pending; k++) {
        uint32_t id = ordcopy[k];
        uint32_t e = route_edge(S, id, 0);
        uint32_t chosen = NONE32;
        for (uint32_t l = 0; l < S->lanes[e] && chosen == NONE32; l++) {
            uint64_t base = S->row_off[S->first_row[e] + l];
            int free_window = 1;
            for (uint32_t c = 0; c <= S->L_c; c++)
                if (S->occ[A][base + c]) free_window = 0;
            if (free_window) chosen = S->first_row[e] + l;
        }
        S->nx_claim[id] = chosen;
        if (chosen != NONE32 && (uint64_t)id < S->claim[chosen]) S->claim[chosen] = id; /* smallest id wins */
    }
    uint32_t n_keep = 0;
    for (uint32_t k = 0; k < S->n_pending; k++) {
        uint32_t id = S->pending[k];
        uint32_t row = S->nx_claim[id];
        if (row != NONE32 && S->claim[row] == (uint64_t)id) {
            uint32_t e = route_edge(S, id, 0);
            S->status[id] = MO_ACTIVE;
            S->x_fx[id] = 0;
            S->v[id] = 0.0f;
            S->tag[id] = 0;
            S->wait[id] = 0;
            S->rpos[id] = 0;
            S->lane[id] = (uint8_t)(row - S->first_row[e]);
            S->admit_step[id] = S->t;
            S->edge_entries[e] += 1;
            S->active[S->n_active++] = id;
            mark_cell(S, A, e, S->lane[id], 0, 0.0f); /* visible to everybody in this step's P1 */
        } else {
            S->pending[n_keep++] = id;
        }
    }
    for (uint32_t k = 0; k < S->n_pending; k++) { /* reset the claim words used */
        uint32_t row = S->nx_claim[ordcopy[k]];
        if (row != NONE32) S->claim[row] = NONE64;
    }
    S->n_pending = n_keep;
    free(ordcopy);
}

/* ---------------------------------------------------------------- R2 */
/* Leader search along the own lane and on along the route ("looking up the
 * status of neighboring cells"; G16).  Returns 1 and (lead_abs_fx, v_lead) if found. */
static int leader_search(mo_sim *S, int A, uint32_t id, uint32_t r, uint32_t l, uint32_t c, int32_t *lead_abs_fx,
                         float *v_lead)
{
    uint32_t nroute = route_len(S, id);
    uint32_t e = route_edge(S, id, r);
    uint32_t base_cells = 0, examined = 0, j = c + 1;
    while (examined < S->p.lookahead_cells) {
        if (j >= S->len_c[e]) {
            if (r + 1 >= nroute) return 0;
            base_cells += S->len_c[e];
            r += 1;
            e = route_edge(S, id, r);
            if (l > (uint32_t)S->lanes[e] - 1u) l = (uint32_t)S->lanes[e] - 1u;
            j = 0;
            continue;
        }
        uint64_t cell = S->row_off[S->first_row[e] + l] + j;
        examined++;
        S->n_cells_examined++;
        if (S->occ[A][cell]) {
            *lead_abs_fx = (int32_t)(((base_cells + j) << 10) | S->frac[A][cell]);
            *v_lead = S->spd[A][cell];
            return 1;
        }
        j++;
    }
    return 0;
}

/* ---------------------------------------------------------------- R5 */
static int lead_in_lane(mo_sim *S, int A, uint32_t e, uint32_t lt, uint32_t c, int32_t *x_a, float *v_a)
{
    uint64_t base = S->row_off[S->first_row[e] + lt];
    for (uint32_t k = 0; k < S->p.lookahead_cells; k++) {
        uint32_t j = c + k;
        if (j >= S->len_c[e]) return 0;
        if (S->occ[A][base + j]) {
            *x_a = (int32_t)((j << 10) | S->frac[A][base + j]);
            *v_a = S->spd[A][base + j];
            return 1;
        }
    }
    return 0;
}
static int lag_in_lane(mo_sim *S, int A, uint32_t e, uint32_t lt, uint32_t c, int32_t *x_b, float *v_b)
{
    uint64_t base = S->row_off[S->first_row[e] + lt];
    for (uint32_t k = 1; k <= S->p.lookback_cells; k++) {
        if (k > c) return 0;
        uint32_t j = c - k;
        if (S->occ[A][base + j]) {
            *x_b = (int32_t)((j << 10) | S->frac[A][base + j]);
            *v_b = S->spd[A][base + j];
            return 1;
        }
    }
    return 0;
}

enum { KIND_STAY = 0, KIND_DONE = 1, KIND_CAND = 2, KIND_HOLD = 3 };

/* ---------------------------------------------------------------- R2..R8 for one vehicle */
static void update_vehicle(mo_sim *S, uint32_t id)
{
    const mo_params *p = &S->p;
    int A = (int)(S->t & 1u);
    uint32_t r = S->rpos[id], l = S->lane[id];
    uint32_t nroute = route_len(S, id);
    int last = (r + 1 == nroute);
    uint32_t e = route_edge(S, id, r);
    uint32_t n = S->lanes[e], len_c = S->len_c[e];
    int32_t len_fx = (int32_t)(len_c << 10);
    int32_t x = (int32_t)S->x_fx[id];
    uint32_t c = (uint32_t)x >> 10;
    float v = S->v[id], v0 = desired_speed(S, id, r, S->limit[e]);
    S->n_updates++;
    /* per-edge speed statistics (Eq. 5 inputs): instantaneous speeds of time t, every period steps */
    if (S->stat_sum && S->t % p->stat_period_steps == 0u) {
        uint32_t slice = S->t / p->stat_slice_steps;
        if (slice < p->stat_n_slices) {
            S->stat_sum[(size_t)slice * S->n_edges + e] += (uint64_t)lrintf(v * 256.0f);
            S->stat_cnt[(size_t)slice * S->n_edges + e] += 1u;
        }
    }

    /* R2 */
    int32_t lead_abs = 0;
    float v_lead = 0.0f, s = 0.0f;
    int found = leader_search(S, A, id, r, l, c, &lead_abs, &v_lead);
    int32_t bound_cur = BOUND_INF;
    if (found) {
        float sf = (float)(lead_abs - x);
        sf = sf * 0.0009765625f; /* 2^-10 */
        s = sf - p->veh_len;
        bound_cur = lead_abs - S->L_fx;
    }
    /* R3 */
    float acc_cur = idm_acc(S, v, v0, found, s, v_lead);

    /* R4: mandatory tag, Eq. (2) */
    uint8_t tag = S->tag[id];
    if (tag == 0 && !last && n >= 2) {
        uint32_t dcell = len_c - c;
        if (dcell <= S->Lam)
            tag = 1;
        else if (dcell <= 5u * S->Lam) {
            uint32_t u0 = rng32(p->seed, id, S->t, 0);
            if (u0 < S->P_mlc[dcell]) tag = 1;
        }
    }
    /* allowed-lane range [lo, hi] for the next turn (R0, G7) */
    uint32_t lo = 0, hi = n - 1;
    if (!last) {
        uint32_t en = route_edge(S, id, r + 1);
        uint32_t u = S->head[e];
        uint32_t d = S->row_ptr[u + 1] - S->row_ptr[u];
        uint32_t j = en - S->row_ptr[u];
        lo = (j * n) / d;
        uint32_t hi1 = ((j + 1) * n) / d;
        hi = (hi1 >= 1 && hi1 - 1 > lo) ? hi1 - 1 : lo;
    }
    int dir = (S->t & 1u) ? -1 : +1; /* G11 */
    int lt_s = (int)l + dir;
    uint32_t l_new = l;
    float acc = acc_cur;
    int32_t bound = bound_cur;
    int possible = lt_s >= 0 && lt_s < (int)n && c >= S->Z_in && (int64_t)c < (int64_t)len_c - (int64_t)S->Z_out;
    if (possible) {
        uint32_t lt = (uint32_t)lt_s;
        int l_in = (l >= lo && l <= hi), lt_in = (lt >= lo && lt <= hi);
        int mand = tag == 1 && !l_in && ((l < lo && dir > 0) || (l > hi && dir < 0));
        /* discretionary pre-test: impeded in the own lane (G9) */
        int disc_pre = 0;
        if (!(tag == 1 && !lt_in) && found) {
            float rr = v / v0;
            float rr2 = rr * rr;
            float fr = rr2 * rr2;
            float af = 1.0f - fr;
            af = p->a * af;
            float g = af - acc_cur;
            disc_pre = g > p->dlc_gain_thr;
        }
        if (mand || disc_pre) {
            S->n_lc_evals++;
            /* R5 */
            int32_t x_a = 0, x_b = 0;
            float v_a = 0.0f, v_b = 0.0f, gap_lead = 0.0f, gap_lag = 0.0f;
            int has_a = lead_in_lane(S, A, e, lt, c, &x_a, &v_a);
            int has_b = lag_in_lane(S, A, e, lt, c, &x_b, &v_b);
            if (has_a) {
                float gf = (float)(x_a - x);
                gf = gf * 0.0009765625f;
                gap_lead = gf - p->veh_len;
            }
            if (has_b) {
                float gf = (float)(x - x_b);
                gf = gf * 0.0009765625f;
                gap_lag = gf - p->veh_len;
            }
            float acc_tgt = idm_acc(S, v, v0, has_a, gap_lead, v_a);
            float gain = acc_tgt - acc_cur;
            int want = mand || (disc_pre && gain > p->dlc_gain_thr);
            if (want) {
                /* R6: gap acceptance, Eq. (3), (4) */
                float g0 = (v < 11.176f) ? p->lc_gap_low : p->lc_gap_high;
                int ok = 1;
                if (has_a) {
                    float t1 = p->lc_alpha * v;
                    float t2 = v - v_a;
                    t2 = p->lc_alpha * t2;
                    float g = g0 + t1;
                    g = g + t2;
                    g = fmaxf(g0, g);
                    g = g + eps_draw(S, id, S->t, 1);
                    g = fmaxf(g, 0.0f);
                    if (!(gap_lead >= g)) ok = 0;
                }
                if (has_b) {
                    float t1 = p->lc_alpha * v;
                    float t2 = v - v_b;
                    t2 = p->lc_alpha * t2;
                    float g = g0 + t1;
                    g = g + t2;
                    g = fmaxf(g0, g);
                    g = g + eps_draw(S, id, S->t, 4);
                    float fl = v_b + S->ADT; /* hard safety floor */
                    fl = fl * p->dt;
                    fl = fl + 0.01f;
                    g = fmaxf(g, fl);
                    if (!(gap_lag >= g)) ok = 0;
                }
                if (ok) {
                    l_new = lt;
                    acc = fminf(acc_cur, acc_tgt);
                    if (has_a) {
                        int32_t bt = x_a - S->L_fx;
                        if (bt < bound) bound = bt;
                    }
                    S->n_lane_changes++;
                }
            }
        }
    }
    /* R7: ballistic update ("double integrating"; G4) and hard clamp */
    float vn = acc * p->dt;
    vn = v + vn;
    vn = fmaxf(0.0f, vn);
    float m = v + vn;
    m = m * S->HALF_DT;
    int32_t dx = (int32_t)lrintf(m * 1024.0f); /* round to nearest, ties to even */
    int32_t xn = x + dx;
    if (xn > bound) {
        xn = bound > x ? bound : x;
        float vc = (float)(xn - x);
        vc = vc * S->VSCALE;
        vn = fminf(vn, vc);
    }
    S->acc_last[id] = acc;
    /* R8 */
    S->nx_lane[id] = (uint8_t)l_new;
    S->nx_tag[id] = tag;
    S->nx_v[id] = vn;
    if (xn < len_fx) {
        S->nx_kind[id] = KIND_STAY;
        S->nx_x[id] = (uint32_t)xn;
    } else if (last) {
        S->nx_kind[id] = KIND_DONE; /* G18 */
    } else {
        uint32_t en = route_edge(S, id, r + 1);
        uint32_t lplus = l_new;
        if (lplus > (uint32_t)S->lanes[en] - 1u) lplus = (uint32_t)S->lanes[en] - 1u;
        uint32_t u = S->head[e];
        uint32_t word = (S->ctrl[u] == 0) ? S->first_row[en] + lplus /* GREEN: lane entry */
                                          : S->n_rows + u;           /* PRIORITY, STOP: the node */
        uint64_t key = id;
        S->nx_x[id] = (uint32_t)(xn - len_fx);
        if (S->ctrl[u] == 2 && S->wait[id] < S->W_stop) {
            /* R8s ("every vehicle is designed to stop at the intersection for 2 seconds before
             * proceeding"): it stands at the stop line for W_stop steps before it may ask for the node */
            S->nx_kind[id] = KIND_HOLD;
            return;
        }
        if (S->ctrl[u] == 2) {
            /* R8s ("a round-robin of the nm combinations ... based on their position in their lane
             * queue"): the n inbound x m outbound combinations take turns; at step t combination (c - t) mod nm = 0
             * is first, then 1, ...; only the front vehicle of a lane can be here; equal combinations: smallest id */
            uint32_t m = S->row_ptr[u + 1] - S->row_ptr[u], nm = S->indeg[u] * m;
            uint32_t c = S->in_idx[e] * m + (en - S->row_ptr[u]);
            uint32_t rank = (c + nm - S->t % nm) % nm;
            key = ((uint64_t)rank << 32) | id;
        }
        S->nx_kind[id] = KIND_CAND;
        S->nx_claim[id] = word;
        S->nx_key[id] = key;
        if (key < S->claim[word]) S->claim[word] = key;
    }
}

/* ---------------------------------------------------------------- R8 (resolution) + R9 */
static void commit(mo_sim *S)
{
    int A = (int)(S->t & 1u), B = A ^ 1;
    uint32_t n_keep = 0;
    /* clear the time-t marks: atlas_t is the write buffer of step t+1 */
    for (uint32_t k = 0; k < S->n_active; k++) {
        uint32_t id = S->active[k];
        clear_cell(S, A, route_edge(S, id, S->rpos[id]), S->lane[id], S->x_fx[id]);
    }
    const uint32_t *ord = ordered(S, S->active, S->n_active);
    uint32_t *ordcopy = (uint32_t *)malloc(sizeof(uint32_t) * (S->n_active + 1));
    memcpy(ordcopy, ord, sizeof(uint32_t) * S->n_active);
    for (uint32_t k = 0; k < S->n_active; k++) {
        uint32_t id = ordcopy[k];
        uint32_t r = S->rpos[id];
        uint32_t e = route_edge(S, id, r);
        S->tag[id] = S->nx_tag[id];
        if (S->nx_kind[id] == KIND_STAY) {
            S->lane[id] = S->nx_lane[id];
            S->x_fx[id] = S->nx_x[id];
            S->v[id] = S->nx_v[id];
        } else if (S->nx_kind[id] == KIND_DONE) {
            S->status[id] = MO_DONE;
            S->arrive_step[id] = S->t + 1;
            S->n_done++;
            S->sum_travel += (uint64_t)(S->arrive_step[id] - S->admit_step[id]);
            continue;
        } else if (S->nx_kind[id] == KIND_HOLD) { /* R8s: stands at the stop line, one more step done */
            S->lane[id] = S->nx_lane[id];
            S->x_fx[id] = (S->len_c[e] << 10) - 1u;
            S->v[id] = 0.0f;
            S->wait[id] += 1;
        } else if (S->claim[S->nx_claim[id]] == S->nx_key[id]) { /* winner crosses */
            uint32_t en = route_edge(S, id, r + 1);
            uint32_t lplus = S->nx_lane[id];
            if (lplus > (uint32_t)S->lanes[en] - 1u) lplus = (uint32_t)S->lanes[en] - 1u;
            S->rpos[id] = r + 1;
            S->lane[id] = (uint8_t)lplus;
            S->x_fx[id] = S->nx_x[id];
            S->v[id] = S->nx_v[id];
            S->tag[id] = 0;
            S->wait[id] = 0;
            S->edge_entries[en] += 1;
        } else { /* loser holds at the stop line (G15) */
            S->lane[id] = S->nx_lane[id];
            S->x_fx[id] = (S->len_c[e] << 10) - 1u;
            S->v[id] = 0.0f;
        }
        mark_cell(S, B, route_edge(S, id, S->rpos[id]), S->lane[id], S->x_fx[id], S->v[id]);
    }
    for (uint32_t k = 0; k < S->n_active; k++) { /* reset claim words */
        uint32_t id = S->active[k];
        if (S->nx_kind[id] == KIND_CAND) S->claim[S->nx_claim[id]] = NONE64;
    }
    for (uint32_t k = 0; k < S->n_active; k++) {
        uint32_t id = S->active[k];
        if (S->status[id] == MO_ACTIVE) S->active[n_keep++] = id;
    }
    S->n_active = n_keep;
    free(ordcopy);
    S->t += 1;
}

int mo_step(mo_sim *S, uint32_t n_steps)
{
    if (!S->n_trips) return -6;
    for (uint32_t k = 0; k < n_steps; k++) {
        admission(S);
        const uint32_t *ord = ordered(S, S->active, S->n_active);
        uint32_t n = S->n_active;
        if (ord != S->active) {
            uint32_t *tmp = (uint32_t *)malloc(sizeof(uint32_t) * (n + 1));
            memcpy(tmp, ord, sizeof(uint32_t) * n);
            for (uint32_t i = 0; i < n; i++) update_vehicle(S, tmp[i]);
            free(tmp);
        } else {
            for (uint32_t i = 0; i < n; i++) update_vehicle(S, ord[i]);
        }
        commit(S);
    }
    return 0;
}

/* ---------------------------------------------------------------- state injection (tests only) */
/* Replace the whole dynamic state by the caller's (arrays in CALLER trip order) and rebuild the
 * atlas and the lists from it.  No arithmetic of the method happens here: it lets a test start the
 * oracle from a snapshot (e.g. the peak of a large run) and compare ONE step.  edge_entries may be NULL
 * (kept as is). */
int mo_set_state(mo_sim *S, uint32_t t, const uint8_t *status, const uint32_t *route_pos, const uint8_t *lane,
                 const uint8_t *tag, const uint32_t *x_fx, const float *v, const uint32_t *admit_step,
                 const uint32_t *arrive_step, const uint32_t *edge_entries)
{
    if (!S->n_trips) return -6;
    for (int k = 0; k < 2; k++) memset(S->occ[k], 0, S->n_cells);
    S->t = t;
    S->n_active = 0;
    S->n_pending = 0;
    S->next_dep = 0;
    S->n_done = 0;
    S->sum_travel = 0;
    for (uint32_t id = 0; id < S->n_trips; id++) {
        uint32_t tr = S->trip_of_id[id];
        S->status[id] = status[tr];
        S->rpos[id] = route_pos[tr];
        S->lane[id] = lane[tr];
        S->tag[id] = tag[tr];
        S->x_fx[id] = x_fx[tr];
        S->v[id] = v[tr];
        S->admit_step[id] = admit_step[tr];
        S->arrive_step[id] = arrive_step[tr];
        S->wait[id] = 0;
        if (status[tr] == MO_ACTIVE) {
            uint32_t e;
            if (route_pos[tr] >= route_len(S, id)) return -3;
            e = route_edge(S, id, route_pos[tr]);
            if (lane[tr] >= S->lanes[e] || (x_fx[tr] >> 10) >= S->len_c[e]) return -3;
            S->active[S->n_active++] = id;
            mark_cell(S, (int)(t & 1u), e, lane[tr], x_fx[tr], v[tr]);
        } else if (status[tr] == MO_DONE) {
            S->n_done++;
            S->sum_travel += (uint64_t)(arrive_step[tr] - admit_step[tr]);
        }
    }
    if (edge_entries) memcpy(S->edge_entries, edge_entries, sizeof(uint32_t) * S->n_edges);
    return 0;
}

void mo_set_wait(mo_sim *S, const uint8_t *wait)
{
    for (uint32_t tr = 0; tr < S->n_trips; tr++) S->wait[S->id_of_trip[tr]] = wait[tr];
}
void mo_get_wait(const mo_sim *S, uint8_t *wait)
{
    for (uint32_t tr = 0; tr < S->n_trips; tr++) wait[tr] = S->wait[S->id_of_trip[tr]];
}
void mo_get_edge_speed_stats(const mo_sim *S, uint64_t *sum_q8, uint32_t *samples)
{
    size_t n = (size_t)S->p.stat_n_slices * S->n_edges;
    if (!S->stat_sum) return;
    if (sum_q8) memcpy(sum_q8, S->stat_sum, n * sizeof(uint64_t));
    if (samples) memcpy(samples, S->stat_cnt, n * sizeof(uint32_t));
}
float mo_v0(const mo_sim *S, uint32_t id, uint32_t r)
{
    return desired_speed(S, id, r, S->limit[route_edge(S, id, r)]);
}
uint64_t mo_n_stopped(const mo_sim *S)
{
    uint64_t n = 0;
    for (uint32_t k = 0; k < S->n_active; k++) n += (S->v[S->active[k]] == 0.0f);
    return n;
}

/* ---------------------------------------------------------------- outputs */
void mo_get_state(const mo_sim *S, uint8_t *status, uint32_t *route_pos, uint8_t *lane, uint8_t *tag,
                  uint32_t *x_fx, float *v, float *acc_last)
{
    for (uint32_t tr = 0; tr < S->n_trips; tr++) {
        uint32_t id = S->id_of_trip[tr];
        if (status) status[tr] = S->status[id];
        if (route_pos) route_pos[tr] = S->rpos[id];
        if (lane) lane[tr] = S->lane[id];
        if (tag) tag[tr] = S->tag[id];
        if (x_fx) x_fx[tr] = S->x_fx[id];
        if (v) v[tr] = S->v[id];
        if (acc_last) acc_last[tr] = S->acc_last[id];
    }
}
void mo_get_trip_results(const mo_sim *S, uint32_t *admit_step, uint32_t *arrive_step)
{
    for (uint32_t tr = 0; tr < S->n_trips; tr++) {
        uint32_t id = S->id_of_trip[tr];
        if (admit_step) admit_step[tr] = S->admit_step[id];
        if (arrive_step) arrive_step[tr] = S->arrive_step[id];
    }
}
void mo_get_edge_entries(const mo_sim *S, uint32_t *edge_entries)
{
    memcpy(edge_entries, S->edge_entries, sizeof(uint32_t) * S->n_edges);
}
void mo_get_summary(const mo_sim *S, uint64_t out[9])
{
    uint64_t nw = 0;
    for (uint32_t id = 0; id < S->n_trips; id++) nw += (S->status[id] == MO_WAITING);
    out[0] = S->t; out[1] = nw; out[2] = S->n_active; out[3] = S->n_done; out[4] = S->sum_travel;
    out[5] = S->n_updates; out[6] = S->n_lane_changes; out[7] = S->n_cells_examined; out[8] = S->n_lc_evals;
}
void mo_get_derived(const mo_sim *S, uint32_t out[6])
{
    out[0] = S->L_c; out[1] = S->Z_out; out[2] = S->Z_in; out[3] = S->LEN_MIN; out[4] = (uint32_t)S->L_fx; out[5] = S->Lam;
}
void mo_get_vehicle_ids(const mo_sim *S, uint32_t *id_of_trip)
{
    memcpy(id_of_trip, S->id_of_trip, sizeof(uint32_t) * S->n_trips);
}
uint64_t mo_n_cells(const mo_sim *S) { return S->n_cells; }
uint32_t mo_n_rows(const mo_sim *S) { return S->n_rows; }
void mo_get_atlas(const mo_sim *S, uint8_t *occ, uint16_t *frac, float *spd)
{
    int A = (int)(S->t & 1u);
    if (occ) memcpy(occ, S->occ[A], S->n_cells);
    if (frac) memcpy(frac, S->frac[A], S->n_cells * sizeof(uint16_t));
    if (spd) memcpy(spd, S->spd[A], S->n_cells * sizeof(float));
}
void mo_get_row_offsets(const mo_sim *S, uint32_t *first_row, uint64_t *row_off)
{
    if (first_row) memcpy(first_row, S->first_row, sizeof(uint32_t) * S->n_edges);
    if (row_off) memcpy(row_off, S->row_off, sizeof(uint64_t) * S->n_rows);
}
