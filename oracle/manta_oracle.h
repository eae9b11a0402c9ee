/*
 * oracle/manta_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU microsimulator of MANTA's per-timestep
 * vehicle update (arxiv 2007.03614; Eq. (1)-(4)).  It is the
 * oracle the CUDA path is compared against.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table generator or constant with
 * paper_2007_03614_b200/csrc; the rule numbers R0..R9 and the readings G1..G23
 * it cites are written out in DESIGN.md (section "Rules").
 */
#ifndef MANTA_ORACLE_H
#define MANTA_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mo_sim mo_sim;

typedef struct {
    float dt;            /* timestep, s (0.5)                    */
    float a;             /* IDM acceleration potential, m/s^2  (Eq. 1)        */
    float b;             /* IDM braking deceleration, m/s^2    (Eq. 1)        */
    float T;             /* IDM desired time headway, s        (Eq. 1)        */
    float s0;            /* IDM standstill spacing, m          (Eq. 1)        */
    float veh_len;       /* vehicle length L, m                               */
    uint32_t lookahead_cells;  /* H   (reading G16)                           */
    uint32_t lookback_cells;   /* lag search range (R5)                       */
    float mlc_scale_m;   /* Lambda: unit of x_i, x_0 in Eq. 2 (reading G6)    */
    float dlc_gain_thr;  /* discretionary gain threshold, m/s^2 (reading G9)  */
    float lc_alpha;      /* anticipation time alpha, s (Eq. 3, 4)             */
    float lc_gap_low;    /* g_a = g_b below 25 mph, m          */
    float lc_gap_high;   /* g_a = g_b above 25 mph, m                         */
    float lc_eps_sigma;  /* std-dev of epsilon, m (Eq. 3, 4: 1)               */
    uint64_t seed;       /* seed of the counter-based generator (G22)         */
    float stop_time_s;   /* STOP nodes: time every vehicle stands at the stop line, s (2) */
    float v0_sigma_rel;  /* per-driver desired speed: v0 = limit * clamp(1 + v0_sigma_rel * z, 1/2, 3/2),
                            z ~ N(0,1) per (vehicle, route position) (reading G27); 0 = off  */
    uint32_t stat_period_steps; /* per-edge speed statistics (Eq. 5 inputs): every this many
                                   steps each ACTIVE vehicle adds its speed to its edge's accumulators; 0 = off  */
    uint32_t stat_slice_steps;  /* steps per time slice of the statistics                                     */
    uint32_t stat_n_slices;     /* number of time slices kept                                                 */
} mo_params;

enum { MO_WAITING = 0, MO_ACTIVE = 1, MO_DONE = 2 };

/* node_ctrl may be NULL (= all GREEN).  0 GREEN (case 2), 1 PRIORITY (one vehicle per node per step, smallest id),
 * 2 STOP (case 1 in full: every vehicle stands stop_time_s at the stop line, then one vehicle per
 * node per step in a round-robin over the (inbound edge, outbound edge) combinations; rule R8s of DESIGN.md). */
mo_sim *mo_create(uint32_t n_nodes, uint32_t n_edges, const uint32_t *row_ptr, const uint32_t *head,
                  const float *length_m, const uint8_t *lanes, const float *speed_limit,
                  const uint8_t *node_ctrl, const mo_params *p);
/* returns 0 or a negative error; init_pos_m / init_speed may be NULL; init_pos_m[i] < 0 = not pre-placed */
int mo_load_trips(mo_sim *S, uint32_t n_trips, const uint64_t *route_ptr, const uint32_t *route_edges,
                  const float *depart_time_s, const float *init_pos_m, const float *init_speed);
/* processing order of the per-vehicle loops: 0 id order, 1 reversed, 2 shuffled every step (pin K10) */
void mo_set_order(mo_sim *S, int mode, uint64_t seed);
int mo_step(mo_sim *S, uint32_t n_steps);
/* tests only: overwrite the dynamic state (arrays in caller trip order) and rebuild atlas + lists */
int mo_set_state(mo_sim *S, uint32_t t, const uint8_t *status, const uint32_t *route_pos, const uint8_t *lane,
                 const uint8_t *tag, const uint32_t *x_fx, const float *v, const uint32_t *admit_step,
                 const uint32_t *arrive_step, const uint32_t *edge_entries);
/* tests only: the stop-line counters of R8s (steps already stood at a STOP node on the current edge), caller order */
void mo_set_wait(mo_sim *S, const uint8_t *wait);
void mo_get_wait(const mo_sim *S, uint8_t *wait);
/* per-edge speed statistics: sum_q8[slice * n_edges + e] = sum of rint(v * 256) over the samples, samples[...] their
 * number; either may be NULL */
void mo_get_edge_speed_stats(const mo_sim *S, uint64_t *sum_q8, uint32_t *samples);
/* desired speed of vehicle `id` at route position r (R3s / G27) */
float mo_v0(const mo_sim *S, uint32_t id, uint32_t r);
/* ACTIVE vehicles standing still (v = 0) now: the "stuck count" of a gridlocked network */
uint64_t mo_n_stopped(const mo_sim *S);
void mo_destroy(mo_sim *S);

/* outputs, indexed by the CALLER's trip index; any pointer may be NULL */
void mo_get_state(const mo_sim *S, uint8_t *status, uint32_t *route_pos, uint8_t *lane, uint8_t *tag,
                  uint32_t *x_fx, float *v, float *acc_last);
void mo_get_trip_results(const mo_sim *S, uint32_t *admit_step, uint32_t *arrive_step);
void mo_get_edge_entries(const mo_sim *S, uint32_t *edge_entries);
/* summary[0]=t, [1]=n_waiting, [2]=n_active, [3]=n_done, [4]=sum travel steps, [5]=vehicle-updates,
 * [6]=lane changes executed, [7]=cells examined by R2 (sum), [8]=updates that ran R5 */
void mo_get_summary(const mo_sim *S, uint64_t summary[9]);
/* derived constants of R0: out[0]=L_c, [1]=Z_out, [2]=Z_in, [3]=LEN_MIN, [4]=L_fx, [5]=Lambda cells */
void mo_get_derived(const mo_sim *S, uint32_t out[6]);
/* vehicle id (rank in depart order) of each caller trip index */
void mo_get_vehicle_ids(const mo_sim *S, uint32_t *id_of_trip);
/* logical atlas of the current step: for every lane-cell, occ (0/1), frac10, speed; row r of edge e
 * starts at cell_off[first_row[e] + lane]; n_cells total.  Used by tests only. */
uint64_t mo_n_cells(const mo_sim *S);
void mo_get_atlas(const mo_sim *S, uint8_t *occ, uint16_t *frac, float *spd);
void mo_get_row_offsets(const mo_sim *S, uint32_t *first_row /*[n_edges]*/, uint64_t *row_off /*[n_rows]*/);
uint32_t mo_n_rows(const mo_sim *S);

/* single functions exposed for the pins */
float mo_idm_acc(const mo_sim *S, float v, float v0, int has_leader, float s, float v_lead); /* R3 */
uint32_t mo_rng(const mo_sim *S, uint32_t id, uint32_t t, uint32_t k);                       /* G22 */
float mo_eps(const mo_sim *S, uint32_t id, uint32_t t, uint32_t k0);                         /* R6 epsilon */
uint32_t mo_pmlc(const mo_sim *S, uint32_t dcell);                                           /* R0 table */

#ifdef __cplusplus
}
#endif
#endif
