"""Pins of six conventions of the oracle that no other pin held ("What's weak" 1): each is a
[proposed] reading of DESIGN.md section 3 with a hand-computed case here, and each comes with the mutation of
oracle/manta_oracle.c it must kill.  CPU only.

  pin_clamped_speed_is_distance_over_dt   R7: a vehicle stopped short by the no-overlap clamp leaves the
                                          step with v' = min(v', (x' - x) / dt)
  pin_dx_rounds_to_nearest_even           R7: dx = rint(m * 1024), ties to even
  pin_entry_window_is_L_c_plus_one_cells  R1: admission needs cells [0, L_c] of the lane empty
  pin_gap_floor_is_one_centimetre         R3: Eq. 1 is evaluated with max(s, 0.01 m)
  pin_depart_step_is_floor                R0: depart_step = floor(depart_time_s / dt)
  pin_vehicle_id_is_departure_rank        R0 / SURVEY 8(b): id = rank in (depart_step, caller index) order, and that id is
                                          the priority at a PRIORITY node
"""
import numpy as np
import pytest

from paper_2007_03614_b200 import workloads as wl
from tests.test_oracle_lane_change_pins import load_mutant


def preplaced(oracle_mod, length, xs, vs, limit=50 / 3.6, params=None, extra_departures=()):
    """one single-lane edge; vehicles pre-placed at xs with speeds vs (+ trips that depart later from cell 0)"""
    n0, n1 = len(xs), len(extra_departures)
    net = wl.straight_road(n_edges=1, length_m=length, limit=limit)
    trips = dict(route_ptr=np.arange(n0 + n1 + 1, dtype=np.uint64), route_edges=np.zeros(n0 + n1, np.uint32),
                 depart_time_s=np.array([0.0] * n0 + list(extra_departures), np.float32),
                 init_pos_m=np.array(list(xs) + [-1.0] * n1, np.float32),
                 init_speed=np.array(list(vs) + [0.0] * n1, np.float32))
    return oracle_mod.Oracle(net, params, trips)


def pin_clamped_speed_is_distance_over_dt(m):
    # a = 0.1 m/s^2 makes Eq. 1 brake too weakly, so the hard clamp of R7 acts.  Follower at 100 m, leader at 107 m,
    # both 10 m/s, L = 5 m: s = 2 m.  v0 = 50/3.6: free = (10 / 13.889)^4 = 0.26874; s* = s0 + T v = 17 (dv = 0);
    # inter = (17 / 2)^2 = 72.25; acc = 0.1 (1 - 0.26874 - 72.25) = -7.1519; v' = 10 - 3.576 = 6.424;
    # dx = (10 + 6.424) / 2 * 0.5 = 4.106 m > s: clamped to x' = x + 2 m, and v' = min(6.424, 2 m / 0.5 s) = 4 exactly.
    o = preplaced(m, 500.0, [100.0, 107.0], [10.0, 10.0], params=dict(a=0.1))
    o.step(1)
    st = o.state()
    assert int(st["x_fx"][0]) == 100 * 1024 + 2048
    assert abs(float(st["acc"][0]) - (-7.1519)) < 1e-3          # the case is the one computed above
    assert float(st["v"][0]) == 4.0, float(st["v"][0])


def pin_dx_rounds_to_nearest_even(m):
    # one free vehicle at v = v0: acc = 0 exactly, m = (v + v) * dt / 2 = v / 2, dx = rint(512 v) (all exact in fp32)
    for v, dx in ((10.0 + 3.0 / 2048.0, 5121),      # 5120.75 -> 5121 (truncation: 5120)
                  (10.0 + 1.0 / 1024.0, 5120),      # 5120.5  -> 5120, the even neighbour (half-up: 5121)
                  (10.0 + 3.0 / 1024.0, 5122)):     # 5121.5  -> 5122, the even neighbour (truncation: 5121)
        assert float(np.float32(v)) == v
        o = preplaced(m, 400.0, [50.0], [v], limit=v)
        o.step(1)
        st = o.state()
        assert float(st["acc"][0]) == 0.0 and float(st["v"][0]) == v
        assert int(st["x_fx"][0]) - 50 * 1024 == dx, (v, int(st["x_fx"][0]) - 50 * 1024)


def pin_entry_window_is_L_c_plus_one_cells(m):
    # L = 5 m: L_c = 5, the window is cells 0..5.  A vehicle standing in cell 6 leaves it free: admitted at step 0.
    o = preplaced(m, 300.0, [6.0], [0.0], extra_departures=[0.0])
    o.step(1)
    assert int(o.state()["admit_step"][1]) == 0
    # Standing in cell 5 (the window's last cell) it blocks.  From rest with a = 1, dt = 0.5 the blocker moves
    # 0.125, 0.375, 0.625 m in its first three steps: 5.125, 5.5 (cell 5), 6.125 (cell 6) => admission at step 3.
    o = preplaced(m, 300.0, [5.0], [0.0], extra_departures=[0.0])
    o.step(3)
    st = o.state()
    assert int(st["status"][1]) == m.WAITING and [int(x) for x in (st["x_fx"][0],)] == [5 * 1024 + 128 + 384 + 640]
    o.step(1)
    assert int(o.state()["admit_step"][1]) == 3


def pin_gap_floor_is_one_centimetre(m):
    # v = v_lead = 0: s* = s0 = 2 m; gap floor 0.01 m: z = 200, acc = a (1 - 0 - 40000) = -39999 (a = 1), for every s <= 0.01
    o = preplaced(m, 300.0, [10.0], [0.0])
    v0 = float(np.float32(50 / 3.6))
    assert o.idm_acc(0.0, v0, 0.005, 0.0) == -39999.0
    assert o.idm_acc(0.0, v0, 0.0, 0.0) == -39999.0
    assert o.idm_acc(0.0, v0, -3.0, 0.0) == -39999.0          # (overlap: the floor, not a negative gap)
    assert o.idm_acc(0.0, v0, 0.02, 0.0) == -9999.0           # above the floor: z = 100
    assert o.idm_acc(0.0, v0, 0.1, 0.0) == -399.0


def pin_depart_step_is_floor(m):
    # dt = 0.5: 0.7 s -> step 1 (ceil: 2); 0.49 s -> 0; 1.0 s -> 2; 1.2 s -> 2 (ceil: 3).  Own origin edges: no queueing.
    times = [0.7, 0.49, 1.0, 1.2]
    n = len(times)
    net = dict(n_nodes=2 * n, n_edges=n, row_ptr=np.repeat(np.arange(n + 1, dtype=np.uint32), 2)[1:], head=np.arange(1, 2 * n, 2, dtype=np.uint32),
               length_m=np.full(n, 100.0, np.float32), lanes=np.ones(n, np.uint8), speed_limit=np.full(n, 10.0, np.float32))
    assert net["row_ptr"].tolist() == [0, 1, 1, 2, 2, 3, 3, 4, 4][:2 * n + 1]
    trips = dict(route_ptr=np.arange(n + 1, dtype=np.uint64), route_edges=np.arange(n, dtype=np.uint32),
                 depart_time_s=np.array(times, np.float32))
    o = m.Oracle(net, None, trips)
    o.step(5)
    assert o.state()["admit_step"].tolist() == [1, 0, 2, 2]


def merge_network(len_a, len_b):
    """0 -> 2 (edge 0), 1 -> 2 (edge 1), 2 -> 3 (edge 2); node 2 is a PRIORITY node: one vehicle per step"""
    return dict(n_nodes=4, n_edges=3, row_ptr=np.array([0, 1, 2, 3, 3], np.uint32), head=np.array([2, 2, 3], np.uint32),
                length_m=np.array([len_a, len_b, 300.0], np.float32), lanes=np.ones(3, np.uint8),
                speed_limit=np.full(3, 10.0, np.float32), node_ctrl=np.array([0, 0, 1, 0], np.uint8))


def pin_vehicle_id_is_departure_rank(m):
    # ids: rank in (depart_step, caller index); trips given in reverse order of departure, two of them in one step
    net = merge_network(200.0, 200.0)
    trips = dict(route_ptr=np.array([0, 2, 4, 6, 8], np.uint64), route_edges=np.array([0, 2, 1, 2, 0, 2, 1, 2], np.uint32),
                 depart_time_s=np.array([30.0, 10.2, 20.0, 10.0], np.float32))        # steps 60, 20, 40, 20
    assert m.Oracle(net, None, trips).vehicle_ids().tolist() == [3, 0, 2, 1]
    # and that id is the priority: trip 1 leaves 2 s BEFORE trip 0 on an approach 22 m longer, so both
    # reach node 2 in the same step (cruising at 10 m/s = 5 m per step; 4 steps = 20 m).  Trip 1, the earlier
    # departure with the LARGER caller index, passes; trip 0 holds at the stop line with v = 0.
    net = merge_network(200.0, 222.0)
    trips = dict(route_ptr=np.array([0, 2, 4], np.uint64), route_edges=np.array([0, 2, 1, 2], np.uint32),
                 depart_time_s=np.array([2.0, 0.0], np.float32))
    o = m.Oracle(net, None, trips)
    assert o.vehicle_ids().tolist() == [1, 0]
    for _ in range(80):
        before = o.state()
        o.step(1)
        st = o.state()
        if (st["route_pos"] > 0).any():
            break
    assert before["route_pos"].tolist() == [0, 0] and (before["status"] == m.ACTIVE).all()
    # both were at the node in this step: whoever did not pass was stopped at the last position of its edge
    stop_line = {0: 200 * 1024 - 1, 1: 222 * 1024 - 1}
    loser = int(np.argmin(st["route_pos"]))
    assert int(st["x_fx"][loser]) == stop_line[loser] and float(st["v"][loser]) == 0.0
    assert float(before["v"][loser]) > 9.9                     # (it was cruising: only the lost claim stops it there)
    assert st["route_pos"].tolist() == [0, 1], st["route_pos"].tolist()


PINS = [pin_clamped_speed_is_distance_over_dt, pin_dx_rounds_to_nearest_even, pin_entry_window_is_L_c_plus_one_cells,
        pin_gap_floor_is_one_centimetre, pin_depart_step_is_floor, pin_vehicle_id_is_departure_rank]


@pytest.mark.parametrize("pin", PINS, ids=[p.__name__ for p in PINS])
def test_pin(oracle_mod, pin):
    pin(oracle_mod)


# (name, text in oracle/manta_oracle.c, replacement, the pin that must fail): the six mistakes that passed every pin of round 2
MUTATIONS = [
    ("speed of a clamped vehicle not reduced", "vn = fminf(vn, vc);", ";", pin_clamped_speed_is_distance_over_dt),
    ("dx truncated instead of rounded", "(int32_t)lrintf(m * 1024.0f);", "(int32_t)(m * 1024.0f);", pin_dx_rounds_to_nearest_even),
    ("dx rounded half up", "(int32_t)lrintf(m * 1024.0f);", "(int32_t)floorf(m * 1024.0f + 0.5f);", pin_dx_rounds_to_nearest_even),
    ("entry window one cell short", "c <= S->L_c;", "c < S->L_c;", pin_entry_window_is_L_c_plus_one_cells),
    ("gap floor 0.1 m", "fmaxf(s, 0.01f)", "fmaxf(s, 0.1f)", pin_gap_floor_is_one_centimetre),
    ("depart_step rounded up", "floor((double)depart_time_s[i] / (double)S->p.dt)", "ceil((double)depart_time_s[i] / (double)S->p.dt)", pin_depart_step_is_floor),
    ("vehicle ids in caller order", "if (x->key != y->key) return x->key < y->key ? -1 : 1;", "", pin_vehicle_id_is_departure_rank),
]


def test_mutations_of_the_oracle_fail_their_pin(tmp_path, oracle_mod):
    survivors = []
    for idx, (name, old, new, pin) in enumerate(MUTATIONS):
        m = load_mutant(tmp_path, 100 + idx, old, new)
        try:
            pin(m)
            survivors.append(name)
        except AssertionError:
            pass
    assert not survivors, "mutations that pass the pin written for them: %s" % survivors
