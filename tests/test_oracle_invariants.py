"""Pins K6-K11: invariants, order independence, lane-change safety and brute-force intersection
conflicts of the oracle.  CPU only."""
import itertools

import numpy as np
import pytest

from paper_2007_03614_b200 import workloads as wl
from tests.helpers import (ACTIVE, DONE, WAITING, check_conservation, check_entries, check_monotone,
                           check_no_overlap, states_equal)


def small_grid_case(n=5, lanes=2, n_trips=500, horizon=300.0, ctrl=wl.PRIORITY, seed=7):
    net = wl.grid_network(nx=n, ny=n, lanes=lanes, ctrl=ctrl)
    o, d = wl.uniform_od(net, n_trips, seed)
    trips = wl.make_trips(net, o, d, wl.depart_uniform(n_trips, 0.0, horizon, seed + 1), n_threads=2)
    return net, trips


def test_K6_K7_K8_config0_full_run(oracle_mod):
    net, trips, params, n_steps = wl.config0()
    o = oracle_mod.Oracle(net, params, trips)
    L_fx = o.derived()["L_fx"]
    n = len(trips["depart_time_s"])
    prev = o.state()
    lane_changes = 0
    for k in range(n_steps // 8):
        o.step(8)
        st = o.state()
        check_conservation(st, n, o.summary())
        check_entries(st, o.edge_entries())
        check_no_overlap(net, trips, st, L_fx)
        check_monotone(prev, st)
        prev = st
    s = o.summary()
    assert s["n_done"] == n and s["n_active"] == 0 and s["n_waiting"] == 0     # everybody arrives within the hour
    assert s["lane_changes"] > 100                                             # the lane-change path is exercised
    assert s["sum_travel_steps"] == int((st["arrive_step"].astype(np.int64) - st["admit_step"]).sum())
    # per-edge counts: every route edge entered exactly once per trip
    want = np.bincount(trips["route_edges"], minlength=net["n_edges"])
    assert np.array_equal(o.edge_entries(), want)
    # free-flow lower bound on travel time: route length / limit
    rl = np.diff(trips["route_ptr"].astype(np.int64)) * 200.0
    tt = (st["arrive_step"].astype(np.int64) - st["admit_step"]) * 0.5
    assert (tt >= rl / (50 / 3.6) - 0.5).all()


def test_K8_every_step_dense_priority_grid(oracle_mod):
    net, trips = small_grid_case(n=4, lanes=2, n_trips=600, horizon=120.0)
    o = oracle_mod.Oracle(net, dict(lookahead_cells=128), trips)
    L_fx = o.derived()["L_fx"]
    prev = o.state()
    for k in range(1500):
        o.step(1)
        st = o.state()
        check_no_overlap(net, trips, st, L_fx)
        check_monotone(prev, st)
        prev = st
    check_conservation(st, 600, o.summary())


@pytest.mark.parametrize("ctrl", [wl.GREEN, wl.PRIORITY])
def test_K10_order_independence(oracle_mod, ctrl):
    net, trips = small_grid_case(n=5, lanes=3, n_trips=700, horizon=200.0, ctrl=ctrl)
    sims = []
    for mode in (0, 1, 2):
        o = oracle_mod.Oracle(net, dict(lookahead_cells=128), trips)
        o.set_order(mode, 12345)
        sims.append(o)
    for k in range(1200):
        for o in sims:
            o.step(1)
        a = sims[0].state()
        for o in sims[1:]:
            b = o.state()
            assert states_equal(a, b) == [], (k, states_equal(a, b))
            assert np.array_equal(a["acc"], b["acc"])
        if k % 100 == 0:
            assert np.array_equal(sims[0].edge_entries(), sims[2].edge_entries())
    assert sims[0].summary() == sims[1].summary() == sims[2].summary()
    assert sims[0].summary()["lane_changes"] > 0


def _lane_change_audit(oracle_mod, net, trips, params, n_steps):
    o = oracle_mod.Oracle(net, params, trips)
    d = o.derived()
    lens = np.round(net["length_m"].astype(np.float64)).astype(np.int64)
    rp = trips["route_ptr"].astype(np.int64)
    prev = o.state()
    n_changes = 0
    for t in range(n_steps):
        o.step(1)
        st = o.state()
        check_no_overlap(net, trips, st, d["L_fx"])
        both = (prev["status"] == ACTIVE) & (st["status"] == ACTIVE) & (prev["route_pos"] == st["route_pos"])
        ch = both & (prev["lane"] != st["lane"])
        if ch.any():
            idx = np.nonzero(ch)[0]
            delta = st["lane"][idx].astype(np.int64) - prev["lane"][idx].astype(np.int64)
            assert (delta == (1 if t % 2 == 0 else -1)).all(), (t, delta)        # G11: one direction per step
            c = prev["x_fx"][idx].astype(np.int64) >> 10
            e = trips["route_edges"][rp[idx] + prev["route_pos"][idx].astype(np.int64)].astype(np.int64)
            assert (c >= d["Z_in"]).all() and (c < lens[e] - d["Z_out"]).all()      # no change near the ends
            n_changes += len(idx)
        prev = st
    assert n_changes == o.summary()["lane_changes"]
    return n_changes


def test_K11_lane_change_safety_ring(oracle_mod):
    # dense multi-lane ring with heterogeneous speeds: discretionary changes only
    net = wl.ring_network(n_edges=4, edge_len=300.0, lanes=3)
    trips = wl.ring_trips(net, n_veh=150, laps_steps=6000, jitter=1.5, vmax=12.0, seed=11)
    n = _lane_change_audit(oracle_mod, net, trips, dict(lookahead_cells=128), 6000)
    assert n > 50


def test_K11_lane_change_safety_grid_mandatory(oracle_mod):
    net, trips = small_grid_case(n=4, lanes=3, n_trips=500, horizon=150.0, ctrl=wl.GREEN, seed=3)
    n = _lane_change_audit(oracle_mod, net, trips, dict(lookahead_cells=128), 2500)
    assert n > 50


@pytest.mark.slow
def test_K11_lane_change_safety_long(oracle_mod):
    net = wl.ring_network(n_edges=4, edge_len=300.0, lanes=2)
    trips = wl.ring_trips(net, n_veh=110, laps_steps=100000, jitter=1.5, vmax=12.0, seed=5)
    _lane_change_audit(oracle_mod, net, trips, dict(lookahead_cells=128), 100000)


# ----------------------------------------------------------------------------- K9
def star_network(ctrl, out_lanes=(2, 1)):
    """3 inbound edges (nodes 0,1,2 -> 3) with 2 lanes, outbound 3 -> 4 and 3 -> 5."""
    tail = np.array([0, 1, 2, 3, 3], np.int64)
    head = np.array([3, 3, 3, 4, 5], np.int64)
    net = wl._csr_from_edges(6, tail, head, length_m=np.full(5, 100.0, np.float32),
                             lanes=np.array([2, 2, 2, out_lanes[0], out_lanes[1]], np.uint8),
                             speed_limit=np.full(5, 50 / 3.6, np.float32))
    c = np.zeros(6, np.uint8)
    c[3] = ctrl
    net["node_ctrl"] = c
    return net


def run_star(oracle_mod, net, veh):
    """veh: list of (in_edge, lane, out_edge) in ID order; all sit 2 m before the node at 10 m/s."""
    n = len(veh)
    trips = dict(route_ptr=np.arange(0, 2 * n + 1, 2, dtype=np.uint64),
                 route_edges=np.array([[a, c] for a, _, c in veh], np.uint32).ravel(),
                 depart_time_s=np.zeros(n, np.float32), init_pos_m=None, init_speed=None)
    o = oracle_mod.Oracle(net, dict(lookahead_cells=64), trips)
    st = dict(status=np.full(n, ACTIVE, np.uint8), route_pos=np.zeros(n, np.uint32),
              lane=np.array([l for _, l, _ in veh], np.uint8), tag=np.zeros(n, np.uint8),
              x_fx=np.full(n, 98 * 1024 + 100, np.uint32), v=np.full(n, 10.0, np.float32),
              admit_step=np.zeros(n, np.uint32), arrive_step=np.full(n, 0xFFFFFFFF, np.uint32))
    o.set_state(0, st)
    o.step(1)
    return o.state(), o.edge_entries()


@pytest.mark.parametrize("ctrl", [wl.GREEN, wl.PRIORITY])
def test_K9_intersection_bruteforce(oracle_mod, ctrl):
    net = star_network(ctrl)
    # inbound choices: edge 0/1/2 x lane 0/1 ; outbound: edge 3 (2 lanes) or 4 (1 lane)
    slots = [(e, l) for e in (0, 1, 2) for l in (0, 1)]
    n_cases = 0
    for k in (2, 3):
        for inb in itertools.combinations(slots, k):
            for outs in itertools.product((3, 4), repeat=k):
                for perm in itertools.permutations(range(k)):
                    veh = [(inb[p][0], inb[p][1], outs[p]) for p in perm]
                    solo = [run_star(oracle_mod, net, [v])[0] for v in veh]
                    assert all(s["route_pos"][0] == 1 for s in solo)        # alone, everybody crosses
                    st, ee = run_star(oracle_mod, net, veh)
                    # expected winners: smallest id per claim word
                    words = {}
                    for i, (e, l, oe) in enumerate(veh):
                        w = "node" if ctrl == wl.PRIORITY else (oe, min(l, int(net["lanes"][oe]) - 1))
                        words.setdefault(w, i)
                    for i, (e, l, oe) in enumerate(veh):
                        w = "node" if ctrl == wl.PRIORITY else (oe, min(l, int(net["lanes"][oe]) - 1))
                        if words[w] == i:
                            for key in ("route_pos", "lane", "x_fx", "v"):
                                assert st[key][i] == solo[i][key][0], (veh, i, key)
                        else:                                                # loser holds at the stop line (G15)
                            assert st["route_pos"][i] == 0 and st["x_fx"][i] == 100 * 1024 - 1
                            assert st["v"][i] == 0.0 and st["lane"][i] == l
                    assert ee[3] + ee[4] == len(words)
                    n_cases += 1
    assert n_cases > 500


def test_K9_capacity_blocking(oracle_mod):
    """an edge whose entry is occupied admits nobody -- the follower stops behind it."""
    net = star_network(wl.GREEN, out_lanes=(1, 1))
    trips = dict(route_ptr=np.array([0, 2, 3], np.uint64), route_edges=np.array([0, 3, 3], np.uint32),
                 depart_time_s=np.zeros(2, np.float32), init_pos_m=None, init_speed=None)
    o = oracle_mod.Oracle(net, dict(lookahead_cells=64), trips)
    st = dict(status=np.full(2, ACTIVE, np.uint8), route_pos=np.zeros(2, np.uint32), lane=np.zeros(2, np.uint8),
              tag=np.zeros(2, np.uint8), x_fx=np.array([94 * 1024, 1 * 1024], np.uint32),
              v=np.array([10.0, 0.0], np.float32), admit_step=np.zeros(2, np.uint32),
              arrive_step=np.full(2, 0xFFFFFFFF, np.uint32))
    o.set_state(1, st)
    o.step(1)
    s1 = o.state()
    assert s1["route_pos"][0] == 0                                   # did not cross
    assert s1["x_fx"][0] < 100 * 1024
    # gap to the blocker (which moved a little) is kept >= L across the node
    lead_abs = 100 * 1024 + int(s1["x_fx"][1])
    assert lead_abs - int(s1["x_fx"][0]) >= 0                        # ordering kept
    # ballistic step would reach 96.5 m; the hard clamp (R7) stops it L behind the blocker's time-t position
    assert int(s1["x_fx"][0]) == 100 * 1024 + 1024 - o.derived()["L_fx"] and s1["v"][0] == 0.0


def test_admission_rules(oracle_mod):
    """R1 / G17: smallest id first, one admission per (edge, lane) per step, blocked entries wait."""
    net = wl.straight_road(n_edges=1, length_m=300.0, lanes=2)
    n = 6
    trips = dict(route_ptr=np.arange(n + 1, dtype=np.uint64), route_edges=np.zeros(n, np.uint32),
                 depart_time_s=np.zeros(n, np.float32), init_pos_m=None, init_speed=None)
    o = oracle_mod.Oracle(net, None, trips)
    o.step(1)
    st = o.state()
    # all six choose lane 0 (first free) -> only trip 0 admitted at t = 0
    assert st["status"].tolist() == [ACTIVE] + [WAITING] * 5 and st["lane"][0] == 0
    o.step(1)
    st = o.state()
    # lane 0 window still occupied -> trip 1 goes to lane 1
    assert st["status"].tolist() == [ACTIVE, ACTIVE] + [WAITING] * 4 and st["lane"][1] == 1
    assert st["admit_step"][:2].tolist() == [0, 1]
    o.step(40)
    st = o.state()
    assert (st["status"] != WAITING).all()
    adm = np.sort(st["admit_step"])
    assert (np.diff(adm) >= 0).all() and st["admit_step"].tolist() == sorted(st["admit_step"].tolist())


def test_K6_K8_config3_congestion_stress(oracle_mod):
    """configs[3] shape (lane-reduced network, doubled demand squeezed into three hours) at 1/256 scale, the
    densest 15 minutes: conservation, no overlap and monotone progress hold under spill-back, and admission is
    actually being refused (vehicles wait for a free entry window)."""
    net, trips, params, _ = wl.config3(scale=1 / 256.0, window=(4200.0, 5100.0), n_threads=2)
    n = len(trips["depart_time_s"])
    assert n > 3000
    o = oracle_mod.Oracle(net, params, trips)
    L_fx = o.derived()["L_fx"]
    prev = o.state()
    late = 0
    for k in range(60):
        o.step(40)
        st = o.state()
        check_conservation(st, n, o.summary())
        check_entries(st, o.edge_entries())
        check_no_overlap(net, trips, st, L_fx)
        check_monotone(prev, st)
        prev = st
    adm = st["status"] != WAITING
    dep_step = np.floor(trips["depart_time_s"].astype(np.float64) / 0.5).astype(np.int64)
    late = int((st["admit_step"][adm].astype(np.int64) > dep_step[adm]).sum())
    assert late > 50                      # entry windows were occupied: R1 held vehicles back
    assert o.summary()["lane_changes"] > 100


def test_config4_tiled_network_is_one_component(oracle_mod):
    """configs[4] shape: the 2 x 2 tiling is joined by seam edges, so gravity OD pairs across tiles are routable
    and vehicles do cross the seams."""
    net, trips, params, _ = wl.config4(scale=1 / 256.0, window=(9000.0, 9300.0), n_threads=2)
    n_tile = net["n_nodes"] // 4
    rp = trips["route_ptr"].astype(np.int64)
    tail = np.repeat(np.arange(net["n_nodes"]), np.diff(net["row_ptr"].astype(np.int64)))
    first_tile = tail[trips["route_edges"][rp[:-1]]] // n_tile
    last_tile = net["head"][trips["route_edges"][rp[1:] - 1]] // n_tile
    assert (first_tile != last_tile).sum() > 10
    o = oracle_mod.Oracle(net, params, trips)
    o.step(1500)
    st = o.state()
    check_conservation(st, len(trips["depart_time_s"]), o.summary())
    check_no_overlap(net, trips, st, o.derived()["L_fx"])
    assert o.summary()["n_done"] > 100
