"""Pins of the SURVEY 8(f) rows N1 (STOP control: "flashing red light ... round-robin of the nm
combinations", "every vehicle is designed to stop at the intersection for 2 seconds") and N2 (per-driver
desired speed; per-edge speed statistics, the inputs of Eq. 5) of the oracle.
Expected values are worked out here from the rules R8s / R3s / R9s of DESIGN.md, not taken from the oracle.  CPU only."""
import itertools
import math

import numpy as np
import pytest

from paper_2007_03614_b200 import workloads as wl
from tests.helpers import ACTIVE, DONE, check_conservation, check_entries, check_no_overlap, states_equal
from tests.test_oracle_lane_change_pins import load_mutant, rng

V0 = 50 / 3.6
STOP = 2
NONE32 = 0xFFFFFFFF


def two_edge_road(ctrl, lanes=1):
    net = wl.straight_road(n_edges=2, length_m=200.0, lanes=lanes)
    c = np.zeros(3, np.uint8)
    c[1] = ctrl
    net["node_ctrl"] = c
    return net


def one_vehicle(om, ctrl, params=None):
    trips = dict(route_ptr=np.array([0, 2], np.uint64), route_edges=np.array([0, 1], np.uint32),
                 depart_time_s=np.zeros(1, np.float32), init_pos_m=np.zeros(1, np.float32),
                 init_speed=np.array([V0], np.float32))
    return om.Oracle(two_edge_road(ctrl), params, trips)


# ------------------------------------------------------------------------------------------------- N1: STOP
def pin_stop_lone_vehicle(om):
    """K1's vehicle (free flow, 7111 units per step) into a STOP node: it reaches the end of the 200-cell edge on its
    29th step, stands at len_fx - 1 with v = 0 for exactly ceil(2 s / 0.5 s) = 4 steps, and crosses on step 33 from
    rest: acc = a = 1, v' = 0.5, dx = (0 + 0.5) / 2 * 0.5 m = 128 units -> x = 204799 + 128 - 204800 = 127."""
    o = one_vehicle(om, STOP)
    line = 200 * 1024 - 1
    for k in range(1, 34):
        o.step(1)
        st = o.state()
        if k <= 28:
            assert st["x_fx"][0] == 7111 * k and st["route_pos"][0] == 0 and st["v"][0] == np.float32(V0)
        elif k <= 32:
            assert st["x_fx"][0] == line and st["v"][0] == 0.0 and st["route_pos"][0] == 0, k
            assert st["wait"][0] == k - 28
        else:
            assert st["route_pos"][0] == 1 and st["x_fx"][0] == 127 and st["v"][0] == np.float32(0.5), k
            assert st["wait"][0] == 0
    assert o.edge_entries().tolist() == [1, 1]
    # the same vehicle through a GREEN node is on the second edge after step 29, at full speed
    g = one_vehicle(om, 0)
    g.step(29)
    st = g.state()
    assert st["route_pos"][0] == 1 and st["x_fx"][0] == 29 * 7111 - 200 * 1024 and st["v"][0] == np.float32(V0)
    # other stop times: 1 s = 2 steps, 0.7 s = 2 steps (ceil), 0 = no stop at all
    for stop_s, n_hold in ((1.0, 2), (0.7, 2), (0.0, 0), (3.0, 6)):
        o = one_vehicle(om, STOP, dict(stop_time_s=stop_s))
        o.step(28)
        held = 0
        for k in range(12):
            o.step(1)
            st = o.state()
            if st["route_pos"][0] == 1:
                break
            assert st["x_fx"][0] == line and st["v"][0] == 0.0
            held += 1
        assert held == n_hold, (stop_s, held)


def star(ctrl):
    """3 inbound edges (nodes 0, 1, 2 -> 3, two lanes each), outbound 3 -> 4 (edge 3) and 3 -> 5 (edge 4), one lane."""
    tail = np.array([0, 1, 2, 3, 3], np.int64)
    head = np.array([3, 3, 3, 4, 5], np.int64)
    net = wl._csr_from_edges(6, tail, head, length_m=np.full(5, 100.0, np.float32),
                             lanes=np.array([2, 2, 2, 1, 1], np.uint8), speed_limit=np.full(5, V0, np.float32))
    c = np.zeros(6, np.uint8)
    c[3] = ctrl
    net["node_ctrl"] = c
    return net


def run_star(om, veh, t, wait):
    """veh: (in_edge, lane, out_edge) in id order, all standing at the stop line, having stood `wait` steps."""
    n = len(veh)
    trips = dict(route_ptr=np.arange(0, 2 * n + 1, 2, dtype=np.uint64),
                 route_edges=np.array([[a, c] for a, _, c in veh], np.uint32).ravel(),
                 depart_time_s=np.zeros(n, np.float32), init_pos_m=None, init_speed=None)
    o = om.Oracle(star(STOP), dict(lookahead_cells=64), trips)
    st = dict(status=np.full(n, ACTIVE, np.uint8), route_pos=np.zeros(n, np.uint32),
              lane=np.array([l for _, l, _ in veh], np.uint8), tag=np.zeros(n, np.uint8),
              x_fx=np.full(n, 100 * 1024 - 1, np.uint32), v=np.zeros(n, np.float32),
              admit_step=np.zeros(n, np.uint32), arrive_step=np.full(n, NONE32, np.uint32),
              wait=np.full(n, wait, np.uint8))
    o.set_state(t, st)
    o.step(1)
    out = o.state()
    o.close()
    return out


def pin_stop_round_robin(om):
    """n = 3 inbound, m = 2 outbound -> 6 combinations c = in_idx * m + out_idx taking turns: at step t
    the vehicle whose combination is nearest after t (smallest (c - t) mod 6) enters the node, the others hold; two
    vehicles of one combination (two lanes of one inbound edge): the smaller id.  Brute force over 2-3 vehicles."""
    slots = [(e, l) for e in (0, 1, 2) for l in (0, 1)]
    n_cases = 0
    for k in (2, 3):
        for inb in itertools.combinations(slots, k):
            for outs in itertools.product((3, 4), repeat=k):
                for t in (0, 1, 4, 9, 14):
                    veh = [(inb[i][0], inb[i][1], outs[i]) for i in range(k)]
                    st = run_star(om, veh, t, 4)
                    rank = [((e * 2 + (oe - 3)) - t) % 6 for e, _, oe in veh]
                    win = min(range(k), key=lambda i: (rank[i], i))
                    for i in range(k):
                        if i == win:
                            assert st["route_pos"][i] == 1 and st["x_fx"][i] == 127 and st["wait"][i] == 0, (veh, t, i)
                        else:
                            assert st["route_pos"][i] == 0 and st["x_fx"][i] == 100 * 1024 - 1 and st["v"][i] == 0.0
                            assert st["wait"][i] == 4
                    n_cases += 1
    assert n_cases > 700
    # ids only break ties inside one combination: a larger id with the better turn beats a smaller id
    st = run_star(om, [(2, 0, 4), (0, 0, 3)], 0, 4)            # combinations 5 and 0 at t = 0: vehicle 1 goes
    assert st["route_pos"].tolist() == [0, 1]
    st = run_star(om, [(2, 0, 4), (0, 0, 3)], 5, 4)            # at t = 5 combination 5 is first
    assert st["route_pos"].tolist() == [1, 0]
    # vehicles that have not stood their 4 steps yet do not take part: nobody crosses, everybody counts one more step
    st = run_star(om, [(0, 0, 3), (1, 1, 4)], 3, 2)
    assert st["route_pos"].tolist() == [0, 0] and st["wait"].tolist() == [3, 3]
    # one of them done, the other not: the done one has the node to itself whatever the turn
    n = 2
    veh = [(0, 0, 3), (1, 0, 3)]
    trips = dict(route_ptr=np.arange(0, 2 * n + 1, 2, dtype=np.uint64),
                 route_edges=np.array([[a, c] for a, _, c in veh], np.uint32).ravel(),
                 depart_time_s=np.zeros(n, np.float32), init_pos_m=None, init_speed=None)
    o = om.Oracle(star(STOP), dict(lookahead_cells=64), trips)
    st = dict(status=np.full(n, ACTIVE, np.uint8), route_pos=np.zeros(n, np.uint32), lane=np.zeros(n, np.uint8),
              tag=np.zeros(n, np.uint8), x_fx=np.full(n, 100 * 1024 - 1, np.uint32), v=np.zeros(n, np.float32),
              admit_step=np.zeros(n, np.uint32), arrive_step=np.full(n, NONE32, np.uint32),
              wait=np.array([1, 4], np.uint8))
    o.set_state(0, st)
    o.step(1)
    out = o.state()
    assert out["route_pos"].tolist() == [0, 1] and out["wait"].tolist() == [2, 0]


def pin_stop_queue(om):
    """A platoon into a STOP node: every vehicle stands at least 4 steps at the line, one vehicle enters the node per
    step at most, nobody overlaps (queue spill-back)."""
    n = 6
    net = two_edge_road(STOP)
    trips = dict(route_ptr=np.arange(0, 2 * n + 1, 2, dtype=np.uint64), route_edges=np.tile([0, 1], n).astype(np.uint32),
                 depart_time_s=np.zeros(n, np.float32), init_pos_m=(150.0 - 20.0 * np.arange(n)).astype(np.float32),
                 init_speed=np.full(n, 8.0, np.float32))
    o = om.Oracle(net, None, trips)
    L_fx = o.derived()["L_fx"]
    stood = np.zeros(n, int)
    crossed_at = np.full(n, -1)
    line = 200 * 1024 - 1
    for k in range(1, 400):
        o.step(1)
        st = o.state()
        check_no_overlap(net, trips, st, L_fx)
        at_line = (st["status"] == ACTIVE) & (st["route_pos"] == 0) & (st["x_fx"] == line) & (st["v"] == 0.0)
        stood += at_line
        newly = (st["route_pos"] == 1) & (crossed_at < 0) & (st["status"] == ACTIVE)
        crossed_at[newly] = k
    assert (crossed_at > 0).all() and (stood >= 4).all(), (crossed_at, stood)
    assert (np.diff(crossed_at) >= 5).all()          # the follower reaches the line only after the leader left it


def pin_stop_grid_invariants_and_order(om):
    """K6-K8 and K10 on a grid whose nodes are all STOP: conservation, no overlap, per-edge counts, and the result does
    not depend on the processing order."""
    net = wl.grid_network(nx=4, ny=4, lanes=2, ctrl=STOP)
    o_, d_ = wl.uniform_od(net, 400, 17)
    trips = wl.make_trips(net, o_, d_, wl.depart_uniform(400, 0.0, 200.0, 18), n_threads=2)
    sims = []
    for mode in (0, 1, 2):
        o = om.Oracle(net, dict(lookahead_cells=128), trips)
        o.set_order(mode, 99)
        sims.append(o)
    L_fx = sims[0].derived()["L_fx"]
    for k in range(40):
        for o in sims:
            o.step(50)
        a = sims[0].state()
        check_no_overlap(net, trips, a, L_fx)
        check_conservation(a, 400, sims[0].summary())
        check_entries(a, sims[0].edge_entries(), trips)
        for o in sims[1:]:
            b = o.state()
            assert states_equal(a, b) == [] and np.array_equal(a["wait"], b["wait"]), k
    s = sims[0].summary()
    assert s["n_done"] > 300 and sims[0].summary() == sims[2].summary()
    # against the same demand through PRIORITY nodes: every node crossing costs at least the four steps
    p = om.Oracle(dict(net, node_ctrl=np.full(16, 1, np.uint8)), dict(lookahead_cells=128), trips)
    p.step(2000)
    ps, ss = p.state(), sims[0].state()
    both = (ps["status"] == DONE) & (ss["status"] == DONE)
    tt_p = (ps["arrive_step"].astype(np.int64) - ps["admit_step"])[both]
    tt_s = (ss["arrive_step"].astype(np.int64) - ss["admit_step"])[both]
    n_cross = (np.diff(trips["route_ptr"].astype(np.int64)) - 1)[both]
    assert both.sum() > 300 and (tt_s >= tt_p + 4 * n_cross - 1).mean() > 0.9


# ------------------------------------------------------------------------------------------------- N2: v0, statistics
def v0_factor(seed, vid, r, sigma):
    """R3s written out a second time: Irwin-Hall normal of generator words 7..9 at counter 0xFFFFFFFF - r, fp32 steps"""
    s = 0
    for k in (7, 8, 9):
        w = rng(seed, vid, 0xFFFFFFFF - r, k)
        s += (w & 255) + ((w >> 8) & 255) + ((w >> 16) & 255) + (w >> 24)
    z = np.float32(s - 1530) * np.float32(1.0 / 256.0)
    f = np.float32(1.0) + np.float32(sigma) * z
    return np.float32(min(max(f, np.float32(0.5)), np.float32(1.5)))


def pin_per_driver_v0(om):
    seed, sigma = 20070361, 0.1
    n = 64
    net = wl.straight_road(n_edges=3, length_m=2000.0, lanes=1)
    trips = dict(route_ptr=np.arange(0, 3 * n + 1, 3, dtype=np.uint64), route_edges=np.tile([0, 1, 2], n).astype(np.uint32),
                 depart_time_s=(np.arange(n) * 400.0).astype(np.float32), init_pos_m=None, init_speed=None)
    o = om.Oracle(net, dict(v0_sigma_rel=sigma, seed=seed), trips)
    lim = np.float32(V0)
    f = np.array([[v0_factor(seed, i, r, sigma) for r in range(3)] for i in range(n)])
    for i in range(n):
        for r in range(3):
            assert np.float32(o.v0(i, r)) == lim * f[i, r], (i, r)
    assert abs(f.mean() - 1.0) < 0.03 and abs(f.std() - sigma) < 0.02 and f.min() >= 0.5 and f.max() <= 1.5
    assert abs(np.corrcoef(f[:, 0], f[:, 1])[0, 1]) < 0.35          # a new draw on every edge
    # a lone driver on an empty road settles at ITS desired speed: free-road equilibrium of Eq. 1 is v = v0
    o.step(200)                                                     # vehicle 0 left at t = 0, nobody else yet
    st = o.state()
    assert st["status"][0] == ACTIVE and st["route_pos"][0] == 0
    assert abs(float(st["v"][0]) - float(lim * f[0, 0])) < 2e-3
    # a huge sigma is clamped to [limit / 2, 3 limit / 2]
    o2 = om.Oracle(net, dict(v0_sigma_rel=5.0, seed=seed), trips)
    fs = np.array([o2.v0(i, 0) / float(lim) for i in range(n)])
    assert fs.min() >= 0.5 - 1e-6 and fs.max() <= 1.5 + 1e-6 and (np.abs(fs - 0.5) < 1e-6).any() and (np.abs(fs - 1.5) < 1e-6).any()
    # sigma = 0: v0 is the limit, bit for bit
    o3 = om.Oracle(net, dict(v0_sigma_rel=0.0), trips)
    assert all(np.float32(o3.v0(i, r)) == lim for i in range(4) for r in range(3))


def pin_edge_speed_statistics(om):
    """Eq. 5 inputs: per edge and time slice, the sum and number of sampled vehicle speeds.  K1's
    vehicle at constant v0 = 13.8889 m/s: rint(v0 * 256) = 3556 per sample; samples at t = 0, 4, 8, ...; 200-cell
    edges are left after 29 steps (t = 28 is the last step spent on edge 0, so samples t = 0..28 -> 8 on edge 0)."""
    p = dict(stat_period_steps=4, stat_slice_steps=20, stat_n_slices=3)
    net = wl.straight_road(n_edges=2, length_m=200.0)
    trips = dict(route_ptr=np.array([0, 2], np.uint64), route_edges=np.array([0, 1], np.uint32),
                 depart_time_s=np.zeros(1, np.float32), init_pos_m=np.zeros(1, np.float32),
                 init_speed=np.array([V0], np.float32))
    o = om.Oracle(net, p, trips)
    o.step(57)                                            # arrives on step 58 (2 * 28.8 = 57.6)
    assert o.state()["status"][0] == ACTIVE
    sm, cn = o.edge_speed_stats()
    q = int(round(float(np.float32(V0)) * 256.0))
    assert q == 3556
    # sampled steps 0, 4, ..., 56; on edge 0 while t <= 28, then on edge 1; slices of 20 steps
    want = np.zeros((3, 2), int)
    for t in range(0, 57, 4):
        want[t // 20, 0 if t <= 28 else 1] += 1
    assert cn.tolist() == want.tolist() and sm.tolist() == (want * q).tolist()
    o.step(10)
    assert o.state()["status"][0] == DONE
    sm2, cn2 = o.edge_speed_stats()
    assert np.array_equal(cn2, cn)                        # nothing is sampled after the trip ended
    # mean speed per edge = sum / (256 * samples)
    assert abs(sm[0, 0] / 256.0 / cn[0, 0] - V0) < 2e-3
    # off by default
    o = om.Oracle(net, None, trips)
    o.step(20)
    assert o.edge_speed_stats()[1].size == 0
    # a decelerating platoon: the statistics equal the speeds read back at the sampled steps
    n = 5
    trips = dict(route_ptr=np.arange(0, 2 * n + 1, 2, dtype=np.uint64), route_edges=np.tile([0, 1], n).astype(np.uint32),
                 depart_time_s=np.zeros(n, np.float32), init_pos_m=(120.0 - 25.0 * np.arange(n)).astype(np.float32),
                 init_speed=np.linspace(2.0, 12.0, n).astype(np.float32))
    o = om.Oracle(net, dict(stat_period_steps=3, stat_slice_steps=1000, stat_n_slices=1), trips)
    tot = np.zeros(2, np.int64)
    cnt = np.zeros(2, np.int64)
    for t in range(60):
        if t % 3 == 0:
            st = o.state()
            for i in np.nonzero(st["status"] == ACTIVE)[0]:
                tot[st["route_pos"][i]] += int(np.rint(np.float32(st["v"][i]) * np.float32(256.0)))
                cnt[st["route_pos"][i]] += 1
        o.step(1)
    sm, cn = o.edge_speed_stats()
    assert cn[0].tolist() == cnt.tolist() and sm[0].tolist() == tot.tolist()


def pin_stuck_count(om):
    """summary.n_stopped = ACTIVE vehicles with v = 0 (the stuck count of a gridlocked network)."""
    o = one_vehicle(om, STOP)
    o.step(28)
    assert o.summary()["n_stopped"] == 0
    o.step(2)
    assert o.summary()["n_stopped"] == 1 and o.summary()["n_active"] == 1
    o.step(4)
    assert o.summary()["n_stopped"] == 0


PINS = [pin_stop_lone_vehicle, pin_stop_round_robin, pin_stop_queue, pin_stop_grid_invariants_and_order,
        pin_per_driver_v0, pin_edge_speed_statistics, pin_stuck_count]


@pytest.mark.parametrize("pin", PINS, ids=[p.__name__ for p in PINS])
def test_pin(oracle_mod, pin):
    pin(oracle_mod)


MUTATIONS = [
    ("one stop step too many", "if (S->ctrl[u] == 2 && S->wait[id] < S->W_stop) {", "if (S->ctrl[u] == 2 && S->wait[id] <= S->W_stop) {"),
    ("stop time rounded down", "S->W_stop = (uint32_t)ceil((double)p->stop_time_s / (double)p->dt - 1e-9);",
     "S->W_stop = (uint32_t)floor((double)p->stop_time_s / (double)p->dt);"),
    ("round-robin turns the other way", "uint32_t rank = (c + nm - S->t % nm) % nm;", "uint32_t rank = (c + S->t % nm) % nm;"),
    ("combination index by in-degree", "uint32_t c = S->in_idx[e] * m + (en - S->row_ptr[u]);",
     "uint32_t c = S->in_idx[e] * S->indeg[u] + (en - S->row_ptr[u]);"),
    ("id before turn", "key = ((uint64_t)rank << 32) | id;", "key = ((uint64_t)id << 32) | rank;"),
    ("stop counter kept across the node", "            S->wait[id] = 0;\n            S->edge_entries[en] += 1;", "            S->edge_entries[en] += 1;"),
    ("held vehicle keeps its speed", "            S->v[id] = 0.0f;\n            S->wait[id] += 1;", "            S->wait[id] += 1;"),
    ("v0 clamp dropped", "    f = fmaxf(f, 0.5f);\n    f = fminf(f, 1.5f);", ""),
    ("one v0 draw per driver instead of per edge", "rng32(S->p.seed, id, 0xFFFFFFFFu - r, k);", "rng32(S->p.seed, id, 0xFFFFFFFFu, k);"),
    ("statistics sample every step", "if (S->stat_sum && S->t % p->stat_period_steps == 0u) {", "if (S->stat_sum) {"),
    ("statistics in the wrong slice", "uint32_t slice = S->t / p->stat_slice_steps;", "uint32_t slice = S->t / p->stat_period_steps;"),
    ("speed truncated instead of rounded", "(uint64_t)lrintf(v * 256.0f);", "(uint64_t)(v * 256.0f);"),
]


def test_mutations_of_the_oracle_fail_a_pin(tmp_path, oracle_mod):
    survivors = []
    for idx, (name, old, new) in enumerate(MUTATIONS):
        m = load_mutant(tmp_path, idx, old, new)
        killed = False
        for pin in PINS:
            try:
                pin(m)
            except AssertionError:
                killed = True
                break
        if not killed:
            survivors.append(name)
    assert not survivors, "mutations that pass every pin: %s" % survivors
