"""Pins K1-K5, K12 and the table values: the oracle against closed forms of Eq. (1), (2)
 and a textbook IDM loop.  CPU only."""
import math
import os

import numpy as np
import pytest

from paper_2007_03614_b200 import workloads as wl

V0 = 50 / 3.6
G = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")) as f:
    for line in f:
        line = line.split("#")[0].split()
        if len(line) == 2:
            G[line[0]] = float(line[1])


def s_e(v, v0=V0, s0=2.0, T=1.5):
    return (s0 + T * v) / math.sqrt(1.0 - (v / v0) ** 4)


def solve_v_e(gap):
    lo, hi = 0.0, V0 * (1 - 1e-12)
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if s_e(mid) < gap:
            lo = mid
        else:
            hi = mid
    return lo


def single_vehicle(oracle_mod, length, v_init, n_edges=1):
    net = wl.straight_road(n_edges=n_edges, length_m=length)
    trips = dict(route_ptr=np.array([0, n_edges], np.uint64), route_edges=np.arange(n_edges, dtype=np.uint32),
                 depart_time_s=np.zeros(1, np.float32), init_pos_m=np.zeros(1, np.float32),
                 init_speed=np.array([v_init], np.float32))
    return oracle_mod.Oracle(net, None, trips)


def test_golden_values_are_the_closed_forms():
    # the stored numbers are what the formulas give (guards the fixture itself)
    for v, k in ((2, "s_e_v2"), (5, "s_e_v5"), (10, "s_e_v10"), (12, "s_e_v12")):
        assert abs(s_e(v) - G[k]) < 1e-4
    assert abs(solve_v_e(20.0) - G["v_e_ring200"]) < 1e-4
    assert abs(solve_v_e(10.0 / 3.0) - G["v_e_ring600"]) < 1e-5
    assert abs(600 / 5.0 * G["v_e_ring600"] * 3.6 - G["flow_ring600_veh_per_h"]) < 0.5
    for fr, k in ((0.5, "t_to_0.5v0"), (0.9, "t_to_0.9v0"), (0.99, "t_to_0.99v0")):
        assert abs(V0 * (0.5 * math.atanh(fr) + 0.5 * math.atan(fr)) - G[k]) < 0.006
    for d, k in ((150, "p_mlc_150m"), (200, "p_mlc_200m"), (300, "p_mlc_300m")):
        assert abs(math.exp(-(d / 100.0 - 1) ** 2) - G[k]) < 1e-6


def test_K1_free_flow_crossing(oracle_mod):
    o = single_vehicle(oracle_mod, 200.0, V0)
    xs = []
    for k in range(1, 40):
        o.step(1)
        st = o.state()
        if st["status"][0] == oracle_mod.DONE:
            assert k == int(G["k1_steps"]) and st["arrive_step"][0] == k
            break
        assert st["acc"][0] == 0.0                      # Eq. (1), s -> inf, v = v0: exactly zero
        assert st["v"][0] == np.float32(V0)
        xs.append(int(st["x_fx"][0]))
    else:
        raise AssertionError("never arrived")
    assert set(np.diff([0] + xs)) == {int(G["k1_dx_fx"])}
    assert o.summary()["sum_travel_steps"] == int(G["k1_steps"])


def test_K2_acceleration_from_rest(oracle_mod):
    o = single_vehicle(oracle_mod, 5000.0, 0.0)
    # fine reference: dv/dt = a(1-(v/v0)^4) at dt = 1e-4 in double (closed form checked in the golden test)
    vs, xs = [0.0], [0.0]
    v = x = 0.0
    h = 1e-4
    for k in range(int(60 / h)):
        a = 1.0 - (v / V0) ** 4
        x += v * h + 0.5 * a * h * h
        v += a * h
        if (k + 1) % 5000 == 0:
            vs.append(v)
            xs.append(x)
    t_cross = {}
    for k in range(1, 121):
        o.step(1)
        st = o.state()
        vk, xk = float(st["v"][0]), st["x_fx"][0] / 1024.0
        for fr in (0.5, 0.9, 0.99):
            if fr not in t_cross and vk >= fr * V0:
                t_cross[fr] = k * 0.5
        # explicit Euler on v: O(dt) error, always ahead of the exact solution by < a*dt
        assert vs[k] - 1e-4 <= vk <= vs[k] + 0.5 + 1e-4
        assert abs(xk - xs[k]) <= 0.02 * xs[k] + 0.2
    assert abs(t_cross[0.5] - G["t_to_0.5v0"]) <= 0.5
    assert abs(t_cross[0.9] - G["t_to_0.9v0"]) <= 0.75
    assert abs(t_cross[0.99] - G["t_to_0.99v0"]) <= 1.5


def test_K3_idm_equilibrium_function(oracle_mod):
    o = single_vehicle(oracle_mod, 200.0, 0.0)
    for v, k in ((2.0, "s_e_v2"), (5.0, "s_e_v5"), (10.0, "s_e_v10"), (12.0, "s_e_v12")):
        acc = o.idm_acc(v, V0, s=s_e(v), v_lead=v)
        assert abs(acc) < 2e-6, (v, acc)
        assert abs(o.idm_acc(v, V0, s=G[k], v_lead=v)) < 2e-4     # the printed 4-decimal gap
        assert o.idm_acc(v, V0, s=0.9 * s_e(v), v_lead=v) < -1e-2   # closer than s_e: brake
        assert o.idm_acc(v, V0, s=1.1 * s_e(v), v_lead=v) > 1e-2    # farther: accelerate
        assert o.idm_acc(v, V0, s=s_e(v), v_lead=v - 1.0) < -1e-2   # approaching: brake (sign of v*dv term)
        assert o.idm_acc(v, V0, s=s_e(v), v_lead=v + 1.0) > 1e-3
    assert o.idm_acc(0.0, V0) == 1.0                                   # a(1 - 0) with no leader
    assert o.idm_acc(float(np.float32(V0)), float(np.float32(V0))) == 0.0
    # dependence on b only through 1/(2 sqrt(ab)): at dv = 1, v = 10, s = 20 the interaction term is
    # ((s0 + T v + v dv/(2 sqrt(ab)))/s)^2 = ((2 + 15 + 10/2.8284)/20)^2
    want = 1.0 * (1 - (10 / V0) ** 4 - ((2 + 15 + 10 * 1.0 / (2 * math.sqrt(2.0))) / 20.0) ** 2)
    assert abs(o.idm_acc(10.0, V0, s=20.0, v_lead=9.0) - want) < 1e-5
    # guard G5: strongly receding leader cannot make the desired gap smaller than s0
    assert abs(o.idm_acc(10.0, V0, s=20.0, v_lead=30.0) - (1 - (10 / V0) ** 4 - (2.0 / 20.0) ** 2)) < 1e-6


@pytest.mark.parametrize("n_veh", [100, 150, 200])  # string-stable densities (N <= 200)
def test_K3_K4_ring_converges_to_equilibrium_gap(oracle_mod, n_veh):
    net = wl.ring_network()
    gap = 5000.0 / n_veh - 5.0
    v_e = solve_v_e(gap)
    trips = wl.ring_trips(net, n_veh=n_veh, laps_steps=6000, jitter=1.0, speeds=v_e * 0.8)
    o = oracle_mod.Oracle(net, None, trips)
    o.step(6000)
    st = o.state()
    rp = trips["route_ptr"].astype(np.int64)
    e = trips["route_edges"][rp[:-1] + st["route_pos"].astype(np.int64)].astype(np.int64)
    pos = np.sort((e * 500.0 + st["x_fx"] / 1024.0) % 5000.0)
    gaps = np.diff(np.concatenate([pos, pos[:1] + 5000.0])) - 5.0
    assert abs(gaps.sum() - (5000.0 - 5.0 * n_veh)) < 1e-6            # conservation of road length
    assert np.abs(gaps - gap).max() < 0.1, np.abs(gaps - gap).max()    # all gaps equal (2^-10 m grid dead band) ...
    assert np.abs(st["v"] - v_e).max() < 0.01                         # ... at the closed-form speed
    if n_veh == 200:
        assert abs(float(st["v"].mean()) - G["v_e_ring200"]) < 0.01
    # and (gap, v) satisfy s_e(v) = gap to 2^-10 m + fp32
    assert abs(s_e(float(st["v"].mean())) - gaps.mean()) < 0.05


def test_K5_config1_ring(oracle_mod):
    net, trips, params, n_steps = wl.config1()
    o = oracle_mod.Oracle(net, params, trips)
    L_fx = o.derived()["L_fx"]
    from tests.helpers import check_no_overlap
    v_mean = []
    for k in range(24):
        o.step(n_steps // 24)
        st = o.state()
        check_no_overlap(net, trips, st, L_fx)
        rp = trips["route_ptr"].astype(np.int64)
        e = trips["route_edges"][rp[:-1] + st["route_pos"].astype(np.int64)].astype(np.int64)
        pos = np.sort((e * 500.0 + st["x_fx"] / 1024.0) % 5000.0)
        gaps = np.diff(np.concatenate([pos, pos[:1] + 5000.0])) - 5.0
        assert abs(gaps.mean() - 10.0 / 3.0) < 1e-9                   # mean gap fixed by conservation
        assert gaps.min() >= -1e-9
        v_mean.append(float(st["v"].mean()))
    assert (st["status"] == oracle_mod.ACTIVE).all()
    # marginally string-unstable regime (growth rate +5.6e-4 1/s): within two hours the waves stay small,
    # so the space-mean speed stays within 2 % of the closed-form v_e = 0.88887 (and not above it: s_e(v) is convex,
    # so a spread of gaps around the fixed mean gap lowers the mean speed)
    assert all(0.98 * G["v_e_ring600"] < x < 1.002 * G["v_e_ring600"] for x in v_mean), v_mean


def test_K12_textbook_idm_platoon(oracle_mod):
    """One lane, GREEN, no RNG: the oracle equals a plain IDM loop (Treiber & Kesting ballistic update,
    the scheme of [27] which PAPER.md:84 cites) fed with exact gaps, up to the 2^-10 m position grid."""
    n = 12
    net = wl.straight_road(n_edges=1, length_m=4000.0)
    x0 = np.arange(n)[::-1] * 30.0 + 10.0          # vehicle 0 is the leader, farthest ahead
    v0s = np.linspace(12.0, 3.0, n)
    trips = dict(route_ptr=np.arange(n + 1, dtype=np.uint64), route_edges=np.zeros(n, np.uint32),
                 depart_time_s=np.zeros(n, np.float32), init_pos_m=x0.astype(np.float32),
                 init_speed=v0s.astype(np.float32))
    o = oracle_mod.Oracle(net, dict(lookahead_cells=512), trips)
    a, b, T, s0, L, dt = 1.0, 2.0, 1.5, 2.0, 5.0, 0.5
    x, v = x0.astype(np.float64).copy(), v0s.astype(np.float64).copy()
    for step in range(300):
        acc = np.empty(n)
        for i in range(n):
            free = (v[i] / V0) ** 4
            if i == 0:
                inter = 0.0
            else:
                s = x[i - 1] - x[i] - L
                dv = v[i] - v[i - 1]
                sstar = s0 + max(0.0, v[i] * T + v[i] * dv / (2 * math.sqrt(a * b)))
                inter = (sstar / s) ** 2
            acc[i] = a * (1 - free - inter)
        vn = np.maximum(0.0, v + acc * dt)
        x = x + 0.5 * (v + vn) * dt
        v = vn
        o.step(1)
        st = o.state()
        assert np.abs(st["v"] - v).max() < 2e-3, step
        assert np.abs(st["x_fx"] / 1024.0 - x).max() < 0.05 + 1e-3 * step, step


def test_eq2_table(oracle_mod):
    o = single_vehicle(oracle_mod, 200.0, 0.0)
    for d in (0, 1, 50, 100):
        assert o.pmlc(d) == 0xFFFFFFFF                                  # x_i <= x_0: m_i = 1
    for d, k in ((150, "p_mlc_150m"), (200, "p_mlc_200m"), (300, "p_mlc_300m")):
        assert abs(o.pmlc(d) / 2.0 ** 32 - G[k]) < 1e-6
    assert o.pmlc(501) == 0 and o.pmlc(10 ** 6) == 0
    vals = [o.pmlc(d) for d in range(100, 501)]
    assert all(x >= y for x, y in zip(vals, vals[1:]))                   # monotone decreasing in distance


def test_rng_and_epsilon(oracle_mod):
    o = single_vehicle(oracle_mod, 200.0, 0.0)
    n = 40000
    w = np.array([o.rng(i % 997, i // 997, (i * 7) % 7) for i in range(n)], dtype=np.uint64)
    # chi^2 of the top byte and of the low byte against uniform (255 dof: mean 255, sd 22.6)
    for sh in (24, 0, 11):
        h = np.bincount(((w >> np.uint64(sh)) & np.uint64(255)).astype(np.int64), minlength=256)
        chi2 = ((h - n / 256.0) ** 2 / (n / 256.0)).sum()
        assert chi2 < 255 + 5 * 22.6, (sh, chi2)
    # each argument matters
    assert len({o.rng(1, 2, 3), o.rng(2, 2, 3), o.rng(1, 3, 3), o.rng(1, 2, 4)}) == 4
    e = np.array([o.eps(i, 17, 1) for i in range(n)])
    assert abs(e.mean()) < 4 * 1.0 / math.sqrt(n)
    assert abs(e.std() - G["eps_sigma"]) < 0.02
    e2 = np.array([o.eps(i, 17, 4) for i in range(n)])
    assert abs(np.corrcoef(e, e2)[0, 1]) < 0.03                          # eps_a, eps_b independent draws
    # Irwin-Hall(12) is close to normal: P(|e| < 1) ~ 0.68
    assert abs((np.abs(e) < 1.0).mean() - 0.683) < 0.02
