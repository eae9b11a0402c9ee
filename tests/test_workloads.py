"""Seeded synthetic inputs: determinism, structural validity and the shapes BASELINE.json
names.  No simulator arithmetic here; CPU only."""
import numpy as np
import pytest

from paper_2007_03614_b200 import workloads as wl

MPH = 0.44704


def check_network(net):
    n, m = net["n_nodes"], net["n_edges"]
    rp = net["row_ptr"].astype(np.int64)
    assert rp[0] == 0 and rp[-1] == m and (np.diff(rp) >= 0).all() and len(rp) == n + 1
    assert (net["head"] < n).all()
    assert (net["lanes"] >= 1).all() and (net["lanes"] <= 8).all()
    assert (net["length_m"] >= 20.0).all() and (net["speed_limit"] > 0).all()


def check_routes(net, trips):
    rp = trips["route_ptr"].astype(np.int64)
    re_ = trips["route_edges"].astype(np.int64)
    assert (np.diff(rp) >= 1).all()
    tail = np.repeat(np.arange(net["n_nodes"]), np.diff(net["row_ptr"].astype(np.int64)))
    inner = np.ones(len(re_), bool)
    inner[rp[1:-1] - 1] = False        # last entry of every trip but the last
    inner[-1] = False
    k = np.nonzero(inner)[0]
    assert (net["head"][re_[k]] == tail[re_[k + 1]]).all()          # consecutive route edges are connected


def test_generators_are_deterministic():
    a = wl.config2(scale=1 / 256.0, n_threads=2)
    b = wl.config2(scale=1 / 256.0, n_threads=1)
    for k in ("row_ptr", "head", "length_m", "lanes", "speed_limit"):
        assert np.array_equal(a[0][k], b[0][k]), k
    for k in ("route_ptr", "route_edges", "depart_time_s"):
        assert np.array_equal(a[1][k], b[1][k]), k


def test_config0_and_config1_shapes():
    net, trips, params, n_steps = wl.config0()
    check_network(net)
    check_routes(net, trips)
    assert (net["n_nodes"], net["n_edges"], n_steps) == (100, 360, 7200)
    assert len(trips["depart_time_s"]) == 2000 and trips["depart_time_s"].max() < 900.0
    assert (net["lanes"] == 2).all() and np.allclose(net["length_m"], 200.0) and np.allclose(net["speed_limit"], 50 / 3.6)
    net, trips, params, n_steps = wl.config1()
    assert net["n_edges"] == 10 and np.isclose(net["length_m"].sum(), 5000.0) and n_steps == 14400
    assert len(trips["init_pos_m"]) == 600 and (trips["init_speed"] >= 0).all() and (trips["init_speed"] <= 15.0).all()
    pos = np.sort(trips["init_pos_m"].astype(np.float64) + 500.0 * trips["route_edges"][trips["route_ptr"][:-1].astype(np.int64)])
    assert np.abs(np.diff(pos) - 5000.0 / 600).max() <= 2.0 + 1e-3            # even spacing with +/- 1 m jitter


def test_config2_shape_at_reduced_scale():
    net, trips, params, n_steps = wl.config2(scale=1 / 16.0, n_threads=4)
    check_network(net)
    check_routes(net, trips)
    assert params["lookahead_cells"] == 256 and n_steps == 50400
    assert 0.8 * 224000 / 16 < net["n_nodes"] < 1.2 * 224000 / 16
    assert 2.2 < net["n_edges"] / net["n_nodes"] < 2.8                           # ~ 550 k / 224 k directed edges per node
    share = np.bincount(net["lanes"], minlength=6)[1:6] / net["n_edges"]
    assert 0.5 < share[0] < 0.7 and 0.15 < share[1] < 0.35 and share[3] + share[4] < 0.1
    assert 100.0 < np.median(net["length_m"]) < 140.0                            # lognormal, median 120 m
    lim = net["speed_limit"] / MPH
    assert lim.min() >= 24.9 and lim.max() <= 65.1
    dep = trips["depart_time_s"].astype(np.float64) / 3600.0 + 5.0
    assert dep.min() >= 5.0 and dep.max() < 12.0
    hist = np.histogram(dep, bins=np.arange(5.0, 12.5, 0.5))[0]
    assert hist.argmax() in (4, 5, 6, 7) and hist[5] > 3 * hist[0]              # peak 07:00-09:00, far above 05:00
    km = np.add.reduceat(net["length_m"][trips["route_edges"]].astype(np.float64), trips["route_ptr"][:-1].astype(np.int64)) / 1000.0
    assert 3.0 < np.median(km) < 10.0                                             # median ~ 6.5 km


def test_config3_and_config4_shapes():
    base = wl.config2(scale=1 / 64.0, n_threads=4)[0]
    net3, trips3, _, n3 = wl.config3(scale=1 / 64.0, n_threads=4)
    check_network(net3)
    check_routes(net3, trips3)
    assert n3 == 43200 and net3["n_edges"] == base["n_edges"]
    multi = base["lanes"] >= 2
    cut = (net3["lanes"] == 1) & multi
    assert 0.15 < cut.sum() / multi.sum() < 0.25 and np.array_equal(net3["lanes"][~multi], base["lanes"][~multi])
    assert len(trips3["depart_time_s"]) == 100000 and trips3["depart_time_s"].max() < 3 * 3600.0
    net4, trips4, _, n4 = wl.config4(scale=1 / 64.0, n_threads=4)
    check_network(net4)
    check_routes(net4, trips4)
    assert n4 == 50400 and net4["n_nodes"] == 4 * base["n_nodes"] and net4["n_edges"] > 4 * base["n_edges"]
    assert len(trips4["depart_time_s"]) == 200000
