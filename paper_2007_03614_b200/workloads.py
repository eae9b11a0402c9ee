"""Seeded synthetic workload generators (networks, demand, routes) for the MANTA hot path.

These stand in for the paper's OSM network, MTC demand (47-51), departure-time law
(67) and routed trips (55-57), none of which are in the container; shapes follow BASELINE.json
`configs` and SURVEY.md section 8(d).  This module holds NONE of the simulator's arithmetic: it only makes
inputs, and is the one module that serves both the CUDA path and the oracle tests.

net   = dict(n_nodes, n_edges, row_ptr u32[n_nodes+1], head u32, length_m f32, lanes u8,
             speed_limit f32, node_ctrl u8 | None, [xy f32[n_nodes,2]])   edges are CSR-ordered by tail node
trips = dict(route_ptr u64[n+1], route_edges u32, depart_time_s f32[n], init_pos_m f32[n] | None,
             init_speed f32[n] | None)
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_RSRC = os.path.join(_HERE, "csrc", "workload_routing.c")
_RSO = os.path.join(_HERE, "libmanta_workloads.so")

MPH = 0.44704
SEED_NET, SEED_DEMAND, SEED_JITTER = 20070361, 20070362, 20070363
GREEN, PRIORITY = 0, 1


def build_routing(force=False):
    if not force and os.path.exists(_RSO) and os.path.getmtime(_RSO) >= os.path.getmtime(_RSRC):
        return _RSO
    subprocess.check_call(["gcc", "-O2", "-Wall", "-shared", "-fPIC", "-pthread", "-o", _RSO, _RSRC])
    return _RSO


_rlib = None


def _routing_lib():
    global _rlib
    if _rlib is None:
        L = C.CDLL(build_routing())
        L.wl_route_trips.restype = C.c_int
        L.wl_route_trips.argtypes = [C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p,
                                     C.c_void_p, C.c_int, C.c_void_p, C.POINTER(C.c_void_p)]
        L.wl_free.argtypes = [C.c_void_p]
        _rlib = L
    return _rlib


def route_trips(net, origin, dest, weight=None, n_threads=None):
    """Shortest routes (edge sequences) for node pairs; weight defaults to free-flow time length/limit."""
    L = _routing_lib()
    origin = np.ascontiguousarray(origin, np.uint32)
    dest = np.ascontiguousarray(dest, np.uint32)
    if weight is None:
        weight = net["length_m"].astype(np.float64) / net["speed_limit"].astype(np.float64)
    weight = np.ascontiguousarray(weight, np.float64)
    n = len(origin)
    rp = np.zeros(n + 1, np.uint64)
    out = C.c_void_p()
    if n_threads is None:
        n_threads = max(1, min(64, os.cpu_count() or 1))
    row_ptr = np.ascontiguousarray(net["row_ptr"], np.uint32)
    head = np.ascontiguousarray(net["head"], np.uint32)
    rc = L.wl_route_trips(int(net["n_nodes"]), row_ptr.ctypes.data, head.ctypes.data, weight.ctypes.data, n,
                          origin.ctypes.data, dest.ctypes.data, int(n_threads), rp.ctypes.data, C.byref(out))
    total = int(rp[-1])
    edges = np.ctypeslib.as_array(C.cast(out, C.POINTER(C.c_uint32)), shape=(max(total, 1),))[:total].copy()
    L.wl_free(out)
    if rc != 0:
        raise ValueError("route_trips: some destination is unreachable")
    return rp, edges


# ----------------------------------------------------------------------------- networks
def _csr_from_edges(n_nodes, tail, head, **attrs):
    order = np.lexsort((head, tail))
    tail, head = tail[order], head[order]
    row_ptr = np.zeros(n_nodes + 1, np.uint32)
    np.add.at(row_ptr, tail + 1, 1)
    row_ptr = np.cumsum(row_ptr).astype(np.uint32)
    net = dict(n_nodes=int(n_nodes), n_edges=int(len(head)), row_ptr=row_ptr, head=head.astype(np.uint32),
               tail=tail.astype(np.uint32))
    for k, v in attrs.items():
        net[k] = v[order]
    return net


def straight_road(n_edges=1, length_m=200.0, lanes=1, limit=50 / 3.6, ctrl=GREEN):
    """A chain of n_edges edges: node 0 -> 1 -> ... (closed forms K1-K3, K12)."""
    tail = np.arange(n_edges, dtype=np.int64)
    head = tail + 1
    net = _csr_from_edges(n_edges + 1, tail, head,
                          length_m=np.full(n_edges, length_m, np.float32),
                          lanes=np.full(n_edges, lanes, np.uint8),
                          speed_limit=np.full(n_edges, limit, np.float32))
    net["node_ctrl"] = np.full(n_edges + 1, ctrl, np.uint8)
    return net


def grid_network(nx=10, ny=10, edge_len=200.0, lanes=2, limit=50 / 3.6, ctrl=PRIORITY):
    """configs[0]: nx x ny lattice, both directions, uniform attributes."""
    idx = np.arange(nx * ny).reshape(ny, nx)
    a = np.concatenate([idx[:, :-1].ravel(), idx[:-1, :].ravel()])
    b = np.concatenate([idx[:, 1:].ravel(), idx[1:, :].ravel()])
    tail = np.concatenate([a, b]).astype(np.int64)
    head = np.concatenate([b, a]).astype(np.int64)
    m = len(tail)
    net = _csr_from_edges(nx * ny, tail, head, length_m=np.full(m, edge_len, np.float32),
                          lanes=np.full(m, lanes, np.uint8), speed_limit=np.full(m, limit, np.float32))
    net["node_ctrl"] = np.full(nx * ny, ctrl, np.uint8)
    yy, xx = np.divmod(np.arange(nx * ny), nx)
    net["xy"] = np.stack([xx * edge_len, yy * edge_len], 1).astype(np.float32)
    return net


def ring_network(n_edges=10, edge_len=500.0, limit=50 / 3.6, lanes=1):
    """configs[1]: a one-way ring of n_edges edges."""
    tail = np.arange(n_edges, dtype=np.int64)
    head = (tail + 1) % n_edges
    net = _csr_from_edges(n_edges, tail, head, length_m=np.full(n_edges, edge_len, np.float32),
                          lanes=np.full(n_edges, lanes, np.uint8), speed_limit=np.full(n_edges, limit, np.float32))
    net["node_ctrl"] = np.zeros(n_edges, np.uint8)
    return net


def ring_trips(net, n_veh=600, laps_steps=14400, dt=0.5, seed=SEED_JITTER, jitter=1.0, vmax=15.0,
               speeds=None):
    """configs[1]: n_veh vehicles pre-placed at k*(C/n) + U(-jitter, jitter), speeds U(0, vmax), routes that
    cycle the ring long enough for laps_steps steps at the speed limit."""
    rng = np.random.default_rng(seed)
    n_e = net["n_edges"]
    el = float(net["length_m"][0])
    circ = n_e * el
    pos = (np.arange(n_veh) * (circ / n_veh) + rng.uniform(-jitter, jitter, n_veh)) % circ
    pos = np.sort(pos)
    v = rng.uniform(0.0, vmax, n_veh) if speeds is None else np.full(n_veh, speeds, np.float64)
    e0 = np.minimum((pos // el).astype(np.int64), n_e - 1)
    x0 = pos - e0 * el
    n_route = int(np.ceil(float(net["speed_limit"][0]) * dt * laps_steps / el)) + 3
    # edge ids equal tail ids on the ring (CSR order), successor of edge e is (e+1) % n_e
    routes = (e0[:, None] + np.arange(n_route)[None, :]) % n_e
    rp = (np.arange(n_veh + 1, dtype=np.uint64) * np.uint64(n_route))
    return dict(route_ptr=rp, route_edges=routes.astype(np.uint32).ravel(), depart_time_s=np.zeros(n_veh, np.float32),
                init_pos_m=x0.astype(np.float32), init_speed=v.astype(np.float32))


def _largest_component(n, a, b):
    """labels of the largest connected component of an undirected graph (a[i]-b[i]); iterative union-find."""
    parent = np.arange(n, dtype=np.int64)
    # pointer-jumping label propagation (numpy-vectorised)
    while True:
        pa, pb = parent[a], parent[b]
        lo = np.minimum(pa, pb)
        changed = False
        newp = parent.copy()
        np.minimum.at(newp, pa, lo)
        np.minimum.at(newp, pb, lo)
        for _ in range(64):
            nn = newp[newp]
            if np.array_equal(nn, newp):
                break
            newp = nn
        changed = not np.array_equal(newp, parent)
        parent = newp
        if not changed:
            break
    lab, cnt = np.unique(parent, return_counts=True)
    return parent == lab[np.argmax(cnt)]


# (share of lattice LINES, lanes choices, limit choices in mph, keep probability of a link).  Arterial links are
# kept more often than local ones, so the line shares are set to give the EDGE shares of BASELINE.json
# configs[2] (60 % 1 lane, 25 % 2, 10 % 3, 5 % 4-5) after removal.
LANE_CLASSES = (
    (0.706, (1,), (25.0,), 0.50),
    (0.184, (2,), (35.0,), 0.80),
    (0.0735, (3,), (45.0,), 0.80),
    (0.0365, (4, 5), (55.0, 65.0), 0.80),
)


def bay_network(nx=492, ny=490, spacing=159.0, seed=SEED_NET, len_median=120.0, len_sigma=0.75,
                len_min=24.0, len_max=10000.0):
    """configs[2]: jittered square lattice with random edge removal, largest component, both directions;
    lognormal lengths; lane class per lattice LINE (so arterials form corridors), limits by class."""
    rng = np.random.default_rng(seed)
    idx = np.arange(nx * ny).reshape(ny, nx)
    # class per horizontal / vertical line
    shares = np.array([c[0] for c in LANE_CLASSES])
    shares = shares / shares.sum()
    cls_h = rng.choice(len(LANE_CLASSES), ny, p=shares)
    cls_v = rng.choice(len(LANE_CLASSES), nx, p=shares)
    a = np.concatenate([idx[:, :-1].ravel(), idx[:-1, :].ravel()])
    b = np.concatenate([idx[:, 1:].ravel(), idx[1:, :].ravel()])
    cls = np.concatenate([np.repeat(cls_h, nx - 1), np.tile(cls_v, ny - 1)])
    pk = np.array([c[3] for c in LANE_CLASSES])[cls]
    kept = rng.random(len(a)) < pk
    a, b, cls = a[kept], b[kept], cls[kept]
    inside = _largest_component(nx * ny, a, b)
    ok = inside[a] & inside[b]
    a, b, cls = a[ok], b[ok], cls[ok]
    new_id = np.full(nx * ny, -1, np.int64)
    new_id[inside] = np.arange(int(inside.sum()))
    n_nodes = int(inside.sum())
    a, b = new_id[a], new_id[b]
    m = len(a)
    length = np.exp(rng.normal(np.log(len_median), len_sigma, m))
    length = np.clip(length, len_min, len_max)
    lanes = np.ones(m, np.int64)
    limit = np.zeros(m)
    for k, (_, lane_opts, lim_opts, _k) in enumerate(LANE_CLASSES):
        sel = np.nonzero(cls == k)[0]
        pick = rng.integers(0, len(lane_opts), len(sel))
        lanes[sel] = np.array(lane_opts)[pick]
        limit[sel] = np.array(lim_opts)[pick % len(lim_opts)] * MPH
    tail = np.concatenate([a, b])
    head = np.concatenate([b, a])
    net = _csr_from_edges(n_nodes, tail, head, length_m=np.tile(length, 2).astype(np.float32),
                          lanes=np.tile(lanes, 2).astype(np.uint8), speed_limit=np.tile(limit, 2).astype(np.float32))
    net["node_ctrl"] = np.zeros(n_nodes, np.uint8)  # all GREEN
    yy, xx = np.divmod(np.nonzero(inside)[0], nx)
    jit = rng.uniform(-0.3, 0.3, (n_nodes, 2))
    net["xy"] = ((np.stack([xx, yy], 1) + jit) * spacing).astype(np.float32)
    net["lattice"] = (nx, ny, spacing, new_id)
    return net


def tile_network(net, kx=2, ky=2, seed=SEED_NET + 7):
    """configs[4]: kx x ky copies of a bay_network laid side by side, joined by seam edges between
    boundary nodes of neighbouring tiles (both directions, 2 lanes, 35 mph, 150 m)."""
    rng = np.random.default_rng(seed)
    n, m = net["n_nodes"], net["n_edges"]
    xy = net["xy"]
    w, h = float(xy[:, 0].max() - xy[:, 0].min()) + 300.0, float(xy[:, 1].max() - xy[:, 1].min()) + 300.0
    tails, heads, L, ln, lim, xys = [], [], [], [], [], []
    for ty in range(ky):
        for tx in range(kx):
            off = (ty * kx + tx) * n
            tails.append(net["tail"].astype(np.int64) + off)
            heads.append(net["head"].astype(np.int64) + off)
            L.append(net["length_m"]); ln.append(net["lanes"]); lim.append(net["speed_limit"])
            xys.append(xy + np.array([tx * w, ty * h], np.float32))
    right = np.nonzero(xy[:, 0] > xy[:, 0].max() - 250.0)[0]
    left = np.nonzero(xy[:, 0] < xy[:, 0].min() + 250.0)[0]
    top = np.nonzero(xy[:, 1] > xy[:, 1].max() - 250.0)[0]
    bot = np.nonzero(xy[:, 1] < xy[:, 1].min() + 250.0)[0]

    def seam(src_nodes, dst_nodes, axis, off_a, off_b):
        # join each src boundary node to the dst boundary node nearest along the seam axis
        order = np.argsort(xy[dst_nodes, axis])
        pos = np.searchsorted(xy[dst_nodes, axis][order], xy[src_nodes, axis]).clip(0, len(dst_nodes) - 1)
        s = src_nodes.astype(np.int64) + off_a
        d = dst_nodes[order][pos].astype(np.int64) + off_b
        k = len(s)
        tails.extend([s, d]); heads.extend([d, s])
        for _ in range(2):
            L.append(np.full(k, 150.0, np.float32)); ln.append(np.full(k, 2, np.uint8))
            lim.append(np.full(k, 35.0 * MPH, np.float32))

    for ty in range(ky):
        for tx in range(kx):
            off = (ty * kx + tx) * n
            if tx + 1 < kx:
                seam(right, left, 1, off, off + n)
            if ty + 1 < ky:
                seam(top, bot, 0, off, off + kx * n)
    _ = rng
    big = _csr_from_edges(kx * ky * n, np.concatenate(tails), np.concatenate(heads),
                          length_m=np.concatenate(L).astype(np.float32), lanes=np.concatenate(ln).astype(np.uint8),
                          speed_limit=np.concatenate(lim).astype(np.float32))
    big["node_ctrl"] = np.zeros(big["n_nodes"], np.uint8)
    big["xy"] = np.concatenate(xys).astype(np.float32)
    return big


def reduce_lanes(net, frac=0.2, seed=SEED_NET + 3):
    """configs[3]: a fraction of the >= 2-lane edges reduced to one lane (bottlenecks)."""
    rng = np.random.default_rng(seed)
    out = dict(net)
    lanes = net["lanes"].copy()
    multi = np.nonzero(lanes >= 2)[0]
    pick = multi[rng.random(len(multi)) < frac]
    lanes[pick] = 1
    out["lanes"] = lanes
    return out


# ----------------------------------------------------------------------------- demand
def uniform_od(net, n_trips, seed=SEED_DEMAND):
    rng = np.random.default_rng(seed)
    o = rng.integers(0, net["n_nodes"], n_trips)
    d = rng.integers(0, net["n_nodes"] - 1, n_trips)
    d = np.where(d >= o, d + 1, d)
    return o.astype(np.uint32), d.astype(np.uint32)


def gravity_od(net, n_trips, seed=SEED_DEMAND, n_origins=16384, dist_median=4300.0, dist_sigma=1.0,
               n_centres=12, centre_share=0.0):
    """Gravity-style OD on a coordinate-carrying network: origins drawn from a weighted set of origin nodes
    (the paper samples nodes inside 1454 TAZs); destination at a lognormal crow-fly distance
    (tuned so routed lengths have median ~6.5 km / mean ~11 km) in a uniform direction, or,
    with probability centre_share, near one of n_centres attraction centres picked by weight x deterrence."""
    rng = np.random.default_rng(seed)
    xy = net["xy"].astype(np.float64)
    n = net["n_nodes"]
    n_origins = min(n_origins, n)
    onodes = rng.choice(n, n_origins, replace=False)
    wts = rng.lognormal(0.0, 0.6, n_origins)
    o = onodes[rng.choice(n_origins, n_trips, p=wts / wts.sum())]
    lo, hi = xy.min(0), xy.max(0)
    # nearest-node lookup through a coarse bucket grid
    cell = 400.0
    gx = np.floor((xy[:, 0] - lo[0]) / cell).astype(np.int64)
    gy = np.floor((xy[:, 1] - lo[1]) / cell).astype(np.int64)
    nbx, nby = int(gx.max()) + 1, int(gy.max()) + 1
    rep = np.full(nbx * nby, -1, np.int64)
    rep[gy * nbx + gx] = np.arange(n)  # any node of the bucket
    filled = np.nonzero(rep >= 0)[0]

    def nearest(pts):
        bx = np.clip(np.floor((pts[:, 0] - lo[0]) / cell).astype(np.int64), 0, nbx - 1)
        by = np.clip(np.floor((pts[:, 1] - lo[1]) / cell).astype(np.int64), 0, nby - 1)
        r = rep[by * nbx + bx]
        miss = np.nonzero(r < 0)[0]
        if len(miss):  # empty bucket: take a random filled one nearby in index space
            r[miss] = rep[filled[np.searchsorted(filled, by[miss] * nbx + bx[miss]).clip(0, len(filled) - 1)]]
        return r

    d = np.empty(n_trips, np.int64)
    todo = np.arange(n_trips)
    centres = lo + rng.random((n_centres, 2)) * (hi - lo) * 0.8 + 0.1 * (hi - lo)
    cw = rng.lognormal(0.0, 0.8, n_centres)
    for _ in range(40):
        if len(todo) == 0:
            break
        k = len(todo)
        src = xy[o[todo]]
        dist = rng.lognormal(np.log(dist_median), dist_sigma, k)
        ang = rng.uniform(0, 2 * np.pi, k)
        tgt = src + dist[:, None] * np.stack([np.cos(ang), np.sin(ang)], 1)
        use_c = rng.random(k) < centre_share
        if use_c.any():
            dc = np.linalg.norm(src[use_c, None, :] - centres[None, :, :], axis=2)
            pr = cw[None, :] * np.exp(-dc / 15000.0)
            pr /= pr.sum(1, keepdims=True)
            pick = (pr.cumsum(1) > rng.random((int(use_c.sum()), 1))).argmax(1)
            tgt[use_c] = centres[pick] + rng.normal(0, 2000.0, (int(use_c.sum()), 2))
        inside = ((tgt >= lo) & (tgt <= hi)).all(1)
        cand = nearest(tgt)
        good = inside & (cand != o[todo])
        d[todo[good]] = cand[good]
        todo = todo[~good]
    if len(todo):
        d[todo] = (o[todo] + 1 + rng.integers(0, n - 1, len(todo))) % n
    return o.astype(np.uint32), d.astype(np.uint32)


def depart_uniform(n_trips, t0=0.0, t1=900.0, seed=SEED_DEMAND + 1):
    return np.random.default_rng(seed).uniform(t0, t1, n_trips).astype(np.float32)


def depart_bimodal(n_trips, seed=SEED_DEMAND + 1, t_open=5 * 3600.0, t_close=12 * 3600.0,
                   peaks=((0.55, 7.5 * 3600.0, 35 * 60.0), (0.45, 8.5 * 3600.0, 35 * 60.0))):
    """Departure seconds after t_open: mixture of normals truncated to [t_open, t_close] (BASELINE.json configs[2]
    'bimodal peak 07:30-08:30'; the paper itself uses one N(07:30, 45 min))."""
    rng = np.random.default_rng(seed)
    out = np.empty(n_trips)
    todo = np.arange(n_trips)
    w = np.array([p[0] for p in peaks])
    while len(todo):
        which = rng.choice(len(peaks), len(todo), p=w / w.sum())
        mu = np.array([p[1] for p in peaks])[which]
        sd = np.array([p[2] for p in peaks])[which]
        t = rng.normal(mu, sd)
        ok = (t >= t_open) & (t < t_close)
        out[todo[ok]] = t[ok] - t_open
        todo = todo[~ok]
    return out.astype(np.float32)


def make_trips(net, origin, dest, depart_time_s, n_threads=None, weight="length"):
    """Routes are shortest paths by edge LENGTH ("the length of the road link in meters ... is used
    as the weight of the edge"), fixed for the whole run; weight="time" gives free-flow time."""
    w = net["length_m"].astype(np.float64)
    if weight == "time":
        w = w / net["speed_limit"].astype(np.float64)
    rp, re_ = route_trips(net, origin, dest, weight=w, n_threads=n_threads)
    return dict(route_ptr=rp, route_edges=re_, depart_time_s=np.asarray(depart_time_s, np.float32),
                init_pos_m=None, init_speed=None)


# ----------------------------------------------------------------------------- the BASELINE.json configs
def config0(n_trips=2000, seed=SEED_DEMAND):
    net = grid_network()
    o, d = uniform_od(net, n_trips, seed)
    return net, make_trips(net, o, d, depart_uniform(n_trips, 0.0, 900.0, seed + 1)), dict(lookahead_cells=128), 7200


def config1(n_veh=600, n_steps=14400):
    net = ring_network()
    return net, ring_trips(net, n_veh=n_veh, laps_steps=n_steps), dict(lookahead_cells=128), n_steps


def config2(scale=1.0, n_trips=None, seed=SEED_DEMAND, net=None, window=None, n_threads=None, weight="time",
            centre_share=0.0):
    """Bay-Area-shaped run.  scale < 1 shrinks the lattice side and the trip count together (parity cases);
    window=(t0, t1) keeps only trips departing in [t0, t1) seconds after 05:00, shifted to start at 0."""
    if net is None:
        side = np.sqrt(scale)
        net = bay_network(nx=max(12, int(round(492 * side))), ny=max(12, int(round(490 * side))))
    if n_trips is None:
        n_trips = int(round(3_200_000 * scale))
    dep = depart_bimodal(n_trips, seed + 1)
    o, d = gravity_od(net, n_trips, seed, n_origins=max(64, int(16384 * scale)), centre_share=centre_share)
    if window is not None:
        sel = (dep >= window[0]) & (dep < window[1])
        o, d, dep = o[sel], d[sel], dep[sel] - np.float32(window[0])
    return net, make_trips(net, o, d, dep, n_threads=n_threads, weight=weight), dict(lookahead_cells=256), 50400


def config3(scale=1.0, seed=SEED_DEMAND + 100, window=None, n_threads=None):
    """BASELINE.json configs[3], congestion stress: the configs[2] network with 20 % of its >= 2-lane edges reduced
    to one lane, demand x 2 (6.4 M trips at scale 1) compressed into 06:00-09:00 (same bimodal law squeezed into
    the three hours), same gravity OD; runs until all trips are done or 43,200 steps (6 simulated hours).
    Times are seconds after 06:00."""
    side = np.sqrt(scale)
    net = reduce_lanes(bay_network(nx=max(12, int(round(492 * side))), ny=max(12, int(round(490 * side)))))
    n_trips = int(round(6_400_000 * scale))
    dep = depart_bimodal(n_trips, seed + 1, t_open=6 * 3600.0, t_close=9 * 3600.0,
                         peaks=((0.55, 7.25 * 3600.0, 20 * 60.0), (0.45, 7.9 * 3600.0, 20 * 60.0)))
    o, d = gravity_od(net, n_trips, seed, n_origins=max(64, int(16384 * scale)))
    if window is not None:
        sel = (dep >= window[0]) & (dep < window[1])
        o, d, dep = o[sel], d[sel], dep[sel] - np.float32(window[0])
    return net, make_trips(net, o, d, dep, n_threads=n_threads, weight="time"), dict(lookahead_cells=256), 43200


def config4(scale=1.0, seed=SEED_DEMAND + 200, window=None, n_threads=None):
    """BASELINE.json configs[4], scale-out on one GPU: 2 x 2 tiling of the configs[2] network joined by seam edges
    (~ 900 k nodes, ~ 2.2 M directed edges at scale 1) with 12.8 M trips of the same distributions (gravity OD over
    the whole tiled network, bimodal departures 05:00-12:00); 50,400 steps (7 simulated hours)."""
    side = np.sqrt(scale)
    net = tile_network(bay_network(nx=max(12, int(round(492 * side))), ny=max(12, int(round(490 * side)))), 2, 2)
    n_trips = int(round(12_800_000 * scale))
    dep = depart_bimodal(n_trips, seed + 1)
    o, d = gravity_od(net, n_trips, seed, n_origins=max(64, int(65536 * scale)))
    if window is not None:
        sel = (dep >= window[0]) & (dep < window[1])
        o, d, dep = o[sel], d[sel], dep[sel] - np.float32(window[0])
    return net, make_trips(net, o, d, dep, n_threads=n_threads, weight="time"), dict(lookahead_cells=256), 50400
