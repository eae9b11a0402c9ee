"""Shared test helpers: invariant checks on oracle / GPU state snapshots (no simulator arithmetic)."""
import numpy as np

WAITING, ACTIVE, DONE = 0, 1, 2


def row_keys(net, trips, st):
    """(edge, lane) key and x of every ACTIVE vehicle."""
    act = np.nonzero(st["status"] == ACTIVE)[0]
    rp = trips["route_ptr"].astype(np.int64)
    e = trips["route_edges"][rp[act] + st["route_pos"][act].astype(np.int64)].astype(np.int64)
    return act, e, st["lane"][act].astype(np.int64), st["x_fx"][act].astype(np.int64)


def check_no_overlap(net, trips, st, L_fx):
    """K8: consecutive vehicles of one (edge, lane) row are >= L apart; no two share a cell."""
    act, e, l, x = row_keys(net, trips, st)
    if len(act) < 2:
        return
    key = e * 16 + l
    order = np.lexsort((x, key))
    k, xs = key[order], x[order]
    same = k[1:] == k[:-1]
    gap = xs[1:] - xs[:-1]
    bad = same & (gap < L_fx)
    assert not bad.any(), "overlap: trips %s gap %s" % (act[order][1:][bad][:5], gap[bad][:5])
    lens = np.round(net["length_m"].astype(np.float64)).astype(np.int64)
    assert (x < (lens[e] << 10)).all()
    assert (l < net["lanes"][e]).all()


def check_conservation(st, n_trips, summary=None):
    """K6 (first half)."""
    nw, na, nd = [(st["status"] == k).sum() for k in (WAITING, ACTIVE, DONE)]
    assert nw + na + nd == n_trips
    if summary is not None:
        assert (summary["n_waiting"], summary["n_active"], summary["n_done"]) == (nw, na, nd)


def check_entries(st, edge_entries, trips=None):
    """K6 (second half): sum of edge entries == sum over admitted vehicles of (route_pos + 1); a DONE vehicle
    has entered every edge of its route (its route_pos is taken from the route length when trips is given)."""
    rpos = st["route_pos"].astype(np.int64)
    if trips is not None:
        rl = np.diff(trips["route_ptr"].astype(np.int64))
        rpos = np.where(st["status"] == DONE, rl - 1, rpos)
    adm = st["status"] != WAITING
    assert int(edge_entries.astype(np.int64).sum()) == int((rpos[adm] + 1).sum())


def check_monotone(prev, cur):
    """K7: route_pos never decreases; on the same edge x never decreases; v >= 0."""
    both = (prev["status"] == ACTIVE) & (cur["status"] == ACTIVE)
    assert (cur["route_pos"][both] >= prev["route_pos"][both]).all()
    same = both & (cur["route_pos"] == prev["route_pos"])
    assert (cur["x_fx"][same] >= prev["x_fx"][same]).all()
    assert (cur["v"][cur["status"] == ACTIVE] >= 0).all()
    assert ((prev["status"] == DONE) <= (cur["status"] == DONE)).all()


def states_equal(a, b, keys=("status", "route_pos", "lane", "tag", "x_fx", "v", "admit_step", "arrive_step", "wait")):
    """bit-exact comparison (v compared by bit pattern); returns list of (key, first bad indices)."""
    bad = []
    act = (a["status"] == ACTIVE)
    for k in keys:
        x, y = a[k], b[k]
        if x.dtype == np.float32:
            x, y = x.view(np.uint32), y.view(np.uint32)
        m = x != y
        if k in ("route_pos", "lane", "tag", "x_fx", "v", "acc", "wait"):
            m = m & (act | (b["status"] == ACTIVE))  # only meaningful while ACTIVE
        if m.any():
            bad.append((k, np.nonzero(m)[0][:8].tolist()))
    return bad
