"""ctypes binding of oracle/manta_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It builds libmanta_oracle.so with gcc (IEEE op-by-op fp32:
-O2 -ffp-contract=off -fno-fast-math) and exposes the mo_* calls on numpy arrays.
It imports nothing from paper_2007_03614_b200.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "manta_oracle.c")
_HDR = os.path.join(_HERE, "manta_oracle.h")
_SO = os.path.join(_HERE, "libmanta_oracle.so")

WAITING, ACTIVE, DONE = 0, 1, 2
NONE32 = 0xFFFFFFFF


def build(force=False):
    """Compile the oracle (gcc only; no CUDA).  Returns the path of the shared object."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))):
        return _SO
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-shared", "-fPIC",
           "-o", _SO, _SRC, "-lm"]
    subprocess.check_call(cmd)
    return _SO


class _Params(C.Structure):
    _fields_ = [("dt", C.c_float), ("a", C.c_float), ("b", C.c_float), ("T", C.c_float), ("s0", C.c_float),
                ("veh_len", C.c_float), ("lookahead_cells", C.c_uint32), ("lookback_cells", C.c_uint32),
                ("mlc_scale_m", C.c_float), ("dlc_gain_thr", C.c_float), ("lc_alpha", C.c_float),
                ("lc_gap_low", C.c_float), ("lc_gap_high", C.c_float), ("lc_eps_sigma", C.c_float),
                ("seed", C.c_uint64), ("stop_time_s", C.c_float), ("v0_sigma_rel", C.c_float),
                ("stat_period_steps", C.c_uint32), ("stat_slice_steps", C.c_uint32), ("stat_n_slices", C.c_uint32)]


DEFAULT_PARAMS = dict(dt=0.5, a=1.0, b=2.0, T=1.5, s0=2.0, veh_len=5.0, lookahead_cells=128, lookback_cells=64,
                      mlc_scale_m=100.0, dlc_gain_thr=0.2, lc_alpha=0.2, lc_gap_low=3.0, lc_gap_high=7.5,
                      lc_eps_sigma=1.0, seed=20070361, stop_time_s=2.0, v0_sigma_rel=0.0, stat_period_steps=0,
                      stat_slice_steps=7200, stat_n_slices=0)

_lib = None


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.mo_create.restype = C.c_void_p
        L.mo_create.argtypes = [C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                C.c_void_p, C.c_void_p, C.POINTER(_Params)]
        L.mo_load_trips.restype = C.c_int
        L.mo_load_trips.argtypes = [C.c_void_p, C.c_uint32] + [C.c_void_p] * 5
        L.mo_set_order.argtypes = [C.c_void_p, C.c_int, C.c_uint64]
        L.mo_step.restype = C.c_int
        L.mo_step.argtypes = [C.c_void_p, C.c_uint32]
        L.mo_set_state.restype = C.c_int
        L.mo_set_state.argtypes = [C.c_void_p, C.c_uint32] + [C.c_void_p] * 9
        L.mo_set_wait.argtypes = [C.c_void_p, C.c_void_p]
        L.mo_get_wait.argtypes = [C.c_void_p, C.c_void_p]
        L.mo_get_edge_speed_stats.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.mo_v0.restype = C.c_float
        L.mo_v0.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32]
        L.mo_n_stopped.restype = C.c_uint64
        L.mo_n_stopped.argtypes = [C.c_void_p]
        L.mo_destroy.argtypes = [C.c_void_p]
        L.mo_get_state.argtypes = [C.c_void_p] + [C.c_void_p] * 7
        L.mo_get_trip_results.argtypes = [C.c_void_p] * 3
        L.mo_get_edge_entries.argtypes = [C.c_void_p] * 2
        L.mo_get_summary.argtypes = [C.c_void_p] * 2
        L.mo_get_derived.argtypes = [C.c_void_p] * 2
        L.mo_get_vehicle_ids.argtypes = [C.c_void_p] * 2
        L.mo_n_cells.restype = C.c_uint64
        L.mo_n_cells.argtypes = [C.c_void_p]
        L.mo_n_rows.restype = C.c_uint32
        L.mo_n_rows.argtypes = [C.c_void_p]
        L.mo_get_atlas.argtypes = [C.c_void_p] * 4
        L.mo_get_row_offsets.argtypes = [C.c_void_p] * 3
        L.mo_idm_acc.restype = C.c_float
        L.mo_idm_acc.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_int, C.c_float, C.c_float]
        L.mo_rng.restype = C.c_uint32
        L.mo_rng.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32]
        L.mo_eps.restype = C.c_float
        L.mo_eps.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32]
        L.mo_pmlc.restype = C.c_uint32
        L.mo_pmlc.argtypes = [C.c_void_p, C.c_uint32]
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


class Oracle:
    """One simulation.  `net` and `trips` are the dicts made by the workload generators:
    net = {n_nodes, n_edges, row_ptr u32, head u32, length_m f32, lanes u8, speed_limit f32, node_ctrl u8|None}
    trips = {route_ptr u64, route_edges u32, depart_time_s f32, init_pos_m f32|None, init_speed f32|None}"""

    def __init__(self, net, params=None, trips=None):
        L = lib()
        pd = dict(DEFAULT_PARAMS)
        pd.update(params or {})
        self.params = pd
        self._P = _Params(**pd)
        self.net = net
        self.n_edges = int(net["n_edges"])
        self._keep = [np.ascontiguousarray(net["row_ptr"], np.uint32), np.ascontiguousarray(net["head"], np.uint32),
                      np.ascontiguousarray(net["length_m"], np.float32), np.ascontiguousarray(net["lanes"], np.uint8),
                      np.ascontiguousarray(net["speed_limit"], np.float32),
                      None if net.get("node_ctrl") is None else np.ascontiguousarray(net["node_ctrl"], np.uint8)]
        self.h = L.mo_create(int(net["n_nodes"]), self.n_edges, *[_ptr(a) for a in self._keep], C.byref(self._P))
        if not self.h:
            raise ValueError("mo_create rejected the network")
        self.n_trips = 0
        if trips is not None:
            self.load_trips(trips)

    def load_trips(self, trips):
        rp = np.ascontiguousarray(trips["route_ptr"], np.uint64)
        re_ = np.ascontiguousarray(trips["route_edges"], np.uint32)
        dep = np.ascontiguousarray(trips["depart_time_s"], np.float32)
        ip = trips.get("init_pos_m")
        iv = trips.get("init_speed")
        ip = None if ip is None else np.ascontiguousarray(ip, np.float32)
        iv = None if iv is None else np.ascontiguousarray(iv, np.float32)
        n = len(dep)
        rc = lib().mo_load_trips(self.h, n, _ptr(rp), _ptr(re_), _ptr(dep), _ptr(ip), _ptr(iv))
        if rc != 0:
            raise ValueError("mo_load_trips failed: %d" % rc)
        self.n_trips = n

    def set_order(self, mode, seed=1):
        lib().mo_set_order(self.h, mode, seed)

    def step(self, n=1):
        rc = lib().mo_step(self.h, int(n))
        if rc != 0:
            raise RuntimeError("mo_step failed: %d" % rc)

    def set_state(self, t, st, edge_entries=None):
        a = [np.ascontiguousarray(st["status"], np.uint8), np.ascontiguousarray(st["route_pos"], np.uint32),
             np.ascontiguousarray(st["lane"], np.uint8), np.ascontiguousarray(st["tag"], np.uint8),
             np.ascontiguousarray(st["x_fx"], np.uint32), np.ascontiguousarray(st["v"], np.float32),
             np.ascontiguousarray(st["admit_step"], np.uint32), np.ascontiguousarray(st["arrive_step"], np.uint32),
             None if edge_entries is None else np.ascontiguousarray(edge_entries, np.uint32)]
        rc = lib().mo_set_state(self.h, int(t), *[_ptr(x) for x in a])
        if rc != 0:
            raise ValueError("mo_set_state failed: %d" % rc)
        if st.get("wait") is not None:
            w = np.ascontiguousarray(st["wait"], np.uint8)
            lib().mo_set_wait(self.h, _ptr(w))

    def state(self):
        n = self.n_trips
        out = dict(status=np.zeros(n, np.uint8), route_pos=np.zeros(n, np.uint32), lane=np.zeros(n, np.uint8),
                   tag=np.zeros(n, np.uint8), x_fx=np.zeros(n, np.uint32), v=np.zeros(n, np.float32),
                   acc=np.zeros(n, np.float32))
        lib().mo_get_state(self.h, *[_ptr(out[k]) for k in ("status", "route_pos", "lane", "tag", "x_fx", "v", "acc")])
        adm = np.zeros(n, np.uint32)
        arr = np.zeros(n, np.uint32)
        lib().mo_get_trip_results(self.h, _ptr(adm), _ptr(arr))
        out["admit_step"], out["arrive_step"] = adm, arr
        out["wait"] = np.zeros(n, np.uint8)
        lib().mo_get_wait(self.h, _ptr(out["wait"]))
        return out

    def edge_speed_stats(self):
        """(sum of rint(v * 256), samples), each [stat_n_slices, n_edges]"""
        ns = int(self.params["stat_n_slices"])
        sm, cn = np.zeros((ns, self.n_edges), np.uint64), np.zeros((ns, self.n_edges), np.uint32)
        if ns and self.params["stat_period_steps"]:
            lib().mo_get_edge_speed_stats(self.h, _ptr(sm), _ptr(cn))
        return sm, cn

    def v0(self, vid, r):
        return float(lib().mo_v0(self.h, vid, r))

    def n_stopped(self):
        return int(lib().mo_n_stopped(self.h))

    def edge_entries(self):
        e = np.zeros(self.n_edges, np.uint32)
        lib().mo_get_edge_entries(self.h, _ptr(e))
        return e

    def summary(self):
        s = np.zeros(9, np.uint64)
        lib().mo_get_summary(self.h, _ptr(s))
        keys = ("t", "n_waiting", "n_active", "n_done", "sum_travel_steps", "vehicle_updates", "lane_changes",
                "cells_examined", "lc_evals")
        out = {k: int(x) for k, x in zip(keys, s)}
        out["n_stopped"] = self.n_stopped()
        return out

    def derived(self):
        d = np.zeros(6, np.uint32)
        lib().mo_get_derived(self.h, _ptr(d))
        return dict(zip(("L_c", "Z_out", "Z_in", "LEN_MIN", "L_fx", "Lambda"), (int(x) for x in d)))

    def vehicle_ids(self):
        ids = np.zeros(self.n_trips, np.uint32)
        lib().mo_get_vehicle_ids(self.h, _ptr(ids))
        return ids

    def atlas(self):
        n = int(lib().mo_n_cells(self.h))
        occ, frac, spd = np.zeros(n, np.uint8), np.zeros(n, np.uint16), np.zeros(n, np.float32)
        lib().mo_get_atlas(self.h, _ptr(occ), _ptr(frac), _ptr(spd))
        nr = int(lib().mo_n_rows(self.h))
        first_row, row_off = np.zeros(self.n_edges, np.uint32), np.zeros(nr, np.uint64)
        lib().mo_get_row_offsets(self.h, _ptr(first_row), _ptr(row_off))
        return dict(occ=occ, frac=frac, spd=spd, first_row=first_row, row_off=row_off)

    def idm_acc(self, v, v0, s=None, v_lead=0.0):
        return float(lib().mo_idm_acc(self.h, v, v0, 0 if s is None else 1, 0.0 if s is None else s, v_lead))

    def rng(self, vid, t, k):
        return int(lib().mo_rng(self.h, vid, t, k))

    def eps(self, vid, t, k0):
        return float(lib().mo_eps(self.h, vid, t, k0))

    def pmlc(self, dcell):
        return int(lib().mo_pmlc(self.h, dcell))

    def close(self):
        if self.h:
            lib().mo_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
