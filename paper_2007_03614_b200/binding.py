"""Thin ctypes binding of libmanta.so (include/manta.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for plumbing: device memory
(the library's allocator callbacks hand out torch caching-allocator blocks) and the CUDA stream.  There is no
CPU fallback: loading fails loudly if the library is missing, and Sim() fails if no CUDA device is present.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# MANTA_LIB_VARIANT=check loads the bounds-checking build (tests; every Sim.close() then fails on a recorded violation),
# MANTA_LIB_VARIANT=fast the fast-mode build (FMA contraction allowed: not bit-exact against the oracle)
VARIANT = os.environ.get("MANTA_LIB_VARIANT", "")
LIB_PATH = os.path.join(_HERE, {"check": "libmanta_check.so", "fast": "libmanta_fast.so"}.get(VARIANT, "libmanta.so"))

OK, ERR_INVALID_ARG, ERR_BAD_NETWORK, ERR_BAD_ROUTE, ERR_OOM, ERR_CUDA, ERR_STATE = 0, -1, -2, -3, -4, -5, -6
GREEN, PRIORITY, STOP = 0, 1, 2
WAITING, ACTIVE, DONE = 0, 1, 2
NONE = 0xFFFFFFFF
NOALLOC_MAX_TRIPS = 262144   # MANTA_NOALLOC_MAX_TRIPS
FLAG_MULTI_KERNEL, FLAG_RECORD_ACC = 2, 4

EXPORTS = ("manta_set_allocator", "manta_create", "manta_load_trips", "manta_step", "manta_step_async", "manta_sync",
           "manta_step_batch",
           "manta_step_timed",
           "manta_readback", "manta_readback_noalloc", "manta_load_state", "manta_readback_edge_speeds", "manta_atlas_cells", "manta_readback_atlas", "manta_set_stream", "manta_set_default_stream",
           "manta_set_multi_kernel",
           "manta_launch_count",
           "manta_device_bytes", "manta_destroy", "manta_last_error", "manta_check_failures",
           "manta_selftest_grid_barrier")


class MantaError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("manta error %d: %s" % (code, msg))
        self.code = code


class Network(C.Structure):
    _fields_ = [("n_nodes", C.c_uint32), ("n_edges", C.c_uint32), ("row_ptr", C.c_void_p), ("head", C.c_void_p),
                ("length_m", C.c_void_p), ("lanes", C.c_void_p), ("speed_limit", C.c_void_p),
                ("node_ctrl", C.c_void_p)]


class Params(C.Structure):
    _fields_ = [("size", C.c_uint32), ("dt", C.c_float), ("a", C.c_float), ("b", C.c_float), ("T", C.c_float),
                ("s0", C.c_float), ("veh_len", C.c_float), ("lookahead_cells", C.c_uint32),
                ("lookback_cells", C.c_uint32), ("mlc_scale_m", C.c_float), ("dlc_gain_thr", C.c_float),
                ("lc_alpha", C.c_float), ("lc_gap_low", C.c_float), ("lc_gap_high", C.c_float),
                ("lc_eps_sigma", C.c_float), ("seed", C.c_uint64), ("flags", C.c_uint32), ("stop_time_s", C.c_float),
                ("v0_sigma_rel", C.c_float), ("stat_period_steps", C.c_uint32), ("stat_slice_steps", C.c_uint32),
                ("stat_n_slices", C.c_uint32)]


class State(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("status", "route_pos", "lane", "tag", "x_fx", "v", "acc", "wait")]


class Summary(C.Structure):
    _fields_ = [(k, C.c_uint64) for k in ("t", "n_waiting", "n_active", "n_done", "sum_travel_steps",
                                          "vehicle_updates", "lane_changes", "cells_examined", "lc_evals", "n_stopped")]


DEFAULT_PARAMS = dict(dt=0.5, a=1.0, b=2.0, T=1.5, s0=2.0, veh_len=5.0, lookahead_cells=128, lookback_cells=64,
                      mlc_scale_m=100.0, dlc_gain_thr=0.2, lc_alpha=0.2, lc_gap_low=3.0, lc_gap_high=7.5,
                      lc_eps_sigma=1.0, seed=20070361, flags=0, stop_time_s=2.0, v0_sigma_rel=0.0, stat_period_steps=0,
                      stat_slice_steps=7200, stat_n_slices=0)

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_uint64, C.c_int, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_int, C.c_void_p)

_lib = None
_blocks = {}
_cb = None
_alloc_stream = None   # torch.cuda.Stream the library's allocations are made for (set by Sim(stream=...))


def load_library():
    """dlopen libmanta.so and declare the prototypes.  Raises if the CUDA library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libmanta.so is missing: run `python -m paper_2007_03614_b200.build` (nvcc, sm_100a). "
                          "There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    L.manta_set_allocator.argtypes = [ALLOC_FN, FREE_FN, C.c_void_p]
    L.manta_create.argtypes = [C.POINTER(Network), C.POINTER(Params), C.c_int, C.POINTER(C.c_void_p)]
    L.manta_load_trips.argtypes = [C.c_void_p, C.c_uint32] + [C.c_void_p] * 5
    for f in ("manta_step", "manta_step_async"):
        getattr(L, f).argtypes = [C.c_void_p, C.c_uint32]
    L.manta_sync.argtypes = [C.c_void_p]
    L.manta_step_batch.argtypes = [C.POINTER(C.c_void_p), C.c_uint32, C.c_uint32]
    L.manta_step_timed.argtypes = [C.c_void_p, C.c_uint32, C.POINTER(C.c_double * 3)]
    L.manta_readback.argtypes = [C.c_void_p, C.POINTER(State), C.c_void_p, C.c_void_p, C.POINTER(Summary)]
    L.manta_readback_noalloc.argtypes = L.manta_readback.argtypes
    L.manta_readback_edge_speeds.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.manta_load_state.argtypes = [C.c_void_p, C.c_uint32, C.POINTER(State), C.c_void_p, C.c_void_p]
    L.manta_atlas_cells.argtypes = [C.c_void_p]
    L.manta_atlas_cells.restype = C.c_uint64
    L.manta_readback_atlas.argtypes = [C.c_void_p] * 5
    L.manta_set_stream.argtypes = [C.c_void_p, C.c_void_p]
    L.manta_set_default_stream.argtypes = [C.c_void_p]
    L.manta_set_multi_kernel.argtypes = [C.c_void_p, C.c_int]
    L.manta_launch_count.argtypes = [C.c_void_p]
    L.manta_launch_count.restype = C.c_uint64
    L.manta_device_bytes.argtypes = [C.c_void_p]
    L.manta_device_bytes.restype = C.c_uint64
    L.manta_destroy.argtypes = [C.c_void_p]
    L.manta_destroy.restype = None
    L.manta_check_failures.argtypes = [C.c_void_p]
    L.manta_selftest_grid_barrier.argtypes = [C.c_int, C.c_uint32, C.POINTER(C.c_uint64), C.POINTER(C.c_uint32)]
    L.manta_last_error.argtypes = [C.c_void_p]
    L.manta_last_error.restype = C.c_char_p
    _lib = L
    return L


def use_torch_allocator():
    """Route the library's device allocations through PyTorch's caching allocator."""
    global _cb
    import torch
    L = load_library()

    def _alloc(nbytes, device, _ctx):
        # the caching allocator hands out stream-ordered blocks: allocate for the stream the library works on
        try:
            if _alloc_stream is not None:
                with torch.cuda.stream(_alloc_stream):
                    t = torch.empty(int(nbytes), dtype=torch.uint8, device="cuda:%d" % device)
            else:
                t = torch.empty(int(nbytes), dtype=torch.uint8, device="cuda:%d" % device)
        except Exception:
            return None
        _blocks[t.data_ptr()] = t
        return t.data_ptr()

    def _free(ptr, _device, _ctx):
        _blocks.pop(ptr, None)

    _cb = (ALLOC_FN(_alloc), FREE_FN(_free))
    L.manta_set_allocator(_cb[0], _cb[1], None)


def _ptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


def selftest_grid_barrier(n_rounds, device=0):
    """manta_selftest_grid_barrier: (words read stale, blocks launched)"""
    stale, blocks = C.c_uint64(0), C.c_uint32(0)
    rc = load_library().manta_selftest_grid_barrier(int(device), int(n_rounds), C.byref(stale), C.byref(blocks))
    if rc != OK:
        raise MantaError(rc, load_library().manta_last_error(None).decode())
    return int(stale.value), int(blocks.value)


def step_batch(sims, n=1):
    """manta_step_batch: advance several simulations (same device, stream, step counter) in one launch."""
    arr = (C.c_void_p * len(sims))(*[s.h for s in sims])
    rc = load_library().manta_step_batch(arr, len(sims), int(n))
    if rc != OK:
        raise MantaError(rc, load_library().manta_last_error(sims[0].h).decode())


class Sim:
    """One simulation on one GPU: manta_create + manta_load_trips + manta_step + manta_readback."""

    def __init__(self, net, params=None, trips=None, device=0, torch_alloc=True, stream=None):
        L = load_library()
        if torch_alloc and _cb is None:
            use_torch_allocator()
        pd = dict(DEFAULT_PARAMS)
        pd.update(params or {})
        self.params = pd
        P = Params(size=C.sizeof(Params), **pd)
        self._net_arrays = [np.ascontiguousarray(net["row_ptr"], np.uint32), np.ascontiguousarray(net["head"], np.uint32),
                            np.ascontiguousarray(net["length_m"], np.float32), np.ascontiguousarray(net["lanes"], np.uint8),
                            np.ascontiguousarray(net["speed_limit"], np.float32),
                            None if net.get("node_ctrl") is None else np.ascontiguousarray(net["node_ctrl"], np.uint8)]
        N = Network(int(net["n_nodes"]), int(net["n_edges"]), *[_ptr(a) for a in self._net_arrays])
        self.n_edges = int(net["n_edges"])
        self.h = C.c_void_p()
        # one stream from manta_create on: uploads, kernels and the allocator's blocks are all ordered on it
        self._stream = stream
        self._use()
        L.manta_set_default_stream(C.c_void_p(int(getattr(stream, "cuda_stream", stream or 0))))
        rc = L.manta_create(C.byref(N), C.byref(P), int(device), C.byref(self.h))
        L.manta_set_default_stream(None)
        if rc != OK:
            self.h = None
            raise MantaError(rc, L.manta_last_error(None).decode())
        self.n_trips = 0
        if trips is not None:
            self.load_trips(trips)

    def _use(self):
        """allocations made by the next library call are for this simulation's stream"""
        global _alloc_stream
        _alloc_stream = self._stream if hasattr(self._stream, "cuda_stream") else None

    def _check(self, rc):
        if rc != OK:
            raise MantaError(rc, load_library().manta_last_error(self.h).decode())

    def set_stream(self, stream):
        """stream: torch.cuda.Stream or a raw cudaStream_t integer."""
        self._stream = stream
        handle = getattr(stream, "cuda_stream", stream)
        self._check(load_library().manta_set_stream(self.h, C.c_void_p(int(handle))))

    def load_trips(self, trips):
        rp = np.ascontiguousarray(trips["route_ptr"], np.uint64)
        re_ = np.ascontiguousarray(trips["route_edges"], np.uint32)
        dep = np.ascontiguousarray(trips["depart_time_s"], np.float32)
        ip, iv = trips.get("init_pos_m"), trips.get("init_speed")
        ip = None if ip is None else np.ascontiguousarray(ip, np.float32)
        iv = None if iv is None else np.ascontiguousarray(iv, np.float32)
        self._use()
        self._check(load_library().manta_load_trips(self.h, len(dep), _ptr(rp), _ptr(re_), _ptr(dep), _ptr(ip), _ptr(iv)))
        self.n_trips = len(dep)

    def step(self, n=1):
        self._check(load_library().manta_step(self.h, int(n)))

    def set_multi_kernel(self, on):
        self._check(load_library().manta_set_multi_kernel(self.h, int(bool(on))))

    def step_async(self, n=1):
        self._check(load_library().manta_step_async(self.h, int(n)))

    def step_timed(self, n=1):
        """manta_step with per-phase CUDA-event timing; returns [admit_ms, update_ms, second_phase_ms] summed over n."""
        ms = (C.c_double * 3)(0.0, 0.0, 0.0)
        self._check(load_library().manta_step_timed(self.h, int(n), C.byref(ms)))
        return [float(x) for x in ms]

    def sync(self):
        self._check(load_library().manta_sync(self.h))

    def readback(self, state=True, edge_entries=True, trips=True, summary=True, noalloc=False):
        """manta_readback; noalloc=True calls manta_readback_noalloc instead (same outputs, no device allocation, at most
        NOALLOC_MAX_TRIPS trips -- see include/manta.h for who needs that and what it costs)."""
        n = self.n_trips
        out = {}
        S = None
        if state:
            out.update(status=np.zeros(n, np.uint8), route_pos=np.zeros(n, np.uint32), lane=np.zeros(n, np.uint8),
                       tag=np.zeros(n, np.uint8), x_fx=np.zeros(n, np.uint32), v=np.zeros(n, np.float32),
                       acc=np.zeros(n, np.float32), wait=np.zeros(n, np.uint8))
            S = State(*[_ptr(out[k]) for k in ("status", "route_pos", "lane", "tag", "x_fx", "v", "acc", "wait")])
        ee = np.zeros(self.n_edges, np.uint32) if edge_entries else None
        tr = np.zeros((n, 2), np.uint32) if trips else None
        sm = Summary() if summary else None
        self._use()
        fn = load_library().manta_readback_noalloc if noalloc else load_library().manta_readback
        self._check(fn(self.h, None if S is None else C.byref(S), _ptr(ee), _ptr(tr), None if sm is None else C.byref(sm)))
        if trips:
            out["admit_step"], out["arrive_step"] = tr[:, 0].copy(), tr[:, 1].copy()
        if edge_entries:
            out["edge_entries"] = ee
        if summary:
            out["summary"] = {k: int(getattr(sm, k)) for k, _ in Summary._fields_}
        return out

    def load_state(self, t, st, edge_entries=None):
        """manta_load_state: st = dict with status, route_pos, lane, tag, x_fx, v, admit_step, arrive_step (as readback
        returns them) and optionally wait."""
        n = self.n_trips
        a = dict(status=np.ascontiguousarray(st["status"], np.uint8), route_pos=np.ascontiguousarray(st["route_pos"], np.uint32),
                 lane=np.ascontiguousarray(st["lane"], np.uint8), tag=np.ascontiguousarray(st["tag"], np.uint8),
                 x_fx=np.ascontiguousarray(st["x_fx"], np.uint32), v=np.ascontiguousarray(st["v"], np.float32),
                 acc=None, wait=None if st.get("wait") is None else np.ascontiguousarray(st["wait"], np.uint8))
        assert all(x is None or len(x) == n for x in a.values())
        S = State(*[_ptr(a[k]) for k in ("status", "route_pos", "lane", "tag", "x_fx", "v", "acc", "wait")])
        tr = np.ascontiguousarray(np.stack([np.asarray(st["admit_step"], np.uint32), np.asarray(st["arrive_step"], np.uint32)], 1))
        ee = None if edge_entries is None else np.ascontiguousarray(edge_entries, np.uint32)
        self._use()
        self._check(load_library().manta_load_state(self.h, int(t), C.byref(S), _ptr(tr), _ptr(ee)))

    def readback_edge_speeds(self):
        """(sum of rint(v * 256), samples), each [stat_n_slices, n_edges] (manta_readback_edge_speeds)"""
        ns = int(self.params["stat_n_slices"])
        sm, cn = np.zeros((ns, self.n_edges), np.uint64), np.zeros((ns, self.n_edges), np.uint32)
        self._check(load_library().manta_readback_edge_speeds(self.h, _ptr(sm), _ptr(cn)))
        return sm, cn

    def readback_atlas(self):
        n = int(load_library().manta_atlas_cells(self.h))
        occ, spd = np.zeros(n, np.uint16), np.zeros(n, np.float32)
        off, pitch = np.zeros(self.n_edges, np.uint32), np.zeros(self.n_edges, np.uint32)
        self._use()
        self._check(load_library().manta_readback_atlas(self.h, _ptr(occ), _ptr(spd), _ptr(off), _ptr(pitch)))
        return dict(occ=occ, spd=spd, cell_off=off, pitch=pitch)

    @property
    def launch_count(self):
        return int(load_library().manta_launch_count(self.h))

    @property
    def device_bytes(self):
        return int(load_library().manta_device_bytes(self.h))

    def check_failures(self):
        """largest bounds-check failure code of the MANTA_CHECK build (0 = none); -1 in the product build"""
        return int(load_library().manta_check_failures(self.h))

    def close(self):
        if getattr(self, "h", None):
            bad = self.check_failures() if VARIANT == "check" and self.n_trips else 0
            load_library().manta_destroy(self.h)
            self.h = None
            if bad > 0:
                raise MantaError(ERR_STATE, "bounds check %d failed in the MANTA_CHECK build" % bad)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
