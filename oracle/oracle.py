"""ctypes front-end of oracle/libnecsim_oracle.so -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
It imports nothing from paper_2108_05815_b200. See necsim_oracle.c for citations into PAPER.md.
"""
import ctypes as C
import os
import numpy as np

from . import build as _build

NONSPATIAL, SPATIALLY_IMPLICIT, EXPLICIT_MATRIX, EXPLICIT_GAUSSIAN = 0, 1, 2, 3

_lib = None


class Stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("richness", "n_lineages", "n_events", "n_culled", "n_epochs",
                                         "resample_attempts", "n_unfinished")]


EVENT_DTYPE = np.dtype({"names": ["loc", "k", "j", "f", "abundance", "time"],
                        "formats": ["<u4", "<u4", "<u4", "<u8", "<u4", "<f8"],
                        "offsets": [0, 4, 8, 16, 24, 32], "itemsize": 40})
KEY_DTYPE = np.dtype({"names": ["loc", "k", "j", "f"], "formats": ["<u4", "<u4", "<u4", "<u8"],
                      "offsets": [0, 4, 8, 16], "itemsize": 24})


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        u32, u64, i64, dbl, vp = C.c_uint32, C.c_uint64, C.c_int64, C.c_double, C.c_void_p
        L.orc_F.restype = u64; L.orc_F.argtypes = [u64]
        L.orc_key_schedule.restype = None; L.orc_key_schedule.argtypes = [u64, vp]
        L.orc_prime.restype = u64; L.orc_prime.argtypes = [vp, u32, u32]
        for nm in ("time", "spec", "index", "migr"):
            f = getattr(L, "orc_draw_" + nm); f.restype = u64; f.argtypes = [u64, u32]
        L.orc_draw_disp.restype = u64; L.orc_draw_disp.argtypes = [u64, u32, u32]
        L.orc_neglog.restype = u64; L.orc_neglog.argtypes = [u64]
        L.orc_turnover_scale.restype = C.c_int; L.orc_turnover_scale.argtypes = [dbl, dbl, vp, vp]
        L.orc_scale.restype = u64; L.orc_scale.argtypes = [u64, u32, u32]
        L.orc_time.restype = dbl; L.orc_time.argtypes = [u32, u64, dbl]
        L.orc_next_event.restype = C.c_int
        L.orc_next_event.argtypes = [vp, u32, vp, i64, u32, u32, u32, vp, vp, vp]
        L.orc_gauss_R.restype = C.c_int; L.orc_gauss_R.argtypes = [dbl]
        L.orc_gauss_table.restype = None; L.orc_gauss_table.argtypes = [dbl, C.c_int, vp]
        L.orc_gauss_lookup.restype = C.c_int; L.orc_gauss_lookup.argtypes = [vp, C.c_int, u32]
        L.orc_alias_row.restype = C.c_int; L.orc_alias_row.argtypes = [vp, u32, vp, vp]
        L.orc_thr.restype = u64; L.orc_thr.argtypes = [dbl]
        L.orc_scenario_create.restype = vp
        L.orc_scenario_create.argtypes = [C.c_int, u32, u32, vp, u32, vp, dbl, vp, dbl, u64, u64, dbl, dbl, C.c_char_p, C.c_int]
        L.orc_scenario_destroy.restype = None; L.orc_scenario_destroy.argtypes = [vp]
        L.orc_scenario_num_individuals.restype = u64; L.orc_scenario_num_individuals.argtypes = [vp]
        L.orc_scenario_thresh.restype = vp; L.orc_scenario_thresh.argtypes = [vp]
        L.orc_scenario_alias.restype = vp; L.orc_scenario_alias.argtypes = [vp]
        L.orc_scenario_gauss.restype = vp; L.orc_scenario_gauss.argtypes = [vp, vp]
        L.orc_scenario_cell_scale.restype = None; L.orc_scenario_cell_scale.argtypes = [vp, u32, vp, vp]
        L.orc_debug_disperse.restype = C.c_int; L.orc_debug_disperse.argtypes = [vp, u64, dbl, u32, u32, u32, vp]
        L.orc_simulate.restype = C.c_int
        L.orc_simulate.argtypes = [vp, u64, dbl, vp, C.c_int, u64, u64, vp, vp, vp, vp, vp]
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


# ---- primitives -------------------------------------------------------------------------------
def F(x): return lib().orc_F(int(x) & (2**64 - 1))

def key_schedule(seed):
    K = np.zeros(6, dtype=np.uint32); lib().orc_key_schedule(int(seed), _ptr(K)); return K

def prime(K, loc, k): return lib().orc_prime(_ptr(K), int(loc), int(k))
def draw_time(s, j): return lib().orc_draw_time(s, j)
def draw_spec(s, j): return lib().orc_draw_spec(s, j)
def draw_disp(s, j, r=0): return lib().orc_draw_disp(s, j, r)
def draw_index(s, j): return lib().orc_draw_index(s, j)
def draw_migr(s, j): return lib().orc_draw_migr(s, j)
def neglog(x): return lib().orc_neglog(int(x))
def scale(E, Cm, sh): return lib().orc_scale(int(E), int(Cm), int(sh))
def thr(p): return lib().orc_thr(float(p))
def time_of(k, f, delta_t): return lib().orc_time(int(k), int(f), float(delta_t))

def turnover_scale(lam, delta_t):
    cm, sh = C.c_uint32(), C.c_uint32()
    rc = lib().orc_turnover_scale(float(lam), float(delta_t), C.byref(cm), C.byref(sh))
    if rc != 0: raise ValueError("turnover*delta_t out of range")
    return cm.value, sh.value

def next_event(K, loc, k, f_last, Cm, sh, k_stop=0xFFFFFFFF):
    """returns (rc, k, j, T, s); rc 0 found, 1 horizon reached."""
    kk, j, T, s = C.c_uint32(int(k)), C.c_uint32(), C.c_uint64(), C.c_uint64()
    rc = lib().orc_next_event(_ptr(K), int(loc), C.byref(kk), int(f_last), int(Cm), int(sh), int(k_stop),
                              C.byref(j), C.byref(T), C.byref(s))
    return rc, kk.value, j.value, T.value, s.value

def gauss_table(sigma):
    R = lib().orc_gauss_R(float(sigma)); TG = np.zeros(2 * R, dtype=np.uint32)
    lib().orc_gauss_table(float(sigma), R, _ptr(TG)); return R, TG

def gauss_lookup(TG, R, u): return lib().orc_gauss_lookup(_ptr(TG), int(R), int(u))

def alias_row(w):
    w = np.ascontiguousarray(w, dtype=np.float64); n = len(w)
    th = np.zeros(n, dtype=np.uint32); al = np.zeros(n, dtype=np.uint32)
    rc = lib().orc_alias_row(_ptr(w), n, _ptr(th), _ptr(al))
    if rc != 0: raise ValueError("alias_row rc=%d" % rc)
    return th, al


# ---- scenario + simulation --------------------------------------------------------------------
class Scenario:
    """Mirror of the paper's scenario = habitat + turnover + dispersal (+ sizes)."""

    def __init__(self, kind, width=1, height=1, deme=None, uniform_deme=0, turnover=None, uniform_turnover=1.0,
                 matrix=None, sigma=0.0, local_size=0, meta_size=0, migration=0.0, delta_t=2.0, sampler=0, past_deme=None, past_start_k=None):
        self.kind = kind
        d = None if deme is None else np.ascontiguousarray(deme, dtype=np.uint32).ravel()
        t = None if turnover is None else np.ascontiguousarray(turnover, dtype=np.float64).ravel()
        m = None if matrix is None else np.ascontiguousarray(matrix, dtype=np.float64)
        err = C.create_string_buffer(256)
        self._h = lib().orc_scenario_create(kind, width, height, _ptr(d), int(uniform_deme), _ptr(t), float(uniform_turnover),
                                            _ptr(m), float(sigma), int(local_size), int(meta_size), float(migration),
                                            float(delta_t), err, 256)
        if not self._h:
            raise ValueError("oracle scenario: " + err.value.decode())
        L = lib(); L.orc_scenario_set_sampler.restype = C.c_int; L.orc_scenario_set_sampler.argtypes = [C.c_void_p, C.c_int]
        if past_deme is not None:   # temporally varying habitat: eras 1.. of the past
            pd = np.ascontiguousarray(past_deme, dtype=np.uint32).reshape(-1, width * height)
            ps = np.ascontiguousarray(past_start_k, dtype=np.uint32).ravel()
            assert len(ps) == pd.shape[0]
            L.orc_scenario_set_eras.restype = C.c_int; L.orc_scenario_set_eras.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p]
            if L.orc_scenario_set_eras(self._h, pd.shape[0], _ptr(pd), _ptr(ps)) != 0:
                raise ValueError("oracle scenario: bad eras (gaussian kind only, start_k increasing, habitat only lost towards the present)")
        if L.orc_scenario_set_sampler(self._h, int(sampler)) != 0:
            raise ValueError("oracle scenario: unknown sampler")
        self.sampler = int(sampler)
        self.delta_t = float(delta_t)
        self.ncells = 2 if kind == SPATIALLY_IMPLICIT else width * height

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_scenario_destroy(self._h); self._h = None

    @property
    def n_individuals(self): return lib().orc_scenario_num_individuals(self._h)

    def alias_tables(self):
        n = self.ncells
        th = np.ctypeslib.as_array(C.cast(lib().orc_scenario_thresh(self._h), C.POINTER(C.c_uint32)), shape=(n, n)).copy()
        al = np.ctypeslib.as_array(C.cast(lib().orc_scenario_alias(self._h), C.POINTER(C.c_uint32)), shape=(n, n)).copy()
        return th, al

    def poisson_table(self):
        """(mu_max, PC[256]) of the Poisson sampler."""
        L = lib(); L.orc_scenario_poisson.restype = C.c_void_p; L.orc_scenario_poisson.argtypes = [C.c_void_p, C.c_void_p]
        mu = C.c_double(); p = L.orc_scenario_poisson(self._h, C.byref(mu))
        return mu.value, np.ctypeslib.as_array(C.cast(p, C.POINTER(C.c_uint64)), shape=(256,)).copy()

    def thin(self, cell):
        L = lib(); L.orc_scenario_thin.restype = C.c_uint32; L.orc_scenario_thin.argtypes = [C.c_void_p, C.c_uint32]
        return L.orc_scenario_thin(self._h, int(cell))

    def batch_next_event_poisson(self, seed, loc, cell, k, f_last):
        loc = np.ascontiguousarray(loc, dtype=np.uint32); n = len(loc)
        cell = _u32(cell, n); k = _u32(k, n)
        f_last = np.ascontiguousarray(np.broadcast_to(np.asarray(f_last, dtype=np.int64), (n,)))
        ko = np.zeros(n, np.uint32); jo = np.zeros(n, np.uint32); To = np.zeros(n, np.uint64); rc = np.zeros(n, np.int32)
        L = lib(); L.orc_batch_next_event_poisson.restype = None
        L.orc_batch_next_event_poisson.argtypes = [C.c_void_p, C.c_uint64] + [C.c_void_p] * 8 + [C.c_uint64]
        L.orc_batch_next_event_poisson(self._h, int(seed), _ptr(loc), _ptr(cell), _ptr(k), _ptr(f_last), _ptr(ko), _ptr(jo), _ptr(To), _ptr(rc), n)
        return ko, jo, To, rc

    def disperse(self, seed, loc, k, j):
        out = C.c_uint32()
        rc = lib().orc_debug_disperse(self._h, int(seed), 0.0, int(loc), int(k), int(j), C.byref(out))
        if rc != 0: raise RuntimeError("disperse rc=%d" % rc)
        return out.value

    def simulate_stream(self, seed, nu, mask=None, capacity=10_000_000, **kw):
        """simulate() with exact dedup plus the full event stream: dict gains `stream`, a structured array
        (loc, k, j, f, loc2) of the distinct executed events sorted by (k, f, loc, j); loc2 = 0xFFFFFFFF marks a speciation."""
        L = lib()
        L.orc_set_event_sink.restype = None; L.orc_set_event_sink.argtypes = [C.c_void_p] * 5 + [C.c_uint64, C.c_void_p]
        a = [np.zeros(capacity, np.uint32) for _ in range(3)]; f = np.zeros(capacity, np.uint64); l2 = np.zeros(capacity, np.uint32)
        n = C.c_uint64()
        L.orc_set_event_sink(_ptr(a[0]), _ptr(a[1]), _ptr(a[2]), _ptr(f), _ptr(l2), capacity, C.byref(n))
        try:
            out = self.simulate(seed, nu, mask, dedup=True, **kw)
        finally:
            L.orc_set_event_sink(None, None, None, None, None, 0, None)
        if n.value > capacity:
            raise RuntimeError("event stream capacity exceeded: %d" % n.value)
        m = n.value
        st = np.zeros(m, dtype=[("loc", "<u4"), ("k", "<u4"), ("j", "<u4"), ("f", "<u8"), ("loc2", "<u4")])
        st["loc"], st["k"], st["j"], st["f"], st["loc2"] = a[0][:m], a[1][:m], a[2][:m], f[:m], l2[:m]
        out["stream"] = st[np.lexsort((st["j"], st["loc"], st["f"], st["k"]))]
        return out

    def simulate(self, seed, nu, mask=None, dedup=True, epoch_events=0, max_steps=0, per_lineage=False):
        """Returns dict(events, labels, richness, stats[, per_lineage, steps])."""
        n_ind = self.n_individuals
        if mask is not None:
            mask = np.ascontiguousarray(mask, dtype=np.uint8)
            assert mask.shape == (n_ind,)
            ns = int(np.count_nonzero(mask))
        else:
            ns = n_ind
        labels = np.zeros(ns, dtype=np.uint32)
        events = np.zeros(ns, dtype=EVENT_DTYPE)
        pl = np.zeros(ns, dtype=KEY_DTYPE) if per_lineage else None
        st = np.zeros(ns, dtype=np.uint32) if per_lineage else None
        stats = Stats()
        rc = lib().orc_simulate(self._h, int(seed), float(nu), _ptr(mask), 1 if dedup else 0, int(epoch_events),
                                int(max_steps), _ptr(labels), _ptr(events), _ptr(pl), _ptr(st), C.byref(stats))
        if rc != 0:
            raise RuntimeError("orc_simulate rc=%d" % rc)
        out = dict(events=events[: stats.richness].copy(), labels=labels, richness=int(stats.richness),
                   stats={n: int(getattr(stats, n)) for n, _ in Stats._fields_})
        if per_lineage:
            out["per_lineage"] = pl; out["steps"] = st
        return out


# ---- vectorised primitives --------------------------------------------------------------------
LANES = dict(time=0, spec=1, disp=2, index=3, migr=4, state=5)

def _u32(a, n=None):
    a = np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.uint32), (n,) if n is not None else np.shape(a)))
    return a

def batch_draw(seed, lane, loc, k, j, r=None):
    loc = np.ascontiguousarray(loc, dtype=np.uint32); n = len(loc)
    k = _u32(k, n); j = _u32(j, n); rr = None if r is None else _u32(r, n)
    out = np.zeros(n, dtype=np.uint64)
    L = lib(); L.orc_batch_draw.restype = None
    L.orc_batch_draw.argtypes = [C.c_uint64, C.c_int] + [C.c_void_p] * 5 + [C.c_uint64]
    L.orc_batch_draw(int(seed), LANES[lane], _ptr(loc), _ptr(k), _ptr(j), _ptr(rr), _ptr(out), n)
    return out

def batch_F(x):
    x = np.ascontiguousarray(x, dtype=np.uint64); out = np.zeros_like(x)
    L = lib(); L.orc_batch_F.restype = None; L.orc_batch_F.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
    L.orc_batch_F(_ptr(x), _ptr(out), len(x)); return out

def batch_neglog(x):
    x = np.ascontiguousarray(x, dtype=np.uint64); out = np.zeros_like(x)
    L = lib(); L.orc_batch_neglog.restype = None; L.orc_batch_neglog.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
    L.orc_batch_neglog(_ptr(x), _ptr(out), len(x)); return out

def batch_next_event(seed, loc, k, f_last, Cm, sh):
    loc = np.ascontiguousarray(loc, dtype=np.uint32); n = len(loc)
    k = _u32(k, n); Cm = _u32(Cm, n); sh = _u32(sh, n)
    f_last = np.ascontiguousarray(np.broadcast_to(np.asarray(f_last, dtype=np.int64), (n,)))
    ko = np.zeros(n, np.uint32); jo = np.zeros(n, np.uint32); To = np.zeros(n, np.uint64); rc = np.zeros(n, np.int32)
    L = lib(); L.orc_batch_next_event.restype = None
    L.orc_batch_next_event.argtypes = [C.c_uint64] + [C.c_void_p] * 9 + [C.c_uint64]
    L.orc_batch_next_event(int(seed), _ptr(loc), _ptr(k), _ptr(f_last), _ptr(Cm), _ptr(sh), _ptr(ko), _ptr(jo), _ptr(To), _ptr(rc), n)
    return ko, jo, To, rc

def batch_disperse(sc, seed, loc, k, j):
    loc = np.ascontiguousarray(loc, dtype=np.uint32); n = len(loc)
    k = _u32(k, n); j = _u32(j, n)
    out = np.zeros(n, np.uint32); rc = np.zeros(n, np.int32)
    L = lib(); L.orc_batch_disperse.restype = None
    L.orc_batch_disperse.argtypes = [C.c_void_p, C.c_uint64] + [C.c_void_p] * 5 + [C.c_uint64]
    L.orc_batch_disperse(sc._h, int(seed), _ptr(loc), _ptr(k), _ptr(j), _ptr(out), _ptr(rc), n)
    if (rc != 0).any(): raise RuntimeError("disperse failed")
    return out
