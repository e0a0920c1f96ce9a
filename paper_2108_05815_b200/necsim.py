"""ctypes binding of include/necsim.h (libnecsim_b200.so). Argument marshalling only: every step of the
hot path runs in the CUDA kernels of csrc/. torch is used for device memory and streams.

There is no CPU fallback: importing works anywhere, but every compute call raises without the built
library and a CUDA device.
"""
import ctypes as C
import os

import numpy as np

NONSPATIAL, SPATIALLY_IMPLICIT, EXPLICIT_MATRIX, EXPLICIT_GAUSSIAN = 0, 1, 2, 3
_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libnecsim_b200.so")

EXPORTS = ["necsim_scenario_workspace_size", "necsim_create_scenario", "necsim_scenario_num_individuals",
           "necsim_simulate_workspace_size", "necsim_simulate", "necsim_simulate_host", "necsim_destroy", "necsim_last_error",
           "necsim_debug_draw", "necsim_debug_neglog", "necsim_debug_next_event", "necsim_debug_disperse", "necsim_debug_tables",
           "necsim_debug_int_peak", "necsim_debug_next_event_poisson", "necsim_debug_poisson_table",
           "necsim_merge_workspace_size", "necsim_merge_species", "necsim_merge_species_static", "necsim_debug_approx_time", "necsim_debug_gather_peak"]


class ScenarioDesc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("width", C.c_uint32), ("height", C.c_uint32), ("sampler", C.c_uint32), ("deme", C.c_void_p),
                ("uniform_deme", C.c_uint32), ("turnover", C.c_void_p), ("uniform_turnover", C.c_double),
                ("dispersal_matrix", C.c_void_p), ("sigma", C.c_double), ("local_size", C.c_uint64),
                ("meta_size", C.c_uint64), ("migration", C.c_double), ("delta_t", C.c_double),
                ("n_past_eras", C.c_uint32), ("past_deme", C.c_void_p), ("past_start_k", C.c_void_p)]


class SimParams(C.Structure):
    _fields_ = [("block_threads", C.c_uint32), ("grid_blocks", C.c_uint32), ("dedup", C.c_uint32),
                ("dedup_log2_slots", C.c_uint32), ("epoch_events", C.c_uint64), ("max_steps", C.c_uint64),
                ("tail_threshold", C.c_uint32), ("dedup_probe", C.c_uint32), ("record_events", C.c_uint32), ("stream_sort_bytes", C.c_uint32),
                ("event_ring_capacity", C.c_uint64), ("event_stream_capacity", C.c_uint64)]


class Result(C.Structure):
    _fields_ = [("richness", C.c_uint64), ("n_lineages", C.c_uint64), ("n_unfinished", C.c_uint64),
                ("d_events", C.c_void_p), ("d_labels", C.c_void_p),
                ("d_term_loc", C.c_void_p), ("d_term_k", C.c_void_p), ("d_term_j", C.c_void_p), ("d_steps", C.c_void_p),
                ("d_term_f", C.c_void_p), ("d_state", C.c_void_p),
                ("n_events_raw", C.c_uint64), ("n_culled", C.c_uint64), ("n_speciation_raw", C.c_uint64),
                ("n_epochs", C.c_uint64), ("n_tail_epochs", C.c_uint64), ("resample_attempts", C.c_uint64),
                ("n_events_tail", C.c_uint64), ("ms_simulate", C.c_float), ("ms_simulate_tail", C.c_float),
                ("ms_total", C.c_float), ("n_kernel_launches", C.c_uint32),
                ("d_stream_loc", C.c_void_p), ("d_stream_k", C.c_void_p), ("d_stream_j", C.c_void_p), ("d_stream_loc2", C.c_void_p),
                ("d_stream_f", C.c_void_p), ("n_stream_events", C.c_uint64), ("n_tail_rounds_exact", C.c_uint64)]


EVENT_DTYPE = np.dtype({"names": ["loc", "k", "j", "abundance", "f", "time"],
                        "formats": ["<u4", "<u4", "<u4", "<u4", "<u8", "<f8"], "offsets": [0, 4, 8, 12, 16, 24], "itemsize": 32})

_lib = None


class NecsimError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("necsim error %d: %s" % (code, msg))
        self.code = code


def lib():
    """Loads the C-ABI library (fails loudly if it was not built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libnecsim_b200.so is not built: run `python -m paper_2108_05815_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.necsim_last_error.restype = C.c_char_p
        for name in EXPORTS:
            if name != "necsim_last_error":
                getattr(L, name).restype = C.c_int
        vp, u64, u32, dbl = C.c_void_p, C.c_uint64, C.c_uint32, C.c_double
        L.necsim_scenario_workspace_size.argtypes = [vp, vp]
        L.necsim_create_scenario.argtypes = [vp, vp, C.c_size_t, vp, vp]
        L.necsim_scenario_num_individuals.argtypes = [vp, vp]
        L.necsim_simulate_workspace_size.argtypes = [vp, u64, vp, vp]
        L.necsim_simulate.argtypes = [vp, u64, dbl, vp, u64, vp, vp, C.c_size_t, vp, vp]
        L.necsim_simulate_host.argtypes = [vp, u64, dbl, vp, u64, vp, vp, C.c_size_t, vp, vp, vp, vp]
        L.necsim_destroy.argtypes = [vp]
        L.necsim_debug_draw.argtypes = [u64, C.c_int, vp, vp, vp, vp, vp, u64, vp]
        L.necsim_debug_neglog.argtypes = [vp, vp, u64, vp]
        L.necsim_debug_next_event.argtypes = [u64] + [vp] * 9 + [u64, vp]
        L.necsim_debug_disperse.argtypes = [vp, u64, vp, vp, vp, vp, u64, vp]
        L.necsim_debug_tables.argtypes = [vp] * 8
        L.necsim_debug_int_peak.argtypes = [C.c_int, u32, vp, vp, vp, vp]
        L.necsim_debug_next_event_poisson.argtypes = [vp, u64] + [vp] * 8 + [u64, vp]
        L.necsim_debug_poisson_table.argtypes = [vp] * 5
        L.necsim_debug_approx_time.argtypes = [vp, u32, u32, vp, vp, vp, u64, vp]
        L.necsim_debug_gather_peak.argtypes = [vp, u64, u32, vp, vp, vp, vp]
        L.necsim_merge_workspace_size.argtypes = [u64, vp]
        L.necsim_merge_species.argtypes = [vp, u64, vp, C.c_size_t, vp, vp, vp, vp]
        L.necsim_merge_species_static.argtypes = [vp, u64, vp, vp, vp, vp]
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise NecsimError(rc, lib().necsim_last_error().decode())


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("necsim needs a CUDA device (there is no CPU fallback)")
    return torch


def _stream_ptr(torch):
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _hptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dev_u32(torch, a, n=None):
    """numpy / scalar -> contiguous device tensor holding the u32 bit patterns (int32 storage)."""
    a = np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.uint32), (n,) if n is not None else np.shape(a)))
    return torch.from_numpy(a.view(np.int32)).cuda()


def make_params(block_threads=0, grid_blocks=0, dedup=None, dedup_log2_slots=0, epoch_events=0, max_steps=0, tail_threshold=0,
                dedup_probe=0, record_events=False, event_ring_capacity=0, event_stream_capacity=0, stream_sort_bytes=0):
    p = SimParams()
    p.block_threads, p.grid_blocks = block_threads, grid_blocks
    p.dedup = 0 if dedup is None else (1 if dedup else 2)
    p.dedup_log2_slots, p.epoch_events, p.max_steps, p.tail_threshold = dedup_log2_slots, epoch_events, max_steps, tail_threshold
    p.dedup_probe = dedup_probe
    p.record_events = 1 if record_events else 0
    p.stream_sort_bytes = int(stream_sort_bytes)
    p.event_ring_capacity, p.event_stream_capacity = int(event_ring_capacity), int(event_stream_capacity)
    return p


class Scenario:
    """necsim_create_scenario / necsim_simulate / necsim_destroy (include/necsim.h)."""

    def __init__(self, kind, width=1, height=1, deme=None, uniform_deme=0, turnover=None, uniform_turnover=1.0, matrix=None,
                 sigma=0.0, local_size=0, meta_size=0, migration=0.0, delta_t=2.0, sampler=0, past_deme=None, past_start_k=None):
        torch = _torch()
        L = lib()
        self._h = None
        d = ScenarioDesc()
        keep = []
        d.kind, d.width, d.height, d.sampler = int(kind), int(width), int(height), int(sampler)
        if deme is not None:
            a = np.ascontiguousarray(deme, dtype=np.uint32).ravel(); keep.append(a); d.deme = a.ctypes.data
        d.uniform_deme = int(uniform_deme)
        if turnover is not None:
            a = np.ascontiguousarray(turnover, dtype=np.float64).ravel(); keep.append(a); d.turnover = a.ctypes.data
        d.uniform_turnover = float(uniform_turnover)
        if matrix is not None:
            a = np.ascontiguousarray(matrix, dtype=np.float64); keep.append(a); d.dispersal_matrix = a.ctypes.data
        d.sigma, d.local_size, d.meta_size = float(sigma), int(local_size), int(meta_size)
        d.migration, d.delta_t = float(migration), float(delta_t)
        if past_deme is not None:   # temporally varying habitat
            pd = np.ascontiguousarray(past_deme, dtype=np.uint32).reshape(-1, int(width) * int(height)); keep.append(pd)
            ps = np.ascontiguousarray(past_start_k, dtype=np.uint32).ravel(); keep.append(ps)
            assert len(ps) == pd.shape[0]
            d.n_past_eras, d.past_deme, d.past_start_k = pd.shape[0], pd.ctypes.data, ps.ctypes.data
        nbytes = C.c_size_t()
        _check(L.necsim_scenario_workspace_size(C.byref(d), C.byref(nbytes)))
        self._ws = torch.empty(max(nbytes.value, 256), dtype=torch.uint8, device="cuda")
        h = C.c_void_p()
        _check(L.necsim_create_scenario(C.byref(d), C.c_void_p(self._ws.data_ptr()), nbytes.value, _stream_ptr(torch), C.byref(h)))
        self._h = h
        n = C.c_uint64()
        _check(L.necsim_scenario_num_individuals(self._h, C.byref(n)))
        self.n_individuals = n.value
        self.kind, self.ncells, self.delta_t = int(kind), (2 if kind == SPATIALLY_IMPLICIT else int(width) * int(height)), float(delta_t)
        self._sim_ws = None

    def close(self):
        if getattr(self, "_h", None):
            lib().necsim_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:       # interpreter shutdown: the module globals may be gone already
            pass

    def _workspace(self, cap, params):
        torch = _torch()
        nbytes = C.c_size_t()
        _check(lib().necsim_simulate_workspace_size(self._h, cap, C.byref(params), C.byref(nbytes)))
        if self._sim_ws is None or self._sim_ws.numel() < nbytes.value:
            self._sim_ws = None
            self._sim_ws = torch.empty(nbytes.value, dtype=torch.uint8, device="cuda")
        return self._sim_ws

    def simulate_raw(self, seed, nu, d_mask=None, n_sampled=None, params=None):
        """Device in, device out: d_mask is a torch uint8 CUDA tensor (or None). Returns the Result struct."""
        torch = _torch()
        params = params if params is not None else SimParams()
        cap = int(n_sampled) if n_sampled is not None else self.n_individuals
        ws = self._workspace(cap, params)
        res = Result()
        mp = None if d_mask is None else C.c_void_p(d_mask.data_ptr())
        _check(lib().necsim_simulate(self._h, int(seed), float(nu), mp, cap, C.byref(params), C.c_void_p(ws.data_ptr()), ws.numel(),
                                     _stream_ptr(torch), C.byref(res)))
        return res

    def simulate_host_raw(self, seed, nu, h_mask, n_sampled, params, h_events, h_labels):
        """Host in, host out (pinned numpy views): the end-to-end entry point necsim_simulate_host."""
        torch = _torch()
        params = params if params is not None else SimParams()
        ws = self._workspace(int(n_sampled), params)
        res = Result()
        _check(lib().necsim_simulate_host(self._h, int(seed), float(nu), _hptr(h_mask), int(n_sampled), C.byref(params),
                                          C.c_void_p(ws.data_ptr()), ws.numel(), _stream_ptr(torch), C.byref(res), _hptr(h_events),
                                          _hptr(h_labels)))
        return res

    def result_tensors(self, res):
        """CUDA views (no copy) of a Result's species table (uint8 [richness * 32]) and labels (int32 [n_lineages]) inside the workspace."""
        ws = self._sim_ws
        eo, lo = int(res.d_events) - ws.data_ptr(), int(res.d_labels) - ws.data_ptr()
        return ws[eo:eo + int(res.richness) * 32], ws[lo:lo + int(res.n_lineages) * 4].view(_torch().int32)

    def simulate(self, seed, nu, mask=None, per_lineage=False, **param_kw):
        """Convenience: numpy mask in, numpy results out. dict(events, labels, richness, stats[, per_lineage, steps, state])."""
        torch = _torch()
        params = make_params(**param_kw)
        d_mask, ns = None, self.n_individuals
        if mask is not None:
            m = np.ascontiguousarray(mask, dtype=np.uint8)
            assert m.shape == (self.n_individuals,)
            ns = max(int(np.count_nonzero(m)), 1)
            d_mask = torch.from_numpy(m).cuda()
        res = self.simulate_raw(seed, nu, d_mask, ns, params)
        n, S = int(res.n_lineages), int(res.richness)
        out = dict(richness=S, events=_read(self._sim_ws, res.d_events, S * 32, np.uint8).view(EVENT_DTYPE) if S else np.zeros(0, EVENT_DTYPE),
                   labels=_read(self._sim_ws, res.d_labels, n * 4, np.uint32),
                   stats={k: getattr(res, k) for k in ("n_lineages", "n_unfinished", "n_events_raw", "n_culled", "n_speciation_raw",
                                                       "n_epochs", "n_tail_epochs", "resample_attempts", "n_events_tail", "ms_simulate",
                                                       "ms_simulate_tail", "ms_total", "n_kernel_launches", "n_stream_events", "n_tail_rounds_exact")})
        if params.record_events:
            m = int(res.n_stream_events)
            st = np.zeros(m, dtype=[("loc", "<u4"), ("k", "<u4"), ("j", "<u4"), ("f", "<u8"), ("loc2", "<u4")])
            for name, ptr, dt, w in (("loc", res.d_stream_loc, np.uint32, 4), ("k", res.d_stream_k, np.uint32, 4), ("j", res.d_stream_j, np.uint32, 4),
                                     ("f", res.d_stream_f, np.uint64, 8), ("loc2", res.d_stream_loc2, np.uint32, 4)):
                st[name] = _read(self._sim_ws, ptr, m * w, dt)
            out["stream"] = st
        if per_lineage:
            pl = np.zeros(n, dtype=[("loc", "<u4"), ("k", "<u4"), ("j", "<u4"), ("f", "<u8")])
            pl["loc"] = _read(self._sim_ws, res.d_term_loc, n * 4, np.uint32); pl["k"] = _read(self._sim_ws, res.d_term_k, n * 4, np.uint32)
            pl["j"] = _read(self._sim_ws, res.d_term_j, n * 4, np.uint32); pl["f"] = _read(self._sim_ws, res.d_term_f, n * 8, np.uint64)
            out["per_lineage"] = pl
            out["steps"] = _read(self._sim_ws, res.d_steps, n * 4, np.uint32)
            out["state"] = _read(self._sim_ws, res.d_state, n, np.uint8)
        return out

    # ---- test-only -----------------------------------------------------------------------------------
    def debug_next_event_poisson(self, seed, loc, cell, k, f_last):
        torch = _torch()
        loc = np.ascontiguousarray(loc, dtype=np.uint32); n = len(loc)
        dl, dc, dk = _dev_u32(torch, loc), _dev_u32(torch, cell, n), _dev_u32(torch, k, n)
        df = torch.from_numpy(np.ascontiguousarray(np.broadcast_to(np.asarray(f_last, dtype=np.int64), (n,)))).cuda()
        ko = torch.empty(n, dtype=torch.int32, device="cuda"); jo = torch.empty_like(ko); rc = torch.empty_like(ko)
        To = torch.empty(n, dtype=torch.int64, device="cuda")
        _check(lib().necsim_debug_next_event_poisson(self._h, int(seed), dl.data_ptr(), dc.data_ptr(), dk.data_ptr(), df.data_ptr(), ko.data_ptr(),
                                                     jo.data_ptr(), To.data_ptr(), rc.data_ptr(), n, _stream_ptr(torch)))
        return (ko.cpu().numpy().view(np.uint32), jo.cpu().numpy().view(np.uint32), To.cpu().numpy().view(np.uint64), rc.cpu().numpy())

    def debug_poisson_table(self):
        torch = _torch()
        pc = np.zeros(256, np.uint64); thin = np.zeros(self.ncells, np.uint32); mu = C.c_double()
        _check(lib().necsim_debug_poisson_table(self._h, _hptr(pc), _hptr(thin), C.byref(mu), _stream_ptr(torch)))
        return mu.value, pc, thin

    def debug_disperse(self, seed, loc, k, j):
        torch = _torch()
        loc = np.ascontiguousarray(loc, dtype=np.uint32); n = len(loc)
        dl, dk, dj = _dev_u32(torch, loc), _dev_u32(torch, k, n), _dev_u32(torch, j, n)
        out = torch.empty(n, dtype=torch.int32, device="cuda")
        _check(lib().necsim_debug_disperse(self._h, int(seed), dl.data_ptr(), dk.data_ptr(), dj.data_ptr(), out.data_ptr(), n, _stream_ptr(torch)))
        return out.cpu().numpy().view(np.uint32)

    def debug_tables(self):
        torch = _torch()
        n = self.ncells
        out = {}
        th = al = None
        if self.kind == EXPLICIT_MATRIX:
            th = np.zeros((n, n), np.uint32); al = np.zeros((n, n), np.uint32)
        R = C.c_int32()
        g = np.zeros(2048, np.uint32)
        cm, sh = np.zeros(n, np.uint32), np.zeros(n, np.uint32)
        _check(lib().necsim_debug_tables(self._h, _hptr(th), _hptr(al), _hptr(g), C.byref(R), _hptr(cm), _hptr(sh), _stream_ptr(torch)))
        out.update(thresh=th, alias=al, R=R.value, gauss=g[: 2 * R.value].copy(), Cm=cm, sh=sh)
        return out


def _read(ws, ptr, nbytes, dtype):
    """Result pointers point into the caller's workspace tensor `ws`: slice it and copy to the host."""
    if nbytes == 0 or not ptr:
        return np.zeros(0, dtype)
    off = int(ptr) - ws.data_ptr()
    assert 0 <= off and off + nbytes <= ws.numel(), "result pointer outside the workspace"
    return ws[off:off + nbytes].cpu().numpy().view(dtype).copy()


def merge_species(d_events):
    """necsim_merge_species: d_events = CUDA uint8 tensor holding n necsim_event records (the concatenated species tables
    of isolated partitions). Returns (merged table as a CUDA uint8 tensor [richness * 32], map as a CUDA int64 tensor [n])."""
    torch = _torch()
    assert d_events.is_cuda and d_events.dtype == torch.uint8 and d_events.numel() % 32 == 0
    n = d_events.numel() // 32
    d_events = d_events.contiguous()
    nbytes = C.c_size_t()
    _check(lib().necsim_merge_workspace_size(n, C.byref(nbytes)))
    ws = torch.empty(nbytes.value, dtype=torch.uint8, device="cuda")
    out = torch.empty(n * 32, dtype=torch.uint8, device="cuda")
    dmap = torch.empty(n, dtype=torch.int32, device="cuda")
    rich = C.c_uint64()
    _check(lib().necsim_merge_species(C.c_void_p(d_events.data_ptr()), n, C.c_void_p(ws.data_ptr()), ws.numel(), _stream_ptr(torch),
                                      C.c_void_p(out.data_ptr()), C.c_void_p(dmap.data_ptr()), C.byref(rich)))
    return out[: rich.value * 32], dmap.to(torch.int64)


MERGE_STATIC_MAX = 65536   # NECSIM_MERGE_STATIC_MAX of include/necsim.h


def merge_species_static(d_events, out=None, dmap=None):
    """necsim_merge_species_static: the merge with the library's static scratch (no workspace, nothing allocated by the call when
    `out` [n * 32] uint8 and `dmap` [n] int32 are passed in). Returns (merged table [richness * 32] uint8, map [n] int32) as views."""
    torch = _torch()
    assert d_events.is_cuda and d_events.dtype == torch.uint8 and d_events.numel() % 32 == 0 and d_events.is_contiguous()
    n = d_events.numel() // 32
    if out is None: out = torch.empty(n * 32, dtype=torch.uint8, device="cuda")
    if dmap is None: dmap = torch.empty(n, dtype=torch.int32, device="cuda")
    assert out.numel() >= n * 32 and dmap.numel() >= n
    rich = C.c_uint64()
    _check(lib().necsim_merge_species_static(C.c_void_p(d_events.data_ptr()), n, _stream_ptr(torch), C.c_void_p(out.data_ptr()),
                                             C.c_void_p(dmap.data_ptr()), C.byref(rich)))
    return out[: rich.value * 32], dmap[:n]


# ---- vectorised device primitives (test-only exports) ------------------------------------------------
LANES = dict(time=0, spec=1, disp=2, index=3, migr=4, state=5)


def debug_draw(seed, lane, loc, k, j, r=None):
    torch = _torch()
    loc = np.ascontiguousarray(loc, dtype=np.uint32); n = len(loc)
    dl, dk, dj = _dev_u32(torch, loc), _dev_u32(torch, k, n), _dev_u32(torch, j, n)
    dr = None if r is None else _dev_u32(torch, r, n)
    out = torch.empty(n, dtype=torch.int64, device="cuda")
    _check(lib().necsim_debug_draw(int(seed), LANES[lane], dl.data_ptr(), dk.data_ptr(), dj.data_ptr(), None if dr is None else dr.data_ptr(),
                                   out.data_ptr(), n, _stream_ptr(torch)))
    return out.cpu().numpy().view(np.uint64)


def debug_neglog(x):
    torch = _torch()
    x = np.ascontiguousarray(x, dtype=np.uint64)
    dx = torch.from_numpy(x.view(np.int64)).cuda()
    out = torch.empty_like(dx)
    _check(lib().necsim_debug_neglog(dx.data_ptr(), out.data_ptr(), len(x), _stream_ptr(torch)))
    return out.cpu().numpy().view(np.uint64)


def debug_approx_time(x, Cm, sh):
    """(binary32 offsets of the fast round, exact Q16.48 offsets, the kernel's margin) for an array of 64-bit draws."""
    torch = _torch()
    x = np.ascontiguousarray(x, dtype=np.uint64)
    dx = torch.from_numpy(x.view(np.int64)).cuda()
    ap = torch.empty(len(x), dtype=torch.float32, device="cuda"); ex = torch.empty_like(dx); mg = torch.zeros(1, dtype=torch.float32, device="cuda")
    _check(lib().necsim_debug_approx_time(dx.data_ptr(), int(Cm), int(sh), ap.data_ptr(), ex.data_ptr(), mg.data_ptr(), len(x), _stream_ptr(torch)))
    return ap.cpu().numpy(), ex.cpu().numpy().view(np.uint64), float(mg.item())


def debug_next_event(seed, loc, k, f_last, Cm, sh):
    torch = _torch()
    loc = np.ascontiguousarray(loc, dtype=np.uint32); n = len(loc)
    dl, dk, dc, ds = _dev_u32(torch, loc), _dev_u32(torch, k, n), _dev_u32(torch, Cm, n), _dev_u32(torch, sh, n)
    df = torch.from_numpy(np.ascontiguousarray(np.broadcast_to(np.asarray(f_last, dtype=np.int64), (n,)))).cuda()
    ko = torch.empty(n, dtype=torch.int32, device="cuda"); jo = torch.empty_like(ko); rc = torch.empty_like(ko)
    To = torch.empty(n, dtype=torch.int64, device="cuda")
    _check(lib().necsim_debug_next_event(int(seed), dl.data_ptr(), dk.data_ptr(), df.data_ptr(), dc.data_ptr(), ds.data_ptr(), ko.data_ptr(),
                                         jo.data_ptr(), To.data_ptr(), rc.data_ptr(), n, _stream_ptr(torch)))
    return (ko.cpu().numpy().view(np.uint32), jo.cpu().numpy().view(np.uint32), To.cpu().numpy().view(np.uint64), rc.cpu().numpy())


def gather_peak(table_bytes, loads_per_thread=256):
    """Random 32-byte-sector gather micro-benchmark over a table of table_bytes: returns (sector bytes per second, ms)."""
    torch = _torch()
    table = torch.zeros(int(table_bytes), dtype=torch.uint8, device="cuda")
    sink = torch.zeros(1, dtype=torch.int32, device="cuda")
    v, ms = C.c_double(), C.c_float()
    _check(lib().necsim_debug_gather_peak(C.c_void_p(table.data_ptr()), int(table_bytes), int(loads_per_thread), C.c_void_p(sink.data_ptr()),
                                          _stream_ptr(torch), C.byref(v), C.byref(ms)))
    return v.value, ms.value


def int_peak(kind, iters=4096):
    """Integer-pipe micro-benchmark: returns (thread-level integer instructions per second, ms)."""
    torch = _torch()
    v, ms = C.c_double(), C.c_float()
    sink = torch.zeros(1, dtype=torch.int32, device="cuda")
    _check(lib().necsim_debug_int_peak(int(kind), int(iters), C.c_void_p(sink.data_ptr()), _stream_ptr(torch), C.byref(v), C.byref(ms)))
    return v.value, ms.value
