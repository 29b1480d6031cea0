"""Thin ctypes binding of libgcmcrt.so (include/gcmcrt.h): argument marshalling only.

Every step of the method runs inside the library's CUDA kernels.  Arrays may be numpy arrays (host memory) or torch
tensors (host or CUDA memory); torch is used for device memory and streams only.  If the library has not been built
(`python -m paper_2110_15640_b200.build`) or cannot be loaded, every call raises -- there is no CPU fallback.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# GCMCRT_LIB selects another build of the same library (the checked variant, build.py --checked)
LIB_PATH = os.environ.get("GCMCRT_LIB") or os.path.join(_HERE, "libgcmcrt.so")
_lib = None

OK, E_INVALID, E_NOMEM, E_CUDA, E_STATE = 0, -1, -2, -3, -4
EXPORTS = ["gcmcrt_grid_create", "gcmcrt_set_opacity", "gcmcrt_set_opacity_nodes", "gcmcrt_run_albedo", "gcmcrt_run_emission",
           "gcmcrt_run_transmission", "gcmcrt_destroy",
           "gcmcrt_last_error", "gcmcrt_debug_ray_tau", "gcmcrt_debug_philox", "gcmcrt_emission_ltot_static", "gcmcrt_version"]


class GcmcrtError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("gcmcrt error %d: %s" % (code, msg))
        self.code = code


class RunParams(C.Structure):
    _fields_ = [("star_dir", C.c_double * 3), ("n_obs", C.c_int), ("obs_dir", C.c_void_p),
                ("packets_per_channel", C.c_uint64), ("pkt_begin", C.c_uint64), ("pkt_end", C.c_uint64),
                ("seed", C.c_uint64), ("chan_begin", C.c_int), ("chan_end", C.c_int),
                ("max_events", C.c_int), ("scatter_on", C.c_int), ("doppler_on", C.c_int),
                ("doppler_halfwidth", C.c_int), ("emission_bias", C.c_double), ("tau_vert_max", C.c_double),
                ("tau_cut", C.c_double), ("npix", C.c_int), ("n_batches", C.c_int),
                ("survival_bias", C.c_int), ("roulette_w_min", C.c_double), ("roulette_survive", C.c_double),
                ("star_radius", C.c_double), ("planet_xy", C.c_double * 2), ("ld_c1", C.c_double), ("ld_c2", C.c_double), ("cloud_phase", C.c_int), ("forced_scatter", C.c_int), ("continuous_absorption", C.c_int),
                ("star_solid_angle", C.c_double), ("stretch_alpha", C.c_double), ("timing", C.c_int), ("concurrency", C.c_int)]


class Counters(C.Structure):
    _fields_ = [("events", C.c_uint64), ("segments_transport", C.c_uint64), ("segments_peel", C.c_uint64),
                ("packets_escaped", C.c_uint64), ("packets_absorbed", C.c_uint64), ("packets_surface", C.c_uint64),
                ("packets_stuck", C.c_uint64), ("escaped_weight", C.c_double), ("passes", C.c_uint64),
                ("rays_peel", C.c_uint64), ("launches", C.c_uint64), ("ms_stage", C.c_double),
                ("ms_emission_cdf", C.c_double), ("ms_transport", C.c_double), ("ms_peel", C.c_double),
                ("ms_sort", C.c_double), ("device_status", C.c_uint64)]


class Result(C.Structure):
    _fields_ = [("flux_sum", C.c_void_p), ("L_tot", C.c_void_p), ("value", C.c_void_p), ("sigma", C.c_void_p),
                ("image", C.c_void_p), ("event_count", C.c_void_p), ("counters", C.c_void_p),
                ("contrib", C.c_void_p)]


def lib():
    """Load libgcmcrt.so; raises if it is missing (the product has no other execution path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise GcmcrtError(E_STATE, "libgcmcrt.so is not built: run `python -m paper_2110_15640_b200.build` "
                                       "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.gcmcrt_last_error.restype = C.c_char_p
        L.gcmcrt_last_error.argtypes = [C.c_void_p]
        L.gcmcrt_version.restype = C.c_char_p
        L.gcmcrt_grid_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int] + [C.c_void_p] * 8 + \
            [C.c_double, C.c_float, C.c_void_p]
        L.gcmcrt_set_opacity.argtypes = [C.c_void_p, C.c_int, C.c_int] + [C.c_void_p] * 6
        L.gcmcrt_set_opacity_nodes.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_int] + \
            [C.c_void_p] * 7
        L.gcmcrt_run_albedo.argtypes = [C.c_void_p, C.POINTER(RunParams), C.POINTER(Result), C.c_void_p]
        L.gcmcrt_run_emission.argtypes = [C.c_void_p, C.POINTER(RunParams), C.POINTER(Result), C.c_void_p]
        L.gcmcrt_run_transmission.argtypes = [C.c_void_p, C.POINTER(RunParams), C.POINTER(Result), C.c_void_p]
        L.gcmcrt_destroy.argtypes = [C.c_void_p]
        L.gcmcrt_debug_ray_tau.argtypes = [C.c_void_p, C.c_int, C.c_long] + [C.c_void_p] * 5
        L.gcmcrt_debug_philox.argtypes = [C.c_long] + [C.c_void_p] * 4
        L.gcmcrt_emission_ltot_static.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _is_torch(x):
    return type(x).__module__.startswith("torch")


def _ptr(x, dtype=None):
    """Address of a contiguous numpy array or torch tensor (or None)."""
    if x is None:
        return None
    if _is_torch(x):
        if not x.is_contiguous():
            raise ValueError("tensor must be contiguous")
        if dtype is not None and str(x.dtype).replace("torch.", "") != np.dtype(dtype).name:
            raise ValueError("tensor dtype %s, expected %s" % (x.dtype, np.dtype(dtype).name))
        return x.data_ptr()
    if not isinstance(x, np.ndarray) or not x.flags["C_CONTIGUOUS"]:
        raise ValueError("array must be a C-contiguous numpy array or torch tensor")
    if dtype is not None and x.dtype != np.dtype(dtype):
        raise ValueError("array dtype %s, expected %s" % (x.dtype, np.dtype(dtype).name))
    return x.ctypes.data


def _stream_ptr(stream):
    if stream is None:
        return None
    return getattr(stream, "cuda_stream", stream)


def _check(handle, rc):
    if rc != 0:
        raise GcmcrtError(rc, lib().gcmcrt_last_error(handle).decode())


# --------------------------------------------------------------------------- the C-ABI calls, same names
def version():
    return lib().gcmcrt_version().decode()


def grid_create(r_edges, colat_edges, lon_edges, T, rho, u=None, v=None, w=None, Omega=0.0, surface_albedo=0.0,
                stream=None):
    r = np.ascontiguousarray(r_edges, dtype=np.float64)
    th = np.ascontiguousarray(colat_edges, dtype=np.float64)
    ph = np.ascontiguousarray(lon_edges, dtype=np.float64)
    h = C.c_void_p()
    rc = lib().gcmcrt_grid_create(C.byref(h), r.size - 1, th.size - 1, ph.size - 1, _ptr(r), _ptr(th), _ptr(ph),
                                  _ptr(T, np.float32), _ptr(rho, np.float32), _ptr(u, np.float32), _ptr(v, np.float32),
                                  _ptr(w, np.float32), float(Omega), float(surface_albedo), _stream_ptr(stream))
    _check(None, rc)
    return h


def set_opacity(handle, chan0, lam, k_abs, k_sca_ray=None, k_sca_cld=None, g_cld=None, stream=None):
    lam = np.ascontiguousarray(lam, dtype=np.float32)
    rc = lib().gcmcrt_set_opacity(handle, int(chan0), lam.size, _ptr(lam), _ptr(k_abs, np.float32),
                                  _ptr(k_sca_ray, np.float32), _ptr(k_sca_cld, np.float32), _ptr(g_cld, np.float32),
                                  _stream_ptr(stream))
    _check(handle, rc)


def set_opacity_nodes(handle, chan0, lam, node_kabs, T_nodes, logp_nodes, p_cell, k_sca_ray=None, k_sca_cld=None,
                      g_cld=None, stream=None):
    lam = np.ascontiguousarray(lam, dtype=np.float32)
    tn = np.ascontiguousarray(T_nodes, dtype=np.float32)
    lpn = np.ascontiguousarray(logp_nodes, dtype=np.float32)
    rc = lib().gcmcrt_set_opacity_nodes(handle, int(chan0), lam.size, _ptr(lam), _ptr(node_kabs, np.float32), tn.size,
                                        lpn.size, _ptr(tn), _ptr(lpn), _ptr(p_cell, np.float32),
                                        _ptr(k_sca_ray, np.float32), _ptr(k_sca_cld, np.float32), _ptr(g_cld, np.float32),
                                        _stream_ptr(stream))
    _check(handle, rc)


def destroy(handle):
    if handle:
        lib().gcmcrt_destroy(handle)


def make_params(prm):
    """dict (names of gcmcrt_run_params) -> (RunParams, keepalive)."""
    obs = np.ascontiguousarray(prm.get("obs_dir", np.zeros((0, 3))), dtype=np.float64).reshape(-1, 3)
    p = RunParams()
    p.star_dir[:] = [float(x) for x in prm.get("star_dir", (1.0, 0.0, 0.0))]
    p.n_obs = obs.shape[0]
    p.obs_dir = obs.ctypes.data if obs.size else None
    p.packets_per_channel = int(prm["packets_per_channel"])
    p.pkt_begin = int(prm.get("pkt_begin", 0))
    p.pkt_end = int(prm.get("pkt_end", 0))
    p.seed = int(prm.get("seed", 0))
    p.chan_begin = int(prm.get("chan_begin", 0))
    p.chan_end = int(prm.get("chan_end", 0))
    for name in ("max_events", "doppler_on", "doppler_halfwidth", "npix"):
        setattr(p, name, int(prm.get(name, 0)))
    p.scatter_on = int(prm.get("scatter_on", 1))
    p.emission_bias = float(prm.get("emission_bias", 0.0))
    p.tau_vert_max = float(prm.get("tau_vert_max", 30.0))
    p.tau_cut = float(prm.get("tau_cut", 50.0))
    p.n_batches = int(prm.get("n_batches", 32))
    p.survival_bias = int(prm.get("survival_bias", 0))
    p.roulette_w_min = float(prm.get("roulette_w_min", 0.0))
    p.roulette_survive = float(prm.get("roulette_survive", 0.0))
    p.star_radius = float(prm.get("star_radius", 0.0))
    xy = prm.get("planet_xy", (0.0, 0.0))
    p.planet_xy[0], p.planet_xy[1] = float(xy[0]), float(xy[1])
    p.ld_c1, p.ld_c2 = float(prm.get("ld_c1", 0.0)), float(prm.get("ld_c2", 0.0))
    p.cloud_phase = int(prm.get("cloud_phase", 0))
    p.forced_scatter = int(prm.get("forced_scatter", 0))
    p.continuous_absorption = int(prm.get("continuous_absorption", 0))
    p.star_solid_angle = float(prm.get("star_solid_angle", 0.0))
    p.stretch_alpha = float(prm.get("stretch_alpha", 0.0))
    p.timing = int(prm.get("timing", 0))
    p.concurrency = int(prm.get("concurrency", 0))
    return p, obs


def read_counters(dev_counters):
    """The gcmcrt_counters struct a run wrote into device memory (counters="device"), as a dict.  Synchronises."""
    raw = dev_counters.cpu().numpy().tobytes()
    cnt = Counters.from_buffer_copy(raw)
    return {name: getattr(cnt, name) for name, _ in Counters._fields_}


def _run(fn, handle, prm, n_chan_table, want_event_count, want_image, device_outputs, stream, want_contrib=0,
         counters="host"):
    """counters: "host" (dict in out["counters"]; the call waits for the device), "device" (out["counters_dev"]: a byte
    tensor holding the struct, read it with read_counters(); with device_outputs the call then only enqueues work), or
    None."""
    p, keep = make_params(prm)
    N = p.packets_per_channel
    lo, hi = p.pkt_begin, (p.pkt_end or N)
    cb, ce = p.chan_begin, (p.chan_end or n_chan_table)
    ncr, nobs, nb = max(ce - cb, 0), max(p.n_obs, 1), (p.n_batches or 32)
    hi = max(hi, lo)          # invalid ranges are reported by the library (E_INVALID), not by numpy
    shapes = {"flux_sum": ((ncr, nobs, nb), np.float64), "L_tot": ((ncr, nobs), np.float64),
              "value": ((ncr, nobs), np.float64), "sigma": ((ncr, nobs), np.float64)}
    if want_image and p.npix > 0:
        shapes["image"] = ((ncr, nobs, p.npix, p.npix), np.float32)
    if want_event_count:
        shapes["event_count"] = ((ncr, hi - lo), np.uint32)
    if want_contrib:             # = ncell: contribution functions (Sect. 6, Eq. 32), [chan][obs][thermal|scattered][cell]
        shapes["contrib"] = ((ncr, nobs, 2, int(want_contrib)), np.float32)
    out = {}
    if device_outputs:
        import torch
        tmap = {np.float64: torch.float64, np.float32: torch.float32, np.uint32: torch.int32}
        for k, (shp, dt) in shapes.items():
            out[k] = torch.empty(shp, dtype=tmap[dt], device="cuda")
    else:
        for k, (shp, dt) in shapes.items():
            out[k] = np.zeros(shp, dtype=dt)
    cnt = Counters()
    res = Result()
    for k in ("flux_sum", "L_tot", "value", "sigma", "image", "event_count", "contrib"):
        setattr(res, k, _ptr(out[k]) if k in out else None)
    if counters == "device":
        import torch
        out["counters_dev"] = torch.zeros(C.sizeof(Counters), dtype=torch.uint8, device="cuda")
        res.counters = out["counters_dev"].data_ptr()
    elif counters == "host":
        res.counters = C.addressof(cnt)
    else:
        res.counters = None
    rc = fn(handle, C.byref(p), C.byref(res), _stream_ptr(stream))
    _check(handle, rc)
    if counters == "host":
        out["counters"] = {name: getattr(cnt, name) for name, _ in Counters._fields_}
    out["n_batches"], out["packets_per_channel"], out["pkt_range"] = nb, N, (lo, hi)
    del keep
    return out


def run_albedo(handle, prm, n_chan_table, want_event_count=False, want_image=True, device_outputs=False, stream=None,
               want_contrib=0, counters="host"):
    return _run(lib().gcmcrt_run_albedo, handle, prm, n_chan_table, want_event_count, want_image, device_outputs, stream,
                want_contrib, counters)


def run_emission(handle, prm, n_chan_table, want_event_count=False, want_image=True, device_outputs=False, stream=None,
                 want_contrib=0, counters="host"):
    return _run(lib().gcmcrt_run_emission, handle, prm, n_chan_table, want_event_count, want_image, device_outputs, stream,
                want_contrib, counters)


def run_transmission(handle, prm, n_chan_table, want_event_count=False, device_outputs=False, stream=None, counters="host"):
    return _run(lib().gcmcrt_run_transmission, handle, prm, n_chan_table, want_event_count, False, device_outputs, stream, 0,
                counters)


STATIC_SCRATCH_BYTES = 8 << 20   # GCMCRT_STATIC_SCRATCH_BYTES of include/gcmcrt.h


def emission_ltot_static(handle, chan_begin, chan_end, tau_vert_max, out=None, stream=None):
    """gcmcrt_emission_ltot_static: L_tot of the staged tables through the entry point that allocates nothing.
    out: a torch CUDA float64 tensor (the call only enqueues) or None (a numpy array is returned; the call waits)."""
    n = chan_end - chan_begin
    if out is None:
        out = np.zeros(max(n, 0), dtype=np.float64)
    rc = lib().gcmcrt_emission_ltot_static(handle, int(chan_begin), int(chan_end), float(tau_vert_max), _ptr(out), _stream_ptr(stream))
    _check(handle, rc)
    return out


def debug_ray_tau(handle, chan, pos, dirs, stream=None):
    pos = np.ascontiguousarray(pos, dtype=np.float32).reshape(-1, 3)
    dirs = np.ascontiguousarray(dirs, dtype=np.float32).reshape(-1, 3)
    n = pos.shape[0]
    tau = np.zeros(n, dtype=np.float32)
    hit = np.zeros(n, dtype=np.int32)
    rc = lib().gcmcrt_debug_ray_tau(handle, int(chan), n, _ptr(pos), _ptr(dirs), _ptr(tau), _ptr(hit), _stream_ptr(stream))
    _check(handle, rc)
    return tau, hit


def debug_philox(ctr, key, stream=None):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    out = np.zeros_like(ctr)
    rc = lib().gcmcrt_debug_philox(ctr.shape[0], _ptr(ctr), _ptr(key), _ptr(out), _stream_ptr(stream))
    _check(None, rc)
    return out


# --------------------------------------------------------------------------- convenience wrapper
class Grid:
    """Owns a gcmcrt_grid handle.  `grid`/`opac` are the plain dicts of workloads.py (numpy or torch arrays)."""

    def __init__(self, grid, stream=None):
        self.stream = stream
        self.n_chan = 0
        self.handle = grid_create(grid["r_edges"], grid["colat_edges"], grid["lon_edges"], _as32(grid["T"]),
                                  _as32(grid["rho"]), _as32(grid.get("u")), _as32(grid.get("v")), _as32(grid.get("w")),
                                  grid.get("Omega", 0.0), grid.get("surface_albedo", 0.0), stream)

    def set_opacity(self, opac):
        lam = opac["lambda"]
        self._keep = [_as32(opac.get(k)) for k in ("k_abs", "k_sca_ray", "k_sca_cld", "g_cld")]
        set_opacity(self.handle, opac.get("chan0", 0), lam, *self._keep, stream=self.stream)
        self.n_chan = int(np.asarray(lam).size) if not _is_torch(lam) else int(lam.numel())

    def set_opacity_nodes(self, opac):
        """k_abs from opac['node_kabs'][n_chan][nT][nP] at opac['T_nodes'], opac['logp_nodes'] (uniform), cell pressures
        opac['p_cell'] [nlon][nlat][nlev] in Pa; scattering tables as in set_opacity."""
        lam = opac["lambda"]
        self._keep = [_as32(opac.get(k)) for k in ("node_kabs", "p_cell", "k_sca_ray", "k_sca_cld", "g_cld")]
        set_opacity_nodes(self.handle, opac.get("chan0", 0), lam, self._keep[0], opac["T_nodes"], opac["logp_nodes"],
                          self._keep[1], *self._keep[2:], stream=self.stream)
        self.n_chan = int(np.asarray(lam).size) if not _is_torch(lam) else int(lam.numel())

    def run_albedo(self, prm, **kw):
        return run_albedo(self.handle, prm, self.n_chan, stream=self.stream, **kw)

    def run_emission(self, prm, **kw):
        return run_emission(self.handle, prm, self.n_chan, stream=self.stream, **kw)

    def run_transmission(self, prm, **kw):
        return run_transmission(self.handle, prm, self.n_chan, stream=self.stream, **kw)

    def ray_tau(self, chan, pos, dirs):
        return debug_ray_tau(self.handle, chan, pos, dirs, self.stream)

    def emission_ltot_static(self, chan_begin, chan_end, tau_vert_max, out=None):
        return emission_ltot_static(self.handle, chan_begin, chan_end, tau_vert_max, out, self.stream)

    def close(self):
        if self.handle:
            destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _as32(a):
    if a is None or _is_torch(a):
        return a
    return np.ascontiguousarray(a, dtype=np.float32)
