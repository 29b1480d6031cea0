"""CPU oracle for the gCMCRT hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes wrapper around oracle/gcmcrt_oracle.c (plain serial fp64 C written from
/root/reference/PAPER.md).  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package; the product
package paper_2110_15640_b200 never does, and this package never imports it.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


class _Grid(C.Structure):
    _fields_ = [("nlev", C.c_int), ("nlat", C.c_int), ("nlon", C.c_int),
                ("r_edges", C.c_void_p), ("colat_edges", C.c_void_p), ("lon_edges", C.c_void_p),
                ("T", C.c_void_p), ("rho", C.c_void_p),
                ("u", C.c_void_p), ("v", C.c_void_p), ("w", C.c_void_p),
                ("Omega", C.c_double), ("surface_albedo", C.c_double)]


class _Opacity(C.Structure):
    _fields_ = [("n_chan", C.c_int), ("chan0", C.c_int), ("lam", C.c_void_p), ("k_abs", C.c_void_p),
                ("k_sca_ray", C.c_void_p), ("k_sca_cld", C.c_void_p), ("g_cld", C.c_void_p)]


class _Params(C.Structure):
    _fields_ = [("star_dir", C.c_double * 3), ("n_obs", C.c_int), ("obs_dir", C.c_void_p),
                ("packets_per_channel", C.c_uint64), ("pkt_begin", C.c_uint64), ("pkt_end", C.c_uint64),
                ("seed", C.c_uint64), ("max_events", C.c_int), ("scatter_on", C.c_int),
                ("doppler_on", C.c_int), ("doppler_halfwidth", C.c_int),
                ("emission_bias", C.c_double), ("tau_vert_max", C.c_double), ("tau_cut", C.c_double),
                ("npix", C.c_int), ("n_batches", C.c_int), ("n_threads", C.c_int),
                ("survival_bias", C.c_int), ("roulette_w_min", C.c_double), ("roulette_survive", C.c_double),
                ("star_radius", C.c_double), ("planet_xy", C.c_double * 2), ("ld_c1", C.c_double), ("ld_c2", C.c_double), ("cloud_phase", C.c_int), ("forced_scatter", C.c_int), ("continuous_absorption", C.c_int),
                ("star_solid_angle", C.c_double), ("stretch_alpha", C.c_double)]


class _Counters(C.Structure):
    _fields_ = [("events", C.c_uint64), ("segments_transport", C.c_uint64), ("segments_peel", C.c_uint64),
                ("packets_escaped", C.c_uint64), ("packets_absorbed", C.c_uint64),
                ("packets_surface", C.c_uint64), ("packets_stuck", C.c_uint64),
                ("escaped_weight", C.c_double)]


class _Result(C.Structure):
    _fields_ = [("flux_sum", C.c_void_p), ("L_tot", C.c_void_p), ("image", C.c_void_p),
                ("event_count", C.c_void_p), ("counters", _Counters), ("contrib", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_u32_to_zeta.restype = C.c_double
        L.orc_u32_to_zeta.argtypes = [C.c_uint32]
        for name in ("orc_sample_isotropic", "orc_sample_lambert", "orc_sample_rayleigh", "orc_phase_rayleigh"):
            getattr(L, name).restype = C.c_double
            getattr(L, name).argtypes = [C.c_double]
        L.orc_sample_tthg.restype = C.c_double
        L.orc_sample_tthg.argtypes = [C.c_double] * 3
        L.orc_draine_G.restype = C.c_double
        L.orc_draine_G.argtypes = [C.c_double]
        for name in ("orc_sample_hg", "orc_phase_hg", "orc_phase_tthg", "orc_planck", "orc_phase_draine", "orc_sample_draine"):
            getattr(L, name).restype = C.c_double
            getattr(L, name).argtypes = [C.c_double, C.c_double]
        L.orc_cell_volume.restype = C.c_double
        L.orc_cell_volume.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.orc_vlos_eq33.restype = C.c_double
        L.orc_vlos_eq33.argtypes = [C.c_double] * 9
        L.orc_vlos_vector.restype = C.c_double
        L.orc_vlos_vector.argtypes = [C.c_double] * 7 + [C.c_void_p]
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


# ---------------------------------------------------------------- small functions
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xffffffff for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xffffffff for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def u32_to_zeta(u):
    return lib().orc_u32_to_zeta(int(u))


def zeta_block(seed, chan, pkt, event, purpose):
    z = (C.c_double * 4)()
    lib().orc_zeta_block(C.c_uint64(seed), C.c_uint32(chan), C.c_uint32(pkt), C.c_uint32(event),
                         C.c_uint32(purpose), z)
    return [float(x) for x in z]


def sample_isotropic(z): return lib().orc_sample_isotropic(z)
def sample_lambert(z): return lib().orc_sample_lambert(z)
def sample_rayleigh(z): return lib().orc_sample_rayleigh(z)
def sample_hg(g, z): return lib().orc_sample_hg(g, z)
def phase_rayleigh(mu): return lib().orc_phase_rayleigh(mu)
def phase_hg(g, mu): return lib().orc_phase_hg(g, mu)
def phase_tthg(g, mu): return lib().orc_phase_tthg(g, mu)
def sample_tthg(g, zl, z): return lib().orc_sample_tthg(g, zl, z)
def draine_G(g): return lib().orc_draine_G(g)
def phase_draine(g, mu): return lib().orc_phase_draine(g, mu)
def sample_draine(g, z): return lib().orc_sample_draine(g, z)
def planck(lam, T): return lib().orc_planck(lam, T)


def rotate(n, ct, psi):
    a = (C.c_double * 3)(*n)
    o = (C.c_double * 3)()
    lib().orc_rotate(a, C.c_double(ct), C.c_double(psi), o)
    return np.array(list(o))


def vlos_eq33(u, v, w, Omega, r, theta, phi, theta_v, phi_v):
    return lib().orc_vlos_eq33(u, v, w, Omega, r, theta, phi, theta_v, phi_v)


def vlos_vector(u, v, w, Omega, r, theta, phi, obs):
    o = _f64(obs)
    return lib().orc_vlos_vector(u, v, w, Omega, r, theta, phi, _ptr(o))


# ---------------------------------------------------------------- marshalling
class _Keep:
    """Holds the numpy arrays a ctypes struct points into."""

    def __init__(self):
        self.refs = []

    def __call__(self, a):
        self.refs.append(a)
        return _ptr(a)


def _grid_struct(grid, keep):
    r = _f64(grid["r_edges"]); th = _f64(grid["colat_edges"]); ph = _f64(grid["lon_edges"])
    nlev, nlat, nlon = len(r) - 1, len(th) - 1, len(ph) - 1
    ncell = nlev * nlat * nlon
    T = _f32(grid["T"]).reshape(-1); rho = _f32(grid["rho"]).reshape(-1)
    assert T.size == ncell and rho.size == ncell
    g = _Grid(nlev, nlat, nlon, keep(r), keep(th), keep(ph), keep(T), keep(rho),
              keep(_f32(grid.get("u"))) if grid.get("u") is not None else None,
              keep(_f32(grid.get("v"))) if grid.get("v") is not None else None,
              keep(_f32(grid.get("w"))) if grid.get("w") is not None else None,
              float(grid.get("Omega", 0.0)), float(grid.get("surface_albedo", 0.0)))
    return g, ncell


def _opac_struct(opac, ncell, keep):
    lam = _f32(opac["lambda"])
    n_chan = lam.size
    ka = _f32(opac["k_abs"]).reshape(n_chan, ncell)
    o = _Opacity(n_chan, int(opac.get("chan0", 0)), keep(lam), keep(ka), None, None, None)
    for name in ("k_sca_ray", "k_sca_cld", "g_cld"):
        a = opac.get(name)
        if a is not None:
            setattr(o, name, keep(_f32(a).reshape(n_chan, ncell)))
    return o, n_chan


def _params_struct(prm, keep):
    obs = _f64(prm.get("obs_dir", np.zeros((0, 3)))).reshape(-1, 3)
    N = int(prm["packets_per_channel"])
    p = _Params()
    p.star_dir[:] = [float(x) for x in prm.get("star_dir", (1.0, 0.0, 0.0))]
    p.n_obs = obs.shape[0]
    p.obs_dir = keep(obs)
    p.packets_per_channel = N
    p.pkt_begin = int(prm.get("pkt_begin", 0))
    p.pkt_end = int(prm.get("pkt_end", N))
    p.seed = int(prm.get("seed", 0))
    p.max_events = int(prm.get("max_events", 0))
    p.scatter_on = int(prm.get("scatter_on", 1))
    p.doppler_on = int(prm.get("doppler_on", 0))
    p.doppler_halfwidth = int(prm.get("doppler_halfwidth", 0))
    p.emission_bias = float(prm.get("emission_bias", 0.0))
    p.tau_vert_max = float(prm.get("tau_vert_max", 30.0))
    p.tau_cut = float(prm.get("tau_cut", 50.0))
    p.npix = int(prm.get("npix", 0))
    p.n_batches = int(prm.get("n_batches", 32))
    p.n_threads = int(prm.get("n_threads", 1))
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
    return p


def _run(mode, grid, opac, prm, want_event_count=False, want_contrib=False):
    keep = _Keep()
    g, ncell = _grid_struct(grid, keep)
    o, n_chan = _opac_struct(opac, ncell, keep)
    p = _params_struct(prm, keep)
    nobs, nb, N, npix = p.n_obs, p.n_batches, p.packets_per_channel, p.npix
    flux = np.zeros((n_chan, nobs, nb), dtype=np.float64)
    ltot = np.zeros((n_chan, nobs), dtype=np.float64)
    image = np.zeros((n_chan, nobs, npix, npix), dtype=np.float64) if npix > 0 else None
    evc = np.zeros((n_chan, N), dtype=np.uint32) if want_event_count else None
    contrib = np.zeros((n_chan, nobs, 2, ncell), dtype=np.float64) if want_contrib else None
    res = _Result(_ptr(flux), _ptr(ltot), _ptr(image), _ptr(evc), _Counters(), _ptr(contrib))
    fn = {"albedo": lib().orc_run_albedo, "emission": lib().orc_run_emission,
          "transmission": lib().orc_run_transmission}[mode]
    fn.restype = C.c_int
    rc = fn(C.byref(g), C.byref(o), C.byref(p), C.byref(res))
    if rc != 0:
        raise RuntimeError("oracle run failed: %d" % rc)
    cnt = {name: getattr(res.counters, name) for name, _ in _Counters._fields_}
    return {"flux_sum": flux, "L_tot": ltot, "image": image, "event_count": evc, "counters": cnt, "contrib": contrib,
            "n_batches": nb, "packets_per_channel": N, "pkt_range": (p.pkt_begin, p.pkt_end)}


def run_albedo(grid, opac, prm, want_event_count=False, want_contrib=False):
    """O3,O5-O8: albedo mode.  Returns raw sums flux_sum[n_chan][n_obs][n_batches] (Eq. 14) etc.; contrib
    [n_chan][n_obs][2][ncell] = Eq. 32 numerators (thermal, scattered) when asked for."""
    return _run("albedo", grid, opac, prm, want_event_count, want_contrib)


def run_emission(grid, opac, prm, want_event_count=False, want_contrib=False):
    """O4-O8: emission mode."""
    return _run("emission", grid, opac, prm, want_event_count, want_contrib)


def run_transmission(grid, opac, prm, want_event_count=False):
    """Sect. 5.1, Eq. 20-23: random transit chords; with scatter_on and star_solid_angle > 0 the packets go on to
    scatter (L259, reading N12).  reduce(.., "transmission") gives <I_p> of Eq. 21 in m^2: see reduce()."""
    res = _run("transmission", grid, opac, prm, want_event_count)
    r = np.asarray(grid["r_edges"], dtype=np.float64)
    res["annulus_width"] = float(r[-1] - r[0])
    return res


def reduce(result, mode):
    """O8 / A10: value[c][o] and its batch-means sigma (C12).

    albedo: reflected fraction S/N (A_g = pi * value at zero phase, Eq. 24).
    emission: L_obs = L_tot S/N (Eq. 28) in W m^-1 sr^-1.
    Batches partly outside the simulated packet range are weighted by the packets they hold.
    """
    S = result["flux_sum"]
    nb = result["n_batches"]
    N = result["packets_per_channel"]
    lo, hi = result["pkt_range"]
    edges = [(b * N + nb - 1) // nb for b in range(nb + 1)]
    cnt = np.array([max(0, min(edges[b + 1], hi) - max(edges[b], lo)) for b in range(nb)], dtype=np.float64)
    n_run = cnt.sum()
    used = cnt > 0
    mean = S.sum(axis=2) / n_run
    bm = S[:, :, used] / cnt[used]
    nbu = int(used.sum())
    sigma = bm.std(axis=2, ddof=1) / np.sqrt(nbu) if nbu > 1 else np.zeros_like(mean)
    if mode == "emission":
        mean = mean * result["L_tot"]
        sigma = sigma * result["L_tot"]
    if mode == "transmission":          # Eq. 21: <I_p> = (R_TOA - R_p0) / N * sum, m^2
        mean = mean * result["annulus_width"]
        sigma = sigma * result["annulus_width"]
    return mean, sigma


def ray_tau(grid, opac, chan, pos, dirs):
    """O5: optical depth from pos along dirs to the TOA; also hit_surface, segment count, path length."""
    keep = _Keep()
    g, ncell = _grid_struct(grid, keep)
    o, _ = _opac_struct(opac, ncell, keep)
    pos = _f64(pos).reshape(-1, 3); dirs = _f64(dirs).reshape(-1, 3)
    n = pos.shape[0]
    tau = np.zeros(n); hit = np.zeros(n, dtype=np.int32); nseg = np.zeros(n, dtype=np.int64); path = np.zeros(n)
    rc = lib().orc_ray_tau(C.byref(g), C.byref(o), C.c_int(chan), C.c_long(n), _ptr(pos), _ptr(dirs),
                           _ptr(tau), _ptr(hit), _ptr(nseg), _ptr(path))
    if rc != 0:
        raise RuntimeError("orc_ray_tau failed")
    return tau, hit, nseg, path


def channel_prep(grid, opac, prm, chan, obs_index=-1, emission=True):
    """O2: staged alpha_ext, omega, P_gas, g, L_i, L_tot of one channel."""
    keep = _Keep()
    g, ncell = _grid_struct(grid, keep)
    o, _ = _opac_struct(opac, ncell, keep)
    p = _params_struct(prm, keep)
    arrs = [np.zeros(ncell) for _ in range(5)]
    ltot = C.c_double(0.0)
    rc = lib().orc_channel_prep(C.byref(g), C.byref(o), C.byref(p), C.c_int(chan), C.c_int(obs_index),
                                _ptr(arrs[0]), _ptr(arrs[1]), _ptr(arrs[2]), _ptr(arrs[3]),
                                _ptr(arrs[4]) if emission else None, C.byref(ltot))
    if rc != 0:
        raise RuntimeError("orc_channel_prep failed")
    return {"alpha": arrs[0], "omega": arrs[1], "pgas": arrs[2], "g": arrs[3], "L_cell": arrs[4],
            "L_tot": ltot.value}


def cell_volume(grid, i, j, k):
    keep = _Keep()
    g, _ = _grid_struct(grid, keep)
    return lib().orc_cell_volume(C.byref(g), i, j, k)


def locate(grid, p):
    keep = _Keep()
    g, _ = _grid_struct(grid, keep)
    pp = (C.c_double * 3)(*[float(x) for x in p])
    out = (C.c_int * 3)()
    lib().orc_locate(C.byref(g), pp, out)
    return tuple(int(x) for x in out)


def interp_nodes(node_kabs, T_nodes, logp_nodes, T_cell, p_cell):
    """k_abs[c][cell] from (T, log10 p) node tables node_kabs[c][nT][nP]: bilinear in (T, log10 p), the cell's
    (T, log10 p) clamped to the table (the interpolation of opacity tables to the GCM cells, PAPER.md L374 / L85;
    gcmcrt_set_opacity_nodes in include/gcmcrt.h states the same definition).  fp64, written out term by term."""
    node = np.asarray(node_kabs, dtype=np.float64)
    Tn = np.asarray(T_nodes, dtype=np.float64)
    lpn = np.asarray(logp_nodes, dtype=np.float64)
    T = np.asarray(T_cell, dtype=np.float64)
    lp = np.log10(np.asarray(p_cell, dtype=np.float64))
    out = np.empty((node.shape[0],) + T.shape, dtype=np.float64)
    for idx in np.ndindex(T.shape):
        t = min(max(T[idx], Tn[0]), Tn[-1])
        q = min(max(lp[idx], lpn[0]), lpn[-1])
        a = min(int(np.searchsorted(Tn, t, side="right")) - 1, Tn.size - 2)
        b = min(int(np.searchsorted(lpn, q, side="right")) - 1, lpn.size - 2)
        x = (t - Tn[a]) / (Tn[a + 1] - Tn[a])
        y = (q - lpn[b]) / (lpn[b + 1] - lpn[b])
        out[(slice(None),) + idx] = ((1 - x) * (1 - y) * node[:, a, b] + x * (1 - y) * node[:, a + 1, b]
                                     + (1 - x) * y * node[:, a, b + 1] + x * y * node[:, a + 1, b + 1])
    return out
