"""Seeded synthetic inputs shared by the CPU oracle and the CUDA path.

This module holds NONE of the method's arithmetic: it only builds grids, GCM-shaped
fields and opacity tables (plain numpy, fp32 where the C-ABI takes fp32) and the
run parameters of BASELINE.json's configs.  The paper's GCM outputs and opacity
tables are not available, so these stand in for them; the
recipe follows SURVEY.md section 8(d) and is restated in DESIGN.md.

Every generator returns (grid, opac, prm) as plain dicts of numpy arrays / scalars:
  grid: r_edges[nlev+1] f64, colat_edges[nlat+1] f64, lon_edges[nlon+1] f64,
        T, rho (and optionally u, v, w) f32 [nlon][nlat][nlev], Omega, surface_albedo
  opac: lambda[n_chan] f32 (m), k_abs / k_sca_ray / k_sca_cld / g_cld f32 [n_chan][nlon][nlat][nlev]
        (absent keys = not present), chan0, and for correlated-k: band[n_chan], g_weight[n_chan]
  prm:  star_dir, obs_dir[n_obs][3], packets_per_channel, seed, ... (names of gcmcrt_run_params)
"""
import numpy as np

K_B = 1.380649e-23
M_U = 1.66053906660e-27
BAR = 1.0e5


def sph_dir(colat, lon):
    return np.array([np.sin(colat) * np.cos(lon), np.sin(colat) * np.sin(lon), np.cos(colat)])


def orbital_phase_dirs(n_obs):
    """C11: observer directions for orbital phases m/n_obs; sub-stellar point at lon 0, phase 0.5 = dayside."""
    return np.array([sph_dir(np.pi / 2, np.pi + 2 * np.pi * m / n_obs) for m in range(n_obs)])


def default_params(**kw):
    prm = dict(star_dir=np.array([1.0, 0.0, 0.0]), obs_dir=np.array([[1.0, 0.0, 0.0]]),
               packets_per_channel=10000, seed=1, max_events=0, scatter_on=1, doppler_on=0,
               doppler_halfwidth=0, emission_bias=0.0, tau_vert_max=30.0, tau_cut=50.0, npix=0, n_batches=32,
               survival_bias=0, roulette_w_min=0.0, roulette_survive=0.0, cloud_phase=0, forced_scatter=0, continuous_absorption=0)
    prm.update(kw)
    prm["star_dir"] = np.asarray(prm["star_dir"], dtype=np.float64)
    prm["obs_dir"] = np.asarray(prm["obs_dir"], dtype=np.float64).reshape(-1, 3)
    return prm


def uniform_edges(nlat, nlon):
    return np.linspace(0.0, np.pi, nlat + 1), np.linspace(0.0, 2 * np.pi, nlon + 1)


def make_grid(r_edges, nlat, nlon, T=1000.0, rho=1.0, surface_albedo=0.0, colat_edges=None, lon_edges=None):
    r_edges = np.asarray(r_edges, dtype=np.float64)
    nlev = r_edges.size - 1
    th, ph = uniform_edges(nlat, nlon)
    if colat_edges is not None:
        th = np.asarray(colat_edges, dtype=np.float64)
    if lon_edges is not None:
        ph = np.asarray(lon_edges, dtype=np.float64)
    shape = (nlon, nlat, nlev)
    return dict(r_edges=r_edges, colat_edges=th, lon_edges=ph,
                T=np.broadcast_to(np.asarray(T, dtype=np.float32), shape).copy(),
                rho=np.broadcast_to(np.asarray(rho, dtype=np.float32), shape).copy(),
                Omega=0.0, surface_albedo=float(surface_albedo))


def uniform_medium(nlev, nlat, nlon, R0, Rtoa, k_ext, omega, g=0.0, pgas=0.0, n_chan=1, lam=1.0e-6,
                   T=1000.0, rho=1.0, surface_albedo=0.0):
    """Homogeneous shell R0..Rtoa (radially uniform edges) with extinction rho*k_ext, albedo omega."""
    grid = make_grid(np.linspace(R0, Rtoa, nlev + 1), nlat, nlon, T=T, rho=rho, surface_albedo=surface_albedo)
    shape = (n_chan, nlon, nlat, nlev)
    k_ext = np.broadcast_to(np.asarray(k_ext, dtype=np.float64).reshape(-1, 1, 1, 1), shape)
    omega = np.broadcast_to(np.asarray(omega, dtype=np.float64).reshape(-1, 1, 1, 1), shape)
    ks = k_ext * omega
    opac = dict(lam_note="synthetic", chan0=0)
    opac["lambda"] = np.broadcast_to(np.asarray(lam, dtype=np.float32), (n_chan,)).copy()
    opac["k_abs"] = (k_ext - ks).astype(np.float32)
    opac["k_sca_ray"] = (ks * pgas).astype(np.float32)
    opac["k_sca_cld"] = (ks * (1.0 - pgas)).astype(np.float32)
    opac["g_cld"] = np.full(shape, g, dtype=np.float32)
    return grid, opac


def _hydrostatic_edges(nlev, p_bot_bar, p_top_bar, R0, T_ref, mu=2.33, grav=10.0):
    p_edges = np.logspace(np.log10(p_bot_bar), np.log10(p_top_bar), nlev + 1) * BAR
    H = K_B * T_ref / (mu * M_U * grav)
    z = H * np.log(p_edges[0] / p_edges)
    p_mid = np.sqrt(p_edges[:-1] * p_edges[1:])
    return R0 + z, p_mid


def cfg1(packets=100000, seed=1):
    """BASELINE config 1: 1D, 50 layers 100 bar..1e-6 bar, isothermal 1500 K, grey absorber + Rayleigh, 8 wavelengths."""
    nlev, mu = 50, 2.33
    r_edges, p_mid = _hydrostatic_edges(nlev, 100.0, 1e-6, 1.0e8, 1500.0, mu=mu)
    rho = (p_mid * mu * M_U / (K_B * 1500.0)).astype(np.float32)
    grid = make_grid(r_edges, 1, 1, T=1500.0, rho=rho.reshape(1, 1, nlev))
    lam = np.logspace(np.log10(0.3e-6), np.log10(1.0e-6), 8).astype(np.float32)
    shape = (8, 1, 1, nlev)
    opac = dict(chan0=0)
    opac["lambda"] = lam
    opac["k_abs"] = np.full(shape, 1e-3, dtype=np.float32)
    opac["k_sca_ray"] = np.broadcast_to((3e-5 * (lam.astype(np.float64) / 0.5e-6) ** -4).reshape(8, 1, 1, 1),
                                        shape).astype(np.float32)
    prm = default_params(packets_per_channel=packets, seed=seed)
    return grid, opac, prm


def gcm_grid(nlon=64, nlat=32, nlev=60, seed=2, R0=1.0e8, T_ref=1600.0, T_d=2200.0, T_n=1000.0, mu=2.33):
    """GCM-like 3D grid of BASELINE configs 2-5: day-night temperature contrast + 2 % noise, ideal-gas density."""
    rng = np.random.default_rng(seed)
    r_edges, p_mid = _hydrostatic_edges(nlev, 100.0, 1e-6, R0, T_ref, mu=mu)
    th, ph = uniform_edges(nlat, nlon)
    thc = 0.5 * (th[:-1] + th[1:])
    phc = 0.5 * (ph[:-1] + ph[1:])
    lat = np.pi / 2 - thc
    mu0 = np.maximum(np.cos(phc)[:, None] * np.cos(lat)[None, :], 0.0)        # [nlon][nlat]
    T2 = T_n + (T_d - T_n) * mu0 ** 0.25
    T = T2[:, :, None] * (1.0 + 0.02 * rng.standard_normal((nlon, nlat, nlev)))
    T = np.maximum(T, 100.0)
    rho = p_mid[None, None, :] * mu * M_U / (K_B * T)
    grid = dict(r_edges=r_edges, colat_edges=th, lon_edges=ph, T=T.astype(np.float32), rho=rho.astype(np.float32),
                Omega=0.0, surface_albedo=0.0)
    grid["p_mid"] = p_mid
    return grid, rng


def corrk_opacity(grid, rng, nbands=11, ng=16):
    """Correlated-k tables of configs 2/3: nbands x ng Gauss-Legendre g-points, per-cell k log-uniform 1e-6..1e1
    sorted ascending in g, cloud scattering with omega0 ~ U(0, 0.9), HG g = 0.5, no Rayleigh."""
    nlon, nlat, nlev = grid["T"].shape
    x, wq = np.polynomial.legendre.leggauss(ng)
    g_weight = 0.5 * wq
    band_centres = np.logspace(np.log10(0.5e-6), np.log10(20e-6), nbands)
    n_chan = nbands * ng
    k_abs = np.empty((nbands, ng, nlon, nlat, nlev), dtype=np.float32)
    k_cld = np.empty_like(k_abs)
    for b in range(nbands):
        logk = rng.uniform(-6.0, 1.0, size=(ng, nlon, nlat, nlev))
        logk.sort(axis=0)
        ka = 10.0 ** logk
        w0 = rng.uniform(0.0, 0.9, size=(nlon, nlat, nlev))
        k_abs[b] = ka.astype(np.float32)
        k_cld[b] = (ka * (w0 / (1.0 - w0))[None]).astype(np.float32)
    opac = dict(chan0=0)
    opac["lambda"] = np.repeat(band_centres, ng).astype(np.float32)
    opac["k_abs"] = k_abs.reshape(n_chan, nlon, nlat, nlev)
    opac["k_sca_cld"] = k_cld.reshape(n_chan, nlon, nlat, nlev)
    opac["g_cld"] = np.full((n_chan, nlon, nlat, nlev), 0.5, dtype=np.float32)
    opac["band"] = np.repeat(np.arange(nbands), ng)
    opac["g_weight"] = np.tile(g_weight, nbands)
    return opac


def cfg2(nlon=64, nlat=32, nlev=60, nbands=11, ng=16, packets=1000000, seed=2):
    """BASELINE config 2: 3D correlated-k albedo, observer at phase angle 0 (o^ = s^)."""
    grid, rng = gcm_grid(nlon, nlat, nlev, seed=seed)
    opac = corrk_opacity(grid, rng, nbands, ng)
    s = sph_dir(np.pi / 2, 0.0)
    prm = default_params(star_dir=s, obs_dir=s[None, :], packets_per_channel=packets, seed=seed)
    return grid, opac, prm


def cfg3(nlon=64, nlat=32, nlev=60, nbands=11, ng=16, packets=1000000, seed=2, n_obs=8):
    """BASELINE config 3: same grid, emission with scattering, 8 orbital phases peeled in one pass."""
    grid, rng = gcm_grid(nlon, nlat, nlev, seed=seed)
    opac = corrk_opacity(grid, rng, nbands, ng)
    prm = default_params(star_dir=sph_dir(np.pi / 2, 0.0), obs_dir=orbital_phase_dirs(n_obs),
                         packets_per_channel=packets, seed=seed + 1, tau_vert_max=30.0)
    return grid, opac, prm


def add_winds(grid, U0=5000.0, Udn=1000.0, period_days=3.0):
    """Config 4/5 wind field: superrotating equatorial jet (<= U0) tapered with pressure, plus a day-night
    divergent flow (<= Udn); w = 0; solid-body rotation Omega = 2 pi / period."""
    nlon, nlat, nlev = grid["T"].shape
    th, ph = grid["colat_edges"], grid["lon_edges"]
    lat = np.pi / 2 - 0.5 * (th[:-1] + th[1:])
    phc = 0.5 * (ph[:-1] + ph[1:])
    p_mid = grid["p_mid"]
    taper = np.clip((np.log10(10.0 * BAR) - np.log10(p_mid)) / 3.0, 0.0, 1.0)    # 0 below 10 bar -> 1 above 10 mbar
    u = U0 * (np.cos(lat) ** 2)[None, :, None] * taper[None, None, :] * np.ones((nlon, 1, 1))
    # day-night flow diverging from the sub-stellar point (lon 0, equator)
    u_dn = Udn * np.sin(phc)[:, None, None] * np.cos(lat)[None, :, None] * taper[None, None, :]
    v_dn = -Udn * np.cos(phc)[:, None, None] * np.sin(lat)[None, :, None] * np.cos(lat)[None, :, None] * taper[None, None, :]
    mag = np.maximum(np.abs(u + u_dn).max(), 1e-30)
    grid["u"] = ((u + u_dn) * min(1.0, U0 / mag)).astype(np.float32)
    grid["v"] = np.broadcast_to(v_dn, (nlon, nlat, nlev)).astype(np.float32)
    grid["w"] = np.zeros((nlon, nlat, nlev), dtype=np.float32)
    grid["Omega"] = 2 * np.pi / (period_days * 86400.0)
    return grid


def _voigt_profile(x, sigma, gamma):
    """Voigt via the pseudo-Voigt approximation of Thompson et al. (synthetic line shapes only need to be smooth)."""
    fg = 2.0 * sigma * np.sqrt(2.0 * np.log(2.0))
    fl = 2.0 * gamma
    f = (fg ** 5 + 2.69269 * fg ** 4 * fl + 2.42843 * fg ** 3 * fl ** 2 + 4.47163 * fg ** 2 * fl ** 3
         + 0.07842 * fg * fl ** 4 + fl ** 5) ** 0.2
    eta = 1.36603 * (fl / f) - 0.47719 * (fl / f) ** 2 + 0.11116 * (fl / f) ** 3
    G = np.exp(-4.0 * np.log(2.0) * (x / f) ** 2) * (2.0 / f) * np.sqrt(np.log(2.0) / np.pi)
    Lz = (f / (2.0 * np.pi)) / (x ** 2 + 0.25 * f ** 2)
    return eta * Lz + (1.0 - eta) * G


def hires_opacity(grid, rng, n_chan=10000, lam0=2.19e-6, R=1.0e5, n_lines=500, nT=16, nP=16, k_cont=1e-4,
                  chan_block=512, cells=True):
    """Config 4/5 high-resolution table: kappa_abs from n_lines synthetic Voigt lines evaluated on an nT x nP
    (T, log p) node grid and bilinearly interpolated to every cell; no scattering."""
    nlon, nlat, nlev = grid["T"].shape
    lam = lam0 * (1.0 + 1.0 / R) ** np.arange(n_chan)
    nu = 1.0e-2 / lam                               # cm^-1
    nu_c = rng.uniform(nu.min(), nu.max(), n_lines)
    S = 10.0 ** rng.uniform(-4.0, 0.0, n_lines)     # relative strengths over 4 decades
    E = rng.uniform(0.0, 5000.0, n_lines)           # lower-state energy, cm^-1
    Tn = np.linspace(500.0, 3000.0, nT)
    lpn = np.linspace(np.log10(1e-6 * BAR), np.log10(100.0 * BAR), nP)
    mass = 28.0 * M_U
    c2 = 1.438776877                                # hc/k in cm K
    node = np.empty((n_chan, nT, nP), dtype=np.float64)
    for a, Tv in enumerate(Tn):
        sig = nu_c * np.sqrt(K_B * Tv / mass) / 299792458.0
        # line strengths are quoted at T_ref = 1500 K, the middle of the grid's temperature range (quoted at 296 K the
        # Boltzmann factor of a 5000 cm^-1 level is e^22 at 3000 K and every channel is opaque in the top cell)
        boltz = np.exp(-c2 * E * (1.0 / Tv - 1.0 / 1500.0)) * (1500.0 / Tv)
        for b, lp in enumerate(lpn):
            gam = 0.07 * (10.0 ** lp / 101325.0) * (Tv / 296.0) ** -0.5
            acc = np.zeros(n_chan)
            for l in range(n_lines):
                acc += S[l] * boltz[l] * _voigt_profile(nu - nu_c[l], sig[l], gam)
            node[:, a, b] = k_cont + 1.0e-2 * acc
    T = grid["T"].astype(np.float64)
    lp_cell = np.broadcast_to(np.log10(grid["p_mid"])[None, None, :], T.shape)
    ft = np.clip((T - Tn[0]) / (Tn[1] - Tn[0]), 0.0, nT - 1 - 1e-9)
    fp = np.clip((lp_cell - lpn[0]) / (lpn[1] - lpn[0]), 0.0, nP - 1 - 1e-9)
    it, ip = ft.astype(int), fp.astype(int)
    wt, wp = ft - it, fp - ip
    opac = dict(chan0=0)
    opac["lambda"] = lam.astype(np.float32)
    opac["lambda64"] = lam
    if cells:   # per-cell table (config 4); config 5 hands the node tables to gcmcrt_set_opacity_nodes instead
        k_abs = np.empty((n_chan, nlon, nlat, nlev), dtype=np.float32)
        for c0 in range(0, n_chan, chan_block):
            nd = node[c0:c0 + chan_block]
            k_abs[c0:c0 + chan_block] = ((1 - wt) * (1 - wp) * nd[:, it, ip] + wt * (1 - wp) * nd[:, it + 1, ip]
                                         + (1 - wt) * wp * nd[:, it, ip + 1] + wt * wp * nd[:, it + 1, ip + 1])
        opac["k_abs"] = k_abs
    # the same table in the form gcmcrt_set_opacity_nodes takes: node values + the cells' pressures
    opac["node_kabs"] = node.astype(np.float32)
    opac["T_nodes"] = Tn.astype(np.float32)
    opac["logp_nodes"] = lpn.astype(np.float32)
    opac["p_cell"] = np.broadcast_to(grid["p_mid"][None, None, :], T.shape).astype(np.float32)
    return opac


def cfg4(nlon=64, nlat=32, nlev=60, n_chan=10000, packets=100000, seed=4, n_lines=500):
    """BASELINE config 4: high-resolution emission with Doppler-shifted opacities, one dayside observer."""
    grid, rng = gcm_grid(nlon, nlat, nlev, seed=seed)
    add_winds(grid)
    opac = hires_opacity(grid, rng, n_chan=n_chan, n_lines=n_lines)
    prm = default_params(star_dir=sph_dir(np.pi / 2, 0.0), obs_dir=sph_dir(np.pi / 2, 0.0)[None, :],
                         packets_per_channel=packets, seed=seed, scatter_on=0, doppler_on=1, doppler_halfwidth=4)
    return grid, opac, prm


def cfg5(nlon=128, nlat=64, nlev=100, n_chan=100000, packets=100000, seed=5, n_lines=500, lam0=0.95e-6):
    """BASELINE config 5: large high-resolution run, emission + albedo at 4 orbital phases, opacities as (T, log p) node
    tables streamed in wavelength batches (the first n_chan points of lambda_n = 0.95 um
    (1 + 1e-5)^n; synthetic lines as in config 4).  The per-cell absorption table (328 GB at full size) is never
    built: `opac` carries the node tables, and a per-channel Rayleigh coefficient `k_ray_chan` (kappa_Ray =
    3e-5 (lambda / 0.5 um)^-4 m^2/kg in every cell, the law of config 1) from which the caller fills the
    [n_chan][ncell] scattering table of a batch."""
    grid, rng = gcm_grid(nlon, nlat, nlev, seed=seed)
    add_winds(grid)
    opac = hires_opacity(grid, rng, n_chan=n_chan, n_lines=n_lines, lam0=lam0, cells=False)
    opac["k_ray_chan"] = (3.0e-5 * (opac["lambda64"] / 0.5e-6) ** -4).astype(np.float32)
    phases = (np.arange(4) + 0.5) / 4.0
    obs = np.stack([sph_dir(np.pi / 2, np.pi + 2 * np.pi * ph) for ph in phases])
    prm = default_params(star_dir=sph_dir(np.pi / 2, 0.0), obs_dir=obs, packets_per_channel=packets, seed=seed,
                         scatter_on=1, doppler_on=1, doppler_halfwidth=4)
    return grid, opac, prm


def cfg5_batches(opac, batch=1024, halo=4):
    """Wavelength batches of config 5: (c0, c1, lo, hi) = channels [c0, c1) are run from a table that holds channels
    [lo, hi), i.e. `halo` extra channels on each side for the Doppler window."""
    n = int(opac["lambda"].size)
    return [(c0, min(c0 + batch, n), max(c0 - halo, 0), min(c0 + batch + halo, n)) for c0 in range(0, n, batch)]
