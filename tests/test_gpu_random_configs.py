"""GPU parity on seeded random configurations: grids from 1 x 1 x 1 to 31 x 17 x 70 cells with stratified, laterally
varying density, temperature and opacities (log-uniform extinction per cell, single-scattering albedo, gas fraction and
asymmetry varying from cell to cell), random star and observer directions, sub-ranges of packets and channels, and
every switch of the run parameters drawn at random (event cap, survival biasing + roulette, forced scattering, continuous
absorption, path-length stretching, the three cloud phase functions, Doppler shifts with winds, composite emission bias,
depth cut, images, limb darkening, multiple scattering in transmission, concurrent parts of a run).  Every case runs in albedo, emission and
transmission mode and is compared with the CPU oracle on the bar of BASELINE.json's north_star: per channel and observer
|delta| <= 4 sigma_MC + 1e-5 relative, >= 99 % of packets with identical event counts, L_tot within 1e-5.  Each run is
repeated with run_params.timing = 1 (the host-driven pass loop): same packets, event for event.

Event counts stay identical while a packet's history is short: positions are fp32 (8 m at 1e8 m), so each event has a
chance of ~3e-4 to fall on the other side of a cell face than in the oracle's fp64, after which the two histories part
(DESIGN.md section 7).  The generator therefore caps the events of a packet at 6 wherever the medium is not absorbing
enough to end histories early -- the paper's workloads have 2 - 4 events per packet -- so that the 99 % bar applies.
"""
import numpy as np
import pytest

from paper_2110_15640_b200 import workloads as wl

pytestmark = pytest.mark.gpu

N_CASES = 48


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2110_15640_b200 import binding, build
    build.build()
    binding.lib()
    return binding


def _unit(rng):
    v = rng.normal(size=3)
    return v / np.linalg.norm(v)


def make_case(seed):
    """Inputs only: shapes, value distributions and switches; none of the method's arithmetic."""
    rng = np.random.default_rng(7000 + seed)
    nlev = int(rng.choice([1, 2, 5, 13, 33, 60, 70]))
    nlat = int(rng.choice([1, 1, 2, 3, 8, 17]))
    nlon = int(rng.choice([1, 1, 2, 5, 12, 31]))
    n_chan = int(rng.choice([1, 2, 3, 5]))
    R0 = 10 ** rng.uniform(6.5, 8.0)
    H = R0 * rng.uniform(0.01, 0.3)
    r_edges = R0 + H * np.linspace(0, 1, nlev + 1) ** rng.uniform(0.7, 1.5)
    grid = wl.make_grid(r_edges, nlat, nlon, surface_albedo=float(rng.choice([0.0, 0.0, 0.3, 1.0])))
    shape = (nlon, nlat, nlev)
    z = (0.5 * (r_edges[1:] + r_edges[:-1]) - R0) / H
    grid["T"] = (rng.uniform(600, 2500) * (1 + 0.3 * rng.uniform(-1, 1, size=shape)) * np.exp(-0.5 * z)[None, None, :]).astype(np.float32)
    grid["rho"] = (np.exp(-z * rng.uniform(0, 6))[None, None, :] * (1 + 0.5 * rng.uniform(-1, 1, size=shape))).astype(np.float32)
    tau_tot = 10 ** rng.uniform(-1.5, 1.7)
    cs = (n_chan,) + shape
    kext = tau_tot / (H * grid["rho"].mean()) * 10 ** rng.uniform(-0.7, 0.7, size=cs) * 10 ** rng.uniform(-1, 1, size=(n_chan, 1, 1, 1))
    omega_max = float(rng.choice([0.0, 0.5, 0.7, 0.95, 1.0]))
    omega = omega_max * rng.uniform(0.3, 1.0, size=cs) if omega_max < 1.0 else np.ones(cs)
    pgas = rng.uniform(0, 1, size=cs) if rng.random() < 0.7 else np.full(cs, float(rng.choice([0.0, 1.0])))
    ks = kext * omega
    opac = dict(chan0=int(rng.integers(0, 1000)))
    opac["lambda"] = (10 ** rng.uniform(-6.3, -5.0) * (1 + 2.0e-5 * np.arange(n_chan))).astype(np.float32)
    opac["k_abs"] = (kext - ks).astype(np.float32)
    opac["k_sca_ray"] = (ks * pgas).astype(np.float32)
    opac["k_sca_cld"] = (ks * (1 - pgas)).astype(np.float32)
    opac["g_cld"] = rng.uniform(-0.3, 0.9, size=cs).astype(np.float32)
    if rng.random() < 0.3:
        grid["u"] = rng.uniform(-6000, 6000, size=shape).astype(np.float32)
        grid["v"] = rng.uniform(-2000, 2000, size=shape).astype(np.float32)
        grid["w"] = rng.uniform(-100, 100, size=shape).astype(np.float32)
        grid["Omega"] = float(rng.uniform(0, 5e-5))
    n_obs = int(rng.choice([1, 1, 2, 4]))
    star = _unit(rng)
    obs = np.array([_unit(rng) for _ in range(n_obs)])
    if rng.random() < 0.3:
        obs[0] = star
    N = int(rng.choice([4000, 20000, 33333]))
    # short histories (see the module docstring): an absorbing medium ends them by itself, otherwise the event cap does
    max_events = int(rng.choice([0, 0, 1, 3, 6])) if omega_max <= 0.7 else int(rng.choice([1, 2, 4, 6]))
    prm = wl.default_params(star_dir=star, obs_dir=obs, packets_per_channel=N, seed=int(rng.integers(1, 10 ** 6)),
                            max_events=max_events, scatter_on=int(rng.random() < 0.85),
                            tau_vert_max=float(rng.choice([0.0, 2.0, 30.0])), tau_cut=float(rng.choice([20.0, 50.0])),
                            n_batches=32, cloud_phase=int(rng.choice([0, 0, 1, 2])))
    vr = rng.random()
    if vr < 0.2:
        prm.update(survival_bias=1, roulette_w_min=float(rng.choice([0.0, 0.1])), roulette_survive=0.3)
    elif vr < 0.4:
        prm.update(forced_scatter=int(rng.choice([1, 2])), survival_bias=1, roulette_w_min=0.1, roulette_survive=0.3)
    elif vr < 0.5:
        prm.update(continuous_absorption=1, max_events=int(rng.choice([4, 6])))
    elif vr < 0.65:
        prm.update(stretch_alpha=float(rng.uniform(0.2, 0.8)), forced_scatter=int(rng.choice([0, 1])))
    if rng.random() < 0.3 and n_chan > 1:
        prm.update(doppler_on=1, doppler_halfwidth=int(rng.choice([1, 2])))
    if rng.random() < 0.3:
        prm.update(emission_bias=float(rng.uniform(0.1, 0.9)))
    if rng.random() < 0.3:     # a sub-range of the packets that still spans several batches (sigma needs more than one)
        lo = int(rng.integers(0, N // 2))
        prm.update(pkt_begin=lo, pkt_end=int(rng.integers(lo + N // 4, N + 1)))
    if rng.random() < 0.3 and n_chan > 2:
        prm.update(chan_begin=1, chan_end=n_chan - int(rng.integers(0, 2)))
    if rng.random() < 0.3:
        prm.update(npix=int(rng.choice([4, 16])))
    tr = dict(star_radius=7.0e8, planet_xy=[float(rng.uniform(-3e8, 3e8)), float(rng.uniform(-3e8, 3e8))], ld_c1=0.3, ld_c2=0.2)
    if rng.random() < 0.5:
        tr["star_solid_angle"] = float(10 ** rng.uniform(-4, -2))
    if rng.random() < 0.4:     # the run's channels in parts side by side (ignored where it does not apply)
        prm.update(concurrency=int(rng.choice([2, 3])))
    return grid, opac, prm, tr


@pytest.mark.parametrize("block", range(4))
def test_random_configurations_meet_the_parity_bar(gpu, orc, block):
    per = N_CASES // 4
    for case in range(block * per, (block + 1) * per):
        grid, opac, prm, tr = make_case(case)
        for mode in ("albedo", "emission", "transmission"):
            p = dict(prm)
            if mode == "transmission":
                p.update(tr)
                p["continuous_absorption"] = 0
                p["obs_dir"] = p["obs_dir"][:2]
            if mode != "emission":
                p["emission_bias"] = 0.0
            tag = (case, mode)
            with gpu.Grid(grid) as G:
                G.set_opacity(opac)
                fn = dict(albedo=G.run_albedo, emission=G.run_emission, transmission=G.run_transmission)[mode]
                g = fn(p, want_event_count=True)
                h = fn(dict(p, timing=1), want_event_count=True)
            ofn = dict(albedo=orc.run_albedo, emission=orc.run_emission, transmission=orc.run_transmission)[mode]
            o = ofn(grid, opac, dict(p, n_threads=16), want_event_count=True)
            vo, so = orc.reduce(o, mode)
            cb = int(p.get("chan_begin", 0) or 0)
            ce = cb + g["value"].shape[0]          # the oracle computes every channel of the table
            vo, so = vo[cb:ce], so[cb:ce]
            tol = 4 * so + 1e-5 * np.abs(vo) + 1e-300
            assert np.all(np.abs(g["value"] - vo) <= tol), (tag, (np.abs(g["value"] - vo) / tol).max())
            if mode == "emission":
                assert np.allclose(g["L_tot"], o["L_tot"][cb:ce], rtol=1e-5), tag
            lo, hi = o["pkt_range"]
            oe = o["event_count"][cb:ce, lo:hi]
            if oe.size:
                assert (g["event_count"] == oe).mean() >= 0.99, (tag, (g["event_count"] == oe).mean(), oe.mean())
            assert g["counters"]["packets_stuck"] == 0 and o["counters"]["packets_stuck"] == 0, tag
            assert g["counters"]["device_status"] == 0, tag
            # the device-driven pass loop and the host-driven one run the same packets, event for event
            assert np.array_equal(g["event_count"], h["event_count"]), tag
            assert np.allclose(g["value"], h["value"], rtol=2e-5, atol=1e-300), tag
