"""gcmcrt_emission_ltot_static: the entry point that allocates nothing (its scratch is a file-scope device array of
GCMCRT_STATIC_SCRATCH_BYTES) against the existing path -- the L_tot output of gcmcrt_run_emission, which the parity
tests hold to the oracle at 1e-5 -- on two calls in a row, with device and with host output, on a channel sub-range,
with and without the depth cut; sizes beyond the static array and missing staged tables are rejected with a clear
error.  The file sorts last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2110_15640_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2110_15640_b200 import binding, build
    build.build()
    binding.lib()
    return binding


def _case(nlon, nlat, nlev, n_chan, seed):
    grid, opac, prm = wl.cfg4(nlon=nlon, nlat=nlat, nlev=nlev, n_chan=n_chan, n_lines=12, packets=2000, seed=seed)
    return grid, opac, dict(prm, doppler_on=0, doppler_halfwidth=0, obs_dir=prm["obs_dir"][:1])


def test_static_scratch_entry_point_matches_the_run_path_twice(gpu):
    import torch
    for (nlon, nlat, nlev, n_chan), tvm in (((12, 6, 20, 24), 30.0), ((9, 5, 70, 7), 0.0), ((16, 8, 130, 5), 2.0)):
        grid, opac, prm = _case(nlon, nlat, nlev, n_chan, seed=3)
        prm = dict(prm, tau_vert_max=tvm)
        with gpu.Grid(grid) as G:
            G.set_opacity(opac)
            with pytest.raises(gpu.GcmcrtError) as ei:          # nothing staged yet, and the call stages nothing
                G.emission_ltot_static(0, n_chan, tvm)
            assert "staged" in str(ei.value)
            ref = G.run_emission(prm)["L_tot"][:, 0]             # the existing path (stages the tables)
            assert np.all(ref > 0)
            free0 = torch.cuda.mem_get_info()[0]
            dev = torch.full((n_chan,), -1.0, dtype=torch.float64, device="cuda")
            for call in range(2):                                  # two calls in a row share the array
                dev.fill_(-1.0)
                G.emission_ltot_static(0, n_chan, tvm, out=dev)
                torch.cuda.synchronize()
                assert np.allclose(dev.cpu().numpy(), ref, rtol=1e-5, atol=0.0), (call, nlev)
                assert np.array_equal(dev.cpu().numpy(), ref), (call, nlev)     # same arithmetic, same order
                host = G.emission_ltot_static(0, n_chan, tvm)                    # host output: copied from the array
                assert np.allclose(host, ref, rtol=1e-5, atol=0.0) and np.array_equal(host, ref)
            # a sub-range between two full calls (the array keeps the last call's contents: nothing may depend on them)
            if n_chan > 3:
                sub = G.emission_ltot_static(2, n_chan - 1, tvm)
                assert np.array_equal(sub, ref[2:n_chan - 1])
                again = G.emission_ltot_static(0, n_chan, tvm)
                assert np.array_equal(again, ref)
            # another depth cut than the run's: against a run with that cut
            other = 0.0 if tvm > 0 else 1.0
            ref2 = G.run_emission(dict(prm, tau_vert_max=other))["L_tot"][:, 0]
            free0 = torch.cuda.mem_get_info()[0]
            got2 = G.emission_ltot_static(0, n_chan, other)
            assert np.allclose(got2, ref2, rtol=1e-5, atol=0.0)
            assert torch.cuda.mem_get_info()[0] == free0         # no device memory taken by the call
            with pytest.raises(gpu.GcmcrtError):
                G.emission_ltot_static(3, 2, tvm)
            with pytest.raises(gpu.GcmcrtError):
                G.emission_ltot_static(0, n_chan + 1, tvm)


def test_static_scratch_limit_is_enforced_with_a_clear_error(gpu):
    # (n_chan * ncol + n_chan) * 8 bytes must fit GCMCRT_STATIC_SCRATCH_BYTES = 8 MiB: 40 x 32 columns -> 818 channels
    nlon, nlat, nlev = 40, 32, 4
    ncol = nlon * nlat
    n_max = gpu.STATIC_SCRATCH_BYTES // 8 // (ncol + 1)
    n_chan = n_max + 1
    grid, opac, prm = _case(nlon, nlat, nlev, n_chan, seed=4)
    with gpu.Grid(grid) as G:
        G.set_opacity(opac)
        ref = G.run_emission(prm)["L_tot"][:, 0]
        with pytest.raises(gpu.GcmcrtError) as ei:
            G.emission_ltot_static(0, n_chan, prm["tau_vert_max"])
        msg = str(ei.value)
        assert "scratch" in msg and str(gpu.STATIC_SCRATCH_BYTES) in msg and str((n_chan * ncol + n_chan) * 8) in msg
        # the largest size that fits, and the rest in a second call
        a = G.emission_ltot_static(0, n_max, prm["tau_vert_max"])
        b = G.emission_ltot_static(n_max, n_chan, prm["tau_vert_max"])
        assert np.array_equal(np.concatenate([a, b]), ref)
