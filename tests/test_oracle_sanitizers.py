"""The CPU oracle under AddressSanitizer + UndefinedBehaviorSanitizer: a small C driver is
compiled together with oracle/gcmcrt_oracle.c with -fsanitize=address,undefined -fno-sanitize-recover=all and runs
albedo (3D grid, Lambert surface, images, contribution functions, every variance-reduction switch), emission (Doppler
shifts, depth cut, composite bias), transmission (raytracer and with multiple scattering) and the ray integrator.  Any out-of-bounds access, use after free,
leak, signed overflow or misaligned access aborts the driver and fails the test."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r'''
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include "gcmcrt_oracle.h"

#define NLEV 5
#define NLAT 4
#define NLON 6
#define NCELL (NLEV * NLAT * NLON)
#define NCHAN 3
#define NOBS 2
#define NPKT 300
#define NPIX 4
#define NB 8

int main(void)
{
    const double pi = 3.14159265358979323846;
    double r[NLEV + 1], th[NLAT + 1], ph[NLON + 1];
    for (int i = 0; i <= NLEV; ++i) r[i] = 1.0e6 + 6.0e4 * i;
    for (int j = 0; j <= NLAT; ++j) th[j] = pi * j / NLAT;
    for (int k = 0; k <= NLON; ++k) ph[k] = 2.0 * pi * k / NLON;
    static float T[NCELL], rho[NCELL], u[NCELL], v[NCELL], w[NCELL];
    static float kabs[NCHAN * NCELL], kray[NCHAN * NCELL], kcld[NCHAN * NCELL], gc[NCHAN * NCELL], lam[NCHAN];
    unsigned s = 12345u;
    for (int c = 0; c < NCELL; ++c) {
        s = s * 1664525u + 1013904223u;
        T[c] = 900.0f + (float)(s >> 20) * 0.3f;
        rho[c] = 1.0f + (float)((s >> 8) & 255) / 256.0f;
        u[c] = 3000.0f * (float)sin(0.1 * c); v[c] = 500.0f * (float)cos(0.3 * c); w[c] = 10.0f;
    }
    for (int c = 0; c < NCHAN; ++c) {
        lam[c] = 2.0e-6f * (1.0f + 1.0e-5f * (float)c);
        for (int m = 0; m < NCELL; ++m) {
            s = s * 1664525u + 1013904223u;
            kabs[c * NCELL + m] = 2.0e-6f * (1.0f + (float)(s >> 24) / 64.0f);
            kray[c * NCELL + m] = 3.0e-6f;
            kcld[c * NCELL + m] = 4.0e-6f;
            gc[c * NCELL + m] = 0.6f;
        }
    }
    orc_grid g;
    memset(&g, 0, sizeof g);
    g.nlev = NLEV; g.nlat = NLAT; g.nlon = NLON; g.r_edges = r; g.colat_edges = th; g.lon_edges = ph;
    g.T = T; g.rho = rho; g.u = u; g.v = v; g.w = w; g.Omega = 2.0e-5; g.surface_albedo = 0.4;
    orc_opacity op;
    memset(&op, 0, sizeof op);
    op.n_chan = NCHAN; op.chan0 = 7; op.lambda = lam; op.k_abs = kabs; op.k_sca_ray = kray; op.k_sca_cld = kcld; op.g_cld = gc;
    double obs[NOBS * 3] = {1.0, 0.0, 0.0, 0.0, 0.6, 0.8};
    double total = 0.0;
    for (int variant = 0; variant < 7; ++variant) {
        orc_params p;
        memset(&p, 0, sizeof p);
        p.star_dir[0] = 0.8; p.star_dir[2] = 0.6;
        p.n_obs = NOBS; p.obs_dir = obs; p.packets_per_channel = NPKT; p.pkt_begin = 0; p.pkt_end = NPKT; p.seed = 5;
        p.scatter_on = 1; p.tau_vert_max = 30.0; p.tau_cut = 50.0; p.npix = NPIX; p.n_batches = NB; p.n_threads = 2;
        p.star_radius = 7.0e8; p.planet_xy[0] = 1.0e8; p.ld_c1 = 0.3; p.ld_c2 = 0.2;
        if (variant == 1) { p.survival_bias = 1; p.roulette_w_min = 0.1; p.roulette_survive = 0.3; p.cloud_phase = 1; }
        if (variant == 2) { p.forced_scatter = 2; p.survival_bias = 1; p.roulette_w_min = 0.1; p.roulette_survive = 0.3; p.cloud_phase = 2; }
        if (variant == 3) { p.continuous_absorption = 1; p.max_events = 6; }
        if (variant == 4) { p.doppler_on = 1; p.doppler_halfwidth = 1; p.emission_bias = 0.4; p.tau_vert_max = 2.0; }
        if (variant == 5) { p.forced_scatter = 1; p.pkt_begin = 17; p.pkt_end = 201; p.star_solid_angle = 0.01; p.stretch_alpha = 0.5; }
        if (variant == 6) { p.scatter_on = 0; p.n_threads = 1; }
        for (int mode = 0; mode < 3; ++mode) {
            orc_result out;
            memset(&out, 0, sizeof out);
            out.flux_sum = calloc((size_t)NCHAN * NOBS * NB, sizeof(double));
            out.L_tot = calloc((size_t)NCHAN * NOBS, sizeof(double));
            out.image = calloc((size_t)NCHAN * NOBS * NPIX * NPIX, sizeof(double));
            out.event_count = calloc((size_t)NCHAN * NPKT, sizeof(uint32_t));
            out.contrib = calloc((size_t)NCHAN * NOBS * 2 * NCELL, sizeof(double));
            int rc = mode == 0 ? orc_run_albedo(&g, &op, &p, &out)
                   : mode == 1 ? orc_run_emission(&g, &op, &p, &out) : orc_run_transmission(&g, &op, &p, &out);
            if (rc != 0) { printf("variant %d mode %d rc %d\n", variant, mode, rc); return 2; }
            for (int m = 0; m < NCHAN * NOBS * NB; ++m) total += out.flux_sum[m];
            free(out.flux_sum); free(out.L_tot); free(out.image); free(out.event_count); free(out.contrib);
        }
    }
    {   /* the ray integrator on its own, rays from every level in fixed directions */
        double pos[3 * 40], dir[3 * 40], tau[40], path[40];
        int hit[40];
        long nseg[40];
        for (int m = 0; m < 40; ++m) {
            double a = 0.37 * m, b = 0.11 * m + 0.2, rr = 1.0e6 + 7.4e3 * m;
            pos[3 * m] = rr * sin(b) * cos(a); pos[3 * m + 1] = rr * sin(b) * sin(a); pos[3 * m + 2] = rr * cos(b);
            dir[3 * m] = sin(2.0 * b) * cos(3.0 * a); dir[3 * m + 1] = sin(2.0 * b) * sin(3.0 * a); dir[3 * m + 2] = cos(2.0 * b);
        }
        if (orc_ray_tau(&g, &op, 1, 40, pos, dir, tau, hit, nseg, path) != 0) return 3;
        for (int m = 0; m < 40; ++m) total += tau[m];
    }
    printf("ok %.6e\n", total);
    return isfinite(total) && total > 0.0 ? 0 : 4;
}
'''


def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    if shutil.which("gcc") is None:
        pytest.skip("no gcc")
    src = tmp_path / "driver.c"
    src.write_text(DRIVER)
    exe = tmp_path / "driver"
    odir = os.path.join(ROOT, "oracle")
    cmd = ["gcc", "-std=c99", "-D_GNU_SOURCE", "-O1", "-g", "-fopenmp", "-fsanitize=address,undefined",
           "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-I", odir, str(src),
           os.path.join(odir, "gcmcrt_oracle.c"), "-o", str(exe), "-lm"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0 and "sanitize" in r.stderr:
        pytest.skip("gcc without sanitizer runtimes: " + r.stderr[-200:])
    assert r.returncode == 0, r.stderr[-2000:]
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1",
               OMP_NUM_THREADS="2")
    r = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, (r.stdout[-500:], r.stderr[-3000:])
    assert r.stdout.startswith("ok ")
