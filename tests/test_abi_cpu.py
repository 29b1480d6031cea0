"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol include/gcmcrt.h declares,
the ctypes structs match the header, and calls fail loudly (never fall back) without a CUDA device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2110_15640_b200 import binding, build, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def test_library_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "gcmcrt.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(gcmcrt_[a-z_0-9]+)\s*\(", hdr)))
    assert set(declared) == set(binding.EXPORTS)
    for name in ("gcmcrt_grid_create", "gcmcrt_set_opacity", "gcmcrt_run_albedo", "gcmcrt_run_emission",
                 "gcmcrt_destroy"):
        assert name in declared          # the five calls north_star names
    for name in declared:
        assert getattr(lib, name) is not None
    assert b"sm_100a" in lib.gcmcrt_version()


def test_struct_layouts_match_header():
    # gcmcrt_run_params: 3 doubles, int(+pad), ptr, 4 u64, 6 int, 3 doubles, 2 int  (natural alignment)
    assert C.sizeof(binding.RunParams) == 24 + 8 + 8 + 32 + 24 + 24 + 8 + 24 + 40 + 8 + 8 + 24   # + survival_bias (int + pad), 2 doubles; + 5 doubles (transmission); + cloud_phase, forced_scatter; + continuous_absorption (int + pad); + star_solid_angle, stretch_alpha, timing + concurrency (2 ints)
    assert binding.RunParams.survival_bias.offset == 128 and binding.RunParams.roulette_survive.offset == 144
    assert binding.RunParams.obs_dir.offset == 32 and binding.RunParams.seed.offset == 64
    assert binding.RunParams.emission_bias.offset == 96 and binding.RunParams.n_batches.offset == 124
    assert C.sizeof(binding.Counters) == 136     # 11 u64/double + 5 ms doubles + device_status
    assert binding.RunParams.star_solid_angle.offset == binding.RunParams.continuous_absorption.offset + 8 and binding.RunParams.stretch_alpha.offset == binding.RunParams.star_solid_angle.offset + 8 and binding.RunParams.timing.offset == binding.RunParams.stretch_alpha.offset + 8 and binding.RunParams.concurrency.offset == binding.RunParams.timing.offset + 4
    assert C.sizeof(binding.Result) == 64      # 8 pointers (contrib added with the contribution functions)


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    grid, opac, prm = wl.cfg1(packets=10)
    with pytest.raises(binding.GcmcrtError) as e:
        binding.Grid(grid)
    assert e.value.code == binding.E_CUDA
    # argument validation comes first and reports E_INVALID with a message
    h = C.c_void_p()
    r = np.array([2.0, 1.0]); th = np.array([0.0, np.pi]); ph = np.array([0.0, 2 * np.pi])
    one = np.ones(1, dtype=np.float32)
    rc = lib.gcmcrt_grid_create(C.byref(h), 1, 1, 1, r.ctypes.data, th.ctypes.data, ph.ctypes.data, one.ctypes.data,
                                one.ctypes.data, None, None, None, 0.0, 0.0, None)
    assert rc == binding.E_INVALID and h.value is None
    assert b"ascending" in lib.gcmcrt_last_error(None)
    assert lib.gcmcrt_destroy(None) == 0
    assert lib.gcmcrt_run_albedo(None, None, None, None) == binding.E_INVALID


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2110_15640_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                # no import / load / link of anything under oracle/ (prose may mention the word)
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "libgcmcrt_oracle" not in src and "gcmcrt_oracle.h" not in src and "orc_" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2110_15640_b200" not in src and "from paper_2110_15640_b200" not in src
            assert "libgcmcrt.so" not in src and "csrc" not in src


def test_header_is_plain_c_and_links(lib, tmp_path):
    """include/gcmcrt.h compiles as C11 (no C++, no torch types), a C program links against libgcmcrt.so, the struct
    sizes the C compiler sees are the ones the ctypes binding uses, and a call without a device fails with a status."""
    import shutil
    import subprocess
    if shutil.which("gcc") is None:
        pytest.skip("no gcc")
    src = tmp_path / "client.c"
    src.write_text(r'''
#include <stdio.h>
#include "gcmcrt.h"
int main(void)
{
    gcmcrt_grid *g = NULL;
    double r[2] = {1.0e6, 2.0e6}, th[2] = {0.0, 3.14159265358979323846}, ph[2] = {0.0, 6.28318530717958647692};
    float T[1] = {1000.0f}, rho[1] = {1.0f};
    int rc = gcmcrt_grid_create(&g, 1, 1, 1, r, th, ph, T, rho, NULL, NULL, NULL, 0.0, 0.0f, NULL);
    printf("%zu %zu %zu %d %s\n", sizeof(gcmcrt_run_params), sizeof(gcmcrt_result), sizeof(gcmcrt_counters), rc,
           gcmcrt_version());
    if (g) gcmcrt_destroy(g);
    return 0;
}
''')
    exe = tmp_path / "client"
    libdir = os.path.dirname(binding.LIB_PATH)
    subprocess.run(["gcc", "-std=c11", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe),
                    "-L", libdir, "-lgcmcrt", "-Wl,-rpath," + libdir], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()
    assert int(out[0]) == C.sizeof(binding.RunParams)
    assert int(out[1]) == C.sizeof(binding.Result)
    assert int(out[2]) == C.sizeof(binding.Counters)
    assert int(out[3]) in (binding.OK, binding.E_CUDA)      # no device here: a status, not a crash or a CPU fallback
    assert "sm_100a" in " ".join(out[4:])
