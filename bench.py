#!/usr/bin/env python
"""bench.py -- throughput of the gCMCRT hot path (packet transport + peel-off) on B200, BASELINE.json's metric.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg2|cfg3|cfg1]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

One *step* is one pass of the whole hot path over one batch of synthetic input:
gcmcrt_set_opacity (opacity staging) followed by gcmcrt_run_albedo / gcmcrt_run_emission over every channel of the
workload with the full packet count.  The default workload is BASELINE.json configs[1] ("cfg2": 64x32x60 grid,
11 bands x 16 g-points = 176 channels, 1e6 packets per channel, albedo).  `value` is packet-events per second with
the opacity tables already resident in HBM; `e2e` is the same metric through the same C-ABI calls with HOST
(pinned) opacity tables and host result buffers, so that the host->device copies of the tables and the
device->host copies of the spectra are inside the timed region.

N > 1: channels are independent, so every rank runs the same per-GPU workload on its own
range of global channel indices (chan0 = rank * n_chan keys the Philox streams: different channels, no data-path
collective); "scaling": "weak".  Timing: CUDA events around the K steps on the launching stream, barrier +
synchronize on both sides, max over ranks.

--impl reference times the CPU oracle (oracle/, test infrastructure) on the host cores on a bounded packet sample of
the same workload; it is the slow baseline, not the target.
"""
import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2110_15640_b200 import workloads as wl  # noqa: E402  (input generators only: no method arithmetic)

METRIC = "packet_events_per_second"
UNIT = "events/s"

# Lane-instructions (FP32/INT issue slots) per unit of work, audited from the executed instruction counts of the ncu
# source page (profiles/ncu_full_r02_cfg2.txt, _cfg3.txt, _cfg4.txt): what the kernels execute on
# ACTIVE lanes for the method itself -- idle lanes, unissued cycles, the per-CTA geometry-table load and the vote /
# shuffle / atomic helper instructions are not work.
#   segment = the plain-crossing loop (17.7: 18 issued instructions per crossing) + ray_run entry / exit (amortised over
#             the segments of a round) + cone / half-plane / column updates
#   peel ray = record read, phase function, ray set-up (ray_init), round control, exp, bin accumulation
I_UNITS = {            # workload: (per peel segment, per peel ray)
    "cfg2": (28.9, 450.0),
    "cfg3": (37.3, 292.0),     # ~9 segments per ray (rays toward 8 phases; those that end on the lower boundary are not marched,
                               # and half of the rays are not even set up): entry / exit weighs more; the record and the
                               # phase-function inputs serve 8 rays
    "cfg4": (28.4, 450.0),
}
I_SEG_1D = 23.0      # nlat = nlon = 1: loop + entry / exit, no lateral crossings
I_SEG_T = 24.3       # one crossing on a packet flight (first flights + generations, same march code)
I_EVENT = 1000.0     # per event on the transport side: Philox block, absorb / scatter, phase-function sample, rotation, ray
                     # set-up, record write + read, flight hand-over (executed: 785 per first flight, 637 per later event)
# dram__bytes_read.sum + dram__bytes_write.sum per peel_kernel launch at the default sizes, from ncu --set full captures
PEEL_DRAM_BYTES_PER_LAUNCH = {
    "cfg2": (7.955e9, "profiles/ncu_full_r02_cfg2.txt: 4 launches of a step, ~94 M events each"),
    "cfg3": (11.941e9, "profiles/ncu_full_r02_cfg3.txt: 6 launches of a step, ~1e8 events x 8 observers each"),
    "cfg4": (3.643e9, "profiles/ncu_full_r02_cfg4.txt: 2000 wavelengths, ~5e7 events per launch"),
}


def make_workload(name, packets=None, channels=None):
    if name == "cfg1":
        grid, opac, prm = wl.cfg1(packets=packets or 100000)
        mode = "albedo"
    elif name == "cfg2":
        grid, opac, prm = wl.cfg2(packets=packets or 1000000)
        mode = "albedo"
    elif name == "cfg3":
        grid, opac, prm = wl.cfg3(packets=packets or 1000000)
        mode = "emission"
    elif name == "cfg4":
        # high-resolution Doppler-shifted emission; the full 1e4 wavelength points take ~2 min of numpy to generate
        # (4.9 GB of tables), so --channels can cut the wavelength range for a quick look (say so when quoting it)
        grid, opac, prm = wl.cfg4(packets=packets or 100000, **({"n_chan": channels} if channels else {}))
        mode = "emission"
    elif name == "cfg5":
        # large high-resolution run, emission + albedo at 4 phases, node tables streamed in wavelength batches; the
        # default 4096 of the 1e5 wavelength points keep a step at a few seconds (--channels 100000 for all of them)
        grid, opac, prm = wl.cfg5(packets=packets or 100000, n_chan=channels or 4096)
        mode = "emission+albedo"
    else:
        raise SystemExit("unknown workload %s" % name)
    return grid, opac, prm, mode


def peaks():
    """Roofline denominators: MEASURED_PEAKS.json (driver-written) else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": float(p.get("hbm_gbs", 6650.0)), "sm_max_mhz": float(p.get("sm_max_mhz", 1965.0)),
                "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


def rank_chan0(rank, n_chan_per_gpu):
    """Weak scaling over channels: rank r runs its own n_chan_per_gpu channels, whose global
    indices start here; the index keys the Philox streams, so the ranks simulate different channels."""
    return rank * n_chan_per_gpu


def reduce_over_ranks(ms, sums, world, device="cpu"):
    """Step time = max over ranks (device-timed on every rank), work counters = sum over ranks.  The only
    communication of the multi-GPU path: no data-path collective.  Works with any torch.distributed backend."""
    if world <= 1:
        return float(ms), [float(x) for x in sums]
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    u = torch.tensor([float(x) for x in sums], device=device, dtype=torch.float64)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), [float(x) for x in u.tolist()]


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md): ONE nvidia-smi process polling
    every 200 ms, as the recipe does.  (A new nvidia-smi process per sample initialises NVML every time, and that was
    measured to stall the device-driven pass loop by up to 30 ms a sample; the polling process does not.)"""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            time.sleep(0.3)     # the first sample is on its way before the timed region starts
        except Exception:
            self.proc = None

    def summary(self):
        rows = []
        if self.proc is not None:
            self.proc.terminate()
            try:
                out, _ = self.proc.communicate(timeout=5)
            except Exception:
                self.proc.kill()
                out = ""
            for line in (out or "").splitlines():
                f = [x.strip() for x in line.split(",")]
                if len(f) >= 7:
                    rows.append(f)
        sm = [float(r[0]) for r in rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if r[1].replace(".", "").isdigit()]
        reasons = []
        for name, col in (("hw_slowdown", 3), ("hw_thermal_slowdown", 4), ("sw_thermal_slowdown", 5), ("sw_power_cap", 6)):
            if any(r[col].lower().startswith("active") for r in rows):
                reasons.append(name)
        pw = [float(r[2]) for r in rows if r[2].replace(".", "").isdigit()]
        # the samples taken under load: the idle ones before / after the steps sit at a lower clock
        load = [c for c, w in zip(sm, pw)] if len(sm) == len(pw) else sm
        return {"sm_mhz": float(np.median(load)) if load else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(rows), "reasons": reasons}


def oracle_leg(name, grid, opac, prm, mode, budget_s=15.0, threads=None):
    """Time the CPU oracle, as it stands, on a bounded sample: the first n packets of every channel.
    threads = None: all host cores (OpenMP over the packet batches); 1: the serial oracle."""
    import oracle  # test infrastructure; allowed here (cpu_baseline / --impl reference)
    cores = threads or os.cpu_count() or 1
    run = oracle.run_albedo if mode == "albedo" else oracle.run_emission

    def once(n):
        # the first n packets of every channel as a run of their own (streams are keyed by packet id only): its 32
        # batches spread over the host threads, which a sub-range of the full run (all in batch 0) would not
        p = dict(prm, packets_per_channel=n, pkt_begin=0, pkt_end=n, n_threads=cores)
        t0 = time.perf_counter()
        o = run(grid, opac, p)
        return time.perf_counter() - t0, o["counters"]

    full = int(prm["packets_per_channel"])
    once(64)                      # thread pool and page-in, untimed
    n1, n2 = min(full, 256 if cores == 1 else 1024), min(full, 1024 if cores == 1 else 4096)
    t1, c = once(n1)              # two calibration points: per-channel table preparation is a fixed cost
    n_run, dt = n1, t1
    if n2 > n1:
        t2, c = once(n2)
        n_run, dt = n2, t2
        per_pkt = max((t2 - t1) / (n2 - n1), 1e-9)
        fixed = max(t1 - per_pkt * n1, 0.0)
        n3 = int(min(full, max(n2, (budget_s - fixed) / per_pkt)))
        n3 = max(32, (n3 // 32) * 32)
        if n3 > n2:
            dt, c = once(n3)
            n_run = n3
    n2 = n_run
    nseg = c["segments_transport"] + c["segments_peel"]
    n_chan = int(np.asarray(opac["lambda"]).size)
    return {"value": c["events"] / dt, "unit": UNIT, "cores": min(cores, int(prm.get("n_batches", 32))), "kind": "oracle",
            "sample": "%s: first %d of %d packets of each of %d channels (%.1f s wall, %s)"
                      % (name, n2, full, n_chan, dt, "serial" if cores == 1 else "OpenMP over batches"),
            "segments_per_s": nseg / dt, "seconds": dt, "events": int(c["events"])}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    grid, opac, prm, mode = make_workload(args.workload, args.packets, args.channels)
    vals = []
    base = None
    budget = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for it in range(args.warmup + args.steps):
        base = oracle_leg(args.workload, grid, opac, prm, mode, budget_s=budget)
        if it >= args.warmup:
            vals.append(base)
    v = float(np.mean([b["value"] for b in vals]))
    ms = float(np.mean([b["seconds"] for b in vals])) * 1e3
    n_chan = int(np.asarray(opac["lambda"]).size)
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "mode": mode, "n_chan_per_gpu": n_chan,
                       "packets_per_channel": int(prm["packets_per_channel"]),
                       "grid": list(np.asarray(grid["T"]).shape), "note": "CPU oracle on a bounded packet sample"},
            "cpu_baseline": {k: base[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    line["cpu_baseline"]["value"] = v
    print(json.dumps(line), flush=True)


COUNTER_KEYS = ("events", "segments_transport", "segments_peel", "rays_peel", "packets_escaped", "packets_absorbed",
                "packets_surface", "packets_stuck", "passes", "launches", "ms_stage", "ms_emission_cdf", "ms_transport",
                "ms_peel", "ms_sort", "device_status")


class Leg:
    """One workload on one handle: device-resident tables, the step function, and the three measurements taken of it --
    `value` (K steps only enqueued: device outputs, counters assembled on the device and read after the timed region),
    the kernel split (steps with run_params.timing = 1: the library records cudaEvents on the launching stream around
    its kernels) and, for the headline workload, `e2e` (host tables in, host spectra out)."""

    def __init__(self, name, args, binding, torch, stream, rank, grid=None, opac=None, prm=None, mode=None, dev_tables=None):
        self.name, self.args, self.binding, self.torch, self.stream = name, args, binding, torch, stream
        if grid is None:
            grid, opac, prm, mode = make_workload(name, args.packets if name == args.workload else None,
                                                  args.channels if name == args.workload else (2000 if name == "cfg4" else None))
        self.grid, self.opac, self.prm, self.mode = grid, dict(opac), prm, mode
        self.n_chan = int(np.asarray(opac["lambda"]).size)
        self.opac["chan0"] = rank_chan0(rank, self.n_chan)   # this rank's global channel range (keys the Philox streams)
        self.tab_keys = [k for k in ("k_abs", "k_sca_ray", "k_sca_cld", "g_cld", "node_kabs", "p_cell") if opac.get(k) is not None]
        self.streamed = name == "cfg5"
        self.dev = dict(self.opac)
        self.host = None
        for k in self.tab_keys:
            if dev_tables is not None and k in dev_tables:
                self.dev[k] = dev_tables[k]
            else:
                self.dev[k] = torch.from_numpy(np.ascontiguousarray(opac[k], dtype=np.float32)).cuda()
        self.G = binding.Grid(grid, stream=stream)
        self.ncell = int(np.asarray(grid["T"]).size)
        if self.streamed:
            self.coef = torch.from_numpy(opac["k_ray_chan"]).cuda()

    def pin_host_tables(self):
        self.host = dict(self.opac)
        for k in self.tab_keys:
            self.host[k] = self.torch.from_numpy(np.ascontiguousarray(self.opac[k], dtype=np.float32)).pin_memory()
        h2d = sum(self.host[k].numel() * 4 for k in self.tab_keys) + self.n_chan * 4
        if self.streamed:   # the cells' pressures travel with every batch
            h2d += self.host["p_cell"].numel() * 4 * (len(wl.cfg5_batches(self.opac, batch=self.args.batch)) - 1)
        return h2d

    def step(self, op, device_outputs, timing=0, counters="host"):
        """One pass of the whole hot path over the workload; returns the list of run results."""
        # run_params.concurrency: the run's channels in K parts side by side on internal handles and streams (the library
        # ignores it for timing = 1); two parts for cfg5, whose handles hold 48 GB each
        K = 0 if timing else (min(self.args.concurrency, 2) if self.streamed else self.args.concurrency)
        prm = dict(self.prm, timing=timing, concurrency=K)
        G = self.G
        if not self.streamed:
            G.set_opacity(op)
            fn = G.run_albedo if self.mode == "albedo" else G.run_emission
            return [fn(prm, device_outputs=device_outputs, counters=counters)]
        # config 5: per wavelength batch (+ halo channels for the Doppler window) the node tables go through
        # gcmcrt_set_opacity_nodes, the batch's Rayleigh table is filled on the device, and the batch is run in
        # emission and in albedo mode toward the 4 phases
        outs = []
        obs = np.asarray(prm["obs_dir"], dtype=np.float64).reshape(-1, 3)
        for c0, c1, lo, hi in wl.cfg5_batches(self.opac, batch=self.args.batch, halo=int(prm["doppler_halfwidth"])):
            sub = dict(op, chan0=op["chan0"] + lo, node_kabs=op["node_kabs"][lo:hi])
            sub["lambda"] = self.opac["lambda"][lo:hi]
            sub["k_sca_ray"] = self.coef[lo:hi, None].expand(hi - lo, self.ncell).contiguous()
            G.set_opacity_nodes(sub)
            # with doppler_on every observer is a run of its own on its own shifted table (L326-328): phases outermost,
            # so that the emission and the albedo run toward a phase share one Doppler staging (4 per batch, not 8)
            for o in range(obs.shape[0]):
                for fn in (G.run_emission, G.run_albedo):
                    outs.append(fn(dict(prm, obs_dir=obs[o:o + 1], chan_begin=c0 - lo, chan_end=c1 - lo),
                                   device_outputs=device_outputs, counters=counters))
        return outs

    def sum_counters(self, outs):
        acc = dict.fromkeys(COUNTER_KEYS, 0)
        for o in outs:
            c = o["counters"] if "counters" in o else self.binding.read_counters(o["counters_dev"])
            for k in COUNTER_KEYS:
                acc[k] += c[k]
        return acc

    def timed(self, op, device_outputs, steps, barrier, timing=0, counters="device"):
        torch = self.torch
        outs = []
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(self.stream)
        for _ in range(steps):
            outs += self.step(op, device_outputs, timing=timing, counters=counters)
        e1.record(self.stream)
        host_s = time.perf_counter() - t0      # what the host spent enqueueing (the calls return before the work is done)
        barrier()
        return e0.elapsed_time(e1), self.sum_counters(outs), outs, host_s

    def d2h_bytes(self, outs, steps):
        return sum(o[k].nbytes for o in outs for k in ("flux_sum", "L_tot", "value", "sigma") if k in o) // max(steps, 1)

    def roofline(self, acc, ms_total, steps, pk):
        """Roofline of the dominant kernel (peel_kernel) from a timing = 1 leg: algorithmic lane-instructions over the
        kernel's device time (cudaEvents the library records on the launching stream around every launch)."""
        is3d = np.asarray(self.grid["T"]).shape[0] > 1 or np.asarray(self.grid["T"]).shape[1] > 1
        i_seg, i_ray = I_UNITS.get(self.name, I_UNITS["cfg2"])
        if not is3d:
            i_seg = I_SEG_1D
        work_seg = acc["segments_peel"] * i_seg
        work = work_seg + acc["rays_peel"] * i_ray
        dur_ms = acc["ms_peel"]
        work_t = acc["segments_transport"] * (I_SEG_T if is3d else I_SEG_1D) + acc["events"] * I_EVENT
        n_dom = max(1, acc["passes"])
        peak = 148 * 128 * pk["sm_max_mhz"] * 1e6 / 1e12          # T lane-instr/s
        achieved = work / (dur_ms * 1e-3) / 1e12 if dur_ms > 0 else 0.0
        hbm_bytes = self.n_chan * self.ncell * 4 * (len(self.tab_keys) + 1 + 4)   # tables read once + alpha/prop written once
        if self.streamed:   # Rayleigh table written once; 4 Doppler stagings (one per phase) each read it and write alpha + prop
            hbm_bytes = self.n_chan * self.ncell * (4 + 4 * (4 + 4 + 16))
        tr = PEEL_DRAM_BYTES_PER_LAUNCH.get(self.name) if self.args.packets is None else None
        return {"bound": "alu", "kernel": "peel_kernel", "achieved": achieved, "peak": peak,
                "unit": "Tlane-instr/s", "frac": achieved / peak if peak else None,
                # the floor of that fraction: the ray segments alone (the per-segment count is the audited loop body), no
                # per-ray set-up counted as work
                "frac_segments_only": work_seg / (dur_ms * 1e-3) / 1e12 / peak if dur_ms > 0 else None,
                "traffic": tr[0] if tr else None,
                "traffic_unit": "dram__bytes_read + write per peel_kernel launch, ncu --set full" + (" (%s)" % tr[1] if tr else ""),
                "peak_source": "148 SM x 128 FP32 lanes x sm_max_mhz (%s)" % pk["source"],
                "lane_instr_per_unit": {"peel_segment": i_seg, "peel_ray": i_ray, "transport_segment": I_SEG_T, "event": I_EVENT,
                                        "source": "executed thread-instructions per unit, ncu source page (profiles/ncu_full_r02_*.txt)"},
                "work_lane_instr_per_launch": work / n_dom, "ms_per_launch": dur_ms / n_dom,
                "timing_steps": steps,
                "hbm_term": {"bytes_per_step": hbm_bytes, "ms_at_peak": hbm_bytes / (pk["hbm_gbs"] * 1e9) * 1e3,
                             "peak_gbs": pk["hbm_gbs"]},
                "kernel_ms_per_step": {k: acc[k] / steps for k in ("ms_stage", "ms_emission_cdf", "ms_transport", "ms_sort", "ms_peel")},
                "transport_kernels": {"achieved": work_t / (acc["ms_transport"] * 1e-3) / 1e12 if acc["ms_transport"] > 0 else 0.0,
                                      "frac": work_t / (acc["ms_transport"] * 1e-3) / 1e12 / peak if acc["ms_transport"] > 0 else None,
                                      "note": "launch sort + first flights + interact generations + persistent tail, same units"},
                "whole_step": {"achieved": (work + work_t) / (ms_total * 1e-3) / 1e12,
                               "frac": (work + work_t) / (ms_total * 1e-3) / 1e12 / peak,
                               "ms_per_step_timing_mode": ms_total / steps}}

    def close(self):
        self.G.close()


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2110_15640_b200 import binding, build

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU path)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    binding.lib()
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    leg = Leg(args.workload, args, binding, torch, stream, rank)
    N = int(leg.prm["packets_per_channel"])
    warm = max(args.warmup, 3)
    for _ in range(warm):
        leg.step(leg.dev, True, counters="device")
    sampler = ClockSampler(local)
    sampler.start()
    ms, acc, _, host_s = leg.timed(leg.dev, True, args.steps, barrier)
    clocks = sampler.summary()
    # kernel split / roofline: the same steps with run_params.timing = 1 (host-driven pass loop, cudaEvents around the kernels)
    t_steps = max(1, min(args.steps, 5))
    leg.step(leg.dev, True, timing=1)
    ms_t, acc_t, _, _ = leg.timed(leg.dev, True, t_steps, barrier, timing=1, counters="host")
    # e2e: host tables in, host spectra out
    h2d = leg.pin_host_tables()
    leg.step(leg.host, False)
    ms_e2e, acc_e2e, outs_e2e, _ = leg.timed(leg.host, False, args.steps, barrier, counters="host")
    d2h = leg.d2h_bytes(outs_e2e, args.steps)

    ms, (ev_all, seg_all) = reduce_over_ranks(ms, [acc["events"], acc["segments_transport"] + acc["segments_peel"]],
                                              world, "cuda")
    ms_e2e, (ev_all_e2e,) = reduce_over_ranks(ms_e2e, [acc_e2e["events"]], world, "cuda")
    value = ev_all / (ms * 1e-3)
    e2e_value = ev_all_e2e / (ms_e2e * 1e-3)

    if rank == 0:
        pk = peaks()
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": warm, "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": args.workload, "mode": leg.mode, "n_chan_per_gpu": leg.n_chan, "packets_per_channel": N,
                           "n_obs": int(np.asarray(leg.prm["obs_dir"]).reshape(-1, 3).shape[0]),
                           "grid": list(np.asarray(leg.grid["T"]).shape), "parallelism": "channels x %d" % world,
                           "concurrency": "run_params.concurrency = %d (channel parts side by side on one GPU)" % (min(args.concurrency, 2) if leg.streamed else args.concurrency),
                           "l2": "opacity tables (%.0f MB) + staged tables exceed the 126 MB L2; no flush" % (h2d / 1e6)},
                "events_per_step": ev_all / args.steps, "segments_per_s": seg_all / (ms * 1e-3),
                "spectra_per_s": world * args.steps / (ms * 1e-3),
                "host_enqueue_ms_per_step": host_s * 1e3 / args.steps,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                        "ms_per_step": ms_e2e / args.steps},
                "gpu_launches": int(acc["launches"]), "clocks": clocks, "roofline": leg.roofline(acc_t, ms_t, t_steps, pk),
                "counters_per_step": {k: acc[k] / args.steps for k in
                                      ("events", "segments_transport", "segments_peel", "rays_peel", "packets_escaped",
                                       "packets_absorbed", "packets_surface", "packets_stuck", "passes")}}
        assert acc["device_status"] == 0, "pass loop reported an error"
        # config 5 has no per-cell table for the oracle to read (328 GB at full size): no cpu_baseline leg there
        if world == 1 and not args.no_cpu and not leg.streamed:
            o0 = dict(leg.opac, chan0=0)
            cpu = oracle_leg(args.workload, leg.grid, o0, leg.prm, leg.mode)
            line["cpu_baseline"] = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}
            cpu1 = oracle_leg(args.workload, leg.grid, o0, leg.prm, leg.mode, budget_s=8.0, threads=1)
            line["cpu_baseline_1core"] = {k: cpu1[k] for k in ("value", "unit", "cores", "kind", "sample")}
        # the other configurations north_star names (3D correlated-k emission, high resolution): short legs of their
        # own after the headline, outside its timed region
        if world == 1 and args.workload == "cfg2" and args.packets is None and not args.no_extra:
            extra = {}

            def short_leg(lg):
                for _ in range(3):
                    lg.step(lg.dev, True, counters="device")
                ms_x, acc_x, _, _ = lg.timed(lg.dev, True, 3, barrier)
                lg.step(lg.dev, True, timing=1)
                ms_xt, acc_xt, _, _ = lg.timed(lg.dev, True, 2, barrier, timing=1, counters="host")
                return {"ms_per_step": ms_x / 3, "value": acc_x["events"] / (ms_x * 1e-3), "unit": UNIT, "steps": 3, "warmup": 3,
                        "config": {"workload": lg.name, "mode": lg.mode, "n_chan_per_gpu": lg.n_chan,
                                   "packets_per_channel": int(lg.prm["packets_per_channel"]),
                                   "n_obs": int(np.asarray(lg.prm["obs_dir"]).reshape(-1, 3).shape[0]),
                                   "grid": list(np.asarray(lg.grid["T"]).shape), "concurrency": args.concurrency},
                        "rays_per_s": acc_x["rays_peel"] / (ms_x * 1e-3),
                        "counters_per_step": {k: acc_x[k] / 3 for k in ("events", "segments_transport", "segments_peel", "rays_peel", "passes")},
                        "roofline": lg.roofline(acc_xt, ms_xt, 2, pk)}

            # config 3: the same grid and tables as config 2, so the tables already on the device serve it
            _, _, p3 = wl.cfg3(packets=1000000)
            leg.close()      # the handle's working buffers (and its internal handles'); the tables in leg.dev stay
            lg = Leg("cfg3", args, binding, torch, stream, rank, leg.grid, leg.opac, p3, "emission", dev_tables=leg.dev)
            extra["cfg3"] = short_leg(lg)
            lg.close()
            leg.dev = lg.dev = None
            torch.cuda.empty_cache()
            # config 4 on 2000 of its 1e4 wavelength points (the full table takes minutes of numpy to generate)
            lg = Leg("cfg4", args, binding, torch, stream, rank)
            extra["cfg4"] = short_leg(lg)
            lg.close()
            line["workloads"] = extra
        print(json.dumps(line), flush=True)
    if leg.G.handle:
        leg.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--channels", type=int, default=None, help="cfg4 / cfg5: number of wavelength points (default 10000 / 4096)")
    ap.add_argument("--batch", type=int, default=1024, help="cfg5: wavelength points per streamed opacity batch")
    ap.add_argument("--packets", type=int, default=None, help="override packets per channel (debugging only)")
    ap.add_argument("--concurrency", type=int, default=3, help="run_params.concurrency of the timed steps (0 = one run per call)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline legs")
    ap.add_argument("--no-extra", action="store_true", help="skip the cfg3 / cfg4 legs of the default run")
    args = ap.parse_args()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "ours" and world != args.gpus and world == 1 and args.gpus > 1:
        # plain `python bench.py --gpus N`: relaunch under torchrun, one rank per GPU
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 1000), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
