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
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2110_15640_b200 import workloads as wl  # noqa: E402  (input generators only: no method arithmetic)

METRIC = "packet_events_per_second"
UNIT = "events/s"

# Algorithmic lane-instructions (FP32/INT issue slots) per unit of work; DESIGN.md section "Roofline" derives them
# from the audited SASS of the march loop, the event handler and the launch code.
I_SEG_3D = 27.0      # one 3D cell crossing: radial run 22 executed thread-instructions per segment (PTX loops, 19 issued per
                     # crossing + the run's entry / exit code) + cone / half-plane / column updates 4.7 per segment
                     # (ncu source page, profiles/ncu_full_r01d_ptx_loops.txt)
I_SEG_1D = 22.0      # nlat = nlon = 1: the same radial run, no lateral crossings
I_EVENT = 420.0      # Philox block, phase sampling, rotation, ray setup, event record write + read
PEEL_DRAM_BYTES_PER_LAUNCH_CFG2 = 7.96e9   # ncu: 4 launches of a cfg2 step average 7.946 GB read + 9.2 MB written
I_PEEL_RAY = 300.0   # record + prop read, phase function, ray setup for one (event, observer), exp, bin accumulation


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


class ClockSampler(threading.Thread):
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.rows = []
        self.stop_flag = threading.Event()

    def run(self):
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 7:
                    self.rows.append(f)
            except Exception:
                pass
            self.stop_flag.wait(0.1)

    def summary(self):
        self.stop_flag.set()
        self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        reasons = []
        for name, col in (("hw_slowdown", 3), ("hw_thermal_slowdown", 4), ("sw_thermal_slowdown", 5), ("sw_power_cap", 6)):
            if any(r[col].lower().startswith("active") for r in self.rows):
                reasons.append(name)
        pw = [float(r[2]) for r in self.rows if r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(self.rows), "reasons": reasons}


def oracle_leg(name, grid, opac, prm, mode, budget_s=15.0):
    """Time the CPU oracle, as it stands, on a bounded sample: the first n packets of every channel."""
    import oracle  # test infrastructure; allowed here (cpu_baseline / --impl reference)
    cores = os.cpu_count() or 1
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
    n1, n2 = min(full, 1024), min(full, 4096)
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
            "sample": "%s: first %d of %d packets of each of %d channels (%.1f s wall, OpenMP over batches)"
                      % (name, n2, full, n_chan, dt),
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
            "config": {"workload": args.workload, "mode": mode, "n_chan": n_chan,
                       "packets_per_channel": int(prm["packets_per_channel"]),
                       "grid": list(np.asarray(grid["T"]).shape), "note": "CPU oracle on a bounded packet sample"},
            "cpu_baseline": {k: base[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    line["cpu_baseline"]["value"] = v
    print(json.dumps(line), flush=True)


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

    grid, opac, prm, mode = make_workload(args.workload, args.packets, args.channels)
    n_chan = int(np.asarray(opac["lambda"]).size)
    opac["chan0"] = rank_chan0(rank, n_chan)   # this rank's global channel range (keys the Philox streams)
    N = int(prm["packets_per_channel"])
    tab_keys = [k for k in ("k_abs", "k_sca_ray", "k_sca_cld", "g_cld", "node_kabs", "p_cell") if opac.get(k) is not None]
    stream = torch.cuda.current_stream()
    streamed = args.workload == "cfg5"

    # device-resident tables for `value`, pinned host tables for `e2e`
    dev_opac = dict(opac)
    host_opac = dict(opac)
    for k in tab_keys:
        t = torch.from_numpy(np.ascontiguousarray(opac[k], dtype=np.float32))
        host_opac[k] = t.pin_memory()
        dev_opac[k] = t.cuda()
    h2d = sum(host_opac[k].numel() * 4 for k in tab_keys) + n_chan * 4
    if streamed:   # the cells' pressures travel with every batch
        h2d += host_opac["p_cell"].numel() * 4 * (len(wl.cfg5_batches(opac, batch=args.batch)) - 1)
    G = binding.Grid(grid, stream=stream)

    def step_streamed(op, device_outputs):
        # config 5: per wavelength batch (+ halo channels for the Doppler window) the node tables go through
        # gcmcrt_set_opacity_nodes, the batch's Rayleigh table is filled on the device, and the batch is run in
        # emission and in albedo mode toward the 4 phases; counters and output bytes are summed over the runs
        ncell = int(np.asarray(grid["T"]).size)
        coef = torch.from_numpy(opac["k_ray_chan"]).cuda()
        tot, nbytes = {}, 0
        for c0, c1, lo, hi in wl.cfg5_batches(opac, batch=args.batch, halo=int(prm["doppler_halfwidth"])):
            sub = dict(op, chan0=op["chan0"] + lo, node_kabs=op["node_kabs"][lo:hi])
            sub["lambda"] = opac["lambda"][lo:hi]
            sub["k_sca_ray"] = coef[lo:hi, None].expand(hi - lo, ncell).contiguous()
            G.set_opacity_nodes(sub)
            for fn in (G.run_emission, G.run_albedo):
                out = fn(dict(prm, chan_begin=c0 - lo, chan_end=c1 - lo), device_outputs=device_outputs)
                for k, v in out["counters"].items():
                    tot[k] = tot.get(k, 0) + v
                nbytes += sum(out[k].nbytes for k in ("flux_sum", "L_tot", "value", "sigma") if k in out and not device_outputs)
        return {"counters": tot, "d2h_bytes": nbytes}

    def step(op, device_outputs):
        if streamed:
            return step_streamed(op, device_outputs)
        G.set_opacity(op)
        fn = G.run_albedo if mode == "albedo" else G.run_emission
        return fn(prm, device_outputs=device_outputs)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(op, device_outputs, steps):
        acc = {}
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        out = None
        for _ in range(steps):
            out = step(op, device_outputs)
            for k, v in out["counters"].items():
                acc[k] = acc.get(k, 0) + v
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        return ms, acc, out

    for _ in range(max(args.warmup, 3)):
        step(dev_opac, True)
    sampler = ClockSampler(local)
    sampler.start()
    ms, acc, out = timed(dev_opac, True, args.steps)
    clocks = sampler.summary()
    # e2e: host tables in, host spectra out
    step(host_opac, False)
    ms_e2e, acc_e2e, out_e2e = timed(host_opac, False, args.steps)
    d2h = out_e2e["d2h_bytes"] if streamed else sum(out_e2e[k].nbytes for k in ("flux_sum", "L_tot", "value", "sigma") if k in out_e2e)

    ms, (ev_all, seg_all) = reduce_over_ranks(ms, [acc["events"], acc["segments_transport"] + acc["segments_peel"]],
                                              world, "cuda")
    ms_e2e, (ev_all_e2e,) = reduce_over_ranks(ms_e2e, [acc_e2e["events"]], world, "cuda")
    value = ev_all / (ms * 1e-3)
    e2e_value = ev_all_e2e / (ms_e2e * 1e-3)

    if rank == 0:
        pk = peaks()
        is3d = np.asarray(grid["T"]).shape[0] > 1 or np.asarray(grid["T"]).shape[1] > 1
        i_seg = I_SEG_3D if is3d else I_SEG_1D
        # dominant kernel: peel_kernel, one launch per pass (the transport side of a pass is a sequence of smaller
        # kernels: launch-order sort, first flights, one interact kernel per generation, the persistent tail).
        # cudaEvents recorded by the library on the caller's stream around every launch give its device time.
        dom = "peel"
        work = acc["segments_peel"] * i_seg + acc["rays_peel"] * I_PEEL_RAY
        dur_ms = acc["ms_peel"]
        work_t = acc["segments_transport"] * i_seg + acc["events"] * I_EVENT
        n_dom = max(1, acc["passes"])
        peak = 148 * 128 * pk["sm_max_mhz"] * 1e6 / 1e12          # T lane-instr/s
        achieved = work / (dur_ms * 1e-3) / 1e12 if dur_ms > 0 else 0.0
        ncell = int(np.asarray(grid["T"]).size)
        hbm_bytes = n_chan * ncell * 4 * (len(tab_keys) + 1 + 4)   # tables read once + alpha/prop written once
        if streamed:   # Rayleigh table written once; 8 Doppler stagings (4 phases x 2 modes) each read it and write alpha + prop
            hbm_bytes = n_chan * ncell * (4 + 8 * (4 + 4 + 16))
        roofline = {"bound": "alu", "kernel": dom + "_kernel", "achieved": achieved, "peak": peak,
                    "unit": "Tlane-instr/s", "frac": achieved / peak if peak else None,
                    # dram__bytes_read + write per peel_kernel launch from one ncu --set full capture of the default
                    # workload (profiles/ncu_full_r01d_ptx_loops.txt); other workloads: not captured
                    "traffic": PEEL_DRAM_BYTES_PER_LAUNCH_CFG2 if (args.workload == "cfg2" and args.packets is None) else None,
                    "traffic_unit": "bytes per launch (94 M events: 64 B record + 4 B permutation entry + extinction gathers)",
                    "peak_source": "148 SM x 128 FP32 lanes x sm_max_mhz (%s)" % pk["source"],
                    "work_lane_instr_per_launch": work / n_dom, "ms_per_launch": dur_ms / n_dom,
                    "hbm_term": {"bytes_per_step": hbm_bytes, "ms_at_peak": hbm_bytes / (pk["hbm_gbs"] * 1e9) * 1e3 * 1.0,
                                 "peak_gbs": pk["hbm_gbs"]},
                    "kernel_ms_per_step": {k: acc[k] / args.steps for k in ("ms_stage", "ms_emission_cdf", "ms_transport", "ms_sort", "ms_peel")},
                    "transport_kernels": {"achieved": work_t / (acc["ms_transport"] * 1e-3) / 1e12 if acc["ms_transport"] > 0 else 0.0,
                                          "frac": work_t / (acc["ms_transport"] * 1e-3) / 1e12 / peak if acc["ms_transport"] > 0 else None,
                                          "note": "launch sort + first flights + interact generations + persistent tail, same units"},
                    "whole_step": {"achieved": (work + work_t) / (ms / args.steps * 1e-3 * args.steps) / 1e12,
                                   "frac": (work + work_t) / (ms * 1e-3) / 1e12 / peak}}
        # config 5 has no per-cell table for the oracle to read (328 GB at full size): no cpu_baseline leg there
        cpu = oracle_leg(args.workload, grid, dict(opac, chan0=0), prm, mode) if world == 1 and not args.no_cpu and not streamed else None
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": args.workload, "mode": mode, "n_chan_per_gpu": n_chan, "packets_per_channel": N,
                           "n_obs": int(np.asarray(prm["obs_dir"]).reshape(-1, 3).shape[0]),
                           "grid": list(np.asarray(grid["T"]).shape), "parallelism": "channels x %d" % world,
                           "l2": "opacity tables (%.0f MB) + staged tables exceed the 126 MB L2; no flush" % (h2d / 1e6)},
                "events_per_step": ev_all / args.steps, "segments_per_s": seg_all / (ms * 1e-3),
                "spectra_per_s": world * args.steps / (ms * 1e-3),
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                        "ms_per_step": ms_e2e / args.steps},
                "gpu_launches": int(acc["launches"]), "clocks": clocks, "roofline": roofline,
                "counters_per_step": {k: acc[k] / args.steps for k in
                                      ("events", "segments_transport", "segments_peel", "rays_peel", "packets_escaped",
                                       "packets_absorbed", "packets_surface", "packets_stuck", "passes")}}
        if cpu is not None:
            line["cpu_baseline"] = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}
        print(json.dumps(line), flush=True)
    G.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--channels", type=int, default=None, help="cfg4 / cfg5: number of wavelength points (default 10000 / 4096)")
    ap.add_argument("--batch", type=int, default=1024, help="cfg5: wavelength points per streamed opacity batch")
    ap.add_argument("--packets", type=int, default=None, help="override packets per channel (debugging only)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
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
