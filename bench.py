#!/usr/bin/env python
"""bench.py -- MLUPS / HBM roofline of the fused thermal two-component LB step on B200.

    python bench.py --gpus N --steps K --warmup W [--config 1..5] [--impl reference]

A "step" is one lattice-Boltzmann time step (rows a1-a9 of SURVEY.md section 8: fused
force+collide+stream kernel + boundary kernel) over the whole lattice of the workload.  Default
workload: BASELINE.json configs[3], the 4096x2048 headline config (4000 droplets r = 14, 4x4 posts
period 16 on both walls, thermal + buoyancy, fp64), synthetic seeded input.
N > 1 (torchrun): the lattice is split into N contiguous y-slabs, one process per GPU; per step and interior
face the 3 rows next to the face travel to the neighbour (NCCL point-to-point on a side stream, overlapped with
the interior rows).  Default: the SAME lattice split N ways ("scaling": "strong");
--scaling weak stacks N copies of the workload in y (ny = N * ny of the config).  value = all site updates over the
max-over-ranks device time.
"""
import hashlib
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

ALG_BYTES_PER_SITE = 432  # 27 fp64 populations read + 27 written
NOMINAL_HBM_GBS = 8000.0
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def kernel_source_hash():
    """sha256 of the sources that define the fused kernel (what a committed ncu capture is valid for)."""
    h = hashlib.sha256()
    for f in ("tlb_step.cu", "tlb_internal.cuh"):
        with open(os.path.join(ROOT, "paper_2109_12565_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def committed_traffic(name):
    """dram bytes per fused-kernel launch from the committed ncu --set full summary (profiles/traffic.json), or None
    when there is no capture for this workload or the kernel sources have changed since it was taken."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            e = json.load(f).get(name)
        if not isinstance(e, dict) or e.get("kernel_source_sha256") != kernel_source_hash():
            return None
        return e["dram_bytes_per_launch"]
    except Exception:
        return None


class ClockSampler(threading.Thread):
    """Samples the SM clock and the throttle reasons (NVML, else nvidia-smi) while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False
        self.nvml = None
        try:  # initialised here, outside the timed region
            import pynvml
            pynvml.nvmlInit()
            self.nvml = (pynvml, pynvml.nvmlDeviceGetHandleByIndex(index))
            pynvml.nvmlDeviceGetClockInfo(self.nvml[1], pynvml.NVML_CLOCK_SM)  # the first query of a kind takes milliseconds
            (getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or pynvml.nvmlDeviceGetCurrentClocksThrottleReasons)(self.nvml[1])
        except Exception:
            self.nvml = None  # no NVML binding: nvidia-smi at 10 Hz

    def _run_nvml(self):
        """NVML polled every millisecond: a 20-step region (13 ms) still gets a dozen samples."""
        pynvml, h = self.nvml
        mx = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
        get_reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
        bits = (0x8, 0x40, 0x20, 0x4)  # hw_slowdown, hw_thermal_slowdown, sw_thermal_slowdown, sw_power_cap
        while not self.stop_flag:
            r = get_reasons(h)
            self.rows.append([str(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)), str(mx)] +
                             ["Active" if r & b else "Not Active" for b in bits])
            time.sleep(0.001)

    def run(self):
        if self.nvml is not None:
            try:
                self._run_nvml()
                return
            except Exception:
                pass
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5)
                self.rows.append([c.strip() for c in out.stdout.strip().split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        self.stop_flag = True
        self.join(timeout=6)
        mhz = sorted(int(r[0]) for r in self.rows if len(r) >= 6 and r[0].isdigit())
        mx = [int(r[1]) for r in self.rows if len(r) >= 6 and r[1].isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) >= 6 and r[2 + k] == "Active" for r in self.rows)]
        return {"sm_mhz": mhz[len(mhz) // 2] if mhz else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(mhz)}


def time_oracle(cfg, solid, rA, rB, T, steps):
    """MLUPS of the oracle as it stands, single-threaded, on this host."""
    from oracle import tlb_oracle
    tlb_oracle.build()
    o = tlb_oracle.Oracle(cfg["nx"], cfg["ny"], **cfg["params"])
    o.set_solid(solid)
    o.set_fields(rA, rB, T)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    return cfg["nx"] * cfg["ny"] * steps / dt / 1e6, dt


def slab_of(cfg, rows):
    """A full-width slab of `rows` rows of the workload (walls, posts, droplets, same physics)."""
    import inputs
    if rows >= cfg["ny"]:
        return cfg, inputs.make_config_inputs(cfg)
    c = dict(cfg, ny=rows)
    dens = cfg["init"]["n_droplets"] / float(cfg["nx"] * cfg["ny"])
    c["init"] = dict(cfg["init"], n_droplets=max(0, int(dens * cfg["nx"] * rows * 0.8)))
    try:
        return c, inputs.make_config_inputs(c)
    except ValueError:
        c["init"] = dict(cfg["init"], n_droplets=0)
        return c, inputs.make_config_inputs(c)


def run_reference(args, rank):
    """--impl reference: the oracle itself (this tier has no reference implementation), timed on the
    host cores, each step a bounded slab of the workload sized so the run ends within minutes."""
    if rank != 0:
        return
    import inputs
    cfg = inputs.config(args.config)
    budget_sites = 90e6  # about 90 s at ~1 MLUPS
    rows = int(budget_sites / max(1, args.steps + args.warmup) / cfg["nx"])
    rows = max(2 * cfg["posts"][1] + 8, min(cfg["ny"], rows))
    c, (solid, rA, rB, T) = slab_of(cfg, rows)
    from oracle import tlb_oracle
    tlb_oracle.build()
    o = tlb_oracle.Oracle(c["nx"], c["ny"], **c["params"])
    o.set_solid(solid)
    o.set_fields(rA, rB, T)
    o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    mlups = c["nx"] * c["ny"] * args.steps / dt / 1e6
    sample = "%dx%d full-width slab of %s per step (walls, posts, droplets kept)" % (c["nx"], c["ny"], cfg["name"])
    print(json.dumps({
        "impl": "reference", "metric": "MLUPS", "value": mlups, "unit": "MLUPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
        "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "sample": sample},
        "cpu_baseline": {"value": mlups, "unit": "MLUPS", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": mlups, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_ours(args, rank, world):
    import torch
    import torch.distributed as dist
    from paper_2109_12565_b200 import binding, replicas
    import inputs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    binding.load_library()  # raises if libtlb.so is missing
    if world > 1 or args.force_slabs:
        return run_slabs(args, rank, world, local)
    cfg = inputs.config(args.config)
    nx, ny = cfg["nx"], cfg["ny"]
    sites = nx * ny
    alg_bytes = ALG_BYTES_PER_SITE * args.pop_precision // 64  # 432 B (fp64 storage) or 216 B (fp32 storage)
    t = binding.TLB(nx, ny, params=binding.params_from_config(cfg), device=dev, pop_precision=args.pop_precision)
    t.init(cfg["seed"])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: K steps, CUDA events on the launch stream, max over ranks
    t.step(max(3, args.warmup))
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = t.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(t.stream)
    t.step(args.steps)
    e1.record(t.stream)
    barrier()
    launches = t.launch_count() - l0
    ms = e0.elapsed_time(e1)
    clocks = sampler.summary()
    mlups, ms = replicas.aggregate_mlups(sites, args.steps, ms, dev)  # all ranks' updates / max-over-ranks time

    # ---- roofline of the dominant (fused) kernel.  Its average launch duration inside the timed region
    # is the step time (CUDA events around the K back-to-back steps above) minus the boundary kernel's
    # duration (events around 200 back-to-back launches of it); recording events around every launch of
    # the real sequence serialises the front end and inflates both.  `kernel_ms_isolated` is the fused
    # kernel launched 50 times on the same buffers: no part of its input is left in L2 by a previous step.
    iso_ms, boundary_ms = t.profile_step(50)
    _, boundary_ms = t.profile_step(200)
    step_ms = ms / args.steps
    fused_ms = step_ms - boundary_ms
    peak, peak_src = measured_peak()
    achieved = alg_bytes * sites / fused_ms / 1e6  # GB/s
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": committed_traffic(cfg["name"]) if args.pop_precision == 64 else None, "peak_source": peak_src, "kernel": "tlb::fused_kernel<0, false, %s, %s>" % ("double" if args.pop_precision == 64 else "float", "true" if cfg["params"]["tau"] == 1.0 else "false"),
                "kernel_ms": fused_ms, "kernel_ms_isolated": iso_ms, "boundary_kernel_ms": boundary_ms,
                "method": "kernel_ms = ms_per_step - boundary_kernel_ms (CUDA events on the launch stream)",
                "alg_bytes_per_launch": alg_bytes * sites, "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                "kernel_share_of_step": fused_ms / step_ms}
    ob = t.observables()
    finite = all(v == v and abs(v) != float("inf") for v in ob.values())
    u = t.fields()[2]
    umax = float((u[0] * u[0] + u[1] * u[1]).max().sqrt())  # print max |u^(H)| of every run
    del u

    # ---- optional: cost of the droplet analysis (section 2.4, first stage) in LB steps; the paper quotes "roughly two LB
    # time steps" for its whole Delaunay procedure (L218)
    droplets = None
    if args.droplets < 0:  # default: threshold half way between the two bulk densities of the input recipe
        args.droplets = 0.5 * (cfg["init"]["rho_in"] + cfg["init"]["rho_out"]) if cfg["init"]["n_droplets"] > 0 else 0.0
    if args.droplets > 0:
        import ctypes
        cap = max(1, min(sites // 4, 8 * max(1, cfg["init"]["n_droplets"])))
        lab = torch.empty((ny, nx), dtype=torch.int32, device=dev)
        nd = torch.zeros(1, dtype=torch.int32, device=dev)
        st = torch.zeros((cap, 4), dtype=torch.float64, device=dev)
        call = lambda: t.lib.tlb_droplets(t.h, ctypes.c_double(args.droplets), lab.data_ptr(), cap, nd.data_ptr(), st.data_ptr())
        assert call() == 0
        torch.cuda.synchronize()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(t.stream)
        for _ in range(20):
            call()
        d1.record(t.stream)
        torch.cuda.synchronize()
        dms = d0.elapsed_time(d1) / 20
        k = int(nd.item())
        droplets = {"B_th": args.droplets, "n_droplets": k, "ms": dms, "lb_steps": dms / step_ms,
                    "sites_min": float(st[:min(k, cap), 1].min()) if k else None,
                    "sites_max": float(st[:min(k, cap), 1].max()) if k else None,
                    "call": "tlb_droplets (rho_A from the first fluid's 9 planes, threshold + run labels, union-find on the remaining bonds, flatten, statistics)"}
        # second stage (R23-R26): digital Voronoi colouring of the centres, Delaunay links, droplet Nusselt numbers
        kk = min(k, cap)
        if kk > 0:
            cen = st[:kk, 2:4].contiguous()
            col = torch.empty((ny, nx), dtype=torch.int32, device=dev)
            nl = torch.zeros(1, dtype=torch.int32, device=dev)
            lk = torch.zeros((16 * kk, 2), dtype=torch.int32, device=dev)
            nu = torch.zeros(kk, dtype=torch.float64, device=dev)

            def stage2():
                assert t.lib.tlb_voronoi(t.h, cen.data_ptr(), kk, col.data_ptr()) == 0
                assert t.lib.tlb_delaunay(t.h, col.data_ptr(), kk, 16 * kk, nl.data_ptr(), lk.data_ptr()) == 0
                assert t.lib.tlb_droplet_nusselt(t.h, cen.data_ptr(), kk, nu.data_ptr()) == 0
            stage2()
            torch.cuda.synchronize()
            d0.record(t.stream)
            for _ in range(20):
                stage2()
            d1.record(t.stream)
            torch.cuda.synchronize()
            s2 = d0.elapsed_time(d1) / 20
            droplets.update({"stage2_ms": s2, "stage2_lb_steps": s2 / step_ms, "n_links": int(nl.item()),
                             "whole_analysis_lb_steps": (dms + s2) / step_ms,
                             "stage2_call": "tlb_voronoi + tlb_delaunay + tlb_droplet_nusselt on the centres of tlb_droplets"})
            del cen, col, nl, lk, nu
        del lab, nd, st

    # ---- the config's own step count (BASELINE config 4: "2000 steps timed"): seconds of back-to-back steps put the GPU
    # under its power cap, the regime a 1e5-1e6-step run (Table A.3) lives in; the K-step region above is a burst when
    # K is small.  Timed the same way, clocks sampled during it.
    sustained = None
    long_steps = min(int(cfg["steps"]), 5000)
    if args.steps < long_steps and not args.no_sustained:
        sampler2 = ClockSampler(local)
        sampler2.start()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(t.stream)
        t.step(long_steps)
        s1.record(t.stream)
        barrier()
        sms = s0.elapsed_time(s1) / long_steps
        sustained = {"steps": long_steps, "ms_per_step": sms, "value": sites / sms / 1e3, "unit": "MLUPS", "gpu_launches": 2 * long_steps,
                     "frac": alg_bytes * sites / (sms - boundary_ms) / 1e6 / peak, "clocks": sampler2.summary()}
    elif args.steps >= long_steps:
        sustained = {"steps": args.steps, "ms_per_step": step_ms, "value": mlups, "unit": "MLUPS", "frac": achieved / peak,
                     "clocks": clocks, "note": "the timed region itself"}
    roofline["sustained"] = sustained  # (timed after the droplet analysis above, which wants the state the K steps left)

    # ---- optional long run with the observables logged (BASELINE config 2: Nu and mass every 1000 steps)
    obs_log = None
    if args.observe_every > 0:
        t.init(cfg["seed"])
        m0 = t.observables()
        obs_log = []
        for k in range(args.observe_every, cfg["steps"] + 1, args.observe_every):
            t.step(args.observe_every)
            o = t.observables()
            uu = t.fields()[2]
            obs_log.append({"step": k, "Nu": o["Nu"], "mass_A": o["mass_A"], "mass_B": o["mass_B"], "E": o["E"],
                            "mass_A_drift": o["mass_A"] / m0["mass_A"] - 1, "mass_B_drift": o["mass_B"] / m0["mass_B"] - 1,
                            "max_uH": float((uu[0] * uu[0] + uu[1] * uu[1]).max().sqrt())})
            print("step %6d  Nu %.9f  mass_A %.12e (%+.2e)  mass_B %.12e (%+.2e)  max|uH| %.4e"
                  % (k, o["Nu"], o["mass_A"], obs_log[-1]["mass_A_drift"], o["mass_B"], obs_log[-1]["mass_B_drift"],
                     obs_log[-1]["max_uH"]), file=sys.stderr)

    # ---- end to end through the host-buffer ABI: per step H2D of the three input fields from pinned
    # memory, one LB step, D2H of the four observables
    solid_h = torch.zeros((ny, nx), dtype=torch.uint8)
    fa, fb, ft = (torch.empty((ny, nx), dtype=torch.float64).pin_memory() for _ in range(3))
    t.fields_host(fa, fb, None, ft)
    e2e_steps = max(3, min(args.steps, 20))
    for _ in range(2):
        t.set_fields_host(fa, fb, ft); t.step(1); t.observables()
    barrier()
    w0 = time.perf_counter()
    for _ in range(e2e_steps):
        t.set_fields_host(fa, fb, ft)
        t.step(1)
        t.observables()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - w0) * 1e3
    e2e_mlups, e2e_ms = replicas.aggregate_mlups(sites, e2e_steps, e2e_ms, dev)
    e2e_observables = {"value": e2e_mlups, "unit": "MLUPS", "h2d_bytes_per_step": 3 * 8 * sites,
                       "d2h_bytes_per_step": 32, "steps": e2e_steps,
                       "call": "tlb_set_fields_host + tlb_step(1) + tlb_observables_host per step"}
    del solid_h
    # the same with the step's full result read back: tlb_fields_host(rho_A, rho_B, u, T), 5 planes
    ha, hb, ht = (torch.empty((ny, nx), dtype=torch.float64).pin_memory() for _ in range(3))
    hu = torch.empty((2, ny, nx), dtype=torch.float64).pin_memory()
    for _ in range(2):
        t.set_fields_host(fa, fb, ft); t.step(1); t.fields_host(ha, hb, hu, ht)
    barrier()
    w0 = time.perf_counter()
    for _ in range(e2e_steps):
        t.set_fields_host(fa, fb, ft)
        t.step(1)
        t.fields_host(ha, hb, hu, ht)
    torch.cuda.synchronize()
    e2f_ms = (time.perf_counter() - w0) * 1e3
    # the headline end-to-end figure is the loop that returns the step's result, the five field planes
    e2e = {"value": sites * e2e_steps / e2f_ms / 1e3, "unit": "MLUPS", "h2d_bytes_per_step": 3 * 8 * sites,
           "d2h_bytes_per_step": 5 * 8 * sites, "steps": e2e_steps,
           "call": "tlb_set_fields_host + tlb_step(1) + tlb_fields_host(rho_A, rho_B, u, T) per step; every step starts "
                   "from the rest equilibrium of the fields it was given"}
    del ha, hb, ht, hu

    # ---- CPU baseline: the oracle as it stands on this host, rank 0 at N = 1 only
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        rows = min(ny, max(64, int(20e6 / nx / 2)))
        c, (solid, rA, rB, T) = slab_of(cfg, rows)
        v, dt = time_oracle(c, solid, rA, rB, T, 2)
        cpu = {"value": v, "unit": "MLUPS", "cores": 1, "kind": "oracle", "seconds": dt,
               "sample": "2 steps of a %dx%d full-width slab of %s (host has %d cores; the oracle is single-threaded)"
                         % (c["nx"], c["ny"], cfg["name"], os.cpu_count())}

    if rank == 0:
        print(json.dumps({
            "metric": "MLUPS", "value": mlups, "unit": "MLUPS", "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "nx": nx, "ny": ny, "droplets": cfg["init"]["n_droplets"],
                       "posts": list(cfg["posts"]), "state_bytes": alg_bytes // 2 * sites, "pop_precision": args.pop_precision,
                       "l2": "state (%.2f GB per buffer) exceeds the 126 MB L2; no flush needed" % (216 * sites / 1e9)
                       if 216 * sites > 4 * 126e6 else "state fits in L2: HBM figures are not meaningful",
                       "parallelism": "1 GPU, whole lattice", "finite": finite, "mass_A": ob["mass_A"], "Nu": ob["Nu"],
                       "max_uH": umax},
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "e2e_observables": e2e_observables, "observables_log": obs_log, "droplet_analysis": droplets,
            "gpu_launches": launches, "clocks": clocks,
            "effective_GBs": alg_bytes * mlups / 1e3, "roofline_frac_whole_step": alg_bytes * mlups / 1e3 / peak / world}))


def run_slabs(args, rank, world, local):
    """N > 1: y-slab decomposition, one process per GPU."""
    import torch
    import torch.distributed as dist
    from paper_2109_12565_b200 import binding, replicas, slabs
    import inputs

    dev = "cuda:%d" % local
    dist.init_process_group("nccl", device_id=torch.device(dev))
    cfg = inputs.config(args.config)
    nx = cfg["nx"]
    ny = cfg["ny"] * (world if args.scaling == "weak" else 1)
    par = binding.params_from_config(cfg)
    if args.scaling == "weak":
        par.n_droplets = cfg["init"]["n_droplets"] * world  # the same emulsion, N times as tall
    alg_bytes = ALG_BYTES_PER_SITE * args.pop_precision // 64
    s = slabs.DistributedSlab(nx, ny, params=par, device=dev, pop_precision=args.pop_precision)
    s.init(cfg["seed"])
    own_sites = nx * (s.y1 - s.y0)

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    s.step(max(3, args.warmup))
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = s.t.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s.t.stream)
    s.step(args.steps)
    e1.record(s.t.stream)
    barrier()
    launches = s.t.launch_count() - l0
    ms = e0.elapsed_time(e1)
    clocks = sampler.summary()
    mlups, ms = replicas.aggregate_mlups(own_sites, args.steps, ms, dev)  # all slabs' updates / max-over-ranks time
    launches = int(replicas.sum_over_ranks(launches, dev))
    ob = s.observables()
    finite = all(v == v and abs(v) != float("inf") for v in ob.values())
    peak, peak_src = measured_peak()
    step_ms = ms / args.steps
    achieved = alg_bytes * own_sites / step_ms / 1e6  # this rank's bytes over the slowest rank's step: a lower bound
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                "peak_source": peak_src, "kernel": "tlb::fused_kernel<0, false, %s, %s>" % ("double" if args.pop_precision == 64 else "float", "true" if cfg["params"]["tau"] == 1.0 else "false"),
                "kernel_ms": step_ms, "method": "per GPU: own rows x alg. bytes / whole step time (edges + interior + halo "
                "exchange + boundary kernel), max over ranks", "alg_bytes_per_launch": alg_bytes * own_sites}

    # ---- end to end: per step H2D of this slab's three input fields, one step with its halo exchange, the observables
    # all-reduced and read back
    nyl = s.t.ny
    fa, fb, ft = (torch.empty((nyl, nx), dtype=torch.float64).pin_memory() for _ in range(3))
    s.t.fields_host(fa, fb, None, ft)
    e2e_steps = max(3, min(args.steps, 20))
    # tlb_fields_host writes the owned rows only; a slab's state-setting calls take the halo rows from the caller's
    # arrays: repeat the nearest owned row there
    for h in (fa, fb, ft):
        h[:s.t.own0] = h[s.t.own0]
        h[s.t.own1:] = h[s.t.own1 - 1]
    for _ in range(2):
        s.t.set_fields_host(fa, fb, ft); s.step(1); s.observables()
    barrier()
    w0 = time.perf_counter()
    for _ in range(e2e_steps):
        s.t.set_fields_host(fa, fb, ft)
        s.step(1)
        s.observables()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - w0) * 1e3
    e2e_mlups, _ = replicas.aggregate_mlups(own_sites, e2e_steps, e2e_ms, dev)
    e2e = {"value": e2e_mlups, "unit": "MLUPS", "h2d_bytes_per_step": int(replicas.sum_over_ranks(3 * 8 * nx * nyl, dev)),
           "d2h_bytes_per_step": 32 * world, "steps": e2e_steps,
           "call": "per rank: tlb_set_fields_host + slab step (edges, interior, NCCL exchange straight out of / into the population buffers, finish) + "
                   "tlb_observable_sums, all-reduce, tlb_observables_from_sums"}
    if rank == 0:
        print(json.dumps({
            "metric": "MLUPS", "value": mlups, "unit": "MLUPS", "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": step_ms, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"] + ("" if args.scaling == "strong" else "_x%d_in_y" % world), "nx": nx, "ny": ny,
                       "posts": list(cfg["posts"]), "pop_precision": args.pop_precision,
                       "parallelism": "%d y-slabs, halo exchange of 3 rows x 27 planes per face and step (NCCL p2p)" % world,
                       "l2": "state exceeds L2; no flush needed" if 216 * own_sites > 4 * 126e6 else
                             "a slab's state fits in L2: HBM figures are not meaningful",
                       "finite": finite, "mass_A": ob["mass_A"], "Nu": ob["Nu"]},
            "roofline": roofline, "cpu_baseline": None, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
            "effective_GBs": alg_bytes * mlups / 1e3, "roofline_frac_whole_step": alg_bytes * mlups / 1e3 / peak / world}))
    dist.destroy_process_group()


def relaunch_under_torchrun(n):
    """`python bench.py --gpus N` without torchrun: start the N ranks here (one process per GPU, 127.0.0.1 rendezvous)
    instead of silently measuring one GPU.  Refuses, with a non-zero exit, when the node has fewer than N GPUs."""
    import socket
    if "--impl" in sys.argv and "reference" in sys.argv:
        have = n  # the oracle arm runs on the host cores of rank 0; no GPU needed
    else:
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < n:
        raise SystemExit("bench.py: --gpus %d asked for, %d CUDA device(s) visible; not running (a line with n_gpus < %d "
                         "would misreport the scaling run)" % (n, have, n))
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n), "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.environ.setdefault("NCCL_DEBUG", "WARN")
    sys.stdout.flush()
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--scaling", default="strong", choices=["strong", "weak"],
                    help="N > 1: split the config's lattice into N y-slabs (strong) or stack N copies of it in y (weak)")
    ap.add_argument("--droplets", type=float, default=-1.0,
                    help="B_th > 0: also time the droplet analysis (threshold B_th on rho_A) on the final state and report it in LB "
                         "steps; < 0 (default): B_th = (rho_in + rho_out) / 2 of the config; 0: skip")
    ap.add_argument("--no-sustained", action="store_true",
                    help="skip the extra leg that times the config's own step count when --steps is smaller")
    ap.add_argument("--observe-every", type=int, default=0,
                    help="also run the config's full step count from its initial state, logging Nu / mass / max|uH| every so many steps")
    ap.add_argument("--force-slabs", action="store_true",
                    help="run the y-slab driver of N > 1 even with one rank (one slab, walls on both faces): a check of that code path")
    ap.add_argument("--pop-precision", type=int, default=64, choices=[64, 32],
                    help="storage of the populations in HBM (32: bandwidth study of BASELINE config 5; arithmetic stays fp64)")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_under_torchrun(args.gpus)  # does not return
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d; launch with --nproc-per-node %d (or let bench.py "
                         "start the ranks itself: run it without torchrun)" % (args.gpus, world, args.gpus))
    if args.impl == "reference":
        run_reference(args, rank)
    else:
        run_ours(args, rank, world)


if __name__ == "__main__":
    main()
