#!/usr/bin/env python
"""Benchmark of the fused two-component TSLB step (BASELINE.json metric: GLUPS of the fused
flow + phase-field step and achieved HBM GB/s against the B200 peak).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c5|c4|c3] [--impl reference]

A "step" is one pass of the whole hot path over the full lattice.
N = 1 runs BASELINE.json configs[4] ("c5": 512x512x1536 fp32 jet, 402 653 184 nodes), the
configuration the metric is quoted on.  N > 1 (torchrun) runs N independent replicas of the same
workload, one per GPU ("replicas only", the default, weak scaling), or with --decomp slabs ONE domain
split into z-slabs whose step kernels push their halo planes into the neighbours' ghost planes
(strong scaling).  The timed region (exactly K steps between CUDA events on the library's
stream) is repeated --reps times; `value` is the median, `reps` lists every repetition.
Prints ONE JSON line (rank 0).
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
sys.path.insert(0, ROOT)

BYTES_PER_NODE = {("f32", True): 88, ("f64", True): 176, ("f32", False): 80, ("f64", False): 160}

CONFIGS = {
    # name: (nx, ny, nz, D, description)
    "c5": (512, 512, 1536, 40, "BASELINE configs[4]: large jet 512x512x1536 fp32, D=40, U=0.05, Re=5000, We=2000"),
    "c4": (256, 256, 512, 20, "BASELINE configs[3]: jet 256x256x512 fp32, D=20, U=0.05, Re=5000, We=200"),
    "t1": (400, 400, 800, 40, "PAPER.md:237-245 Table 1 row 5 / the shape the paper's GLUPS are quoted on: jet 400x400x800 fp32, "
                              "D=40, U=0.05, Re=5000, We=2000 (ragged 12.5 x 50 tiles)"),
    "c3": (128, 128, 128, 0, "BASELINE configs[2]: 128^3 periodic droplets + noise fp32"),
}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", default=os.environ.get("TSLB_BENCH_CONFIG", "c5"))
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--precision", default="f32")
    ap.add_argument("--kernel", default="auto")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slabs"],
                    help="N > 1: independent replicas (default, weak scaling) or ONE domain split into z-slabs "
                         "(strong scaling, halo push fused into the step kernel; DESIGN.md §8)")
    ap.add_argument("--slabs", type=int, default=0, help="with --decomp slabs on one GPU: number of in-process slabs")
    ap.add_argument("--forcing", default="kick", choices=["kick", "guo"],
                    help="how the surface-tension force enters (include/tslb.h): the kick of reading A9 (default, all "
                         "kernels) or the Guo-type forcing of reading A18 (generic kernel only; its cost is a bench line "
                         "of its own, not the headline)")
    ap.add_argument("--reps", type=int, default=3, help="repetitions of the timed region of K steps (value = median)")
    ap.add_argument("--sample", default="slab", help="(--impl cpu-sample) oracle sample: slab | c3 | c4slab")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    return ap.parse_args()


# ------------------------------------------------------------------ synthetic state (device)
def developed_jet_device(torch, nx, ny, nz, D, U, dtype, device, seed=99, ndrop=200, W=4.0):
    """Seeded synthetic 'developed jet' state built on the GPU (input generation only, none of the
    method's arithmetic): axial velocity with the self-similar profile shape of PAPER.md:271, a phi
    core of diameter D over the first third of z and seeded droplets in a cone downstream
    (same recipe as inputs.jet_developed)."""
    g = torch.Generator(device="cpu").manual_seed(seed)
    x1 = torch.arange(nx, device=device, dtype=dtype) - (nx - 1) / 2.0
    y1 = torch.arange(ny, device=device, dtype=dtype) - (ny - 1) / 2.0
    z1 = torch.arange(nz, device=device, dtype=dtype)
    r2 = (y1[:, None] ** 2 + x1[None, :] ** 2)[None]                      # (1, ny, nx)
    z0 = 6.0 * D
    uz = torch.empty((nz, ny, nx), dtype=dtype, device=device)
    phi = torch.zeros((nz, ny, nx), dtype=dtype, device=device)
    zs = 64
    for a in range(0, nz, zs):
        b = min(a + zs, nz)
        zz = z1[a:b, None, None]
        uz[a:b] = U * torch.exp(-75.0 * r2 / (zz + z0) ** 2)
        core = 0.5 * (1.0 - torch.tanh(2.0 * (torch.sqrt(r2) - D / 2.0) / W))
        phi[a:b] = core * (zz < nz / 3.0)
    rnd = torch.rand((ndrop, 4), generator=g).numpy()
    nrm = torch.randn((ndrop, 2), generator=g).numpy()
    for k in range(ndrop):
        cz = nz / 3.0 + rnd[k, 0] * max(1.0, nz - 8.0 - nz / 3.0)
        spread = 0.1 * (cz + z0)
        cx, cy = nrm[k, 0] * spread, nrm[k, 1] * spread
        rad = 3.0 + rnd[k, 1] * 0.2 * D
        lo, hi = int(max(cz - rad - 6, 0)), int(min(cz + rad + 7, nz))
        ylo, yhi = int(max(cy - rad - 6 + (ny - 1) / 2.0, 0)), int(min(cy + rad + 7 + (ny - 1) / 2.0, ny))
        xlo, xhi = int(max(cx - rad - 6 + (nx - 1) / 2.0, 0)), int(min(cx + rad + 7 + (nx - 1) / 2.0, nx))
        if hi <= lo or yhi <= ylo or xhi <= xlo:
            continue
        d = torch.sqrt((z1[lo:hi, None, None] - cz) ** 2 + (y1[None, ylo:yhi, None] - cy) ** 2
                       + (x1[None, None, xlo:xhi] - cx) ** 2)
        sub = phi[lo:hi, ylo:yhi, xlo:xhi]
        torch.maximum(sub, 0.5 * (1.0 - torch.tanh(2.0 * (d - rad) / W)), out=sub)
    rho = torch.ones((nz, ny, nx), dtype=dtype, device=device)
    zero = torch.zeros((nz, ny, nx), dtype=dtype, device=device)
    return dict(rho=rho, ux=zero, uy=zero.clone(), uz=uz, phi=phi)


def droplets_device(torch, inputs, n, dtype, device):
    d = inputs.droplets_noise(n, seed=12345, ndrop=40)
    return {k: torch.tensor(np.asarray(v, dtype=np.float32 if dtype == torch.float32 else np.float64), device=device)
            for k, v in d.items() if v is not None}


# ------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return None
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.rows:
            if ts < t0 or ts > t1 + 0.2:
                continue
            p = [q.strip() for q in line.split(",")]
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except Exception:
                continue
            for nme, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        if not sm:
            return None
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "samples": len(sm),
                "reasons": sorted(reasons)}


# ------------------------------------------------------------------ CPU oracle legs
def oracle_sample(cfg_name, steps, sample="slab"):
    """Time the oracle, as it stands, on a bounded sample of the workload.
    sample: "slab" = the first 16 planes of the bench configuration (64^3 sub-box for c3); "c3" = BASELINE
    configs[2] in full (128^3 droplets + noise); "c4slab" = the first 128 planes of configs[3] (256x256x512 jet).
    -> (GLUPS, threads, description, seconds per step)"""
    from oracle import ref
    from paper_2403_15773_b200 import inputs
    nx, ny, nz, D, _ = CONFIGS[cfg_name]
    if sample == "c3" or (sample == "slab" and cfg_name == "c3"):
        n = 128 if sample == "c3" else 64
        d = inputs.droplets_noise(n, seed=12345, ndrop=40 if n == 128 else 5)
        o = ref.Oracle(n, n, n, 1.95, two_component=True, sigma=0.005, interface_width=4.0)
        desc = ("C3 in full: 128^3 periodic, 40 droplets + noise, %d steps" % steps) if n == 128 else \
               ("64^3 sub-box of the C3 recipe (5 droplets + noise), %d steps" % steps)
        nodes = n ** 3
    else:
        if sample == "c4slab":
            cfg_name = "c4"
            nx, ny, nz, D, _ = CONFIGS["c4"]
            sz = 128
        else:
            sz = 16
        prm = inputs.jet_params(nx, ny, sz, D, We=200.0 if cfg_name == "c4" else 2000.0)
        d = inputs.jet_developed(nx, ny, sz, D, ndrop=4)
        o = ref.Oracle(nx, ny, sz, prm["omega"], two_component=True, sigma=prm["sigma"], interface_width=4.0,
                       bc_zlo=ref.BC_JET_INFLOW, bc_zhi=ref.BC_OUTFLOW, jet_diameter=prm["jet_diameter"],
                       jet_velocity=prm["jet_velocity"], jet_perturbation=prm["jet_perturbation"], seed=prm["seed"])
        desc = "%dx%dx%d slab (first %d planes of the %s jet, inflow/outflow), %d steps" % (nx, ny, sz, sz, cfg_name, steps)
        nodes = nx * ny * sz
    o.init_fields(d["rho"], d["ux"], d["uy"], d["uz"], d["phi"])
    o.step(1)                                   # page in
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    o.close()
    return nodes * steps / dt / 1e9, ref.num_threads(), desc, dt / steps


def cpu_sample_subprocess(cfg_name, steps, sample, threads):
    """The same in a child process with OMP_NUM_THREADS fixed (OpenMP reads it once per process).
    threads = 0: all cores.  -> dict or None"""
    env = dict(os.environ)
    if threads:
        env["OMP_NUM_THREADS"] = str(threads)
    else:
        env.pop("OMP_NUM_THREADS", None)
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        env.pop(k, None)
    try:
        r = subprocess.run([sys.executable, os.path.abspath(__file__), "--impl", "cpu-sample", "--config", cfg_name,
                            "--steps", str(steps), "--sample", sample], env=env, capture_output=True, text=True, timeout=600)
        return json.loads(r.stdout.strip().splitlines()[-1])
    except Exception as ex:      # the baseline is a report, not a gate
        return {"error": repr(ex)[:200], "sample": sample, "threads": threads}


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    nx, ny, nz, D, desc = CONFIGS[args.config]
    # each "step" of this arm is one oracle time step on the bounded slab; at most 4 are run (a step takes
    # seconds), after one untimed step that pages the state in -- the line reports what ran
    steps = max(1, min(args.steps, 4))
    glups, threads, sample, sps = oracle_sample(args.config, steps)
    out = {"impl": "reference", "metric": "GLUPS (fused flow+phase-field step)", "value": glups, "unit": "GLUPS",
           "n_gpus": args.gpus, "steps": steps, "warmup": 1, "requested": {"steps": args.steps, "warmup": args.warmup},
           "ms_per_step": sps * 1e3,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": desc, "grid": [nx, ny, nz]},
           "cpu_baseline": {"value": glups, "unit": "GLUPS", "cores": threads, "kind": "oracle", "sample": sample,
                            "cpu_model": cpu_model()},
           "e2e": {"value": glups, "unit": "GLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


# ------------------------------------------------------------------ z-slab mode (optional)
def run_slabs(args):
    """ONE domain split along z: one slab per rank (slabs.RankSlab, CUDA IPC + a one-element NCCL
    all-reduce per step as the barrier), or --slabs K in-process slabs on a single GPU
    (slabs.LocalSlabs) to measure what the decomposition itself costs.  Strong scaling."""
    import torch
    import torch.distributed as dist
    from paper_2403_15773_b200 import build, inputs, slabs, tslb
    from paper_2403_15773_b200 import dist as tdist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    build.build()
    nx, ny, nz, D, desc = CONFIGS[args.config]
    prec = tslb.F32 if args.precision == "f32" else tslb.F64
    tdt = torch.float32 if prec == tslb.F32 else torch.float64
    if args.config == "c3":
        kw = dict(two_component=True, sigma=0.005, interface_width=4.0)
        omega = 1.95
        state = droplets_device(torch, inputs, nx, tdt, dev)
    else:
        prm = inputs.jet_params(nx, ny, nz, D, We=200.0 if args.config == "c4" else 2000.0)
        omega = prm["omega"]
        kw = {k: v for k, v in prm.items() if k not in ("nx", "ny", "nz", "omega")}
        state = developed_jet_device(torch, nx, ny, nz, D, prm["jet_velocity"], tdt, dev)
    names = ("rho", "ux", "uy", "uz", "phi")
    if world > 1:
        run = slabs.RankSlab(nx, ny, nz, omega, precision=prec, device=local, **kw)
        run.init_fields(*[state[k][run.z0:run.z1].contiguous() for k in names])
        nslabs, sims = world, [run.sim]
    else:
        nslabs = max(1, args.slabs)
        run = slabs.LocalSlabs(nx, ny, nz, omega, nslabs, precision=prec, devices=[local] * nslabs, **kw)
        run.init_fields(*[state[k] for k in names])
        sims = run.sims
    del state
    torch.cuda.empty_cache()

    def barrier():
        torch.cuda.synchronize()
        tdist.barrier()
        torch.cuda.synchronize()

    run.step(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    l0 = sum(s.launch_count for s in sims)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record()
    run.step(args.steps)
    e1.record()
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    ms = tdist.max_over_ranks(e0.elapsed_time(e1), dev)
    launches = sum(s.launch_count for s in sims) - l0
    nodes = nx * ny * nz
    glups = nodes * args.steps / (ms * 1e-3) / 1e9          # one domain: all ranks' nodes / slowest rank's time
    kname = sims[0].kernel_name
    run.close()
    if rank == 0:
        peak = 6650.0
        pth = os.path.join(ROOT, "MEASURED_PEAKS.json")
        if os.path.exists(pth):
            peak = float(json.load(open(pth))["hbm_gbs"])
        bpn = BYTES_PER_NODE[(args.precision, True)]
        ach = bpn * nodes / world / (ms / args.steps * 1e-3) / 1e9     # per GPU
        print(json.dumps({
            "metric": "GLUPS (fused flow+phase-field step)", "value": glups, "unit": "GLUPS", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
            "config": {"workload": desc, "grid": [nx, ny, nz], "parallelism": "z-slabs x%d (%s)" % (
                nslabs, "one per rank, CUDA IPC peer stores" if world > 1 else "in-process on one GPU"),
                "l2": "state far exceeds the 126 MB L2; no flush needed"},
            "roofline": {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                         "traffic": None, "kernel": kname, "bytes_per_node_update": bpn, "nodes_per_launch": nodes // nslabs},
            "cpu_baseline": None, "e2e": None, "gpu_launches": int(launches), "clocks": clocks}))
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------ our arm
def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.impl == "cpu-sample":            # child of the cpu_baseline leg (fixed OMP_NUM_THREADS)
        g, threads, sample, sps = oracle_sample(args.config, max(1, args.steps), args.sample)
        print(json.dumps({"value": g, "unit": "GLUPS", "cores": threads, "sample": sample, "s_per_step": sps}))
        return
    if args.decomp == "slabs":
        run_slabs(args)
        return
    import torch
    import torch.distributed as dist
    from paper_2403_15773_b200 import build, inputs, tslb
    from paper_2403_15773_b200 import dist as tdist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    build.build()

    nx, ny, nz, D, desc = CONFIGS[args.config]
    prec = tslb.F32 if args.precision == "f32" else tslb.F64
    tdt = torch.float32 if prec == tslb.F32 else torch.float64
    kern = {"auto": tslb.KERNEL_AUTO, "generic": tslb.KERNEL_GENERIC, "tiled": tslb.KERNEL_TILED}[args.kernel]
    if args.config == "c3":
        kw = dict(two_component=True, sigma=0.005, interface_width=4.0)
        omega = 1.95
        state = droplets_device(torch, inputs, nx, tdt, dev)
    else:
        prm = inputs.jet_params(nx, ny, nz, D, We=200.0 if args.config == "c4" else 2000.0)
        omega = prm["omega"]
        kw = {k: v for k, v in prm.items() if k not in ("nx", "ny", "nz", "omega")}
        state = developed_jet_device(torch, nx, ny, nz, D, prm["jet_velocity"], tdt, dev)
    if args.forcing == "guo":
        kw["forcing"] = tslb.FORCING_GUO
    sim = tslb.Tslb(nx, ny, nz, omega, precision=prec, device=local, kernel=kern, **kw)
    sim.init_fields(state["rho"], state["ux"], state["uy"], state["uz"], state["phi"])
    nodes = nx * ny * nz

    def barrier():
        torch.cuda.synchronize()
        tdist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then exactly K steps between CUDA events on the
    # library's stream (torch's current stream was handed to tslb_create)
    sim.step(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    l0 = sim.launch_count
    t0 = time.time()
    rep_ms = []
    for _ in range(max(1, args.reps)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        sim.step(args.steps)
        e1.record()
        barrier()
        rep_ms.append(tdist.max_over_ranks(e0.elapsed_time(e1), dev))
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    ms = float(np.median(rep_ms))            # K steps, median over the repetitions (max over ranks each)
    launches = (sim.launch_count - l0) // max(1, args.reps)
    m = sim.get_moments(device=True, want=("rho", "phi"))
    finite = bool(torch.isfinite(m["rho"]).all().item() and torch.isfinite(m["phi"]).all().item())
    del m
    ms_max = ms
    glups = world * nodes * args.steps / (ms * 1e-3) / 1e9      # whole job: all ranks' nodes / slowest rank's time

    # ---- end to end through the C-ABI with HOST buffers: H2D of the inputs, K steps, D2H of the state
    e2e = None
    if not args.no_e2e:
        host = {k: torch.empty((nz, ny, nx), dtype=tdt, pin_memory=True) for k in ("rho", "ux", "uy", "uz", "phi")}
        for k in host:
            host[k].copy_(state[k])
        del state
        torch.cuda.empty_cache()
        out_host = [torch.empty((nz, ny, nx), dtype=tdt, pin_memory=True) for _ in range(11)]
        lib = tslb.lib()
        import ctypes
        arr = (ctypes.c_void_p * 6)(*[t.data_ptr() for t in out_host[4:10]])
        barrier()
        w0 = time.perf_counter()
        rc = lib.tslb_init_fields(sim._h, host["rho"].data_ptr(), host["ux"].data_ptr(), host["uy"].data_ptr(),
                                  host["uz"].data_ptr(), host["phi"].data_ptr(), None, 0)
        assert rc == 0
        rc = lib.tslb_step(sim._h, args.steps)
        assert rc == 0
        rc = lib.tslb_get_moments(sim._h, out_host[0].data_ptr(), out_host[1].data_ptr(), out_host[2].data_ptr(),
                                  out_host[3].data_ptr(), arr, out_host[10].data_ptr(), 0)
        assert rc == 0
        torch.cuda.synchronize()
        w1 = time.perf_counter()
        esz = 4 if prec == tslb.F32 else 8
        e2e = {"value": tdist.job_throughput(nodes * args.steps, w1 - w0, dev) / 1e9, "unit": "GLUPS",
               "h2d_bytes_per_step": 5 * nodes * esz / args.steps, "d2h_bytes_per_step": 11 * nodes * esz / args.steps,
               "what": "tslb_init_fields(host) + tslb_step(K) + tslb_get_moments(host), pinned host buffers, "
                       "wall clock; bytes are the job's total divided by K"}
        del host, out_host
    kname = sim.kernel_name
    sim.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline (HBM): algorithmic bytes per node-update x nodes / kernel time
    bpn = BYTES_PER_NODE[(args.precision, True)]
    peaks, peak_src = None, "fallback 6650 GB/s (B200_PROFILING.md)"
    pth = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pth):
        peaks = json.load(open(pth))
        peak_src = "measured copy bandwidth (MEASURED_PEAKS.json)"
    peak = float(peaks["hbm_gbs"]) if peaks else 6650.0
    ms_step = ms / args.steps
    achieved = bpn * nodes / (ms_step * 1e-3) / 1e9
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        tj = json.load(open(tp)).get(args.config + ("" if args.precision == "f32" else "_" + args.precision))
        if tj and kname.startswith("tiled<"):     # the ncu capture is of the tiled kernel
            traffic = tj.get("dram_bytes_per_launch")
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "peak_source": peak_src, "kernel": kname,
                "bytes_per_node_update": bpn, "nodes_per_launch": nodes}

    cpu = None
    if not args.no_cpu:
        g, threads, sample, _ = oracle_sample(args.config, 6)
        cpu = {"value": g, "unit": "GLUPS", "cores": threads, "kind": "oracle", "sample": sample,
               "cpu_model": cpu_model(),
               # the oracle on C3 and on the C4 shape, one thread and all cores (bounded:
               # each child runs a few seconds to half a minute)
               "more": [cpu_sample_subprocess("c3", 10, "c3", 0), cpu_sample_subprocess("c3", 2, "c3", 1),
                        cpu_sample_subprocess("c4", 2, "c4slab", 0), cpu_sample_subprocess("c4", 1, "slab", 1)]}

    out = {"metric": "GLUPS (fused flow+phase-field step)", "value": glups, "unit": "GLUPS", "n_gpus": world,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
           "config": {"workload": desc, "grid": [nx, ny, nz], "state_bytes_per_gpu": 2 * 11 * nodes * (4 if prec == tslb.F32 else 8),
                      "l2": "state (%.1f GB) far exceeds the 126 MB L2; no flush needed" % (2 * 11 * nodes * (4 if prec == tslb.F32 else 8) / 1e9),
                      "parallelism": "replicas x%d" % world if world > 1 else "single GPU",
                      "initial_state": "seeded synthetic developed jet (device-generated)", "finite": finite,
                      "forcing": args.forcing},
           "reps": {"n": len(rep_ms), "ms_per_step": [x / args.steps for x in rep_ms], "median": ms / args.steps,
                    "min": min(rep_ms) / args.steps},
           "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
           "paper_context": "paper: ~1.5 GLUPS RTX 3090, ~2 GLUPS A100 on 400x400x800 (PAPER.md:283); other hardware, not the target"}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
