#!/usr/bin/env python
"""bench.py -- throughput of the MRHS Wilson-clover stencil hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--sweep OUT.jsonl]

One "step" is one pass of the whole hot path over one batch
of seeded synthetic input, at BASELINE.json's target workload (config 5: 48^4 fine lattice,
N_rhs = 12, mass -0.05, c_sw 1.5; plus config 4's coarsest-style level 6^3x32, nbasis 40,
N_rhs = 12):

    D_hop (full lattice)                                   row a2
    M_eooe (odd <- even) and M_eooe (even <- odd)          row a3
    M_ooee (full lattice)                                  row a4
    Schur sequence M_eooe, M_ooee, M_eooe                  row a7 (M_ooee fused into the first hop: 2 launches)
    coarse 9-point apply, FP32 FMA                         row a5
    coarse 9-point apply, tensor cores (3xTF32, tcgen05)    row a6
    coarse 9-point apply, tensor cores (fp16 hi + lo split, kind::f16; column-maximum and split passes included)  row a6

All fields are resident in HBM in the library's native layout when the timed region starts; the
working set of every launch (>= 0.85 GB) is far larger than the 126 MB L2, so no flush is needed
between iterations.  The metric is nominal GFLOP/s (1320 flops/site/RHS for the hop, 504 for the
clover term, 72 nb^2 for the coarse apply); each kernel's algorithmic GB/s against the measured
HBM copy bandwidth (MEASURED_PEAKS.json) is reported beside it, with mean, median and minimum
launch time.  The line also carries `nrhs_sweep`: D_hop, M_eooe, M_ooee and the coarse apply (both
math modes) at the N_rhs lists of BASELINE.json's configs 2-5 -- the metric is "GFLOP/s and % HBM
roofline vs N_rhs" -- timed launch by launch with an L2 flush in between (--no-sweep leaves it out).

--impl reference times the fp64 CPU oracle (oracle/), as it stands, on a bounded sample of the
same workload (named in its config.workload).  --sweep OUT.jsonl writes one JSON line per
(operator, lattice, N_rhs) for every operator of the library over configs 2-5.
"""
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

FLOPS_HOP = 1320.0      # per output site per RHS (BASELINE.json north_star)
FLOPS_CLOVER = 504.0    # per site per RHS (reading S10)
FINE_DIMS = [48, 48, 48, 48]
COARSE_DIMS = [6, 6, 6, 32]
NBASIS = 40
NRHS = 12
MASS, CSW = -0.05, 1.5
SEED = 5

# bounded sample of the same workload for the CPU oracle (cpu_baseline and --impl reference): the fine operators full-field
# on config 2's 24^4 lattice (1/16 of the sites of the 48^4 bench lattice, same N_rhs, same operators) and config 4 in full
CPU_FINE_DIMS = [24, 24, 24, 24]
CPU_COARSE_DIMS = [6, 6, 6, 32]
CPU_SAMPLE = ("fp64 oracle, OpenMP over sites: the step's fine operators (D_hop, M_eooe x2, M_ooee, M_eooe M_ooee M_eooe) full-field on "
              "config 2's 24^4 lattice at N_rhs=12 (1/16 of the 48^4 sites of the GPU step) + config 4's coarse apply in full (6^3x32, nbasis 40), three times as in the GPU step (once per math mode)")


def coarse_flops(nb):
    return 72.0 * nb * nb


def bytes_dhop(V, N):
    return V * (288.0 + 192.0 * N)


def bytes_meooe(V, N):
    return (V / 2) * (576.0 + 192.0 * N)


def bytes_mooee(nsites, N):
    return nsites * (288.0 + 192.0 * N)


def bytes_coarse(V, nb, N):
    return V * (72.0 * nb * nb + 16.0 * nb * N)


def vol(dims):
    return dims[0] * dims[1] * dims[2] * dims[3]


def step_work(fdims, cdims, nb, N, schur_fused=True):
    """Nominal flops and algorithmic bytes of each launch of one step, in launch order.  The Schur-style sequence is
    credited with the flops of its three operators and with the bytes of the path that runs: fused (sweep kernel, two
    launches) the M_ooee stage moves only the clover blocks of the odd sites (288 B each) -- the intermediate field is
    neither written nor re-read; unfused (gather kernel, three launches) it is a full M_ooee pass."""
    V, Vc = vol(fdims), vol(cdims)
    hop_f, hop_b = FLOPS_HOP * (V / 2) * N, bytes_meooe(V, N)
    clv_h_f = FLOPS_CLOVER * (V / 2) * N
    clv_h_b = 288.0 * (V / 2) if schur_fused else bytes_mooee(V / 2, N)
    return [
        ("dhop", FLOPS_HOP * V * N, bytes_dhop(V, N)),
        ("meooe_oe", hop_f, hop_b),
        ("meooe_eo", hop_f, hop_b),
        ("mooee", FLOPS_CLOVER * V * N, bytes_mooee(V, N)),
        ("schur_meooe_oe", hop_f, hop_b),
        ("schur_mooee_oo", clv_h_f, clv_h_b),
        ("schur_meooe_eo", hop_f, hop_b),
        ("coarse_fma", coarse_flops(nb) * Vc * N, bytes_coarse(Vc, nb, N)),
        ("coarse_tc", coarse_flops(nb) * Vc * N, bytes_coarse(Vc, nb, N)),
        ("coarse_tc_f16", coarse_flops(nb) * Vc * N, bytes_coarse(Vc, nb, N)),
    ]


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(key):
    """DRAM bytes per launch from the committed ncu capture (profiles/dram_traffic.csv), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "dram_traffic.csv")) as f:
            for line in f:
                parts = line.strip().split(",")
                if len(parts) == 2 and parts[0] == key:
                    return float(parts[1])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                smax = float(parts[1])
            except ValueError:
                continue
            for n, v in zip(names, parts[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "samples": len(sm),
                "reasons": sorted(reasons)}


# ------------------------------------------------------------------------ CPU oracle arm

def oracle_step_setup():
    import numpy as np
    import oracle
    import synth_inputs as syn
    fd, cd = CPU_FINE_DIMS, CPU_COARSE_DIMS
    U = syn.gauge_np(fd, SEED).astype(np.complex128)
    psi = syn.spinor_np(vol(fd), NRHS, SEED).astype(np.complex128)
    C, _ = oracle.clover_blocks(fd, U, MASS, CSW)          # setup (row a0), untimed like the GPU side
    pe, po = oracle.cb_split(fd, psi)
    Ce, Co = oracle.cb_split(fd, C)
    A = syn.coarse_links_np(cd, NBASIS, 4).astype(np.complex128)
    v = syn.coarse_vector_np(cd, NBASIS, NRHS, 4).astype(np.complex128)
    return dict(fd=fd, cd=cd, U=U, psi=psi, C=C, pe=pe, po=po, Co=Co, A=A, v=v)


def oracle_step(s):
    import oracle
    oracle.dhop(s["fd"], s["U"], s["psi"])
    oracle.meooe(s["fd"], s["U"], s["pe"], 1)
    oracle.meooe(s["fd"], s["U"], s["po"], 0)
    oracle.mooee(s["C"], s["psi"])
    t = oracle.meooe(s["fd"], s["U"], s["pe"], 1)
    t = oracle.mooee(s["Co"], t)
    oracle.meooe(s["fd"], s["U"], t, 0)
    for _ in range(3):      # the GPU step applies the coarse operator once per math mode (FP32 FMA, tf32 split, fp16 split)
        oracle.coarse_apply(s["cd"], s["A"], s["v"])


def time_oracle(steps, warmup):
    import oracle
    s = oracle_step_setup()
    flops = sum(w[1] for w in step_work(CPU_FINE_DIMS, CPU_COARSE_DIMS, NBASIS, NRHS))
    for _ in range(warmup):
        oracle_step(s)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_step(s)
    dt = (time.perf_counter() - t0) / steps
    return flops / dt / 1e9, dt * 1e3, oracle.get_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    gf, ms, cores = time_oracle(args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": "MRHS Wilson-clover stencil hot path, nominal GFLOP/s", "value": gf,
        "unit": "GFLOP/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": reference_config(),
        "cpu_baseline": {"value": gf, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": CPU_SAMPLE},
        "e2e": {"value": gf, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def workload_config():
    return {"workload": "config 5 (48^4 fine, N_rhs=12, mass -0.05, c_sw 1.5: D_hop, M_eooe x2, M_ooee, Schur sequence) "
                        "+ config 4 (6^3x32 coarse, nbasis 40, N_rhs=12: 9-point apply in the three math modes: FP32 FMA, tf32 split, fp16 split)",
            "fine_dims": FINE_DIMS, "coarse_dims": COARSE_DIMS, "nbasis": NBASIS, "n_rhs": NRHS,
            "precision": "complex64 fields, fp32 FMA",
            "l2": "every launch touches >= 0.85 GB, far above the 126 MB L2; no flush between iterations",
            "parallelism": "replicas only (one GPU per lattice, no collectives; north_star)"}


def reference_config():
    """The oracle arm times a bounded sample, and says so where the workload is named: its config is NOT the GPU arm's."""
    cfg = workload_config()
    cfg["workload"] = "SAMPLE of the GPU arm's workload -- " + CPU_SAMPLE
    cfg["fine_dims"], cfg["coarse_dims"] = CPU_FINE_DIMS, CPU_COARSE_DIMS
    cfg["precision"] = "complex128 (fp64 oracle)"
    cfg["gpu_arm_workload"] = workload_config()["workload"]
    return cfg


# ------------------------------------------------------------------------ replicas (N > 1)

def max_over_ranks(x, dist, device):
    """max of a per-rank scalar over all ranks (the slowest replica sets the job time)."""
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_gflops(flops_step, world, ms_per_step):
    """Whole-job throughput of `world` independent replicas (weak scaling: one lattice per GPU)."""
    return world * flops_step / (ms_per_step * 1e-3) / 1e9


# ------------------------------------------------------------------------ GPU arm

class Workload:
    """Device-resident inputs and handles of one step (native layout), plus host staging for e2e."""

    def __init__(self, torch, mrhs, syn, device, stream, fdims, cdims, nb, N):
        self.torch, self.mrhs, self.fdims, self.cdims, self.nb, self.N = torch, mrhs, fdims, cdims, nb, N
        V = vol(fdims)
        U = syn.gauge_torch(fdims, SEED, device)
        torch.cuda.synchronize()     # the inputs are generated on torch's current stream, the library works on `stream`
        self.w = mrhs.Wilson(fdims, N, MASS, CSW, U, stream=stream)
        del U
        psi = syn.spinor_torch(V, N, SEED, device)
        self.psi = self.w.import_field(psi, mrhs.FULL)
        del psi
        self.out_full = self.w.empty(mrhs.FULL)
        self.in_e, self.in_o = self.w.empty(mrhs.EVEN), self.w.empty(mrhs.ODD)
        mrhs.cb_split(fdims, 12, N, self.psi, self.in_e, self.in_o)
        self.out_e, self.out_o = self.w.empty(mrhs.EVEN), self.w.empty(mrhs.ODD)
        self.t0, self.t1 = self.w.empty(mrhs.ODD), self.w.empty(mrhs.ODD)
        A = syn.coarse_links_torch(cdims, nb, 4, device)
        torch.cuda.synchronize()
        self.c = mrhs.Coarse(cdims, nb, N, A, stream=stream)
        self.c_tc = mrhs.Coarse(cdims, nb, N, A, math_mode=mrhs.COARSE_TENSOR, stream=stream)
        self.c_h16 = mrhs.Coarse(cdims, nb, N, A, math_mode=mrhs.COARSE_TENSOR_F16, stream=stream)
        del A
        v = syn.spinor_torch(vol(cdims), N, 4, device, ncomp=(nb,))
        self.v = self.c.import_field(v)
        self.v_out = self.c.empty()
        torch.cuda.synchronize()

    def launches(self):
        w, c, m = self.w, self.c, self.mrhs
        return [
            ("dhop", lambda: w.dhop(self.psi, self.out_full)),
            ("meooe_oe", lambda: w.meooe(self.in_e, self.out_o, m.ODD)),
            ("meooe_eo", lambda: w.meooe(self.in_o, self.out_e, m.EVEN)),
            ("mooee", lambda: w.mooee(self.psi, self.out_full, m.FULL)),
            ("schur", lambda: w.schur_sequence(self.in_e, self.t0, self.t1, self.out_e)),
            ("coarse_fma", lambda: c.apply(self.v, self.v_out)),
            ("coarse_tc", lambda: self.c_tc.apply(self.v, self.v_out)),
            ("coarse_tc_f16", lambda: self.c_h16.apply(self.v, self.v_out)),
        ]


def run_gpu(args):
    import torch
    import paper_2211_13719_b200 as mrhs
    import synth_inputs as syn

    mrhs.lib()   # fails loudly if libmrhs.so is missing: there is no fallback
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    fdims, cdims, nb, N = FINE_DIMS, COARSE_DIMS, NBASIS, NRHS
    if args.small:
        fdims, cdims = [16, 16, 16, 16], [4, 4, 4, 4]
    stream = torch.cuda.Stream(device)
    wl = Workload(torch, mrhs, syn, device, stream, fdims, cdims, nb, N)
    tiling_note = "library default"
    for which in (0, 1):
        if args.hop_tiling:
            t = [int(x) for x in args.hop_tiling.split(",")]
            mrhs.wilson_set_tiling(wl.w.h, which, t[:3], t[3:5])
        if args.hop_kernel is not None:
            mrhs.wilson_set_hop_kernel(wl.w.h, which, {"gather": mrhs.HOP_GATHER, "sweep": mrhs.HOP_SWEEP}[args.hop_kernel])
        if args.hop_sweep:
            t = [int(x) for x in args.hop_sweep.split(",")]
            mrhs.wilson_set_sweep(wl.w.h, which, t[0], t[1:3])
        if args.hop_prefetch is not None:
            mrhs.wilson_set_prefetch(wl.w.h, which, args.hop_prefetch)
    if args.hop_tiling or args.hop_prefetch is not None or args.hop_kernel or args.hop_sweep:
        tiling_note = "override: kernel %s tiling %s prefetch %s sweep %s" % (args.hop_kernel, args.hop_tiling, args.hop_prefetch, args.hop_sweep)
    launches = wl.launches()
    fused = mrhs.wilson_get_hop_kernel(wl.w.h, 1) == mrhs.HOP_SWEEP
    work = step_work(fdims, cdims, nb, N, schur_fused=fused)
    flops_step = sum(w[1] for w in work)
    K, W = args.steps, args.warmup

    # one event pair per launch group per step, recorded on the stream the kernels run on
    nseg = len(launches)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(nseg + 1)] for _ in range(K)]
    for _ in range(W):
        for _, f in launches:
            f()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    t_wall = time.perf_counter()
    for k in range(K):
        evs[k][0].record(stream)
        for i, (_, f) in enumerate(launches):
            f()
            evs[k][i + 1].record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop() if rank == 0 else None
    total_ms = evs[0][0].elapsed_time(evs[K - 1][nseg])
    seg_all = [sorted(evs[k][i].elapsed_time(evs[k][i + 1]) for k in range(K)) for i in range(nseg)]
    seg_ms = [sum(a) / K for a in seg_all]
    total_ms = max_over_ranks(total_ms, dist, device)
    ms_per_step = total_ms / K
    value = job_gflops(flops_step, world, ms_per_step)

    # ------------------------------------------------------------ end to end, host buffers
    e2e = run_e2e(torch, mrhs, wl, args, barrier, dist, device, world, flops_step)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    peak, peak_src = measured_peaks()
    V = vol(fdims)
    seg_names = [n for n, _ in launches]
    kernels = {}
    for name, ms, allms in zip(seg_names, seg_ms, seg_all):
        if name == "schur":
            fl = sum(w[1] for w in work if w[0].startswith("schur"))
            by = sum(w[2] for w in work if w[0].startswith("schur"))
        else:
            fl, by = [(w[1], w[2]) for w in work if w[0] == name][0]
        gbs = by / (ms * 1e-3) / 1e9
        kernels[name] = {"ms": ms, "ms_median": allms[len(allms) // 2], "ms_min": allms[0], "gflops": fl / (ms * 1e-3) / 1e9,
                         "gbs": gbs, "hbm_frac": gbs / peak, "algorithmic_bytes": by, "share_of_step": ms / sum(seg_ms)}
        if name == "schur":
            # what three separate launches would have to move (22.2 GB), for comparison only
            by3 = 2 * bytes_meooe(V, N) + bytes_mooee(V / 2, N)
            kernels[name]["launches"] = 2 if fused else 3
            kernels[name]["gbs_credited_with_unfused_bytes"] = by3 / (ms * 1e-3) / 1e9
    d = kernels["dhop"]
    kname = {mrhs.HOP_GATHER: "hop_kernel (gather)", mrhs.HOP_SWEEP: "hop_sweep_kernel (slice sweep)"}
    roofline = {"kernel": "%s: D_hop, full lattice %dx%dx%dx%d, N_rhs=%d" % (kname[mrhs.wilson_get_hop_kernel(wl.w.h, 0)], *fdims, N), "bound": "hbm",
                "achieved": d["gbs"], "peak": peak, "unit": "GB/s", "frac": d["gbs"] / peak,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": bytes_dhop(V, N),
                "avg_launch_ms": d["ms"], "median_launch_ms": d["ms_median"], "min_launch_ms": d["ms_min"],
                "traffic": ncu_traffic("dhop_48x48x48x48_n12") if not args.small else None,
                "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of this kernel in the committed ncu capture "
                                  "(profiles/dram_traffic.csv; ncu cannot run inside the timed bench)"}
    cpu = None
    if not args.no_cpu:
        gf, ms, cores = time_oracle(args.cpu_steps, 1)
        cpu = {"value": gf, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": CPU_SAMPLE, "ms_per_sample_step": ms}
    nrhs_sweep = None
    if not args.no_sweep and not args.small:
        # release the step's fields first: the sweep builds its own handles (48^4 at N_rhs = 24 needs 12 GB per field)
        wl = release_fields(wl)
        nrhs_sweep = [r for r in sweep_records(torch, mrhs, syn, device, stream, peak, iters=args.inrun_sweep_iters, subset="north_star")]
    cfg = workload_config()
    def hop_cfg(which):
        k = mrhs.wilson_get_hop_kernel(wl.w.h, which)
        if k == mrhs.HOP_SWEEP:
            lt, chunk = mrhs.wilson_get_sweep(wl.w.h, which)
            return {"kernel": "sweep", "tile_yz": [2, 2], "segment_t": lt, "chunk_tiles_yz": chunk}
        tile, chunk = mrhs.wilson_get_tiling(wl.w.h, which)
        return {"kernel": "gather", "tile_yzt": tile, "chunk_tiles_yz": chunk}
    cfg["hop_tiling"] = {"dhop": hop_cfg(0), "meooe": hop_cfg(1), "source": tiling_note}
    if args.small:
        cfg["workload"] = "SMALL smoke workload (16^4 fine, 4^4 coarse) -- not the benchmark configuration"
        cfg["fine_dims"], cfg["coarse_dims"] = fdims, cdims
    line = {
        "metric": "MRHS Wilson-clover stencil hot path, nominal GFLOP/s", "value": value, "unit": "GFLOP/s",
        "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": cfg, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "clocks": clocks,
        # + 2: the column-maximum and split passes of the fp16-split coarse apply
        "gpu_launches": (len(work) - (1 if fused else 0) + 2) * K, "kernels": kernels, "wall_ms_per_step": t_wall * 1e3 / K,
        "nrhs_sweep": nrhs_sweep,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def release_fields(wl):
    """Drop the step's device fields (keeps the handles, whose tiling the report still reads)."""
    for name in ("psi", "out_full", "in_e", "in_o", "out_e", "out_o", "t0", "t1", "v", "v_out"):
        setattr(wl, name, None)
    wl.torch.cuda.empty_cache()
    return wl


def run_e2e(torch, mrhs, wl, args, barrier, dist, device, world, flops_step):
    """The same step through the host-buffer C-ABI entries: pinned canonical host fields in,
    canonical host fields out, host<->device copies and layout conversion inside the timed region."""
    if args.no_e2e:
        return None
    fdims, N, nb, cdims = wl.fdims, wl.N, wl.nb, wl.cdims
    V = vol(fdims)
    full_shape, half_shape = (V, 4, 3, N), (V // 2, 4, 3, N)
    h_full_in = torch.empty(full_shape, dtype=torch.complex64).pin_memory()
    # one result buffer per call of the step: the calls are in flight together
    h_full_out = [torch.empty(full_shape, dtype=torch.complex64).pin_memory() for _ in range(2)]
    # canonical host inputs: export the device fields the device-timed arm uses
    h_full_in.copy_(wl.w.export_field(wl.psi, mrhs.FULL))
    h_e_in = torch.empty(half_shape, dtype=torch.complex64).pin_memory()
    h_o_in = torch.empty(half_shape, dtype=torch.complex64).pin_memory()
    h_e_in.copy_(wl.w.export_field(wl.in_e, mrhs.EVEN))
    h_o_in.copy_(wl.w.export_field(wl.in_o, mrhs.ODD))
    h_half_out = [torch.empty(half_shape, dtype=torch.complex64).pin_memory() for _ in range(3)]
    h_v_in = torch.empty((vol(cdims), nb, N), dtype=torch.complex64).pin_memory()
    h_v_in.copy_(wl.c.export_field(wl.v))
    h_v_out = [torch.empty_like(h_v_in).pin_memory() for _ in range(3)]
    torch.cuda.synchronize()
    w = wl.w.h
    coarse = (wl.c.h, wl.c_tc.h, wl.c_h16.h)     # one coarse apply per math mode, as in the device-timed step

    def step():
        # the asynchronous host entries: every call's host->device copy, kernels and device->host copy are enqueued, the copy-in
        # of a call runs under the kernels and the copy-out of the call before it; the step ends when every result is on the host
        mrhs.wilson_apply_host_async(w, mrhs.OP_DHOP, 0, h_full_in, h_full_out[0])
        mrhs.wilson_apply_host_async(w, mrhs.OP_MEOOE, mrhs.ODD, h_e_in, h_half_out[0])
        mrhs.wilson_apply_host_async(w, mrhs.OP_MEOOE, mrhs.EVEN, h_o_in, h_half_out[1])
        mrhs.wilson_apply_host_async(w, mrhs.OP_MOOEE, mrhs.FULL, h_full_in, h_full_out[1])
        mrhs.wilson_apply_host_async(w, mrhs.OP_SCHUR, 0, h_e_in, h_half_out[2])
        for c, o in zip(coarse, h_v_out):
            mrhs.coarse_apply_host_async(c, h_v_in, o)
        mrhs.wilson_host_wait(w)
        for c in coarse:
            mrhs.coarse_host_wait(c)

    fb, hb, cb = h_full_in.numel() * 8, h_e_in.numel() * 8, h_v_in.numel() * 8
    h2d = 2 * fb + 3 * hb + 3 * cb
    d2h = 2 * fb + 3 * hb + 3 * cb
    E = max(1, min(args.steps, args.e2e_steps))
    step()   # warm-up: allocates the handle's staging buffers
    barrier()
    t0 = time.perf_counter()
    for _ in range(E):
        step()   # ends with the host waits: every result of the step is in host memory
    barrier()
    dt = time.perf_counter() - t0
    dt = max_over_ranks(dt, dist, device) / E
    return {"value": job_gflops(flops_step, world, dt * 1e3), "unit": "GFLOP/s", "h2d_bytes_per_step": h2d,
            "d2h_bytes_per_step": d2h, "ms_per_step": dt * 1e3, "steps": E,
            "api": "mrhs_wilson_apply_host_async / mrhs_coarse_apply_host_async + mrhs_*_host_wait (pinned canonical host buffers, "
                   "three staging slots: the copy-in of a call overlaps the kernels and the copy-out of the call before)"}


# ------------------------------------------------------------------------ N_rhs sweep

def sweep_records(torch, mrhs, syn, device, stream, peak, iters, subset, warm=10, ops=("fine", "coarse")):
    """Per (operator, lattice, N_rhs) records for configs 2-5: median and min time of individually timed launches on the
    library's stream, L2 flushed between launches (a 512 MB memset), GFLOP/s, algorithmic GB/s, fraction of the measured
    HBM peak, speed-up per RHS over the first N_rhs of the config.  subset "north_star": D_hop, M_eooe, M_ooee and the
    coarse apply in both math modes at the N_rhs lists of BASELINE.json's configs (what the metric names);
    "all": every operator of the library."""
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=device)
    everything = subset == "all"

    def timeit(f):
        with torch.cuda.stream(stream):
            for _ in range(warm):
                f()
            ts = []
            for _ in range(iters):
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                f()
                e1.record(stream)
                e1.synchronize()
                ts.append(e0.elapsed_time(e1))
        ts.sort()
        return ts[len(ts) // 2], ts[0]

    base = {}

    def rec(cfg, op, dims, N, fl, by, t, extra=None):
        med, mn = t
        r = {"config": cfg, "op": op, "dims": dims, "n_rhs": N, "ms_median": med, "ms_min": mn,
             "gflops": fl / (med * 1e-3) / 1e9, "gbs": by / (med * 1e-3) / 1e9,
             "hbm_frac": by / (med * 1e-3) / 1e9 / peak, "alg_bytes": by, "nominal_flops": fl}
        base.setdefault((cfg, op), med / N)
        r["speedup_per_rhs_vs_first_n"] = base[(cfg, op)] / (med / N)
        if extra:
            r.update(extra)
        return r

    fine = [("config2", [24, 24, 24, 24], [1, 4, 12, 24, 48], 2), ("config5", [48, 48, 48, 48], [1, 12, 24], 5)]
    for cfg, dims, ns, seed in (fine if "fine" in ops else []):
        V = vol(dims)
        U = syn.gauge_torch(dims, seed, device)
        for N in ns:
            torch.cuda.synchronize()
            w = mrhs.Wilson(dims, N, MASS, CSW, U, stream=stream)
            psi = w.import_field(syn.spinor_torch(V, N, seed, device), mrhs.FULL)
            o_full = w.empty(mrhs.FULL)
            ie, io = w.empty(mrhs.EVEN), w.empty(mrhs.ODD)
            mrhs.cb_split(dims, 12, N, psi, ie, io)
            oe, oo, t0 = w.empty(mrhs.EVEN), w.empty(mrhs.ODD), w.empty(mrhs.ODD)
            torch.cuda.synchronize()
            kern = {mrhs.HOP_GATHER: "gather", mrhs.HOP_SWEEP: "sweep"}[mrhs.wilson_get_hop_kernel(w.h, 0)]
            yield rec(cfg, "dhop", dims, N, FLOPS_HOP * V * N, bytes_dhop(V, N), timeit(lambda: w.dhop(psi, o_full)), {"hop_kernel": kern})
            yield rec(cfg, "meooe", dims, N, FLOPS_HOP * V / 2 * N, bytes_meooe(V, N), timeit(lambda: w.meooe(ie, oo, mrhs.ODD)), {"hop_kernel": kern})
            yield rec(cfg, "mooee", dims, N, FLOPS_CLOVER * V * N, bytes_mooee(V, N), timeit(lambda: w.mooee(psi, o_full, mrhs.FULL)))
            if everything or N == 12:
                fused = kern == "sweep"
                by = 2 * bytes_meooe(V, N) + (288.0 * V / 2 if fused else bytes_mooee(V / 2, N))
                yield rec(cfg, "schur_seq", dims, N, (2 * FLOPS_HOP + FLOPS_CLOVER) * V / 2 * N, by,
                          timeit(lambda: w.schur_sequence(ie, oo, t0, oe)), {"launches": 2 if fused else 3})
                # the even-odd preconditioned operator C_e - H_eo C_o^-1 H_oe / 4 (NEXT-2): two hops, the even input read twice
                yield rec(cfg, "schur_apply", dims, N, (2 * FLOPS_HOP + 2 * FLOPS_CLOVER + 24) * V / 2 * N,
                          2 * bytes_meooe(V, N) + (V / 2) * (2 * 288.0 + 96.0 * N), timeit(lambda: w.schur_apply(ie, t0, oe)))
                # the full Wilson-clover matrix M = M_ooee - D_hop / 2 in one launch: gauge + clover + one field in, one out
                yield rec(cfg, "wilson_M", dims, N, (FLOPS_HOP + FLOPS_CLOVER + 48) * V * N, V * (576.0 + 192.0 * N), timeit(lambda: w.apply(psi, o_full)))
                yield rec(cfg, "dhop_dag", dims, N, FLOPS_HOP * V * N, bytes_dhop(V, N), timeit(lambda: w.dhop_dag(psi, o_full)))
            if everything:
                # simultaneous inner products <psi_r, out_r> (NEXT-4): two fields read once, 8 flops per complex element
                res = torch.empty(N, dtype=torch.complex128, device=device)
                yield rec(cfg, "inner_products", dims, N, 8.0 * 12 * V * N, 2.0 * 96 * V * N,
                          timeit(lambda: mrhs.inner_products(dims, 12, N, mrhs.FULL, psi, o_full, res, stream=stream)))
                # intergrid operators (NEXT-3): 4^4 aggregates, 20 basis vectors (nbasis 40); basis 1920 B per site
                if N in (12, 24) and cfg == "config5":
                    nvec, bd = 20, [4, 4, 4, 4]
                    cd = [d // b for d, b in zip(dims, bd)]
                    basis = syn.spinor_torch(V * nvec, 1, seed + 1, device).reshape(nvec, V, 4, 3)
                    torch.cuda.synchronize()
                    tr = mrhs.Transfer(dims, bd, nvec, N, basis, stream=stream)
                    del basis
                    vc = mrhs.empty_field(cd, 2 * nvec, N, mrhs.FULL, device)
                    vc.normal_()
                    torch.cuda.synchronize()
                    fl, by = 8.0 * 12 * nvec * V * N, V * (96.0 * nvec + 96.0 * N) + vol(cd) * 16.0 * nvec * N
                    yield rec(cfg, "prolong", dims, N, fl, by, timeit(lambda: tr.prolong(vc, o_full)), {"nvec": nvec, "block": bd})
                    yield rec(cfg, "restrict", dims, N, fl, by, timeit(lambda: tr.restrict(psi, vc)), {"nvec": nvec, "block": bd})
                    tr.close()
                    del vc
            w.close()
            del w, psi, o_full, ie, io, oe, oo, t0
            torch.cuda.empty_cache()
        del U
    coarse = [("config3", [8, 8, 8, 8], 24, [1, 12, 24, 64], 3), ("config4", [6, 6, 6, 32], 40, [12, 24, 48, 96], 4)]
    for cfg, dims, nb, ns, seed in (coarse if "coarse" in ops else []):
        V = vol(dims)
        A = syn.coarse_links_torch(dims, nb, seed, device)
        for N in ns:
            for mode in mrhs.COARSE_MODES:
                torch.cuda.synchronize()
                try:
                    c = mrhs.Coarse(dims, nb, N, A, math_mode=mode, stream=stream)
                except mrhs.MrhsError:
                    continue
                v = c.import_field(syn.spinor_torch(V, N, seed, device, ncomp=(nb,)))
                vo = c.empty()
                torch.cuda.synchronize()
                fl = coarse_flops(nb) * V * N
                t = timeit(lambda: c.apply(v, vo))
                yield rec(cfg, "coarse_mode%d" % mode, dims, N, fl, bytes_coarse(V, nb, N), t,
                          {"nbasis": nb, "fp32_fma_peak_frac": fl / (t[0] * 1e-3) / 74.4e12})
                # the 8-point coarse hopping term alone (what the paper's coarse-level figure measures, reading S12) and coarse
                # M_eooe (NEXT-1): the same term on one parity from the other (all link matrices of the output sites, half the vectors)
                yield rec(cfg, "coarse_hop8_mode%d" % mode, dims, N, 64 * nb * nb * V * N, V * (64 * nb * nb + 16 * nb * N),
                          timeit(lambda: c.apply(v, vo, mrhs.COARSE_HOP)), {"nbasis": nb})
                if all(d % 2 == 0 for d in dims):
                    ve, vod = c.empty(parity=mrhs.EVEN), c.empty(parity=mrhs.ODD)
                    mrhs.coarse_cb_split(dims, nb, N, v, ve, vod)
                    oe = c.empty(parity=mrhs.EVEN)
                    torch.cuda.synchronize()
                    yield rec(cfg, "coarse_meooe_mode%d" % mode, dims, N, 64 * nb * nb * (V / 2) * N, (V / 2) * (64 * nb * nb + 16 * nb * N),
                              timeit(lambda: c.meooe(vod, oe, mrhs.EVEN)), {"nbasis": nb})
                    del ve, vod, oe
                c.close()
                del c, v, vo
        if everything and cfg == "config4":
            # coarse -> coarser intergrid operators (NEXT-3): 40 -> 60 components, 3 x 3 x 3 x 2 aggregates
            nf, nvec, bd, N = nb, 30, [3, 3, 3, 2], 12
            cd = [d // b for d, b in zip(dims, bd)]
            basis = syn.spinor_torch(V * nvec, 1, seed + 1, device, ncomp=(nf,)).reshape(nvec, V, nf)
            torch.cuda.synchronize()
            tr = mrhs.Transfer(dims, bd, nvec, N, basis, stream=stream, nf=nf)
            del basis
            vc = mrhs.empty_field(cd, 2 * nvec, N, mrhs.FULL, device).normal_()
            vf = mrhs.empty_field(dims, nf, N, mrhs.FULL, device).normal_()
            torch.cuda.synchronize()
            fl, by = 8.0 * (nf / 2) * nvec * V * N * 2 / 2, V * (8.0 * nf * nvec + 8.0 * nf * N) + vol(cd) * 16.0 * nvec * N
            yield rec(cfg, "prolong_coarse", dims, N, fl, by, timeit(lambda: tr.prolong(vc, vf)), {"nf": nf, "nvec": nvec, "block": bd})
            yield rec(cfg, "restrict_coarse", dims, N, fl, by, timeit(lambda: tr.restrict(vf, vc)), {"nf": nf, "nvec": nvec, "block": bd})
            tr.close()
        del A


def run_sweep(args):
    """--sweep OUT.jsonl: every operator of the library over configs 2-5, one JSON line each (and a table on stdout)."""
    import torch
    import paper_2211_13719_b200 as mrhs
    import synth_inputs as syn
    device = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    peak, _ = measured_peaks()
    stream = torch.cuda.Stream(device)
    with open(args.sweep, "w") as out:
        for r in sweep_records(torch, mrhs, syn, device, stream, peak, iters=args.sweep_iters, subset="all", ops=tuple(args.sweep_ops.split(","))):
            out.write(json.dumps(r) + "\n")
            out.flush()
            print("%-8s %-20s %-16s N=%-3d %8.4f ms  %9.1f GF/s  %7.1f GB/s  %5.1f%% HBM" %
                  (r["config"], r["op"], "x".join(map(str, r["dims"])), r["n_rhs"], r["ms_median"], r["gflops"], r["gbs"], 100 * r["hbm_frac"]), flush=True)
    return 0


def run_oracle_table(args):
    """--oracle-table OUT.jsonl: the fp64 oracle as it stands, timed per operator (SURVEY.md Sec. 8(d) "Oracle beside it"):
    full-field on configs 1-4 and on config 5 at N_rhs = 1, single-threaded and with OpenMP over sites on all cores the
    process may use.  A reported baseline (needs no GPU); one JSON line per (config, operator, N_rhs, threads)."""
    import numpy as np
    import oracle
    import synth_inputs as syn
    cores = len(os.sched_getaffinity(0))

    def timed(f, reps):
        f()
        ts = []
        for _ in range(reps):
            t0 = time.perf_counter(); f(); ts.append(time.perf_counter() - t0)
        ts.sort()
        return ts[len(ts) // 2]

    fine = [("config1", [4, 4, 4, 4], [4], -0.1, 1.0, 0, 5), ("config2", [24, 24, 24, 24], [1, 4, 12, 24, 48], MASS, CSW, 2, 1),
            ("config5", [48, 48, 48, 48], [1], MASS, CSW, 5, 1)]
    coarse = [("config3", [8, 8, 8, 8], 24, [1, 12, 24, 64], 3), ("config4", [6, 6, 6, 32], 40, [12, 24, 48, 96], 4)]
    with open(args.oracle_table, "w") as out:
        def emit(cfg, op, dims, N, fl, t, thr):
            r = {"config": cfg, "op": op, "dims": dims, "n_rhs": N, "threads": thr, "ms": t * 1e3, "gflops": fl / t / 1e9,
                 "site_rhs_per_s": vol(dims) * N / t, "kind": "oracle", "dtype": "f64"}
            out.write(json.dumps(r) + "\n"); out.flush()
            print("%-8s %-10s %-14s N=%-3d threads=%-3d %10.2f ms %8.2f GF/s" % (cfg, op, "x".join(map(str, dims)), N, thr, r["ms"], r["gflops"]), flush=True)
        for cfg, dims, ns, mass, csw, seed, reps in fine:
            V = vol(dims)
            U = syn.gauge_np(dims, seed).astype(np.complex128)
            oracle.set_threads(cores)
            C, _ = oracle.clover_blocks(dims, U, mass, csw)
            for N in ns:
                psi = syn.spinor_np(V, N, seed).astype(np.complex128)
                pe, _po = oracle.cb_split(dims, psi)
                for thr in (cores, 1):
                    if thr == 1 and V * N > 24 ** 4 * 12:
                        continue          # single-threaded only where it ends in seconds
                    oracle.set_threads(thr)
                    emit(cfg, "dhop", dims, N, 1320.0 * V * N, timed(lambda: oracle.dhop(dims, U, psi), reps), thr)
                    emit(cfg, "meooe", dims, N, 1320.0 * (V / 2) * N, timed(lambda: oracle.meooe(dims, U, pe, 1), reps), thr)
                    emit(cfg, "mooee", dims, N, 504.0 * V * N, timed(lambda: oracle.mooee(C, psi), reps), thr)
                del psi, pe, _po
            del U, C
        for cfg, dims, nb, ns, seed in coarse:
            A = syn.coarse_links_np(dims, nb, seed).astype(np.complex128)
            for N in ns:
                v = syn.coarse_vector_np(dims, nb, N, seed).astype(np.complex128)
                for thr in (cores, 1):
                    if thr == 1 and N > 24:
                        continue
                    oracle.set_threads(thr)
                    emit(cfg, "coarse", dims, N, coarse_flops(nb) * vol(dims) * N, timed(lambda: oracle.coarse_apply(dims, A, v), 1), thr)
            del A
    oracle.set_threads(cores)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--small", action="store_true", help="tiny workload for a functional check (not a benchmark)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-steps", type=int, default=8, help="oracle sample steps timed for cpu_baseline")
    ap.add_argument("--sweep", default=None, help="write the per-operator N_rhs sweep to this .jsonl and exit")
    ap.add_argument("--sweep-iters", type=int, default=50)
    ap.add_argument("--oracle-table", default=None, help="time the fp64 oracle per operator on configs 1-5 (host cores, no GPU), write this .jsonl and exit")
    ap.add_argument("--no-sweep", action="store_true", help="leave the N_rhs sweep (key nrhs_sweep) out of the bench line")
    ap.add_argument("--inrun-sweep-iters", type=int, default=10, help="timed launches per point of the in-run N_rhs sweep")
    ap.add_argument("--sweep-ops", default="fine,coarse", help="which operator families the sweep covers")
    ap.add_argument("--hop-tiling", default=None, help="by,bz,bt,cy,cz for D_hop and M_eooe instead of the library default")
    ap.add_argument("--hop-prefetch", type=int, default=None, help="L2 prefetch distance in tiles (0 = off)")
    ap.add_argument("--hop-kernel", default=None, choices=["gather", "sweep"], help="hop kernel instead of the library default")
    ap.add_argument("--hop-sweep", default=None, help="lt,cy,cz for the sweep kernel instead of the library default")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours" and not args.sweep:
        args.warmup = 3   # timing rule: at least 3 warm-up steps
    if args.impl == "reference":
        return run_reference(args)
    if args.oracle_table:
        return run_oracle_table(args)
    if args.sweep:
        return run_sweep(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
