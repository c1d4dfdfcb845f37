#!/usr/bin/env python
"""bench.py — MD-step site-updates/s of the fused hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4] [--dims Lx,Ly,Lz,Lt]

A "step" is one fused molecular-dynamics step on the whole lattice: P += eps F(U), then
U <- reunit(exp(i eps P) U) — force, projection, momentum update, exponential, link update and
reunitarisation, all rows of SURVEY.md section 8(a)'s MD step.  --path single_pass (default, the faster one as
measured: profiles/r02_*.md) runs it as ONE kernel, qcd_md_step_single_pass, ping-ponging two gauge fields
(8(a) "MD step (single pass)", 288 reals/site); --path two_kernel as qcd_force_mom_update followed by
qcd_link_update(reunit) in place (8(a) "MD step (fused)", 432 reals/site).  Default workload: BASELINE
config 4, 32^3x64 fp64, sigma=0.2, beta=6.0, eps=0.02, seeded synthetic hot start generated on the device.

N > 1 (torchrun): the path is run as N independent replicas (one lattice per GPU, different seeds,
no data-path collective); value = total site-updates/s, scaling "weak".
--decompose instead cuts ONE lattice into N slabs of timeslices, one per rank, with a halo exchange per step
(strong scaling; its own JSON object).

--impl reference times the CPU oracle (oracle/, as it stands, serial) on a bounded sample of the
same workload; rank 0 only.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

SEED_BASE = 0x1212078500000000
CONFIGS = {  # BASELINE.json configs: dims, hot-start sigma, beta, eps
    3: dict(dims=(16, 16, 16, 32), sigma=0.5, beta=5.8, eps=0.05, name="16^3x32"),
    4: dict(dims=(32, 32, 32, 64), sigma=0.2, beta=6.0, eps=0.02, name="32^3x64"),
    5: dict(dims=(48, 48, 48, 96), sigma=0.3, beta=6.2, eps=0.01, name="48^3x96"),
}
# reals/site R+W: force+mom reads U,P writes P; exp+reunit reads P,U writes U; the single-pass
# kernel reads U,P and writes P,U
BYTES_PER_SITE = {"force_mom_update": 216, "link_update_reunit": 216, "md_step_single_pass": 288}
# FP64/FP32 arithmetic instructions per site of the default kernels: the plane-sharing force is
# 6 planes x (108 + 108 + 90) + 12 down staples x 216 + 4 x 90 (U_mu A, TA part only) = 4788 FMA, + projection and
# P += eps F; the link update is about 480 per link (Hermitian Q^2 54, series ~95, two rows of E 40, two rows of
# E U 72, reunit ~100, norm, scaling, det ~70)
FMA_FORCE, FMA_MOM, FMA_LINK = 4788, 112, 4 * 480
METRIC = "md_step_site_updates_per_s"
UNIT = "site-updates/s"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """samples SM clock and throttle reasons through NVML (what nvidia-smi reads) while `active`"""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.mask, self.active, self.stop_flag = index, [], 0, False, False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:  # noqa: BLE001
            self.nv, self.err = None, repr(e)

    def run(self):
        while not self.stop_flag and self.nv is not None:
            if self.active:
                try:
                    self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                    self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:  # noqa: BLE001
                    pass
            time.sleep(0.005)

    def summary(self):
        if self.nv is None or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"], "samples": 0}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz,
                "reasons": [n for b, n in self.REASONS.items() if self.mask & b], "samples": len(s)}


def oracle_step_rate(orc, cfg, dims, steps, warmup):
    """time `steps` fused MD steps of the oracle on lattice `dims` (same sigma, beta, eps as cfg)"""
    seed = SEED_BASE + 4
    U = orc.hot_start(dims, seed, cfg["sigma"])
    P = orc.mom_refresh(dims, seed)
    for _ in range(warmup):
        orc.md_step(dims, cfg["beta"], cfg["eps"], cfg["eps"], U, P, inplace=True)
    t0 = time.perf_counter()
    for _ in range(steps):
        orc.md_step(dims, cfg["beta"], cfg["eps"], cfg["eps"], U, P, inplace=True)
    dt = time.perf_counter() - t0
    V = 1
    for d in dims:
        V *= d
    return V * steps / dt, dt


SAMPLE_LATTICES = [(4, 4, 4, 4), (8, 4, 4, 4), (8, 8, 4, 4), (8, 8, 8, 4), (8, 8, 8, 8), (16, 8, 8, 8), (16, 16, 8, 8),
                   (16, 16, 16, 8), (16, 16, 16, 16), (32, 16, 16, 16), (32, 32, 16, 16), (32, 32, 32, 16)]


def pick_sample(orc, cfg, steps_total, budget_s):
    """largest sample lattice whose `steps_total` oracle steps fit the time budget"""
    rate, _ = oracle_step_rate(orc, cfg, (8, 8, 8, 4), 1, 0)  # calibration, ~20 ms
    best = SAMPLE_LATTICES[0]
    for d in SAMPLE_LATTICES:
        V = d[0] * d[1] * d[2] * d[3]
        if V * steps_total / rate <= budget_s:
            best = d
    return best


def run_reference(args, cfg):
    """the oracle, as it stands (serial build), on the host cores; rank 0 only"""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle.oracle import Oracle
    orc = Oracle(omp=False)
    dims = pick_sample(orc, cfg, args.steps + args.warmup, 150.0)
    rate, dt = oracle_step_rate(orc, cfg, dims, args.steps, args.warmup)
    sample = (f"{'x'.join(map(str, dims))} lattice with the {cfg['name']} parameters (sigma={cfg['sigma']}, "
              f"beta={cfg['beta']}, eps={cfg['eps']}), {args.steps} fused MD steps, serial C oracle")
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg['name']} fp64 fused MD step (bounded sample: {'x'.join(map(str, dims))})"},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def replica_seed(rank):
    """each replica (rank) runs its own lattice: distinct hot-start / momentum seeds"""
    return SEED_BASE + 4 + 1000 * rank


def aggregate(elapsed_ms, sites_per_rank, steps, world, device):
    """whole-job throughput from per-rank device times: MAX elapsed over ranks (one all-reduce, outside the
    timed region), value = world x sites x steps / that time.  Returns (value, max_elapsed_ms)."""
    import torch
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return world * sites_per_rank * steps / (t.item() * 1e-3), t.item()


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist

    from paper_1212_0785_b200 import binding as qcd

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    dtype = torch.float64 if args.dtype == "f64" else torch.float32
    rbytes = 8 if args.dtype == "f64" else 4
    dims, beta, eps = cfg["dims"], cfg["beta"], cfg["eps"]
    lat = qcd.Lattice(dims)
    V = lat.V
    U, P = lat.new_matrix_field(dtype), lat.new_matrix_field(dtype)
    qcd.qcd_hot_start(lat, U, replica_seed(rank), cfg["sigma"])
    qcd.qcd_mom_refresh(lat, P, replica_seed(rank))
    stream = torch.cuda.current_stream()

    single = args.path == "single_pass"
    bufs = [U, lat.new_matrix_field(dtype)] if single else [U]

    def step(k, ev=None):
        """one MD step; k counts steps (the single-pass kernel ping-pongs between two gauge fields)"""
        if single:
            if ev:
                ev[0].record(stream)
            qcd.qcd_md_step_single_pass(lat, bufs[k & 1], P, bufs[(k + 1) & 1], beta, eps, eps)
            if ev:
                ev[1].record(stream)
                ev[2].record(stream)
        else:
            if ev:
                ev[0].record(stream)
            qcd.qcd_force_mom_update(lat, U, P, beta, eps)
            if ev:
                ev[1].record(stream)
            qcd.qcd_link_update(lat, P, U, eps, reunit=True)
            if ev:
                ev[2].record(stream)

    # the FMA denominator: register-resident 3x3 complex product chains, measured now
    prec = qcd.F64 if args.dtype == "f64" else qcd.F32
    fma_peak = qcd.probe_rate(qcd.PROBE_FMA, prec)
    fma_src = "measured in this run: qcd_probe_launch(QCD_PROBE_FMA), best of 3, CUDA events"
    time.sleep(2.0)  # let the board cool off the probe (full-power FMA for 0.1 s) before the timed region

    nwarm = args.warmup + (args.warmup & 1 if single else 0)  # even, so the timed steps start from bufs[0]
    for k in range(nwarm):
        step(k)
    try:  # NVML index of this CUDA device (differs from `local` under CUDA_VISIBLE_DEVICES)
        nvml_index = torch.cuda._get_nvml_device_index(local)
    except Exception:  # noqa: BLE001
        nvml_index = local
    sampler = ClockSampler(nvml_index)
    sampler.start()

    # ---- timed region: K fused MD steps, inputs resident in HBM (2 x field >> L2, see config.l2)
    K = args.steps
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
    barrier()
    sampler.active = True
    for k in range(K):
        step(k, ev[k])
    barrier()
    sampler.active = False
    elapsed_ms = ev[0][0].elapsed_time(ev[K - 1][2])
    force_ms = sum(e[0].elapsed_time(e[1]) for e in ev) / K
    link_ms = sum(e[1].elapsed_time(e[2]) for e in ev) / K
    value, elapsed_ms = aggregate(elapsed_ms, V, K, world, "cuda")
    clocks_timed = sampler.summary()

    # ---- the sustained regime (a trajectory lives there: the fp64 step draws the board's full power and the driver
    # lowers the SM clock after a few tenths of a second): a second, longer loop outside the --steps region
    sustained = None
    if args.sustained_steps > 0:
        Ks = args.sustained_steps + (args.sustained_steps & 1 if single else 0)
        sampler.samples, sampler.mask = [], 0
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        sampler.active = True
        s0.record(stream)
        for k in range(Ks):
            step(k)
        s1.record(stream)
        barrier()
        sampler.active = False
        _, sus_ms = aggregate(s0.elapsed_time(s1), V, Ks, world, "cuda")
        sustained = {"steps": Ks, "ms_per_step": sus_ms / Ks, "site_updates_per_s": world * V * Ks / (sus_ms * 1e-3),
                     "clocks": sampler.summary()}

    # ---- e2e: the C-ABI call on HOST buffers (pinned), H2D + pack + step + unpack + D2H every step
    Ke = max(1, min(K, args.e2e_steps))
    fb = lat.field_bytes(qcd.F64 if args.dtype == "f64" else qcd.F32)
    hU = torch.empty(V * 72, dtype=dtype).pin_memory()
    hP = torch.empty(V * 72, dtype=dtype).pin_memory()
    work = torch.empty(lat.md_host_work_bytes(qcd.F64 if args.dtype == "f64" else qcd.F32) // rbytes, dtype=dtype,
                       device="cuda")
    tmp = work[: V * 72]
    qcd.qcd_unpack(lat, 72, qcd.LAYOUT_PAIRS, U, tmp)
    hU.copy_(tmp)
    qcd.qcd_unpack(lat, 72, qcd.LAYOUT_PAIRS, P, tmp)
    hP.copy_(tmp)
    qcd.qcd_md_host(lat, hU, hP, beta, eps, 1, work)  # warm-up
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(Ke):
        qcd.qcd_md_host(lat, hU, hP, beta, eps, 1, work)
        stream.synchronize()  # the caller reads the step's result on the host
    e1.record(stream)
    barrier()
    e2e_value, _ = aggregate(e0.elapsed_time(e1), V, Ke, world, "cuda")
    sampler.stop_flag = True

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = peaks()
    nslab = max(d for d in range(1, 17) if dims[3] % d == 0)  # qcd_md_host: largest divisor of Lt up to 16
    top = "md_step_single_pass" if single else "force_mom_update"
    force_bytes = BYTES_PER_SITE[top] * rbytes * V
    step_bytes = force_bytes if single else 2 * force_bytes
    achieved = force_bytes / (force_ms * 1e-3) / 1e9
    traffic = None
    tp = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    if os.path.exists(tp):
        traffic = json.load(open(tp)).get(f"{top}_{args.dtype}_{cfg['name']}")
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
        "ms_per_step": elapsed_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": f"{cfg['name']} {'fp64' if args.dtype == 'f64' else 'fp32'} fused MD step "
                               f"({'one single-pass kernel' if single else 'force+momentum, exp+reunit'}), sigma={cfg['sigma']} beta={beta} eps={eps}",
                   "sites_per_gpu": V, "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                   "l2": f"inputs U+P = {2 * fb / 1e6:.0f} MB per GPU, larger than the 126 MB L2: no flush needed"
                         if 2 * fb > 2 * 126e6 else "inputs fit L2: numbers are L2-resident, not HBM",
                   "path": args.path,
                   # `value` is the --steps region the contract defines; when that region is shorter than the few
                   # tenths of a second the board takes to reach its power cap it is a boost-clock BURST number, and
                   # the regime a trajectory lives in is config.sustained (and roofline.frac_sustained)
                   "value_regime": ("burst" if elapsed_ms < 300.0 else "sustained")
                                   + f": {K} steps = {elapsed_ms:.0f} ms at a median SM clock of {clocks_timed['sm_mhz']} MHz",
                   "step_hbm_gbs": step_bytes / (elapsed_ms / K * 1e-3) / 1e9,
                   "step_frac_of_hbm_peak": step_bytes / (elapsed_ms / K * 1e-3) / 1e9 / peak,
                   "kernel_ms": {top: force_ms} if single else
                                {"force_mom_update": force_ms, "link_update_reunit": link_ms},
                   "sustained": sustained},
        "roofline": {"bound": "hbm", "kernel": top, "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak,
                     "frac_sustained": None if (sustained is None or not single) else
                                       force_bytes / (sustained["ms_per_step"] * 1e-3) / 1e9 / peak,
                     "traffic": traffic, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": force_bytes,
                     "traffic_source": "stored ncu capture (profiles/roofline_traffic.json names the report), not measured in this run",
                     # the same kernel against the plain-ALU roofline it also sits near: FMA per site x V
                     # / time over the FMA rate the qcd_probe_launch(QCD_PROBE_FMA) kernel reached a moment ago
                     "fma_frac": (FMA_FORCE + FMA_MOM + (FMA_LINK if single else 0)) * V / (force_ms * 1e-3) / fma_peak,
                     "fma_per_site": FMA_FORCE + FMA_MOM + (FMA_LINK if single else 0),
                     "fma_peak": fma_peak, "fma_peak_source": fma_src},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 2 * fb, "d2h_bytes_per_step": 2 * fb,
                "steps": Ke, "call": "qcd_md_host (pinned host buffers, canonical layout; H2D, pack, "
                                     + (f"single-pass step, unpack, D2H pipelined over {nslab} slabs of timeslices on three streams)"
                                        if nslab >= 8 else "two-kernel step, unpack, D2H on one stream: fewer than 8 slabs)")},
        "gpu_launches": K if single else 2 * K,
        "clocks": clocks_timed,
    }
    if world == 1 and not args.no_cpu_baseline:
        from oracle.oracle import Oracle
        orc = Oracle(omp=False)
        sd = pick_sample(orc, cfg, 6, 20.0)
        rate, dt = oracle_step_rate(orc, cfg, sd, 5, 1)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
                                "sample": f"{'x'.join(map(str, sd))} lattice with the {cfg['name']} parameters, "
                                          f"5 fused MD steps of the serial C oracle ({dt:.1f} s)"}
        # the same oracle source built with -fopenmp on all host cores (SURVEY.md 8(d) oracle timing (ii)); extra key
        omp = Oracle(omp=True)
        if omp.num_threads() > 1:
            sd2 = pick_sample(omp, cfg, 6, 10.0)
            rate2, dt2 = oracle_step_rate(omp, cfg, sd2, 5, 1)
            line["cpu_baseline_openmp"] = {"value": rate2, "unit": UNIT, "cores": omp.num_threads(), "kind": "oracle",
                                           "sample": f"{'x'.join(map(str, sd2))} lattice, 5 fused MD steps of the "
                                                     f"OpenMP build of the same oracle ({dt2:.1f} s)"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# per-kernel table: reals per site read + written, FMA per site (products x 108 + small)
KERNEL_TABLE = [
    # name, reals/site, FMA/site, subsets
    ("gauge_force", 144, FMA_FORCE + 40, True),
    ("mom_update", 216, 72, True),
    ("force_mom_update", 216, FMA_FORCE + FMA_MOM, True),
    ("link_update", 216, 4 * 420, True),
    ("reunit", 144, 4 * 100, True),
    ("link_update_reunit", 216, FMA_LINK, True),
    ("mom_refresh", 72, 0, True),
    ("plaquette", 72, 12 * 108 + 6 * 18, False),
    ("sum_norm2", 72, 72, True),
    ("sum_multi_norm2_per_t", 72, 72, False),
    ("md_step_single_pass", 288, FMA_FORCE + FMA_MOM + FMA_LINK, False),
    ("force_mom_update_sums", 216, FMA_FORCE + FMA_MOM + 180, False),
]
FMA_PEAK_NOMINAL = {"f64": 148 * 64 * 1.965e9, "f32": 148 * 128 * 1.965e9}  # lanes x clock


def run_peaks(args):
    """the measured denominators: FMA (fp64, fp32), L1-resident loads, shared memory, L2-resident loads"""
    import torch

    from paper_1212_0785_b200 import binding as qcd
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    out = {"device": torch.cuda.get_device_name(0), "sms": sms}
    for name, what, prec in (("fma_f64_per_s", qcd.PROBE_FMA, qcd.F64), ("fma_f32_per_s", qcd.PROBE_FMA, qcd.F32),
                             ("l1_resident_ldg128_bytes_per_s", qcd.PROBE_L1, qcd.F64),
                             ("shared_lds128_bytes_per_s", qcd.PROBE_LDS, qcd.F64),
                             ("l2_resident_ldg128_bytes_per_s", qcd.PROBE_L2, qcd.F64)):
        time.sleep(0.5)
        out[name] = qcd.probe_rate(what, prec)
    out["nominal_fma_per_s"] = FMA_PEAK_NOMINAL
    out["l1_bytes_per_clk_per_sm_at_1965MHz"] = out["l1_resident_ldg128_bytes_per_s"] / sms / 1.965e9
    out["lds_bytes_per_clk_per_sm_at_1965MHz"] = out["shared_lds128_bytes_per_s"] / sms / 1.965e9
    print(json.dumps({"peaks": out, "how": "qcd_probe_launch through the C ABI, CUDA events, best of 3 per probe"}), flush=True)


def run_slabs(args, cfg):
    """the single-pass step on the lattice cut into --slabs slabs of timeslices in ONE process on one GPU, halos written
    by the step kernel of the neighbouring slab (qcd_md_step_single_pass_push): what the
    decomposition itself costs (halo timeslices, smaller launches, the push stores) with the transport at device-memory
    speed.  One JSON object; not the headline line."""
    import torch

    from paper_1212_0785_b200 import binding as qcd
    from paper_1212_0785_b200 import slabs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dtype = torch.float64 if args.dtype == "f64" else torch.float32
    dims, beta, eps = cfg["dims"], cfg["beta"], cfg["eps"]
    V = dims[0] * dims[1] * dims[2] * dims[3]
    rows = []
    for nslabs, overlap in ((1, False), (args.slabs, False), (args.slabs, True)):
        ss = slabs.SlabSet(qcd, dims, nslabs, dtype)
        ss.start(SEED_BASE + 4, cfg["sigma"])
        ss.leapfrog_single_pass(beta, eps, 4, overlap=overlap)  # warm-up
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        time.sleep(1.0)
        e0.record()
        ss.leapfrog_single_pass(beta, eps, args.steps, overlap=overlap)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        rows.append({"slabs": nslabs, "boundary_first": overlap, "ms_per_step": ms, "site_updates_per_s": V / (ms * 1e-3)})
        del ss
    print(json.dumps({"slab_steps": rows, "config": {"workload": f"{cfg['name']} {args.dtype} leapfrog of single-pass "
                      f"steps with in-kernel halo push, all slabs in one process on one GPU, {args.steps} steps + the "
                      "closing half kick"}}), flush=True)


def run_decompose(args, cfg):
    """--decompose: ONE lattice cut into --gpus slabs of timeslices, one per rank (paper_1212_0785_b200/slabs.py
    DistSlab): the leapfrog step as a multi-GPU job runs it — link update (exp + reunit),
    one halo exchange (two face messages per rank through torch.distributed: NCCL batch_isend_irecv for N > 1, the
    rank's own boundary for N = 1), force + momentum update.  Strong scaling: the lattice is fixed, value = V x steps /
    the slowest rank's device time.  One JSON object; the headline line stays the replica run."""
    import torch
    import torch.distributed as dist

    from paper_1212_0785_b200 import binding as qcd
    from paper_1212_0785_b200 import slabs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    local = local % torch.cuda.device_count() if args.backend == "gloo" else local
    torch.cuda.set_device(local)
    if world > 1 and args.backend == "nccl":
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    elif world > 1:  # gloo: several ranks may share a GPU (faces staged through the host); a functional check only
        dist.init_process_group("gloo")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    dtype = torch.float64 if args.dtype == "f64" else torch.float32
    dims, beta, eps = cfg["dims"], cfg["beta"], cfg["eps"]
    V = dims[0] * dims[1] * dims[2] * dims[3]
    ds = slabs.DistSlab(qcd, dims, slabs.SlabComm(rank, world, dist if world > 1 else None), dtype)
    ds.start(SEED_BASE + 4, cfg["sigma"])  # the generator is keyed on the global site: every rank uses the same seed
    ds.exchange()
    ds.leapfrog(beta, eps, max(args.warmup, 3))
    K = args.steps
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    ds.leapfrog(beta, eps, K)
    e1.record()
    barrier()
    value, ms = aggregate(e0.elapsed_time(e1), V / world, K, world, "cuda")
    plaq, kin, _ = ds.global_observables(beta)  # collective: every rank takes part
    face = ds.face(ds.n, slabs.MASK_ALL).numel() + ds.face(1, slabs.MASK_SPATIAL).numel()
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": f"{cfg['name']} {args.dtype} leapfrog, the lattice cut into {world} slab(s) of "
                                   f"{ds.n} timeslices, one per rank; per step: link update (exp + reunit), one halo "
                                   "exchange, force + momentum update; the timed region also holds the opening half kick",
                       "mode": "decompose", "transport": "own boundary (one rank)" if world == 1 else "NCCL batch_isend_irecv" if args.backend == "nccl"
                                    else "gloo through host memory (functional check, not a measurement)",
                       "sent_bytes_per_rank_per_step": face * (8 if args.dtype == "f64" else 4)},
            "plaquette": plaq, "kinetic_energy": kin}), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_per_kernel(args, cfg):
    """each kernel alone on ALL / EVEN / ODD with an L2 flush between timed launches (config 3's U + P is about the
    size of L2); one JSON line with a list of rows"""
    import torch

    from paper_1212_0785_b200 import binding as qcd
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dtype = torch.float64 if args.dtype == "f64" else torch.float32
    rb = 8 if args.dtype == "f64" else 4
    dims, beta, eps = cfg["dims"], cfg["beta"], cfg["eps"]
    lat = qcd.Lattice(dims)
    V = lat.V
    U, P, F, W = (lat.new_matrix_field(dtype) for _ in range(4))
    ws = lat.new_workspace()
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    per_t = torch.zeros(dims[3], dtype=torch.float64, device="cuda")
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")  # 4 x L2
    peak, peak_src = peaks()
    fma_peak = qcd.probe_rate(qcd.PROBE_FMA, qcd.F64 if args.dtype == "f64" else qcd.F32)
    stream = torch.cuda.current_stream()

    def reset():
        qcd.qcd_hot_start(lat, U, SEED_BASE + args.config, cfg["sigma"])
        qcd.qcd_perturb(lat, U, SEED_BASE + args.config, 1e-3)  # config 3: reunit input off SU(3) by sigma = 1e-3
        qcd.qcd_mom_refresh(lat, P, SEED_BASE + args.config)
        qcd.qcd_mom_refresh(lat, F, SEED_BASE + args.config, stream_id=1)

    calls = {
        "gauge_force": lambda sub: qcd.qcd_gauge_force(lat, U, F, beta, subset=sub),
        "mom_update": lambda sub: qcd.qcd_mom_update(lat, F, P, eps, subset=sub),
        "force_mom_update": lambda sub: qcd.qcd_force_mom_update(lat, U, P, beta, eps, subset=sub),
        "link_update": lambda sub: qcd.qcd_link_update(lat, P, U, eps, reunit=False, subset=sub),
        "reunit": lambda sub: qcd.qcd_reunit(lat, U, subset=sub),
        "link_update_reunit": lambda sub: qcd.qcd_link_update(lat, P, U, eps, reunit=True, subset=sub),
        "mom_refresh": lambda sub: qcd.qcd_mom_refresh(lat, P, SEED_BASE, subset=sub),
        "plaquette": lambda sub: qcd.qcd_plaquette(lat, U, out[0:1], per_t, ws),
        "sum_norm2": lambda sub: qcd.qcd_sum(lat, qcd.SUM_NORM2, 72, P, out[1:2], ws, subset=sub),
        "sum_multi_norm2_per_t": lambda sub: qcd.qcd_sum_multi(lat, qcd.SUM_NORM2, 72, P, None, dims[3], per_t, ws),
        "md_step_single_pass": lambda sub: qcd.qcd_md_step_single_pass(lat, U, P, W, beta, eps, eps),
        "force_mom_update_sums": lambda sub: qcd.qcd_force_mom_update_sums(lat, U, P, beta, eps, out, ws),
    }
    rows = []
    reps = max(5, min(args.steps, 20))
    for name, reals, fma, has_subsets in KERNEL_TABLE:
        for sub, sname in ((qcd.ALL, "all"), (qcd.EVEN, "even"), (qcd.ODD, "odd")):
            if sub != qcd.ALL and not has_subsets:
                continue
            reset()
            fn = calls[name]
            for _ in range(3):
                fn(sub)
            ts = []
            for _ in range(reps):
                flush.fill_(1)  # evict the fields from L2
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                fn(sub)
                e1.record(stream)
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            ts.sort()
            ms = ts[len(ts) // 2]
            sites = V if sub == qcd.ALL else V // 2
            gbs = reals * rb * sites / (ms * 1e-3) / 1e9
            rows.append({"kernel": name, "subset": sname, "ms": ms, "bytes_per_site": reals * rb, "gbs": gbs,
                         "frac_hbm": gbs / peak, "site_updates_per_s": sites / (ms * 1e-3),
                         "frac_fma": fma * sites / (ms * 1e-3) / fma_peak})
    print(json.dumps({"per_kernel": rows, "config": {"workload": f"{cfg['name']} {args.dtype}, each kernel alone, "
                      "L2 flushed (512 MB write) before every timed launch", "reps": reps},
                      "peak_gbs": peak, "peak_source": peak_src, "fma_peak": fma_peak,
                      "fma_peak_source": "qcd_probe_launch(QCD_PROBE_FMA), measured in this run"}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=sorted(CONFIGS))
    ap.add_argument("--dims", default=None,
                    help="Lx,Ly,Lz,Lt: another lattice shape with the parameters of --config (shape studies; the "
                         "headline workload is the default)")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--path", default="single_pass", choices=["two_kernel", "single_pass"],
                    help="single_pass (default, the faster one as measured): qcd_md_step_single_pass ping-ponging two "
                         "gauge fields; two_kernel: qcd_force_mom_update + qcd_link_update(reunit) in place")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--sustained-steps", type=int, default=600,
                    help="length of the second timed loop that reports the power-capped regime (0: skip)")
    ap.add_argument("--peaks", action="store_true",
                    help="measure the FMA / L1 / shared-memory / L2 denominators with the library's probe kernels")
    ap.add_argument("--slabs", type=int, default=0,
                    help="instead of the MD-step line: the step on the lattice cut into this many slabs of timeslices in one "
                         "process (in-kernel halo push), against the undecomposed step")
    ap.add_argument("--decompose", action="store_true",
                    help="instead of the MD-step line: ONE lattice cut into --gpus slabs of timeslices, one per rank, halo "
                         "faces exchanged through torch.distributed (strong scaling; the default N > 1 run is replicas)")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="--decompose only: gloo lets several ranks share one GPU (faces staged through host memory) to "
                         "check the N > 1 code path on a one-GPU box; its timings are not measurements")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--per-kernel", action="store_true",
                    help="instead of the MD-step line: every kernel alone on ALL/EVEN/ODD with an L2 flush between "
                         "launches (SURVEY.md 8(d), config 3 row); prints one JSON object with the table")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    cfg = dict(CONFIGS[args.config])
    if args.dims:
        cfg["dims"] = tuple(int(x) for x in args.dims.split(","))
        cfg["name"] = "x".join(str(d) for d in cfg["dims"])
    if args.impl == "reference":
        run_reference(args, cfg)
    elif args.peaks:
        run_peaks(args)
    elif args.decompose:
        run_decompose(args, cfg)
    elif args.slabs > 0:
        run_slabs(args, cfg)
    elif args.per_kernel:
        run_per_kernel(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
