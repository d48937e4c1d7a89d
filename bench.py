#!/usr/bin/env python
"""bench.py -- D_tm GFLOPS (1320 flop/site) and HBM GB/s of the even-odd twisted-mass hot path.

Workload (BASELINE.json configs[4], the configuration the metric is quoted on):
32^3 x 64 lattice, complex double, Haar-random SU(3) links, Gaussian source,
kappa = 0.15, mu = 0.1, antiperiodic in time; synthetic seeded inputs
(lqcd_inputs).

One step = one CG iteration on Mhat^dag Mhat:
four hopping launches with fused diagonal-term epilogues (the second with the fused
<p,Ap> partial sums, the fourth applying r -= alpha q in place with the |r|^2 partial
sums) + the fused x/p vector kernel + two one-block finalisation kernels (7 launches).  K steps are run as solves of
SOLVE_LEN iterations each (a real solve at this configuration takes about that
many), the one-launch solve setup included in the timed region; the recursive
residual would otherwise underflow after several hundred iterations.

value   = hopping flops (4 x V/2 x 1320 per step; diagonal and vector-kernel
          flops NOT counted) / time, inputs resident in HBM.
roofline= the hopping kernel.  frac = the plain-epilogue launches (two of the four per step), whose algorithmic
          bytes are exactly SURVEY section 8(d)'s 1536 B per output site, / their CUDA-event durations, recorded live by
          the library (lqcd_profile) on one solve in five of the timed region (an event pair around EVERY launch costs
          2.6% of the step, measured, so the other solves run without them and replay the cached CUDA graph); a timed
          region of fewer than five solves (the driver's --steps 20) runs entirely without event pairs and one extra
          solve right after it is the profiled one.  roofline.all_hopping_launches gives the figure over all four
          launches under each byte count one can book to them; roofline.traffic is a constant from a committed ncu
          capture (traffic_source), not measured here.
sustained= after the timed region the same steps run again for >= 2 s (power cap reached, SM clock settled) with
          their own clocks, ms per step, GFLOPS and roofline fraction: a 25 ms timed region is a burst figure.
e2e     = the same per-step work through lqcd_cg_mdagm_host with pinned HOST
          buffers: every step uploads gauge + source, runs one CG iteration (plus
          the solve's true-residual check, not counted as flops) and downloads x.
roofline.stream_probe_gbs = what lqcd_stream_probe (the paper's copy micro-benchmark, Fig. 5) moves on this
          box in the same run: copy, read-only and 7 reads : 1 write on 16-byte elements (context for frac).
--impl reference times the CPU oracle (oracle/, test infrastructure) on the host cores.
--scaling strong (not the contract's arm, which is N independent replicas): the ONE lattice split over the N ranks
          along t (lqcd_slab_*), a step = one CG iteration of binding.slab_cg with its halo exchanges and all-reduces.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_SITE = 1320          # BASELINE.json metric; SURVEY.md section 8(a) row a5
BYTES_PER_SITE = 1536         # double, 18-real links: 8 links x 144 + 192 in + 192 out (section 8(d))
AUX_BYTES_PER_SITE = 192      # launches with the M_ee * aux epilogue read one more half spinor
# the last hopping launch of an iteration (fused r -= alpha q, |r|^2): 8 links + in + aux + r read + r write
FUSED_R_BYTES_PER_SITE = 8 * 144 + 4 * 192
# whole CG iteration: 3 x (1536 [+192 aux on one]) + fused-r launch + cg_update_xp (x, p, r read; x, p written)
STEP_BYTES_PER_SITE = 3 * BYTES_PER_SITE + AUX_BYTES_PER_SITE + FUSED_R_BYTES_PER_SITE + 5 * 192
DIMS = (32, 32, 32, 64)
REF_DIMS = (16, 16, 16, 32)   # bounded sample for the oracle legs (same recipe, 1/16 of the sites)
REF_DIMS_SMALL = (8, 8, 8, 16)  # used by --impl reference when K + W > 100 steps are asked for
KAPPA, MU = 0.15, 0.1
SOLVE_LEN = 40
PROFILE_EVERY = 5              # per-launch events on one solve in five of the timed region
CPU_BASELINE_STEPS = 8         # oracle leg of the default run on all cores: ~7 s on the workload itself ...
CPU_BASELINE_STEPS_1T = 1      # ... and one application single-threaded (~14 s): SURVEY.md section 8(d)
SUSTAINED_MS = 2000.0          # the `sustained` leg runs the same steps for at least this long
REFERENCE_BUDGET_S = 240.0     # --impl reference stays on the workload's own lattice while K + W steps fit this
METRIC = "D_tm GFLOPS (1320 flop/site) & achieved HBM GB/s vs B200 peak, double"
# dram__bytes_read.sum + dram__bytes_write.sum per PLAIN hopping launch (MODE 0, exactly 1536 B/site algorithmic =
# 1.610613 GB) at this workload, from the committed `ncu --set full` capture named in NCU_TRAFFIC_SOURCE; a constant
# typed in from that file, NOT measured in this run -- refreshed whenever the hopping kernel changes.
NCU_TRAFFIC_BYTES_PER_LAUNCH = 1586016000
NCU_TRAFFIC_SOURCE = ("profiles/r02_hopping_staged.md, section 'The branch per hop' (ncu --set full of the default kernel "
                      "hopping_kernel<double,18,0,0,...,REALPH>, raw page in profiles/r02z_hop_default_raw.csv): "
                      "dram__bytes_read 1.415661 GB + dram__bytes_write 0.170355 GB")


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (pynvml, else nvidia-smi)."""

    def __init__(self, index):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None

    def _run_nvml(self):
        import pynvml as nv
        nv.nvmlInit()
        h = nv.nvmlDeviceGetHandleByIndex(self.index)
        self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
        names = {
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
            nv.nvmlDeviceGetCurrentClocksThrottleReasons
        while not self._stop.is_set():
            self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
            r = get_reasons(h)
            for bit, name in names.items():
                if r & bit:
                    self.reasons.add(name)
            time.sleep(0.005)

    def _run_smi(self):
        import subprocess
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
            "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        keys = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        while not self._stop.is_set():
            out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={q}",
                                  "--format=csv,noheader,nounits"], capture_output=True, text=True).stdout
            f = [s.strip() for s in out.strip().split(",")]
            if len(f) >= 6:
                self.samples.append(float(f[0]))
                self.max_mhz = float(f[1])
                for k, v in zip(keys, f[2:6]):
                    if v.lower().startswith("active"):
                        self.reasons.add(k)

    def _run(self):
        try:
            self._run_nvml()
        except Exception:
            try:
                self._run_smi()
            except Exception:
                pass

    def __enter__(self):
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._thr.join(timeout=5)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def oracle_gflops(dims, steps, warmup, U=None, x=None):
    """Oracle as it stands: one application of Mhat^dag Mhat (4 hopping terms = one CG iteration's
    operator work) per step on the host cores; returns (gflops, ms_per_step, threads).  U, x: the
    seeded inputs if the caller has them already (generating 32^3 x 64 links takes ~20 s)."""
    import lqcd_inputs as gen
    import oracle
    oracle.build()
    Vh = int(np.prod(dims)) // 2
    if U is None:
        U = gen.gauge_haar(dims)
    if x is None:
        x = gen.spinor_gaussian(Vh, stream=gen.STREAM_SOURCE)
    ph = gen.antiperiodic_t()
    for _ in range(warmup):
        oracle.mdagm(dims, ph, U, x, KAPPA, MU)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.mdagm(dims, ph, U, x, KAPPA, MU)
    dt = (time.perf_counter() - t0) / steps
    return 4 * Vh * FLOP_PER_SITE / dt / 1e9, dt * 1e3, oracle.num_threads()


def max_over_ranks(x, world, device):
    """Max of a per-rank scalar over all ranks (the contract's max-over-ranks timing)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gflops(world, steps, sites_per_rank, ms_max):
    """Replicas only: every rank does `steps` steps on its own lattice; whole-job rate."""
    return world * steps * 4 * sites_per_rank * FLOP_PER_SITE / (ms_max * 1e-3) / 1e9


def run_reference(args, rank):
    """The CPU oracle as the reference arm: one application of Mhat^dag Mhat per step on the host cores, on the
    workload's own 32^3 x 64 lattice whenever K + W steps of it fit REFERENCE_BUDGET_S (one application is timed
    first), else on a bounded 16^3 x 32 / 8^3 x 16 sample of the same recipe -- and then `config` says so."""
    if rank != 0:
        return
    import lqcd_inputs as gen
    import oracle
    oracle.build()
    n = args.steps + args.warmup
    cfg = workload_config()
    dims, U, x = DIMS, gen.gauge_haar(DIMS), gen.spinor_gaussian(int(np.prod(DIMS)) // 2, stream=gen.STREAM_SOURCE)
    t0 = time.perf_counter()
    oracle.mdagm(dims, gen.antiperiodic_t(), U, x, KAPPA, MU)
    t1 = time.perf_counter() - t0
    if n * t1 > REFERENCE_BUDGET_S:
        dims = REF_DIMS if n * t1 / 16 <= REFERENCE_BUDGET_S else REF_DIMS_SMALL
        U = x = None
        cfg["reference_lattice"] = (f"{'x'.join(map(str, dims))} sample of the same recipe: {n} steps of the oracle at "
                                    f"{t1:.2f} s each on the workload's own lattice exceed {REFERENCE_BUDGET_S:.0f} s")
    gf, ms, threads = oracle_gflops(dims, args.steps, args.warmup, U, x)
    sample = (f"oracle Mhat^dag Mhat (4 hopping terms = the operator work of one step) per step on "
              + ("the workload's own 32x32x32x64 lattice, links and source" if dims == DIMS else
                 f"a {'x'.join(map(str, dims))} lattice of the same recipe ({np.prod(dims) / np.prod(DIMS):.4f} of the workload's sites)")
              + ", OpenMP over sites; a plain test oracle, not a tuned CPU code")
    line = {
        "impl": "reference", "metric": METRIC, "value": gf, "unit": "GFLOPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": cfg,
        "cpu_baseline": {"value": gf, "unit": "GFLOPS", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": gf, "unit": "GFLOPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config():
    return {"workload": "32^3x64 complex double, Haar SU(3) links, Gaussian source, kappa=0.15 mu=0.1, "
                        "antiperiodic t; one step = one CG iteration on Mhat^dag Mhat (4 hopping launches, the last with the fused r-update, + 1 vector + 2 one-block finalise launches)",
            "lattice": list(DIMS), "precision": "double", "recon": 18, "kappa": KAPPA, "mu": MU,
            "solve_len": SOLVE_LEN,
            "l2": "inputs larger than L2 (gauge 1.21 GB + 6 half spinors of 201 MB per step vs 126 MB L2)"}


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    import lqcd_inputs as gen
    import paper_1209_5942_b200.binding as B

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    Vh = int(np.prod(DIMS)) // 2
    ph = gen.antiperiodic_t()
    # "replicas only": every rank solves its own seeded system of the same shape
    seed = gen.BASE_SEED + rank
    U = gen.gauge_haar(DIMS, seed)
    b = gen.spinor_gaussian(Vh, seed, gen.STREAM_SOURCE)

    B.lqcd_init(DIMS, ph)
    stream = torch.cuda.Stream()
    B.lqcd_set_stream(stream)
    with torch.cuda.stream(stream):
        g = B.upload_gauge(U)
        src = B.upload_spinor(b, 0)
        x = B.alloc_spinor()
    stream.synchronize()

    def run_steps(n, sample_profile=False):
        """n steps as solves of SOLVE_LEN iterations.  sample_profile: the library's per-launch event pairs are
        recorded on one solve in PROFILE_EVERY (recording every launch costs 2.6% of the step); returns the
        (event, event, steps) brackets of those solves."""
        done, idx, marks = 0, 0, []
        while done < n:
            k = min(SOLVE_LEN, n - done)
            prof_this = sample_profile and idx % PROFILE_EVERY == 0
            if prof_this:
                ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                ea.record(stream)
                B.lqcd_profile(2)
            B.lqcd_cg_setup(g, src, x, KAPPA, MU, 0.0)
            B.lqcd_cg_iterate(k)
            if prof_this:
                B.lqcd_profile(0)
                eb.record(stream)
                marks.append((ea, eb, k))
            done += k
            idx += 1
        return marks

    peak, peak_src = measured_peak()

    def measure(n_steps):
        """One timed region of n_steps steps: CUDA events on the library's stream around the whole region, clocks
        sampled inside it, per-launch event pairs on one solve in PROFILE_EVERY when the region holds that many."""
        sample = -(-n_steps // SOLVE_LEN) >= PROFILE_EVERY
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        B.lqcd_profile(1)      # discard earlier records ...
        B.lqcd_profile(0)      # ... and record only inside the sampled solves of this region
        n0 = B.lqcd_launch_count()
        barrier()
        with ClockSampler(local_rank) as clk:
            e0.record(stream)
            marks = run_steps(n_steps, sample_profile=sample)
            e1.record(stream)
            stream.synchronize()
        barrier()
        m = {"steps": n_steps, "launches": int(B.lqcd_launch_count() - n0), "ms_total": e0.elapsed_time(e1),
             "clocks": clk.summary(), "prof": {c: B.lqcd_profile_read(c) for c in range(6)},
             "ms_sampled": sum(a.elapsed_time(b_) for a, b_, _ in marks), "steps_sampled": sum(k for _, _, k in marks),
             "solves_sampled": len(marks)}
        st = B.lqcd_cg_finish()
        iters, _, _ = B.lqcd_cg_stats()
        last = n_steps % SOLVE_LEN or min(SOLVE_LEN, n_steps)
        if iters != last or st < 0:
            raise SystemExit(f"bench: the last solve ran {iters} iterations, expected {last} (status {st})")
        return m

    def profile_one_solve():
        """Per-launch event pairs on ONE extra solve of SOLVE_LEN steps (for regions too short to sample)."""
        B.lqcd_profile(1)
        B.lqcd_profile(0)
        ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ea.record(stream)
        B.lqcd_profile(2)
        B.lqcd_cg_setup(g, src, x, KAPPA, MU, 0.0)
        B.lqcd_cg_iterate(SOLVE_LEN)
        B.lqcd_profile(0)
        eb.record(stream)
        stream.synchronize()
        B.lqcd_cg_finish()
        return {"prof": {c: B.lqcd_profile_read(c) for c in range(6)}, "ms_sampled": ea.elapsed_time(eb),
                "steps_sampled": SOLVE_LEN, "solves_sampled": 1}

    def hopping_roofline(m, where):
        """roofline of the hopping kernel from per-launch CUDA events.  frac: the plain-epilogue launches (MODE 0,
        two of the four per step), whose algorithmic bytes are exactly section 8(d)'s 1536 B per output site; the
        figure over all four launches is given with each of the byte counts one can book to them."""
        prof = m["prof"]
        hop_ms = prof[0][0] + prof[1][0] + prof[2][0] + prof[5][0]
        hop_n = prof[0][1] + prof[1][1] + prof[2][1] + prof[5][1]
        iters = prof[5][1]
        plain_ms, plain_n = prof[0]
        achieved = Vh * BYTES_PER_SITE * plain_n / (plain_ms * 1e-3) / 1e9
        full_bytes = Vh * (BYTES_PER_SITE * (hop_n - iters) + AUX_BYTES_PER_SITE * (prof[1][1] + prof[2][1])
                           + FUSED_R_BYTES_PER_SITE * iters)
        gbs = lambda nbytes: nbytes / (hop_ms * 1e-3) / 1e9
        return {
            "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH, "traffic_source": NCU_TRAFFIC_SOURCE, "peak_source": peak_src,
            "frac_of_nominal_8000": achieved / 8000.0,
            "kernel": "hopping_kernel<double,18,*,0> (the plain-epilogue launches: 2 of the 4 hopping launches of a step)",
            "launches": plain_n, "avg_launch_us": plain_ms / plain_n * 1e3,
            "algorithmic_bytes_per_launch": Vh * BYTES_PER_SITE,
            "plain_epilogue_gflops": Vh * FLOP_PER_SITE * plain_n / (plain_ms * 1e-3) / 1e9,
            "all_hopping_launches": {
                "launches": hop_n, "avg_launch_us": hop_ms / hop_n * 1e3,
                "gbs_with_fused_reads": gbs(full_bytes), "frac_with_fused_reads": gbs(full_bytes) / peak,
                "bytes_with_fused_reads": "3 x 1536 + 192 (aux of the <p,Ap> launch) + 1920 (fused r -= alpha q launch: 8 links, in, aux, r read, r written) = 6720 B per site and step",
                "gbs_a9": gbs(Vh * 6528 * iters), "frac_a9": gbs(Vh * 6528 * iters) / peak,
                "bytes_a9": "SURVEY section 8(a) a9: 4 x 1536 + 2 x 192 = 6528 B per site and step",
                "gbs_1536_each": gbs(Vh * BYTES_PER_SITE * hop_n), "frac_1536_each": gbs(Vh * BYTES_PER_SITE * hop_n) / peak,
            },
            "share_of_step": hop_ms / m["ms_sampled"],
            "vector_kernels_share_of_step": prof[3][0] / m["ms_sampled"],
            "sampled": f"{where}: event pairs around every launch of {m['solves_sampled']} solve(s), {m['steps_sampled']} steps, "
                       f"{m['ms_sampled'] / m['steps_sampled']:.4f} ms per step there (direct launches; solves without event pairs "
                       f"replay four iterations at a time as the library's cached CUDA graph)",
        }

    # ---- device-resident timing -------------------------------------------------------------
    run_steps(args.warmup)
    stream.synchronize()
    m = measure(args.steps)
    launches = m["launches"]
    ms_max = max_over_ranks(m["ms_total"], world, "cuda")
    ms_per_step = ms_max / args.steps
    value = whole_job_gflops(world, args.steps, Vh, ms_max)
    if m["solves_sampled"]:
        roofline = hopping_roofline(m, f"inside the timed region of {args.steps} steps")
    else:   # too short to sample one solve in PROFILE_EVERY: the timed region stays free of event pairs
        roofline = hopping_roofline(profile_one_solve(), "one extra solve right after the timed region (which ran without event pairs)")
    achieved = roofline["achieved"]

    # ---- sustained: the same steps for >= SUSTAINED_MS, so that a short (burst-clock) timed region is not read as it
    n_sus = max(args.steps, int(np.ceil(SUSTAINED_MS / ms_per_step)), PROFILE_EVERY * SOLVE_LEN)
    n_sus = -(-n_sus // SOLVE_LEN) * SOLVE_LEN
    ms_ = measure(n_sus)
    sus_ms = max_over_ranks(ms_["ms_total"], world, "cuda")
    sus_roof = hopping_roofline(ms_, f"inside the sustained leg of {n_sus} steps")
    sustained = {
        "steps": n_sus, "seconds": sus_ms * 1e-3, "ms_per_step": sus_ms / n_sus,
        "value": whole_job_gflops(world, n_sus, Vh, sus_ms), "unit": "GFLOPS", "clocks": ms_["clocks"],
        "gbs_effective_step": world * n_sus * Vh * STEP_BYTES_PER_SITE / (sus_ms * 1e-3) / 1e9,
        "roofline_frac": sus_roof["frac"], "roofline_achieved": sus_roof["achieved"],
        "roofline_avg_launch_us": sus_roof["avg_launch_us"], "all_hopping_launches": sus_roof["all_hopping_launches"],
        "share_of_step": sus_roof["share_of_step"],
        "note": "the timed region above is the contract's K steps; this leg repeats the same steps back to back for at least "
                f"{SUSTAINED_MS / 1e3:.0f} s, where the board sits at its power cap (sw_power_cap) and the SM clock settles",
    }

    line = {
        "metric": METRIC, "value": value, "unit": "GFLOPS", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(),
        "clocks": m["clocks"], "gpu_launches": int(launches), "roofline": roofline,
        "timed_region_seconds": ms_max * 1e-3,
        "timed_region_kind": "burst (shorter than 1 s: the board has not reached its power cap; see `sustained`)" if ms_max < 1000.0
                             else "sustained (>= 1 s under load)",
        "sustained": sustained,
        # whole-step algorithmic bytes (STEP_BYTES_PER_SITE above)
        "gbs_effective_step": world * args.steps * Vh * STEP_BYTES_PER_SITE / (ms_max * 1e-3) / 1e9,
    }

    # ---- end to end through the host-buffer C-ABI call (pinned host memory) -----------------
    n_e2e = max(1, min(args.e2e_steps, args.steps))
    U_pin = torch.from_numpy(U).pin_memory()
    b_pin = torch.from_numpy(b).pin_memory()
    x_pin = torch.empty((Vh, 4, 3), dtype=torch.complex128).pin_memory()
    for _ in range(2):
        B.lqcd_cg_mdagm_host(U_pin, b_pin, x_pin, KAPPA, MU, 0.0, 1)
    barrier()
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        B.lqcd_cg_mdagm_host(U_pin, b_pin, x_pin, KAPPA, MU, 0.0, 1)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    barrier()
    dt = max_over_ranks(dt, world, "cuda")
    # the amortised figure a user sees: one upload, a whole solve to 1e-10, one download
    t0 = time.perf_counter()
    st = B.lqcd_cg_mdagm_host(U_pin, b_pin, x_pin, KAPPA, MU, 1e-10, 2000)
    dt_solve = time.perf_counter() - t0
    it_solve, rr, rt = B.lqcd_cg_stats()
    line["e2e"] = {
        "value": whole_job_gflops(world, n_e2e, Vh, dt * 1e3), "unit": "GFLOPS",
        "h2d_bytes_per_step": int(U_pin.numel() * 16 + b_pin.numel() * 16),
        "d2h_bytes_per_step": int(x_pin.numel() * 16), "steps": n_e2e, "ms_per_step": dt / n_e2e * 1e3,
        "call": "lqcd_cg_mdagm_host(maxit=1): upload gauge+source, pack, 1 CG iteration (+ true-residual check, "
                "not counted), unpack, download x",
        "solve": {"call": "lqcd_cg_mdagm_host(tol=1e-10)", "status": int(st), "iterations": it_solve,
                  "seconds": dt_solve, "true_rel_resid": rt,
                  "gflops": world * it_solve * 4 * Vh * FLOP_PER_SITE / dt_solve / 1e9},
    }
    del U_pin

    # ---- what the memory system of THIS box does on a pure stream (lqcd_stream_probe, 16-byte elements,
    # 1.06 GB read per launch): context for roofline.frac, whose peak stays the driver's measured memcpy figure
    nb = 12096 * 87500
    with torch.cuda.stream(stream):
        ps = torch.randint(0, 256, (nb,), dtype=torch.uint8, device="cuda")
        pd = torch.empty(nb, dtype=torch.uint8, device="cuda")
        ceil = {}
        for name, mode, moved in (("copy", B.LQCD_STREAM_COPY, 2 * nb), ("read", B.LQCD_STREAM_READ, nb),
                                  ("mix_7_reads_1_write", B.LQCD_STREAM_MIX71, nb + nb // 7)):
            for _ in range(3):
                B.lqcd_stream_probe(B.LQCD_ELEM_VEC16, mode, ps, pd, nb)
            p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            p0.record(stream)
            for _ in range(10):
                B.lqcd_stream_probe(B.LQCD_ELEM_VEC16, mode, ps, pd, nb)
            p1.record(stream)
            stream.synchronize()
            ceil[name] = moved * 10 / (p0.elapsed_time(p1) * 1e-3) / 1e9
        # the same 7:1 stream kept up for >= 1 s, with its own clock record: what a pure stream holds on this box when
        # it runs as long as the sustained leg did (it draws less power than the hopping kernel, so its clock stays higher)
        n_probe = max(10, int(1000.0 / ((nb + nb // 7) / ceil["mix_7_reads_1_write"] / 1e6)))
        with ClockSampler(local_rank) as pclk:
            p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            p0.record(stream)
            for _ in range(n_probe):
                B.lqcd_stream_probe(B.LQCD_ELEM_VEC16, B.LQCD_STREAM_MIX71, ps, pd, nb)
            p1.record(stream)
            stream.synchronize()
        mix_sustained = (nb + nb // 7) * n_probe / (p0.elapsed_time(p1) * 1e-3) / 1e9
        del ps, pd
    roofline["stream_probe_gbs"] = ceil
    roofline["frac_of_stream_mix"] = achieved / ceil["mix_7_reads_1_write"]
    roofline["frac_note"] = ("frac is against MEASURED_PEAKS.json's copy bandwidth (1 read : 1 write); the plain hopping launch is "
                             "7 reads : 1 write, which the same-run stream probe moves at mix_7_reads_1_write GB/s, so a burst "
                             "at the maximum clock can read slightly above 1 -- frac_of_stream_mix is the same figure against that probe")
    sustained["frac_of_stream_mix"] = sustained["roofline_achieved"] / ceil["mix_7_reads_1_write"]
    sustained["stream_mix_sustained"] = {"gbs": mix_sustained, "launches": n_probe, "seconds": p0.elapsed_time(p1) * 1e-3,
                                         "clocks": pclk.summary(),
                                         "frac_of_it": sustained["roofline_achieved"] / mix_sustained}

    # ---- oracle on the host cores beside it (rank 0, N = 1 only) ------------------------------
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        # the workload itself (same links, same source): all cores, then one thread
        gf, ms, threads = oracle_gflops(DIMS, CPU_BASELINE_STEPS, 1, U, b)
        oracle.set_num_threads(1)
        gf1, ms1, threads1 = oracle_gflops(DIMS, CPU_BASELINE_STEPS_1T, 0, U, b)
        oracle.set_num_threads(0)
        line["cpu_baseline"] = {
            "value": gf, "unit": "GFLOPS", "cores": threads, "kind": "oracle",
            "sample": f"{CPU_BASELINE_STEPS} applications of the oracle's Mhat^dag Mhat (4 hopping terms each = the operator "
                      f"work of one step) on the workload's own {'x'.join(map(str, DIMS))} lattice, links and source; "
                      f"{ms:.0f} ms per application on {threads} threads; a plain test oracle, not a tuned CPU code",
            "single_thread": {"value": gf1, "unit": "GFLOPS", "cores": threads1, "ms_per_application": ms1,
                              "sample": f"{CPU_BASELINE_STEPS_1T} application of the same call with OpenMP held to one thread"}}
    if rank == 0:
        print(json.dumps(line), flush=True)
    B.lqcd_finalize()
    if world > 1:
        dist.destroy_process_group()


def run_strong(args, rank, world, local_rank):
    """--scaling strong: ONE 32^3 x 64 lattice, its time direction split over the N ranks (lqcd_slab_*, DESIGN.md
    section 7); a step is one CG iteration of binding.slab_cg: four hopping stages, each behind the halo exchange of
    its input field (two blocks per direction, NCCL point-to-point on the library's stream), and two all-reduces of one
    double.  The default arm (replicas) is what BASELINE.json's north_star fixes; this arm exists so that a multi-GPU run
    measures the decomposition.  N = 1 runs the same stages with the rank as its own neighbour."""
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    if DIMS[3] % world or (DIMS[3] // world) % 2:
        raise SystemExit(f"--scaling strong: {world} ranks do not divide N_t = {DIMS[3]} into even slabs")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")      # which transport carried the halos: say so in the log
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    import lqcd_inputs as gen
    import paper_1209_5942_b200.binding as B

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    Vh = int(np.prod(DIMS)) // 2
    ph = gen.antiperiodic_t()
    U = gen.gauge_haar(DIMS, gen.BASE_SEED)                           # the same global field on every rank ...
    b = gen.spinor_gaussian(Vh, gen.BASE_SEED, gen.STREAM_SOURCE)
    s3 = DIMS[0] * DIMS[1] * DIMS[2]
    nt = DIMS[3] // world
    lo, hi = rank * nt * s3, (rank + 1) * nt * s3                      # ... of which this rank keeps its time slab
    B.lqcd_slab_init(DIMS, ph, rank, world)
    stream = torch.cuda.Stream()
    B.lqcd_set_stream(stream)
    with torch.cuda.stream(stream):
        g = B.upload_gauge(U[lo:hi])
        B.slab_exchange_gauge(g, rank, world)
        src = B.upload_spinor(b[lo // 2:hi // 2], 0)
        x = B.alloc_spinor()
    stream.synchronize()
    del U

    def run_steps(n):
        done = 0
        with torch.cuda.stream(stream):
            while done < n:
                k = min(SOLVE_LEN, n - done)
                st = B.slab_cg(g, src, x, KAPPA, MU, 0.0, k, rank, world, overlap=args.overlap, check_every=SOLVE_LEN)
                if st < 0:
                    raise SystemExit(f"bench: slab_cg status {st}")
                done += k

    run_steps(args.warmup)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = B.lqcd_launch_count()
    barrier()
    with ClockSampler(local_rank) as clk:
        e0.record(stream)
        run_steps(args.steps)
        e1.record(stream)
        stream.synchronize()
    barrier()
    launches = max_over_ranks(B.lqcd_launch_count() - n0, world, "cuda")
    ms_max = max_over_ranks(e0.elapsed_time(e1), world, "cuda")
    iters, rr, rt = B.lqcd_cg_stats()
    h = B.lqcd_slab_spinor_halo()
    value = args.steps * 4 * Vh * FLOP_PER_SITE / (ms_max * 1e-3) / 1e9        # the whole lattice, all ranks together
    cfg = workload_config()
    cfg["workload"] = cfg["workload"].replace("one step = one CG iteration", f"time direction split over {world} rank(s) "
                                              f"(slabs of {nt} slices); one step = one CG iteration of binding.slab_cg")
    cfg.update({"ranks": world, "local_lattice": list(DIMS[:3]) + [nt], "overlap_interior_with_halo": bool(args.overlap),
                "halo_bytes_sent_per_rank_and_hopping_stage": 2 * int(h["bytes"]),
                "note": "each solve of %d iterations also pays its setup and the true-residual check (one more "
                        "application of Mhat^dag Mhat) inside the timed region; stages are issued from Python, ~30 calls per "
                        "iteration, so small slabs are launch bound (a native driver is future work)" % SOLVE_LEN})
    line = {"metric": METRIC, "value": value, "unit": "GFLOPS", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": cfg, "clocks": clk.summary(), "gpu_launches": int(launches),
            "last_solve": {"iterations": iters, "rel_resid_recursive": rr, "rel_resid_true": rt},
            "gbs_effective_step": args.steps * Vh * STEP_BYTES_PER_SITE / (ms_max * 1e-3) / 1e9,
            "e2e": None, "roofline": None, "cpu_baseline": None,
            "measured": "kernels and exchange as one region (CUDA events on the library's stream, max over ranks); the "
                        "roofline / e2e / cpu_baseline legs belong to the default arm (--scaling weak)"}
    if rank == 0:
        print(json.dumps(line), flush=True)
    B.lqcd_finalize()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=40)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="weak (default): N independent replicas, the contract's arm; strong: one lattice split over N ranks")
    ap.add_argument("--overlap", action="store_true", help="--scaling strong: interior sites while the halos are in flight")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.scaling == "strong":
        run_strong(args, rank, world, local_rank)
        return
    run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
