#!/usr/bin/env python
"""sweep.py -- timings of the BASELINE.json configurations 3, 4, 5 and of the paper's thermal
lattice shapes (Fig. 7), one JSON line each.  A user-facing companion of bench.py:

    python -m paper_1209_5942_b200.sweep [--configs 3,4,5,solve5,thermal,force,gauge,slab,copy,large] [--out FILE] [--hop-variant N]

config 3: 16^3x32, near-identity links, kappa=.16 mu=.05: 10 warm-up + 100 timed D_eo/D_oe
          applications, 5 repeats, median (working set fits L2: not a HBM roofline figure)
config 4: 24^3x48 Haar links: CG on Mhat^dag Mhat to 1e-10; iterations, time to solution,
          per-iteration split between hopping launches and vector kernels
config 5: 32^3x64, double/single x 18/12-real links: 20 warm-up + 200 timed D-slash applications
solve5  : config 4's three solves (double CG, BiCGStab, mixed-precision CG) on config 5's lattice
thermal : N_sigma in {16,24,32,48} x N_tau in {4,8,12,16}, double/18 D-slash
force   : the fermion-force kernel at 32^3x64 in the four storage variants
gauge   : heatbath and overrelaxation sweeps at 32^3x64 in the four storage variants

GFLOPS at 1320 flop per output site (BASELINE metric); "gbs_effective" counts the algorithmic
bytes (each link, each input site and each output once); "gbs_paper_accounting" counts the
paper's 8 links + 8 spinors + 1 store per site for comparison with its Fig. 7.
"""
import argparse
import json
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import lqcd_inputs as gen  # noqa: E402
from paper_1209_5942_b200 import binding as B  # noqa: E402

FLOP = 1320
NOMINAL_GBS = 8000.0


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"])
    except Exception:
        return 6650.0


def site_bytes(precision, recon):
    real = 8 if precision == 0 else 4
    link, spinor = recon * real, 24 * real
    return 8 * link + 2 * spinor, 8 * link + 9 * spinor


def time_dslash(dims, U, precision, recon, kappa, warm, reps, repeats, stream):
    Vh = int(np.prod(dims)) // 2
    B.lqcd_init(dims, gen.antiperiodic_t())
    B.lqcd_set_format(precision, recon)
    B.lqcd_set_stream(stream)
    with torch.cuda.stream(stream):
        g = B.upload_gauge(U)
        a = B.upload_spinor(gen.spinor_gaussian(Vh), 1)
        b = B.alloc_spinor()
        for _ in range(warm // 2):
            B.lqcd_dslash_eo(g, a, b, 0, kappa)
            B.lqcd_dslash_eo(g, b, a, 1, kappa)
        # the timed loop is captured once in a CUDA graph and replayed: below ~24^3 x 8 one
        # Python/ctypes call per application (~7 us) is slower than the kernel itself
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            for _ in range(reps // 2):
                B.lqcd_dslash_eo(g, a, b, 0, kappa)
                B.lqcd_dslash_eo(g, b, a, 1, kappa)
        graph.replay()
        times = []
        for _ in range(repeats):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            stream.synchronize()
            e0.record(stream)
            graph.replay()
            e1.record(stream)
            stream.synchronize()
            times.append(e0.elapsed_time(e1) / (2 * (reps // 2)))
        del graph
    B.lqcd_finalize()
    ms = float(np.median(times))
    eff, paper = site_bytes(precision, recon)
    peak = measured_peak()
    gbs = Vh * eff / ms / 1e6
    return {"us_per_application": ms * 1e3, "gflops": Vh * FLOP / ms / 1e6, "gbs_effective": gbs,
            "gbs_paper_accounting": Vh * paper / ms / 1e6, "bytes_per_site": eff,
            "frac_of_measured_peak": gbs / peak, "frac_of_nominal_peak": gbs / NOMINAL_GBS,
            "measured_peak_gbs": peak}


def config3(stream):
    dims = (16, 16, 16, 32)
    U = gen.gauge_near_identity(dims, gen.BASE_SEED, 0.3)
    r = time_dslash(dims, U, 0, 18, 0.16, 10, 100, 5, stream)
    r.update({"config": 3, "lattice": list(dims), "precision": "double", "recon": 18,
              "note": "gauge 75 MB + spinors 25 MB fit the 126 MB L2: DRAM traffic is far below the algorithmic "
                      "bytes, the fraction of HBM peak is not a roofline result"})
    return [r]


def config4(stream, dims=(24, 24, 24, 48), label=4):
    kappa, mu, tol = 0.15, 0.1, 1e-10
    Vh = int(np.prod(dims)) // 2
    U = gen.gauge_haar(dims)
    src = gen.spinor_gaussian(Vh, stream=gen.STREAM_SOURCE)
    B.lqcd_init(dims, gen.antiperiodic_t())
    B.lqcd_set_stream(stream)
    out = []
    with torch.cuda.stream(stream):
        g = B.upload_gauge(U)
        b = B.upload_spinor(src, 0)
        x = B.alloc_spinor()
        B.lqcd_cg_mdagm(g, b, x, kappa, mu, tol, 2000)      # warm-up solve
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stream.synchronize()
        e0.record(stream)
        st = B.lqcd_cg_mdagm(g, b, x, kappa, mu, tol, 2000)
        e1.record(stream)
        stream.synchronize()
        iters, rr, rt = B.lqcd_cg_stats()
        ms = e0.elapsed_time(e1)
        # per-iteration split from per-launch events, in a separate profiled solve
        B.lqcd_profile(1)
        B.lqcd_cg_setup(g, b, x, kappa, mu, tol)
        B.lqcd_cg_iterate(iters)
        hop = sum(B.lqcd_profile_read(c)[0] for c in (0, 1, 2, 5))
        vec = B.lqcd_profile_read(3)[0]
        B.lqcd_profile(0)
        B.lqcd_cg_finish()
        # BiCGStab on Mhat x = b (the other solver the paper names): same operator, the system
        # itself instead of the normal equations, two Mhat applications per iteration
        B.lqcd_bicgstab_mhat(g, b, x, kappa, mu, tol, 2000)
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stream.synchronize()
        b0.record(stream)
        bst = B.lqcd_bicgstab_mhat(g, b, x, kappa, mu, tol, 2000)
        b1.record(stream)
        stream.synchronize()
        bit, brr, brt = B.lqcd_cg_stats()
        bicg = {"status": int(bst), "iterations": bit, "time_to_solution_ms": b0.elapsed_time(b1),
                "ms_per_iteration": b0.elapsed_time(b1) / max(bit, 1), "rel_resid_recursive": brr,
                "rel_resid_true": brt, "gflops": 4 * bit * Vh * FLOP / b0.elapsed_time(b1) / 1e6}
        # the same solve by mixed-precision defect correction (single/12 inner CG)
        B.lqcd_set_format(B.LQCD_SINGLE, 12)
        gs = B.upload_gauge(U)
        B.lqcd_set_format(B.LQCD_DOUBLE, 18)
        B.lqcd_cg_mdagm_mixed(g, 18, gs, 12, b, x, kappa, mu, tol, 2000)
        m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stream.synchronize()
        m0.record(stream)
        mst = B.lqcd_cg_mdagm_mixed(g, 18, gs, 12, b, x, kappa, mu, tol, 2000)
        m1.record(stream)
        stream.synchronize()
        mit, mrr, _ = B.lqcd_cg_stats()
        mixed = {"status": int(mst), "inner_iterations": mit, "outer_corrections": B.lqcd_cg_outer_iterations(),
                 "time_to_solution_ms": m0.elapsed_time(m1), "rel_resid_true": mrr,
                 "speedup_vs_double": ms / m0.elapsed_time(m1)}
    B.lqcd_finalize()
    out.append({"config": label, "lattice": list(dims), "precision": "double", "recon": 18, "status": int(st),
                "iterations": iters, "time_to_solution_ms": ms, "rel_resid_recursive": rr, "rel_resid_true": rt,
                "ms_per_iteration": ms / max(iters, 1),
                "gflops": 4 * iters * Vh * FLOP / ms / 1e6,
                "per_iteration_us": {"hopping_4_launches": hop / iters * 1e3, "vector_and_finalize_kernels": vec / iters * 1e3},
                "hopping_share": hop / (hop + vec),
                "mixed_precision_single12_inner": mixed,
                "bicgstab_on_mhat": bicg,
                "note": "time to solution includes the solve setup and the final true-residual check (one extra "
                        "application of Mhat^dag Mhat)"})
    return out


def solve5(stream):
    """Config 4's three solves (double CG, BiCGStab on Mhat, mixed-precision CG with a single/12 inner solve) on config 5's
    32^3x64 lattice, device resident, to 1e-10."""
    return config4(stream, (32, 32, 32, 64), "solve5")


FORMATS = ((0, 18), (0, 12), (1, 18), (1, 12))   # --formats narrows config 5 down (d18,d12,s18,s12)


def config5(stream):
    dims = (32, 32, 32, 64)
    U = gen.gauge_haar(dims)
    out = []
    for precision, recon in FORMATS:
        r = time_dslash(dims, U, precision, recon, 0.15, 20, 200, 3, stream)
        r.update({"config": 5, "lattice": list(dims), "precision": "double" if precision == 0 else "single",
                  "recon": recon})
        out.append(r)
    return out


def force(stream):
    """Fermion-force kernel at 32^3x64: one launch computes all 4 V links.
    Algorithmic bytes per site of V: 4 links + X + Y (each site once) + 4 x 8 force reals."""
    dims = (32, 32, 32, 64)
    V = int(np.prod(dims))
    U = gen.gauge_haar(dims)
    out = []
    for precision, recon in ((0, 18), (0, 12), (1, 18), (1, 12)):
        B.lqcd_init(dims, gen.antiperiodic_t())
        B.lqcd_set_format(precision, recon)
        B.lqcd_set_stream(stream)
        with torch.cuda.stream(stream):
            g = B.upload_gauge(U)
            f = B.alloc_force()
            h = [B.upload_spinor(gen.spinor_gaussian(V // 2, stream=10 + i), i % 2) for i in range(4)]
            for _ in range(10):
                B.lqcd_fermion_force(g, h[0], h[1], h[2], h[3], f, 0.15)
            times = []
            for _ in range(3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                stream.synchronize()
                e0.record(stream)
                for _ in range(100):
                    B.lqcd_fermion_force(g, h[0], h[1], h[2], h[3], f, 0.15)
                e1.record(stream)
                stream.synchronize()
                times.append(e0.elapsed_time(e1) / 100)
        B.lqcd_finalize()
        ms = float(np.median(times))
        real = 8 if precision == 0 else 4
        bytes_site = 4 * recon * real + 2 * 24 * real + 4 * 8 * 8
        paper_bytes = 4 * (2 * recon * real + 4 * 24 * real + 2 * 8 * 8)   # PAPER.md:236 accounting (4736 in double/18)
        peak = measured_peak()
        gbs = V * bytes_site / ms / 1e6
        out.append({"config": "force", "kernel": "fermion_force", "lattice": list(dims),
                    "precision": "double" if precision == 0 else "single", "recon": recon,
                    "us_per_launch": ms * 1e3, "links_per_s": 4 * V / ms * 1e3, "bytes_per_site": bytes_site,
                    "gbs_effective": gbs, "gbs_paper_accounting": V * paper_bytes / ms / 1e6,
                    "frac_of_measured_peak": gbs / peak, "measured_peak_gbs": peak})
    return out


def gauge(stream):
    """Heatbath / overrelaxation sweeps at 32^3x64, thermalised-like links,
    beta = 5.7: one sweep = 8 sub-sweep launches = 4 V link updates.  GFLOPS with the paper's counts
    (3912 / 3846 flop per link); algorithmic bytes per updated link = 9 links (a sub-sweep
    reads every link of the lattice once and writes V/2), paper accounting = 20 links."""
    dims = (32, 32, 32, 64)
    V = int(np.prod(dims))
    U = gen.gauge_near_identity(dims, gen.BASE_SEED, 0.3)
    out = []
    for precision, recon in ((0, 18), (1, 18), (0, 12), (1, 12)):
        B.lqcd_init(dims, gen.antiperiodic_t())
        B.lqcd_set_format(precision, recon)
        B.lqcd_set_stream(stream)
        with torch.cuda.stream(stream):
            g = B.upload_gauge(U)
            for mode, name, flop in ((B.LQCD_HEATBATH, "heatbath", 3912), (B.LQCD_OVERRELAX, "overrelax", 3846)):
                for k in range(3):
                    B.lqcd_gauge_sweep(g, mode, 5.7, gen.BASE_SEED, 100 + k)
                times = []
                for rep in range(3):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    stream.synchronize()
                    e0.record(stream)
                    for k in range(10):
                        B.lqcd_gauge_sweep(g, mode, 5.7, gen.BASE_SEED, 200 + 10 * rep + k)
                    e1.record(stream)
                    stream.synchronize()
                    times.append(e0.elapsed_time(e1) / 10)
                ms = float(np.median(times))
                real = 8 if precision == 0 else 4
                link = recon * real
                peak = measured_peak()
                gbs = 4 * V * 9 * link / ms / 1e6
                out.append({"config": "gauge", "kernel": name, "lattice": list(dims),
                            "precision": "double" if precision == 0 else "single", "recon": recon,
                            "ms_per_sweep": ms, "us_per_subsweep": ms * 1e3 / 8, "links_per_s": 4 * V / ms * 1e3,
                            "gflops_paper_count": 4 * V * flop / ms / 1e6, "bytes_per_link": 9 * link,
                            "gbs_effective": gbs, "gbs_paper_accounting": 4 * V * 20 * link / ms / 1e6,
                            "frac_of_measured_peak": gbs / peak, "measured_peak_gbs": peak,
                            "plaquette_after": B.lqcd_plaquette(g)})
        B.lqcd_finalize()
    return out


def copy(stream):
    """The paper's buffer-copy micro-benchmark by element type (Fig. 5) through
    lqcd_stream_probe, plus the READ and 7:1 mixes that bracket the hopping kernel.  Two buffer sizes: 2.1 GB
    (HBM; every figure that is compared with a kernel) and the paper's 100 MiB, which fits B200's 126 MB L2
    and is reported only to show that.  GB/s counts bytes read + bytes written."""
    names = {0: "float (4 B)", 1: "double (8 B)", 2: "16-byte vector", 3: "su3 AoS (144 B)", 4: "spinor AoS (192 B)"}
    modes = {0: "copy", 1: "read", 2: "mix 7:1"}
    B.lqcd_init((4, 4, 4, 4), gen.antiperiodic_t())
    B.lqcd_set_stream(stream)
    out = []
    peak = measured_peak()
    with torch.cuda.stream(stream):
        for nbytes, where in ((12096 * 175000, "HBM"), (12096 * 8668, "paper's 100 MiB: fits L2")):
            src = torch.randint(0, 256, (nbytes,), dtype=torch.uint8, device="cuda")
            dst = torch.empty(nbytes, dtype=torch.uint8, device="cuda")

            def timed(body, moved):
                for _ in range(5):
                    body()
                ts = []
                for _ in range(3):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    stream.synchronize()
                    e0.record(stream)
                    for _ in range(20):
                        body()
                    e1.record(stream)
                    stream.synchronize()
                    ts.append(e0.elapsed_time(e1) / 20)
                ms = float(np.median(ts))
                return ms * 1e3, moved / ms / 1e6

            for elem in range(5):
                for mode in ((0, 1, 2) if elem < 3 else (0,)):
                    moved = {0: 2 * nbytes, 1: nbytes, 2: nbytes + nbytes // 7}[mode]
                    us, gbs = timed(lambda: B.lqcd_stream_probe(elem, mode, src, dst, nbytes), moved)
                    out.append({"config": "copy", "element": names[elem], "mode": modes[mode], "buffer_bytes": nbytes,
                                "buffer": where, "us": us, "gbs": gbs, "frac_of_measured_peak": gbs / peak,
                                "measured_peak_gbs": peak})
            us, gbs = timed(lambda: dst.copy_(src), 2 * nbytes)
            out.append({"config": "copy", "element": "torch.Tensor.copy_ (what MEASURED_PEAKS.json times)", "mode": "copy",
                        "buffer_bytes": nbytes, "buffer": where, "us": us, "gbs": gbs,
                        "frac_of_measured_peak": gbs / peak, "measured_peak_gbs": peak})
            del src, dst
        # FP64 pipe (the hopping term's secondary bound): 8 independent DFMA chains per thread
        n = B.LQCD_STREAM_PROBE_BLOCKS * 256
        o = torch.empty(n, dtype=torch.float64, device="cuda")
        iters = 20000
        B.lqcd_fp64_probe(0.999999, 1e-3, iters, o)
        ts = []
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            stream.synchronize()
            e0.record(stream)
            B.lqcd_fp64_probe(0.999999, 1e-3, iters, o)
            e1.record(stream)
            stream.synchronize()
            ts.append(e0.elapsed_time(e1))
        ms = float(np.median(ts))
        out.append({"config": "copy", "element": "fp64 pipe: 8 DFMA chains per thread, 1184 CTAs x 256 threads", "mode": "dfma",
                    "iters": iters, "us": ms * 1e3, "tflops_fp64": 16.0 * iters * n / ms / 1e9})
    B.lqcd_finalize()
    return out


def large(stream):
    """A production-size lattice, 48^3 x 96 (gauge field 6.1 GB, beyond the paper's 32^3 x 64 sizes): D-slash in
    the four storage variants and the CG iteration in double.  The links are a fixed gather of a seeded
    16^3 x 32 Haar field (any arrangement of SU(3) matrices is a valid field; 42 M fresh links take minutes)."""
    dims = (48, 48, 48, 96)
    V = int(np.prod(dims))
    small = gen.gauge_haar((16, 16, 16, 32)).reshape(-1, 3, 3)
    U = small[(np.arange(4 * V, dtype=np.int64) * 7919 + 13) % small.shape[0]].reshape(V, 4, 3, 3)
    out = []
    for precision, recon in ((0, 18), (0, 12), (1, 18), (1, 12)):
        r = time_dslash(dims, U, precision, recon, 0.15, 10, 50, 3, stream)
        r.update({"config": "large", "lattice": list(dims), "precision": "double" if precision == 0 else "single",
                  "recon": recon})
        out.append(r)
    Vh = V // 2
    B.lqcd_init(dims, gen.antiperiodic_t())
    B.lqcd_set_stream(stream)
    with torch.cuda.stream(stream):
        g = B.upload_gauge(U)
        b = B.upload_spinor(gen.spinor_gaussian(Vh, stream=gen.STREAM_SOURCE), 0)
        x = B.alloc_spinor()
        B.lqcd_cg_setup(g, b, x, 0.15, 0.1, 0.0)
        B.lqcd_cg_iterate(10)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stream.synchronize()
        e0.record(stream)
        B.lqcd_cg_setup(g, b, x, 0.15, 0.1, 0.0)
        B.lqcd_cg_iterate(40)
        e1.record(stream)
        stream.synchronize()
        B.lqcd_cg_finish()
        ms = e0.elapsed_time(e1) / 40
    B.lqcd_finalize()
    out.append({"config": "large", "lattice": list(dims), "precision": "double", "recon": 18, "what": "CG iteration",
                "ms_per_iteration": ms, "gflops": 4 * Vh * FLOP / ms / 1e6, "gbs_effective_step": Vh * 7680 / ms / 1e6})
    return out


def slab(stream):
    """One rank's share of a 32^3 x 64 lattice cut into R slabs of the time direction (SURVEY.md section
    8(e)), timed on ONE GPU: the hopping launch over the rank's 32^3 x (64/R) sites
    in one piece and split into interior + boundary launches (what overlaps the halo exchange), the
    halo copy itself as two device-to-device block copies, and the bytes a rank sends per application.
    Per-rank figures only: nothing here measures NVLink."""
    gdims = (32, 32, 32, 64)
    kappa = 0.15
    out = []
    for R in (1, 2, 4, 8):
        dims = gdims[:3] + (gdims[3] // R,)
        Vh = int(np.prod(dims)) // 2
        U = gen.gauge_haar(dims)
        B.lqcd_slab_init(gdims, gen.antiperiodic_t(), 0, R)
        B.lqcd_set_stream(stream)
        with torch.cuda.stream(stream):
            g = B.upload_gauge(U)
            a = B.upload_spinor(gen.spinor_gaussian(Vh), 1)
            b = B.alloc_spinor()
            h = B.lqcd_slab_spinor_halo()
            n = h["bytes"]

            def exchange(f):   # the rank as its own neighbour: same bytes moved as between ranks
                f[h["ghost_fwd"]:h["ghost_fwd"] + n].copy_(f[h["send_lo"]:h["send_lo"] + n])
                f[h["ghost_bwd"]:h["ghost_bwd"] + n].copy_(f[h["send_hi"]:h["send_hi"] + n])

            def timed(body, reps=50):
                for _ in range(5):
                    body()
                ts = []
                for _ in range(3):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    stream.synchronize()
                    e0.record(stream)
                    for _ in range(reps):
                        body()
                    e1.record(stream)
                    stream.synchronize()
                    ts.append(e0.elapsed_time(e1) / reps)
                return float(np.median(ts)) * 1e3

            def whole():
                B.lqcd_slab_dslash(g, a, b, 0, kappa, 0)
                B.lqcd_slab_dslash(g, b, a, 1, kappa, 0)

            def split():
                B.lqcd_slab_dslash(g, a, b, 0, kappa, 1)
                B.lqcd_slab_dslash(g, a, b, 0, kappa, 2)
                B.lqcd_slab_dslash(g, b, a, 1, kappa, 1)
                B.lqcd_slab_dslash(g, b, a, 1, kappa, 2)

            exchange(a); exchange(b)
            us_whole = timed(whole) / 2
            us_split = timed(split) / 2
            us_copy = timed(lambda: exchange(a))
        B.lqcd_finalize()
        out.append({"config": "slab", "global_lattice": list(gdims), "ranks": R, "local_lattice": list(dims),
                    "precision": "double", "recon": 18, "us_per_application_whole": us_whole,
                    "us_per_application_interior_plus_boundary": us_split, "us_halo_copies_on_device": us_copy,
                    "halo_bytes_sent_per_application": 2 * n,
                    "us_halo_at_900_GBs_per_direction": n / 900e9 * 1e6,
                    "gflops_per_rank_whole": Vh * FLOP / us_whole / 1e3,
                    "gbs_effective_per_rank_whole": Vh * 1536 / us_whole / 1e3})
    return out


def thermal(stream):
    out = []
    for ns in (16, 24, 32, 48):
        for nt in (4, 8, 12, 16):
            dims = (ns, ns, ns, nt)
            U = gen.gauge_haar(dims)
            r = time_dslash(dims, U, 0, 18, 0.15, 10, 100, 3, stream)
            r.update({"config": "thermal", "lattice": list(dims), "precision": "double", "recon": 18})
            out.append(r)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="3,4,5,thermal")
    ap.add_argument("--out", default=None)
    ap.add_argument("--hop-variant", type=int, default=0,
                    help="hopping kernel variant (lqcd_set_hop_variant): 0 plain (default), 1..3 link ring of that depth, 4 / 5 bulk-staged forward links, 6 the 2 x 2 (z, t) tile order, 7 the general-phase kernel on real phases")
    ap.add_argument("--formats", default="d18,d12,s18,s12", help="storage variants timed by config 5")
    args = ap.parse_args()
    global FORMATS
    FORMATS = tuple({"d18": (0, 18), "d12": (0, 12), "s18": (1, 18), "s12": (1, 12)}[f.strip()] for f in args.formats.split(","))
    if not torch.cuda.is_available():
        raise SystemExit("sweep.py needs a CUDA device: there is no CPU fallback")
    stream = torch.cuda.Stream()
    table = {"3": config3, "4": config4, "5": config5, "solve5": solve5, "thermal": thermal, "force": force, "gauge": gauge, "slab": slab, "copy": copy, "large": large}
    lines = []
    B.lqcd_set_hop_variant(args.hop_variant)
    for key in args.configs.split(","):
        for r in table[key.strip()](stream):
            if args.hop_variant:
                r["hop_variant"] = args.hop_variant
            line = json.dumps(r)
            print(line, flush=True)
            lines.append(line)
    if args.out:
        with open(args.out, "w") as f:
            f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
