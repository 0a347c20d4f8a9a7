#!/usr/bin/env python
"""bench.py -- headline benchmark of the tm-dslash / MdagM / CG / loop library on B200.

A "step" is one pass of the whole hot path over one batch of synthetic input at 32^3x64 (BASELINE.json
configs[3], the paper's ensemble shape): 12 Z2xiZ2 noise sources -> pack -> batched truncated CG (tol 1e-2, fp16
storage / fp32 arithmetic / fp64 reductions, 12-real links, every gauge load shared by the 12 right-hand sides) ->
16-Gamma per-time-slice loop contraction of every solution.  metric = LP solves/s (BASELINE.json "LP solves/sec").
The same run also reports BASELINE.json's other metric, single-RHS tm-dslash GFLOPS and algorithmic HBM GB/s at
fp32 / fp16 x 18 / 12 reals (configs[2]), and a mixed-precision CG to 1e-8.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--no-sweeps]
N > 1: launched under torch.distributed.run; noise sources are independent, so ranks take different batches and
there is no data-path collective (weak scaling, "replicas + gather" of the [16][T] loops through paper_1309_2256_b200.shard).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

DIMS = (32, 32, 32, 64)
NRHS = 12
LP_TOL = 1e-2
FLOPS_HOP, FLOPS_TWIST_INV, FLOPS_XPAY = 1320, 1392, 1416  # per output site
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12          # 148 SMs x 128 FP32 lanes x 2 (FMA) x max SM clock


# DRAM bytes per launch of the dominant kernel: read from the tracked record of its `ncu --set full` capture, and only
# trusted while the kernel the library launches still has the template signature that was profiled
TRAFFIC_RECORD = os.path.join(ROOT, "profiles", "dominant_kernel_traffic.json")


def ncu_traffic(signature):
    """(bytes per launch | None, source string).  None when there is no record or it belongs to another kernel build."""
    try:
        rec = json.load(open(TRAFFIC_RECORD))
    except Exception as e:
        return None, "no usable %s (%s)" % (os.path.relpath(TRAFFIC_RECORD, ROOT), type(e).__name__)
    if rec.get("signature") != signature:
        return None, "stale: %s was captured for %r, the library launches %r" % (os.path.relpath(TRAFFIC_RECORD, ROOT), rec.get("signature"), signature)
    return float(rec["dram_bytes_per_launch"]), "%s: %s" % (os.path.relpath(TRAFFIC_RECORD, ROOT), rec.get("source", ""))


def ncu_pipe_fractions(signature):
    """FMA-pipe and issue-slot utilisation of the dominant kernel from the same signature-checked ncu record ({} when stale):
    the counted flops (1392 / 1416 per site) leave out conversion, projection, link handling and epilogue work, so `frac`
    understates how busy the FP32 pipe is."""
    try:
        rec = json.load(open(TRAFFIC_RECORD))
    except Exception:
        return {}
    if rec.get("signature") != signature:
        return {}
    return {k + "_ncu": rec[k] for k in ("fma_pipe_active_frac", "issue_active_frac") if k in rec}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons),
                "samples": len(sm)}


def cpu_oracle_sample(large=False):
    """The oracle as it stands on the host cores: ONE complete truncated solve (tol 1e-2) + one 16-Gamma loop contraction, on a
    lattice with the workload's generators / kappa / mu, scaled by the site ratio to solves/s at 32^3x64.
    large: the 32^3x64 lattice of the workload itself (one of the 12 sources of a step, nothing extrapolated; 26 s on the 16 host
    cores of the GPU box); else 16^3x32 (1/16 of the sites, 1.5 s: the per-step sample of --impl reference)."""
    import oracle
    import tm_inputs as ti
    dims = DIMS if large else (16, 16, 16, 32)
    U = ti.gauge(dims)
    eta = ti.z4(dims)
    t0 = time.time()
    s, info = oracle.cg_solve(U, eta, ti.KAPPA, ti.MU, LP_TOL, 500)
    oracle.loop(eta, s)
    dt = time.time() - t0
    scale = float(np.prod(DIMS)) / float(np.prod(dims))
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    sample = "one truncated CG solve (tol 1e-2, %d iterations) + one 16-Gamma loop on %dx%dx%dx%d in %.1f s" % ((info["iters"],) + tuple(dims) + (dt,))
    sample += ": 1 of the 12 sources of a step, nothing extrapolated" if scale == 1.0 else " (1/%d of the sites), scaled x1/%d to 32^3x64" % (round(scale), round(scale))
    return {"value": 1.0 / (dt * scale), "unit": "solves/s", "cores": cores, "kind": "oracle", "sample": sample}, dt


def run_reference(args, rank):
    if rank != 0:
        return
    vals, dts = [], []
    base = None
    for _ in range(args.warmup):  # untimed: library load, page faults of the first pass
        cpu_oracle_sample()
    for _ in range(args.steps):
        base, dt = cpu_oracle_sample()
        vals.append(base["value"]); dts.append(dt)
    v = float(np.mean(vals))
    base["value"] = v
    print(json.dumps({
        "impl": "reference", "metric": "LP solves/s", "value": v, "unit": "solves/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(dts)), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "32^3x64 TSM: truncated CG tol 1e-2 + 16-Gamma loop per source (oracle sample on 16^3x32, scaled)"},
        "cpu_baseline": base, "e2e": {"value": v, "unit": "solves/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def dslash_bytes(Vh, prec, recon, has_x, nrhs=1):
    """Minimal-traffic (algorithmic) bytes of one dslash launch: every link once, every input spinor once, output once
    (+ x once); fp16 spinors carry a 4-byte norm."""
    sp = 24 * prec + (4 if prec == 2 else 0)
    return Vh * (8 * recon * prec + nrhs * (2 + (1 if has_x else 0)) * sp)


def time_events(torch, fn, n):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(n):
        fn(i)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n


def run_b200(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    import tm_inputs as ti
    import paper_1309_2256_b200 as tm
    from paper_1309_2256_b200 import shard
    tm.load()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    hbm_peak, peak_src = peaks()
    L = tm.tm_lattice_create(DIMS, True)
    V, Vh, T = L.V, L.V // 2, DIMS[3]
    kappa, mu = ti.KAPPA, ti.MU

    # ---- once per configuration: gauge field -> packed links (a0) ----
    U = torch.from_numpy(ti.gauge(DIMS).view(np.float64)).cuda()
    gauges = {}
    for prec, recon in ((2, 12), (2, 18), (4, 12), (4, 18), (8, 12), (8, 18), (2, 8), (4, 8), (8, 8), (2, 112), (2, 118)):
        gauges[(prec, recon)] = tm.device_buffer(tm.tm_gauge_bytes(L, prec, recon))
        tm.tm_gauge_pack(L, U, prec, recon, gauges[(prec, recon)], 1e-10)
    del U
    torch.cuda.empty_cache()

    # ---- inputs: two batches of 12 Z2xiZ2 sources per rank (302 MB each > L2), alternating ----
    nb = 2
    codes_host = [torch.from_numpy(np.stack([ti.z4_codes(DIMS, seed=ti.NOISE_SEED + (rank * nb + b) * NRHS + r) for r in range(NRHS)]))
                  .pin_memory() for b in range(nb)]
    codes_dev = [c.cuda() for c in codes_host]
    # the e2e leg ships the same noise bit-packed (3 bytes per site instead of 12: tm_tsm_batch_host_bits)
    bits_host = [torch.from_numpy(np.stack([ti.z4_bits(DIMS, seed=ti.NOISE_SEED + (rank * nb + b) * NRHS + r) for r in range(NRHS)]))
                 .pin_memory() for b in range(nb)]
    prec, recon = 2, 12
    g_lp = gauges[(prec, recon)]
    fb = tm.tm_spinor_bytes(L, prec, 1, NRHS)
    eta, sol = tm.device_buffer(fb), tm.device_buffer(fb)
    cg_ws = tm.device_buffer(tm.tm_cg_workspace_bytes(L, 8, prec, tm.TM_CG_LP_TRUNCATED, NRHS))
    loop_ws = tm.device_buffer(tm.tm_loop_workspace_bytes(L, NRHS))
    loops = torch.zeros((NRHS, 16, T, 2), dtype=torch.float64, device="cuda")
    tsm_ws = tm.device_buffer(tm.tm_tsm_workspace_bytes(L, prec, NRHS))
    loops_host = torch.zeros((NRHS, 16, T, 2), dtype=torch.float64).pin_memory()
    prm = tm.make_cg_params(kappa, mu, LP_TOL, 500, tm.TM_CG_LP_TRUNCATED, 0.1, 0, 1)  # truncated mode: no residual recomputation
    iters_log = []
    gather = shard.LoopGather(world * NRHS, NRHS, (16, T, 2), torch.float64, torch.device("cuda", local_rank)) if world > 1 else None

    def step(i):
        tm.tm_spinor_pack_z4(L, codes_dev[i % nb], prec, NRHS, eta)
        rc, info = tm.tm_cg_multi(L, None, 8, g_lp, prec, recon, sol, eta, prm, NRHS, cg_ws)
        assert rc == tm.TM_OK, rc
        tm.tm_loop_contract(L, eta, sol, prec, NRHS, loops, loop_ws)
        if world > 1:  # the path's only exchange: one gather of the [16][T] loops (16 KB per source), SURVEY.md 8(e)
            gather(loops)
        iters_log.append([x.iters for x in info])

    def step_e2e(i):
        rc, info = tm.tm_tsm_batch_host_bits(L, g_lp, prec, recon, bits_host[i % nb], prm, NRHS, loops_host, tsm_ws)
        assert rc == tm.TM_OK, rc

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    table, flat = single_rhs_table(torch, tm, ti, L, gauges, hbm_peak, peak_src) if rank == 0 else (None, None)

    # ---- warm-up, then EXACTLY K timed steps (device-resident inputs) ----
    for i in range(args.warmup):
        step(i)
    iters_log.clear()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    tm.tm_kernel_timing_enable(1)
    tm.tm_kernel_timing_read(True)
    n0 = tm.tm_launch_count()
    torch.cuda.profiler.start()   # no-op unless a profiler runs with --profile-from-start off: then exactly the timed steps are listed
    ms_step = time_events(torch, step, args.steps)
    torch.cuda.profiler.stop()
    launches = tm.tm_launch_count() - n0
    k_ms, k_n = tm.tm_kernel_timing_read(True)
    tm.tm_kernel_timing_enable(0)
    barrier()
    clocks = sampler.stop()
    ms_step = max_over_ranks(ms_step)
    value = world * NRHS / (ms_step * 1e-3)

    # ---- e2e: host buffers through tm_tsm_batch_host_bits, H2D + D2H inside the timed region ----
    for i in range(max(1, args.warmup // 2)):
        step_e2e(i)
    barrier()
    ms_e2e = max_over_ranks(time_events(torch, step_e2e, args.steps))
    e2e = {"value": world * NRHS / (ms_e2e * 1e-3), "unit": "solves/s", "h2d_bytes_per_step": int(bits_host[0].numel()),
           "d2h_bytes_per_step": int(loops_host.numel() * 8), "ms_per_step": ms_e2e}

    # ---- roofline of the dominant kernel: the 12-RHS fp16 dslash launches inside the timed steps ----
    # launches per solve batch: 3 (prepare) + 4 per CG iteration while any rhs is active + 1 (reconstruct);
    # rhs r is active in iterations 1..iters[r]; bytes follow the active right-hand sides exactly.
    sp = 24 * prec + 4
    tot_bytes = tot_flops = 0.0
    for it in iters_log:
        tot_bytes += 4 * dslash_bytes(Vh, prec, recon, False, NRHS) + 3 * Vh * NRHS * sp  # 4 full launches, 3 of them read x
        tot_flops += Vh * NRHS * (3 * FLOPS_XPAY + 1 * FLOPS_TWIST_INV)
        for k in range(1, max(it) + 1):
            act = sum(1 for x in it if x >= k)
            # 4 launches: in + out each, x twice, the residual once; flops: 2 x (TWIST_INV + XPAY) + |M p|^2, r -= alpha A p, |r|^2
            tot_bytes += 4 * Vh * 8 * recon * prec + Vh * act * (4 * 2 + 3) * sp
            tot_flops += Vh * act * (2 * (FLOPS_TWIST_INV + FLOPS_XPAY) + 3 * 48)
    k_avg_ms = k_ms / max(1, k_n)
    ach_gbs = tot_bytes / (k_ms * 1e-3) / 1e9
    ach_tf = tot_flops / (k_ms * 1e-3) / 1e12
    sig = tm.tm_kernel_signature()
    traffic, traffic_src = ncu_traffic(sig)
    roofline = {"kernel": sig + " (fp16 storage, 12-real links, link cache + cp.async.bulk)", "bound": "alu", "achieved": ach_tf, "peak": FP32_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": ach_tf / FP32_PEAK_TFLOPS, "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": "148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (B200_PROFILING.md unit counts and clocks)",
                "avg_launch_ms": k_avg_ms, "launches_timed": int(k_n), "share_of_step": k_ms / (ms_step * args.steps),
                # the same launches in the HBM view (flat scalars: nested objects do not survive the driver's parse)
                "hbm_achieved_GBps": ach_gbs, "hbm_peak_GBps": hbm_peak, "hbm_frac": ach_gbs / hbm_peak, "hbm_peak_source": peak_src}
    roofline.update(ncu_pipe_fractions(sig))

    out = {"metric": "LP solves/s", "value": value, "unit": "solves/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32 (fp16 storage + per-site fp32 norm, fp64 reductions)", "data": "synthetic",
           "config": {"workload": "32^3x64 TSM (BASELINE.json configs[3]): 12 Z2xiZ2 sources per step, truncated CG tol 1e-2, "
                                  "12-real links, 12 RHS per gauge load, + 16-Gamma per-timeslice loop of each solution",
                      "lattice": list(DIMS), "kappa": kappa, "mu": mu, "gauge": "seeded SU(3), eps=0.5", "nrhs": NRHS,
                      "iters_per_solve": float(np.mean(iters_log)), "l2": "inputs larger than L2 (gauge 201 MB + 12x2x54.5 MB vectors)",
                      "parallelism": "independent noise batches per GPU; one all_gather of the loops per step (16 KB per source)"},
           "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline}
    if rank == 0:
        out["roofline"].update(flat)
        out["dslash"] = table
        out["dslash_peak_source"] = peak_src
        extras(torch, tm, ti, L, gauges, hbm_peak, peak_src, out, world, table)
        if not args.no_sweeps and world == 1:
            del gauges, eta, sol, cg_ws, tsm_ws
            torch.cuda.empty_cache()
            sweep_other_configs(torch, tm, ti, hbm_peak, out)
        if "dslash" in out:  # the single-rhs table goes last, so that the tail of the line holds it
            out["dslash"] = out.pop("dslash")
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def single_rhs_table(torch, tm, ti, L, gauges, hbm_peak, peak_src):
    """BASELINE.json's first metric (configs[2]): the single-RHS dslash table at 32^3x64 and MdagM.  Runs BEFORE the TSM steps: the
    steps hold the board at its power cap for seconds, and the clock they leave behind (1.8 GHz instead of 1.95) would be charged to
    these 40-launch measurements (76 vs 84 us for fp16 / 12 reals in the same process).  Returns (table, flat roofline keys)."""
    Vh = L.V // 2
    kappa, mu = ti.KAPPA, ti.MU
    psi = torch.from_numpy(ti.z4(DIMS, seed=777).view(np.float64)).cuda()
    table = {}
    for prec in (4, 2, 8):  # single / half / double of Table A.1
        # every precision gets freshly allocated (2 MB aligned) buffers: blocks recycled from the previous precision by the caching
        # allocator put the four rotating outputs, the source and x at offsets that cost the same kernels up to 8 % (measured: fp32 / 12
        # reals 98.4 vs 102-106 us, fp16 / 12 reals 73.8 vs 78-80 us) -- an artefact of the harness, not of the kernels
        torch.cuda.empty_cache()
        pb = tm.tm_spinor_bytes(L, prec, 0, 1)
        src = tm.device_buffer(2 * pb)
        tm.tm_spinor_pack(L, psi, prec, 1, src)
        # rotate through 4 output/x buffers so the spinor working set (>= 5 x 54..101 MB) exceeds the 126 MB L2
        bufs = [tm.device_buffer(pb) for _ in range(4)]
        xs = [tm.device_buffer(pb) for _ in range(4)]
        for b in bufs + xs:
            b.copy_(src[:pb])
        tmp = tm.device_buffer(2 * pb)
        # 8 = the paper's fastest reconstruction on the GTX Titan (Table A.1), ALU-bound on B200; 118 / 112 = 16-bit fixed-point links
        for recon in (18, 12, 8) + ((118, 112) if prec == 2 else ()):
            g = gauges[(prec, recon)]
            reals = recon % 100
            # "wilson_plain" = the hop alone (Table A.1's Wilson column: no twist in the epilogue)
            for kind, name, fl in ((tm.TM_KIND_TWIST_INV, "twist_inv", FLOPS_TWIST_INV), (tm.TM_KIND_XPAY_TWIST, "xpay_twist", FLOPS_XPAY),
                                   (tm.TM_KIND_PLAIN, "wilson_plain", 1320)):
                def run(i, kind=kind, g=g, prec=prec, recon=recon):
                    tm.tm_dslash(L, g, prec, recon, bufs[i % 4], src[pb:2 * pb], xs[i % 4] if kind == tm.TM_KIND_XPAY_TWIST else None, 0, 0,
                                 kind, kappa, mu)
                for i in range(5):
                    run(i)
                ms = min(time_events(torch, run, 40) for _ in range(3))
                by = dslash_bytes(Vh, prec, reals, kind == tm.TM_KIND_XPAY_TWIST)
                sp = 24 * prec + (4 if prec == 2 else 0)
                naive = Vh * (8 * reals * prec + (9 + (1 if kind == tm.TM_KIND_XPAY_TWIST else 0)) * sp)
                gbs = by / ms / 1e6
                table["%s_fp%d_recon%d%s" % (name, prec * 8, reals, "fix16" if recon >= 100 else "")] = {
                    "us": ms * 1e3, "GFLOPS": Vh * fl / ms / 1e6, "GBps_algorithmic": gbs, "GBps_naive_model": naive / ms / 1e6,
                    "bytes_per_site_minimal": by / Vh, "bytes_per_site_naive": naive / Vh,
                    "frac_of_measured_%.0f" % hbm_peak: gbs / hbm_peak, "frac_of_nominal_8000": gbs / 8000.0}
        def run_mdagm(i, g=gauges[(prec, 12)], prec=prec):
            tm.tm_MdagM(L, g, prec, 12, bufs[i % 4], src[:pb], tmp, 0, kappa, mu)
        for i in range(3):
            run_mdagm(i)
        ms = min(time_events(torch, run_mdagm, 20) for _ in range(3))
        table["MdagM_fp%d_recon12" % (prec * 8)] = {"us": ms * 1e3, "GFLOPS": Vh * 2 * (FLOPS_TWIST_INV + FLOPS_XPAY) / ms / 1e6,
                                                   "GBps_algorithmic": (2 * dslash_bytes(Vh, prec, 12, False) + 2 * dslash_bytes(Vh, prec, 12, True)) / ms / 1e6}
        del bufs, xs, src, tmp
    flat = {}
    # BASELINE.json's first metric where the driver's parse keeps it: flat scalars inside `roofline` (TWIST_INV, 32^3x64, single rhs;
    # algorithmic bytes / time as a fraction of the measured copy bandwidth; north_star's target is >= 0.70)
    fk = "frac_of_measured_%.0f" % hbm_peak
    for prec_, nm in ((4, "fp32"), (2, "fp16")):
        for rc_ in (18, 12):
            row = table["twist_inv_fp%d_recon%d" % (prec_ * 8, rc_)]
            flat["dslash_%s_r%d_frac" % (nm, rc_)] = row[fk]
            flat["dslash_%s_r%d_us" % (nm, rc_)] = row["us"]
            flat["dslash_%s_r%d_frac_of_8000" % (nm, rc_)] = row["frac_of_nominal_8000"]
    del psi
    return table, flat


def extras(torch, tm, ti, L, gauges, hbm_peak, peak_src, out, world, table):
    """Rank 0, N=1 context numbers: the single-rhs kernels in temporal gauge, loop contraction, insertions, unbatched / fp32 solves,
    mixed CG to 1e-8, and the oracle timed on the host cores."""
    Vh = L.V // 2
    kappa, mu = ti.KAPPA, ti.MU
    psi = torch.from_numpy(ti.z4(DIMS, seed=777).view(np.float64)).cuda()
    # the same single-rhs kernels on the temporal-gauge copy of the field, declared as such (TM_RECON_*_TG): temporal hops inside the
    # lattice load no link and multiply by none.  Bytes: 6 + 2/T links per site instead of 8; GFLOPS keep the 1320-flop convention.
    # the field is gauge-fixed by the library's own call on the device (tm_gauge_fix_temporal), as a user would do it
    Utg = torch.from_numpy(ti.gauge(DIMS).view(np.float64)).cuda()
    gtg = torch.empty(L.V * 18, dtype=torch.float64, device="cuda")
    tm.tm_gauge_fix_temporal(L, Utg, gtg)
    del gtg
    tgt = {}
    T_ = DIMS[3]
    for prec in (4, 2):
        pb = tm.tm_spinor_bytes(L, prec, 0, 1)
        src = tm.device_buffer(2 * pb)
        tm.tm_spinor_pack(L, psi, prec, 1, src)
        bufs = [tm.device_buffer(pb) for _ in range(4)]
        xs = [tm.device_buffer(pb) for _ in range(4)]
        for b in bufs + xs:
            b.copy_(src[:pb])
        for reals in (18, 12):
            code = 200 + reals
            g = tm.device_buffer(tm.tm_gauge_bytes(L, prec, code))
            tm.tm_gauge_pack(L, Utg, prec, code, g, 1e-10)
            for kind, name, fl in ((tm.TM_KIND_TWIST_INV, "twist_inv", FLOPS_TWIST_INV), (tm.TM_KIND_XPAY_TWIST, "xpay_twist", FLOPS_XPAY)):
                def run(i, kind=kind, g=g, prec=prec, code=code):
                    tm.tm_dslash(L, g, prec, code, bufs[i % 4], src[pb:2 * pb], xs[i % 4] if kind == tm.TM_KIND_XPAY_TWIST else None, 0, 0,
                                 kind, kappa, mu)
                for i in range(5):
                    run(i)
                ms = min(time_events(torch, run, 40) for _ in range(3))
                sp = 24 * prec + (4 if prec == 2 else 0)
                by = Vh * ((6 + 2.0 / T_) * reals * prec + (2 + (1 if kind == tm.TM_KIND_XPAY_TWIST else 0)) * sp)
                ref_us = table["%s_fp%d_recon%d" % (name, prec * 8, reals)]["us"]
                tgt["%s_fp%d_recon%d" % (name, prec * 8, reals)] = {
                    "us": ms * 1e3, "GFLOPS": Vh * fl / ms / 1e6, "GBps_algorithmic": by / ms / 1e6, "bytes_per_site_minimal": by / Vh,
                    "frac_of_measured_%.0f" % hbm_peak: by / ms / 1e6 / hbm_peak, "time_over_ordinary_field": ms * 1e3 / ref_us}
            del g
        del bufs, xs, src
    del Utg
    out["dslash_temporal_gauge"] = tgt

    # loop contraction alone (fp16, 12 RHS): reads 2 full spinors per rhs
    prec = 2
    fb = tm.tm_spinor_bytes(L, prec, 1, NRHS)
    a, b = tm.device_buffer(fb), tm.device_buffer(fb)
    a.zero_(); b.zero_()
    lo = torch.zeros((NRHS, 16, DIMS[3], 2), dtype=torch.float64, device="cuda")
    lws = tm.device_buffer(tm.tm_loop_workspace_bytes(L, NRHS))
    f = lambda i: tm.tm_loop_contract(L, a, b, prec, NRHS, lo, lws)
    f(0)
    ms = time_events(torch, f, 10)
    out["loop_contract_fp16_x12"] = {"us": ms * 1e3, "GBps_algorithmic": 2 * fb / ms / 1e6, "frac_of_measured": 2 * fb / ms / 1e6 / hbm_peak}
    # NEXT-2 / NEXT-3 rows at 32^3x64: momentum-projected loops for the p^2 <= 9 list (123 momenta), the
    # contraction field, the covariant derivative and the HPE remainder; algorithmic bytes as for the loop kernel
    ins = {}
    r = int(np.floor(np.sqrt(9)))
    mom = np.array([(x, y, z) for x in range(-r, r + 1) for y in range(-r, r + 1) for z in range(-r, r + 1) if x * x + y * y + z * z <= 9],
                   dtype=np.int32)
    lm = torch.zeros((NRHS, 16, DIMS[3], len(mom), 2), dtype=torch.float64, device="cuda")
    mws = tm.device_buffer(tm.tm_loop_momentum_workspace_bytes(L, NRHS, len(mom), r))
    f = lambda i: tm.tm_loop_momentum(L, a, b, prec, NRHS, mom, lm, mws)
    f(0)
    ms = time_events(torch, f, 5)
    ins["loop_momentum_p2le9_fp16_x12"] = {"us": ms * 1e3, "momenta": int(len(mom)), "GBps_algorithmic": 2 * fb / ms / 1e6,
                                           "frac_of_measured": 2 * fb / ms / 1e6 / hbm_peak}
    del lm, mws
    fb1 = tm.tm_spinor_bytes(L, prec, 1, 1)
    cf = torch.empty((L.V, 32), dtype=torch.float64, device="cuda")
    f = lambda i: tm.tm_contract_field(L, a, b, prec, 1, cf)
    f(0)
    ms = time_events(torch, f, 10)
    by = 2 * fb1 + L.V * 256
    ins["contract_field_fp16"] = {"us": ms * 1e3, "GBps_algorithmic": by / ms / 1e6, "frac_of_measured": by / ms / 1e6 / hbm_peak}
    del cf
    for p_, rc_ in ((4, 18), (2, 12)):
        fbp = tm.tm_spinor_bytes(L, p_, 1, 1)
        vin, vout, vtmp = tm.device_buffer(fbp), tm.device_buffer(fbp), tm.device_buffer(fbp)
        tm.tm_spinor_pack(L, psi, p_, 1, vin)
        f = lambda i: tm.tm_covdev(L, gauges[(p_, rc_)], p_, rc_, vout, vin, i % 4, 1)
        f(0)
        ms = time_events(torch, f, 20)
        by = L.V * rc_ * p_ + 2 * fbp  # one link per site (each link serves a forward and a backward hop), spinor in + out
        ins["covdev_fp%d_recon%d" % (8 * p_, rc_)] = {"us": ms * 1e3, "GBps_algorithmic": by / ms / 1e6,
                                                     "frac_of_measured": by / ms / 1e6 / hbm_peak}
        f = lambda i: tm.tm_hpe_remainder(L, gauges[(p_, rc_)], p_, rc_, vout, vin, vtmp, kappa, mu, 1)
        f(0)
        ms = time_events(torch, f, 5)
        by = 8 * dslash_bytes(Vh, p_, rc_, False)
        ins["hpe_remainder_fp%d_recon%d" % (8 * p_, rc_)] = {"us": ms * 1e3, "launches": 8, "GBps_algorithmic": by / ms / 1e6,
                                                            "frac_of_measured": by / ms / 1e6 / hbm_peak}
        del vin, vout, vtmp
    out["insertions_next2_next3"] = ins
    del a, b

    # the truncated solve UNBATCHED (one source per call, single-rhs kernels): the batching gain of configs[3]
    fb2 = tm.tm_spinor_bytes(L, 2, 1, 1)
    e1, s1 = tm.device_buffer(fb2), tm.device_buffer(fb2)
    tm.tm_spinor_pack(L, psi, 2, 1, e1)
    ws1 = tm.device_buffer(tm.tm_cg_workspace_bytes(L, 8, 2, tm.TM_CG_LP_TRUNCATED, 1))
    prm1 = tm.make_cg_params(kappa, mu, LP_TOL, 500, tm.TM_CG_LP_TRUNCATED, 0.1, 0, 1)
    its = []
    def lp1(i):
        rc, info = tm.tm_cg(L, None, 8, gauges[(2, 12)], 2, 12, s1, e1, prm1, ws1)
        its.append(info.iters)
    lp1(0)
    ms = time_events(torch, lp1, 5)
    out["lp_unbatched_fp16_recon12"] = {"ms_per_solve": ms, "solves_per_s": 1e3 / ms, "iters": its[-1],
                                        "batched_over_unbatched": out["value"] / (1e3 / ms)}
    del e1, s1, ws1

    # the same batched TSM step with fp32 storage ("inversions ... in single or half precision")
    T = DIMS[3]
    codes4 = torch.from_numpy(np.stack([ti.z4_codes(DIMS, seed=ti.NOISE_SEED + r) for r in range(NRHS)])).cuda()
    fb4 = tm.tm_spinor_bytes(L, 4, 1, NRHS)
    eta4, sol4 = tm.device_buffer(fb4), tm.device_buffer(fb4)
    ws4 = tm.device_buffer(tm.tm_cg_workspace_bytes(L, 8, 4, tm.TM_CG_LP_TRUNCATED, NRHS))
    lws4 = tm.device_buffer(tm.tm_loop_workspace_bytes(L, NRHS))
    loops4 = torch.zeros((NRHS, 16, T, 2), dtype=torch.float64, device="cuda")
    it4 = []

    def step_fp32(i):
        tm.tm_spinor_pack_z4(L, codes4, 4, NRHS, eta4)
        rc, info = tm.tm_cg_multi(L, None, 8, gauges[(4, 12)], 4, 12, sol4, eta4, prm1, NRHS, ws4)
        assert rc == tm.TM_OK, rc
        tm.tm_loop_contract(L, eta4, sol4, 4, NRHS, loops4, lws4)
        it4.append(info[0].iters)
    step_fp32(0)
    ms4 = time_events(torch, step_fp32, 3)
    out["lp_batched_fp32_recon12"] = {"ms_per_step": ms4, "solves_per_s": NRHS / (ms4 * 1e-3), "iters": it4[-1],
                                      "fp32_over_fp16_time": ms4 / out["ms_per_step"]}
    del eta4, sol4, ws4

    # ... and with fp16 storage + 16-bit fixed-point links (TM_RECON_12_FIX16): the 12-rhs kernel reads the fp32 link cache, so the
    # more accurate links cost nothing there
    fbx = tm.tm_spinor_bytes(L, 2, 1, NRHS)
    etax, solx = tm.device_buffer(fbx), tm.device_buffer(fbx)
    wsx = tm.device_buffer(tm.tm_cg_workspace_bytes(L, 8, 2, tm.TM_CG_LP_TRUNCATED, NRHS))
    itx = []

    def step_fix16(i):
        tm.tm_spinor_pack_z4(L, codes4, 2, NRHS, etax)
        rc, info = tm.tm_cg_multi(L, None, 8, gauges[(2, 112)], 2, 112, solx, etax, prm1, NRHS, wsx)
        assert rc == tm.TM_OK, rc
        tm.tm_loop_contract(L, etax, solx, 2, NRHS, loops4, lws4)
        itx.append(info[0].iters)
    step_fix16(0)
    msx = time_events(torch, step_fix16, 3)
    out["lp_batched_fp16_recon12fix16"] = {"ms_per_step": msx, "solves_per_s": NRHS / (msx * 1e-3), "iters": itx[-1],
                                           "fix16_over_binary16_time": msx / out["ms_per_step"]}
    del codes4, etax, solx, wsx, lws4, loops4

    # mixed-precision CG to 1e-8 on one Z2xiZ2 source (configs[2]): fp64 reliable updates, fp32 and fp16 iterations
    cg = {}
    pb8 = tm.tm_spinor_bytes(L, 8, 1, 1)
    eta8, s8 = tm.device_buffer(pb8), tm.device_buffer(pb8)
    tm.tm_spinor_pack(L, psi, 8, 1, eta8)
    for plp in (4, 2):
        ws = tm.device_buffer(tm.tm_cg_workspace_bytes(L, 8, plp, tm.TM_CG_HP_MIXED, 1))
        prm = tm.make_cg_params(kappa, mu, 1e-8, 5000, tm.TM_CG_HP_MIXED, 0.1, 1)
        torch.cuda.synchronize()
        t0 = time.time()
        rc, info = tm.tm_cg(L, gauges[(8, 12)], 8, gauges[(plp, 12)], plp, 12, s8, eta8, prm, ws)
        torch.cuda.synchronize()
        dt = time.time() - t0
        cg["fp64+fp%d" % (plp * 8)] = {"status": rc, "iters": info.iters, "reliable_updates": info.reliable_updates,
                                       "true_resid": info.true_resid, "seconds": dt, "ms_per_iter": 1e3 * dt / max(1, info.iters)}
        del ws
    # the same tolerance by batched defect correction (TM_CG_HP_DEFECT): 12 sources share every gauge load of the inner solves;
    # stopping rule |eta - M s| <= 1e-8 |eta| on the full lattice
    del eta8, s8
    pb8n = tm.tm_spinor_bytes(L, 8, 1, NRHS)
    etaN, sN = tm.device_buffer(pb8n), tm.device_buffer(pb8n)
    c1 = tm.device_buffer(L.V * 12)
    for r in range(NRHS):
        c1.copy_(torch.from_numpy(ti.z4_codes(DIMS, seed=ti.NOISE_SEED + 900 + r).reshape(-1)))
        tm.tm_spinor_pack_z4(L, c1, 8, 1, etaN[r * pb8:(r + 1) * pb8])
    for plp in (4, 2):
        ws = tm.device_buffer(tm.tm_cg_workspace_bytes(L, 8, plp, tm.TM_CG_HP_DEFECT, NRHS))
        prm = tm.make_cg_params(kappa, mu, 1e-8, 5000, tm.TM_CG_HP_DEFECT, 0.0)
        torch.cuda.synchronize()
        t0 = time.time()
        rc, info = tm.tm_cg_multi(L, gauges[(8, 12)], 8, gauges[(plp, 12)], plp, 12, sN, etaN, prm, NRHS, ws)
        torch.cuda.synchronize()
        dt = time.time() - t0
        cg["defect_x12_fp64+fp%d" % (plp * 8)] = {"status": rc, "nrhs": NRHS, "inner_iters": max(x.iters for x in info),
                                                 "cycles": max(x.reliable_updates for x in info),
                                                 "true_resid_full_system": max(x.true_resid for x in info), "seconds": dt,
                                                 "ms_per_solve": 1e3 * dt / NRHS, "HP_solves_per_s": NRHS / dt}
        del ws
    # ... and ONE source through the same mode (configs[2]'s "mixed-precision CG to 1e-8 on one Z2xiZ2 source"): nrhs = 1 takes the
    # fused single-rhs iteration without a link cache
    for plp in (4, 2):
        ws = tm.device_buffer(tm.tm_cg_workspace_bytes(L, 8, plp, tm.TM_CG_HP_DEFECT, 1))
        prm = tm.make_cg_params(kappa, mu, 1e-8, 5000, tm.TM_CG_HP_DEFECT, 0.0)
        best = None
        for rep in range(2):
            torch.cuda.synchronize()
            t0 = time.time()
            rc, info = tm.tm_cg_multi(L, gauges[(8, 12)], 8, gauges[(plp, 12)], plp, 12, sN[:pb8], etaN[:pb8], prm, 1, ws)
            torch.cuda.synchronize()
            dt = time.time() - t0
            best = dt if best is None else min(best, dt)
        cg["defect_x1_fp64+fp%d" % (plp * 8)] = {"status": rc, "inner_iters": info[0].iters, "cycles": info[0].reliable_updates,
                                                "true_resid_full_system": info[0].true_resid, "seconds": best}
        del ws
    del etaN, sN, c1
    out["cg_mixed_1e-8"] = cg
    # the paper's per-configuration TSM workload (N_HP = 8, N_LP = 200) from the rates measured above
    hp = cg.get("defect_x12_fp64+fp16")
    if hp:
        n_hp, n_lp = 8, 200
        out["tsm_per_configuration"] = {
            "n_hp": n_hp, "n_lp": n_lp, "seconds": n_hp * hp["ms_per_solve"] * 1e-3 + (n_hp + n_lp) / out["value"],
            "R_HP_over_LP": hp["ms_per_solve"] * 1e-3 * out["value"],
            "note": "derived: N_HP solves to 1e-8 (batched defect correction) + (N_HP + N_LP) truncated solves with their loops, at the "
                    "rates measured in this run on the synthetic eps = 0.5 field (9 / 62 iterations; a physical light-quark ensemble "
                    "needs about 10x more).  Context: PAPER.md Table I R_HP/LP = 17-27 (light, strange), Table II 1471 GPU-node-seconds"}
    # ... and the same workload actually RUN: all sources made on the device (tm_noise_z4), N_HP = 8 sources solved to 1e-8 (batched defect
    # correction, fp64 loops), the same 8 and 200 further sources solved in the truncated mode in batches of 12, every solution contracted
    # (16 Gamma x T), Eq. (8) combined on the device (tm_tsm_combine).  Wall clock around the whole configuration, one stream.
    n_hp, n_lp, T = 8, 200, DIMS[3]
    seed0 = ti.NOISE_SEED + 5000
    fb2_ = tm.tm_spinor_bytes(L, 2, 1, NRHS)
    e2_, s2_ = tm.device_buffer(fb2_), tm.device_buffer(fb2_)
    fb8_ = tm.tm_spinor_bytes(L, 8, 1, n_hp)
    e8_, s8_ = tm.device_buffer(fb8_), tm.device_buffer(fb8_)
    ws_lp = tm.device_buffer(tm.tm_cg_workspace_bytes(L, 8, 2, tm.TM_CG_LP_TRUNCATED, NRHS))
    ws_hp = tm.device_buffer(tm.tm_cg_workspace_bytes(L, 8, 2, tm.TM_CG_HP_DEFECT, n_hp))
    lws_ = tm.device_buffer(tm.tm_loop_workspace_bytes(L, NRHS))
    l_hp = torch.zeros((n_hp, 16, T, 2), dtype=torch.float64, device="cuda")
    l_lp = torch.zeros((n_hp + n_lp, 16, T, 2), dtype=torch.float64, device="cuda")
    l_out = torch.zeros((16, T, 2), dtype=torch.float64, device="cuda")
    prm_lp = tm.make_cg_params(kappa, mu, LP_TOL, 500, tm.TM_CG_LP_TRUNCATED, 0.1, 0, 1)
    prm_hp = tm.make_cg_params(kappa, mu, 1e-8, 5000, tm.TM_CG_HP_DEFECT, 0.0)

    def configuration():
        tm.tm_noise_z4(L, seed0, 1, 8, n_hp, e8_)
        rc, _ = tm.tm_cg_multi(L, gauges[(8, 12)], 8, gauges[(2, 12)], 2, 12, s8_, e8_, prm_hp, n_hp, ws_hp)
        assert rc == tm.TM_OK, rc
        tm.tm_loop_contract(L, e8_, s8_, 8, n_hp, l_hp, lws_)
        for first in range(0, n_hp + n_lp, NRHS):
            n = min(NRHS, n_hp + n_lp - first)
            tm.tm_noise_z4(L, seed0 + first, 1, 2, n, e2_)
            rc, _ = tm.tm_cg_multi(L, None, 8, gauges[(2, 12)], 2, 12, s2_, e2_, prm_lp, n, ws_lp)
            assert rc == tm.TM_OK, rc
            tm.tm_loop_contract(L, e2_, s2_, 2, n, l_lp[first:first + n], lws_)
        tm.tm_tsm_combine(T, l_hp, l_lp[:n_hp], n_hp, l_lp[n_hp:], n_lp, l_out)

    configuration()
    torch.cuda.synchronize()
    t0 = time.time()
    configuration()
    torch.cuda.synchronize()
    dt_cfg = time.time() - t0
    tr = l_out.cpu().numpy()
    out["tsm_configuration_measured"] = {"n_hp": n_hp, "n_lp": n_lp, "seconds": dt_cfg, "solves": 2 * n_hp + n_lp,
                                         "loop_Gamma0_t0_re": float(tr[0, 0, 0]), "loop_Gamma15_t0_im": float(tr[15, 0, 1]),
                                         "note": "one configuration of the paper's TSM workload (PAPER.md:106, :226) run end to end on the device: noise, "
                                                 "8 HP + 208 LP solves, 216 contractions, Eq. (8); synthetic field (9 / 63 iterations per solve)"}
    del e2_, s2_, e8_, s8_, ws_lp, ws_hp, lws_
    if world == 1:
        # ~26 s of oracle work on the GPU box; the --impl reference arm keeps the 1.5 s sample so that its K + W steps stay short
        base, _ = cpu_oracle_sample(large=True)
        out["cpu_baseline"] = base


def sweep_other_configs(torch, tm, ti, hbm_peak, out):
    """`--sweeps`: BASELINE.json configs[1] (16^3x32 fp32, 100 applications captured in a CUDA graph: L2 / launch-latency
    regime, NOT an HBM roofline point) and configs[4] (64^3x128: the clean HBM-bound sweep, working set >> L2)."""
    kappa, mu = ti.KAPPA, ti.MU
    # ---- configs[1] ----
    dims = (16, 16, 16, 32)
    L = tm.tm_lattice_create(dims, True)
    Vh = L.V // 2
    U = torch.from_numpy(ti.gauge(dims).view(np.float64)).cuda()
    psi = torch.from_numpy(ti.z4(dims).view(np.float64)).cuda()
    small = {}
    prec = 4
    pb = tm.tm_spinor_bytes(L, prec, 0, 1)
    src = tm.device_buffer(2 * pb)
    tm.tm_spinor_pack(L, psi, prec, 1, src)
    a, b, tmp = tm.device_buffer(pb), tm.device_buffer(pb), tm.device_buffer(2 * pb)
    for recon in (18, 12):
        g = tm.device_buffer(tm.tm_gauge_bytes(L, prec, recon))
        tm.tm_gauge_pack(L, U, prec, recon, g, 1e-10)
        for name, fl, by in (("twist_inv", FLOPS_TWIST_INV, dslash_bytes(Vh, prec, recon, False)),
                             ("MdagM", 2 * (FLOPS_TWIST_INV + FLOPS_XPAY), 2 * dslash_bytes(Vh, prec, recon, False) + 2 * dslash_bytes(Vh, prec, recon, True))):
            st = torch.cuda.Stream()
            def body():
                for i in range(100):
                    o, inp = (a, b) if i % 2 == 0 else (b, a)
                    if name == "twist_inv":
                        tm.tm_dslash(L, g, prec, recon, o, src[pb:2 * pb] if i == 0 else inp, None, 0, 0, tm.TM_KIND_TWIST_INV, kappa, mu)
                    else:
                        tm.tm_MdagM(L, g, prec, recon, o, src[:pb] if i == 0 else inp, tmp, 0, kappa, mu)
            with torch.cuda.stream(st):
                body()  # warm-up (also loads the modules before capture)
                st.synchronize()
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=st):
                    body()
                ts = []
                for _ in range(5):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(st); graph.replay(); e1.record(st); st.synchronize()
                    ts.append(e0.elapsed_time(e1) / 100)
            ms = float(np.median(ts))
            small["%s_fp32_recon%d" % (name, recon)] = {"us": ms * 1e3, "GFLOPS": Vh * fl / ms / 1e6, "GBps_algorithmic": by / ms / 1e6}
    out["config1_16x32_fp32_graph"] = {"note": "L2-resident working set (<= 50 MB), 100 applications in one CUDA graph, median of 5: "
                                       "L2 / launch-latency regime, not an HBM roofline point", "table": small}
    del U, psi, src, a, b, tmp
    # ---- configs[4] ----
    dims = (64, 64, 64, 128)
    X, Y, Z, T = dims
    L = tm.tm_lattice_create(dims, True)
    Vh = L.V // 2
    # 19.3 GB of canonical fp64 links: made on the device by the library's restatement of the input generator (tm_gauge_synthetic)
    U = torch.empty(T * X * Y * Z * 4 * 18, dtype=torch.float64, device="cuda")
    tm.tm_gauge_synthetic(L, ti.GAUGE_SEED, 1.0, ti.EPS, U)
    gauges = {}
    for prec in (4, 2):
        for recon in (18, 12):
            gauges[(prec, recon)] = tm.device_buffer(tm.tm_gauge_bytes(L, prec, recon))
            tm.tm_gauge_pack(L, U, prec, recon, gauges[(prec, recon)], 1e-10)
    del U
    torch.cuda.empty_cache()
    codes = torch.empty((T, Z, Y, X, 4, 3), dtype=torch.uint8, device="cuda")
    for t0 in range(0, T, 16):
        codes[t0:t0 + 16].copy_(torch.from_numpy(ti.z4_codes(dims, t0=t0, t1=t0 + 16)))
    big = {}
    for prec in (4, 2):
        pb = tm.tm_spinor_bytes(L, prec, 0, 1)
        src = tm.device_buffer(2 * pb)
        tm.tm_spinor_pack_z4(L, codes, prec, 1, src)
        o, x, tmp = tm.device_buffer(pb), tm.device_buffer(pb), tm.device_buffer(2 * pb)
        x.copy_(src[:pb])
        for recon in (18, 12):
            g = gauges[(prec, recon)]
            runs = (("twist_inv", FLOPS_TWIST_INV, dslash_bytes(Vh, prec, recon, False),
                     lambda i: tm.tm_dslash(L, g, prec, recon, o, src[pb:2 * pb], None, 0, 0, tm.TM_KIND_TWIST_INV, kappa, mu)),
                    ("xpay_twist", FLOPS_XPAY, dslash_bytes(Vh, prec, recon, True),
                     lambda i: tm.tm_dslash(L, g, prec, recon, o, src[pb:2 * pb], x, 0, 0, tm.TM_KIND_XPAY_TWIST, kappa, mu)),
                    ("MdagM", 2 * (FLOPS_TWIST_INV + FLOPS_XPAY), 2 * dslash_bytes(Vh, prec, recon, False) + 2 * dslash_bytes(Vh, prec, recon, True),
                     lambda i: tm.tm_MdagM(L, g, prec, recon, o, src[:pb], tmp, 0, kappa, mu)))
            for name, fl, by, fn in runs:
                for i in range(3):
                    fn(i)
                ms = min(time_events(torch, fn, 10) for _ in range(3))
                big["%s_fp%d_recon%d" % (name, prec * 8, recon)] = {
                    "us": ms * 1e3, "GFLOPS": Vh * fl / ms / 1e6, "GBps_algorithmic": by / ms / 1e6,
                    "frac_of_measured_%.0f" % hbm_peak: by / ms / 1e6 / hbm_peak, "frac_of_nominal_8000": by / ms / 1e6 / 8000.0}
        del src, o, x, tmp
    for prec_, nm in ((4, "fp32"), (2, "fp16")):  # flat scalars where the driver's parse keeps them (TWIST_INV, single rhs, 64^3x128)
        for rc_ in (18, 12):
            row = big["twist_inv_fp%d_recon%d" % (prec_ * 8, rc_)]
            out["roofline"]["dslash64_%s_r%d_frac" % (nm, rc_)] = row["frac_of_measured_%.0f" % hbm_peak]
            out["roofline"]["dslash64_%s_r%d_us" % (nm, rc_)] = row["us"]
    out["config4_64x128"] = {"note": "33.5 M sites; gauge 3.2-9.7 GB + spinors 0.9-1.6 GB per parity: every launch streams from HBM",
                             "table": big}


def free_port():
    import socket
    sk = socket.socket()
    sk.bind(("127.0.0.1", 0))
    port = sk.getsockname()[1]
    sk.close()
    return port


def run_dry(args, rank, world):
    """--dry-run (CPU, gloo): the launcher and the N > 1 host logic without a GPU -- rendezvous, the source partition, the one
    gather of the [16][T] loops, max-over-ranks of a time -- with stand-in loops that encode their source index."""
    import torch
    import torch.distributed as dist
    from paper_1309_2256_b200 import shard
    if world > 1:
        dist.init_process_group("gloo")
    T = DIMS[3]
    n = world * NRHS
    ids = shard.owned_sources(n, NRHS, rank, world)
    local = torch.stack([torch.full((16, T, 2), float(r), dtype=torch.float64) for r in ids])
    gather = shard.LoopGather(n, NRHS, (16, T, 2), torch.float64, torch.device("cpu"))
    full = gather(local)
    ok = bool(all(torch.all(full[r] == float(r)) for r in range(n)))
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    ranks = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_gather(ranks, torch.tensor([float(rank)], dtype=torch.float64))
    if rank == 0:
        print(json.dumps({"dry_run": True, "n_gpus": world, "ranks_reported": [int(x.item()) for x in ranks], "gather_in_source_order": ok,
                          "max_over_ranks": float(t.item()), "sources": n}))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--sweeps", action="store_true", help="kept for compatibility: configs[1] and [4] are timed by default now")
    ap.add_argument("--no-sweeps", action="store_true", help="skip BASELINE.json configs[1] (16^3x32, CUDA graph) and [4] (64^3x128; needs ~35 GB of HBM, ~6 s)")
    ap.add_argument("--dry-run", action="store_true", help="CPU / gloo run of the launcher and the multi-rank host logic only (no GPU, no timing)")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("--gpus must be >= 1")
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference":
        # started bare: launch one rank per GPU ourselves (the driver's torchrun line sets WORLD_SIZE and skips this)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus), "--master-addr", "127.0.0.1",
               "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
        os.environ.setdefault("NCCL_DEBUG", "WARN")
        sys.stdout.flush()
        os.execv(sys.executable, cmd)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if world != args.gpus:
        raise SystemExit("bench.py --gpus %d was started with WORLD_SIZE=%d: the rank count must equal --gpus" % (args.gpus, world))
    if args.dry_run:
        run_dry(args, rank, world)
        return
    if args.warmup < 3:
        args.warmup = 3
    run_b200(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
