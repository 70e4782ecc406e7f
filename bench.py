#!/usr/bin/env python
"""bench.py -- SFFT subtractions/sec per 2048x4096 fp64 CCD on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

A "step" is one pass of the whole hot path (sfft_build_system + sfft_solve + sfft_subtract) over
one synthetic full-DECam-CCD pair (BASELINE.json configs[3]: 2048x4096 fp64, w=5, DK=2, DB=2,
N=732).  Inputs are seeded synthetic star fields (paper_2603_08593_b200/synth.py) standing in for
the paper's DESIRT exposures.  `value` is device-timed with inputs resident in HBM; `e2e` is the
same metric with pinned HOST buffers, H2D/D2H copies inside the timed region (3 plans on 3 streams
so copies overlap compute).  Prints ONE JSON line on rank 0.  N>1 shards CCDs over ranks (weak
scaling, no data-path collective).

`--impl reference` times the CPU oracle (oracle/sfft_oracle.py) as it stands on host cores, each
step a bounded sample (a 512x1024 crop) of the same workload.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "SFFT subtractions/sec per 2048x4096 fp64 CCD"
UNIT = "CCD/s"
WORKLOAD = "full DECam CCD (BASELINE.json configs[3]): 2048x4096 fp64, w=5, DK=2, DB=2, N=732"
SOLVE_CTAS_PIPELINED = 16   # sfft_plan_set_solve_ctas for the multi-plan legs (e2e, exposure); 8..74 swept: 16 is best
NPAIR = 3  # distinct resident pairs cycled through (3 x 143 MB of inputs > 126 MB L2)

# fp64-pipe peak derived from unit counts and clocks: 148 SMs x 4 SMSPs x 16
# fp64 lanes x 2 flop x clocks.max.sm; one DP-pipe instruction slot is counted as 2 flop.
def alu_peak_tflops(sm_max_mhz):
    return 148 * 4 * 16 * 2 * sm_max_mhz * 1e6 / 1e12


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


class ClockSampler:
    """Samples SM clocks and throttle reasons DURING the timed region: NVML polled every ~2 ms from a
    thread (the timed region is only tens of milliseconds), nvidia-smi as the fallback."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    BITS = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40}

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thr, self.stop_flag = index, [], None, None, False
        self.nvml, self.handle = None, None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[self.index]) if vis and vis.split(",")[self.index].isdigit() else self.index
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.nvml = pynvml
            self.thr = threading.Thread(target=self._poll_nvml, daemon=True)
            self.thr.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thr = threading.Thread(target=self._read, daemon=True)
        self.thr.start()

    def _poll_nvml(self):
        n = self.nvml
        mx = n.nvmlDeviceGetMaxClockInfo(self.handle, n.NVML_CLOCK_SM)
        while not self.stop_flag:
            try:
                sm = n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM)
                try:
                    rs = n.nvmlDeviceGetCurrentClocksEventReasons(self.handle)
                except Exception:
                    rs = n.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle)
                self.rows.append((time.time(), (float(sm), float(mx), int(rs))))
            except Exception:
                pass
            time.sleep(0.002)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def mark(self):
        return time.time()

    def stop(self, t0, t1):
        if self.nvml is not None:
            self.stop_flag = True
            self.thr.join(timeout=1.0)
            rows = [r for (t, r) in self.rows if t0 <= t <= t1] or [r for (_, r) in self.rows[-3:]]
            sm = [r[0] for r in rows]
            reasons = sorted({name for r in rows for name, bit in self.BITS.items() if r[2] & bit})
            return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": rows[0][1] if rows else None,
                    "samples": len(sm), "reasons": reasons, "source": "nvml, polled every 2 ms in the timed region"}
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows[-3:]]
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons), "source": "nvidia-smi"}


def oracle_cores():
    return len(os.sched_getaffinity(0))


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


# ------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle on a bounded sample


def run_reference(args, rank, world):
    if rank != 0:
        return
    import numpy as np
    from oracle import sfft_oracle as orc
    from paper_2603_08593_b200 import synth
    pr = synth.make_pair("full")
    cfg = pr.cfg
    ch, cw = 512, 1024
    y0, x0 = (cfg.H - ch) // 2, (cfg.W - cw) // 2
    R = np.ascontiguousarray(pr.R[y0:y0 + ch, x0:x0 + cw])
    S = np.ascontiguousarray(pr.S[y0:y0 + ch, x0:x0 + cw])
    M = np.ascontiguousarray(pr.mask[y0:y0 + ch, x0:x0 + cw])
    M[:6] = 1; M[-6:] = 1; M[:, :6] = 1; M[:, -6:] = 1
    cores = oracle_cores()
    frac = (ch * cw) / float(cfg.H * cfg.W)

    def step():
        orc.sfft_difference(R, S, M, cfg.w, cfg.DK, cfg.DB, workers=cores)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    value = args.steps * frac / dt
    sample = (f"{ch}x{cw} centre crop (1/{int(round(1 / frac))} of the CCD's pixels) of the configs[3] pair, same w/DK/DB; "
              "CCD/s = crop fraction / time, i.e. extrapolated LINEARLY in pixels -- the full-CCD oracle leg of the "
              "CUDA arm (cpu_baseline) runs ~1.9x slower per pixel (cache effects, N log N), so this line flatters the CPU")
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------------------------
# CUDA arm


def stage_models(plan_dims, peaks, alu_peak):
    """Algorithmic DP-pipe instructions and compulsory HBM bytes of each stage for ONE step
    (DESIGN.md "Cost model").  Returns {stage: (dp_instr, hbm_bytes)}."""
    H, W, w, DK, DB = plan_dims
    NC, P = W // 2, H * W
    TK, TB = (DK + 1) * (DK + 2) // 2, (DB + 1) * (DB + 2) // 2
    L = (2 * w + 1) ** 2
    N = L * TK + TB
    nRow, nSpec = DK + 1 + 1, TK + 1   # lean plan: the kernel-background block needs no transform

    def fft_instr(n):  # Stockham radix-16/8/4 passes as implemented (fft_smem.cuh)
        plans = {8: [8], 16: [16], 32: [8, 4], 64: [8, 8], 128: [16, 8], 256: [16, 16], 512: [8, 8, 8],
                 1024: [16, 8, 8], 2048: [16, 16, 8], 4096: [16, 16, 16]}
        bfly = {4: 16, 8: 56, 16: 160}
        tot = 0.0
        for i, r in enumerate(plans[n]):
            tot += (n / r) * (bfly[r] + (0 if i == 0 else 4 * (r - 1)))
        return tot

    rowfft = fft_instr(NC) + 8.0 * NC
    nKK, nKS = TK * (TK + 1) // 2, TK
    col_pair = lambda D: H * 4.0 + (H / 8.0) * (58.0 + 8.0 * D)
    m = {}
    m["build.row_fwd"] = (nRow * H * rowfft, 2 * P * 8 + P + nRow * P * 8)
    m["build.col_fwd"] = (nSpec * NC * fft_instr(H), (nRow + nSpec) * P * 8)
    # blocked column/cross kernel (k_colb): per column ceil(H/B) blocks of B = 128 - 4w centre rows; per
    # block 2 TK + 1 transforms of 128 points (radix 8 x 16: 16 x (56 + 7 x 4) + 8 x 160), the eta^q
    # weights (2 per element of the sequences with q >= 1), one complex multiply-add per pair and
    # frequency; per column one 16-point inverse per (pair, a) and 8 twiddled terms per lag.  What the
    # METHOD needs, not what the kernel executes.  HBM: the row spectra in, the lag rows out.
    Bc = 128 - 4 * w
    nblk = -(-H // Bc)
    fft128 = 16 * (56 + 7 * 4) + 8 * 160
    nq1 = TK - (DK + 1)                      # monomials with q >= 1 (centre and extended version each)
    per_block = (2 * TK + 1) * fft128 + 2 * nq1 * 2 * 128 + (nKK + nKS) * 128 * 4
    per_col = nblk * per_block + (nKK + nKS) * 8 * 160 + (nKK * (4 * w + 1) + nKS * (2 * w + 1)) * 8 * 4
    m["build.colx"] = ((NC + 1) * per_col,
                       nRow * H * (NC + 1) * 16 + (nKK * (4 * w + 1) + nKS * (2 * w + 1)) * (NC + 1) * 16)
    m["build.cross_KK"] = ((NC + 1) * nKK * col_pair(2 * w), TK * P * 8)
    m["build.cross_KS"] = ((NC + 1) * nKS * col_pair(w), nSpec * P * 8)
    # sparse kernel-background part: ~1% special pixels (border), L shifts, TK*TB products; reads the mask twice
    m["build.kb_sparse"] = (0.01 * P * L * TK * TB, 2.0 * P)
    m["build.lag_gather"] = ((nKK * (4 * w + 1) * (2 * w + 1) + nKS * (2 * w + 1) * (w + 1)) * NC * 4.0, N * N * 8.0)
    m["solve"] = (N ** 3 / 6.0 + 2.0 * N * N, 2.0 * N * N * 8)
    m["subtract.row_fwd"] = ((DK + 1) * H * rowfft, P * 8 + (DK + 1) * P * 8)
    per_v = sum(2 * (DK - p) + 4 for p in range(DK + 1))
    m["subtract.mix"] = (P / 2.0 * (2 * w + 1) * per_v, (DK + 1) * P * 8 + P * 8)
    m["subtract.row_inv"] = (H * rowfft + P * (2 + 2 * TB), 3 * P * 8)
    # textbook flop count of the same kernel (5 n log2 n per complex transform, 8 per complex multiply-add,
    # 2 per real x complex scaling), for the conventional fraction quoted beside the slot-based one
    tb_block = (2 * TK + 1) * 5 * 128 * 7 + 2 * nq1 * 2 * 128 + (nKK + nKS) * 128 * 8
    tb_col = nblk * tb_block + (nKK + nKS) * 8 * 5 * 16 * 4 + (nKK * (4 * w + 1) + nKS * (2 * w + 1)) * 8 * 8
    m["_textbook_flop"] = {"build.colx": (NC + 1) * tb_col}
    return m


def run_exposure(torch, synth, cfg, plans, streams, nccd):
    """BASELINE.json configs[4]: `nccd` independent full-CCD pairs (per-CCD seed 2000+k, sky level
    U[800,3000] ADU, science FWHM U[3.5,6] px), resident in HBM, processed back to back on one GPU
    with len(plans) plans in flight.  Returns host wall-clock from first launch to final sync."""
    import concurrent.futures as cf
    import numpy as np
    rng = np.random.default_rng(2000)
    sky = rng.uniform(800.0, 3000.0, nccd)
    fwhm = rng.uniform(3.5, 6.0, nccd)
    N = plans[0].N
    dev = []
    tg = time.perf_counter()
    with cf.ThreadPoolExecutor(max_workers=min(8, oracle_cores())) as ex:
        for pr in ex.map(lambda k: synth.make_pair("full", seed=2000 + k, sky0=float(sky[k]), fwhm_s=float(fwhm[k])),
                         range(nccd)):
            dev.append((torch.from_numpy(pr.R).cuda(), torch.from_numpy(pr.S).cuda(), torch.from_numpy(pr.mask).cuda()))
    gen_s = time.perf_counter() - tg
    NS = len(plans)
    Ds = [torch.empty((cfg.H, cfg.W), dtype=torch.float64, device="cuda") for _ in range(nccd)]
    cs = torch.empty((nccd, N), dtype=torch.float64, device="cuda")
    infos = torch.zeros(nccd, dtype=torch.int32, device="cuda")
    As = [torch.empty((N, N), dtype=torch.float64, device="cuda") for _ in range(NS)]
    bs = [torch.empty(N, dtype=torch.float64, device="cuda") for _ in range(NS)]

    def run_all():
        for k in range(nccd):
            s = k % NS
            R, S, M = dev[k]
            st, pl = streams[s], plans[s]
            pl.build_system(R, S, M, As[s], bs[s], stream=st)
            pl.subtract_prepare(R, stream=st)
            pl.solve(As[s], bs[s], cs[k], infos[k:k + 1], stream=st)
            pl.subtract(R, S, cs[k], Ds[k], stream=st)

    torch.cuda.synchronize()
    run_all()                       # warm-up pass over the whole exposure
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    run_all()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    ok = bool((infos == 0).all().item())
    inputs_gb = nccd * (2 * cfg.H * cfg.W * 8 + cfg.H * cfg.W) / 1e9

    # the same exposure with the 60 pairs in PINNED HOST memory: every CCD's R, S, mask cross PCIe inside
    # the timed region; D and the coefficients stay in HBM as above
    wall_h2d = None
    try:
        hostp = [tuple(t.cpu().pin_memory() for t in trip) for trip in dev]
        stg = [tuple(torch.empty_like(t) for t in dev[0]) for _ in range(NS)]

        def run_all_h2d():
            for k in range(nccd):
                s = k % NS
                st, pl = streams[s], plans[s]
                R, S, M = stg[s]
                with torch.cuda.stream(st):
                    for d, h in zip((R, S, M), hostp[k]):
                        d.copy_(h, non_blocking=True)
                pl.build_system(R, S, M, As[s], bs[s], stream=st)
                pl.subtract_prepare(R, stream=st)
                pl.solve(As[s], bs[s], cs[k], infos[k:k + 1], stream=st)
                pl.subtract(R, S, cs[k], Ds[k], stream=st)

        torch.cuda.synchronize()
        run_all_h2d()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        run_all_h2d()
        torch.cuda.synchronize()
        wall_h2d = time.perf_counter() - t0
        ok = ok and bool((infos == 0).all().item())
        del hostp
    except RuntimeError as e:       # not enough pinnable host memory on this box
        wall_h2d = None
        h2d_err = str(e).splitlines()[0][:120]
    out = {"ccds": nccd, "wall_s": wall, "ccd_per_s": nccd / wall, "plans_in_flight": NS, "solve_ctas": SOLVE_CTAS_PIPELINED, "all_spd": ok,
           "inputs_resident_gb": round(inputs_gb, 2), "generation_s": round(gen_s, 1),
           "wall_s_incl_h2d": wall_h2d, "ccd_per_s_incl_h2d": (nccd / wall_h2d) if wall_h2d else None,
           "h2d_gb": round(inputs_gb, 2),
           "how": "configs[4]: per-CCD seed 2000+k, sky0~U[800,3000], S FWHM~U[3.5,6]; wall_s: inputs and outputs resident "
                  "in HBM; wall_s_incl_h2d: the 60 pairs start in pinned host memory and R, S, mask of every CCD are copied "
                  "to the device inside the timed region (PCIe-bound); host wall-clock of the second pass from first launch "
                  "to final synchronize; the paper's ~50 s per exposure (PAPER.md:305, whole Stage 2 on 64 cores + 2x A100) "
                  "is context only"}
    if wall_h2d is None:
        out["h2d_error"] = h2d_err
    return out


def run_cuda(args, rank, world, local_rank):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2603_08593_b200 import SfftPlan, shard, synth
    from paper_2603_08593_b200.binding import probe_fp64

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SFFT hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    peaks = load_peaks()
    alu_peak = alu_peak_tflops(peaks["sm_max_mhz"])

    cfg = synth.CONFIGS["full"]
    pairs = [synth.make_pair("full", seed=cfg.seed + 97 * rank + 1000 * i if (i or rank) else None)
             for i in range(NPAIR)]
    host = [(torch.from_numpy(p.R).pin_memory(), torch.from_numpy(p.S).pin_memory(),
             torch.from_numpy(p.mask).pin_memory()) for p in pairs]
    devp = [(r.cuda(), s.cuda(), m.cuda()) for (r, s, m) in host]
    plan = SfftPlan(cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB)
    N = plan.N
    A = torch.empty((N, N), dtype=torch.float64, device="cuda")
    b = torch.empty(N, dtype=torch.float64, device="cuda")
    c = torch.empty(N, dtype=torch.float64, device="cuda")
    info = torch.zeros(1, dtype=torch.int32, device="cuda")
    D = torch.empty((cfg.H, cfg.W), dtype=torch.float64, device="cuda")

    def step(k):
        R, S, M = devp[k % NPAIR]
        plan.build_system(R, S, M, A, b)
        plan.subtract_prepare(R)          # coefficient-independent stage of subtract, overlaps the solve
        plan.solve(A, b, c, info)
        plan.subtract(R, S, c, D)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    warm = max(3, args.warmup)
    for k in range(warm):
        step(k)
    torch.cuda.synchronize()
    assert int(info.item()) == 0, "Cholesky reported a non-positive-definite system"
    launches = sum(plan.last_launch_count(i) for i in range(3))

    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    t0 = sampler.mark()
    evs[0].record()
    for k in range(args.steps):
        step(k)
        evs[k + 1].record()
    barrier()
    t1 = sampler.mark()
    ms = evs[0].elapsed_time(evs[-1])
    ms_median = statistics.median(evs[k].elapsed_time(evs[k + 1]) for k in range(args.steps))
    # per-stage times: a second pass over the same steps with the library's stage events on (the ~18 event
    # records per step cost about 4 % of the step, so they stay out of the timed region above)
    plan.profile_enable(True)
    plan.profile_read(reset=True)
    pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pe0.record()
    for k in range(args.steps):
        step(k)
    pe1.record()
    torch.cuda.synchronize()
    ms_profiled = pe0.elapsed_time(pe1) / args.steps
    stages = plan.profile_read(reset=True)
    if plan.fused:   # stage slot 1 holds the fused column-pass + cross kernel
        stages = {("build.colx" if k == "build.col_fwd" else k): v for k, v in stages.items()}
    plan.profile_enable(False)
    clocks = sampler.stop(t0, t1)
    ms = shard.max_over_ranks(ms, device="cuda")
    value = shard.aggregate_rate(args.steps, world, ms)

    # ---- end to end: pinned host buffers, 3 plans on 3 streams, copies inside the timed region
    NS = 3
    streams = [torch.cuda.Stream() for _ in range(NS)]
    plans = [plan] + [SfftPlan(cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB) for _ in range(NS - 1)]
    for pl in plans:   # several plans in flight: a small Cholesky grid leaves whole SMs to the others
        pl.set_solve_ctas(SOLVE_CTAS_PIPELINED)
    h2d, d2h = SfftPlan.host_bytes_per_call(cfg.H, cfg.W, N)

    def e2e_step(k):
        # the repo's public end-to-end call: pinned host R, S, mask in; D, coefficients, info out
        hR, hS, hM = host[k % NPAIR]
        return plans[k % NS].difference_host_async(hR, hS, hM, stream=streams[k % NS])

    for k in range(warm):
        e2e_step(k)
    barrier()
    main = torch.cuda.current_stream()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(main)
    for st in streams:
        st.wait_event(f0)
    for k in range(args.steps):
        e2e_step(k)
    for st in streams:
        ev = torch.cuda.Event()
        ev.record(st)
        main.wait_event(ev)
    f1.record(main)
    barrier()
    ms_e2e = f0.elapsed_time(f1)
    ms_e2e = shard.max_over_ranks(ms_e2e, device="cuda")
    e2e_value = shard.aggregate_rate(args.steps, world, ms_e2e)
    assert all(int(pl._stage["ih"].item()) == 0 for pl in plans)

    # ---- the two steps after the differencing, timed alone on the device
    post = None
    plan.set_solve_ctas(0)   # the single-plan legs below run with the default solve grid again
    if world == 1:
        from paper_2603_08593_b200 import aperture_stats, median_combine
        nT = 5   # N_TEMP default
        Dt = [torch.randn((cfg.H, cfg.W), dtype=torch.float64, device="cuda") * 40 for _ in range(nT)]
        sc = [1.0, 0.93, 1.1, 0.8, 1.25]
        outm = torch.empty_like(Dt[0])
        gq = torch.Generator(device="cuda").manual_seed(7)
        xs = torch.rand(1024, dtype=torch.float64, device="cuda", generator=gq) * cfg.W
        ys = torch.rand(1024, dtype=torch.float64, device="cuda", generator=gq) * cfg.H
        for _ in range(3):
            median_combine(Dt, sc, out=outm)
            aperture_stats(D, devp[0][2], xs, ys, 0.6731 * 5.0)
        g0, g1, g2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        reps = 10
        g0.record()
        for _ in range(reps):
            median_combine(Dt, sc, out=outm)
        g1.record()
        for _ in range(reps):
            aperture_stats(D, devp[0][2], xs, ys, 0.6731 * 5.0)
        gap = torch.cuda.Event(enable_timing=True)
        gap.record()
        torch.cuda.synchronize()
        from paper_2603_08593_b200 import resample_affine
        Maff = [2.3, 0.9995, 0.004, 1.7, -0.004, 0.9995]   # a small rotation + scale + shift
        rs_out = torch.empty((cfg.H, cfg.W), dtype=torch.float64, device="cuda")
        rs_flag = torch.empty((cfg.H, cfg.W), dtype=torch.uint8, device="cuda")
        for _ in range(3):
            resample_affine(devp[0][1], Maff, cfg.H, cfg.W, 3, out=rs_out, outside=rs_flag)
        g2.record()
        g3 = torch.cuda.Event(enable_timing=True)
        for _ in range(reps):
            resample_affine(devp[0][1], Maff, cfg.H, cfg.W, 3, out=rs_out, outside=rs_flag)
        g3.record()
        torch.cuda.synchronize()
        t_med, t_rs = g0.elapsed_time(g1) / reps, g2.elapsed_time(g3) / reps
        t_ap = g1.elapsed_time(gap) / reps
        rs_bytes = cfg.H * cfg.W * (8 + 8 + 1)
        med_bytes = (nT + 1) * cfg.H * cfg.W * 8
        post = {"median_combine": {"templates": nT, "ms": round(t_med, 4), "hbm_gbs": round(med_bytes / t_med / 1e6, 1),
                                   "frac_of_hbm_peak": round(med_bytes / t_med / 1e6 / peaks["hbm_gbs"], 4),
                                   "bytes": med_bytes},
                "resample_affine": {"lanczos_order": 3, "ms": round(t_rs, 4), "hbm_gbs": round(rs_bytes / t_rs / 1e6, 1),
                                    "frac_of_hbm_peak": round(rs_bytes / t_rs / 1e6 / peaks["hbm_gbs"], 4),
                                    "bytes": rs_bytes, "note": "36 taps from L1 and 12 weights per pixel: L1/fp64-bound, not HBM-bound"},
                "aperture_stats": {"positions": 1024, "radius_px": round(0.6731 * 5.0, 3), "ms": round(t_ap, 4),
                                   "bound": "latency (two small kernels)"}}
        # exact unmasked-pixel objective (NEXT-1): the ordinary build on the unmasked images + the masked
        # pixels' symmetric rank-K update
        Rx, Sx, Mx = devp[0]
        for _ in range(2):
            plan.build_system_exact(Rx, Sx, Mx, A, b)
        g4, g5 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g4.record()
        for _ in range(5):
            plan.build_system_exact(Rx, Sx, Mx, A, b)
        g5.record()
        torch.cuda.synchronize()
        t_ex = g4.elapsed_time(g5) / 5
        nmask = int((Mx != 0).sum().item())
        post["build_system_exact"] = {"ms": round(t_ex, 3), "masked_pixels": nmask,
                                      "note": "ordinary build with no mask + fully masked rows / columns through strip "
                                              "correlations (k_exact_strips.cu) + the other masked pixels (none for this "
                                              "frame mask) through the fp64 tensor-path rank-K update; round 1: 3.7 ms"}
        # multi-template MODE (NEXT-2): S against N_TEMP = 5 templates in one call (the science
        # image's row transform computed once), against 5 x the single-template chain + the median
        from paper_2603_08593_b200 import cut_stamps
        gt = torch.Generator(device="cuda").manual_seed(11)
        Rt = [Rx + 3.0 * torch.randn(Rx.shape, dtype=torch.float64, device="cuda", generator=gt) for _ in range(nT)]
        for _ in range(2):
            mt = plan.multi_template_difference(Rt, Sx, Mx, sc)
        g6, g7, g8 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        g6.record()
        for _ in range(3):
            mt = plan.multi_template_difference(Rt, Sx, Mx, sc)
        g7.record()
        for _ in range(3):
            sep = []
            for k in range(nT):
                plan.build_system(Rt[k], Sx, Mx, A, b)
                plan.subtract_prepare(Rt[k])
                plan.solve(A, b, c, info)
                sep.append(plan.subtract(Rt[k], Sx, c, mt[1][k]))
            median_combine(sep, sc, out=outm)
        g8.record()
        torch.cuda.synchronize()
        assert mt[3].cpu().tolist() == [0] * nT and torch.equal(outm, mt[0])
        t_mt, t_sep = g6.elapsed_time(g7) / 3, g7.elapsed_time(g8) / 3
        # the same mode with the templates spread over three plans (sfft_multi_template_difference_plans: the
        # solve of one template overlaps the transforms of the others; 16-CTA solve grids as in the exposure leg)
        helpers = [SfftPlan(cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB) for _ in range(2)]
        for q in [plan, *helpers]:
            q.set_solve_ctas(SOLVE_CTAS_PIPELINED)
        for _ in range(2):
            mt3 = plan.multi_template_difference(Rt, Sx, Mx, sc, helpers=helpers)
        g9, g10 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
        g9.record()
        for _ in range(3):
            mt3 = plan.multi_template_difference(Rt, Sx, Mx, sc, helpers=helpers)
        g10.record()
        torch.cuda.synchronize()
        assert all(torch.equal(a, b) for a, b in zip(mt3, mt))
        t_mt3 = g9.elapsed_time(g10) / 3
        plan.set_solve_ctas(0)
        for q in helpers:
            q.close()
        post["multi_template"] = {"templates": nT, "ms": round(t_mt, 3), "ms_separate_calls": round(t_sep, 3),
                                  "ms_three_plans": round(t_mt3, 3),
                                  "ccd_per_s": round(1e3 / t_mt, 1), "ccd_per_s_three_plans": round(1e3 / t_mt3, 1),
                                  "note": "one sfft_multi_template_difference call (row transform and moments of m S "
                                          "reused by templates 2..5) vs 5 x (build, prepare, solve, subtract) + "
                                          "sfft_median_combine; ms_three_plans: sfft_multi_template_difference_plans "
                                          "with the 5 templates spread over 3 plans (solves overlap the other "
                                          "templates' transforms); bitwise equal results (asserted)"}
        del mt, mt3, sep, Rt
        # three-channel stamps (NEXT-3): 1024 candidates, 63 x 63 pixels (size is the caller's)
        for _ in range(2):
            stp = cut_stamps(Sx, Rx, D, xs, ys, 63)
        g9, g10 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g9.record()
        for _ in range(reps):
            stp = cut_stamps(Sx, Rx, D, xs, ys, 63)
        g10.record()
        torch.cuda.synchronize()
        t_st = g9.elapsed_time(g10) / reps
        st_bytes = 2 * stp.numel() * 8
        post["cut_stamps"] = {"candidates": 1024, "size": 63, "ms": round(t_st, 4), "bytes": st_bytes,
                              "gbs": round(st_bytes / t_st / 1e6, 1),
                              "note": "gather of 1024 x 3 x 63 x 63 fp64 (read + write bytes counted; the output "
                                      "tensor is allocated inside the timed call)"}
        del Dt, outm, stp
        torch.cuda.empty_cache()

    exposure = None
    if world == 1 and args.exposure_ccds > 0:
        for pl in plans:
            pl._stage = None
            pl.set_solve_ctas(SOLVE_CTAS_PIPELINED)
        torch.cuda.empty_cache()
        exposure = run_exposure(torch, synth, cfg, plans, streams, args.exposure_ccds)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel + per-stage table
    models = stage_models((cfg.H, cfg.W, cfg.w, cfg.DK, cfg.DB), peaks, alu_peak)
    textbook = models.pop("_textbook_flop")
    # fp64 peak = the library's own DFMA probe, measured in this run (the derived figure is quoted beside it)
    alu_nominal = alu_peak
    try:
        dfma_tf, _ = probe_fp64(0, 20000)
    except Exception:
        dfma_tf = None
    if dfma_tf:
        alu_peak = dfma_tf
    table = []
    for name, (tot_ms, cnt) in stages.items():
        if cnt == 0:
            continue
        t_ms = tot_ms / cnt
        instr, byts = models[name]
        t_alu = 2 * instr / (alu_peak * 1e12) * 1e3
        t_hbm = byts / (peaks["hbm_gbs"] * 1e9) * 1e3
        bound = "alu" if t_alu >= t_hbm else "hbm"
        table.append({"stage": name, "ms": round(t_ms, 4), "share": None, "bound": bound,
                      "alu_tflops": round(2 * instr / (t_ms * 1e-3) / 1e12, 3),
                      "hbm_gbs": round(byts / (t_ms * 1e-3) / 1e9, 1),
                      "frac_of_roofline": round(max(t_alu, t_hbm) / t_ms, 4)})
    # the sparse kernel-background chain runs on the plan's side stream concurrently with the row
    # pass and the fused kernel: its span overlaps theirs and is not part of the critical path
    for r in table:
        if r["stage"] == "build.kb_sparse":
            r["overlapped"] = "side stream, concurrent with build.row_fwd / build.colx (span, not busy time)"
        if r["stage"] == "subtract.row_fwd":
            r["overlapped"] = ("side stream (sfft_subtract_prepare), concurrent with solve on about a third of the "
                               "SMs (span, not busy time; ~0.065 ms when run alone on the whole GPU)")
    serial = [r for r in table if "overlapped" not in r]
    tot = sum(r["ms"] for r in serial)
    for r in serial:
        r["share"] = round(r["ms"] / tot, 4)
    # dominant KERNEL: every stage is one kernel launch except `solve` (k_chol_fused + k_chol_back; the ncu
    # launch list under profiles/ puts k_chol_fused at 0.74 of the stage) and `build.lag_gather` (two small ones)
    largest_kernel_share = {"solve": 0.74, "build.lag_gather": 0.7}
    dom = max(serial, key=lambda r: r["ms"] * largest_kernel_share.get(r["stage"], 1.0))
    instr, byts = models[dom["stage"]]
    if dom["bound"] == "alu":
        roof = {"kernel": dom["stage"], "bound": "alu", "achieved": dom["alu_tflops"], "peak": round(alu_peak, 2),
                "unit": "TFLOP/s", "frac": round(dom["alu_tflops"] / alu_peak, 4), "traffic": NCU_TRAFFIC.get(dom["stage"]),
                "traffic_source": NCU_SOURCE,
                "peak_source": "measured in this run: sfft_probe_fp64 (dependent-free DFMA loop on every SM); one DP-pipe "
                               "instruction slot (DFMA, DADD or DMUL) = 2 flop; algorithmic instruction count of the "
                               "blocked column/cross algorithm (DESIGN.md section 5)",
                "peak_nominal": round(alu_nominal, 2),
                "peak_nominal_source": "148 SM x 64 fp64 lanes x 2 x clocks.max.sm", "ms_per_launch": dom["ms"]}
        if dom["stage"] in textbook:
            roof["frac_textbook"] = round(textbook[dom["stage"]] / (dom["ms"] * 1e-3) / 1e12 / alu_peak, 4)
            roof["frac_textbook_note"] = ("textbook flops (5 n log2 n per transform, 8 per complex multiply-add) / time / "
                                          "peak: lower than `frac` because a DADD or DMUL fills a DP issue slot with 1 flop")
    else:
        roof = {"kernel": dom["stage"], "bound": "hbm", "achieved": dom["hbm_gbs"], "peak": peaks["hbm_gbs"],
                "unit": "GB/s", "frac": round(dom["hbm_gbs"] / peaks["hbm_gbs"], 4), "traffic": NCU_TRAFFIC.get(dom["stage"]),
                "traffic_source": NCU_SOURCE,
                "peak_source": peaks["source"] + " (MEASURED_PEAKS.json hbm_gbs)", "ms_per_launch": dom["ms"]}
    roof["alu_peak_probed_tflops"] = dfma_tf

    # ---- CPU baseline: the oracle as it stands, one CCD of the same workload, with all host cores and
    # once more with scipy.fft workers=1 (SURVEY 8(d) "Timing the oracle beside it")
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import sfft_oracle as orc
        cores = oracle_cores()
        p0 = pairs[0]
        tc = time.perf_counter()
        orc.sfft_difference(p0.R, p0.S, p0.mask, cfg.w, cfg.DK, cfg.DB, workers=cores)
        dtc = time.perf_counter() - tc
        tc = time.perf_counter()
        orc.sfft_difference(p0.R, p0.S, p0.mask, cfg.w, cfg.DK, cfg.DB, workers=1)
        dt1 = time.perf_counter() - tc
        cpu = {"value": 1.0 / dtc, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "1 full CCD pair (pair 0 of this run): FFT-route build + Cholesky + FFT-route subtract, "
                         f"scipy.fft workers={cores}; {dtc:.1f} s",
               "workers1": {"value": 1.0 / dt1, "unit": UNIT, "cores": 1, "seconds": round(dt1, 1),
                            "sample": "the same pair and code with scipy.fft workers=1 (numpy's own BLAS/threads untouched)"},
               "cpu_model": cpu_model()}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms / args.steps, "ms_per_step_median": round(ms_median, 4),
        "ms_per_step_with_stage_events": round(ms_profiled, 4),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "l2": f"inputs larger than L2: {NPAIR} resident pairs cycled (429 MB) and "
                   "~1.4 GB of per-step scratch traffic", "parallelism": f"ccd-shard x{world}", "plans": 1,
                   "calls_per_step": "sfft_build_system, sfft_subtract_prepare, sfft_solve, sfft_subtract"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": ms_e2e / args.steps, "how": "pinned host R,S,mask -> device, hot path, D and coeffs "
                "-> pinned host; 3 plans on 3 streams; PCIe-bound: this box moves 51.8 GB/s host->device while the "
                "device->host copy of D runs (55.5 GB/s alone), i.e. 2.9 ms per 143 MB pair"},
        "gpu_launches": launches * args.steps,
        "gpu_launches_per_step": launches,
        "roofline": roof,
        "stages": table,
        "cpu_baseline": cpu,
        "exposure": exposure,
        "post_differencing": post,
    }
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu --set full capture of the final
# kernels of this round, summarised in NCU_SOURCE (null where that capture holds no such kernel).
NCU_SOURCE = "profiles/r02_ncu_full.md"
NCU_TRAFFIC = {"build.colx": 282.8e6, "build.row_fwd": 363.4e6, "subtract.row_fwd": 209.1e6, "subtract.mix": 253.7e6,
               "subtract.row_inv": 172.5e6, "solve": 4.6e6}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--exposure-ccds", type=int, default=60,
                    help="CCD pairs of the exposure-batch leg (BASELINE.json configs[4]); 0 skips it")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_cuda(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
