#!/usr/bin/env python
"""bench.py -- slice.projection pairs/s per MBIR iteration (forward + adjoint) on BASELINE config 4, 1xB200.

A step = one pass of the whole hot path over one batch: tc_radon (F1-F4) then tc_backproject (B1-B4) on
128 slices of 2048^2 with 1024 angles (centre 1027.5), device-resident.  `value` = S * Na * n_gpus / step time.
`e2e` = the same through the C-ABI call with pinned HOST buffers (slab scheduler: H2D, compute, D2H inside the
timed region).  `extra` carries the other north_star figures of the same run: one full MBIR iteration of config 4
(`mbir_*`), config 3's 50 iterations, and config 5 out of core (`ooc`: streamed MBIR with its transfer/compute overlap).
`--impl reference` times the oracle (oracle/nufft.py, float64 numpy, one process per host core) instead.
Prints ONE JSON line on rank 0.
"""
import argparse, json, os, subprocess, sys, threading, time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
METRIC = "slice_projection_pairs_per_s_fwd_adj"
UNIT = "slice*projection pairs/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE config number (4 = the metric's workload)")
    ap.add_argument("--slices", type=int, default=0, help="override slice count (debug)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-mbir", action="store_true", help="skip the MBIR-iteration timings (extra.mbir_*, extra.cfg3_*)")
    ap.add_argument("--ooc", type=int, default=-1, metavar="SLICES",
                    help="config 5's geometry (2560^2, 1313 angles) out of core on SLICES host-resident slices: streamed MBIR, "
                         "transfer/compute overlap (extra.ooc).  -1 (default): as many of the 2160 slices as host memory allows; 0: skip")
    ap.add_argument("--ooc-iters", type=int, default=20)
    return ap.parse_args()


def peak_hbm():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True); self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm = sorted(float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) > 3 + k and r[3 + k].lower().startswith("active") for r in self.rows)]
        mx = next((float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()), None)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": reasons, "samples": len(sm)}


def stage_bytes(n, nd, na, S):
    """algorithmic HBM bytes per launch of each kernel, S slices = ceil(S/8) groups of 32-byte cells."""
    ng = (S + 7) // 8
    G = 2 * n
    cell = 32
    return {
        "fwd_rows": S * n * n * 4 + ng * n * G * cell,
        "fwd_cols": ng * (n * G + G * G) * cell,
        "fwd_gather": ng * G * G * cell + S * na * nd * 4,
        "adj_radial": S * na * nd * 4 + ng * na * nd * cell,
        "adj_spread": ng * na * nd * cell + ng * G * G * cell,
        "adj_cols": ng * (G * G + n * G) * cell,
        "adj_rows": ng * n * G * cell + S * n * n * 4,
        "fwd_radial": ng * na * nd * cell + S * na * nd * 4,       # F4 as its own launch (tile-binned gather): reads cpol, writes the sinogram
    }


# ---- the oracle as it stands, one process per host core (cpu_baseline and --impl reference) ----
def _oracle_job(a):
    import numpy as np
    from oracle import nufft
    vol, ang, nd, centre = a
    s = nufft.radon_nufft(vol, ang, nd, centre)
    nufft.backproject_nufft(s, ang, vol.shape[-1], centre)
    return len(ang)


def oracle_sample(c, n_slices, n_angles_sample, pool, vols=None):
    """oracle forward + adjoint of n_slices slices (one job each) on every (Na / n_angles_sample)-th angle; returns (pairs, seconds)."""
    import numpy as np
    from paper_2304_12934_b200 import inputs
    ang = inputs.angles_uniform(c["Na"]).astype(np.float64)[:: max(1, c["Na"] // n_angles_sample)]
    if vols is None:
        vols = inputs.volume_fibres(n_slices, c["N"], c["seed"], n_fibres=3000 if c["N"] >= 2048 else 300, workers=min(n_slices, os.cpu_count() or 1))
    t0 = time.perf_counter()
    res = pool.map(_oracle_job, [(vols[s], ang, c["Nd"], c["centre"]) for s in range(n_slices)], chunksize=1)
    return sum(res), time.perf_counter() - t0, vols


def oracle_pool():
    import multiprocessing as mp
    cores = max(1, min(16, os.cpu_count() or 1))
    return mp.get_context("fork").Pool(cores), cores


def run_reference(args, c):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    pool, cores = oracle_pool()
    nsl, nsel = cores, 64
    vols = None
    for _ in range(min(args.warmup, 1)):
        _, _, vols = oracle_sample(c, nsl, nsel, pool, vols)
    tot, pairs = 0.0, 0
    for _ in range(args.steps):
        p, t, vols = oracle_sample(c, nsl, nsel, pool, vols)
        tot += t; pairs += p
    pool.close()
    val = pairs / tot
    sample = "%d slices x %d of %d angles (every %dth), %dx%d, oracle/nufft.py forward+adjoint, float64 numpy, %d processes (one slice each)" % (
        nsl, nsel, c["Na"], c["Na"] // nsel, c["N"], c["N"], cores)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config4: 128 slices 2048x2048, 1024 angles, 2048 bins, centre 1027.5 (bounded sample per step: %s)" % sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "cpu": cpu_model()},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def cpu_model():
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def host_mem_available():
    """bytes this process may still take: MemAvailable, capped by the cgroup limit if there is one."""
    avail = None
    try:
        with open("/proc/meminfo") as fh:
            for line in fh:
                if line.startswith("MemAvailable:"):
                    avail = int(line.split()[1]) * 1024
    except Exception:
        pass
    for lim, cur in (("/sys/fs/cgroup/memory.max", "/sys/fs/cgroup/memory.current"),
                     ("/sys/fs/cgroup/memory/memory.limit_in_bytes", "/sys/fs/cgroup/memory/memory.usage_in_bytes")):
        try:
            l = open(lim).read().strip()
            if l != "max" and int(l) < (1 << 60):
                room = int(l) - int(open(cur).read().strip())
                avail = room if avail is None else min(avail, room)
        except Exception:
            pass
    return avail


def step_L(Na, N):
    """the step constant both MBIR timings use: 1.05 * lambda_hat (~ 1.02 Na N for uniform angles) + 4 / (c sigma^2)  (reading G15)"""
    return float(1.05 * 1.02 * Na * N + 4.0 / (1e-4 * (1 / 0.7) ** 2))


def run_ooc(args, tc, inputs, torch, np, nw, pcie_peak=None):
    """BASELINE config 5: 2560^2 x S slices host-resident (pinned), 1313 angles, MBIR streamed by slab over PCIe."""
    c5 = inputs.CONFIGS[5]
    N5, Na5, Nd5 = c5["N"], c5["Na"], c5["Nd"]
    vol_b, sino_b = N5 * N5 * 4, Na5 * Nd5 * 4
    S_full = c5["S"]
    # pinned host memory: the caller's volume (truth, then the output), the library's second volume, the sinogram
    need = lambda S: S * (2 * vol_b + sino_b)
    avail = host_mem_available()
    S5 = S_full if args.ooc < 0 else min(args.ooc, S_full)
    note = "full size"
    if avail is not None and need(S5) > 0.88 * avail:
        S5 = int(0.88 * avail / (2 * vol_b + sino_b)) // 32 * 32
        note = "reduced to fit host memory: need %.1f GB pinned for %d slices, %.1f GB available" % (need(S_full) / 1e9, S_full, avail / 1e9)
    if S5 < 64:
        return {"unavailable": "host memory: %s bytes available, %d needed for 64 slices" % (avail, need(64))}
    t0 = time.perf_counter()
    blk = 120                                                      # a seeded 120-slice fibre block, repeated along z (content does not change the work)
    block = inputs.volume_fibres(blk, N5, c5["seed"], n_fibres=3000, workers=nw)
    pv5, pb5 = tc.PinnedArray((S5, N5, N5)), tc.PinnedArray((S5, Na5, Nd5))     # exact-size pinned memory from the library (tc_host_alloc)
    v5, b5 = pv5.array, pb5.array
    for s0 in range(0, S5, blk):
        ns = min(blk, S5 - s0)
        v5[s0:s0 + ns] = block[:ns]
    del block
    t_gen = time.perf_counter() - t0
    p5 = tc.Plan(N5, Nd5, inputs.angles_uniform(Na5), c5["centre"], max_slab_slices=32)
    p5.radon(v5, out=b5)                                           # b = A truth, by the GPU path itself, slab-wise
    st_f = p5.sched_stats()
    pr5 = tc.prior_params(L=step_L(Na5, N5))
    its = args.ooc_iters
    t0 = time.perf_counter()
    x5, log5 = p5.mbir(b5, pr5, its, out=v5)                       # the truth's array becomes the output (and one of the two host volumes)
    t_call = time.perf_counter() - t0
    st5 = p5.sched_stats()
    p5.close()
    F = [l["F"] for l in log5]
    wall = st5["wall_s"]
    busy = {"h2d": st5["h2d_s"], "compute": st5["compute_s"], "d2h": st5["d2h_s"]}
    h2d_gbps = st5["h2d_bytes"] / max(st5["h2d_s"], 1e-9) / 1e9
    d2h_gbps = st5["d2h_bytes"] / max(st5["d2h_s"], 1e-9) / 1e9
    out = {"workload": "config5: %d of %d slices of 2560x2560 host-resident (pinned; %s), 1313 angles, 2560 bins, slabs of 32, %d MBIR iterations streamed over PCIe; "
                       "volume = a seeded %d-slice fibre block repeated along z, sinogram = A truth by the streamed tc_radon" % (S5, S_full, note, its, blk),
           "slices": S5, "iterations": its, "mbir_iter_s": wall / its, "mbir_total_s": wall, "mbir_pairs_per_s": S5 * Na5 / (wall / its),
           "overlap": st5["overlap"], "overlap_formula": "(h2d + compute + d2h - wall) / (h2d + compute + d2h - max(h2d, compute, d2h))",
           "h2d_s": st5["h2d_s"], "compute_s": st5["compute_s"], "d2h_s": st5["d2h_s"], "wall_s": wall,
           "bound_by": max(busy, key=busy.get), "busiest_fraction_of_wall": max(busy.values()) / wall,
           "setup_s": st5["setup_s"], "handover_s": st5["handover_s"], "call_s": t_call, "input_generation_s": t_gen,
           "h2d_GBps": h2d_gbps, "d2h_GBps": d2h_gbps, "pcie_bytes_per_iter": (st5["h2d_bytes"] + st5["d2h_bytes"]) / its,
           "host_pinned_GB": need(S5) / 1e9,
           "F_first_last": [F[0], F[-1]], "F_monotone": all(F[i + 1] <= F[i] for i in range(len(F) - 1)), "accepted": sum(l["accepted"] for l in log5),
           "radon_streamed": {"wall_s": st_f["wall_s"], "overlap": st_f["overlap"], "pairs_per_s": S5 * Na5 / st_f["wall_s"],
                              "h2d_GBps": st_f["h2d_bytes"] / max(st_f["h2d_s"], 1e-9) / 1e9, "d2h_GBps": st_f["d2h_bytes"] / max(st_f["d2h_s"], 1e-9) / 1e9}}
    if pcie_peak:
        out["pcie_peak_GBps"] = pcie_peak
        out["h2d_frac_of_pcie_peak"] = h2d_gbps / pcie_peak["h2d"]
        out["d2h_frac_of_pcie_peak"] = d2h_gbps / pcie_peak["d2h"]
    del v5, b5, x5
    pv5.free(); pb5.free()
    return out


def measure_pcie(torch):
    """pinned cudaMemcpyAsync peaks of this box, 1 GiB each way (what config 5's copies are reported against)."""
    h = torch.empty(1 << 28, dtype=torch.float32, pin_memory=True)
    dv = torch.empty(1 << 28, dtype=torch.float32, device="cuda")
    res = {}
    for name, (dst, src) in (("h2d", (dv, h)), ("d2h", (h, dv))):
        best = 0.0
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); dst.copy_(src, non_blocking=True); e1.record(); torch.cuda.synchronize()
            best = max(best, h.numel() * 4 / (e0.elapsed_time(e1) * 1e-3) / 1e9)
        res[name] = best
    return res


def main():
    args = parse()
    from paper_2304_12934_b200 import inputs
    c = dict(inputs.CONFIGS[args.config])
    if args.slices:
        c["S"] = args.slices
    if args.impl == "reference":
        return run_reference(args, c)

    import numpy as np, torch, torch.distributed as dist
    from paper_2304_12934_b200 import binding as tc
    from paper_2304_12934_b200.shard import max_over_ranks
    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    S, N, Nd, Na = c["S"], c["N"], c["Nd"], c["Na"]
    ang = inputs.angles_uniform(Na)
    # weak scaling: every rank runs the whole config on its own z-range of a (world x S)-slice job; no data-path collective
    nw = max(1, min(32, (os.cpu_count() or 1) // max(1, min(world, 8))))
    if args.config == 4:
        vol_h = inputs.volume_fibres(S, N, c["seed"] + rank, workers=nw)
    elif args.config == 3:
        vol_h = inputs.volume_porous(S, N, c["seed"] + rank)
    elif args.config == 2:
        vol_h = inputs.volume_cfg2()
    else:
        vol_h = inputs.volume_cfg1() if args.config == 1 else inputs.volume_fibres(S, N, c["seed"], workers=nw)
    plan = tc.Plan(N, Nd, ang, c["centre"])
    vol = torch.from_numpy(vol_h).cuda()
    sino = torch.empty((S, Na, Nd), dtype=torch.float32, device="cuda")
    back = torch.empty_like(vol)

    def step():
        plan.radon(vol, out=sino)
        plan.backproject(sino, out=back)

    def fence():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 1)):
        step()
    fence()
    # ---- the headline: K steps, CUDA events, per-stage recording OFF ----
    plan.profile(False); tc.launch_count(reset=True)
    sampler = ClockSampler(local); sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fence()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    fence()
    secs = max_over_ranks(e0.elapsed_time(e1) * 1e-3)
    clocks = sampler.stop()
    launches = tc.launch_count()
    ms_step = 1e3 * secs / args.steps
    value = world * S * Na / (secs / args.steps)
    # ---- per-kernel times: a second pass with the library's CUDA-event recording on (events on the launching stream) ----
    nprof = min(args.steps, 10)
    plan.profile(True); plan.profile_read()
    for _ in range(nprof):
        step()
    fence()
    stages = plan.profile_read(); plan.profile(False)

    peak, peak_src = peak_hbm()
    sb = stage_bytes(N, Nd, Na, S)
    per = {k: (ms / max(cnt, 1), cnt) for k, (ms, cnt) in stages.items()}
    dom = max(per, key=lambda k: per[k][0] * per[k][1])
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            traffic = json.load(fh).get("config%d" % args.config, {}).get(dom)
    except Exception:
        pass
    ach = sb[dom] / (per[dom][0] * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": traffic,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": sb[dom], "avg_launch_ms": per[dom][0]}
    model_bytes = (104 * N * N + 8 * Na * Nd) * S           # fwd+adj staged-byte model per slice
    extra = {"stage_ms_per_step": {k: per[k][0] * per[k][1] / nprof for k in per},
             "stage_GBps": {k: sb[k] / (per[k][0] * 1e-3) / 1e9 if per[k][0] > 0 else None for k in per},
             "stage_frac_of_hbm_peak": {k: sb[k] / (per[k][0] * 1e-3) / 1e9 / peak if per[k][0] > 0 else None for k in per},
             "fwd_pairs_per_s": S * Na / (sum(per[k][0] * per[k][1] for k in per if k.startswith("fwd")) / nprof * 1e-3),
             "adj_pairs_per_s": S * Na / (sum(per[k][0] * per[k][1] for k in per if k.startswith("adj")) / nprof * 1e-3),
             "step_model_bytes": model_bytes, "step_frac_of_hbm_roofline": model_bytes / (secs / args.steps) / 1e9 / peak,
             "step_frac_of_nominal_8TBs": model_bytes / (secs / args.steps) / 8e12,
             # also against the compulsory bytes (inputs + outputs only, 8 N^2 + 8 Na Nd per slice)
             "step_compulsory_bytes": (8 * N * N + 8 * Na * Nd) * S,
             "step_frac_of_compulsory_roofline": (8 * N * N + 8 * Na * Nd) * S / (secs / args.steps) / 1e9 / peak}

    # ---- e2e: host buffers through the C ABI (slab scheduler) ----
    e2e = None
    if not args.no_e2e:
        pinned = True
        try:
            hv = torch.from_numpy(vol_h).pin_memory()
            hs = torch.empty((S, Na, Nd), dtype=torch.float32).pin_memory()
            hb = torch.empty((S, N, N), dtype=torch.float32).pin_memory()
        except Exception as exc:                                  # seen once right after an ncu run on the same box: fall back to pageable
            sys.stderr.write("bench.py: pinning host buffers failed (%s); e2e uses pageable memory\n" % exc)
            pinned = False
            hv = torch.from_numpy(vol_h)
            hs = torch.empty((S, Na, Nd), dtype=torch.float32)
            hb = torch.empty((S, N, N), dtype=torch.float32)
        plan.radon(hv, out=hs); plan.backproject(hs, out=hb)      # warm-up (allocates staging)
        fence()
        t0 = time.perf_counter()
        ov = []
        for _ in range(args.steps):
            plan.radon(hv, out=hs); ov.append(plan.sched_stats()["overlap"])
            plan.backproject(hs, out=hb); ov.append(plan.sched_stats()["overlap"])
        fence()
        t_e2e = max_over_ranks(time.perf_counter() - t0)
        bytes_in = hv.numel() * 4 + hs.numel() * 4
        bytes_out = hs.numel() * 4 + hb.numel() * 4
        e2e = {"value": world * S * Na / (t_e2e / args.steps), "unit": UNIT, "h2d_bytes_per_step": bytes_in, "d2h_bytes_per_step": bytes_out,
               "ms_per_step": 1e3 * t_e2e / args.steps, "pcie_GBps": (bytes_in + bytes_out) / (t_e2e / args.steps) / 1e9,
               "overlap_mean": float(np.mean(ov)), "pinned_host_buffers": pinned}
        del hv, hs, hb

    if not args.no_mbir:
        # one full MBIR iteration of this config, in core: 1 adjoint + 1 forward + the update / objective kernels
        b = sino
        pr = tc.prior_params(L=step_L(Na, N))
        plan.mbir(b, pr, 1); fence()

        # every iteration ends with a stream synchronisation (the accept test), and the library logs the wall time between two of
        # them (tc_iter_log.ms): the median over the iterations of one call, first iteration left out.  (Differences of whole-call
        # times are useless here: allocation and release of the ~10 GB of state vary by milliseconds from call to call.)
        nit = 24
        _, logm = plan.mbir(b, pr, nit); fence()
        _, logm = plan.mbir(b, pr, nit); fence()
        it_s = max_over_ranks(float(np.median([l["ms"] for l in logm[1:]])) * 1e-3)
        extra["mbir_iter_ms_min_max"] = [float(min(l["ms"] for l in logm[1:])), float(max(l["ms"] for l in logm[1:]))]
        extra["mbir_iter_ms"] = 1e3 * it_s
        extra["mbir_pairs_per_s"] = world * S * Na / it_s
        extra["mbir_model_bytes"] = (128 * N * N + 40 * Na * Nd) * S      # one MBIR iteration per slice
        extra["mbir_frac_of_hbm_roofline"] = extra["mbir_model_bytes"] / it_s / 1e9 / peak
        extra["mbir_slices"] = S
        if rank == 0 and args.config == 4:
            # BASELINE config 3 as stated: 64 x 1024^2, 128 angles, Poisson sinogram, 50 iterations (whole call: allocation, ||b||^2, loop, copy out)
            c3 = inputs.CONFIGS[3]
            p3 = tc.Plan(c3["N"], c3["Nd"], inputs.angles_uniform(c3["Na"]), c3["centre"])
            v3 = torch.from_numpy(inputs.volume_porous(c3["S"], c3["N"], c3["seed"])).cuda()
            b3 = torch.from_numpy(inputs.poisson_sinogram(p3.radon(v3).cpu().numpy(), seed=19)).cuda()
            pr3 = tc.prior_params(L=step_L(c3["Na"], c3["N"]))
            p3.mbir(b3, pr3, 2); fence()
            t0 = time.perf_counter(); x3, log3 = p3.mbir(b3, pr3, 50); fence(); t50 = time.perf_counter() - t0
            it3 = float(np.median([l["ms"] for l in log3[1:]])) * 1e-3
            extra["cfg3_mbir_50it_s"] = t50
            extra["cfg3_mbir_iter_ms"] = 1e3 * it3
            extra["cfg3_mbir_pairs_per_s"] = c3["S"] * c3["Na"] / it3
            extra["cfg3_mbir_frac_of_hbm_roofline"] = (128 * c3["N"] ** 2 + 40 * c3["Na"] * c3["Nd"]) * c3["S"] / it3 / 1e9 / peak
            extra["cfg3_accepted"] = sum(l["accepted"] for l in log3)
            p3.close(); del v3, b3, x3

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        pool, cores = oracle_pool()
        nsel = 128 if Na >= 128 else Na
        nsl = min(cores, S)
        pairs, t, _ = oracle_sample(c, nsl, nsel, pool, vols=vol_h[:nsl])
        pool.close()
        cpu = {"value": pairs / t, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu": cpu_model(),
               "sample": "%d of %d slices x %d of %d angles, %dx%d, oracle/nufft.py forward+adjoint as it stands (float64 numpy), one slice per process, %d processes, %.1f s"
                         % (nsl, S, nsel, Na, N, N, cores, t)}

    if args.ooc != 0 and rank == 0 and world == 1:
        plan.close()
        del vol, sino, back
        torch.cuda.empty_cache()
        try:
            extra["ooc"] = run_ooc(args, tc, inputs, torch, np, nw, measure_pcie(torch))
        except Exception as exc:                                   # the headline must survive a failure of this leg
            extra["ooc"] = {"failed": repr(exc)[:300]}
        plan = None
    if plan is not None:
        plan.close()
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "config%d: %d slices %dx%d float32 fibre-composite phantom (seed %d), %d angles in [0,pi), %d bins, centre %.1f, oversampling 2, KB width 6; step = tc_radon + tc_backproject"
                       % (args.config, S, N, N, c["seed"], Na, Nd, c["centre"]),
                       "l2": "inputs larger than L2 (volume %.2f GB, sinogram %.2f GB, fine grid %.1f GB per step)" % (S * N * N * 4e-9, S * Na * Nd * 4e-9, ((S + 7) // 8) * 4 * N * N * 32e-9),
                       "parallelism": "z-shards, no collective (x%d)" % world},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu, "extra": extra}))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
