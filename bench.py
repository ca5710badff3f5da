"""bench.py -- throughput of the PTEFIT hot path (include/ptefit.h) on synthetic EXL-50U-shaped
slices, with the roofline of the dominant kernel and the FP64 oracle timed beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config cfg4]

A "step" is one ptefit_reconstruct call over one batch: the configured number of Picard
iterations (all SURVEY.md 8(a) rows) for every slice of the batch.  Default workload =
BASELINE.json configs[3] ("cfg4": 129x129, 140 channels, 76 coil columns, batch 512, 20
iterations, FP32) -- the configuration the batched slices/s metric is quoted on; the batch-1
latency of configs[2] ("cfg3") is measured in the same run and reported as `latency_batch1`.
Prints ONE JSON line on rank 0.  DESIGN.md "Measurement" explains every field.
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

METRIC = "slices_per_s_129x129"
UNIT = "slices/s"


def _peaks():
    """Roofline denominators: MEASURED_PEAKS.json (driver-written), else the guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=float(d["hbm_gbs"]), bf16=float(d["bf16_tflops"]),
                    bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), source="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 25 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "25"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


def yardsticks(torch):
    """Library GEMMs timed on this box in this run (yardsticks only): TF32 and FP64
    torch.matmul, best of 5 after warm-up.  TFLOP/s."""
    out = {}
    prev = torch.backends.cuda.matmul.allow_tf32
    for name, dt, n, tf32 in (("tf32_tflops", torch.float32, 8192, True), ("fp64_tflops", torch.float64, 4096, False)):
        torch.backends.cuda.matmul.allow_tf32 = tf32
        a = torch.randn(n, n, dtype=dt, device="cuda"); b = torch.randn(n, n, dtype=dt, device="cuda")
        for _ in range(2):
            a @ b
        best = 1e30
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); a @ b; e1.record(); torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        out[name] = 2.0 * n ** 3 / (best * 1e-3) / 1e12
        del a, b
    torch.backends.cuda.matmul.allow_tf32 = prev
    out["how"] = "torch.matmul 8192^3 with TF32 allowed / 4096^3 FP64, best of 5, CUDA events (library yardsticks)"
    return out


def ncu_traffic():
    """DRAM bytes per launch of the stage kernels from the committed `ncu --set full` summaries
    (profiles/r2_ncu_traffic.json: dram__bytes_read.sum + dram__bytes_write.sum, workload cfg4 batch 512)."""
    p = os.path.join(ROOT, "profiles", "r2_ncu_traffic.json")
    return json.load(open(p)) if os.path.exists(p) else {}


def make_workload(name, batch, first=0):
    """Seeded synthetic device + `batch` slices (synth/)."""
    import synth
    dev = synth.make_device(name)
    sl = synth.make_slices(dev, batch, first=first)
    return dev, sl


def round32(dev, sl):
    """FP32 configs: the oracle consumes the inputs the GPU sees (rounded to nearest FP32)."""
    r32 = lambda a: np.asarray(a, np.float32).astype(np.float64)
    d2 = dict(dev)
    d2["tables"] = {k: r32(v) for k, v in dev["tables"].items()}
    return d2, r32(sl["b"]), r32(sl["ic"])


def oracle_throughput(dev, b, ic, n_iter, n_sample, budget_s=25.0):
    """The oracle as it stands (oracle/picard.py, single process; numpy/LAPACK threads as the box
    provides), timed on up to n_sample slices or until budget_s is spent.  slices/s."""
    from oracle.picard import Device, reconstruct
    od = Device(dev["grid"], dev["geom"], dev["tables"], dev["basis"])   # table copy + banded LU: not timed
    done, t0 = 0, time.perf_counter()
    for q in range(min(n_sample, b.shape[0])):
        reconstruct(od, b[q], ic[q], n_iter)
        done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return done / dt, done, dt


def host_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info()]
        return max(n) if n else 1
    except Exception:
        return 1


def run_reference(args):
    """--impl reference: the FP64 CPU oracle on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfgname = args.config
    import synth
    c = synth.CONFIGS[cfgname]
    per_step = max(1, args.ref_sample)
    n = per_step * (args.steps + args.warmup)
    dev, sl = make_workload(cfgname, min(n, 64))
    dv, b, ic = round32(dev, sl) if c["precision"] == "fp32" else (dev, sl["b"], sl["ic"])
    from oracle.picard import Device, reconstruct
    od = Device(dv["grid"], dv["geom"], dv["tables"], dv["basis"])
    q = 0
    for _ in range(args.warmup * per_step):
        reconstruct(od, b[q % len(b)], ic[q % len(b)], c["n_iter"]); q += 1
    t0 = time.perf_counter()
    for _ in range(args.steps * per_step):
        reconstruct(od, b[q % len(b)], ic[q % len(b)], c["n_iter"]); q += 1
    dt = time.perf_counter() - t0
    val = args.steps * per_step / dt
    sample = f"{per_step} slice(s) per step of {cfgname} ({c['n']}x{c['n']}, {c['n_iter']} Picard iterations), seeded like the GPU arm"
    line = dict(impl="reference", metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * dt / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", config=dict(workload=cfgname, grid=f"{c['n']}x{c['n']}", n_iter=c["n_iter"],
                                              batch=per_step, note="oracle/ on host cores, bounded sample"),
                cpu_baseline=dict(value=val, unit=UNIT, cores=host_threads(), kind="oracle", sample=sample),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line), flush=True)


def stage_roofline(stage, ms_per_launch, dims, peaks, gemm_mode):
    """Roofline entry of the kernel that dominates `stage`.
    Algorithmic work per launch = SURVEY.md 8(d)'s per-slice figure x slices per launch."""
    B, es = dims["B"], dims["es"]
    N, Nint, Nb, M, nt = dims["N"], dims["Nint"], dims["Nb"], dims["M"], dims["nt"]
    tf32 = peaks.get("tf32") or (1.1 / 2.25) * peaks["bf16_sustained"]   # measured yardstick, else the guide's nominal TF32 : bf16 ratio
    tnote = peaks.get("tf32_note", "1.1/2.25 x measured sustained bf16")
    fp64 = peaks.get("fp64") or 37.0
    f64 = es == 8
    if stage == "response":
        flops = 2.0 * M * Nint * nt * B
        return dict(kernel="k_basis_c+k_gemm_dmma+k_resp_reduce_d" if f64 else "k_gemm_3xtf32<144,3,NP,NFF>+k_resp_reduce", bound="tensor",
                    achieved=flops / (ms_per_launch * 1e-3) / 1e12, peak=fp64 if f64 else tf32, unit="TFLOP/s",
                    peak_note=("FP64 yardstick" if f64 else tnote) + f"; gemm mode {gemm_mode}; algorithmic flops on the full node list (2 M N_int nb)")
    if stage == "boundary":
        flops = 2.0 * Nb * Nint * B
        return dict(kernel="k_current_c+k_gemm_dmma+k_pbd_reduce_d" if f64 else "k_current_split+k_gemm_3xtf32<256,2>+k_pbd_reduce", bound="tensor",
                    achieved=flops / (ms_per_launch * 1e-3) / 1e12, peak=fp64 if f64 else tf32, unit="TFLOP/s",
                    peak_note=("FP64 yardstick" if f64 else tnote) + f"; gemm mode {gemm_mode}")
    if stage == "solve" and dims.get("fused"):
        # A7 + A8 read 4 N_int (J) + 4 N (psi_coil), write 4 N (psi); A1 fused behind it writes <= 5 N
        byts = (float(es) * (Nint + 2 * N) + (es + 1.0) * N) * B
        # what the kernel moves with this repo's additions: + old psi (relaxation), + delz column, + boundary flux
        extra = float(es) * (6 * N + Nb) * B
        return dict(kernel="k_solve_tc" if not f64 and dims.get("tcs") else "k_solve_fused", bound="hbm", achieved=byts / (ms_per_launch * 1e-3) / 1e9,
                    peak=peaks["hbm"], unit="GB/s", peak_note=f"{peaks['source']} copy bandwidth; algorithmic bytes per SURVEY.md 8(d)",
                    bytes_per_launch=byts, bytes_incl_additions=extra)
    if stage == "solve":
        byts = float(es) * (Nint + N + N + N) * B    # read I, psi_coil, old psi (relaxation); write psi
        return dict(kernel="k_rhs_dst+k_tridiag+k_idst_total", bound="hbm", achieved=byts / (ms_per_launch * 1e-3) / 1e9,
                    peak=peaks["hbm"], unit="GB/s", peak_note=f"{peaks['source']} copy bandwidth")
    if stage == "search":
        byts = float(es) * (N + N) * B               # read psi, write normalised flux
        return dict(kernel="k_search", bound="hbm", achieved=byts / (ms_per_launch * 1e-3) / 1e9, peak=peaks["hbm"],
                    unit="GB/s", peak_note=f"{peaks['source']} copy bandwidth")
    byts = float(es) * N * B
    return dict(kernel="k_" + stage, bound="hbm", achieved=byts / (ms_per_launch * 1e-3) / 1e9, peak=peaks["hbm"],
                unit="GB/s", peak_note=f"{peaks['source']} copy bandwidth")


def run_ours(args):
    import torch
    import torch.distributed as dist
    import synth
    import paper_2601_12378_b200 as P

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the PTEFIT hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c = synth.CONFIGS[args.config]
    B = args.batch or c["batch"]
    prec = c["precision"]
    n_iter = c["n_iter"]
    # each rank reconstructs its own B slices (weak scaling: slices are independent, tables replicated)
    n_unique = min(B, args.unique) if args.unique > 0 else B
    dev, sl = make_workload(args.config, n_unique, first=rank * n_unique)
    reps = (B + n_unique - 1) // n_unique
    b_np = np.tile(sl["b"], (reps, 1))[:B]
    ic_np = np.tile(sl["ic"], (reps, 1))[:B]
    rec = P.Reconstructor(dev, precision=prec, max_batch=B)
    dt = rec.dtype
    d_b = torch.tensor(b_np, dtype=dt, device="cuda")
    d_ic = torch.tensor(ic_np, dtype=dt, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")      # 256 MB > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        rec.reconstruct(d_b, d_ic, n_iter)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    # ---- timed region: K steps, L2 flushed between steps (outside the per-step event pairs)
    clk = ClockSampler(local)
    clk.start()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    for e0, e1 in evs:
        flush.zero_()
        e0.record()
        step()
        e1.record()
    barrier()
    ms_steps = [e0.elapsed_time(e1) for e0, e1 in evs]
    clocks = clk.stop()
    launches = rec.launch_count() * args.steps
    total_ms = float(sum(ms_steps))
    t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    value = world * B * args.steps / (total_ms * 1e-3)
    status = rec.status[:B].cpu().numpy()
    n_ok = int((status == 0).sum())
    # ---- stage breakdown: K more steps with the library's stage events switched on
    rec.set_profiling(True)
    acc = {}
    for _ in range(args.steps):
        flush.zero_()
        step()
        torch.cuda.synchronize()
        for k, v in rec.stage_ms().items():
            acc[k] = acc.get(k, 0.0) + v / args.steps
    rec.set_profiling(False)
    dims = dict(B=B, es=4 if prec == "fp32" else 8, N=rec.nr * rec.nz, Nint=(rec.nr - 2) * (rec.nz - 2),
                Nb=2 * (rec.nr + rec.nz) - 4, M=rec.M, nt=rec.nt)
    loop_stages = {k: v for k, v in acc.items() if k != "setup" and v > 0.0}
    dims["fused"] = "search" not in loop_stages     # search runs inside k_solve_fused
    top = max(loop_stages, key=loop_stages.get)
    peaks = _peaks()
    yard = None
    if not args.skip_extras:
        yard = yardsticks(torch)
        peaks["tf32"] = yard["tf32_tflops"]; peaks["fp64"] = yard["fp64_tflops"]
        peaks["tf32_note"] = "TF32 torch.matmul yardstick measured in this run"
    dims["tcs"] = (prec == "fp32" and rec.nz == 129 and rec.nr <= 129)
    roof = stage_roofline(top, loop_stages[top] / n_iter, dims, peaks, args.gemm)
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["traffic"] = None
    if args.config == "cfg4" and B == 512:
        roof["traffic"] = ncu_traffic().get(roof["kernel"].split("+")[0].split("<")[0])
    roof["share_of_step"] = loop_stages[top] / max(sum(acc.values()), 1e-9)
    roof["all_stages"] = {}
    for sname, ms in loop_stages.items():
        r = stage_roofline(sname, ms / n_iter, dims, peaks, args.gemm)
        roof["all_stages"][sname] = dict(ms_per_step=ms, bound=r["bound"], achieved=r["achieved"], unit=r["unit"],
                                         frac=r["achieved"] / r["peak"])
        if r["bound"] == "tensor" and prec == "fp32":
            roof["all_stages"][sname]["frac_of_peak_over_3"] = 3.0 * r["achieved"] / r["peak"]     # 3xTF32 issues three MMAs per product
    e2e = None
    if not args.skip_extras:
        e2e = run_e2e(args, torch, dist, rec, b_np, ic_np, dt, B, n_iter, world, barrier)
    rec.close()
    out = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
               ms_per_step=total_ms / args.steps, us_per_slice=1e3 * total_ms / args.steps / B,
               us_per_slice_iteration=1e3 * total_ms / args.steps / B / max(n_iter, 1), higher_is_better=True,
               scaling="weak", vs_baseline=None, dtype="f32" if prec == "fp32" else "f64", data="synthetic",
               config=dict(workload=args.config, grid=f"{rec.nr}x{rec.nz}", batch_per_gpu=B, n_iter=n_iter, n_meas=rec.M,
                           n_coil=rec.nc, n_terms=rec.nt, unique_slices=n_unique, gemm=args.gemm if prec == "fp32" else "fp64-dmma",
                           l2="flushed between timed steps (256 MB memset) and working set > L2",
                           parallelism=f"slices sharded over {world} GPU(s), no collective"),
               clocks=clocks, e2e=e2e, gpu_launches=launches, slices_status_ok=n_ok, roofline=roof,
               stage_ms_per_step=acc, yardsticks=yard)
    if rank == 0 and world == 1 and not args.skip_extras:
        out["latency_batch1"] = latency_batch1(args, torch, P)
        dv, b32, ic32 = round32(dev, sl) if prec == "fp32" else (dev, sl["b"], sl["ic"])
        v, done, secs = oracle_throughput(dv, b32, ic32, n_iter, args.cpu_sample)
        out["cpu_baseline"] = dict(value=v, unit=UNIT, cores=host_threads(), kind="oracle", note="the numpy test oracle as it stands, not a tuned CPU baseline",
                                   sample=f"first {done} slices of the same {args.config} batch, {n_iter} iterations each, {secs:.1f} s")
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_e2e(args, torch, dist, rec, b_np, ic_np, dt, B, n_iter, world, barrier):
    """End to end through the host-buffer C-ABI call: pinned host memory, host<->device copies inside
    the timed region, wall clock around the synchronous call, max over ranks."""
    hb = torch.tensor(b_np, dtype=dt).pin_memory()
    hic = torch.tensor(ic_np, dtype=dt).pin_memory()
    hout = {k: torch.from_numpy(v).pin_memory() for k, v in rec.host_outputs(B).items()}
    hout_np = {k: v.numpy() for k, v in hout.items()}
    for _ in range(2):
        rec.reconstruct_host(hb.numpy(), hic.numpy(), n_iter, hout_np)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        rec.reconstruct_host(hb.numpy(), hic.numpy(), n_iter, hout_np)      # synchronous
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_s = float(t.item())
    h2d = int(hb.numel() * hb.element_size() + hic.numel() * hic.element_size())
    d2h = int(sum(v.numel() * v.element_size() for v in hout.values()))
    e2e = dict(value=world * B * args.steps / e2e_s, unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
               api="ptefit_reconstruct_host (pinned host buffers)")
    return e2e


def latency_batch1(args, torch, P):
    """Batch-1 latency on BASELINE configs[2] (cfg3: 129x129, 20 iterations, FP32): median of 50
    ptefit_reconstruct calls, CUDA events, inputs resident (the whole 42 MB table set fits L2, which
    is the real-time operating mode: consecutive slices reuse it)."""
    import synth
    c = synth.CONFIGS["cfg3"]
    dev, sl = make_workload("cfg3", 1)
    rec = P.Reconstructor(dev, precision=c["precision"], max_batch=1)
    d_b = torch.tensor(sl["b"], dtype=rec.dtype, device="cuda")
    d_ic = torch.tensor(sl["ic"], dtype=rec.dtype, device="cuda")
    for _ in range(5):
        rec.reconstruct(d_b, d_ic, c["n_iter"])
    torch.cuda.synchronize()
    ts = []
    for _ in range(50):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); rec.reconstruct(d_b, d_ic, c["n_iter"]); e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    n = rec.launch_count()
    # the paper's operating mode: one Picard iteration per slice from the previous flux
    tw = []
    for _ in range(5):
        rec.reconstruct(d_b, d_ic, 1, warm_start=True)
    torch.cuda.synchronize()
    for _ in range(50):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); rec.reconstruct(d_b, d_ic, 1, warm_start=True); e1.record()
        torch.cuda.synchronize()
        tw.append(e0.elapsed_time(e1))
    # the same in continue mode (warm_start = 2: the handle's own previous output is the start, its search is not repeated)
    tc2 = []
    for _ in range(50):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); rec.reconstruct(d_b, d_ic, 1, warm_start=2); e1.record()
        torch.cuda.synchronize()
        tc2.append(e0.elapsed_time(e1))
    # flux-surface post-processing of the paper's timing (33 profile points; Sec. II.E): 33 levels x 128
    # chords, 10 bisections, three Q integrals, q profile, LCFS geometry -- a separate call (ptefit_flux_surfaces)
    for _ in range(3):
        rec.flux_surfaces(1, n_prof=33, n_chord=128, n_bisect=10, f_vac=2.5e6, want_vert=False)
    torch.cuda.synchronize()
    tf = []
    for _ in range(30):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); rec.flux_surfaces(1, n_prof=33, n_chord=128, n_bisect=10, f_vac=2.5e6, want_vert=False); e1.record()
        torch.cuda.synchronize()
        tf.append(e0.elapsed_time(e1))
    us_flux = 1e3 * float(np.median(tf))
    # streaming replay (PAPER.md:158, 175 / Fig. 3): 10 000 consecutive slices, one warm-started Picard
    # iteration each (the previous slice's flux is the start), measurements cycling through the stored
    # cfg3 slices; one event pair per slice, read after the loop
    dev8, sl8 = make_workload("cfg3", 8)
    d_b8 = torch.tensor(sl8["b"], dtype=rec.dtype, device="cuda")
    d_ic8 = torch.tensor(sl8["ic"], dtype=rec.dtype, device="cuda")
    n_stream = 400 if args.latency_only else 10000
    # slow flux variation: the measurements drift linearly from one stored equilibrium to the
    # next over 1250 slices
    seg = n_stream // 8
    al = (torch.arange(n_stream, device="cuda") % seg).to(rec.dtype)[:, None] / seg
    k0 = (torch.arange(n_stream, device="cuda") // seg) % 8
    k1 = (k0 + 1) % 8
    b_all = d_b8[k0] * (1 - al) + d_b8[k1] * al
    ic_all = d_ic8[k0] * (1 - al) + d_ic8[k1] * al
    rec.reconstruct(b_all[0:1], ic_all[0:1], c["n_iter"])      # converge on the first slice, then stream
    n_ok = 0
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(n_stream + 1)]
    stat = torch.zeros(n_stream, dtype=torch.int32, device="cuda")
    evs[0].record()
    for q in range(n_stream):
        rec.reconstruct(b_all[q:q + 1], ic_all[q:q + 1], 1, warm_start=2)      # continue mode: slice q starts from what slice q - 1 left
        evs[q + 1].record()
        stat[q:q + 1].copy_(rec.status[0:1], non_blocking=True)    # outside the event pair of slice q, inside that of q + 1
    torch.cuda.synchronize()
    st = np.array([evs[q].elapsed_time(evs[q + 1]) for q in range(n_stream)]) * 1e3
    stream = dict(slices=n_stream, us_mean=float(st.mean()), us_p50=float(np.percentile(st, 50)), us_p99=float(np.percentile(st, 99)),
                  us_max=float(st.max()), status_ok=int((stat == 0).sum().item()),
                  note="one Picard iteration per slice continuing the previous slice (warm_start = 2), back-to-back launches, no post-processing")
    rec.close()
    return dict(workload="cfg3", streaming=stream, us_per_slice=1e3 * float(np.median(ts)), us_min=1e3 * float(min(ts)), n_iter=c["n_iter"],
                us_per_iteration=1e3 * float(np.median(ts)) / c["n_iter"],
                us_one_warm_iteration=1e3 * float(np.median(tw)), us_one_continue_iteration=1e3 * float(np.median(tc2)), us_flux_surfaces=us_flux,
                us_warm_iteration_plus_flux_surfaces=1e3 * float(np.median(tw)) + us_flux,
                launches_per_call=n, paper_context="0.268 ms/slice at 129x129 on the paper's GPU (PAPER.md:175), other hardware")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg4")
    ap.add_argument("--batch", type=int, default=0, help="override the config's batch")
    ap.add_argument("--unique", type=int, default=0, help="distinct seeded slices per rank, tiled to the batch (0 = all distinct)")
    ap.add_argument("--gemm", default="3xtf32", help="contraction arithmetic label recorded in config")
    ap.add_argument("--cpu-sample", type=int, default=24, help="slices the cpu_baseline leg times")
    ap.add_argument("--skip-extras", action="store_true", help="timed region + stage breakdown only (for ncu runs)")
    ap.add_argument("--ref-sample", type=int, default=4, help="--impl reference: slices per step")
    ap.add_argument("--latency-only", action="store_true", help="only the batch-1 latency section (cfg3), for ncu launch lists")
    args = ap.parse_args()
    if args.latency_only:
        import torch
        import paper_2601_12378_b200 as P
        print(json.dumps(dict(latency_batch1=latency_batch1(args, torch, P))), flush=True)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
