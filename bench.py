"""bench.py — demag evaluations/s of boris_demag_apply (+ energy) on synthetic meshes.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C5] [--impl ours|reference]

A step = one pass of the whole hot path: boris_demag_apply
followed by boris_demag_energy on one seeded synthetic magnetization field.  The
headline workload is config C5 (512x512x32, BASELINE.json configs[4]): it is one of
the two meshes the north_star target names, and its compulsory data (M + H + kernel
spectrum = 410 MB) exceed the 126 MB L2, so back-to-back steps are HBM-cold.  The
other four configs are timed too (L2 flushed between steps) and reported under
"all_configs" of the same JSON line.

Multi-GPU: the path does not shard (every output cell depends on every input cell);
`--gpus N` runs N independent replicas, one per rank, no data-path collective
(replicas only), so value = N * evaluations / max-over-ranks time.

`--impl reference` times the fp64 CPU oracle (oracle/, test infrastructure) on the
host cores instead — a deliberately plain program; the ratio to it says nothing about
kernel quality, parity and the roofline fraction do.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2008_02478_b200 import workloads as W  # noqa: E402

METRIC = "demag_evaluations_per_s"
UNIT = "eval/s"
L2_FLUSH_BYTES = 512 << 20
FP32_LANES_PER_SM = 128


def measured_peaks():
    """HBM GB/s and SM clock from MEASURED_PEAKS.json (driver-written), else the guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ----------------------------------------------------------------- ledgers
def kind_bytes(cfg, info):
    """Algorithmic HBM bytes of each kernel kind over one evaluation: its inputs + outputs once."""
    nx, ny, nz = cfg.nx, cfg.ny, cfg.nz
    N = nx * ny * nz
    sp = info["spectrum_bytes"]              # intermediate spectrum (V tiled / W), complex64
    kst = info["kernel_storage_bytes"]
    if info["path"] == 2:
        return {"XFwdT": 12 * N + sp, "YFused": 2 * sp + kst, "XInvT": sp + 12 * N}
    if info["path"] == 3:
        return {"XZFwd": 12 * N + sp, "YFused": 2 * sp + kst, "ZXInv": sp + 12 * N}
    if info["path"] == 4:                    # plane path: X (unpadded) in, partial planes out (cols = ky residues)
        pp = sp * (2 if info["cols"] > 1 else 1)
        return {"XFwdT": 12 * N + sp, "YZFused": sp + kst + pp, "XInvP": pp + 12 * N}
    t = 8 * 3 * (nx + 1) * nz * 2 * ny       # y-padded scratch T over all chunks
    return {"XFwd": 12 * N + sp, "Y2D": 2 * sp + kst, "YFwd": sp + t, "ZFused": 2 * t + kst, "YInv": t + sp,
            "XInv": sp + 12 * N}


def flops_parts(cfg):
    """SURVEY.md §8(d) count: 5 P log2 P per complex FFT, real x FFT as half-length complex + post pass.
    Returns (x one way, y one way, z one way, multiply)."""
    nx, ny, nz = cfg.nx, cfg.ny, cfg.nz
    Px, Py, Pz = 2 * nx, 2 * ny, (2 * nz if nz > 1 else 1)
    NS = nx + 1
    lg = np.log2
    fx = 3 * nz * ny * (5 * nx * lg(nx) + 8 * nx)               # forward; inverse the same
    fy = 3 * nz * NS * 5 * Py * lg(Py)
    fz = 3 * Py * NS * 5 * Pz * lg(Pz) if nz > 1 else 0.0
    mul = (30 if nz > 1 else 20) * NS * Py * Pz
    return float(fx), float(fy), float(fz), float(mul)


def path_flops(cfg):
    fx, fy, fz, mul = flops_parts(cfg)
    return 2 * (fx + fy + fz) + mul


def kind_flops(cfg, info):
    """The same count split over the kernels of the plan's path (which steps each kernel runs: DESIGN.md §5)."""
    fx, fy, fz, mul = flops_parts(cfg)
    if info["path"] == 2:
        return {"XFwdT": fx, "YFused": 2 * fy + mul, "XInvT": fx}
    if info["path"] == 3:
        return {"XZFwd": fx + fz, "YFused": 2 * fy + mul, "ZXInv": fx + fz}
    if info["path"] == 4:
        return {"XFwdT": fx, "YZFused": 2 * (fy + fz) + mul, "XInvP": fx}
    return {"XFwd": fx, "YFwd": fy, "ZFused": 2 * fz + mul, "YInv": fy, "XInv": fx}


# ----------------------------------------------------------------- ncu DRAM traffic (profiles/)
def csrc_sha():
    """Hash of the kernel sources: a stored ncu number is only quoted for the sources it was captured from."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2008_02478_b200", "csrc")
    for name in sorted(os.listdir(d)):
        # the hot path: kernel headers, the launcher, the translation units that instantiate them and the C ABI
        if name.endswith((".h", ".cuh")) or name.startswith("tu_") or name == "boris_demag.cu":
            h.update(name.encode())
            h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(config, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `config`, from the committed ncu
    summary profiles/ncu_traffic.csv (written by paper_2008_02478_b200/ncu_summary.py from an ncu --set full
    report); None when no capture of the CURRENT kernel sources is on file."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None
    sha = csrc_sha()
    best = None
    for line in open(path).read().splitlines()[1:]:
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 5 and f[0] == config and f[1] == kernel and f[4] == sha:
            best = int(f[2]) + int(f[3])
    return best


# ----------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        rows = [r.split(",") for r in open(self.path).read().strip().splitlines() if r.count(",") >= 6]
        os.unlink(self.path)
        if not rows:
            return out
        sm = [float(r[0]) for r in rows if r[0].strip().replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].strip() == "Active" for r in rows)]
        out.update(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=float(rows[0][1]), reasons=reasons,
                   samples=len(rows), power_w_max=max(float(r[2]) for r in rows))
        return out


# ----------------------------------------------------------------- GPU arm
def time_config(torch, binding, cfg, steps, warmup, flush, peak_gbs, sm_max_mhz=1965.0, profile_reps=5):
    """Times `steps` steps of apply+energy on one config.  flush=True: L2 flushed between steps and each
    step timed with its own event pair; flush=False: one event pair around all steps (inputs > L2)."""
    M_host = W.make_input(cfg)
    plan = binding.DemagPlan(cfg.nx, cfg.ny, cfg.nz, *cfg.h)
    info = plan.info()
    M = torch.from_numpy(M_host).cuda()
    H = torch.empty_like(M)
    E = torch.zeros(1, dtype=torch.float64, device="cuda")
    scratch = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda") if flush else None
    st = torch.cuda.current_stream()

    def step():
        plan.apply_energy(M, H, E)      # S1-S8: on the tiled paths the last kernel gathers the energy sum

    for _ in range(max(warmup, 3)):
        step()
    torch.cuda.synchronize()
    if flush:
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in ev:
            scratch.fill_(1)
            a.record(st)
            step()
            b.record(st)
        torch.cuda.synchronize()
        ms = sum(a.elapsed_time(b) for a, b in ev)
    else:
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(st)
        for _ in range(steps):
            step()
        b.record(st)
        torch.cuda.synchronize()
        ms = a.elapsed_time(b)
    # warm regime through one CUDA graph: the step's launches replayed back to back, no host launch cost in
    # between (what an LLG loop that keeps M and H on the device would see; inputs may sit in L2)
    graph_ms = None
    try:
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        side.wait_stream(st)
        with torch.cuda.stream(side):
            step()
            with torch.cuda.graph(g, stream=side):
                step()
        st.wait_stream(side)
        torch.cuda.synchronize()
        reps = max(20, min(steps, 200))
        ga, gb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g.replay()
        ga.record(st)
        for _ in range(reps):
            g.replay()
        gb.record(st)
        torch.cuda.synchronize()
        graph_ms = ga.elapsed_time(gb) / reps
        del g
    except Exception as e:                      # graph capture is an extra measurement, never the headline
        graph_ms = None
        print(f"[bench] CUDA graph timing skipped: {e}", file=sys.stderr)
    # per-kernel device time (event pairs around every launch, on the launching stream)
    kinds = {}
    for _ in range(profile_reps):
        if flush:
            scratch.fill_(1)
        for k, (t, n) in plan.apply_timed(M, H).items():
            kinds.setdefault(k, [0.0, 0])
            kinds[k][0] += t
            kinds[k][1] += n
    ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ems = 0.0
    for _ in range(profile_reps):
        if flush:
            scratch.fill_(1)
        ea.record(st)
        plan.energy(M, H, E)
        eb.record(st)
        torch.cuda.synchronize()
        ems += ea.elapsed_time(eb)
    kb = kind_bytes(cfg, info)
    kf = kind_flops(cfg, info)
    alu_peak = 148 * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6          # flop/s, FMA counted as 2
    comp = info["compulsory_bytes"]
    # every launch of every kind covers the whole mesh (launches_per_eval > 1 only on the chunked fallback, whose
    # launches together cover it once), so the algorithmic bytes of a kind per evaluation are the compulsory bytes
    # of the evaluation (24 B per cell + the reduced kernel spectrum); the bytes the kernel is
    # DESIGNED to move (its inputs and outputs once, intermediate spectra included) are reported beside them
    per_kind = {k: {"ms_per_eval": t / profile_reps, "launches_per_eval": n // profile_reps,
                    "algorithmic_bytes": comp, "gbs": comp / (t / profile_reps) / 1e6,
                    "hbm_frac": comp / (t / profile_reps) / 1e6 / peak_gbs,
                    "designed_bytes": kb[k], "kernel_gbs_designed": kb[k] / (t / profile_reps) / 1e6,
                    "flops_5NlogN": kf.get(k), "alu_frac": (kf[k] / (t / profile_reps * 1e-3) / alu_peak) if k in kf else None}
                for k, (t, n) in kinds.items()}
    # the stand-alone energy kernel (boris_demag_energy); the timed step gathers E inside its last kernel instead
    per_kind["Energy"] = {"ms_per_eval": ems / profile_reps, "launches_per_eval": 1,
                          "algorithmic_bytes": 24 * cfg.cells, "gbs": 24 * cfg.cells / (ems / profile_reps) / 1e6,
                          "hbm_frac": 24 * cfg.cells / (ems / profile_reps) / 1e6 / peak_gbs}
    ms_step = ms / steps
    res = {"config": cfg.name, "mesh": [cfg.nx, cfg.ny, cfg.nz], "padded": list(info["padded"]),
           "ms_per_step": ms_step, "evals_per_s": 1e3 / ms_step, "mcell_per_s": cfg.cells / ms_step / 1e3,
           "compulsory_bytes": info["compulsory_bytes"], "designed_hbm_bytes": info["designed_hbm_bytes"],
           "hbm_roofline_frac": info["compulsory_bytes"] / (ms_step * 1e-3) / (peak_gbs * 1e9),
           "designed_hbm_passes": info["designed_hbm_bytes"] / info["compulsory_bytes"],
           "launches_per_step": info["kernel_launches"] + (0 if info["path"] else 1), "l2": "flushed between steps" if flush else "inputs > L2",
           "ms_per_step_warm_graph": graph_ms, "flops": path_flops(cfg), "kernels": per_kind}
    return res, plan, (M_host, M, H, E)


def time_e2e(torch, plan, cfg, M_host, steps, warmup):
    """Same metric through boris_demag_apply_host with pinned HOST buffers (H2D + kernels + D2H timed)."""
    Mp = torch.from_numpy(M_host).pin_memory()
    Hp = torch.empty_like(Mp).pin_memory()
    for _ in range(max(1, min(warmup, 3))):
        plan.apply_host(Mp, Hp)
    torch.cuda.synchronize()
    n = max(3, min(steps, 20))
    t0 = time.perf_counter()
    for _ in range(n):
        plan.apply_host(Mp, Hp)              # synchronises the stream before returning
    dt = time.perf_counter() - t0
    return n, dt / n, Mp.numel() * 4, Hp.numel() * 4 + 8


# ----------------------------------------------------------------- oracle arm (CPU baseline / --impl reference)
def oracle_setup(cfg):
    """The fp64 oracle on the FULL mesh of the workload (no sub-sampling, nothing scaled); its kernel spectrum is
    precomputed and excluded from the timing, as the GPU plan's is."""
    from oracle.demag_direct import tensor_table          # the only place bench.py touches oracle/
    from oracle.demag_fft import demag_fft, kernel_spectrum
    M = W.make_input(cfg)
    Khat = kernel_spectrum(cfg.shape, cfg.h, table=tensor_table(cfg.shape, cfg.h))
    what = (f"the full {cfg.nx}x{cfg.ny}x{cfg.nz} mesh of {cfg.name}, fp64 zero-padded FFT convolution "
            "oracle/demag_fft.py (scipy pocketfft, all host cores), kernel spectrum precomputed")
    return M, Khat, (lambda: demag_fft(M, cfg.h, Khat=Khat)), what


def cpu_baseline(cfg, budget_s=12.0):
    M, Khat, run, what = oracle_setup(cfg)
    run()
    n, t0 = 0, time.perf_counter()
    while True:
        run()
        n += 1
        dt = time.perf_counter() - t0
        if (dt > budget_s and n >= 3) or n >= 20:
            break
    return {"value": n / dt, "unit": UNIT, "mcell_per_s": cfg.cells * n / dt / 1e6,
            "cores": os.cpu_count(), "kind": "oracle", "sample": f"{n} evaluations of {what}",
            "cpu": cpu_model()}


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def run_reference(args, cfg):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    M, Khat, run, what = oracle_setup(cfg)
    for _ in range(args.warmup):
        run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run()
    dt = time.perf_counter() - t0
    value = args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name} {cfg.nx}x{cfg.ny}x{cfg.nz}", "sample": what},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                             "sample": f"each step = one evaluation of {what}", "cpu": cpu_model()},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ----------------------------------------------------------------- device probes (profiles/*_microbench.md)
def run_micro(torch, binding, build):
    """FP32 lane rate per instruction kind and HBM throughput per piece size, as one JSON line and a table."""
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --micro needs a CUDA device")
    build.build()
    peak_gbs, sm_max_mhz, peak_src = measured_peaks()
    names = ["FADD", "FFMA", "FADD2 (packed)", "FFMA2 (packed)"]
    rate = {n: binding.micro_fp32_rate(i) for i, n in enumerate(names)}
    nominal = 148 * FP32_LANES_PER_SM * sm_max_mhz * 1e6
    seg = {str(sb): {"read_gbs": binding.micro_segment_bw(sb, False), "write_gbs": binding.micro_segment_bw(sb, True)}
           for sb in (16, 32, 64, 128, 256, 512)}
    print("| instruction | T lane-ops/s | of 148 SM x 128 lanes x %.0f MHz |" % sm_max_mhz, file=sys.stderr)
    for n in names:
        print(f"| {n} | {rate[n] / 1e12:.2f} | {rate[n] / nominal:.3f} |", file=sys.stderr)
    print("| piece bytes | read GB/s | write GB/s | read / %.0f GB/s (%s) |" % (peak_gbs, peak_src), file=sys.stderr)
    for sb, v in seg.items():
        print(f"| {sb} | {v['read_gbs']:.0f} | {v['write_gbs']:.0f} | {v['read_gbs'] / peak_gbs:.3f} |", file=sys.stderr)
    print(json.dumps({"micro": {"fp32_lane_ops_per_s": rate, "nominal_lane_rate": nominal, "segments": seg,
                                "hbm_peak_gbs": peak_gbs, "peak_source": peak_src}}))


# ----------------------------------------------------------------- multi-GPU: replicas only
def max_over_ranks(x, dist, device):
    """The slowest rank's time: every multi-GPU number is the max over ranks (no data-path collective exists)."""
    if dist is None:
        return x
    import torch
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_throughput(world, ms_per_step):
    """Whole-job evaluations/s of `world` independent replicas that each take ms_per_step (weak scaling)."""
    return world * 1e3 / ms_per_step


# ----------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="C5", choices=sorted(W.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-all-configs", action="store_true", help="skip the four secondary configs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--micro", action="store_true",
                    help="print the table of the two device probes of include/boris_micro.h and exit")
    args = ap.parse_args()
    cfg = W.CONFIGS[args.config]
    args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    from paper_2008_02478_b200 import binding, build
    if args.micro:
        run_micro(torch, binding, build)
        return
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    if rank == 0:
        build.build()
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist.barrier()
    binding.lib()
    peak_gbs, sm_max_mhz, peak_src = measured_peaks()
    warmup = max(args.warmup, 3)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- headline: K steps, barrier + synchronize on both sides, device time, max over ranks
    flush = 24 * cfg.cells < (192 << 20)          # M + H smaller than ~1.5 x L2: flush L2 between steps
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    res, plan, (M_host, M, H, E) = time_config(torch, binding, cfg, args.steps, warmup, flush, peak_gbs, sm_max_mhz)
    barrier()
    clocks = sampler.stop()
    ms_step = res["ms_per_step"]
    ms_step = max_over_ranks(ms_step, dist, "cuda")
    n_e2e, e2e_s, h2d, d2h = time_e2e(torch, plan, cfg, M_host, args.steps, warmup)
    e2e_s = max_over_ranks(e2e_s, dist, "cuda")
    if rank != 0:
        barrier()
        dist.destroy_process_group()
        return

    kernels = res["kernels"]
    dom = max((k for k in kernels if k != "Energy"), key=lambda k: kernels[k]["ms_per_eval"])
    dk = kernels[dom]
    launches = max(dk["launches_per_eval"], 1)
    # achieved = algorithmic (compulsory) bytes of the work one launch covers / its duration;
    # the throughput over the bytes the kernel is designed to move is reported under its own key
    roofline = {"kernel": dom, "bound": "hbm", "achieved": dk["gbs"], "peak": peak_gbs, "unit": "GB/s",
                "frac": dk["gbs"] / peak_gbs, "traffic": ncu_traffic(cfg.name, dom), "peak_source": peak_src,
                "algorithmic_bytes_per_launch": dk["algorithmic_bytes"] / launches,
                "avg_launch_ms": dk["ms_per_eval"] / launches, "launches_per_eval": launches,
                "kernel_gbs_designed": dk["kernel_gbs_designed"], "designed_bytes_per_launch": dk["designed_bytes"] / launches,
                "alu_frac": dk["alu_frac"],
                "share_of_eval": dk["ms_per_eval"] / sum(v["ms_per_eval"] for k, v in kernels.items() if k != "Energy")}
    alu_peak = 148 * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    path = {"compulsory_bytes": res["compulsory_bytes"], "hbm_frac_of_peak": res["compulsory_bytes"] / (ms_step * 1e-3) / (peak_gbs * 1e9),
            "designed_hbm_passes": res["designed_hbm_passes"], "flops_5NlogN": res["flops"],
            "tflops": res["flops"] / (ms_step * 1e-3) / 1e12, "fp32_fma_peak_tflops": alu_peak,
            "alu_frac_of_peak": res["flops"] / (ms_step * 1e-3) / 1e12 / alu_peak}
    line = {"metric": METRIC, "value": replica_throughput(world, ms_step), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{cfg.name} {cfg.nx}x{cfg.ny}x{cfg.nz} cells, padded {'x'.join(map(str, res['padded']))}, "
                                   f"seeded {cfg.texture} texture; step = boris_demag_apply_energy (H and E)",
                       "l2": res["l2"], "parallelism": "replicas only" if world > 1 else "single GPU"},
            "mcell_per_s": world * cfg.cells / ms_step / 1e3,
            "e2e": {"value": world / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": n_e2e, "api": "boris_demag_apply_host (pinned host M in, H and E out)"},
            "gpu_launches": res["launches_per_step"] * args.steps,
            "clocks": clocks, "roofline": roofline, "path_roofline": path, "kernels": kernels}
    # the paper's own benchmark unit: time per evaluation of an RK4 step with demag,
    # exchange and applied field (include/boris_llg.h); side information, not the headline metric
    if world == 1:
        try:
            solver = binding.LLG(plan, cfg.Ms, 1.3e-11, 0.02, Hext=(0.0, 0.0, 1e4))
            mu = (M / cfg.Ms).contiguous()
            solver.rk4(mu, 1e-13, 2)
            torch.cuda.synchronize()
            nst = 5
            la, lb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            la.record(torch.cuda.current_stream())
            solver.rk4(mu, 1e-13, nst)
            lb.record(torch.cuda.current_stream())
            torch.cuda.synchronize()
            ms_eval = la.elapsed_time(lb) / (4 * nst)
            line["llg"] = {"ms_per_evaluation": ms_eval, "evaluations_per_s": 1e3 / ms_eval, "ms_per_rk4_step": 4 * ms_eval,
                           "terms": "demag + exchange (6-neighbour, Neumann) + applied field, LLG torque, RK4 bookkeeping",
                           "demag_share": res["kernels"] and sum(v["ms_per_eval"] for k, v in res["kernels"].items()
                                                                 if k != "Energy") / ms_eval}
            solver.close()
            del mu
        except Exception as e:
            print(f"[bench] LLG evaluation timing skipped: {e}", file=sys.stderr)
    # boris_demag_apply_ex(ACCUMULATE): fused into the kernel that writes H on the tiled / plane paths
    if world == 1:
        try:
            def timed(fn, nrep=5):
                fn()
                torch.cuda.synchronize()
                ta, tb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                ta.record(torch.cuda.current_stream())
                for _ in range(nrep):
                    fn()
                tb.record(torch.cuda.current_stream())
                torch.cuda.synchronize()
                return ta.elapsed_time(tb) / nrep
            Hacc = torch.zeros_like(H)
            t_plain = timed(lambda: plan.apply(M, H))
            t_acc = timed(lambda: plan.apply_ex(M, Hacc, plan.ACCUMULATE))
            line["apply_ex"] = {"apply_ms": t_plain, "accumulate_ms": t_acc, "accumulate_over_apply": t_acc / t_plain}
            del Hacc
        except Exception as e:
            print(f"[bench] apply_ex timing skipped: {e}", file=sys.stderr)
    # the double-precision variant (include/boris_demag_f64.h; "single or double"): side information
    if world == 1:
        try:
            p64 = binding.DemagPlanF64(cfg.nx, cfg.ny, cfg.nz, *cfg.h)
            M64 = M.double()
            H64 = torch.empty_like(M64)
            for _ in range(2):
                p64.apply(M64, H64)
            torch.cuda.synchronize()
            fa, fb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            nrep = 5
            fa.record(torch.cuda.current_stream())
            for _ in range(nrep):
                p64.apply(M64, H64)
            fb.record(torch.cuda.current_stream())
            torch.cuda.synchronize()
            ms64 = fa.elapsed_time(fb) / nrep
            dev = (H64.float() - H).abs().max().item() / cfg.Ms
            line["f64"] = {"ms_per_evaluation": ms64, "evaluations_per_s": 1e3 / ms64, "kernel_launches": 5,
                           "max_abs_diff_to_f32_over_Ms": dev, "workspace_bytes": p64.info()["workspace_bytes"]}
            p64.close()
            del M64, H64
        except Exception as e:
            print(f"[bench] fp64 variant timing skipped: {e}", file=sys.stderr)
    del plan, M, H, E
    torch.cuda.empty_cache()
    # the next size up from the headline mesh (same plane path, eight ky residues): time per cell against C5's
    if world == 1 and not args.no_all_configs and cfg.name == "C5":
        try:
            big = W.Config("C5x4", 1024, 1024, 32, cfg.hx, cfg.hy, cfg.hz, cfg.Ms, 2005, "random")
            pb = binding.DemagPlan(big.nx, big.ny, big.nz, *big.h)
            Mb = torch.randn(3, big.nz, big.ny, big.nx, device="cuda") * (cfg.Ms / 3 ** 0.5)
            Hb = torch.empty_like(Mb)
            for _ in range(3):
                pb.apply(Mb, Hb)
            torch.cuda.synchronize()
            ba, bb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ba.record(torch.cuda.current_stream())
            for _ in range(5):
                pb.apply(Mb, Hb)
            bb.record(torch.cuda.current_stream())
            torch.cuda.synchronize()
            msb = ba.elapsed_time(bb) / 5
            line["next_size"] = {"mesh": [big.nx, big.ny, big.nz], "path": pb.layout()["path"], "ms_per_apply": msb,
                                 "ns_per_cell": msb * 1e6 / big.cells,
                                 "per_cell_over_headline": (msb / big.cells) / (ms_step / cfg.cells)}
            pb.close()
            del Mb, Hb
            torch.cuda.empty_cache()
        except Exception as e:
            print(f"[bench] next-size timing skipped: {e}", file=sys.stderr)
    if world == 1 and not args.no_all_configs:
        allc = {cfg.name: {k: v for k, v in res.items() if k != "kernels"}}
        for name in sorted(W.CONFIGS):
            if name == cfg.name:
                continue
            c = W.CONFIGS[name]
            steps = 200 if c.cells <= (1 << 20) else 50
            r, p, bufs = time_config(torch, binding, c, steps, 5, 24 * c.cells < (192 << 20), peak_gbs, sm_max_mhz, profile_reps=3)
            allc[name] = r
            p.close()
            del bufs
            torch.cuda.empty_cache()
        line["all_configs"] = allc
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(cfg)
    print(json.dumps(line))
    if dist is not None:
        barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
