#!/usr/bin/env python
"""bench.py -- throughput of the projection cycle (BASELINE.json `metric`).

    python bench.py --gpus N --steps K --warmup W            # this build (CUDA path, C ABI), config 2
    python bench.py --config {1,2,3,4} [--alg DM|EPIE_MB|LSQML]   # the other configurations of BASELINE.json
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle as it stands
    python bench.py --cufft-ref                              # harness-side reference point: the cycle as unfused torch.fft ops

A "step" is one iteration over all J scan positions.  The default is config 2 (BASELINE.json configs[2]: DM,
256x256 frames, 10 000 Fermat-spiral positions, 4096^2 object, uint16 Poisson counts) -- the
configuration the metric "diffraction patterns/sec per DM iteration (256x256, 1 B200)" is quoted
on.  `value` = J * K / (device time of K iterations), inputs resident in HBM; `e2e` = the same
through the C ABI from pinned HOST buffers: ptycho_init (H2D of intensities, object, probe,
positions) + one iteration + ptycho_fetch_error, all inside the timed region (that one iteration is the FIRST
one after init: for DM it forms psi = P O_j inside the kernel instead of reading the exit-wave store).
N > 1: the path does not shard in this build ("replicas only"): every rank
reconstructs its own replica scan, no data-path collective; time = max over ranks.

Prints ONE JSON line (rank 0).  Inputs are seeded synthetic scans (paper_2202_03144_b200/synth.py).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

_ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, _ROOT)

METRIC = "diffraction patterns/sec per DM iteration (256x256, 1 B200); % HBM roofline"
UNIT = "patterns/s"
CFG = 2                      # default: BASELINE.json configs[2]
DEFAULT_ALG = {1: "EPIE_MB", 2: "DM", 3: "LSQML", 4: "DM"}
FULL_J = {1: 1024, 2: 10000, 3: 20000, 4: 16384}
REF_SAMPLE = {1: 256, 2: 256, 3: 96, 4: 64}   # frames of the bounded oracle sample (first positions of the same scan)
TRAFFIC_FILE = os.path.join(_ROOT, "profiles", "r02_traffic.json")   # ncu dram__bytes per launch of the dominant kernel, per config


def ncu_traffic(cfg: int, alg: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, from the committed ncu summary
    (profiles/r02_traffic.json, written from the `ncu --set full` captures named in profiles/r02.md); None if not captured."""
    try:
        with open(TRAFFIC_FILE) as f:
            return json.load(f).get(f"cfg{cfg}_{alg}")
    except Exception:
        return None


def flops_per_pattern(n: int, k: int) -> float:
    """nominal K (2 * 10 N^2 log2 N + 40 N^2) (two 2-D transforms of 5 N^2 log2 N^2 flops + point-wise work)."""
    return k * (2 * 10 * n * n * np.log2(n) + 40 * n * n)


def algorithmic_bytes_per_pattern(n: int, k: int, bytes_i: int) -> int:
    """DM streams psi in, psi out and I in: N^2 (16 K + b_I)."""
    return n * n * (16 * k + bytes_i)


def measured_peaks():
    p = os.path.join(_ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# --------------------------------------------------------------------------- clocks during the run
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML every `period` seconds."""

    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTE = {"sw_power_cap": 0x4, "hw_power_brake": 0x80, "sync_boost": 0x10}

    def __init__(self, index: int, period: float = 0.01, uuid: str | None = None):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples: list[tuple[float, int, int]] = []
        self.max_mhz = None
        self._stop_ev = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:                                             # CUDA_VISIBLE_DEVICES may renumber
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if uuid and not uuid.startswith("GPU-") else uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:                               # NVML missing: report that
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        while not self._stop_ev.is_set():
            try:
                mhz = int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                try:
                    rs = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    rs = int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.samples.append((time.perf_counter(), mhz, rs))
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_ev.set()

    def summary(self, t0: float, t1: float) -> dict:
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml_unavailable"]}
        inside = [(m, r) for (t, m, r) in self.samples if t0 <= t <= t1]
        if not inside:                                       # region shorter than one period
            inside = [(m, r) for (_, m, r) in self.samples[-3:]]
        mhz = sorted(m for m, _ in inside)
        bits = 0
        for _, r in inside:
            bits |= r
        reasons = [k for k, v in {**self.BAD, **self.NOTE}.items() if bits & v]
        return {"sm_mhz": mhz[len(mhz) // 2] if mhz else None, "sm_max_mhz": self.max_mhz,
                "reasons": reasons, "samples": len(inside)}


# --------------------------------------------------------------------------- reference arm (oracle)
def scan_params(s, alg: str) -> dict:
    """Parameters of the run: the config's own (synth.params) for the chosen algorithm."""
    par = {}
    if alg == "DM":
        par["pbound"] = s.params.get("pbound", s.params.get("pbound_dm", 0.0))
    else:
        par["batch_size"] = s.params.get("batch_size", 0)
        par["disable_dm"] = 1
    return par


def workload_name(cfg: int, alg: str, s, J: int) -> str:
    return (f"cfg{cfg} {alg} {s.n}x{s.n} J={J} H={s.obj0.shape[0]} {s.intensities.dtype} K={s.n_modes}"
            +  (f" pbound={scan_params(s, alg)['pbound']}" if alg == "DM" else f" batch={s.params.get('batch_size', 0)}"))


def run_oracle_sample(cfg: int, alg: str, steps: int, warmup: int):
    """Times the CPU oracle (oracle/, as it stands) on the first REF_SAMPLE[cfg] positions of the config:
    one step = one oracle iteration over those frames.  Returns (patterns/s, ms/step, cores, sample)."""
    import oracle
    from paper_2202_03144_b200 import synth
    oracle.build()
    sample = REF_SAMPLE[cfg]
    s = synth.make_config(cfg, n_pos=sample)
    par = {k: v for k, v in scan_params(s, alg).items() if k != "disable_dm"}
    o = oracle.Oracle(s.obj0, s.probe0, s.pos, s.intensities, par)
    for _ in range(warmup):
        o.iterate(alg, 1)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.iterate(alg, 1)
    dt = time.perf_counter() - t0
    cores = int(os.environ.get("OMP_NUM_THREADS", 0)) or (os.cpu_count() or 1)
    return sample * steps / dt, dt / steps * 1e3, cores, sample


def reference_line(args) -> dict:
    from paper_2202_03144_b200 import synth
    cfg, alg = args.config, args.alg or DEFAULT_ALG[args.config]
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    val, ms, cores, sample = run_oracle_sample(cfg, alg, steps, warmup)
    s = synth.make_config(cfg, n_pos=4)
    what = (f"first {sample} positions of config {cfg} (same generator), one oracle {alg} iteration "
            f"(fp64, OpenMP over frames) per step")
    return {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg, alg, s, FULL_J[cfg]) + " (bounded sample)", "sample_frames": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


def cufft_reference_line(args) -> dict:
    """B:ns "cuFFT is reported only as a reference point": the DM cycle of config 2's frame size written as unfused torch
    operations on resident frames (reflector, fft2, modulus replacement, ifft2, exit-wave update; no object gather, no
    overlap sums, no error) and the two bare transforms alone.  Harness-side only; the library never calls cuFFT."""
    import torch
    from paper_2202_03144_b200 import synth
    dev = torch.device("cuda", 0)
    n, f = (synth.make_config(args.config, n_pos=4).n), 2000
    g = torch.Generator(device=dev).manual_seed(0)
    psi = torch.randn((f, n, n), dtype=torch.complex64, device=dev, generator=g)
    po = torch.randn((f, n, n), dtype=torch.complex64, device=dev, generator=g)
    amp = torch.rand((f, n, n), device=dev, generator=g) * 30
    def bare():
        return torch.fft.ifft2(torch.fft.fft2(psi))
    def cycle():
        phi = torch.fft.fft2(2 * po - psi)
        phi = phi * (amp / phi.abs().clamp_min(1e-30))
        return psi + torch.fft.ifft2(phi) - po
    out = {}
    for name, fn in (("fft2_ifft2", bare), ("unfused_cycle", cycle)):
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(10):
            fn()
        e1.record()
        torch.cuda.synchronize()
        out[name] = f * 10 / (e0.elapsed_time(e1) * 1e-3)
    return {"impl": "cufft_reference_point", "unit": "frames/s", "frame": n, "frames_resident": f, **out,
            "note": "torch.fft (cuFFT) on resident complex64 frames; a reference point, not part of the library"}


def mma_dft_line(args) -> dict:
    """B:ns "tensor cores ... DFT-as-GEMM ... only if it beats the packed-fp32 line FFT at <= 2e-6 error": the micro-benchmark.
    The forward FFT of every row of resident 256 x 256 complex64 frames by (0) the row pass of the product kernels and (1) the
    tensor-core kernel of csrc/fft_mma.cuh, on 2048 frames (1 GB, 524 288 lines per launch; a working set small enough to stay in
    L2 would make launches of ~20 us, which measure the launch); CUDA events, 20 repetitions after 3 warm-ups; error of each
    against numpy's FFT in double.  torch.fft (cuFFT) rows beside them as a reference point.  At 4 KB per line the HBM bound is
    1.6 G lines/s."""
    import torch
    from paper_2202_03144_b200 import binding
    dev = torch.device("cuda", 0)
    n = 256
    g = torch.Generator(device=dev).manual_seed(1)
    out = {"impl": "mma_dft_microbenchmark", "unit": "lines/s", "line": n}
    small = torch.randn((6, n, n), dtype=torch.complex64, device=dev, generator=g)
    want = np.fft.fft(small.cpu().numpy().astype(np.complex128), axis=-1)
    for impl, name in ((0, "packed_fp32"), (1, "mma_tf32x3")):
        got = binding.test_fft_rows(small.clone(), impl=impl).cpu().numpy()
        out[name + "_rel_l2_error"] = float(np.linalg.norm(got - want) / np.linalg.norm(want))
    for frames, tag in ((2048, "hbm_streamed_1GB"),):
        x = torch.randn((frames, n, n), dtype=torch.complex64, device=dev, generator=g)
        fns = {"packed_fp32": lambda: binding.test_fft_rows(x, impl=0), "mma_tf32x3": lambda: binding.test_fft_rows(x, impl=1),
               "cufft_rows": lambda: torch.fft.fft(x, dim=-1, out=x)}
        for name, fn in fns.items():
            x.normal_(generator=g); x *= 1e-30               # unscaled transforms applied repeatedly in place (x16 each): stays finite
            for _ in range(3):
                fn()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(20):
                fn()
            e1.record()
            torch.cuda.synchronize()
            out[f"{name}_{tag}"] = frames * n * 20 / (e0.elapsed_time(e1) * 1e-3)
    out["note"] = ("rows only (load, 256-point FFT, store); lines/s; the product's DM iteration needs 4 x 2.56 M line FFTs at config 2. "
                   "A micro-benchmark: the tensor-core kernel is not part of any product path")
    return out


# --------------------------------------------------------------------------- this build's arm
def dist_env():
    return (int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)),
            int(os.environ.get("WORLD_SIZE", 1)))


def max_over_ranks(x: float, world: int, device=None) -> float:
    """Slowest rank's time (the contract's max over ranks); identity for a single process."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device if dist.get_backend() == "nccl" else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def ours_line(args) -> dict | None:
    import torch
    rank, local, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the projection cycle has no CPU path "
                         "(use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    from paper_2202_03144_b200 import binding, synth
    binding.lib()                                            # fails loudly if the .so is missing

    cfg, alg = args.config, args.alg or DEFAULT_ALG[args.config]
    steps, warmup = max(1, args.steps), max(3, args.warmup)
    s = synth.make_config(cfg, n_pos=args.n_pos, replica=rank, threads=max(2, (os.cpu_count() or 8) // world))
    J, N, K = s.n_pos, s.n, s.n_modes
    par = scan_params(s, alg)
    obj0 = torch.from_numpy(s.obj0.astype(np.complex64))
    probe0 = torch.from_numpy(s.probe0.astype(np.complex64))
    inten_h = torch.from_numpy(s.intensities).pin_memory()
    obj_h, probe_h = obj0.pin_memory(), probe0.pin_memory()

    # ---- device-resident timing: inputs in HBM before the timed region
    inten_d = inten_h.to(dev)
    g = binding.Ptycho(obj0.to(dev), probe0.to(dev), s.pos, inten_d, binding.default_params(**par), device=dev)
    stream = torch.cuda.current_stream(dev)
    for _ in range(warmup):
        g.iterate(alg, 1)
    try:
        uuid = str(torch.cuda.get_device_properties(dev).uuid)
    except Exception:
        uuid = None
    sampler = ClockSampler(local, uuid=uuid)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    barrier(world)
    g.profile(True)
    l0 = g.launch_count()
    t0 = time.perf_counter()
    e0.record(stream)
    for _ in range(steps):
        g.iterate(alg, 1)
    e1.record(stream)
    torch.cuda.synchronize(dev)
    t1 = time.perf_counter()
    barrier(world)
    ms = max_over_ranks(float(e0.elapsed_time(e1)), world, dev)
    launches = g.launch_count() - l0
    prof = g.profile_fetch()
    g.profile(False)
    clocks = sampler.summary(t0, t1)
    err_hist = g.fetch_error()
    assert np.all(np.isfinite(err_hist)), "non-finite error history"
    g.destroy()
    del g, inten_d
    torch.cuda.empty_cache()

    # ---- end to end through the C ABI from pinned host buffers (H2D + iterate + D2H inside)
    e2e_steps = min(steps, 10 if cfg != 4 else 3)
    h2d = inten_h.numel() * inten_h.element_size() + obj_h.numel() * 8 + probe_h.numel() * 8 + s.pos.nbytes
    e2e_ms = []
    for i in range(e2e_steps + 1):
        torch.cuda.synchronize(dev)
        barrier(world)
        e0.record(stream)
        ge = binding.Ptycho(obj_h, probe_h, s.pos, inten_h, binding.default_params(**par), device=dev)
        ge.iterate(alg, 1)
        ev = ge.fetch_error()                                # D2H of the step's result (8 bytes)
        e1.record(stream)
        torch.cuda.synchronize(dev)
        if i > 0:                                            # first one is the warm-up (allocator)
            e2e_ms.append(float(e0.elapsed_time(e1)))
        assert np.isfinite(ev[-1])
        ge.destroy()
        del ge
    sampler.stop()
    e2e_ms_step = max_over_ranks(sum(e2e_ms) / len(e2e_ms), world, dev)

    # ---- roofline of the dominant kernel chain
    hbm_peak, peak_src = measured_peaks()
    chain = ("mega",) if prof.get("mega", (0.0, 0))[1] > 0 else ("rows_fwd", "cols", "rows_inv")
    chain_ms = sum(prof[k][0] for k in chain)
    n_chain = sum(prof[k][1] for k in chain)
    bytes_i = s.intensities.dtype.itemsize
    full = args.n_pos is None
    if alg == "DM":                                          # HBM-bound: psi in, psi out, I in per pattern
        alg_bytes = algorithmic_bytes_per_pattern(N, K, bytes_i)
        achieved = alg_bytes * J * steps / (chain_ms * 1e-3) / 1e9 if chain_ms > 0 else 0.0
        roofline = {"bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s", "frac": achieved / hbm_peak,
                    "peak_source": peak_src, "algorithmic_bytes_per_pattern": alg_bytes,
                    "step_frac_of_hbm_roofline": (alg_bytes * J * steps * world / (ms * 1e-3) / 1e9) / (hbm_peak * world)}
    else:                                                    # no exit-wave traffic: the fp32 ALUs bind
        mhz = clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965
        peak = 148 * 128 * 2 * mhz * 1e6 / 1e12             # SMs x fp32 lanes x 2 flop (FMA) x SM clock sampled in this run
        fl = flops_per_pattern(N, K)
        achieved = fl * J * steps / (chain_ms * 1e-3) / 1e12 if chain_ms > 0 else 0.0
        roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                    "peak_source": f"148 SMs x 128 fp32 lanes x 2 x {mhz} MHz (median SM clock of this run)",
                    "nominal_flops_per_pattern": fl,
                    "frac_of_hbm_roofline": (N * N * bytes_i * J * steps / (ms * 1e-3) / 1e9) / hbm_peak}
    roofline.update({
        "traffic": ncu_traffic(cfg, alg) if full else None,
        "traffic_source": "profiles/r02_traffic.json: ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum per launch (profiles/r02.md)",
        "kernel": ("k_dm_mega (one persistent launch per DM iteration: a1-a9 of all frames)" if chain == ("mega",)
                   else "k_rows_fwd + k_cols + k_rows_inv (one launch triple per chunk of a minibatch)"),
        "launches_timed": n_chain, "avg_launch_ms": chain_ms / max(n_chain, 1),
        "kernel_ms_per_step": {k: prof[k][0] / steps for k in prof},
    })
    line = {
        "metric": METRIC, "value": J * steps * world / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
        "steps": steps, "warmup": warmup, "ms_per_step": ms / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg, alg, s, J),
                   "l2": "inputs larger than L2 (%.2f GB streamed per step)" % ((J * K * N * N * 16 * (alg == "DM") + J * N * N * bytes_i) / 1e9),
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "e2e_step": f"ptycho_init from pinned host buffers + the FIRST {alg} iteration + ptycho_fetch_error",
                   "e2e_steps": e2e_steps,
                   "timed_iterations": f"{warmup}..{warmup + steps - 1} of a run from the flat object (DM: frames inside the power bound "
                                       "take the short pass 3; see DESIGN.md section 5)"},
        "clocks": clocks,
        "e2e": {"value": J * world / (e2e_ms_step * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": 8, "ms_per_step": e2e_ms_step},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "error_first_last": [float(err_hist[0]), float(err_hist[-1])],
    }
    if world == 1 and rank == 0 and not args.no_cpu_baseline:
        val, _, cores, sample = run_oracle_sample(cfg, alg, steps=4 if cfg in (3, 4) else 6, warmup=1)
        line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"first {sample} positions of config {cfg}, oracle {alg} iterations (fp64, OpenMP)"}
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return line if rank == 0 else None


def sharded_line(args) -> dict | None:
    """--sharded: ONE scan of the config split over the N ranks: strong scaling.  Not the
    driver's mode (B:ns asks for replicas); kept so that the sharded path can be timed the same way.  Timed region = `steps` DM
    iterations, each ptycho_shard_begin + neighbour exchange of the correction canvas + all-reduce of the probe sums +
    ptycho_shard_end, CUDA events, max over ranks."""
    import torch
    import torch.distributed as dist
    rank, local, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the projection cycle has no CPU path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if "RANK" in os.environ and "MASTER_ADDR" in os.environ:       # launched by torchrun (any world size): its rendezvous
        dist.init_process_group("nccl", device_id=dev)
    else:                                                            # plain `python bench.py --sharded`: a group of one
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % (29500 + os.getpid() % 2000), rank=0, world_size=1, device_id=dev)
    from paper_2202_03144_b200 import binding, sharded, synth
    binding.lib()
    cfg = args.config
    if DEFAULT_ALG[cfg] != "DM" or (args.alg or "DM") != "DM":
        raise SystemExit("bench.py --sharded: DM configurations only (2, 4, or 1 with --alg DM is not sharded)")
    steps, warmup = max(1, args.steps), max(3, args.warmup)
    s = synth.make_config(cfg, n_pos=args.n_pos, replica=0, threads=max(2, (os.cpu_count() or 8) // world))   # the same scan on every rank
    par = scan_params(s, "DM")
    plan = sharded.shard_plan(s.pos, s.n, s.obj0.shape[0], s.obj0.shape[1], world)
    mine = plan.frames[rank]
    inten_d = torch.from_numpy(np.ascontiguousarray(s.intensities[mine])).to(dev)
    comm = sharded.DistComm()
    g = sharded.ShardedPtycho(plan, rank, torch.from_numpy(s.obj0.astype(np.complex64)).to(dev), torch.from_numpy(s.probe0.astype(np.complex64)).to(dev),
                              s.pos, inten_d, comm=comm, device=dev, **par)
    stream = torch.cuda.current_stream(dev)
    g.iterate(warmup)
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    barrier(world)
    l0 = g.core.launch_count()
    t0 = time.perf_counter()
    e0.record(stream)
    g.iterate(steps)
    e1.record(stream)
    torch.cuda.synchronize(dev)
    t1 = time.perf_counter()
    barrier(world)
    ms = max_over_ranks(float(e0.elapsed_time(e1)), world, dev)
    launches = g.core.launch_count() - l0
    sampler.stop()
    err = g.fetch_error()
    assert np.all(np.isfinite(err))
    halo_rows = sum(hi - lo for _, lo, hi in plan.exchange[rank])
    g.destroy()
    dist.destroy_process_group()
    J = s.n_pos
    alg_bytes = algorithmic_bytes_per_pattern(s.n, 1, s.intensities.dtype.itemsize)
    hbm_peak, peak_src = measured_peaks()
    achieved = alg_bytes * J * steps / (ms * 1e-3) / 1e9
    line = {"metric": METRIC, "value": J * steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(cfg, "DM", s, J), "parallelism": f"one scan sharded over {world} GPU(s): row bands, per iteration "
                       "a neighbour exchange of the correction canvas on shared rows and an all-reduce of the probe sums",
                       "halo_bytes_sent_per_step_rank0": int(halo_rows * s.obj0.shape[1] * 8), "frames_rank0": int(len(mine)),
                       "timed_iterations": f"{warmup}..{warmup + steps - 1}"},
            "clocks": sampler.summary(t0, t1), "e2e": None, "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": hbm_peak * world, "unit": "GB/s", "frac": achieved / (hbm_peak * world),
                         "peak_source": peak_src + f" x {world}", "algorithmic_bytes_per_pattern": alg_bytes, "traffic": None,
                         "kernel": "whole step (k_dm_mega + exchange + updates), all ranks"},
            "error_first_last": [float(err[0]), float(err[-1])]}
    return line if rank == 0 else None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=CFG, choices=[1, 2, 3, 4], help="BASELINE.json configs[i] (default 2: the metric's)")
    ap.add_argument("--alg", default=None, choices=["DM", "EPIE_MB", "LSQML"], help="default: the config's own algorithm")
    ap.add_argument("--cufft-ref", action="store_true", help="print the torch.fft reference point instead (harness-side)")
    ap.add_argument("--mma-dft", action="store_true", help="print the DFT-as-GEMM micro-benchmark instead (csrc/fft_mma.cuh)")
    ap.add_argument("--n-pos", type=int, default=None, help="truncate the scan (debugging only; invalidates the metric)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sharded", action="store_true", help="split ONE scan over the ranks instead of running replicas (SURVEY 8(f) f4)")
    args = ap.parse_args()
    rank, _, world = dist_env()
    if args.cufft_ref:
        if rank == 0:
            print(json.dumps(cufft_reference_line(args)), flush=True)
        return
    if args.mma_dft:
        if rank == 0:
            print(json.dumps(mma_dft_line(args)), flush=True)
        return
    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(reference_line(args)), flush=True)
        return
    line = sharded_line(args) if args.sharded else ours_line(args)
    if line is not None:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
