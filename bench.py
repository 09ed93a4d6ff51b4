#!/usr/bin/env python
"""bench.py -- series star-products per second on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg2|staple|batched4|exp|exp4|sweep]
    python bench.py --impl reference ...        # the CPU oracle as the reference arm

A step is one pass of the whole hot path over one synthetic input: for the default workload
(cfg3: N=225, N_trunc=63, the configuration the north-star target is quoted on) that is one
nspt_series_mul = forward transforms of A and B, 128 mode-wise 225^3 complex matrix products,
inverse transform with truncation.  Inputs are seeded synthetic unitary series
(paper_2001_02835_b200.workloads), resident in HBM before the timed region; the timed steps
rotate over R buffer sets whose total size exceeds twice the L2 so every step reads HBM.

Reported beside `value`:
  e2e          the same metric through the host-buffer C-ABI call (pinned host memory, H2D of A, B
               and D2H of C inside every step);
  roofline     the dominant kernel (mode-wise matrix product): conventional 8 N^3 L flops per launch
               / its mean launch duration (CUDA events on the library stream, second pass of K steps
               with the library's stage profiler on) against the FP64 tensor-pipe peak measured
               in-run by nspt_probe_fp64_peak (MEASURED_PEAKS.json has no FP64 entry);
  cpu_baseline the oracle (naive O(N_trunc^2) convolution, C + OpenMP) on this box's host cores,
               one full product of the same workload, rank 0 at N=1 only.

Multi-GPU: the path does not shard ("replicas only"): --gpus N runs N independent
replicas, one process per GPU (torchrun), no data-path collective; value = products of all ranks
/ max-over-ranks time, scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "series_star_products_per_sec"
L2_BYTES = 126e6

WORKLOADS = {
    # name: (kind, N, Ntrunc, batch, seed)
    "cfg3": ("product", 225, 63, 1, 3),
    "cfg2": ("product", 225, 31, 1, 2),
    "batched4": ("batched", 225, 31, 4, 2),
    "staple": ("staple", 225, 31, 1, 4),
    "mdstep": ("mdstep", 225, 31, 1, 4),          # staple + four forces + batched link update: one NSPT update of the four links
    "staple_split": ("staple", 225, 31, 1, 4),     # the paper's direction split: nspt_staple_dir per owned direction + all-gather
    "small": ("product", 9, 7, 1, 0),
    "sweep": ("sweep", 225, 31, 1, 5),
    "exp": ("exp", 225, 31, 1, 6),
    "exp4": ("exp", 225, 31, 4, 6),
}


WORKLOAD_DESC = {
    "cfg3": "single star-product A*B, N=225, N_trunc=63 (L=128), complex128, A,B = exp(i sum g^k H_k) series (BASELINE.json configs[2])",
    "cfg2": "single star-product A*B, N=225, N_trunc=31 (L=64), complex128 (BASELINE.json configs[1])",
    "batched4": "batch of 4 star-products, N=225, N_trunc=31 (the four P_mu*U_mu of a link update)",
    "staple": "full TEK staple S_mu, mu=1..4, N=225, N_trunc=31, k=4 twist (BASELINE.json configs[3]); 36 mode-wise products per step (literal eq. 2.3: 52)",
    "mdstep": "one update of the four TEK links at N=225, N_trunc=31 (PAPER.md:50-55): nspt_staple (36 products), four nspt_force, nspt_link_update_batched U <- exp(i eps F) * U (4 x 11 products); the integrator's momentum update is outside the library, the force series stands in for P",
    "staple_split": "full TEK staple S_mu, mu=1..4, N=225, N_trunc=31, k=4 twist (BASELINE.json configs[3]), directions split over the ranks (PAPER.md:140): 15 mode-wise products per owned direction, one all-gather of the four S_mu per step",
    "small": "single star-product A*B, N=9, N_trunc=7 (BASELINE.json configs[0])",
    "exp": "series exponential exp(X), X anti-Hermitian series, N=225, N_trunc=31 (link-update exponential; 10 mode-wise products, Paterson-Stockmeyer)",
    "exp4": "batch of 4 series exponentials (the four links of an update), N=225, N_trunc=31; 10 batched mode-wise products",
}


def transform_length(Ntrunc: int) -> int:
    L = 1
    while L < 2 * Ntrunc + 1:
        L *= 2
    return L


def exp_products(Ntrunc: int) -> int:
    """Mode-wise products nspt_series_exp executes: Paterson-Stockmeyer (s - 1) + (r - 1) with s = ceil(sqrt(n + 1)),
    r = ceil((n + 1) / s) for n = N_trunc >= 6, plain Horner n - 1 below."""
    if Ntrunc < 6:
        return max(Ntrunc - 1, 0)
    s = 1
    while s * s < Ntrunc + 1:
        s += 1
    r = (Ntrunc + 1 + s - 1) // s
    return (s - 1) + (r - 1)


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    return rank, local, world


def max_over_ranks(value: float, world: int, device=None) -> float:
    """Max of a scalar over all ranks (torch.distributed if initialised; identity otherwise)."""
    if world <= 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, world: int, device=None) -> float:
    if world <= 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(units_this_rank: float, ms_this_rank: float, world: int, device=None):
    """Whole-job throughput: units of all ranks / max-over-ranks time.  Returns (units/s, ms)."""
    ms = max_over_ranks(ms_this_rank, world, device)
    units = sum_over_ranks(units_this_rank, world, device)
    return units / (ms * 1e-3), ms


def read_traffic(workload: str, kernel: str):
    """DRAM bytes per launch of a kernel from the committed ncu summary table (profiles/traffic.csv:
    dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full` capture), or None."""
    tfile = ROOT / "profiles" / "traffic.csv"
    if not tfile.exists():
        return None
    try:
        for line in tfile.read_text().splitlines()[1:]:
            cols = line.split(",")
            if len(cols) >= 3 and cols[0] == workload and cols[1] == kernel:
                return float(cols[2])
    except Exception:
        return None
    return None


# ------------------------------------------------------------------------------------ clocks

class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.index = index
        self.samples = []
        self.reasons = set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        self._nvml = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nvml = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nvml = None
            return self
        self._thread = threading.Thread(target=self._run, daemon=True)
        self._thread.start()
        return self

    def _run(self):
        nv = self._nvml
        names = {
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def stop(self):
        self._stop.set()
        if self._thread is not None:
            self._thread.join(timeout=2.0)
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ------------------------------------------------------------------------------------ inputs

def make_inputs(kind, N, Ntrunc, batch, seed):
    from paper_2001_02835_b200 import workloads as wl
    if kind in ("staple", "mdstep"):
        U, z = wl.config_staple(N, Ntrunc, seed=seed)
        return {"U": U, "z": z}
    if kind == "batched":
        rng = np.random.default_rng(seed)
        A = np.stack([wl.unitary_series(N, Ntrunc, rng) for _ in range(batch)])
        B = np.stack([wl.unitary_series(N, Ntrunc, rng) for _ in range(batch)])
        return {"A": A, "B": B}
    if N <= 16:
        A, B = wl.config1_gaussian()
    else:
        A, B = wl.config_product(N, Ntrunc, seed=seed)
    return {"A": A, "B": B}


# ------------------------------------------------------------------------------------ reference arm

def run_reference(args):
    """The oracle as the reference arm: the same program as `cpu_baseline` (one full oracle.series_mul per step), the same
    metric and the same `config.workload` string as the CUDA arm.  Workloads that are not a single product (staple,
    exponential, sweep, batch) fall back to the headline product cfg3."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    import oracle
    name = args.workload if WORKLOADS[args.workload][0] == "product" else "cfg3"
    kind, N, Ntrunc, batch, seed = WORKLOADS[name]
    inp = make_inputs("product", N, Ntrunc, 1, seed)
    A, B = inp["A"], inp["B"]
    for _ in range(args.warmup):
        oracle.series_mul(A, B)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.series_mul(A, B)
    dt = time.perf_counter() - t0
    value = args.steps / dt
    cores = oracle.num_threads()
    sample = f"1 full star-product N={N} N_trunc={Ntrunc} per step (oracle.series_mul, naive O(N_trunc^2))"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "products/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_DESC[name], "N": N, "N_trunc": Ntrunc, "L": transform_length(Ntrunc), "batch": 1},
        "cpu_baseline": {"value": value, "unit": "products/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "products/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def cpu_fftconv(A, B):
    """The paper's own CPU algorithm (FFT-CONV: batched FFT along the order index, one ZGEMM per mode,
    inverse FFT, truncation) with numpy's pocketfft and BLAS -- a second reported CPU baseline next to the naive oracle,
    because the paper's CPU-vs-GPU factor is quoted against FFT-CONV, not against the naive convolution.  Not the oracle
    and not on the product path."""
    n = A.shape[0]
    L = transform_length(n - 1)
    FA = np.fft.ifft(A, n=L, axis=0)          # forward transform with the paper's sign (eq. 2.7), up to a factor L
    FB = np.fft.ifft(B, n=L, axis=0)
    FC = np.matmul(FA, FB)                    # one N x N complex product per mode (eq. 2.8)
    return (np.fft.fft(FC, axis=0) * L)[:n]   # eq. 2.9 and Step 5


# ------------------------------------------------------------------------------------ config 5 sweep

def device_unitary_series(nspt, torch, N, Ntrunc, seed, dev):
    """U = exp(i sum_{k>=1} g^k H_k), H_k Hermitian traceless with E|H_ij|^2 = 1/N (the config-2 recipe), built on
    the device: generators from torch's generator, exponential by the library's own nspt_series_exp.  Used for
    TIMING inputs of the sweep only (the numpy generation costs minutes at N_trunc = 127); the parity of every
    sweep point is tests/test_gpu_parity.py::test_config5_sweep_points_sampled_rows with numpy-generated inputs."""
    g = torch.Generator(device=dev)
    g.manual_seed(int(seed))
    G = torch.randn(Ntrunc + 1, N, N, dtype=torch.complex128, device=dev, generator=g)   # re, im ~ N(0, 1/2)
    H = (G + G.conj().transpose(1, 2)) / (2.0 * N) ** 0.5
    tr = torch.diagonal(H, dim1=1, dim2=2).sum(dim=1) / N
    H = H - tr[:, None, None] * torch.eye(N, dtype=torch.complex128, device=dev)
    X = (1j * H).contiguous()
    X[0] = 0
    return nspt.nspt_series_exp(X)


def run_sweep(args):
    """BASELINE.json configs[4]: time per product over N_trunc in {7..127} at N = 225 and N in {16..400} at
    N_trunc = 31, FFT-CONV on the GPU against the naive O(N_trunc^2) convolution (the oracle, host cores)."""
    import torch
    rank, local, world = dist_env()
    if rank != 0:
        return 0
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    from paper_2001_02835_b200 import build as nspt_build
    nspt_build.build()
    from paper_2001_02835_b200 import binding as nspt
    from paper_2001_02835_b200 import workloads as wl
    stream = torch.cuda.Stream(device=dev)
    nspt.nspt_set_stream(stream.cuda_stream)
    nspt.nspt_set_order_scale(1.0)
    nspt.nspt_set_gemm_variant(args.gemm_variant)
    fp64_peak = probe_fp64_peak(nspt)
    peaks = {}
    pfile = ROOT / "MEASURED_PEAKS.json"
    if pfile.exists():
        try:
            peaks = json.loads(pfile.read_text())
        except Exception:
            peaks = {}
    hbm = peaks.get("hbm_gbs", 6650.0)
    W, K = max(3, args.warmup), args.steps
    # BASELINE.json configs[4] plus the paper's other matrix sizes (Table 3) at N_trunc = 31
    points = sorted(set(wl.sweep_points() + [(225, 31), (121, 31), (169, 31), (289, 31)]), key=lambda p: (p[0] != 225, p[0], p[1]))
    rows_out = []
    launches0 = nspt.nspt_launch_count()
    sampler = ClockSampler(local).start()
    headline = None
    for (N, Ntrunc) in points:
        n, L = Ntrunc + 1, transform_length(Ntrunc)
        per_set = 3 * n * N * N * 16
        R = max(2, int(np.ceil(2 * L2_BYTES / per_set)))
        R = min(R, 64)
        with torch.cuda.stream(stream):
            A0 = device_unitary_series(nspt, torch, N, Ntrunc, 1000 * N + Ntrunc, dev)
            B0 = device_unitary_series(nspt, torch, N, Ntrunc, 1000 * N + Ntrunc + 500, dev)
            sets = [(A0.roll(r, dims=-1).contiguous() if r else A0, B0.roll(r, dims=-2).contiguous() if r else B0,
                     torch.empty_like(A0)) for r in range(R)]
            for i in range(W):
                nspt.nspt_series_mul(*sets[i % R])
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            stream.synchronize()
            ev0.record(stream)
            for i in range(K):
                nspt.nspt_series_mul(*sets[i % R])
            ev1.record(stream)
            stream.synchronize()
            us = ev0.elapsed_time(ev1) / K * 1e3
            nspt.nspt_profile(True)
            for name in nspt.STAGES:
                nspt.nspt_profile_read(name)
            for i in range(K):
                nspt.nspt_series_mul(*sets[i % R])
            st = {name: nspt.nspt_profile_read(name) for name in ("fft_forward", "zgemm_modes", "fft_inverse", "int8_slicing")}
            nspt.nspt_profile(False)
        t_gemm = 8.0 * N ** 3 * L / (fp64_peak * 1e12)
        t_fft = 9.0 * n * N * N * 16 / (hbm * 1e9)
        row = {"N": N, "N_trunc": Ntrunc, "L": L, "us_per_product": us, "products_per_s": 1e6 / us,
               "fft_forward_us": st["fft_forward"][0] / K * 1e3, "zgemm_modes_us": st["zgemm_modes"][0] / K * 1e3,
               "fft_inverse_us": st["fft_inverse"][0] / K * 1e3,
               "int8_slicing_us": st["int8_slicing"][0] / K * 1e3,
               "mode_wise_product": "int8 tensor cores" if st["int8_slicing"][1] else "fp64 tensor pipe",
               "fftconv_roofline_us": max(t_gemm, t_fft) * 1e6, "bound": "fp64" if t_gemm >= t_fft else "hbm",
               "fftconv_roofline_frac": max(t_gemm, t_fft) * 1e6 / us, "buffer_sets": R}
        if not args.no_cpu_baseline:
            import oracle
            A = A0.cpu().numpy()
            B = B0.cpu().numpy()
            # naive O(N_trunc^2) convolution (eq. 2.5) on the host cores: a row sample sized for ~1 s, scaled to a product
            flops = 8.0 * N ** 3 * n * (n + 1) / 2
            nrows = int(max(1, min(N, round(N * 30e9 / flops))))
            rows = np.linspace(0, N - 1, nrows).astype(np.int32)
            t0 = time.perf_counter()
            ref = oracle.series_mul_rows(A, B, rows)
            dt = (time.perf_counter() - t0) * N / nrows
            with torch.cuda.stream(stream):
                C = nspt.nspt_series_mul(A0, B0)
            stream.synchronize()
            got = C[:, torch.from_numpy(rows.astype(np.int64)).to(dev), :].cpu().numpy()
            bound = oracle.product_bound(A, B) * np.sqrt(nrows / N)
            err = (np.sqrt((np.abs(got - ref) ** 2).sum(axis=(1, 2))) / bound).max()
            row.update({"naive_oracle_s_per_product": dt, "naive_rows_sampled": nrows, "cores": oracle.num_threads(),
                        "fftconv_gpu_vs_naive_cpu": dt / (us * 1e-6), "parity_sampled_rows_err_over_bound": float(err)})
        rows_out.append(row)
        if (N, Ntrunc) == (225, 31):
            headline = row
        del sets, A0, B0
        torch.cuda.empty_cache()
    clocks = sampler.stop()
    line = {
        "metric": METRIC, "value": headline["products_per_s"], "unit": "products/s", "n_gpus": 1, "steps": K, "warmup": W,
        "ms_per_step": headline["us_per_product"] * 1e-3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "scaling sweep of A*B (BASELINE.json configs[4]): N_trunc in {7,15,31,63,127} at N=225 and N in "
                               "{16,49,100,225,400} at N_trunc=31, plus the paper's other sizes N in {121,169,289}; value is the shared point N=225, N_trunc=31; timing inputs are "
                               "unitary series generated on the device with nspt_series_exp",
                   "l2": "each point rotates over buffer sets larger than 2 x L2 (up to 64 sets)"},
        "clocks": clocks, "gpu_launches": nspt.nspt_launch_count() - launches0,
        "fp64_peak_tflops": fp64_peak, "hbm_peak_GB_s": hbm, "sweep": rows_out,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------ CUDA arm

def probe_fp64_peak(nspt) -> float:
    """FP64 tensor-pipe peak (TFLOP/s) of this GPU: best of three probe runs a short pause apart, so that a power-capped
    moment right after the timed loops does not lower the denominator (a lower peak would flatter every fraction)."""
    best = 0.0
    for _ in range(3):
        best = max(best, nspt.nspt_probe_fp64_peak())
        time.sleep(0.2)
    return best


def run_cuda(args):
    import torch
    rank, local, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    from paper_2001_02835_b200 import build as nspt_build
    nspt_build.build()
    from paper_2001_02835_b200 import binding as nspt

    kind, N, Ntrunc, batch, seed = WORKLOADS[args.workload]
    L = transform_length(Ntrunc)
    n = Ntrunc + 1
    inp = make_inputs(kind, N, Ntrunc, batch, seed) if kind != "exp" else {}

    stream = torch.cuda.Stream(device=dev)
    nspt.nspt_set_stream(stream.cuda_stream)
    nspt.nspt_set_order_scale(1.0)
    nspt.nspt_set_gemm_variant(args.gemm_variant)

    series_bytes = n * N * N * 16 * batch
    with torch.cuda.stream(stream):
        if kind == "exp":
            # series exponential of an anti-Hermitian series (the link-update exponential)
            per_set = 2 * series_bytes
            R = max(2, int(np.ceil(2 * L2_BYTES / per_set)))
            gen = torch.Generator(device=dev)
            gen.manual_seed(seed)
            sets = []
            for r in range(R):
                G = torch.randn(batch, n, N, N, dtype=torch.complex128, device=dev, generator=gen)
                H = (G + G.conj().transpose(2, 3)) / (2.0 * N) ** 0.5
                X = (1j * H).contiguous()
                X[:, 0] = 0
                if batch == 1:
                    X = X[0].contiguous()
                sets.append((X, torch.empty_like(X)))

            def step(i):
                X, E = sets[i % R]
                if batch == 1:
                    nspt.nspt_series_exp(X, E)
                else:
                    nspt.nspt_series_exp_batched(X, E)
            products_per_step = exp_products(Ntrunc)
            units_name = "exponentials"
        elif kind == "mdstep":
            per_set = 16 * series_bytes
            R = max(2, int(np.ceil(2 * L2_BYTES / per_set)))
            U0 = torch.stack([torch.from_numpy(u) for u in inp["U"]]).to(dev)          # (4, n, N, N)
            sets = []
            for r in range(R):
                Ub = U0.roll(r, dims=-1).contiguous() if r else U0
                sets.append((Ub, [torch.empty_like(Ub[0]) for _ in range(4)], torch.empty_like(Ub), torch.empty_like(Ub)))
            z = inp["z"]
            eps_md, c_md = 0.05, 1.0

            def step(i):
                Ub, S, F, Un = sets[i % R]
                nspt.nspt_staple([Ub[mu] for mu in range(4)], z, S)
                for mu in range(4):
                    nspt.nspt_force(S[mu], c_md, F[mu])
                nspt.nspt_link_update_batched(F, Ub, eps_md, Un)
            products_per_step = 36 + 4 * (exp_products(Ntrunc) + 1)
            units_name = "link_updates"
        elif kind == "staple":
            per_set = 8 * series_bytes
            R = max(2, int(np.ceil(2 * L2_BYTES / per_set)))
            U0 = [torch.from_numpy(u).to(dev) for u in inp["U"]]
            sets = []
            for r in range(R):
                U = [u.roll(r, dims=-1).contiguous() for u in U0] if r else U0
                S = [torch.empty_like(u) for u in U]
                sets.append((U, S))
            z = inp["z"]

            if args.workload == "staple_split":
                from paper_2001_02835_b200 import parallel
                owned = parallel.owned_directions(rank, world if world in (1, 2, 4) else 1)

                def step(i):
                    U, S = sets[i % R]
                    mine = [nspt.nspt_staple_dir(U, z, mu, S[mu]) for mu in owned]
                    if world > 1:
                        with torch.cuda.stream(stream):
                            parallel.all_gather_series(mine, rank, world)
                products_per_step = 15 * len(owned)
            else:
                def step(i):
                    U, S = sets[i % R]
                    nspt.nspt_staple(U, z, S)
                products_per_step = 36
            units_name = "staples"
        else:
            per_set = 3 * series_bytes
            R = max(2, int(np.ceil(2 * L2_BYTES / per_set)))
            A0 = torch.from_numpy(inp["A"]).to(dev)
            B0 = torch.from_numpy(inp["B"]).to(dev)
            sets = []
            for r in range(R):
                A = A0.roll(r, dims=-1).contiguous() if r else A0
                B = B0.roll(r, dims=-2).contiguous() if r else B0
                sets.append((A, B, torch.empty_like(A)))
            if kind == "batched":
                def step(i):
                    A, B, C = sets[i % R]
                    nspt.nspt_series_mul_batched(A, B, C)
            else:
                def step(i):
                    A, B, C = sets[i % R]
                    nspt.nspt_series_mul(A, B, C)
            products_per_step = batch
            units_name = "products"
    stream.synchronize()

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize(dev)

    W, K = max(3, args.warmup), args.steps
    for i in range(W):
        step(i)
    stream.synchronize()

    # ---- timed region 1: K steps, inputs resident in HBM, CUDA events on the library stream
    ev0 = torch.cuda.Event(enable_timing=True)
    ev1 = torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local).start()
    launches0 = nspt.nspt_launch_count()
    barrier()
    ev0.record(stream)
    for i in range(K):
        step(i)
    ev1.record(stream)
    barrier()
    ms_local = ev0.elapsed_time(ev1)
    launches = nspt.nspt_launch_count() - launches0
    clocks = sampler.stop()
    units_per_step = 1 if kind in ("staple", "mdstep") else (batch if kind == "exp" else products_per_step)
    if args.workload == "staple_split":
        units_per_step = 1.0 / world          # the ranks share ONE staple per step (strong scaling)
    value, ms_total = aggregate_throughput(K * units_per_step, ms_local, world, dev)

    # ---- timed region 2: the same K steps with the stage profiler on -> per-kernel durations
    nspt.nspt_profile(True)
    for name in nspt.STAGES:
        nspt.nspt_profile_read(name)
    for i in range(K):
        step(i)
    stage_ms = {}
    for name in nspt.STAGES:
        ms, cnt = nspt.nspt_profile_read(name)
        if cnt:
            stage_ms[name] = {"ms_total": ms, "launches": cnt, "ms_per_launch": ms / cnt}
    nspt.nspt_profile(False)

    # ---- roofline of the dominant kernel (mode-wise matrix product)
    line_extra = {}
    if rank == 0:
        fp64_peak = probe_fp64_peak(nspt)
        gemm = stage_ms.get("zgemm_modes")
        flops_per_launch = 8.0 * N ** 3 * L * batch
        # a launch may carry several independent products (staple): flops of all mode-wise products of a step
        # over the summed duration of the step's GEMM launches
        gemm_products_per_step = products_per_step if kind in ("staple", "exp", "mdstep") else 1
        achieved = (gemm_products_per_step * flops_per_launch * K / (gemm["ms_total"] * 1e-3) * 1e-12) if gemm else None
        traffic = read_traffic(args.workload, "zgemm_modes")
        peaks = {}
        pfile = ROOT / "MEASURED_PEAKS.json"
        if pfile.exists():
            try:
                peaks = json.loads(pfile.read_text())
            except Exception:
                peaks = {}
        hbm = peaks.get("hbm_gbs", 6650.0)
        hbm_src = "MEASURED_PEAKS.json" if "hbm_gbs" in peaks else "fallback 6.65 TB/s"
        e_bytes = N * N * 16
        if kind == "staple":
            retrunc_spectra = 18          # W, Y (12) and T (6): two launches
        elif kind == "exp":
            s_ps = 1
            while s_ps * s_ps < Ntrunc + 1:
                s_ps += 1
            r_ps = (Ntrunc + 1 + s_ps - 1) // s_ps
            retrunc_spectra = ((s_ps - 1) + max(r_ps - 2, 0)) * batch if Ntrunc >= 6 else max(Ntrunc - 2, 0) * batch
            poly_bytes = (s_ps - 1 + r_ps) * L * e_bytes * batch     # reads X^1..X^(s-1), writes B_0..B_(r-1)
        else:
            retrunc_spectra = 0
        fwd_ops = {"exp": 1, "staple": 4}.get(kind, 2)               # operands transformed per step
        inv_ops = 4 if kind == "staple" else 1
        fft_step_bytes = {  # algorithmic bytes per STEP: all launches of a stage together
            "fft_forward": fwd_ops * (n + L) * e_bytes * batch,       # per operand: read n*e, write L*e
            "fft_inverse": inv_ops * (L + n) * e_bytes * batch,
            "fft_retruncate": 2 * L * e_bytes * retrunc_spectra,      # per spectrum: read L*e, write L*e
        }
        if kind == "exp" and Ntrunc >= 6:
            fft_step_bytes["freq_block_polys"] = poly_bytes
        if kind == "mdstep":
            fft_step_bytes = {}       # a mix of the staple's and the exponentials' launches: per-stage bytes are in those workloads' lines
        stages_out = {}
        for name, st in stage_ms.items():
            o = {"launches_per_step": st["launches"] / K, "us_per_launch": st["ms_per_launch"] * 1e3}
            if name in fft_step_bytes and st["ms_total"] > 0:
                gbs = fft_step_bytes[name] * K / (st["ms_total"] * 1e-3) * 1e-9
                o.update({"algorithmic_bytes_per_step": fft_step_bytes[name], "algorithmic_GB_s": gbs, "frac_of_hbm_peak": gbs / hbm})
            stages_out[name] = o
        t_gemm_roof = flops_per_launch / (fp64_peak * 1e12)
        t_fft_roof = 9.0 * n * N * N * 16 * batch / (hbm * 1e9)
        roof_time = max(t_gemm_roof, t_fft_roof)
        int8_path = "int8_slicing" in stage_ms      # the library chose (or was told to use) the INT8 tensor-core product
        if int8_path and gemm:
            # the dominant kernel is a contraction in INT8: 28 slice pairs x 3 planes of N^3 multiply-adds per mode, against
            # the INT8 peak = measured dense bf16 peak x the nominal ratio 2 (B200_PROFILING.md); beside it the FP64 work it stands for
            int8_ops = 84 * 2.0 * N ** 3 * L * batch * gemm_products_per_step   # all mode-wise products of a step
            bf16 = peaks.get("bf16_tflops", 1630.0)
            int8_peak = 2.0 * bf16
            ach_i8 = int8_ops * K / (gemm["ms_total"] * 1e-3) * 1e-12
            k_chunks = N // 32 if (N >= 64 and 0 < N % 32 <= 2) else -(-N // 32)
            padded_ratio = (-(-N // 128) * 128) * (-(-N // 64) * 64) * (k_chunks * 32) / float(N) ** 3
            traffic = read_traffic(args.workload, "zgemm_modes_i8")
            line_extra["roofline"] = {
                "bound": "tensor", "kernel": "zgemm_modes_i8_kernel (tcgen05.mma.kind::i8, TMEM accumulators; FP64 product emulated with 7 int8 slices per plane)",
                "achieved": ach_i8, "peak": int8_peak, "unit": "TOP/s", "frac": ach_i8 / int8_peak, "traffic": traffic,
                # what the tensor cores execute: tiles of 128 (j) x 64 (i) x 32 (k), K without the columns the FP64 tail takes
                "achieved_executed": ach_i8 * padded_ratio, "frac_executed": ach_i8 * padded_ratio / int8_peak,
                "executed_over_algorithmic": padded_ratio,
                "flops_basis": "84 INT8 matrix products (28 slice pairs x 3 planes of the 3M complex product) of 2*N^3 ops per mode; tiles are padded to 128 x 64 x 32, the executed count is higher",
                "peak_source": ("MEASURED_PEAKS.json bf16_tflops (burst) x 2 (nominal INT8 : bf16 ratio, B200_PROFILING.md)" if "bf16_tflops" in peaks
                                else "fallback 1630 TFLOP/s bf16 x 2"),
                "fp64_equivalent": {"achieved": achieved, "unit": "TFLOP/s", "basis": "conventional 8*N^3*L", "fp64_tensor_peak": fp64_peak,
                                    "ratio_to_fp64_tensor_peak": (achieved / fp64_peak) if achieved else None},
                "hbm_peak_GB_s": hbm, "hbm_peak_source": hbm_src,
            }
            if kind == "staple":
                # 8 + 12 + 6 spectra are cut per staple: 18 of them into both layouts (read 16, write 2 x 21 bytes per element), 8 into one
                fft_step_bytes["int8_slicing"] = (18 * (16 + 42) + 8 * (16 + 21)) * L * N * N
            elif kind == "exp":
                # the powers in the layouts the products read them in (left factors of the doubling waves X^1, X^2, X^4, ...;
                # right factors X^1..X^cnt of each wave and X^s), the r-1 Horner left factors, one max pass over B_{r-1}
                lf, rt, h = set(), {s_ps}, 1
                while h < s_ps:
                    cnt = min(s_ps - h, h)
                    lf.add(h)
                    rt.update(range(1, cnt + 1))
                    h += cnt
                fft_step_bytes["int8_slicing"] = (len(lf & rt) * (16 + 42) + len(lf ^ rt) * (16 + 21) + (r_ps - 1) * (16 + 21) + 16) * L * N * N * batch
            elif kind != "mdstep":
                fft_step_bytes["int8_slicing"] = 2 * (16 + 21) * L * N * N * batch   # per operand: read L*e, write 21 bytes per element
            if "int8_slicing" in fft_step_bytes and "int8_slicing" in stages_out and stage_ms["int8_slicing"]["ms_total"] > 0:
                gbs = fft_step_bytes["int8_slicing"] * K / (stage_ms["int8_slicing"]["ms_total"] * 1e-3) * 1e-9
                stages_out["int8_slicing"].update({"algorithmic_bytes_per_step": fft_step_bytes["int8_slicing"], "algorithmic_GB_s": gbs,
                                                   "frac_of_hbm_peak": gbs / hbm})
        else:
          line_extra["roofline"] = {
            "bound": "tensor", "kernel": "zgemm_modes_dmma_kernel (FP64 tensor pipe, DMMA.8x8x4)",
            "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s",
            "frac": (achieved / fp64_peak) if achieved else None, "traffic": traffic,
            "flops_basis": "conventional 8*N^3*L per mode-wise product (all products of a step / summed GEMM launch time); the kernel executes 6*N^3*L (3-multiplication complex product)",
            "achieved_executed": (achieved * 0.75) if achieved else None,
            "frac_executed": (achieved * 0.75 / fp64_peak) if achieved else None,
            "peak_source": "nspt_probe_fp64_peak: DMMA m8n8k4 chain, best of 3 in this run (MEASURED_PEAKS.json has no FP64 entry)",
            "hbm_peak_GB_s": hbm, "hbm_peak_source": hbm_src,
          }
        if kind == "exp":
            step_s = ms_local / K * 1e-3
            line_extra["exp_roofline"] = {
                "definition": "the (s-1)+(r-1) mode-wise products of the Paterson-Stockmeyer form of sum_m X^m/m! (s = ceil(sqrt(N_trunc+1)); the Horner form needs N_trunc-1) of 8*N^3*L flops each at FP64 peak",
                "products_horner": max(Ntrunc - 1, 0),
                "t_roof_ms": products_per_step * t_gemm_roof * 1e3, "products_executed": products_per_step,
                "frac": products_per_step * t_gemm_roof / step_s if step_s else None,
            }
        elif kind == "mdstep":
            step_s = ms_local / K * 1e-3
            line_extra["mdstep_roofline"] = {
                "definition": "the 36 + 4 x 11 mode-wise products of the step (staple; four Paterson-Stockmeyer exponentials and their products with U) of 8*N^3*L flops each at FP64 peak",
                "t_roof_ms": products_per_step * t_gemm_roof * 1e3, "products_executed": products_per_step,
                "frac": products_per_step * t_gemm_roof / step_s if step_s else None,
            }
        elif kind != "staple":
            step_s = ms_local / K * 1e-3
            line_extra["fftconv_roofline"] = {
                "definition": "slower of 8*N^3*L flops at FP64 peak and 9*n*16*N^2 bytes at HBM peak (SURVEY.md 8d)",
                "roofline_products_per_s": batch / roof_time, "t_gemm_us": t_gemm_roof * 1e6, "t_fft_us": t_fft_roof * 1e6,
                "frac": roof_time / step_s if step_s else None,
                "mode_wise_product": ("INT8 tensor cores (FP64 emulated by exact integer slices): the FP64-peak bound above does not bind this path"
                                      if int8_path else "FP64 tensor pipe"),
                # the kernel executes the 3-multiplication product (6*N^3*L), for which 8*N^3*L / peak is NOT a lower bound:
                # the same fraction against the bound of the arithmetic actually executed, transforms not overlapped
                "frac_vs_3m_bound": (0.75 * t_gemm_roof + t_fft_roof) / step_s if step_s else None,
                "t_3m_bound_us": (0.75 * t_gemm_roof + t_fft_roof) * 1e6,
            }
        else:
            step_s = ms_local / K * 1e-3
            line_extra["staple_roofline"] = {
                "definition": "36 mode-wise products (the fewest this organisation of eq. 2.3 needs; literal form: 52) of 8*N^3*L flops each at FP64 peak (SURVEY.md 8d)",
                "roofline_staples_per_s": 1.0 / (36 * t_gemm_roof), "t_roof_ms": 36 * t_gemm_roof * 1e3,
                "products_executed": products_per_step, "frac": 36 * t_gemm_roof / step_s if step_s else None,
            }
        line_extra["stages"] = stages_out

    # ---- e2e: host buffers through the C ABI, H2D and D2H inside the timed region
    e2e = None
    if kind in ("product", "batched"):
        hA = torch.from_numpy(inp["A"]).pin_memory()
        hB = torch.from_numpy(inp["B"]).pin_memory()
        hC = torch.empty_like(hA).pin_memory()
        call = nspt.nspt_series_mul_batched_host if kind == "batched" else nspt.nspt_series_mul_host
        Ke = max(3, min(K, 20))
        for _ in range(2):
            call(hA, hB, hC)
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            call(hA, hB, hC)          # synchronous: returns after the D2H copy
        torch.cuda.synchronize(dev)
        dt_ms = (time.perf_counter() - t0) * 1e3
        e2e_value, _ = aggregate_throughput(Ke * products_per_step, dt_ms, world, dev)
        e2e = {"value": e2e_value, "unit": f"{units_name}/s", "h2d_bytes_per_step": 2 * series_bytes,
               "d2h_bytes_per_step": series_bytes, "steps": Ke,
               "how": ("nspt_series_mul_batched_host" if kind == "batched" else "nspt_series_mul_host") +
                      " with pinned host buffers; wall clock around synchronous calls"}
    elif kind == "staple":
        hU = [torch.from_numpy(u).pin_memory() for u in inp["U"]]
        hS = [torch.empty_like(u).pin_memory() for u in hU]
        Ke = max(2, min(K, 5))
        nspt.nspt_staple_host(hU, z, hS)
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            nspt.nspt_staple_host(hU, z, hS)
        torch.cuda.synchronize(dev)
        dt_ms = (time.perf_counter() - t0) * 1e3
        e2e_value, _ = aggregate_throughput(Ke, dt_ms, world, dev)
        e2e = {"value": e2e_value, "unit": "staples/s", "h2d_bytes_per_step": 4 * series_bytes,
               "d2h_bytes_per_step": 4 * series_bytes, "steps": Ke,
               "how": "nspt_staple_host with pinned host buffers; wall clock around synchronous calls"}
    elif kind in ("exp", "mdstep") and args.workload != "staple_split":
        # no _host entry point for these: the caller's own sequence -- pinned host buffers, copies on the library stream
        # around the device-pointer calls, one stream synchronisation per step
        d_in, d_out = (sets[0][0], sets[0][1]) if kind == "exp" else (sets[0][0], sets[0][3])
        h_in = d_in.cpu().pin_memory()
        h_out = torch.empty_like(h_in).pin_memory()

        def e2e_step():
            with torch.cuda.stream(stream):
                d_in.copy_(h_in, non_blocking=True)
                step(0)
                h_out.copy_(d_out, non_blocking=True)
            stream.synchronize()
        Ke = max(2, min(K, 5))
        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            e2e_step()
        dt_ms = (time.perf_counter() - t0) * 1e3
        e2e_value, _ = aggregate_throughput(Ke * units_per_step, dt_ms, world, dev)
        nbytes = h_in.numel() * 16
        e2e = {"value": e2e_value, "unit": f"{units_name}/s", "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes, "steps": Ke,
               "how": "pinned host buffers copied on the library stream around the device-pointer calls of the step "
                      "(no _host form of these entry points); wall clock, one stream synchronisation per step"}

    # ---- CPU baseline: the oracle on this box's cores (rank 0, single-GPU runs only)
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        if kind in ("exp", "mdstep"):
            # the oracle's exponential is the Horner form of the Taylor sum: N_trunc - 1 star-products (oracle.series_exp);
            # the step's CPU cost is estimated from ONE timed oracle product of the same shape
            X1 = (sets[0][0][0] if (kind == "mdstep" or batch > 1) else sets[0][0]).cpu().numpy()
            t0 = time.perf_counter()
            oracle.series_mul(X1, X1)
            dt = time.perf_counter() - t0
            horner = max(Ntrunc - 1, 1)
            nprod = horner * batch if kind == "exp" else 52 + 4 * (horner + 1)
            cpu_baseline = {"value": (batch if kind == "exp" else 1) / (nprod * dt), "unit": f"{units_name}/s",
                            "cores": oracle.num_threads(), "kind": "oracle",
                            "sample": f"1 star-product N={N} N_trunc={Ntrunc} (oracle.series_mul), scaled by the {nprod} products of the "
                                      + ("oracle's Horner exponential(s)" if kind == "exp" else
                                         "literal staple (52) and of four Horner exponentials times U")}
        elif kind == "staple":
            # one of the 52 products of the literal staple, scaled
            t0 = time.perf_counter()
            oracle.series_mul(inp["U"][0], inp["U"][1])
            dt = time.perf_counter() - t0
            cpu_baseline = {"value": 1.0 / (52 * dt), "unit": "staples/s", "cores": oracle.num_threads(), "kind": "oracle",
                            "sample": "1 of the 52 star-products of the literal staple (oracle.series_mul), scaled by 52"}
        else:
            A = inp["A"] if kind == "product" else inp["A"][0]
            B = inp["B"] if kind == "product" else inp["B"][0]
            t0 = time.perf_counter()
            ref = oracle.series_mul(A, B)
            dt = time.perf_counter() - t0
            cpu_baseline = {"value": 1.0 / dt, "unit": "products/s", "cores": oracle.num_threads(), "kind": "oracle",
                            "sample": f"1 full star-product N={N} N_trunc={Ntrunc} (oracle.series_mul, naive O(N_trunc^2))"}
            # the paper's own CPU algorithm (FFT-CONV with library FFT + ZGEMM), same inputs, reported beside the oracle
            t0 = time.perf_counter()
            cpu_fftconv(A, B)
            dt2 = time.perf_counter() - t0
            line_extra["cpu_fftconv_baseline"] = {
                "value": 1.0 / dt2, "unit": "products/s", "kind": "numpy pocketfft + BLAS zgemm per mode (PAPER.md:68-102, Table 2)",
                "note": "the paper's CPU-vs-GPU factor 9 is against its CPU FFT-CONV; numpy uses the BLAS threads of this box"}
            # parity check of the timed call on the timed buffers: the same entry point, every element of a batch
            with torch.cuda.stream(stream):
                step(0)
            stream.synchronize()
            got = sets[0][2].cpu().numpy()
            if kind == "product":
                err = oracle.per_order_error(got, ref, oracle.product_bound(A, B)).max()
            else:
                err = 0.0
                for b in range(batch):
                    rb = ref if b == 0 else oracle.series_mul(inp["A"][b], inp["B"][b])
                    err = max(err, oracle.per_order_error(got[b], rb, oracle.product_bound(inp["A"][b], inp["B"][b])).max())
            line_extra["parity_max_err_over_bound"] = float(err)
            line_extra["parity_checked"] = ("nspt_series_mul_batched, all %d elements" % batch) if kind == "batched" else "nspt_series_mul"

    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return 0

    desc = WORKLOAD_DESC[args.workload]
    line = {
        "metric": {"staple": "tek_staples_per_sec", "exp": "series_exponentials_per_sec", "mdstep": "tek_link_updates_per_sec"}.get(kind, METRIC),
        "value": value, "unit": f"{units_name}/s", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "strong" if args.workload == "staple_split" else "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "N": N, "N_trunc": Ntrunc, "L": L, "batch": batch,
                   "parallelism": "replicas only (no data-path collective)" if world > 1 else "single GPU",
                   "l2": f"inputs rotate over {R} buffer sets, {R * per_set / 1e6:.0f} MB total > 2 x L2 (126 MB)"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
    }
    line.update(line_extra)
    if "i8" in line.get("roofline", {}).get("kernel", ""):
        line["dtype_detail"] = ("transforms, slicing and recombination in f64; the mode-wise product in exact integer arithmetic "
                                "(int8 slices, int32 tensor-core accumulators) that reproduces the f64 product to 2^-50")
    if cpu_baseline is not None:
        line["cpu_baseline"] = cpu_baseline
    print(json.dumps(line))
    return 0


def replica_env(rank: int, world: int, port: int) -> dict:
    """Environment of replica `rank` when bench.py spawns its own ranks (no torchrun): one process per GPU."""
    env = dict(os.environ)
    env.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": str(world), "MASTER_ADDR": "127.0.0.1",
                "MASTER_PORT": str(port)})
    return env


def spawn_replicas(n: int, argv) -> int:
    """`python bench.py --gpus N` outside torchrun: start the N replica processes (one per GPU, rank = local rank = GPU
    index), let rank 0's JSON line through and return the worst exit code."""
    import socket
    import subprocess
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
    procs = [subprocess.Popen([sys.executable, str(Path(__file__).resolve()), *argv], env=replica_env(r, n, port),
                              stdout=None if r == 0 else subprocess.DEVNULL) for r in range(n)]
    return max(p.wait() for p in procs)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--gemm-variant", type=int, default=-1, choices=[-1, 1, 2, 3, 4],
                    help="mode-wise product kernel (include/nspt_debug.h): -1 = the library's automatic choice (default), 1 = FP64 tensor pipe "
                         "(DMMA), 2 = INT8 tensor cores (tcgen05, Ozaki slicing), 3 = persistent DMMA, 4 = INT8 on CTA pairs")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference":
        return spawn_replicas(args.gpus, sys.argv[1:])
    if args.impl == "reference":
        args.steps = args.steps if args.steps is not None else 5
        args.warmup = args.warmup if args.warmup is not None else 1
        return run_reference(args)
    if args.workload == "sweep":
        args.steps = args.steps if args.steps is not None else 50
        args.warmup = args.warmup if args.warmup is not None else 3
        return run_sweep(args)
    args.steps = args.steps if args.steps is not None else (200 if args.workload not in ("staple", "staple_split", "mdstep", "exp", "exp4") else 10)
    args.warmup = args.warmup if args.warmup is not None else 5
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
