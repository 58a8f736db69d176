#!/usr/bin/env python
"""bench.py — throughput of the PWA likelihood hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

Workload (default cfg4 = BASELINE.json configs[4], the largest config and the one the
north_star's HBM target is stated on): n = 64 waves, N_data = 5e6 events, fp32 amplitude storage
(2.56 GB, >> the 126 MB L2, so nothing is cache-resident between steps), fp64 arithmetic.
A STEP is one lnL + gradient evaluation at a fresh random V over all data events of the rank:
steps A2-A5 + A7 of DESIGN.md section 2 (one pass over the amplitude matrix in HBM); with
N > 1 ranks the events are sharded (weak scaling: every rank holds a full cfg-sized shard) and
the step adds the rank-ordered sum of the (2 + 2n)-double data-term record.  The normalisation
matrix M (step A6) is built once per fit at constant resonances and is
therefore outside the step; its build, the batched K-start path (A8) and the floating-resonance
iteration (A1, cfg3) are timed separately and reported under "extra" on the same JSON line.

value = event-waves/s = (events x waves evaluated by all ranks) / time, device-timed with CUDA
events on the library's stream, max over ranks.  e2e = the same through the synchronous C-ABI
call pwa_nll_grad with HOST V in and HOST results out (wall clock).

--impl reference times the CPU oracle (oracle/, test infrastructure) on the box's host cores on
a bounded sample of the same workload; it is a deliberately plain program, reported as context.
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

import numpy as np  # noqa: E402

WORKLOADS = {"cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg0": 0}
SAMPLE_TARGET_S = 0.6          # reference arm: aim for this much oracle time per step


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=sorted(WORKLOADS))
    ap.add_argument("--no-extra", action="store_true", help="skip the M-build / batched / cfg3 side measurements")
    ap.add_argument("--n-data", type=int, default=0, help="override N_data (debugging only; makes the line invalid)")
    ap.add_argument("--n-mc", type=int, default=0, help="override N_MC accepted (debugging only)")
    return ap.parse_args()


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)", d
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)", {}


def load_traffic(kernel_key):
    """dram bytes per launch of the dominant kernel from the committed ncu capture
    (profiles/traffic.csv: key,dram_bytes_per_launch,source) or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None
    for line in open(p):
        f = line.strip().split(",")
        if len(f) >= 2 and f[0] == kernel_key:
            try:
                return float(f[1])
            except ValueError:
                return None
    return None


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    BAD = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown"}
    NOTE = {0x4: "sw_power_cap", 0x80: "hw_power_brake", 0x2: "applications_clocks_setting"}

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz, self.ok = [], set(), None, False
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def _once(self):
        nv = self.nv
        self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
        try:
            r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
        except Exception:
            r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
        for bit, name in list(self.BAD.items()) + list(self.NOTE.items()):
            if r & bit:
                self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._once()
            except Exception:
                pass
            self._stop.wait(0.02)

    def start(self):
        if self.ok:
            self._stop.clear()
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr:
            self._stop.set()
            self._thr.join()
            self._thr = None

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    ws = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, ws, local


def sizes_for(args, spec):
    n_data = args.n_data or spec["n_data"]
    n_mc = args.n_mc or spec["n_mc"]
    return int(n_data), int(n_mc)


def workload_config(workload, n, n_data, storage, ws, backend):
    """The `config` object of the JSON line: the same for our arm and for the reference arm (which times the oracle on a
    bounded sample of exactly this workload)."""
    bytes_data = n_data * n * 2 * (8 if storage == "f64" else 4)
    return {"workload": workload, "n_waves": n, "n_data_per_gpu": n_data, "storage": storage,
            "parallelism": (f"event-sharded x{ws}" + ("" if backend == "nccl" else f" ({backend} exchange, test mode)")) if ws > 1 else "single GPU",
            "l2": f"input {bytes_data / 1e6:.0f} MB per step vs 126 MB L2: "
                  + ("larger than L2, no flush needed" if bytes_data > 2.5e8 else "L2-RESIDENT (latency-bound config)")}


# --------------------------------------------------------------------------- reference arm
def oracle_sample_size(oracle, A, M, V, n_total, target_s):
    """Largest prefix of the data whose oracle evaluation takes about target_s seconds."""
    probe = min(n_total, 20_000)
    oracle.nll_grad(A[:probe], M, V)                     # page in / warm up threads
    t0 = time.perf_counter()
    oracle.nll_grad(A[:probe], M, V)
    dt = max(time.perf_counter() - t0, 1e-6)
    s = int(probe * target_s / dt)
    return max(1000, min(n_total, s))


def small_oracle_norm(synth, oracle, cfg, n_mc=50_000):
    wm = synth.make_workload(cfg, n_data=1, n_mc=n_mc, want_data=False)
    A_mc = wm.A_mc
    if A_mc is None:   # factored config
        A_mc = synth.amplitudes(wm, wm.kin_mc)
    return oracle.norm_matrix(A_mc, wm.n_gen)


def run_reference(args):
    rank, ws, _ = dist_env()
    if rank != 0:
        return 0
    from oracle import oracle
    from paper_1108_5882_b200.inputs import synth
    cfg = WORKLOADS[args.workload]
    spec = synth._CFG[cfg]
    n_data, _ = sizes_for(args, spec)
    K, W = args.steps, args.warmup
    target = min(SAMPLE_TARGET_S, 150.0 / max(1, K + W))
    # generate a bounded prefix of the data sample (the generator is sequential in candidate
    # order, so the first S accepted events of the full workload are exactly these)
    cap = min(n_data, 400_000)
    w = synth.make_workload(cfg, n_data=cap, n_mc=1, want_mc=False)
    A = w.A_data if w.A_data is not None else synth.amplitudes(w, w.kin_data)
    M = small_oracle_norm(synth, oracle, cfg)
    Vs = synth.eval_points(w, K + W)
    S = oracle_sample_size(oracle, A, M, Vs[0], cap, target)
    A = np.ascontiguousarray(A[:S])
    for i in range(W):
        oracle.nll_grad(A, M, Vs[i])
    t0 = time.perf_counter()
    for i in range(K):
        oracle.nll_grad(A, M, Vs[W + i])
    dt = time.perf_counter() - t0
    value = S * w.n * K / dt
    sample = f"first {S} of {n_data} data events of {args.workload} (n={w.n}, {w.storage} storage), full lnL+gradient per step"
    line = {
        "impl": "reference", "metric": "event-waves/s (lnL+gradient evaluation)", "value": value,
        "unit": "event-waves/s", "n_gpus": args.gpus, "steps": K, "warmup": W,
        "ms_per_step": dt / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": workload_config(args.workload, w.n, n_data, w.storage, ws, os.environ.get("PWA_BENCH_BACKEND", "nccl")),   # our arm's config
        "sample_events": S,
        "evals_per_s": K / dt * (S / n_data),
        "cpu_baseline": {"value": value, "unit": "event-waves/s", "cores": oracle.threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": "event-waves/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------- our arm
class Timer:
    """CUDA-event timing on torch's current stream (the stream every pwa context here uses)."""

    def __init__(self, torch):
        self.torch = torch

    def run(self, fn, steps, warmup, barrier=None):
        torch = self.torch
        for i in range(warmup):
            fn(i)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        if barrier:
            barrier()
            torch.cuda.synchronize()
        t0 = time.perf_counter()
        e0.record()
        for i in range(steps):
            fn(warmup + i)
        e1.record()
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        if barrier:
            barrier()
        return e0.elapsed_time(e1) / steps, wall / steps * 1e3      # ms per step (device, wall)


SIDE_STEPS, SIDE_WARMUP = 10, 3      # every side measurement: >= 10 timed steps after 3 warm-ups


def measure_peaks(pwa, ctx, mp_hbm, mp_src):
    """Roofline denominators.  HBM: MEASURED_PEAKS.json (driver-written copy bandwidth).  FP64: MEASURED_PEAKS has
    no fp64 figure, so the register-resident DFMA and mma.sync.m8n8k4.f64 loops of pwa_microbench are run here
    (SURVEY 8(d) "Denominators").  int8 tensor: pwa_microbench(3), a loop of tcgen05.mma.kind::i8 M = 128, N = 256, K = 32
    with both operands in shared memory on every SM (nominal dense int8: 4.5 Pop/s)."""
    return {"hbm_gbs": mp_hbm, "hbm_source": mp_src,
            "dfma_tflops": pwa.pwa_microbench(ctx, 0), "dmma_tflops": pwa.pwa_microbench(ctx, 1),
            "hbm_read_gbs": pwa.pwa_microbench(ctx, 2, 4 << 30),
            "fp64_source": "measured here: pwa_microbench(0 | 1), register-resident loops, best of 5",
            "hbm_read_source": "measured here: pwa_microbench(2), read-only stream over 4 GiB",
            "int8_tops": pwa.pwa_microbench(ctx, 3), "int8_tops_n128": pwa.pwa_microbench(ctx, 4),
            "int8_tops_n64": pwa.pwa_microbench(ctx, 5), "tmem_read_gbs": pwa.pwa_microbench(ctx, 7),
            "int8_source": "measured here: pwa_microbench(3 | 4 | 5), tcgen05.mma.kind::i8 from shared memory, all SMs",
            "int8_tops_nominal": 4500.0,
            "tensor_overlap_ms": overlap_probe(pwa, ctx)}


def overlap_probe(pwa, ctx):
    """pwa_microbench(8): a stream of int8 tcgen05.mma next to 12 warps of one kind of epilogue work (the issuer's scheduler
    kept free).  overlap = (t_mma + t_work - t_both) / min(t_mma, t_work): 1 = the work hides under the MMAs, 0 = serial.
    fp64 arithmetic comes out at 0 (why the batched int8 kernel cannot hide its epilogue)."""
    out = {"mma_alone": pwa.pwa_microbench(ctx, 8, 16)}
    for mode, name in ((0, "fp64_fma"), (6, "fp64_diluted_1_in_4"), (5, "fp32_fma"), (3, "int_mad"), (1, "tcgen05_ld"), (2, "st_shared")):
        alone = pwa.pwa_microbench(ctx, 8, mode + 32 + 64)
        both = pwa.pwa_microbench(ctx, 8, mode + 48 + 64)
        out[name] = {"alone": alone, "with_mma": both, "overlap": (out["mma_alone"] + alone - both) / min(out["mma_alone"], alone)}
    # window mode: one fp64 window and one integer window, in either order (who waits for whom)
    for flag, name in ((0, "windows_fp64_first"), (128, "windows_int_first")):
        alone = pwa.pwa_microbench(ctx, 8, 8 + 32 + 64 + flag + (8192 << 8))
        both = pwa.pwa_microbench(ctx, 8, 8 + 48 + 64 + flag + (8192 << 8))
        out[name] = {"alone": alone, "with_mma": both, "added": both - alone}
    return out


def rl_hbm(peaks, nbytes, ms, **kw):
    a = nbytes / ms * 1e-6
    r = {"bound": "hbm", "achieved": a, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": a / peaks["hbm_gbs"],
         "peak_source": peaks["hbm_source"], "algorithmic_bytes_per_launch": nbytes}
    r.update(kw)
    return r


def rl_flops(peaks, bound, flops, ms, **kw):
    """bound: 'tensor' (fp64 DMMA), 'alu' (fp64 FMA) or 'tensor_int8' (nominal peak)."""
    a = flops / ms * 1e-9
    if bound == "tensor":
        peak, src, unit = peaks["dmma_tflops"], peaks["fp64_source"], "TFLOP/s"
    elif bound == "alu":
        peak, src, unit = peaks["dfma_tflops"], peaks["fp64_source"], "TFLOP/s"
    else:
        peak, src, unit = peaks["int8_tops"], peaks["int8_source"], "Top/s"
    r = {"bound": bound.split("_")[0], "achieved": a, "peak": peak, "unit": unit, "frac": a / peak, "peak_source": src,
         "algorithmic_flops_per_launch": flops}
    r.update(kw)
    return r


def upload_constant(pwa, ctx, w):
    t0 = time.perf_counter()
    pwa.pwa_upload_events(ctx, pwa.PWA_DATA, w.A_data)
    pwa.pwa_sync(ctx)
    return time.perf_counter() - t0


def upload_mc(torch, pwa, tm, ctx, w):
    """Uploads the MC sample; -> device time (ms) of what an MC upload does besides the copy: for fp32 storage the column
    maxima of the int8 path (k_colmax_f32, one read of the sample, once per upload), timed on a borrowed device copy."""
    t_mc = torch.from_numpy(w.A_mc).cuda()
    ms_pre, _ = tm.run(lambda i: pwa.pwa_upload_events(ctx, pwa.PWA_MC, t_mc, n_events=w.n_acc, n_generated=w.n_gen,
                                                       flags=pwa.PWA_BORROW), 3, 1)
    pwa.pwa_upload_events(ctx, pwa.PWA_MC, w.A_mc, n_generated=w.n_gen)
    del t_mc
    return ms_pre


def m_build_record(pwa, tm, ctx, w, n, elem, peaks):
    ms_m, _ = tm.run(lambda i: pwa.pwa_build_norm(ctx, want_M=False), SIDE_STEPS, SIDE_WARMUP)
    bound, path = pwa.pwa_norm_error_bound(ctx)
    nbytes = w.n_acc * n * 2 * elem
    flops_sym = 4.0 * n * n * w.n_acc                       # Hermitian symmetry used: half of the 8 n^2 N full Gram
    rec = {"ms": ms_m, "n_mc": w.n_acc, "gflops_full_gram": 2 * flops_sym / ms_m * 1e-6, "mc_gbs": nbytes / ms_m * 1e-6,
           "path": "int8 tcgen05 (digit planes, int32 TMEM)" if path == 1 else "fp64 DMMA", "error_bound_abs": bound}
    hb = rl_hbm(peaks, nbytes, ms_m, kernel="i8::k_norm_i8" if path == 1 else "k_norm_dmma")
    if path == 1:
        rec["roofline"] = hb                                 # exact integer GEMM keeps up with the stream: HBM-bound
        # opt-in variant with three digit planes ("norm" = 3): faster, larger a-priori bound; measured against the default's M
        M4 = pwa.pwa_build_norm(ctx)
        pwa.pwa_set_option(ctx, "norm", 3)
        ms3, _ = tm.run(lambda i: pwa.pwa_build_norm(ctx, want_M=False), SIDE_STEPS, SIDE_WARMUP)
        M3 = pwa.pwa_build_norm(ctx)
        bound3, _ = pwa.pwa_norm_error_bound(ctx)
        pwa.pwa_set_option(ctx, "norm", 0)
        pwa.pwa_build_norm(ctx, want_M=False)                # leave the default's M in the context
        rec["three_planes"] = {"ms": ms3, "roofline": rl_hbm(peaks, nbytes, ms3, kernel="i8::k_norm_i8<3>"),
                               "error_bound_abs": bound3, "max_abs_M": float(np.abs(M4).max()),
                               "measured_diff_to_default_abs": float(np.abs(M3 - M4).max())}
    else:
        tb = rl_flops(peaks, "tensor", flops_sym, ms_m, kernel="k_norm_dmma")
        rec["roofline"] = hb if hb["frac"] >= tb["frac"] else tb    # the floor that is closer is the binding one
        rec["roofline_other"] = tb if hb["frac"] >= tb["frac"] else hb
    return rec


def bench_constant(torch, pwa, synth, w, steps, warmup, elem, peaks):
    """Single-rank side measurement of a constant-resonance config -> dict."""
    tm = Timer(torch)
    stream = torch.cuda.current_stream().cuda_stream
    ctx = pwa.pwa_create(w.n, w.storage, torch.cuda.current_device(), stream)
    out = {}
    try:
        up_s = upload_constant(pwa, ctx, w)
        n = w.n
        M0 = np.zeros((n, n, 2)); M0[np.arange(n), np.arange(n), 0] = 1.0
        if w.A_mc is not None:
            ms_pre = upload_mc(torch, pwa, tm, ctx, w)
            out["m_build"] = m_build_record(pwa, tm, ctx, w, n, elem, peaks)
            out["m_build"]["upload_prepass_ms"] = ms_pre
            out["m_build"]["upload_prepass_note"] = ("device work of pwa_upload_events(MC) on a borrowed buffer, once per upload: "
                                                     "column maxima for the int8 digit planes (fp32 storage), nothing for fp64")
        else:
            pwa.pwa_set_norm(ctx, M0)
        Vs = synth.eval_points(w, steps + warmup)
        ms, _ = tm.run(lambda i: pwa.pwa_nll_grad_enqueue(ctx, Vs[i]), steps, warmup)
        t0 = time.perf_counter()
        for i in range(steps):
            pwa.pwa_nll_grad(ctx, Vs[warmup + i])
        wall = (time.perf_counter() - t0) / steps * 1e3
        nbytes = w.n_data * n * 2 * elem
        out.update({"n_waves": n, "n_data": w.n_data, "storage": w.storage, "evaluations_timed": steps, "ms_per_eval": ms,
                    "evals_per_s": 1e3 / ms, "event_waves_per_s": w.n_data * n / ms * 1e3,
                    "e2e_ms_per_eval": wall, "e2e_evals_per_s": 1e3 / wall, "upload_s": up_s})
        if nbytes < 100e6:
            # latency-bound sample: the same evaluations through the resident grid (no launch per evaluation)
            pwa.pwa_set_option(ctx, "resident", 1)
            try:
                for i in range(warmup):
                    pwa.pwa_nll_grad(ctx, Vs[i])
                t0 = time.perf_counter()
                for i in range(steps):
                    pwa.pwa_nll_grad(ctx, Vs[warmup + i])
                wall_r = (time.perf_counter() - t0) / steps * 1e3
                out["resident"] = {"e2e_ms_per_eval": wall_r, "e2e_evals_per_s": 1e3 / wall_r,
                                   "note": "pwa_set_option('resident', 1): host V in, host record out, through the binding"}
                # what a fit sees: the host BFGS driver on this sample, evaluations by launches and through the resident grid
                if w.A_mc is not None:
                    V0 = synth.eval_points(w, 1, stream=synth.S_START)[0]
                    fit = {}
                    for mode, key in ((0, "launched"), (1, "resident")):
                        pwa.pwa_set_option(ctx, "resident", mode)
                        t0 = time.perf_counter()
                        _, nll_f, ev, _, it = pwa.pwa_minimize_bfgs(ctx, V0, max_iter=100, gtol=0.0, want_iters=True)
                        dt = time.perf_counter() - t0
                        fit[key] = {"iterations": it, "evaluations": ev, "wall_ms": dt * 1e3, "us_per_evaluation": dt / max(ev, 1) * 1e6,
                                    "nll": nll_f}
                    out["resident"]["bfgs_100_iterations"] = fit
            except pwa.PwaError as e:       # e.g. under a profiler that makes launches synchronous: the grid never sees a command
                out["resident"] = {"unavailable": str(e)}
            pwa.pwa_set_option(ctx, "resident", 0)
            out["roofline"] = {"bound": "latency", "achieved": nbytes / ms * 1e-6, "peak": None, "unit": "GB/s", "frac": None,
                               "algorithmic_bytes_per_launch": nbytes, "kernel": "k_data_term_tma",
                               "note": "sample is L2-RESIDENT (< 126 MB): launch / reduction latency bound, not an HBM fraction; "
                                       f"the HBM floor would be {nbytes / peaks['hbm_gbs'] * 1e-3:.1f} us"}
        else:
            l2mb = pwa.pwa_get_option(ctx, "l2_resident_mb")
            res_mb = (48 if 64e6 <= nbytes <= (1 << 30) else 0) if l2mb < 0 else l2mb
            out["roofline"] = rl_hbm(peaks, nbytes, ms, kernel="k_data_term_tma")
            if res_mb:
                out["roofline"]["note"] = (f"ALGORITHMIC GB/s: {res_mb} MB of the sample are kept L2-resident between "
                                           "evaluations by cache hints, so DRAM moves less than the algorithmic bytes")
                out["roofline"]["dram_gbs_estimate"] = (nbytes - res_mb * 1e6) / ms * 1e-6
                out["roofline"]["dram_frac_estimate"] = (nbytes - res_mb * 1e6) / ms * 1e-6 / peaks["hbm_gbs"]
        # NEXT-2: Fumili-style approximate Hessian (synchronous call: one row-scaled Gram pass over the data)
        for i in range(SIDE_WARMUP):
            pwa.pwa_fumili_hessian(ctx, Vs[i])
        t0 = time.perf_counter()
        for i in range(SIDE_STEPS):
            pwa.pwa_fumili_hessian(ctx, Vs[(SIDE_WARMUP + i) % len(Vs)])
        ms_f = (time.perf_counter() - t0) / SIDE_STEPS * 1e3
        out["fumili"] = {"ms_per_call_e2e": ms_f,
                         "roofline": rl_flops(peaks, "tensor", 4.0 * n * n * w.n_data + 16.0 * n * w.n_data, ms_f,
                                              kernel="k_norm_dmma (row-scaled, DATA)", timed="synchronous call incl. D2H of H")}
        if w.K > 1:
            Vk = synth.eval_points(w, w.K, stream=synth.S_START)
            ms_b, _ = tm.run(lambda i: pwa.pwa_nll_grad_batch_enqueue(ctx, Vk), SIDE_STEPS, SIDE_WARMUP)
            path, err_rel = pwa.pwa_batch_path(ctx)
            flops = 16.0 * w.n_data * n * w.K
            out["batch"] = {"K": w.K, "ms_per_call": ms_b, "evals_per_s": w.K / ms_b * 1e3,
                            "event_waves_per_s": w.n_data * n * w.K / ms_b * 1e3,
                            "fp64_equivalent_gflops": flops / ms_b * 1e-6,
                            "path": {0: "K streaming passes", 1: "fp64 DMMA chained GEMMs",
                                     2: "int8 tcgen05 chained GEMMs (digit planes, int32 TMEM)"}[path],
                            "per_term_error_estimate": err_rel}
            if path == 2:
                # digit-pair products of 128 x 128 x 128 int8 MACs per 128-event tile (pwa_batch_path documents the count)
                pairs = 20
                ops = 2.0 * 128 * 128 * pairs * w.n_data
                out["batch"]["roofline"] = rl_flops(peaks, "tensor_int8", ops, ms_b, kernel="bi8::k_batch_i8",
                                                    digit_pair_gemms_per_tile=pairs)
                out["batch"]["roofline_hbm"] = rl_hbm(peaks, nbytes, ms_b, kernel="bi8::k_batch_i8")
                pwa.pwa_set_option(ctx, "batch", 1)
                ms_d, _ = tm.run(lambda i: pwa.pwa_nll_grad_batch_enqueue(ctx, Vk), SIDE_STEPS, SIDE_WARMUP)
                pwa.pwa_set_option(ctx, "batch", 0)
                out["batch"]["fp64_dmma"] = {"ms_per_call": ms_d,
                                             "roofline": rl_flops(peaks, "tensor", flops, ms_d, kernel="k_batch_dmma")}
            elif path == 1:
                out["batch"]["roofline"] = rl_flops(peaks, "tensor", flops, ms_b, kernel="k_batch_dmma")
            # NEXT-3: the same evaluation with per-event weights (8 B/event weight stream)
            wts = np.random.default_rng(7).uniform(0.5, 1.5, size=w.n_data)
            pwa.pwa_set_weights(ctx, pwa.PWA_DATA, wts)
            ms_w, _ = tm.run(lambda i: pwa.pwa_nll_grad_enqueue(ctx, Vs[i % len(Vs)]), SIDE_STEPS, SIDE_WARMUP)
            pwa.pwa_set_weights(ctx, pwa.PWA_DATA, None)
            out["weighted"] = {"ms_per_eval": ms_w, "roofline": rl_hbm(peaks, nbytes + 8 * w.n_data, ms_w, kernel="k_data_term_tma<.., WT> (weighted)")}
    finally:
        pwa.pwa_destroy(ctx)
    return out


# algorithmic fp64 flops per event of the fused Breit-Wigner passes at configs[3] (8 resonances x 2 angular structures;
# "flops ~ n_res (complex reciprocal ~ 25) + n 6 + 16 n + 60 ~ 600 / event")
FLOPS_FACT_DATA = 600.0
FLOPS_RES_GRAD = 450.0      # res_grad.cu: one Breit-Wigner per resonance, w BW^2, 8 complex MACs, 1 / S
FLOPS_FACT_RG = 750.0       # fused pass of pwa_nll_grad_floating: the 600 above + Q2[r][s] += BW_r^2 Z_s f (16 complex MACs + 8 BW^2)


def bench_floating(torch, pwa, synth, w, steps, warmup, peaks):
    """cfg3: one evaluation of a floating-resonance fit (value, V gradient, d/dM_r, d/dG_r; reading A9), timed two ways:
    the two-pass call pwa_nll_grad_floating (explicit MC sum: what pwa_minimize_bfgs_floating uses) and, as configs[3]
    words it ("M is rebuilt every iteration"), set_resonances + build_norm (fused BW over MC) + nll_grad + res_grad."""
    tm = Timer(torch)
    stream = torch.cuda.current_stream().cuda_stream
    ctx = pwa.pwa_create(w.n, w.storage, torch.cuda.current_device(), stream)
    try:
        pwa.pwa_upload_events_factored(ctx, pwa.PWA_DATA, w.mass_data, w.Z_data)
        pwa.pwa_upload_events_factored(ctx, pwa.PWA_MC, w.mass_mc, w.Z_mc, n_generated=w.n_gen)
        pwa.pwa_set_wave_map(ctx, w.n_res, w.res_of_wave, w.ang_of_wave)
        Mr0, Gr0 = synth.floating_start(w)
        Vs = synth.eval_points(w, steps + warmup)
        jit = synth.cnormal(w.seed, synth.S_START + 1, steps + warmup)

        def params(i):
            Mr, Gr = Mr0.copy(), Gr0.copy()
            Mr[: w.n_free] *= 1.0 + 1e-3 * jit[i, 0]
            Gr[: w.n_free] *= 1.0 + 1e-3 * jit[i, 1]
            return Mr, Gr

        def it_dev(i):
            Mr, Gr = params(i)
            pwa.pwa_set_resonances(ctx, Mr, Gr)
            pwa.pwa_build_norm(ctx, want_M=False)
            pwa.pwa_nll_grad_enqueue(ctx, Vs[i])

        def it_full(i):
            Mr, Gr = params(i)
            pwa.pwa_set_resonances(ctx, Mr, Gr)
            pwa.pwa_build_norm(ctx, want_M=False)
            pwa.pwa_nll_grad(ctx, Vs[i])
            pwa.pwa_res_grad(ctx, Vs[i])

        def it_two_pass(i):
            Mr, Gr = params(i)
            pwa.pwa_nll_grad_floating(ctx, Vs[i], Mr, Gr)

        def only_norm(i):
            Mr, Gr = params(i)
            pwa.pwa_set_resonances(ctx, Mr, Gr)
            pwa.pwa_build_norm(ctx, want_M=False)

        pwa.pwa_set_resonances(ctx, Mr0, Gr0)
        pwa.pwa_build_norm(ctx, want_M=False)
        ms_data, _ = tm.run(lambda i: pwa.pwa_nll_grad_enqueue(ctx, Vs[i]), steps, warmup)
        ms_it, _ = tm.run(it_dev, steps, warmup)
        ms_norm, _ = tm.run(only_norm, steps, warmup)
        _, wall_full = tm.run(it_full, steps, warmup)
        ms_two, wall_two = tm.run(it_two_pass, steps, warmup)       # synchronous call: device time between events ~ e2e
        ms_rg = max(wall_full - ms_it, 1e-6)
        # configs[3] as stated: 200 quasi-Newton iterations driven from the host, M rebuilt in every evaluation
        free = np.arange(w.n_free, dtype=np.int32)
        pwa.pwa_set_resonances(ctx, Mr0, Gr0)
        t0 = time.perf_counter()
        _, Mf, Gf, nll_f, its, evs, _, why = pwa.pwa_minimize_bfgs_floating_ex(ctx, w.V_true, Mr0, Gr0, free, max_iter=200, gtol=0.0)
        fit_s = time.perf_counter() - t0
        fit = {"max_iter_requested": 200, "iterations_run": its, "evaluations": evs,
               "stopped_because": {0: "converged", 1: "max_iter", 2: "line search exhausted (fp64 resolution of nll)"}[why],
               "wall_s": fit_s, "e2e_ms_per_evaluation": fit_s / max(evs, 1) * 1e3,
               "nll": nll_f, "free_parameters": 2 * w.n + 2 * w.n_free}
        n = w.n
        mc_bytes = w.n_acc * (8 + 16 * w.n_ang)
        data_bytes = w.n_data * (8 + 16 * w.n_ang)
        return {"n_waves": n, "n_data": w.n_data, "n_mc": w.n_acc, "storage": w.storage, "floating_fit": fit,
                "two_pass_evaluation": {"e2e_ms": wall_two, "ms_between_events": ms_two,
                                        "what": "pwa_nll_grad_floating: nll, V gradient, d/dM_r, d/dG_r from one MC pass + one data pass (no M)",
                                        "event_waves_per_s": (w.n_data + w.n_acc) * n / wall_two * 1e3,
                                        "roofline": rl_flops(peaks, "alu", FLOPS_FACT_RG * (w.n_data + w.n_acc), wall_two,
                                                             kernel="k_data_term_fact<.., RG> (MC pass + data pass)",
                                                             timed="synchronous call, host V / parameters in, host results out",
                                                             hbm_frac=(mc_bytes + data_bytes) / wall_two * 1e-6 / peaks["hbm_gbs"])},
                "ms_per_iteration_nll_grad_plus_norm": ms_it, "ms_norm_build_fused_bw": ms_norm,
                "ms_data_term_fused_bw": ms_data,
                "e2e_ms_per_iteration_with_res_grad": wall_full,
                "iterations_per_s": 1e3 / ms_it,
                "event_waves_per_s": (w.n_data + w.n_acc) * n / ms_it * 1e3,
                "roofline_m_rebuild": rl_flops(peaks, "tensor", 4.0 * n * n * w.n_acc, ms_norm, kernel="k_norm_dmma (fused BW)",
                                               hbm_frac=mc_bytes / ms_norm * 1e-6 / peaks["hbm_gbs"]),
                "roofline_data_term": rl_flops(peaks, "alu", FLOPS_FACT_DATA * w.n_data, ms_data, kernel="k_data_term_fact",
                                               hbm_frac=data_bytes / ms_data * 1e-6 / peaks["hbm_gbs"]),
                "roofline_res_grad": rl_flops(peaks, "alu", FLOPS_RES_GRAD * (w.n_data + w.n_acc), ms_rg,
                                              kernel="k_res_grad_fast (data + MC pass)",
                                              timed="e2e iteration with res_grad minus device time of the iteration without")}
    finally:
        pwa.pwa_destroy(ctx)


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank, ws, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    # PWA_BENCH_BACKEND=gloo (tests only): several ranks share the visible GPUs and exchange through host memory, so that
    # the N > 1 code below can be exercised on a one-GPU box (tests/test_gpu_sharded.py); the driver's runs use nccl
    backend = os.environ.get("PWA_BENCH_BACKEND", "nccl")
    if backend != "nccl":
        local = local % torch.cuda.device_count()
    torch.cuda.set_device(local)
    if ws > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)
    if args.gpus != ws and rank == 0:
        sys.stderr.write(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={ws}; using {ws}\n")
    import __graft_entry__
    if rank == 0:
        __graft_entry__.build()
    if ws > 1:
        dist.barrier()
    from paper_1108_5882_b200 import binding as pwa
    from paper_1108_5882_b200 import sharded
    from paper_1108_5882_b200.inputs import synth

    cfg = WORKLOADS[args.workload]
    spec = synth._CFG[cfg]
    n_data, n_mc = sizes_for(args, spec)
    K, W = args.steps, args.warmup
    if W < 3:
        raise SystemExit("bench.py: --warmup must be >= 3")
    mp_hbm, mp_src, _ = load_peaks()
    elem = 8 if spec["storage"] == "f64" else 4
    extra_on = (not args.no_extra) and ws == 1
    tm = Timer(torch)
    barrier = (lambda: dist.barrier()) if ws > 1 else None
    stream = torch.cuda.current_stream().cuda_stream
    dev = torch.device("cuda", local)
    pctx = pwa.pwa_create(4, "f64", local, stream)
    try:
        peaks = measure_peaks(pwa, pctx, mp_hbm, mp_src)
    finally:
        pwa.pwa_destroy(pctx)
    t_gen = time.perf_counter()

    if spec["factored"]:
        # cfg3 as the main workload: a step is one floating-resonance iteration (M rebuild + lnL + gradient)
        w = synth.make_workload(cfg, n_data=n_data, n_mc=n_mc, full_amplitudes=False, shard=rank)
        if ws > 1:
            raise SystemExit("bench.py: the cfg3 step is single-GPU here; use the default workload for N > 1")
        clk = ClockSampler(local); clk.start()
        r = bench_floating(torch, pwa, synth, w, K, W, peaks)
        clk.stop()
        ms = r["two_pass_evaluation"]["ms_between_events"]
        line = {"metric": "event-waves/s (floating-resonance evaluation: lnL, V gradient, mass / width gradient)",
                "value": (w.n_data + w.n_acc) * w.n / ms * 1e3, "unit": "event-waves/s", "n_gpus": ws, "steps": K, "warmup": W,
                "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": args.workload, "n_waves": w.n, "n_data": w.n_data, "n_mc": w.n_acc,
                           "storage": w.storage, "l2": "factored inputs 200 MB > L2 126 MB"},
                "e2e": {"value": r["two_pass_evaluation"]["event_waves_per_s"],
                        "unit": "event-waves/s", "h2d_bytes_per_step": 16 * w.n + 16 * w.n_res,
                        "d2h_bytes_per_step": 8 * (4 + 2 * w.n) + 16 * w.n_res},
                "roofline": dict(r["two_pass_evaluation"]["roofline"], traffic=load_traffic("k_data_term_fact_rg")),
                "peaks": peaks, "clocks": clk.summary(), "extra": {"cfg3": r}, "gpu_launches": 2 * K}
        print(json.dumps(line), flush=True)
        return 0

    w = synth.make_workload(cfg, n_data=n_data, n_mc=(n_mc if extra_on or ws > 1 else 1),
                            want_mc=(extra_on or ws > 1), shard=rank)
    gen_s = time.perf_counter() - t_gen
    n = w.n
    ctx = pwa.pwa_create(n, w.storage, local, stream)
    extra = {"generate_s": gen_s}
    try:
        up_s = upload_constant(pwa, ctx, w)
        bytes_data = w.n_data * n * 2 * elem
        extra["upload_data_s"] = up_s
        # ---- normalisation matrix (once per fit; not part of the step)
        if w.A_mc is not None:
            ms_pre = upload_mc(torch, pwa, tm, ctx, w)
            extra["m_build"] = m_build_record(pwa, tm, ctx, w, n, elem, peaks)
            extra["m_build"]["upload_prepass_ms"] = ms_pre
            M_all = pwa.pwa_build_norm(ctx)
            if ws > 1:
                M_all, _ = sharded.combine_norm(ctx, device=dev if backend == "nccl" else None)
            w.A_mc = None   # free 10 GB of host memory
        else:
            M_all = np.zeros((n, n, 2)); M_all[np.arange(n), np.arange(n), 0] = 1.0
            pwa.pwa_set_norm(ctx, M_all)
        Vs = synth.eval_points(w, 2 * (K + W))
        out_dev = torch.zeros(2 + 2 * n, dtype=torch.float64, device=dev)

        # ---- the timed region: K steps, device-timed
        if ws == 1:
            step = lambda i: pwa.pwa_nll_grad_enqueue(ctx, Vs[i])          # noqa: E731
        else:
            def step(i):
                sharded.nll_grad(ctx, Vs[i], M_all, out_dev)
        clk = ClockSampler(local)
        # the peak probes and the M builds above load the board at ~1 kW for a second or two; its power limiter works on a
        # moving average, so let that decay before the warm-up (the sustained figure is reported separately: extra.sustained)
        torch.cuda.synchronize()
        time.sleep(2.0)
        for i in range(W):
            step(i)
        torch.cuda.synchronize()
        l0 = pwa.pwa_launch_count(ctx)
        clk.start()
        ms, _ = tm.run(step, K, 0, barrier)
        clk.stop()
        launches = pwa.pwa_launch_count(ctx) - l0
        # kernel-only loop for the roofline when the step also holds a collective
        if ws > 1:
            ms_kernel, _ = tm.run(lambda i: pwa.pwa_data_term_enqueue(ctx, Vs[i], out_dev), K, W)
        else:
            ms_kernel = ms
        # ---- end to end: synchronous C-ABI call, host V in, host results out
        def e2e_step(i):
            if ws == 1:
                return pwa.pwa_nll_grad(ctx, Vs[K + W + i])
            return sharded.nll_grad(ctx, Vs[K + W + i], M_all, out_dev)
        for i in range(W):
            e2e_step(i)
        torch.cuda.synchronize()
        if barrier:
            barrier()
        t0 = time.perf_counter()
        for i in range(K):
            e2e_step(W + i)
        torch.cuda.synchronize()
        wall_ms = (time.perf_counter() - t0) / K * 1e3
        gpu_at_V0 = pwa.pwa_nll_grad(ctx, Vs[0]) if ws == 1 else None
        # ---- the same step sustained for ~1 s (what a long fit sees: the board may reach its power cap)
        if extra_on and bytes_data > 1e9:
            clk_s = ClockSampler(local)
            n_sus = 2000
            clk_s.start()
            ms_sus, _ = tm.run(lambda i: pwa.pwa_nll_grad_enqueue(ctx, Vs[i % len(Vs)]), n_sus, 0)
            clk_s.stop()
            extra["sustained"] = {"steps": n_sus, "ms_per_step": ms_sus, "roofline": rl_hbm(peaks, bytes_data, ms_sus, kernel=f"k_data_term_{w.storage}_n{n}"),
                                  "clocks": clk_s.summary()}
            time.sleep(2.0)                                # let the board cool before the side measurements
        # ---- configs[4] as stated: K = 64 independent fits x 300 host BFGS iterations, in lock-step on the batched
        # call (A8 path); gtol = 0 so that every fit runs its 300 iterations unless its line search is exhausted
        if ws == 1 and w.K > 1 and w.A_mc is None and "m_build" in extra and not args.no_extra:
            iters = 300
            V0 = synth.eval_points(w, w.K, stream=synth.S_START)
            t0 = time.perf_counter()
            Vf, nllf, evals, _, its, why = pwa.pwa_minimize_bfgs_batch_ex(ctx, V0, max_iter=iters, gtol=0.0)
            dt = time.perf_counter() - t0
            path, _ = pwa.pwa_batch_path(ctx)
            extra["cfg4_multistart"] = {"K": w.K, "bfgs_iterations_requested": iters,
                                        "iterations_run_min_max": [int(its.min()), int(its.max())],
                                        "stop_reasons": {"max_iter": int((why == 1).sum()), "line_search": int((why == 2).sum()),
                                                         "converged": int((why == 0).sum())},
                                        "batched_evaluations": evals, "wall_s": dt,
                                        "e2e_ms_per_batched_evaluation": dt / max(evals, 1) * 1e3,
                                        "last_batch_path": path,
                                        "nll_best": float(np.min(nllf)), "nll_worst": float(np.max(nllf))}
        if ws > 1:
            t = torch.tensor([ms, wall_ms, ms_kernel], dtype=torch.float64, device=dev if backend == "nccl" else "cpu")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms, wall_ms, ms_kernel = (float(x) for x in t.tolist())
    finally:
        pwa.pwa_destroy(ctx)

    if rank != 0:
        if ws > 1:
            dist.barrier(); dist.destroy_process_group()
        return 0

    units = w.n_data * n * ws                      # event-waves per step, all ranks (weak scaling)
    kernel_key = f"k_data_term_{w.storage}_n{n}"
    roof = rl_hbm(peaks, bytes_data, ms_kernel, kernel=kernel_key, traffic=load_traffic(kernel_key))
    roof["frac_of_nominal_8TBs"] = roof["achieved"] / 8000.0
    if bytes_data > 2.5e8:
        roof["note"] = ("back-to-back evaluations: up to L2 / sample = %.1f %% of the bytes may still be L2-resident from the "
                        "previous evaluation; the cold-cache ncu launch list (profiles/) bounds the effect" % (126e6 / bytes_data * 100))
    line = {
        "metric": "event-waves/s (lnL+gradient evaluation)", "value": units / ms * 1e3, "unit": "event-waves/s",
        "n_gpus": ws, "steps": K, "warmup": W, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args.workload, n, w.n_data, w.storage, ws, backend),
        "evals_per_s": 1e3 / ms,
        "e2e": {"value": units / wall_ms * 1e3, "unit": "event-waves/s", "ms_per_step": wall_ms,
                "evals_per_s": 1e3 / wall_ms, "h2d_bytes_per_step": 16 * n, "d2h_bytes_per_step": 8 * (4 + 2 * n),
                "note": "events are uploaded once per fit (upload_data_s in extra), V and results cross every step"},
        "roofline": roof, "peaks": peaks,
        "clocks": clk.summary(), "gpu_launches": int(launches),
    }
    if ws == 1:
        line["cpu_baseline"], line["parity"] = cpu_baseline(synth, w, M_all, Vs[0], args.workload, gpu_at_V0)
    line["extra"] = side_measurements(torch, pwa, synth, args, extra, peaks) if extra_on else extra
    print(json.dumps(line), flush=True)
    if ws > 1:
        dist.barrier(); dist.destroy_process_group()
    return 0


def cpu_baseline(synth, w, M, V, name, gpu_result):
    """The oracle as it stands on this box's host cores, on a prefix of the same data.  When the prefix is the whole
    sample, the oracle's result at V is also compared with the GPU's at the same V (max parity error of the benched
    config, norm-wise as in DESIGN.md C8)."""
    from oracle import oracle
    S = oracle_sample_size(oracle, w.A_data, M, V, w.n_data, 5.0)
    A = np.ascontiguousarray(w.A_data[:S])
    reps, t0 = 3, time.perf_counter()
    for _ in range(reps):
        ref = oracle.nll_grad(A, M, V)
    dt = (time.perf_counter() - t0) / reps
    base = {"value": S * w.n / dt, "unit": "event-waves/s", "cores": oracle.threads(), "kind": "oracle",
            "sample": f"first {S} of {w.n_data} data events of {name}, {reps} full lnL+gradient evaluations, {dt:.2f} s each"}
    # the same oracle on ONE thread, on a prefix of about a second
    nt = oracle.threads()
    try:
        oracle.set_threads(1)
        S1 = max(1, min(S, int(S / max(nt, 1) / max(dt, 1e-3))))
        A1 = A[:S1]
        t0 = time.perf_counter()
        oracle.nll_grad(A1, M, V)
        dt1 = time.perf_counter() - t0
        base["one_thread"] = {"value": S1 * w.n / dt1, "unit": "event-waves/s", "sample": f"first {S1} events, 1 evaluation, {dt1:.2f} s"}
    finally:
        oracle.set_threads(nt)
    parity = None
    if gpu_result is not None and S == w.n_data:
        nll_o, g_o, parts_o = ref[0], ref[1], ref[2]
        parity = {"vs": "oracle, same V, all events of the benched config",
                  "nll_rel": abs(gpu_result[0] - nll_o) / max(abs(nll_o), abs(parts_o[0])),
                  "L_data_rel": abs(gpu_result[2][0] - parts_o[0]) / abs(parts_o[0]),
                  "grad_rel_maxnorm": float(np.abs(gpu_result[1] - g_o).max() / np.abs(g_o).max()),
                  "tolerance": 1e-12 if w.storage == "f64" else 1e-6}
    return base, parity


def side_measurements(torch, pwa, synth, args, extra, peaks):
    """Other configs of BASELINE.json, single GPU, each in the launch configuration the tests check; the iteration
    counts are the ones the configs state (cfg1: 100 evaluations, cfg2: 1000, cfg3: 200 quasi-Newton iterations)."""
    try:
        w2 = synth.make_workload(2)
        extra["cfg2"] = bench_constant(torch, pwa, synth, w2, 1000, 5, 4, peaks)
        del w2
        w1 = synth.make_workload(1)
        extra["cfg1"] = bench_constant(torch, pwa, synth, w1, 100, 5, 8, peaks)
        del w1
        w3 = synth.make_workload(3, full_amplitudes=False)
        extra["cfg3"] = bench_floating(torch, pwa, synth, w3, 20, 3, peaks)
        del w3
        if args.workload == "cfg4":
            w4 = synth.make_workload(4, n_mc=1, want_mc=False)
            w4.A_mc = None
            r = bench_constant(torch, pwa, synth, w4, SIDE_STEPS, SIDE_WARMUP, 4, peaks)
            extra["cfg4_batch"] = r.get("batch")
            extra["cfg4_fumili"] = r.get("fumili")
            extra["cfg4_weighted"] = r.get("weighted")
    except Exception as e:   # side measurements must never lose the main line
        extra["error"] = repr(e)
    return extra


if __name__ == "__main__":
    a = parse_args()
    sys.exit(run_reference(a) if a.impl == "reference" else run_ours(a))
