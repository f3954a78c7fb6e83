#!/usr/bin/env python
"""bench.py -- throughput of the hot path (Cartesian gradient + Yn tensor filter, FP64) on B200.

A "step" is one pass of the whole hot path over one synthetic state of the chosen configuration:
sp_cartesian_gradient of all fields, then sp_tensor_filter of all tensors (SURVEY.md 8(a) rows G1-G4,
F1-F5).  metric = grid-point*fields/s (BASELINE.json).  Contract: one JSON line on stdout (rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

N > 1 (torchrun): the path shards with no exchange step: every rank runs the full
configuration on its own seeded state (independent shells), weak scaling, no data-path collective.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "grid-point*fields/s, gradient + Yn filter (FP64)"
UNIT = "grid-point*fields/s"
L2_BYTES = 126e6


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=4,
                    help="BASELINE.json config (1-based); default 4 = the largest single-GPU configuration (58 fields at 65x96x192)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-others", action="store_true", help="skip the short runs of the other configs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--leg", default="main", choices=["main", "ghg", "ghg_rhs", "filters", "fft", "convergence"],
                    help="ghg: run only the GHG single-black-hole leg (SURVEY.md 8(f) NEXT-1) and print its JSON")
    ap.add_argument("--t-end", type=float, default=20000.0, help="--leg filters: evolve every filter variant to this time")
    ap.add_argument("--no-graph", action="store_true", help="time eager launches instead of replayed CUDA graphs of the step")
    return ap.parse_args()


def flops_per_unit(cfg):
    """Algorithmic flops per grid-point*field: per stage."""
    Nr, Nt, Np, L = cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["L"]
    return {
        "grad_dphi": 2.0 * Np,
        "grad_rtheta": 2.0 * Nr + 4.0 * Nt + 13.0,
        "filt_project": 0.0,
        "filt_analysis": 2.0 * (2 * L + 1),
        "filt_theta": 1.0 * (2 * L + 1),
        "filt_synthesis": 2.0 * (2 * L + 1),
        "filt_recombine": 0.0,
    }


def workload_name(cfg):
    return (f"config {cfg['id']}: {cfg['nfields']} fields ({'+'.join(t['name'] for t in cfg['tensors'])}), "
            f"Nr x Ntheta x Nphi = {cfg['Nr']}x{cfg['Nt']}x{cfg['Np']}, shell [{cfg['rmin']},{cfg['rmax']}], L = {cfg['L']}")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.stop_flag, self.index, self.nv = [], False, index, None
        self.t = threading.Thread(target=self._run, daemon=True)

    def _nvml_setup(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.mx = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.bits = [pynvml.nvmlClocksEventReasonHwSlowdown, pynvml.nvmlClocksEventReasonHwThermalSlowdown,
                         pynvml.nvmlClocksEventReasonSwThermalSlowdown, pynvml.nvmlClocksEventReasonSwPowerCap]
            self._nvml_sample()
            return True
        except Exception:
            self.nv = None
            return False

    def _nvml_sample(self):
        nv = self.nv
        sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
        try:
            rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            rs = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1e3
        self.rows.append([str(sm), str(self.mx), str(pw)] + ["Active" if (rs & bit) else "Not Active" for bit in self.bits])

    def _run(self):
        if self.nv is not None:               # NVML in-process: a sample every few ms
            while not self.stop_flag:
                try:
                    self._nvml_sample()
                except Exception:
                    break
                time.sleep(0.002)
            return
        while not self.stop_flag:
            self._one_smi()
            time.sleep(0.05)

    def _one_smi(self):
        try:
            out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                 capture_output=True, text=True, timeout=10).stdout.strip()
            if out:
                self.rows.append([x.strip() for x in out.split(",")])
        except Exception:
            pass

    def start(self):
        self.rows = []
        self._nvml_setup()                    # NVML is initialised here, before the timed region, not in the thread
        self.rows = []
        self.t.start()

    def stop(self):
        self.stop_flag = True
        self.t.join(timeout=6)
        if not self.rows:                      # the sampling thread got nothing (NVML unavailable): one direct reading
            self._one_smi()
        sm = sorted(float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit())
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            for q, nm in enumerate(names):
                if len(r) > 3 + q and r[3 + q].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None,
                "sm_max_mhz": float(self.rows[0][1]) if self.rows and self.rows[0][1].replace(".", "").isdigit() else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline and --impl reference): the oracle as it stands, on a bounded sample
# ---------------------------------------------------------------------------------------------------
ORACLE_SAMPLE = {   # config -> (fields differentiated on the full grid, radii on which ALL tensors of the state are filtered)
    1: (1, 9), 2: (50, 17), 3: (16, 8), 4: (16, 4), 5: (5, 8),
}


def oracle_sample(cfg, u, threads):
    """One bounded sample of the workload through the oracle, as it stands.  Returns (seconds per unit, seconds, description).
    A unit is one grid-point*field that went through the gradient AND the filter.  The gradient leg differentiates the first
    fields of the state on the full grid (OpenMP over fields); the filter leg filters ALL tensors of the state on the spheres
    at evenly spaced radii in ONE oracle call (the filter acts on every radius independently, so a state thinned
    to those radii is the same work per unit; OpenMP over (tensor, radius) spheres).  The one-off filter-matrix table (start-up
    cost) is built by an untimed call on one sphere first."""
    import numpy as np
    import oracle
    oracle.set_threads(threads)
    Nr, Nt, Np = cfg["Nr"], cfg["Nt"], cfg["Np"]
    nfg, nrad = ORACLE_SAMPLE[cfg["id"]]
    nfg, nrad = min(nfg, cfg["nfields"]), min(nrad, Nr)
    ug = np.ascontiguousarray(u[:nfg])
    a = time.perf_counter()
    oracle.gradient(ug, Nr, Nt, Np, cfg["rmin"], cfg["rmax"])
    tg = time.perf_counter() - a
    radii = sorted({int(round(q * (Nr - 1) / max(nrad - 1, 1))) for q in range(nrad)})
    us = np.ascontiguousarray(u[..., radii])
    oracle.tensor_filter(np.ascontiguousarray(us[..., :1]), 1, Nt, Np, cfg["L"], cfg["tensors"])      # table build, untimed
    a = time.perf_counter()
    oracle.tensor_filter(us, len(radii), Nt, Np, cfg["L"], cfg["tensors"])
    tf = time.perf_counter() - a
    nff = sum(len(t["fields"]) for t in cfg["tensors"])
    per_unit = tg / (nfg * Nr * Nt * Np) + tf / (nff * len(radii) * Nt * Np)
    desc = (f"oracle (plain C, long double, OpenMP x{threads}): gradient of {nfg} field(s) on the full grid + Yn filter of "
            f"all {len(cfg['tensors'])} tensors ({nff} fields) on the spheres at {len(radii)} of {Nr} radii "
            f"(one-off filter-matrix table built before the timed call)")
    return per_unit, tg + tf, desc


def paper_style_cpu_gradient(cfg, u, threads):
    """The paper's own CPU formulation of the derivative (eq. 13-19): one dgemm per direction on the
    whole state array with explicit transposes, in double precision through numpy/BLAS, then the chain rule (eq. 6).
    A timing baseline of the harness (not the oracle, not the product); returns seconds for the gradient of all fields."""
    import numpy as np
    from threadpoolctl import threadpool_limits
    Nr, Nt, Np = cfg["Nr"], cfg["Nt"], cfg["Np"]
    nv = u.shape[0]
    k = np.arange(Nr)
    x = -np.cos(np.pi * k / (Nr - 1))
    c = np.where((k == 0) | (k == Nr - 1), 2.0, 1.0)
    with np.errstate(divide="ignore"):
        CD = (c[:, None] / c[None, :]) * (-1.0) ** (k[:, None] + k[None, :]) / (x[:, None] - x[None, :])
    CD[k, k] = 0.0
    CD[k, k] = -CD.sum(axis=1)
    CD *= 2.0 / (cfg["rmax"] - cfg["rmin"])

    def FD(n):
        i = np.arange(n)
        d = i[:, None] - i[None, :]
        with np.errstate(divide="ignore"):
            M = (-1.0) ** d / (2.0 * np.tan(d * np.pi / n))
        M[i, i] = 0.0
        return M
    F2, F3 = FD(2 * Nt)[:Nt], FD(Np)
    r = 0.5 * (cfg["rmax"] + cfg["rmin"]) + 0.5 * (cfg["rmax"] - cfg["rmin"]) * x
    th = np.pi * (np.arange(Nt) + 0.5) / Nt
    ph = 2 * np.pi * np.arange(Np) / Np
    st, ct, sp, cp = np.sin(th)[None, :, None], np.cos(th)[None, :, None], np.sin(ph)[:, None, None], np.cos(ph)[:, None, None]
    ir = (1.0 / r)[None, None, :]
    with threadpool_limits(limits=threads):
        a = time.perf_counter()
        U = u.reshape(nv, Np, Nt, Nr)
        dr = (U.reshape(-1, Nr) @ CD.T).reshape(U.shape)                           # eq. 13: contiguous direction
        ext = np.concatenate([U, np.roll(U, Nt, axis=1)[:, :, ::-1, :]], axis=2)   # double cover
        T = np.ascontiguousarray(ext.transpose(0, 1, 3, 2))                        # transpose, eq. 14-16
        dth = np.ascontiguousarray((T.reshape(-1, 2 * Nt) @ F2.T).reshape(nv, Np, Nr, Nt).transpose(0, 1, 3, 2))
        T = np.ascontiguousarray(U.transpose(0, 2, 3, 1))                          # transpose, eq. 17-19
        dph = np.ascontiguousarray((T.reshape(-1, Np) @ F3.T).reshape(nv, Nt, Nr, Np).transpose(0, 3, 1, 2))
        out = np.empty((3,) + U.shape)
        out[0] = st * cp * dr + ct * cp * ir * dth - sp / st * ir * dph
        out[1] = st * sp * dr + ct * sp * ir * dth + cp / st * ir * dph
        out[2] = ct * dr - st * ir * dth
        return time.perf_counter() - a, out


def run_reference(args):
    import numpy as np
    import synth
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:                                # the oracle runs on rank 0's host cores only; the other ranks check in and leave
        import torch.distributed as dist
        dist.init_process_group("gloo")
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return 0
    cfg = synth.config(args.config)
    u = synth.make_state(cfg)
    threads = os.cpu_count() or 1
    for _ in range(args.warmup):
        oracle_sample(cfg, u, threads)
    tot_units_time, wall, desc = 0.0, 0.0, ""
    for _ in range(args.steps):
        pu, w, desc = oracle_sample(cfg, u, threads)
        tot_units_time += pu
        wall += w
    value = 1.0 / (tot_units_time / max(args.steps, 1))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": max(world, 1), "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(args.steps, 1), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "sample": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------------
# GPU leg
# ---------------------------------------------------------------------------------------------------
def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def aggregate_over_ranks(ms_local, units_local, dist=None):
    """Whole-job numbers from per-rank ones: time = MAX over ranks, units = SUM over ranks.
    (No data-path collective exists; these two scalars are the only cross-rank traffic.)"""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return ms_local, units_local
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    n = torch.tensor([units_local], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t.item()), float(n.item())


class GpuWorkload:
    """State, outputs and workspaces of one configuration resident in HBM; step() = gradient + filter."""

    def __init__(self, cfg, seed_offset=0, nsets=None):
        import torch
        import synth
        from paper_1104_3408_b200 import Shell
        self.torch, self.cfg = torch, cfg
        self.sh = Shell(cfg["Nr"], cfg["Nt"], cfg["Np"], cfg["rmin"], cfg["rmax"], cfg["L"])
        u = synth.make_state(cfg, seed=cfg["seed"] + 1000 * seed_offset)
        self.u_host = u
        state_bytes = u.nbytes
        # rotate over enough distinct input sets that consecutive steps never find their input in L2
        self.nsets = nsets if nsets is not None else max(2, int(2 * L2_BYTES // state_bytes) + 1)
        self.nsets = min(self.nsets, 8)
        self.u = [torch.from_numpy(u).cuda() for _ in range(self.nsets)]
        nf = cfg["nfields"]
        self.du = torch.empty((3, nf, cfg["Np"], cfg["Nt"], cfg["Nr"]), dtype=torch.float64, device="cuda")
        self.fu = torch.empty_like(self.u[0])
        g, f, _ = self.sh.workspace_bytes(nf)
        self.ws_g = torch.empty(g // 8, dtype=torch.float64, device="cuda")
        self.ws_f = torch.empty(f // 8, dtype=torch.float64, device="cuda")
        self.descs = self.sh.make_descs(cfg["tensors"])
        self.units = float(cfg["npts"] * nf)
        self.it = 0

    def step(self, sg=None, sf=None):
        """One pass of the hot path over one state: gradient of all fields and Yn filter of all tensors.  The two calls are
        independent (both read u), so with two streams they are issued side by side -- the "parallel kernels" the paper
        names as its next optimisation."""
        u = self.u[self.it % self.nsets]
        self.it += 1
        self.sh.cartesian_gradient(u, out=self.du, workspace=self.ws_g, stream=sg)
        self.sh.tensor_filter(u, self.cfg["tensors"], out=self.fu, workspace=self.ws_f, descs=self.descs, stream=sf)

    def capture(self):
        """CUDA graphs of the step (every pointer of a step is fixed, the library allocates nothing and its internal side
        stream is forked/joined by events, so the calls are capturable as they are): one graph per input copy holding ONE
        step (gradient and filter forked onto two streams, joined at the end), and one graph holding a ROUND of nsets steps,
        one per input copy, whose gradient chain and filter chain run side by side and are joined only at the end of the
        round (as with eager launches on two streams).  Returns launches per step."""
        torch = self.torch
        from paper_1104_3408_b200 import launch_count
        side = torch.cuda.Stream()
        sg, sf = torch.cuda.Stream(), torch.cuda.Stream()
        self.graphs, per_step = [], 0

        def one_graph(first, count):
            self.it = first
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                ev = torch.cuda.Event(); ev.record(side); sg.wait_event(ev); sf.wait_event(ev)
                for _ in range(count):
                    self.step(sg, sf)
                for q in (sg, sf):
                    ev = torch.cuda.Event(); ev.record(q); side.wait_event(ev)
            return g
        for i in range(self.nsets):
            l0 = launch_count()
            self.graphs.append(one_graph(i, 1))
            per_step = launch_count() - l0
        self.round_graph = one_graph(0, self.nsets)
        self.it = 0
        return per_step

    def time_graph_steps(self, steps, warmup):
        """EXACTLY `steps` steps: whole rounds of nsets steps by the round graph, the remainder by single-step graphs."""
        torch = self.torch
        self.round_graph.replay()
        for n in range(warmup):
            self.graphs[n % self.nsets].replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        rounds, rest = divmod(steps, self.nsets)
        e0.record()
        for _ in range(rounds):
            self.round_graph.replay()
        for n in range(rest):
            self.graphs[n].replay()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    def time_steps(self, steps, warmup, concurrent=True):
        torch = self.torch
        cur = torch.cuda.current_stream()
        sg = sf = None
        if concurrent:
            sg, sf = torch.cuda.Stream(), torch.cuda.Stream()
        for _ in range(warmup):
            self.step(sg, sf)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        if concurrent:
            sg.wait_event(e0); sf.wait_event(e0)
        for _ in range(steps):
            self.step(sg, sf)
        if concurrent:
            for s_ in (sg, sf):
                ev = torch.cuda.Event(); ev.record(s_); cur.wait_event(ev)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    def time_call(self, which, steps, warmup=3):
        """Device time (ms per call) of ONE of the two hot calls alone, back to back on the current stream."""
        torch = self.torch

        def one():
            u = self.u[self.it % self.nsets]
            self.it += 1
            if which == "gradient":
                self.sh.cartesian_gradient(u, out=self.du, workspace=self.ws_g)
            else:
                self.sh.tensor_filter(u, self.cfg["tensors"], out=self.fu, workspace=self.ws_f, descs=self.descs)
        for _ in range(warmup):
            one()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            one()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / steps

    def latency_floor_ms(self, nlaunch, reps=200):
        """Launch/latency floor of a step: a CUDA graph of `nlaunch` DEPENDENT near-empty kernels (one 8-byte fill each) replayed
        back to back -- what a step of that many launches costs on this device when every kernel has nothing to do."""
        torch = self.torch
        x = torch.zeros(1, dtype=torch.float64, device="cuda")
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            for _ in range(nlaunch):
                x.add_(1.0)
        g.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            g.replay()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    def time_call_graph(self, which, steps, warmup=1):
        """The same call alone, replayed from a CUDA graph holding one call per input copy (the headline's launch mode)."""
        torch = self.torch
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        self.it = 0
        with torch.cuda.graph(g, stream=side):
            for _ in range(self.nsets):
                u = self.u[self.it % self.nsets]
                self.it += 1
                if which == "gradient":
                    self.sh.cartesian_gradient(u, out=self.du, workspace=self.ws_g, stream=side)
                else:
                    self.sh.tensor_filter(u, self.cfg["tensors"], out=self.fu, workspace=self.ws_f, descs=self.descs, stream=side)
        rounds = max(1, steps // self.nsets)
        for _ in range(warmup):
            g.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(rounds):
            g.replay()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / (rounds * self.nsets)

    def calls_report(self, steps, peak_tf):
        """each call alone -- units/s, achieved algorithmic TFLOP/s, fraction of the FP64 peak."""
        fl = flops_per_unit(self.cfg)
        fg = fl["grad_dphi"] + fl["grad_rtheta"]
        ff = fl["filt_analysis"] + fl["filt_theta"] + fl["filt_synthesis"]
        out = {}
        for which, f in (("gradient", fg), ("filter", ff)):
            ms = sorted(self.time_call(which, steps) for _ in range(3))[1]      # median of three runs
            tf = f * self.units / (ms * 1e-3) * 1e-12
            out[which] = {"ms": ms, "value": self.units / (ms * 1e-3), "algorithmic_flops_per_unit": f, "tflops": tf,
                          "frac_of_fp64_peak": tf / peak_tf}
            try:                                                             # same call replayed from a CUDA graph
                msg = sorted(self.time_call_graph(which, steps) for _ in range(3))[1]
                out[which]["graph_ms"] = msg
                out[which]["graph_frac_of_fp64_peak"] = f * self.units / (msg * 1e-3) * 1e-12 / peak_tf
            except Exception as ex:                                          # capture refused: the eager figure stands alone
                out[which]["graph_ms"] = None
                print(f"bench.py: per-call graph capture failed ({ex!r})", file=sys.stderr)
        return out

    def stage_times(self, reps=5):
        """Per-stage device times (ms), median over reps, from CUDA events recorded inside the library
        on the launching stream (sp_profile_enable)."""
        import statistics
        self.sh.profile(True)
        rows = []
        for _ in range(reps):
            self.step()
            rows.append(self.sh.profile_read())
        self.sh.profile(False)
        return {k: statistics.median(r[k] for r in rows) for k in rows[0]}

    def e2e(self, steps):
        """Same metric through the public API with HOST buffers: every step copies its state from pinned host
        memory to the device, runs gradient + filter, and copies the gradient and the filtered state back to
        pinned host memory; all of it inside the timed region.  Copies and kernels of neighbouring steps overlap
        on three streams (H2D, compute, D2H) with double-buffered device arrays -- PCIe is full duplex."""
        torch = self.torch
        hu = torch.from_numpy(self.u_host).pin_memory()
        hdu = torch.empty(self.du.shape, dtype=torch.float64).pin_memory()
        hfu = torch.empty(self.fu.shape, dtype=torch.float64).pin_memory()
        s_in, s_c, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
        ud = [self.u[0], self.u[1 % self.nsets]]
        du = [self.du, torch.empty_like(self.du)]
        fu = [self.fu, torch.empty_like(self.fu)]
        ev_in = [torch.cuda.Event() for _ in range(2)]
        ev_c = [torch.cuda.Event() for _ in range(2)]
        ev_out = [torch.cuda.Event() for _ in range(2)]

        def one(n):
            b = n & 1
            with torch.cuda.stream(s_in):
                s_in.wait_event(ev_c[b])              # compute of step n-2 has finished reading ud[b]
                ud[b].copy_(hu, non_blocking=True)
                ev_in[b].record(s_in)
            with torch.cuda.stream(s_c):
                s_c.wait_event(ev_in[b])
                s_c.wait_event(ev_out[b])             # D2H of step n-2 has drained du[b], fu[b]
                self.sh.cartesian_gradient(ud[b], out=du[b], workspace=self.ws_g, stream=s_c)
                self.sh.tensor_filter(ud[b], self.cfg["tensors"], out=fu[b], workspace=self.ws_f, descs=self.descs, stream=s_c)
                ev_c[b].record(s_c)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_c[b])
                hdu.copy_(du[b], non_blocking=True)
                hfu.copy_(fu[b], non_blocking=True)
                ev_out[b].record(s_out)

        torch.cuda.synchronize()
        for n in range(2):
            one(n)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for s_ in (s_in, s_c, s_out):
            s_.wait_event(e0)
        for n in range(steps):
            one(n)
        cur = torch.cuda.current_stream()
        for s_ in (s_in, s_c, s_out):
            ev = torch.cuda.Event(); ev.record(s_); cur.wait_event(ev)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        return ms, hu.numel() * 8, (hdu.numel() + hfu.numel()) * 8


def ghg_e1_leg(evolve=True):
    """The paper's own application (Sec. 4.1, Tab. 4): 1000 RK4 steps of the GHG system for the
    Kerr-Schild black hole on the shell R10 = [1.8, 11.8] at the paper's three grids, Yn filter with n_f = 4 after every
    step, lambda = 4, freezing outer boundary; each RK4 step is one replayed CUDA graph.  Reports the wall time of the 1000
    steps next to the paper's GTX580 / one-core i7-870 times (context: other hardware) and rhs(g_tt) on the innermost sphere
    at t = 0 and at the end (Fig. 2: the run must settle, not grow)."""
    import torch
    import synth
    from paper_1104_3408_b200 import Shell
    from paper_1104_3408_b200.ghg import GhgRK4
    from paper_1104_3408_b200.wave import wave_dt
    out = {"what": "1000 RK4 steps, 50-field GHG system, single Kerr-Schild black hole, shell [1.8, 11.8], Yn filter n_f = 4, lambda = 4",
           "paper_tab4_seconds": {"25x9x18": {"gtx580": 16, "i7_870_one_core": 165}, "37x15x30": {"gtx580": 49, "i7_870_one_core": 823},
                                  "49x21x42": {"gtx580": 133, "i7_870_one_core": 2903}}, "grids": {}}
    rmin, rmax = 1.8, 11.8
    for Nr, Nt, Np in (((25, 9, 18), (37, 15, 30), (49, 21, 42)) if evolve else ()):
        sh = Shell(Nr, Nt, Np, rmin, rmax, Nt - 1 - 4)
        g = torch.from_numpy(synth.kerr_schild_metric(Nr, Nt, Np, rmin, rmax)).cuda()
        u, H, dH = sh.ghg_init(g)
        rk = GhgRK4(sh, H, dH)
        r_init = rk.rhs(u)
        n0, m0 = float(r_init[0, :, :, 0].abs().max()), float(r_init.abs().max())
        dt = wave_dt(Nr, Nt, Np, rmin, rmax, lam=4.0)
        keep = u.clone()
        rk.evolve(u, dt, 3, graph=True)
        u.copy_(keep)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record()
        rk.evolve(u, dt, 1000, graph=True)
        e1.record()
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        r_end = rk.rhs(u)
        n1, m1 = float(r_end[0, :, :, 0].abs().max()), float(r_end.abs().max())
        out["grids"][f"{Nr}x{Nt}x{Np}"] = {"seconds_1000_steps": e0.elapsed_time(e1) * 1e-3, "wall_seconds": wall, "dt": dt,
                                           "t_end": 1000 * dt, "rhs_gtt_inner_sphere_t0": n0, "rhs_gtt_inner_sphere_end": n1,
                                           "rhs_all_fields_t0": m0, "rhs_all_fields_end": m1,
                                           "max_drift_of_state": float((u - keep).abs().max())}
    # the right-hand side alone on the config-3 grid (152 064 points x 50 fields): gradient + pointwise algebra + boundary
    Nr, Nt, Np = 33, 48, 96
    sh = Shell(Nr, Nt, Np, 1.8, 20.0, 43)
    g = torch.from_numpy(synth.kerr_schild_metric(Nr, Nt, Np, 1.8, 20.0)).cuda()
    u, H, dH = sh.ghg_init(g)
    rk = GhgRK4(sh, H, dH)
    du = torch.empty((3, 50, Np, Nt, Nr), dtype=torch.float64, device="cuda")
    ws = torch.empty(50 * Np * Nt * Nr, dtype=torch.float64, device="cuda")

    def timeit(fn, reps=50):
        for _ in range(5):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps
    t_rhs = timeit(lambda: rk.rhs(u))
    t_grad = timeit(lambda: sh.cartesian_gradient(u, out=du, workspace=ws))
    npts = Nr * Nt * Np
    out["rhs_on_config3_grid"] = {"rhs_total_ms": t_rhs, "gradient_ms": t_grad, "pointwise_and_boundary_ms": t_rhs - t_grad,
                                  "pointwise_bytes": 266 * 8 * npts,
                                  "pointwise_GBs": 266 * 8 * npts / ((t_rhs - t_grad) * 1e-3) * 1e-9,
                                  "note": "pointwise kernel: 216 doubles read + 50 written per point (HBM-bound by design)"}
    return out


def filter_comparison_leg(t_end, every=5000.0):
    """PAPER.md Sec. 4.1, Fig. 5-6 (SURVEY.md experiment E3, NEXT-2): the single black hole on 25 x 9 x 18 evolved with the
    scalar Y-filter, the graded Yg-filter (eq. 59) and the tensor Yn-filter; max |rhs(g_tt)| on the innermost sphere is
    sampled every `every` in t.  The paper: Y fails by t ~ 7 000, Yg by ~ 70 000, Yn runs beyond 200 000."""
    import torch
    import synth
    from paper_1104_3408_b200 import Shell
    from paper_1104_3408_b200.ghg import GhgRK4
    from paper_1104_3408_b200.wave import wave_dt
    Nr, Nt, Np, rmin, rmax = 25, 9, 18, 1.8, 11.8
    dt = wave_dt(Nr, Nt, Np, rmin, rmax, lam=4.0)
    out = {"what": "single black hole, 25x9x18, shell [1.8, 11.8], n_f = 4, lambda = 4: max|rhs(g_tt)| on the inner sphere vs t",
           "paper": "Y fails by t ~ 7e3, Yg by ~ 7e4, Yn lasts beyond 2e5 (PAPER.md:523-543)", "dt": dt, "runs": {}}
    for mode in ("Y", "Yg", "Yn"):
        sh = Shell(Nr, Nt, Np, rmin, rmax, Nt - 1 - 4)
        g = torch.from_numpy(synth.kerr_schild_metric(Nr, Nt, Np, rmin, rmax)).cuda()
        u, H, dH = sh.ghg_init(g)
        rk = GhgRK4(sh, H, dH, filter=mode)
        chunk = max(1, int(every / dt))
        t, rows, t0, failed_at = 0.0, [], time.perf_counter(), None
        while t < t_end:
            rk.evolve(u, dt, chunk, graph=True)
            t += chunk * dt
            n = float(rk.rhs(u)[0, :, :, 0].abs().max())
            rows.append([round(t, 1), n])
            if not (n == n) or n > 1.0:
                failed_at = t
                break
        out["runs"][mode] = {"samples_t_rhs": rows, "failed_by_t": failed_at, "reached_t": t, "wall_seconds": time.perf_counter() - t0}
    return out


def convergence_leg(t_end=1000.0):
    """PAPER.md Sec. 4.1, Fig. 2: the single black hole evolved to t = 1000 at Ntheta x Nphi = 9 x 18 and Nr = 13 ... 37;
    max |rhs(g_tt)| on the innermost sphere against t.  The paper: exponential convergence with Nr, the oscillation dies out
    and the runs settle; round-off (1e-12 ... 1e-13) is reached at Nr ~ 37-40."""
    import torch
    import synth
    from paper_1104_3408_b200 import Shell
    from paper_1104_3408_b200.ghg import GhgRK4
    from paper_1104_3408_b200.wave import wave_dt
    Nt, Np, rmin, rmax = 9, 18, 1.8, 11.8
    out = {"what": "single black hole, Nr x 9 x 18, shell [1.8, 11.8], Yn filter n_f = 4, lambda = 4: max|rhs(g_tt)| on the inner sphere",
           "paper": "Fig. 2 (PAPER.md:487-505): exponential convergence with Nr; round-off 1e-12..1e-13 near Nr = 37-40", "runs": {}}
    for Nr in (13, 17, 21, 25, 29, 33, 37):
        sh = Shell(Nr, Nt, Np, rmin, rmax, Nt - 1 - 4)
        g = torch.from_numpy(synth.kerr_schild_metric(Nr, Nt, Np, rmin, rmax)).cuda()
        u, H, dH = sh.ghg_init(g)
        rk = GhgRK4(sh, H, dH)
        dt = wave_dt(Nr, Nt, Np, rmin, rmax, lam=4.0)
        rows, t = [], 0.0
        chunk = max(1, int(round(50.0 / dt)))
        peak = 0.0
        while t < t_end:
            # the oscillation: sample the maximum over the chunk's last 20 steps rather than one phase of it
            rk.evolve(u, dt, max(chunk - 20, 1), graph=True)
            m = 0.0
            for _ in range(20):
                rk.evolve(u, dt, 1, graph=True)
                m = max(m, float(rk.rhs(u)[0, :, :, 0].abs().max()))
            t += (max(chunk - 20, 1) + 20) * dt
            rows.append([round(t, 1), m])
            peak = max(peak, m)
        out["runs"][str(Nr)] = {"dt": dt, "samples_t_rhs": rows, "max_over_run": peak, "final": rows[-1][1]}
    return out


def fft_comparison_leg():
    """PAPER.md Sec. 4.2, Fig. 9: one-directional periodic derivative of n1 x (20*20*54) values, by matrix
    multiplication and by FFT, against n1.  A measurement with library calls on both sides (cuBLAS DGEMM through torch.matmul,
    cuFFT through torch.fft, each in its best layout), plus this library's own d/dphi stage (GEMM + chain-rule epilogue, two
    outputs) on a shell with Nphi = n1 and about the same number of columns."""
    import torch
    from paper_1104_3408_b200 import Shell
    cols = 20 * 20 * 54
    out = {"what": "derivative along one periodic direction of an n1 x 21600 array, FP64: time in microseconds",
           "paper": "matmul competitive with CUFFT up to n1 ~ 100 on GTX580/M2070 (PAPER.md:563-567, Fig. 9)", "rows": []}

    def timeit(fn, reps=50):
        for _ in range(5):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps * 1e3
    for n1 in (16, 24, 32, 48, 64, 96, 128, 160, 192, 256):
        x = torch.randn(n1, cols, dtype=torch.float64, device="cuda")          # GEMM layout: D [n1 x n1] @ X [n1 x cols]
        xt = x.t().contiguous()                                                   # FFT layout: cols transforms of length n1, contiguous
        D = torch.randn(n1, n1, dtype=torch.float64, device="cuda")
        ik = (1j * torch.fft.rfftfreq(n1, 1.0 / n1).to("cuda")).to(torch.complex128)
        t_mm = timeit(lambda: torch.matmul(D, x))
        t_fft = timeit(lambda: torch.fft.irfft(torch.fft.rfft(xt, dim=1) * ik, n=n1, dim=1))
        row = {"n1": n1, "cublas_dgemm_us": t_mm, "cufft_rfft_mul_irfft_us": t_fft}
        Nt = n1 // 2
        if Nt >= 4:
            Nr = 15
            nf = max(1, round(cols / (Nr * Nt)))
            sh = Shell(Nr, Nt, n1, 1.0, 2.0, Nt - 1)
            u = torch.randn(nf, n1, Nt, Nr, dtype=torch.float64, device="cuda")
            du = torch.empty((3, nf, n1, Nt, Nr), dtype=torch.float64, device="cuda")
            ws = torch.empty(nf * n1 * Nt * Nr, dtype=torch.float64, device="cuda")
            sh.profile(True)
            ts = []
            for _ in range(7):
                sh.cartesian_gradient(u, out=du, workspace=ws)
                ts.append(sh.profile_read()["grad_dphi"])
            sh.profile(False)
            row["ours_dphi_with_chain_rule_us"] = sorted(ts)[len(ts) // 2] * 1e3
            row["ours_columns"] = nf * Nr * Nt
        out["rows"].append(row)
    # the d/dphi product of config 3 in its own layout: 50 fields x [96 x 96] @ [96 x 1584] (K stride 1584), cuBLAS batched
    X = torch.randn(50, 96, 1584, dtype=torch.float64, device="cuda")
    D = torch.randn(96, 96, dtype=torch.float64, device="cuda")
    Y = torch.empty_like(X)
    t = timeit(lambda: torch.matmul(D, X, out=Y))
    out["config3_dphi_shape"] = {"cublas_batched_dgemm_us": t, "tflops": 2.0 * 96 * 96 * 50 * 1584 / t * 1e-6,
                                 "note": "product only; the library's stage (grad_dphi in the main line) also applies the chain rule "
                                         "and writes d_x and d_y (another 2 x 61 MB read and 2 x 61 MB written)"}
    return out


def roofline_for(cfg, stages_ms, units, peak_tf, hbm_gbs, hbm_src):
    fl = flops_per_unit(cfg)
    table = {}
    for k, ms in stages_ms.items():
        if ms is None or ms <= 0:
            continue
        table[k] = {"ms": ms, "tflops": fl[k] * units / (ms * 1e-3) * 1e-12}
    dom = max(table, key=lambda k: table[k]["ms"])
    ach = table[dom]["tflops"]
    traffic, executed, tsrc = None, {}, None
    tp = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tp):
        try:
            tj = json.load(open(tp))
            traffic = tj.get(f"config{cfg['id']}", {}).get(dom)
            executed = tj.get(f"config{cfg['id']}_executed_flops", {})
            tsrc = tj.get("source")
        except Exception:
            traffic, executed, tsrc = None, {}, None
    for k in table:                      # executed (ncu instruction counts, profiles/) next to the algorithmic count
        if k in executed:
            table[k]["executed_tflops"] = executed[k] / (table[k]["ms"] * 1e-3) * 1e-12
    roof = {"bound": "alu", "kernel": dom, "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach / peak_tf,
            "traffic": traffic, "traffic_source": tsrc,
            "achieved_executed": table[dom].get("executed_tflops"),
            "frac_executed": (table[dom]["executed_tflops"] / peak_tf) if "executed_tflops" in table[dom] else None,
            "executed_flops_per_step": sum(executed.values()) if executed else None,
            "peak_source": "FP64 DMMA issue peak measured live by sp_probe_fp64_peak (148 SMs x 64 FMA/clk x 2 x 1.965 GHz = 37.2 nominal)",
            "hbm_gbs": hbm_gbs, "hbm_source": hbm_src}
    return roof, table


def run_ours(args):
    import torch
    import torch.distributed as dist
    import synth
    from paper_1104_3408_b200 import launch_count, probe_fp64_peak

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = synth.config(args.config)
    wl = GpuWorkload(cfg, seed_offset=rank)
    peak_tf = probe_fp64_peak(0)
    hbm_gbs, hbm_src = measured_peaks()

    use_graph = not args.no_graph
    per_step = 0
    if use_graph:
        try:
            wl.time_steps(2, 1)                      # lazy initialisation outside the capture
            per_step = wl.capture()
        except Exception as ex:                      # capture unsupported: time eager launches, say so
            print(f"bench.py: CUDA graph capture failed ({ex!r}); timing eager launches", file=sys.stderr)
            use_graph = False
        torch.cuda.synchronize()
    sampler = ClockSampler(local) if rank == 0 else None
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    if use_graph:
        ms = wl.time_graph_steps(args.steps, args.warmup)
        launches = per_step * args.steps
    else:
        l0 = launch_count()
        ms = wl.time_steps(args.steps, args.warmup)
        launches = (launch_count() - l0) * args.steps // (args.steps + args.warmup)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None
    ms_all, units_all = aggregate_over_ranks(ms, wl.units * args.steps, dist if world > 1 else None)
    value = units_all / (ms_all * 1e-3)

    # end to end with host buffers (every rank, max over ranks)
    e2e_ms, h2d, d2h = wl.e2e(max(4, min(args.steps, 20)))
    e2e_ms_all, e2e_units = aggregate_over_ranks(e2e_ms, wl.units, dist if world > 1 else None)
    stages = wl.stage_times()
    nsec = max(10, args.steps // 4)                  # secondary figures: median of three short runs each
    serial_ms = sorted(wl.time_steps(nsec, 2, concurrent=False) / nsec for _ in range(3))[1]
    eager_ms = sorted(wl.time_steps(nsec, 2) / nsec for _ in range(3))[1]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    roof, table = roofline_for(cfg, stages, wl.units, peak_tf, hbm_gbs, hbm_src)
    fl = flops_per_unit(cfg)
    tot_fl = sum(fl.values())
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_all / args.steps, "serial_ms_per_step": serial_ms, "eager_ms_per_step": eager_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "parallelism": f"replicas x{world} (independent shells, no collective)",
                   "streams": "gradient and filter of a step are issued on two CUDA streams (independent calls on the same input); "
                              "serial_ms_per_step is the same step on one stream",
                   "launch": ("CUDA graphs captured from the two library calls: rounds of one step per input copy (gradient chain and "
                              "filter chain on two streams, joined at the end of the round), remainder by single-step graphs; "
                              "eager_ms_per_step is the same two-stream stepping launched eagerly") if use_graph
                             else "eager launches",
                   "l2": f"inputs rotate over {wl.nsets} distinct state copies ({wl.nsets * wl.u_host.nbytes / 1e6:.0f} MB > 126 MB L2); "
                         f"each step also streams {4 * wl.u_host.nbytes / 1e6:.0f} MB of outputs and the workspaces"},
        "clocks": clocks,
        "e2e": {"value": e2e_units / (e2e_ms_all * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms_all},
        "gpu_launches": int(launches),
        "roofline": roof,
        "path": {"algorithmic_flops_per_unit": tot_fl, "tflops": tot_fl * wl.units / (ms / args.steps * 1e-3) * 1e-12,
                 "frac_of_fp64_peak": tot_fl * wl.units / (ms / args.steps * 1e-3) * 1e-12 / peak_tf,
                 "hbm_min_bytes_per_unit": 48, "stages": table,
                 "executed_tflops": (roof["executed_flops_per_step"] / (ms / args.steps * 1e-3) * 1e-12)
                 if roof.get("executed_flops_per_step") else None,
                 "note": "algorithmic = dense products as the paper defines them (SURVEY.md 8(d)); executed = FP64 instructions counted "
                         "by ncu (profiles/): the reflection folds execute fewer flops than the algorithmic count"},
        "fp64_peak_tflops": {"dmma": peak_tf, "dfma": probe_fp64_peak(1)},
        "kernel_variants": wl.sh.tuning(),
    }
    line["calls"] = wl.calls_report(max(10, args.steps // 4), peak_tf)
    wl_units = wl.units
    if not args.no_others and world == 1:
        others = {}
        for cid in (2, 3, 4, 5):
            if cid == args.config:
                continue
            try:
                del wl
            except NameError:
                pass
            torch.cuda.empty_cache()
            c2 = synth.config(cid)
            w2 = GpuWorkload(c2)
            k2 = {2: 200, 3: 100, 4: 20, 5: 100}[cid]

            def timed(w, k, warm):                   # same launch mode as the headline
                if use_graph:
                    w.time_steps(2, 1)
                    w.capture()
                    return w.time_graph_steps(k, warm)
                return w.time_steps(k, warm)
            m2 = timed(w2, k2, 3)
            st2 = w2.stage_times()
            r2, t2 = roofline_for(c2, st2, w2.units, peak_tf, hbm_gbs, hbm_src)
            f2 = sum(flops_per_unit(c2).values())
            others[f"config{cid}"] = {"workload": workload_name(c2), "value": w2.units * k2 / (m2 * 1e-3), "ms_per_step": m2 / k2,
                                      "path_frac_of_fp64_peak": f2 * w2.units / (m2 / k2 * 1e-3) * 1e-12 / peak_tf,
                                      "dominant": r2["kernel"], "dominant_frac": r2["frac"],
                                      "stages_ms": {k: v["ms"] for k, v in t2.items()}}
            others[f"config{cid}"]["calls"] = w2.calls_report(max(10, k2 // 4), peak_tf)
            if cid in (2, 5):  # these states fit L2: the figure above rotates inputs (HBM-cold); this one re-reads one copy
                from paper_1104_3408_b200 import launch_count
                l0 = launch_count()
                w2.step()
                nl = launch_count() - l0
                torch.cuda.synchronize()
                others[f"config{cid}"]["launches_per_step"] = nl
                # the gradient chain and the filter chain run side by side: the floor is the longer chain (about half the launches)
                others[f"config{cid}"]["latency_floor_ms"] = {"all_launches_in_one_chain": w2.latency_floor_ms(nl),
                                                              "half_of_them_per_chain": w2.latency_floor_ms((nl + 1) // 2)}
                w2.nsets = 1
                others[f"config{cid}"]["ms_per_step_l2_warm"] = timed(w2, k2, 3) / k2
            if cid == 5:      # the configuration's own workload: 200 RK4 steps with the Yn filter after every substep
                from paper_1104_3408_b200.wave import WaveRK4, wave_dt
                uw = torch.from_numpy(synth.wave_exact(c2, 0.0)).cuda()
                rk = WaveRK4(w2.sh, c2["tensors"])
                dt = wave_dt(c2["Nr"], c2["Nt"], c2["Np"], c2["rmin"], c2["rmax"])
                rk.evolve(uw.clone(), dt, 5)
                torch.cuda.synchronize()
                ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                ev0.record()
                rk.evolve(uw, dt, 200)
                ev1.record()
                torch.cuda.synchronize()
                msw = ev0.elapsed_time(ev1)
                others["config5"]["rk4_200_steps_ms"] = msw
                ug = torch.from_numpy(synth.wave_exact(c2, 0.0)).cuda()
                rk.evolve(ug, dt, 2, graph=True)                 # captures the step for this state array
                ug.copy_(torch.from_numpy(synth.wave_exact(c2, 0.0)))
                torch.cuda.synchronize()
                ev0.record()
                rk.evolve(ug, dt, 200, graph=True)
                ev1.record()
                torch.cuda.synchronize()
                msg = ev0.elapsed_time(ev1)
                others["config5"]["rk4_200_steps_graph_ms"] = msg
                others["config5"]["rk4_steps_per_s"] = 200.0 / (min(msw, msg) * 1e-3)
            wl = w2
        line["other_configs"] = others
        try:
            line["ghg_single_black_hole"] = ghg_e1_leg()
        except Exception as ex:                       # the widened path must never cost the headline line
            line["ghg_single_black_hole"] = {"error": repr(ex)}
    if not args.no_cpu_baseline and world == 1:
        threads = os.cpu_count() or 1
        pu, wall, desc = oracle_sample(cfg, synth.make_state(cfg), threads)
        pu1, _, _ = oracle_sample(cfg, synth.make_state(cfg), 1)
        line["cpu_baseline"] = {"value": 1.0 / pu, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc,
                                "seconds": wall, "value_1_thread": 1.0 / pu1}
        # the paper's own CPU formulation of the derivative (dgemm + transposes, double precision), 1 thread and all threads
        uh = synth.make_state(cfg)
        paper_style_cpu_gradient(cfg, uh, threads)
        t1 = min(paper_style_cpu_gradient(cfg, uh, 1)[0] for _ in range(2))
        tn = min(paper_style_cpu_gradient(cfg, uh, threads)[0] for _ in range(2))
        line["cpu_paper_style"] = {
            "what": "gradient only: numpy/BLAS dgemm per direction with explicit transposes (PAPER.md:135-168), double precision",
            "unit": "grid-point*fields/s (gradient call alone; compare with calls.gradient.value)",
            "value_1_thread": wl_units / t1, "value_all_threads": wl_units / tn, "cores": threads,
            "paper_context": "PAPER.md Tab. 4: GTX580 vs one i7-870 core 10.0x / 16.7x / 21.8x for the whole time step"}
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def self_launch(args):
    """`python bench.py --gpus N` without torchrun: start the N ranks ourselves (one process per GPU, the launch line the
    contract gives for the driver) and return the launcher's exit code.  Rank 0 of the child job prints the JSON line."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.run(cmd).returncode


def main():
    args = parse()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return self_launch(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.leg == "convergence":
        print(json.dumps({"leg": "radial_convergence", **convergence_leg()}))
        return 0
    if args.leg == "fft":
        print(json.dumps({"leg": "fft_comparison", **fft_comparison_leg()}))
        return 0
    if args.leg == "filters":
        print(json.dumps({"leg": "filter_comparison", **filter_comparison_leg(args.t_end)}))
        return 0
    if args.leg in ("ghg", "ghg_rhs"):           # ghg_rhs: only the right-hand side on the config-3 grid (for profiling)
        print(json.dumps({"leg": "ghg_single_black_hole", **ghg_e1_leg(evolve=args.leg == "ghg")}))
        return 0
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
