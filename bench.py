#!/usr/bin/env python
"""bench.py — OCI unknown-updates/s and time-to-converge per time step on one B200 (BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: one `oci_step`
(c_fix, all OCI iterations to tol 1e-10 on the scalar flux with the device-side stop, commit) of
the headline workload, config 3 of BASELINE.json (S32, 131,072 cells: the largest in unknowns, the
shared-block tensor path).  The other configs are parity-test cases; a compact per-config table
(OCI and the GPU SI comparator, S4..S128) rides along in `per_config` because the metric is quoted
"S4-S128", but the headline `value` is config 3 (or --config).

Timing: W untimed warm-up steps, state reset to the initial condition (untimed), then exactly K
steps between CUDA events on the library's stream, barrier + synchronize on both sides, max over
ranks.  The working set (three 128 MiB arrays) is larger than the 126 MB L2.

--gpus N (under torchrun, one rank per GPU): row f4, ONE slab of N x 131,072 cells sharded by contiguous cell
ranges (weak scaling); the edge half rows and the two norms of the stopping rule travel per iteration as peer-memory
stores (csrc/shard_exchange.cu), NCCL is only used for the rendezvous and the timing barrier.

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded
sample of the same workload; see DESIGN.md "Measurement".
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
sys.path.insert(0, ROOT)

from workloads import make_problem, make_multi_region  # noqa: E402

METRIC = "oci_unknown_updates_per_s"
UNIT = "unknown-updates/s"

def load_traffic(cfg, reduced, suffix=""):
    """DRAM bytes per iteration of the dominant kernel from the committed `ncu --set full` capture: profiles/traffic.json,
    written by `python -m paper_2305_13555_b200.ncu_traffic` from the .ncu-rep together with the commit the capture was
    taken at, so that a stale capture is visible next to the number."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(path):
        return None, None
    with open(path) as f:
        t = json.load(f)
    e = t.get("entries", {}).get(f"cfg{cfg}_{'reduced' if reduced else 'full'}{suffix}")
    if not e:
        return None, None
    return e["dram_bytes_per_iteration"], {"file": "profiles/traffic.json", "capture": e.get("capture"), "kernel": e.get("kernel"),
                                           "captured_at_commit": e.get("commit")}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region (B200_PROFILING.md recipe).  The timed
    region is only milliseconds long, so NVML is polled in-process from a thread (every ~2 ms);
    `nvidia-smi -lms` is the fallback when the NVML binding is missing."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index):
        self.index, self.sm, self.bits, self.power = index, [], 0, []
        self.stop_flag, self.thread, self.proc, self.lines, self.h, self.nv = False, None, None, [], None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                ent = vis.split(",")[index].strip()
                phys = int(ent) if ent.isdigit() else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.nv = pynvml
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.h = None

    def _poll(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.bits |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(0.002)

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def start(self):
        self.stop_flag = False
        if self.h is not None:
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def pause(self):
        """Stop sampling (end of a timed region); start() resumes and keeps accumulating."""
        self.stop_flag = True
        if self.h is not None and self.thread:
            self.thread.join(timeout=1)
            self.thread = None
        elif self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
            self._parse_smi()
            self.proc = None

    def _parse_smi(self):
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        inv = {v: k for k, v in self.REASONS.items()}
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                self.sm.append(float(f[0]))
                self.max_mhz = float(f[1])
                self.power.append(float(f[2]))
            except ValueError:
                continue
            for nm, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    self.bits |= inv[nm]
        self.lines = []

    def result(self, note=""):
        if self.h is None and not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": ["clock sampling unavailable"]}
        reasons = sorted(nm for bit, nm in self.REASONS.items() if self.bits & bit)
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": getattr(self, "max_mhz", None),
                "samples": len(self.sm), "power_w_max": max(self.power) if self.power else None,
                "reasons": reasons, "how": ("NVML polled in-process" if self.h is not None else "nvidia-smi -lms 20") + note}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# ------------------------------------------------------------------------------------------ oracle arm
def oracle_sample_problem(cfg):
    """A bounded sample of config `cfg` for the CPU oracle (about 10-30 s of CPU work per run on 16 cores): config 3
    (the bench default) runs at FULL size, the O(N^2)-per-cell configs 4 and 5 on their first 2048 / 512 cells."""
    sample = {1: None, 2: None, 3: None, 4: 2048, 5: 512}[cfg]
    p = make_problem(cfg, cells=sample)
    desc = (f"config {cfg} at full size" if sample is None else
            f"config {cfg} with the first {sample} of {FULL_CELLS[cfg]} cells (same materials, angles, dt, BCs)")
    return p, desc


FULL_CELLS = {1: 20, 2: 1000, 3: 131072, 4: 16384, 5: 4096}


def time_oracle(cfg, steps, warmup, threads, scheme="oci", cells=None):
    from oracle import Oracle
    p, desc = oracle_sample_problem(cfg)
    if cells is not None and cells < p.cells:
        p = make_problem(cfg, cells=cells)
        desc = f"config {cfg} with the first {cells} of {FULL_CELLS[cfg]} cells (same materials, angles, dt, BCs)"
    o = Oracle.from_problem(p, threads=threads)
    step = o.oci_step if scheme == "oci" else o.si_step
    for k in range(warmup):
        o.set_source(p.source(k))
        step(p.tol, p.max_iters)
    o.set_flux(p.psi0)
    updates, iters = 0, []
    t0 = time.perf_counter()
    for k in range(steps):
        o.set_source(p.source(k))
        st, it, _ = step(p.tol, p.max_iters)
        updates += p.unknowns * it
        iters.append(it)
    dt = time.perf_counter() - t0
    return dict(value=updates / dt, seconds=dt, iters=iters,
                sample=f"{desc}, {steps} time steps, {scheme.upper()} to tol {p.tol:g}, {threads} thread(s)",
                ms_per_step=dt / steps * 1e3, cells=p.cells)


def oracle_legs(cfg, threads):
    """SURVEY 8(d) "Oracle timing": the oracle as it stands, OCI and SI, on (i) one thread and (ii) all host cores
    (threads over cells for OCI, over angles for SI, as the paper's CPU runs).  The one-thread legs use a
    quarter of the sample and one step so that the whole baseline stays within tens of seconds."""
    p, _ = oracle_sample_problem(cfg)
    small = max(1, p.cells // 4) if cfg in (3, 4, 5) else None
    steps = 3 if cfg == 3 else 2 if cfg in (4, 5) else 5
    legs = {}
    for scheme in ("oci", "si"):
        legs[f"{scheme}_all_cores"] = time_oracle(cfg, steps, 0, threads, scheme)
        legs[f"{scheme}_1_thread"] = time_oracle(cfg, 1 if cfg in (3, 4, 5) else steps, 0, 1, scheme, cells=small)
    return legs


class CpuBlasReduced:
    """A TUNED CPU restatement of the algorithm the GPU arm runs, for a fair CPU figure next to the (deliberately
    plain) oracle: shared block, the block inverse formed once with LAPACK, and the interface-reduced iteration of
    DESIGN.md 6.7 - y^(l+1) = yfix + inc G^T, phi^(l+1) = phifix + inc H^T - as two threaded BLAS dgemms per
    iteration at the FULL cell count.  The state is kept PACKED the whole time ([O | I] columns, each run a contiguous
    slice: no strided or fancy-indexed passes inside a step), the work arrays are allocated once and the dgemms write
    in place.  The matrix B comes from the oracle's `cell_matrix` (this is bench.py's CPU leg, the one place outside
    tests/ that may call oracle/); everything else is numpy.  Not used for parity."""

    def __init__(self, p):
        from oracle import cell_matrix, gauss_legendre
        assert np.all(p.dx == p.dx[0]) and np.all(p.sigma_t == p.sigma_t[0]) and np.all(p.sigma_s == p.sigma_s[0])
        self.p, N, J = p, p.n_angles, p.cells
        self.mu, self.w = gauss_legendre(N)
        h, hN = float(p.dx[0]), N // 2
        Binv = np.linalg.inv(cell_matrix(self.mu, self.w, h, float(p.sigma_t[0]), float(p.sigma_s[0]), p.v, p.dt))
        m = np.arange(N)
        neg, pos = m[self.mu < 0], m[self.mu > 0]
        assert np.array_equal(neg, m[:hN]) and np.array_equal(pos, m[hN:])      # ascending Gauss-Legendre set
        # I: rows that receive an incident flux, ordered [k | k+1/2 of mu < 0, k | k+1/2 of mu > 0] so that the gather
        # of the neighbours' values is two contiguous half-row slices; O = the partner slots a neighbour reads.
        # Every run of hN columns of [O | I] is (one sign of mu, one slot); runs 2r and 2r+1 are slots k and k+1/2.
        self.I = np.concatenate([4 * neg + 1, 4 * neg + 3, 4 * pos + 0, 4 * pos + 2])
        self.O = self.I ^ 1
        self.perm = np.concatenate([self.O, self.I])
        self.nr = N                                                  # columns [0, nr) of inc: the value comes from cell j+1
        amu = np.abs(self.mu[self.I >> 2])
        W = np.zeros((4, 4 * N))
        for s_ in range(4):
            W[s_, 4 * m + s_] = self.w
        self.G = np.ascontiguousarray((Binv[np.ix_(self.O, self.I)] * amu).T)        # [2N][2N], applied as inc @ G
        self.H = np.ascontiguousarray(((W @ Binv)[:, self.I] * amu).T)               # [2N][4]
        self.F = np.ascontiguousarray((Binv[np.ix_(self.I, self.I)] * amu).T)        # [2N][2N], the FINAL pass
        # phi rides along as four more columns of the iteration operator and of the FIX operator: one dgemm each
        self.GH = np.ascontiguousarray(np.hstack([self.G, self.H]))                  # [2N][2N + 4]
        WB = (W @ Binv)[:, self.perm]
        self.Bp = np.ascontiguousarray(np.vstack([Binv[np.ix_(self.O, self.perm)], WB,
                                                  Binv[np.ix_(self.I, self.perm)]]).T)   # packed c_fix -> [O | phi | I]
        self.W, self.alpha, self.h = W, h / (2 * p.v * p.dt), h
        where = {(int(i) >> 2, (int(i) >> 1) & 1): k for k, i in enumerate(self.I)}
        self.mirror = np.array([where[(N - 1 - (int(i) >> 2), (int(i) >> 1) & 1)] for i in self.I])
        psi = np.empty((J, N, 4))
        psi[:, :, 0] = psi[:, :, 2] = p.psi0[:, :, 0]
        psi[:, :, 1] = psi[:, :, 3] = p.psi0[:, :, 1]
        psi = psi.reshape(J, 4 * N)
        # [O columns | phi], ghost rows 0 and J+1
        self.Y, self.Ynew = np.zeros((J + 2, 2 * N + 4)), np.zeros((J + 2, 2 * N + 4))
        self.Ip = np.ascontiguousarray(psi[:, self.I])                            # I columns
        self.Y[1:-1, :2 * N] = psi[:, self.O]
        self.Y[1:-1, 2 * N:] = psi @ W.T
        # work arrays, allocated once
        self.cfix, self.fix = np.zeros((J, 4 * N)), np.empty((J, 4 * N + 4))
        self.inc, self.dphi = np.empty((J, 2 * N)), np.empty((J, 4))

    @property
    def phi(self):
        return self.Y[1:-1, 2 * self.p.n_angles:]

    @property
    def Psi(self):
        """The angular flux [J][4N] in the library's layout (unpacked on demand)."""
        out = np.empty((self.p.cells, 4 * self.p.n_angles))
        out[:, self.O], out[:, self.I] = self.Y[1:-1, :2 * self.p.n_angles], self.Ip
        return out

    def _ghosts(self):
        p, Y = self.p, self.Y
        for side, bc, row, src in ((0, p.bc_left, 0, 1), (1, p.bc_right, -1, -2)):
            if bc[0] == 2:
                Y[row, :self.mirror.size] = Y[src][self.mirror]
            else:
                Y[row, :self.mirror.size] = bc[1] if bc[0] == 1 else 0.0

    def step(self, q, tol, max_iters):
        p, J, N, nr, hN = self.p, self.p.cells, self.p.n_angles, self.nr, self.p.n_angles // 2
        cfix, fix, inc, dphi = self.cfix, self.fix, self.inc, self.dphi
        # c_fix in packed columns: rows (k, .) take alpha * the committed k+1/2 value of the same angle, plus (h/4) Q
        c4 = cfix.reshape(J, 4, 2, hN)
        for r_ in range(2):
            np.multiply(self.Y[1:-1, (2 * r_ + 1) * hN:(2 * r_ + 2) * hN], self.alpha, out=c4[:, r_, 0, :])
        np.multiply(self.Ip.reshape(J, 2, 2, hN)[:, :, 1, :], self.alpha, out=c4[:, 2:4, 0, :])
        c4[:, :, 1, :] = 0.0
        if q is not None:
            cfix += np.take(0.25 * self.h * np.asarray(q), self.perm & 3, axis=1)
        np.matmul(cfix, self.Bp, out=fix)                              # [yfix | phifix | ifix], once per step
        yfix, ifix = fix[:, :2 * N + 4], fix[:, 2 * N + 4:]
        it, d, r = 0, 0.0, 0.0
        while it < max_iters:
            self._ghosts()
            inc[:, :nr] = self.Y[2:, :nr]
            inc[:, nr:] = self.Y[:-2, nr:2 * N]
            ynew = self.Ynew[1:-1]
            np.matmul(inc, self.GH, out=ynew)
            ynew += yfix
            phinew = ynew[:, 2 * N:]
            np.subtract(phinew, self.phi, out=dphi)
            d, r = max(dphi.max(), -dphi.min()), max(phinew.max(), -phinew.min())
            self.Y, self.Ynew = self.Ynew, self.Y
            it += 1
            if tol >= 0 and d <= tol * r:
                break
        # the I rows of the converged iterate from the last gathered inc (the FINAL pass)
        np.matmul(inc, self.F, out=self.Ip)
        self.Ip += ifix
        return it


def time_cpu_blas(cfg, steps):
    """Unknown-updates/s of the tuned CPU restatement (CpuBlasReduced) at the config's FULL size; None for per-cell
    configs (a batched GEMV over 2 GiB of inverses is not a BLAS-3 problem)."""
    if cfg == 5:
        return None
    p = make_problem(cfg)
    c = CpuBlasReduced(p)
    c.step(p.source(0), p.tol, p.max_iters)                            # warm-up (BLAS thread pool, page faults)
    updates, t0 = 0, time.perf_counter()
    for k in range(1, 1 + steps):
        updates += p.unknowns * c.step(p.source(k), p.tol, p.max_iters)
    dt = time.perf_counter() - t0
    try:
        import threadpoolctl
        th = max([i.get("num_threads", 1) for i in threadpoolctl.threadpool_info()] + [1])
    except Exception:
        th = os.cpu_count()
    return {"value": updates / dt, "unit": UNIT, "ms_per_step": dt / steps * 1e3, "threads": th, "cells": p.cells,
            "kind": "numpy + threaded BLAS, pre-inverted block, interface-reduced iteration (same algorithm as the GPU arm), full size"}


def run_reference(args):
    """The base contract's reference arm = the oracle as it stands on the host cores: EXACTLY --steps timed steps after
    --warmup untimed ones, each on a bounded sample of the config (oracle_sample_problem; one calibration step first, and
    the sample shrinks if the whole run would not end within a few minutes)."""
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    from oracle import threads_available
    threads = threads_available()
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    p, _ = oracle_sample_problem(args.config)
    cells = p.cells
    need = time_oracle(args.config, 1, 0, threads)["seconds"] * (steps + warmup)
    budget = 150.0
    if need > budget:
        cells = max(16, int(cells * budget / need) // 16 * 16)
    r = time_oracle(args.config, steps, warmup, threads, cells=cells)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": make_problem(args.config, cells=1).name},
        "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": threads, "kind": "oracle", "sample": r["sample"]},
        "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "iters_per_step": r["iters"],
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------ GPU arm
def time_gpu_steps(torch, g, p, steps, scheme, sampler=None, barrier=None):
    """Reset to the IC (untimed), then time exactly `steps` steps with CUDA events on the library's
    (= torch's current) stream.  `g`: an OCI context or a ShardedOCI.  Returns (ms, iters, per-step ms)."""
    sharded = hasattr(g, "shards")
    if sharded:
        g.set_flux_from_problem()
    else:
        g.set_flux(p.psi0)
    qdev = {}
    if not sharded:
        for k in range(steps):                  # inputs resident in HBM before the timed region
            q = p.source(k)
            if q is not None and id(q) not in qdev:
                qdev[id(q)] = torch.from_numpy(np.ascontiguousarray(q)).cuda()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    if barrier:
        barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    iters = []
    ev[0].record()
    for k in range(steps):
        if sharded:
            g.set_source(k)
            st, it, _ = g.step(p.tol, p.max_iters)
        else:
            q = p.source(k)
            g.set_source_dev(qdev[id(q)] if q is not None else None)
            st, it, _ = (g.oci_step if scheme == "oci" else g.si_step)(p.tol, p.max_iters)
        iters.append(it)
        ev[k + 1].record()
    torch.cuda.synchronize()
    if sampler:
        sampler.pause()
    if barrier:
        barrier()
    return ev[0].elapsed_time(ev[-1]), iters, [ev[k].elapsed_time(ev[k + 1]) for k in range(steps)]


def time_gpu_e2e(torch, g, p, steps):
    """Same K steps through the C ABI with HOST buffers: the initial condition and every step's source are copied
    host->device from pinned memory and every step's scalar flux is read back into pinned host memory
    (oci_get_scalar_flux_async: the copy of step k's flux overlaps step k+1; oci_synchronize before the clock stops),
    all inside the timed region."""
    sharded = hasattr(g, "shards")
    ctxs = g.shards if sharded else [g]
    probs = [c.problem for c in ctxs] if sharded else [p]
    psi0 = [torch.from_numpy(np.ascontiguousarray(q.psi0)).pin_memory() for q in probs]
    qpin = {}
    for q in probs:
        for k in range(steps):
            a = q.source(k)
            if a is not None and (id(q), k) not in qpin:
                qpin[(id(q), k)] = torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    phi = [[torch.empty((q.cells, 4), dtype=torch.float64).pin_memory() for _ in range(2)] for q in probs]
    h2d = sum(t.numel() * 8 for t in psi0)
    d2h = 0
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for c, t in zip(ctxs, psi0):
        c.set_flux(t.numpy())
    updates = 0
    for k in range(steps):
        for c, q in zip(ctxs, probs):
            a = qpin.get((id(q), k))
            c.set_source(a.numpy() if a is not None else None)
            h2d += q.cells * 32 if a is not None else 0
        st, it, _ = g.step(p.tol, p.max_iters) if sharded else g.oci_step(p.tol, p.max_iters)
        updates += sum(q.unknowns for q in probs) * it
        for c, q, bufs in zip(ctxs, probs, phi):
            c.get_scalar_flux_async(bufs[k & 1])
            d2h += q.cells * 32
    for c in ctxs:
        c.synchronize()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    return updates / (ms * 1e-3), h2d / steps, d2h / steps


def iteration_roofline(P, p, info, cfg, kms, klaunch, aux, steps, peaks, peak_src, peak_live):
    """Roofline of the OCI iteration kernel against the work it EXECUTES per launch (or, for the fused
    loops, per iteration): the full apply is [n x n] per cell; the reduced iteration is
    [(2N+4) x 2N] per cell (G and the four scalar-flux rows H); its FIX pass [(4N+4) x (2N+4)] and FINAL
    pass [2N x 2N] run once per step and are listed in step_breakdown."""
    shared = info["path"] == P.PATH_SHARED
    n = info["block_dim"]
    k_avg_ms = kms / max(klaunch, 1)
    reduced = info["iteration"] == P.ITERATION_REDUCED
    K2 = n // 2
    M_op, K_op = (K2 + 4, K2) if reduced else (n, n)
    fix_ms, fix_n, fin_ms, fin_n = aux["fix_ms"], aux["fix_launches"], aux["final_ms"], aux["final_launches"]
    traffic, traffic_src = load_traffic(cfg, reduced)
    breakdown = {"iteration_kernel_ms": k_avg_ms, "iterations_per_step": klaunch / steps,
                 "fix_pass_ms_per_step": fix_ms / max(fix_n, 1) if reduced else None,
                 "final_pass_ms_per_step": fin_ms / max(fin_n, 1) if reduced else None,
                 "operator_rows_x_cols": [M_op, K_op], "form": "reduced" if reduced else "full"}
    if info["reduced_kernel"] == P.RKERNEL_WOODBURY and reduced:
        # O(N) apply: HBM-bound; algorithmic bytes = the state only, J (6N doubles of y in / yfix in /
        # y out + 96 B of scalar flux), plus 16N doubles of 4x4 pieces, a row of M and the block index with per-cell blocks
        N = n // 4
        bytes_ = p.cells * (48.0 * N + 96.0 + (0.0 if shared else 128.0 * N + 132.0))
        achieved = bytes_ / (k_avg_ms * 1e-3) * 1e-9
        traffic, traffic_src = load_traffic(cfg, reduced, "_woodbury")
        breakdown["operator_rows_x_cols"] = None
        breakdown["form"] = "reduced, rank-4 (Woodbury) apply"
        roofline = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": achieved / peaks["hbm_gbs"], "traffic": traffic, "traffic_source": traffic_src,
                    "kernel": "oci iteration through the rank-4 scattering matrix (eq. 22)", "algorithmic_bytes_per_launch": bytes_,
                    "avg_launch_ms": k_avg_ms, "launches_timed": klaunch, "peak_source": f"MEASURED_PEAKS hbm_gbs ({peak_src})"}
    elif shared:
        flops = 2.0 * M_op * K_op * p.cells
        nominal_ratio = 45.0 / 2250.0        # guide: B200 fp64 tensor 45 TF vs bf16 2250 TF nominal
        peak_scaled = peaks["bf16_tflops"] * nominal_ratio
        peak = max(peak_live, peak_scaled)
        achieved = flops / (k_avg_ms * 1e-3) * 1e-12
        roofline = {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                    "traffic": traffic, "traffic_source": traffic_src,
                    "kernel": "oci %s iteration (eq. 19), fp64 DMMA" % breakdown["form"], "algorithmic_flops_per_launch": flops,
                    "avg_launch_ms": k_avg_ms, "launches_timed": klaunch,
                    "peak_source": f"max(live DMMA issue-rate probe {peak_live:.2f}, MEASURED_PEAKS bf16 {peak_src} x 45/2250 = {peak_scaled:.2f})"}
    else:
        if reduced:   # operator + gathered half rows, yfix in, y out; phifix and old phi in, phi out
            bytes_ = p.cells * (M_op * K_op * 8.0 + 3.0 * K2 * 8.0 + 96.0)
        else:         # inverse + c_fix, 2 half rows, Psi out; phi
            bytes_ = p.cells * (n * n * 8.0 + 4.0 * n * 8.0 + 64.0)
        achieved = bytes_ / (k_avg_ms * 1e-3) * 1e-9
        roofline = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": achieved / peaks["hbm_gbs"], "traffic": traffic, "traffic_source": traffic_src,
                    "kernel": "oci %s iteration (eq. 19), batched GEMV" % breakdown["form"], "algorithmic_bytes_per_launch": bytes_,
                    "avg_launch_ms": k_avg_ms, "launches_timed": klaunch, "peak_source": f"MEASURED_PEAKS hbm_gbs ({peak_src})"}
    roofline["step_breakdown"] = breakdown
    return roofline


def per_config_table(torch, P, peaks=None, peak_src=None, peak_live=None):
    """OCI vs the GPU SI comparator for every BASELINE config (each for its own number of steps)."""
    out = {}
    for cfg in (1, 2, 3, 4, 5):
        p = make_problem(cfg)
        g = P.OCI.from_problem(p)
        row = {"S_N": p.n_angles, "cells": p.cells, "path": "shared" if g.get_info()["path"] == 0 else "per_cell",
               "setup_ms": g.get_setup_time()}
        for scheme in ("oci", "si"):
            for k in range(3):                   # warm-up
                g.set_source(p.source(k))
                (g.oci_step if scheme == "oci" else g.si_step)(p.tol, p.max_iters)
            ms, iters, each = time_gpu_steps(torch, g, p, p.n_steps, scheme)
            row[f"{scheme}_ms_per_step"] = ms / p.n_steps
            row[f"{scheme}_ms_per_step_median"] = float(np.median(each))
            row[f"{scheme}_iters"] = iters
            row[f"{scheme}_updates_per_s"] = p.unknowns * sum(iters) / (ms * 1e-3)
        row["si_over_oci_time"] = row["si_ms_per_step"] / row["oci_ms_per_step"]
        row["oci_woodbury"] = woodbury_row(torch, P, p, peaks)
        row["si_over_oci_woodbury_time"] = row["si_ms_per_step"] / row["oci_woodbury"]["ms_per_step"]
        if cfg >= 3 and peaks is not None:       # cfg 1-2 are launch-latency bound: absolutes only
            g.enable_kernel_timing(True)
            time_gpu_steps(torch, g, p, p.n_steps, "oci")
            kms, klaunch = g.get_kernel_time()
            aux = g.get_aux_kernel_time()
            g.enable_kernel_timing(False)
            r = iteration_roofline(P, p, g.get_info(), cfg, kms, klaunch, aux, p.n_steps, peaks, peak_src, peak_live)
            row["oci_iteration_roofline"] = {k: r[k] for k in ("bound", "achieved", "peak", "unit", "frac", "avg_launch_ms")}
            row["oci_step_breakdown"] = r["step_breakdown"]
        out[f"cfg{cfg}"] = row
        g.close()
        del g
        torch.cuda.empty_cache()
    out["multi_region"] = multi_region_row(torch, P)
    return out


def multi_region_row(torch, P):
    """Context beside the five configs: a multi-region slab of the kind the paper times (Reed-type, S64, v = 4,
    dt = 1, 5 steps; synthetic layout, workloads.make_multi_region): a handful of materials on the K-tiled tensor-core
    kernels (row f2), the same through the Woodbury family, and the GPU SI scan.  Time per step and iterations only.
    Thin cells and a void are the one-cell inversion's worst case (rho_OCI -> 1 as Sigma dx -> 0; information
    crosses the void one cell per iteration), so OCI needs hundreds to thousands of iterations here where SI needs tens:
    the paper's own Table 1 has OCI losing on this kind of problem on the CPU."""
    p = make_multi_region(cells=1024)
    row = {"workload": p.name, "S_N": p.n_angles, "cells": p.cells}
    for name, kw, scheme in (("oci", {}, "oci"), ("oci_woodbury", {"reduced_kernel": P.RKERNEL_WOODBURY}, "oci"), ("si", {}, "si")):
        g = P.OCI.from_problem(p, **kw)
        if name == "oci":
            row["n_blocks"] = g.get_info()["n_blocks"]
            row["reduced_kernel"] = g.get_info()["reduced_kernel"]
        for k in range(2):
            g.set_source(p.source(k))
            (g.oci_step if scheme == "oci" else g.si_step)(p.tol, p.max_iters)
        ms, iters, each = time_gpu_steps(torch, g, p, p.n_steps, scheme)
        row[f"{name}_ms_per_step"] = ms / p.n_steps
        row[f"{name}_iters"] = iters
        g.close()
    return row


def woodbury_row(torch, P, p, peaks):
    """The same time steps with the O(N) apply through the rank-4 scattering matrix (row f3, second half; selected with
    oci_set_reduced_kernel): time to converge, and the iteration kernel against the HBM roofline - its algorithmic bytes
    per iteration are the state only, J (6N doubles of y in / yfix in / y out + 96 B of scalar flux), plus 16N doubles of
    4x4 pieces, one row of M and the block index per cell when every cell has its own block."""
    g = P.OCI.from_problem(p, reduced_kernel=P.RKERNEL_WOODBURY)
    for k in range(3):
        g.set_source(p.source(k))
        g.oci_step(p.tol, p.max_iters)
    ms, iters, each = time_gpu_steps(torch, g, p, p.n_steps, "oci")
    g.enable_kernel_timing(True)
    time_gpu_steps(torch, g, p, p.n_steps, "oci")
    kms, klaunch = g.get_kernel_time()
    aux = g.get_aux_kernel_time()
    g.enable_kernel_timing(False)
    N = p.n_angles
    per_cell = g.get_info()["path"] == P.PATH_PER_CELL
    bytes_ = p.cells * (48.0 * N + 96.0 + ((128.0 * N + 132.0) if per_cell else 0.0))
    k_avg = kms / max(klaunch, 1)
    out = {"ms_per_step": ms / p.n_steps, "ms_per_step_median": float(np.median(each)), "iters": iters,
           "updates_per_s": p.unknowns * sum(iters) / (ms * 1e-3), "iteration_kernel_ms": k_avg,
           "fix_pass_ms_per_step": aux["fix_ms"] / max(aux["fix_launches"], 1),
           "final_pass_ms_per_step": aux["final_ms"] / max(aux["final_launches"], 1)}
    if peaks is not None and p.cfg >= 3:
        ach = bytes_ / (k_avg * 1e-3) * 1e-9
        out["iteration_roofline"] = {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
                                     "algorithmic_bytes_per_iteration": bytes_}
    g.close()
    return out


def aggregate_over_ranks(torch, ms, amount, device):
    """Whole-job figures for N independent replicas: time = MAX over ranks, amount
    (updates, or a per-rank rate) = SUM over ranks.  `device` None = single process."""
    if device is None:
        return float(ms), float(amount)
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    u = torch.tensor([float(amount)], dtype=torch.float64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def run_ours(args):
    import torch
    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        print(json.dumps({"error": "no CUDA device; this benchmark has no CPU fallback"}))
        return 1
    torch.cuda.set_device(local)
    import paper_2305_13555_b200 as P
    barrier = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
        barrier = dist.barrier

    if args.si_only:
        # the comparator alone (rows d1-d3): the SI steps of one config, nothing else - for launch lists and profiles
        p = make_problem(args.config)
        g = P.OCI.from_problem(p, device=f"cuda:{local}")
        for k in range(args.warmup):
            g.set_source(p.source(k))
            g.si_step(p.tol, p.max_iters)
        l0 = g.launch_count()
        ms, iters, each = time_gpu_steps(torch, g, p, args.steps, "si")
        print(json.dumps({"metric": "si_time_to_converge_ms_per_step", "value": ms / args.steps, "unit": "ms", "higher_is_better": False,
                          "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step_median": float(np.median(each)),
                          "iters_per_step": iters, "si_unknown_updates_per_s": p.unknowns * sum(iters) / (ms * 1e-3),
                          "gpu_launches": int(g.launch_count() - l0), "dtype": "f64", "data": "synthetic",
                          "config": {"workload": p.name, "S_N": p.n_angles, "cells": p.cells, "tol": p.tol, "scheme": "source iteration"}}))
        g.close()
        return 0

    peaks, peak_src = load_peaks()
    if world > 1:
        # row f4: ONE slab of world x (config's cells), sharded by contiguous cell ranges (weak scaling)
        from paper_2305_13555_b200.sharding import ShardedOCI
        p = make_problem(args.config, cells=FULL_CELLS[args.config] * world)
        g = ShardedOCI.distributed(p, device=f"cuda:{local}")
        ctx = g.shards[0]

        def warm_step(k):
            g.set_source(k)
            g.step(p.tol, p.max_iters)
    else:
        p = make_problem(args.config)
        g = ctx = P.OCI.from_problem(p, device=f"cuda:{local}", reduced_kernel=P.RKERNEL_WOODBURY if args.family == "woodbury" else None)

        def warm_step(k):
            g.set_source(p.source(k))
            g.oci_step(p.tol, p.max_iters)
    info = ctx.get_info()
    shared = info["path"] == P.PATH_SHARED
    n = info["block_dim"]
    p_local = ctx.problem if world > 1 else p

    for k in range(args.warmup):                # warm-up steps (untimed)
        warm_step(k)

    # ---- headline: K steps, inputs resident in HBM
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = ctx.launch_count()
    ms, iters, each = time_gpu_steps(torch, g, p, args.steps, "oci", sampler, barrier)
    launches = ctx.launch_count() - l0
    updates = p.unknowns * sum(iters)           # the whole slab: every rank advances its share of it
    if world > 1:
        ms, _ = aggregate_over_ranks(torch, ms, 0.0, "cuda")
        each = [aggregate_over_ranks(torch, t, 0.0, "cuda")[0] for t in each]
    value = updates / (ms * 1e-3)

    # ---- the dominant kernel alone (events around every OCI apply launch, same steps again)
    ctx.enable_kernel_timing(True)
    time_gpu_steps(torch, g, p, args.steps, "oci", sampler, barrier)
    clocks = sampler.result(" during the headline and the per-kernel timed regions") if sampler else None
    kms, klaunch = ctx.get_kernel_time()
    aux = ctx.get_aux_kernel_time()
    ctx.enable_kernel_timing(False)
    peak_live = P.probe_fp64_tensor_tflops(f"cuda:{local}") if shared and args.family != "woodbury" else None
    roofline = iteration_roofline(P, p_local, info, args.config, kms, klaunch, aux, args.steps, peaks, peak_src, peak_live)
    reduced = info["iteration"] == P.ITERATION_REDUCED

    # ---- end to end through the C ABI with host buffers
    if barrier:
        barrier()
    e2e_val, h2d, d2h = time_gpu_e2e(torch, g, p, args.steps)
    if world > 1:
        # every rank measured the whole slab's updates over its own clock: the job's figure is the slowest rank's
        t = torch.tensor([e2e_val], dtype=torch.float64, device="cuda")
        torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MIN)
        e2e_val = float(t.item())
        _, h2d = aggregate_over_ranks(torch, 0.0, h2d, "cuda")
        _, d2h = aggregate_over_ranks(torch, 0.0, d2h, "cuda")
    setup_ms = ctx.get_setup_time()
    g.close()
    del g
    torch.cuda.empty_cache()

    # arrays a step streams: reduced form y (x2), z, yfix, ifix of J x 2N doubles each (+ one operator per cell on
    # the per-cell path); full form the two Psi buffers and c_fix
    ws = p_local.unknowns * 4.0 * 5 if reduced else p_local.unknowns * 8.0 * 3
    if not shared:
        ws += p_local.cells * (n // 2 + 4) * (n // 2) * 8.0 if reduced else p_local.cells * n * n * 8.0
    l2_note = ("working set of a step %.0f MiB per GPU, larger than the 126 MB L2" % (ws / 2**20) if ws > 126e6 else
               "working set of a step %.1f MiB fits L2 and is not flushed between steps (launch-latency-bound config)" % (ws / 2**20))
    if rank == 0:
        per_cfg = (per_config_table(torch, P, peaks, peak_src, peak_live or P.probe_fp64_tensor_tflops(f"cuda:{local}"))
                   if (world == 1 and not args.no_table) else None)
        cpu = None
        if world == 1 and not args.no_cpu:
            from oracle import threads_available
            th = threads_available()
            legs = oracle_legs(args.config, th)
            r = legs["oci_all_cores"]
            cpu = {"value": r["value"], "unit": UNIT, "cores": th, "kind": "oracle", "sample": r["sample"],
                   "ms_per_step_on_sample": r["ms_per_step"], "sample_cells": r["cells"],
                   "legs": {k: {"value": v["value"], "ms_per_step_on_sample": v["ms_per_step"], "sample": v["sample"], "iters": v["iters"]}
                            for k, v in legs.items()},
                   "tuned_same_algorithm": time_cpu_blas(args.config, 2)}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "ms_per_step_median": float(np.median(each)), "ms_per_step_each": each,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": p.name, "S_N": p.n_angles, "cells": p.cells, "unknowns": p.unknowns, "tol": p.tol,
                       "path": "shared" if shared else "per_cell",
                       "kernel_family": "dense (the library default)" if args.family == "default" else "woodbury (rank-4 apply, on request)",
                       "parallelism": (f"one slab sharded over {world} GPUs by cell ranges ({p_local.cells} cells each), halo + norm exchange "
                                       "by peer-memory stores per iteration" if world > 1 else "1 gpu"),
                       "l2": l2_note},
            "iters_per_step": iters, "time_to_converge_ms_per_step": ms / args.steps, "setup_ms": setup_ms,
            "roofline": roofline, "cpu_baseline": cpu,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": int(launches), "clocks": clocks, "per_config": per_cfg,
        }
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-table", action="store_true", help="skip the per-config OCI/SI table")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--si-only", action="store_true", help="time only the GPU SI comparator on --config (one small JSON line; for profiles)")
    ap.add_argument("--family", default="default", choices=["default", "woodbury"],
                    help="kernel family of the timed arm: the library default (dense inverse, the headline) or the O(N) rank-4 apply")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
