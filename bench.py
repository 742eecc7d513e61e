#!/usr/bin/env python
"""Benchmark of the B200-native complex CCSD hot path (BASELINE.json metric: CCSD s/iteration and pp-ladder FP64
TFLOP/s as % of the B200 FP64 peak, 1 GPU).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg3|cfg2|cfg1|cfg0] [--no-sweep]
    python bench.py --impl reference ...        # the CPU oracle, timed on the host cores (bounded sample)

One "step" = one ccsd_iterate: the whole hot path (eqs 23-33, Jacobi + DIIS update, energy) on one set of synthetic
inputs (ccsd_inputs.py, recipe in DESIGN.md).  `value` is measured with the tensors resident in HBM; `e2e` adds the
host->device copy of the amplitudes from pinned memory and the device->host copy of the new amplitudes + energy
every step.  The path does not shard (north_star: one GPU, no collectives): N > 1 runs N independent replicas.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

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

import numpy as np  # noqa: E402

import ccsd_inputs as ci  # noqa: E402

FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 * 1e-12   # 148 SMs x 64 FMA/clk x 2 x 1.965 GHz = 37.2
# dram__bytes_read.sum + dram__bytes_write.sum of ONE pp-ladder launch of the 3M + sum-plane DMMA GEMM at cfg3, from
# profiles/r02_ncu_pp_ladder_cfg3.md (ncu --set full).  None until captured for the workload.
NCU_TRAFFIC_BYTES = {"cfg3": 23.10e9 + 0.220e9}
# ... and of the batched launch the pp-ladder is with its Strassen levels: {levels: {workload: bytes}}
# (profiles/r02b_ncu_pp_ladder_strassen_cfg3.md: one level, 7 products; profiles/r02c_ncu_pp_ladder_strassen_cfg3.md: two levels, 49)
NCU_TRAFFIC_BYTES_STRASSEN = {1: {"cfg3": 30.472e9 + 0.389e9}, 2: {"cfg3": 49.517e9 + 0.687e9}}
NCU_TRAFFIC_FILE_STRASSEN = {1: "r02b_ncu_pp_ladder_strassen_cfg3.md", 2: "r02c_ncu_pp_ladder_strassen_cfg3.md"}
NCU_TRAFFIC_SOURCE = ("recorded constant, not measured in this run: dram__bytes_read.sum + dram__bytes_write.sum of one "
                      "pp-ladder launch from the ncu --set full capture summarised in profiles/r02_ncu_pp_ladder_cfg3.md")


def flops_per_iteration(o: int, v: int) -> dict:
    """Algorithmic work of the GEMM-view steps (8 real flop per complex MAC, packed index ranges): DESIGN.md table."""
    oo, vv, ov = o * (o - 1) // 2, v * (v - 1) // 2, o * v
    f = {
        "pp_ladder": 8 * oo * vv * vv,
        "Hvovo_quad": 8 * ov ** 3,
        "ring_gemm": 8 * ov ** 3,
        "C_ovoo": 8 * ov * oo * vv + 8 * ov * o * o * v,
        # the quartic term of A (oo oo vv MACs) is timed with the Fock-like terms: H^k_i reads ITS quartic term (o o o vv MACs as a
        # product of its own) off that product as a partial trace, as G^a_c reads its <ak||cd> t1 term off the linear term of H^{ak}_{ci}
        "A_oooo": 8 * oo * o * o * v,
        "hh_ladder+Goo": 8 * oo * oo * vv,            # algorithmic: hh-ladder oo^2 vv (+ Goo term o*oo*vv*... small)
        "fock_like": 8 * (v * v * oo * v + oo * oo * vv + ov * ov),
        "Hvovo_linear": 8 * (v * ov * o * v + v * o * ov * o),
        "Vdag_t1": 8 * o * vv * o * v,
        "Gvv_t2": 8 * oo * v * v * v,
        "C_t1": 8 * v * oo * v * o,
        # S1: its <ak||cd> tau term (v o o vv MACs as a product of its own) is read off the product of C (a partial trace,
        # ccsd_lib.cu s1_c_trace) on one GPU, so it is not counted as work
        "S1": 8 * (o * v * oo * v + 2 * ov * ov),
    }
    f["total"] = sum(f.values())
    return f


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, power, reasons = [], [], [], set()
        for t, line in self.rows:
            if t < t0 or t > t1 + 0.1:
                continue
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks() -> dict:
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return {"hbm_gbs": float(d["hbm_gbs"]), "source": "MEASURED_PEAKS.json (of measured)"}
    return {"hbm_gbs": 6650.0, "source": "fallback of B200_PROFILING.md (of fallback)"}


# -------------------------------------------------------------------------------------------------------------------
# CPU oracle arm (cpu_baseline leg and --impl reference)
#
# What is timed is always the oracle's OWN loop nests (oracle/ccsd_oracle.c), as they stand:
#   cfg0 / cfg1   real OracleCCSD.iterate() calls (restricted-sum mode), plus each term on its own;
#   cfg2 / cfg3   a whole oracle iteration takes minutes to tens of minutes (recorded once by
#                 tests/golden/make_oracle_energies.py: tests/golden/oracle_iteration_seconds.txt), so every term of
#                 the iteration is timed on a SLAB of its outermost output indices (oracle_*_range / _part: the same
#                 loop nests, true shapes, synthetic values) and scaled by the exact fraction of loop iterations the
#                 slab covers.  The sum is reported as s/iteration and marked "extrapolated": true;
#   cfg4          the pp-ladder evaluator the cfg4 parity tests use, on a bounded number of W rows per shape.
# -------------------------------------------------------------------------------------------------------------------
def workload_string(cfg: str) -> str:
    o, v, L, _ = ci.CONFIGS[cfg]
    vv = ci.pair_count(v)
    return f"{cfg}: nocc={o} nvir={v} naux={L} complex128, DIIS(6), antisymmetry-packed <ab||cd> {vv}x{vv}"


def _timed(fn) -> float:
    t0 = time.perf_counter()
    fn()
    return time.perf_counter() - t0


def _pairs_below(n_first: int, extent: int) -> int:
    """number of pairs x<y with x < n_first in a dimension of size extent"""
    return sum(extent - 1 - x for x in range(min(n_first, extent)))


def _grow_and_time(run, frac, limits, budget_s):
    """run(*sizes) evaluates a slab, frac(*sizes) is the fraction of the term's loop iterations it covers.  Start from the
    smallest slab and grow (last index first) until one evaluation takes about budget_s or the term is complete.  Returns
    (estimated seconds of the complete term, seconds of the largest slab timed, its fraction, its sizes): complete terms
    are measured; otherwise the two largest slabs give a fixed cost (buffers cleared, antisymmetric fill) plus a cost per
    loop iteration, and the term is  t2 + (t2 - t1) / (f2 - f1) * (1 - f2)."""
    sizes = [1] * len(limits)
    hist = []
    while True:
        dt = _timed(lambda: run(*sizes))
        f = frac(*sizes)
        hist.append((dt, f))
        done = dt >= 0.4 * budget_s or f >= 1.0
        if not done:
            want = min(16.0, 0.8 * budget_s / max(dt, 1e-4))
            for k in reversed(range(len(limits))):
                if sizes[k] < limits[k] and want > 1.0:
                    new = int(min(limits[k], max(sizes[k] + 1, sizes[k] * want)))
                    want /= new / sizes[k]
                    sizes[k] = new
            done = frac(*sizes) == f
        if done:
            if f >= 1.0:
                return dt, dt, f, list(sizes)
            if len(hist) < 2 or hist[-2][1] >= f:        # no second point yet: one more slab, twice the size
                for k in reversed(range(len(limits))):
                    if sizes[k] < limits[k]:
                        sizes[k] = min(limits[k], 2 * sizes[k])
                        break
                hist.append((_timed(lambda: run(*sizes)), frac(*sizes)))
                dt, f = hist[-1]
            (t1, f1), (t2, f2) = hist[-2], hist[-1]
            if f2 <= f1:
                return dt / f, dt, f, list(sizes)
            return t2 + max(t2 - t1, 0.0) / (f2 - f1) * (1.0 - f2), dt, f, list(sizes)


def oracle_term_seconds(oc, budget_s: float) -> dict:
    """Seconds per term of one residual evaluation + energy on the oracle object `oc` (tau current), every term by its own
    loop nest; terms that would take longer than budget_s are timed on a slab and scaled (entry "fraction" < 1)."""
    o, v, R = oc.o, oc.v, oc.restricted
    oo, vv = ci.pair_count(o), ci.pair_count(v)
    out = {}

    def rec(name, full, dt, f, slab):
        out[name] = {"seconds": full, "timed_seconds": dt, "fraction": f, "slab": slab}

    dt = _timed(oc.build_tau)
    rec("tau", dt, dt, 1.0, "all")
    for name, extent in zip(oc.PARTS, (v, o, o, v, o, o)):
        full, dt, f, sz = _grow_and_time(lambda n: oc.intermediates_part(name, 0, n), lambda n: n / extent, [extent], budget_s)
        rec(name, full, dt, f, f"outer index [0,{sz[0]}) of {extent}")
    fi = (lambda ni: _pairs_below(ni, o) / oo) if R else (lambda ni: ni / o)
    fa = (lambda na: _pairs_below(na, v) / vv) if R else (lambda na: na / v)
    a_cap = v if oc.vvvv is None or oc.vvvv.shape[0] == v else oc.vvvv_range[1]
    for name in oc.TERMS:
        if name == "ring":      # all j, all b for the slab of (i, a)
            frac = lambda ni, na: (ni / o) * (na / v)
        else:
            frac = lambda ni, na: fi(ni) * fa(na)
        lim_a = a_cap if name == "pp_ladder" else v
        full, dt, f, sz = _grow_and_time(lambda ni, na: oc.s2_term_range(name, 0, ni, 0, na), frac, [o, lim_a], budget_s)
        rec("S2_" + name, full, dt, f, f"i in [0,{sz[0]}) of {o}, a in [0,{sz[1]}) of {v}")
    full, dt, f, sz = _grow_and_time(lambda ni: oc.s1_range(0, ni), lambda ni: ni / o, [o], budget_s)
    rec("S1", full, dt, f, f"i in [0,{sz[0]}) of {o}")
    dt = _timed(oc.energy)
    rec("energy", dt, dt, 1.0, "all")
    return out


def _synthetic_oracle(o: int, v: int, seed: int, vvvv_rows: int):
    """An oracle object of the true shapes on synthetic-valued blocks (timing only): every block is a random row
    broadcast over the leading indices, which costs a memory pass instead of the oracle's own integral build."""
    from oracle import ccsd_oracle as orc
    rng = np.random.default_rng(seed)

    def block(*shape, scale):
        a = np.empty(shape, dtype=np.complex128)
        a[...] = (rng.standard_normal(shape[-1]) + 1j * rng.standard_normal(shape[-1])) * scale
        return a

    n = o + v
    f = block(n, n, scale=0.01)
    f[np.arange(n), np.arange(n)] = np.concatenate([np.linspace(-2.0, -0.5, o), np.linspace(0.3, 5.0, v)])
    oc = orc.OracleCCSD.from_blocks(o, v, f, block(o, o, o, o, scale=5e-3), block(o, o, o, v, scale=5e-3),
                                    block(o, o, v, v, scale=5e-3), block(v, o, v, o, scale=5e-3),
                                    block(v, o, v, v, scale=5e-3), block(vvvv_rows, v, v, v, scale=5e-3), 0, restricted=True)
    oc.set_amplitudes(block(o, v, scale=0.01), block(o, o, v, v, scale=0.01))
    for a in (oc.tau, oc.Hvovo, oc.C, oc.A, oc.S2, oc._scratch):
        a.fill(0.0)                                  # touch the pages outside the timed region
    return oc


def oracle_baseline(cfg: str, budget_s: float = 20.0, iterations: int = 1) -> dict:
    """The oracle on the host cores for workload `cfg`: s/iteration (measured for cfg0/cfg1, slab-scaled for cfg2/cfg3)
    and seconds per term."""
    from oracle import ccsd_oracle as orc
    o, v, L, seed = ci.CONFIGS[cfg]
    cores = orc.num_threads()
    recorded = recorded_oracle_seconds()
    if cfg in ("cfg0", "cfg0_2e", "cfg1"):
        inp = ci.make_config(cfg)
        oc = orc.OracleCCSD(inp.h, inp.B, o, v, restricted=True)
        ts = [_timed(oc.iterate) for _ in range(max(1, iterations))]
        terms = oracle_term_seconds(oc, 1e9)
        return {"value": statistics.median(ts), "unit": "s/iteration", "cores": cores, "kind": "oracle",
                "extrapolated": False, "timed_iterations": len(ts), "timed_seconds": sum(ts),
                "sample": f"{len(ts)} full OracleCCSD.iterate() of {cfg} (restricted-sum loops, DIIS in numpy)",
                "per_term_seconds": {k: round(x["seconds"], 4) for k, x in terms.items()},
                "recorded_full_iterations": recorded.get(cfg)}
    t0 = time.perf_counter()
    oc = _synthetic_oracle(o, v, seed, vvvv_rows=min(v, 8))
    setup = time.perf_counter() - t0
    nterms = 2 + len(oc.PARTS) + len(oc.TERMS) + 1
    t0 = time.perf_counter()
    terms = oracle_term_seconds(oc, max(0.3, budget_s / nterms))
    timed = time.perf_counter() - t0
    total = sum(x["seconds"] for x in terms.values())
    return {"value": total, "unit": "s/iteration", "cores": cores, "kind": "oracle", "extrapolated": True,
            "timed_iterations": 0, "timed_seconds": round(timed, 2), "setup_seconds": round(setup, 2),
            "scale_factor": round(total / max(sum(x["timed_seconds"] for x in terms.values()), 1e-9), 2),
            "sample": f"every term of one {cfg} residual + energy timed with the oracle's own loop nests on a slab of its "
                      "outermost output indices (true shapes, synthetic values); a term's time = largest slab + cost per loop "
                      "iteration (from the two largest slabs) x the iterations left; sum over terms (Jacobi/DIIS in numpy "
                      "not included)",
            "per_term_seconds": {k: round(x["seconds"], 3) for k, x in terms.items()},
            "per_term_fraction_timed": {k: round(x["fraction"], 6) for k, x in terms.items()},
            "recorded_full_iterations": recorded.get(cfg)}


def recorded_oracle_seconds() -> dict:
    """Wall seconds of REAL full oracle iterations at cfg2 / cfg3, recorded by tests/golden/make_oracle_energies.py
    (context for the slab-scaled numbers; another machine, its core count is in the file)."""
    path = os.path.join(ROOT, "tests", "golden", "oracle_iteration_seconds.txt")
    out = {}
    if not os.path.exists(path):
        return out
    with open(path) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            cfg, threads, nit, sec = line.split()[:4]
            out[cfg] = {"seconds_per_iteration": float(sec), "iterations": int(nit), "threads": int(threads),
                        "source": "tests/golden/oracle_iteration_seconds.txt"}
    return out


def oracle_ladder_sweep(budget_s: float = 6.0) -> list:
    """BASELINE config 4 on the host cores: the oracle's pp-ladder evaluator (the one the cfg4 parity tests use) on a
    bounded number of W rows per shape against every tau row, scaled to the whole contraction."""
    from oracle import ccsd_oracle as orc
    out = []
    per = budget_s / len(ci.LADDER_SWEEP)
    for k, (o, v) in enumerate(ci.LADDER_SWEEP):
        oo, vv = ci.pair_count(o), ci.pair_count(v)
        rng = np.random.default_rng(ci.LADDER_SEED0 + k)
        tau = (rng.standard_normal((oo, vv)) + 1j * rng.standard_normal((oo, vv))) * 0.01 / np.sqrt(2)
        nrow, dt = 4, 0.0
        while True:
            W = (rng.standard_normal((nrow, vv)) + 1j * rng.standard_normal((nrow, vv))) * 5e-3 / np.sqrt(2)
            ij, ab = np.meshgrid(np.arange(oo), np.arange(nrow), indexing="ij")
            dt = _timed(lambda: orc.pp_ladder_samples(tau, W, ij.ravel(), ab.ravel()))
            if dt > 0.4 * per or nrow >= vv:
                break
            nrow = int(min(vv, max(nrow * 2, nrow * 0.8 * per / max(dt, 1e-4))))
        sec = dt * vv / nrow
        out.append({"nocc": o, "nvir": v, "seconds": round(sec, 2), "gflops": round(8.0 * oo * vv * vv / sec * 1e-9, 2),
                    "rows_timed": nrow, "of_rows": vv, "timed_seconds": round(dt, 3), "extrapolated": nrow < vv})
    return out


def run_reference(args) -> None:
    """--impl reference: the CPU oracle on this arm's config, metric and unit.  A "step" is one bounded sample of the
    workload (cfg0/cfg1: one real iteration; cfg2/cfg3: one pass of per-term slab timings); `steps` is the number of
    samples actually timed, `ms_per_step` their measured wall time, so that steps x ms_per_step fits the run."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    small = cfg in ("cfg0", "cfg1")
    nsamp = max(1, min(args.steps, 3 if small else 2))
    for _ in range(1 if args.warmup > 0 else 0):
        oracle_baseline(cfg, budget_s=4.0)
    t0 = time.perf_counter()
    infos = [oracle_baseline(cfg, budget_s=20.0) for _ in range(nsamp)]
    wall = time.perf_counter() - t0
    info = sorted(infos, key=lambda d: d["value"])[len(infos) // 2]
    v = info["value"]
    line = {"impl": "reference", "metric": "ccsd_seconds_per_iteration", "value": v, "unit": "s/iteration",
            "n_gpus": args.gpus, "steps": nsamp, "warmup": 1 if args.warmup > 0 else 0, "ms_per_step": wall / nsamp * 1e3,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "complex128 (f64)",
            "data": "synthetic", "config": {"workload": workload_string(cfg)},
            "extrapolated": bool(info["extrapolated"]),
            "value_note": ("measured: median of real oracle iterations" if not info["extrapolated"] else
                           "extrapolated: sum over terms of slab seconds / slab fraction (see cpu_baseline.sample); "
                           "ms_per_step is the measured wall time of one sampling pass, not value x 1000"),
            "cpu_baseline": info,
            "e2e": {"value": v, "unit": "s/iteration", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# -------------------------------------------------------------------------------------------------------------------
# GPU arm
# -------------------------------------------------------------------------------------------------------------------
def time_events(torch, fn, reps, warmup, stream=None):
    """CUDA-event times (ms) of fn(), one pair of events per repetition, recorded on the stream fn launches on
    (torch.cuda.Event.record() without a stream sees only torch's current stream)."""
    stream = stream or torch.cuda.current_stream()
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream); fn(); e1.record(stream)
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    return ts


def ladder_sweep(torch, pkg, peak_tflops, reps=5, warmup=3):
    """BASELINE config 4: isolated pp-ladder R[(i<j)][(a<b)] = sum_{c<d} W tau per shape, with sampled parity."""
    from oracle.ccsd_oracle import pp_ladder_samples
    out = []
    for k, (o, v) in enumerate(ci.LADDER_SWEEP):
        oo, vv = ci.pair_count(o), ci.pair_count(v)
        gen = torch.Generator(device="cuda")
        gen.manual_seed(ci.LADDER_SEED0 + k)
        W = torch.view_as_complex(torch.randn((vv, vv, 2), generator=gen, device="cuda", dtype=torch.float64))
        W.mul_(5e-3 / np.sqrt(2))
        tau = torch.view_as_complex(torch.randn((oo, vv, 2), generator=gen, device="cuda", dtype=torch.float64))
        tau.mul_(0.01 / np.sqrt(2))
        R = torch.zeros((oo, vv), dtype=torch.complex128, device="cuda")
        # as inside ccsd_iterate: the sum plane of the constant W exists once (ccsd_init), tau's is rebuilt per call
        Ws = pkg.sum_plane(W)

        def ladder():
            pkg.contract("pp_ladder_planes", o, v, [tau, W, pkg.sum_plane(tau), Ws], out=R)

        ts = time_events(torch, ladder, reps, warmup)
        t = statistics.median(ts)
        # sampled parity against the oracle (inputs come from torch's RNG, not from the CUDA path)
        rng = np.random.default_rng(k)
        ij = rng.integers(0, oo, 64); ab = rng.integers(0, vv, 64)
        Wrows = W[torch.from_numpy(np.unique(ab)).cuda()].cpu().numpy()
        remap = {a: i for i, a in enumerate(np.unique(ab))}
        ref = pp_ladder_samples(tau.cpu().numpy(), Wrows, ij, np.array([remap[a] for a in ab]))
        got = R[torch.from_numpy(ij).cuda(), torch.from_numpy(ab).cuda()].cpu().numpy()
        err = float(np.abs(got - ref).max() / np.abs(ref).max())
        tf = 8.0 * oo * vv * vv / (t * 1e-3) * 1e-12
        ex = pkg.real_flops_per_cmac() / 8.0
        out.append({"nocc": o, "nvir": v, "ms": round(t, 3), "tflops": round(tf, 2),
                    "tflops_executed": round(tf * ex, 2), "frac_fp64_peak": round(tf * ex / peak_tflops, 4),
                    "sampled_rel_err": err})
        del W, tau, R, Ws
        torch.cuda.empty_cache()
    return out


def transpose_bench(torch, pkg, hbm_gbs, o, v):
    """Transposition GB/s (read + write bytes) on o^2 v^2-shaped complex128 tensors."""
    torch.cuda.empty_cache()       # the legs before this one leave tens of GB of cached blocks behind
    x = torch.view_as_complex(torch.randn((o, o, v, v, 2), device="cuda", dtype=torch.float64))
    nbytes = 2 * x.numel() * 16
    res = {}
    cases = (("ijab->abij", [2, 3, 0, 1]), ("ijab->iajb", [0, 2, 1, 3]), ("ijab->jiba", [1, 0, 3, 2]),
             ("ijab->baji", [3, 2, 1, 0]), ("ijab->aibj", [2, 0, 3, 1]), ("ijab->ibaj", [0, 3, 2, 1]))
    # one untimed pass over every case first: right after the FP64-tensor-heavy legs (900 W) the first memory-bound
    # kernels run below the steady rate for some tens of milliseconds (measured: 4.7 instead of 6.1 TB/s for whichever case
    # is first)
    for _, perm in cases:
        for _ in range(20):
            pkg.transpose(x, perm)
    torch.cuda.synchronize()
    for name, perm in cases:
        ts = time_events(torch, lambda: pkg.transpose(x, perm), 15, 5)
        gbs = nbytes / (statistics.median(ts) * 1e-3) * 1e-9
        res[name] = {"gbs": round(gbs, 1), "frac_hbm": round(gbs / hbm_gbs, 3)}
    return res


def library_yardstick(torch, pkg, o, v, peak):
    """SURVEY 8(d) yardstick (b): the library FP64 GEMMs (cuBLAS through torch.matmul) timed beside this repo's kernel --
    DGEMM 8192^3, and ZGEMM on the workload's pp-ladder shape (oo x vv x vv, both operands K-contiguous) against
    ccsd_contract(PP_LADDER) on the very same tensors.  A comparison only: nothing on the product path calls a library GEMM."""
    torch.cuda.empty_cache()
    oo, vv = o * (o - 1) // 2, v * (v - 1) // 2
    a = torch.randn((8192, 8192), device="cuda", dtype=torch.float64)
    b = torch.randn((8192, 8192), device="cuda", dtype=torch.float64)
    c = torch.empty((8192, 8192), device="cuda", dtype=torch.float64)
    ts = time_events(torch, lambda: torch.matmul(a, b, out=c), 5, 2)
    dgemm_tflops = 2 * 8192 ** 3 / (statistics.median(ts) * 1e-3) * 1e-12
    del a, b, c
    gen = torch.Generator(device="cuda").manual_seed(2021030899)
    W = torch.view_as_complex(torch.randn((vv, vv, 2), generator=gen, device="cuda", dtype=torch.float64)) * 5e-3
    tau = torch.view_as_complex(torch.randn((oo, vv, 2), generator=gen, device="cuda", dtype=torch.float64)) * 1e-2
    out_lib = torch.empty((oo, vv), device="cuda", dtype=torch.complex128)
    Wt = W.t()
    ts = time_events(torch, lambda: torch.matmul(tau, Wt, out=out_lib), 5, 2)
    lib_ms = statistics.median(ts)
    out_own = torch.zeros((oo, vv), device="cuda", dtype=torch.complex128)
    ts = time_events(torch, lambda: pkg.contract("pp_ladder", o, v, [tau, W], out=out_own), 5, 2)
    own_ms = statistics.median(ts)
    diff = float((out_own - out_lib).abs().max() / out_lib.abs().max())
    fl8 = 8.0 * oo * vv * vv
    res = {"dgemm_8192_tflops": round(dgemm_tflops, 2), "dgemm_8192_frac_fp64_peak": round(dgemm_tflops / peak, 4),
           "pp_ladder_shape": [oo, vv, vv],
           "library_zgemm_ms": round(lib_ms, 3), "library_zgemm_tflops_8flop": round(fl8 / (lib_ms * 1e-3) * 1e-12, 2),
           "own_pp_ladder_ms": round(own_ms, 3), "own_pp_ladder_tflops_8flop": round(fl8 / (own_ms * 1e-3) * 1e-12, 2),
           "own_over_library": round(lib_ms / own_ms, 3), "max_rel_diff_own_vs_library": diff,
           "note": "library = cuBLAS via torch.matmul (complex128 ZGEMM, 4 real products per complex MAC); own = "
                   "ccsd_contract(PP_LADDER) without caller-held sum planes (3M, 3 real products)"}
    del W, Wt, tau, out_lib, out_own
    torch.cuda.empty_cache()
    return res


def converge_bench(torch, pkg, inp, o, v, tol=1e-11, max_iterations=400):
    """Time to solution: ccsd_init + ccsd_solve from the MP2 guess to ||S/D||_2 < tol and |dE| < tol (.TCONVERG),
    wall clock; init_seconds includes the host->device copy of h and B.  tests/test_gpu_fullsize.py certifies this converged energy with the oracle."""
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    solver = pkg.CCSD(inp.h, inp.B, o, v, ndiis=6)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    ok, nit, e, sn = solver.solve(tol, max_iterations)
    torch.cuda.synchronize()
    t2 = time.perf_counter()
    t1d = solver.t1_diagnostic()
    solver.close()
    del solver
    torch.cuda.empty_cache()
    return {"converged": bool(ok), "tol": tol, "iterations": nit, "solve_seconds": round(t2 - t1, 3),
            "init_seconds": round(t1 - t0, 3), "E_corr": [e.real, e.imag], "step_norm": sn, "t1_diagnostic": t1d}


def cc2_bench(torch, pkg, inp, o, v, steps=5, warmup=3):
    """NEXT-1 row of SURVEY 8(f): the CC2 iteration on the same workload, device-resident."""
    solver = pkg.CCSD(inp.h, inp.B, o, v, ndiis=6, cc2=True)
    solver.enable_step_timing(True)
    ts = time_events(torch, solver.iterate, steps, warmup, solver.stream)
    st = solver.step_times()
    e, sn = solver.iterate()
    solver.close()
    del solver
    torch.cuda.empty_cache()
    return {"s_per_iteration": round(statistics.median(ts) * 1e-3, 6), "steps": steps, "warmup": warmup,
            "pp_ladder_ms": round(st["pp_ladder"], 3), "C_ovoo_ms": round(st["C_ovoo"], 3),
            "E_last": [e.real, e.imag], "step_norm_last": sn,
            "note": "eq 34 evaluated as eq 32 at t2 = 0 plus the two Fock terms, the <ab||cd> and <bk||cd> terms factorised "
                    "through the auxiliary index (K = naux GEMMs); singles by eq 33"}


def triples_bench(torch, pkg, inp, o, v, peak_tflops):
    """NEXT-3 row of SURVEY 8(f): +T / (T) / -T at the amplitudes after two CCSD iterations.
    One timed call without per-launch events (wall clock around a synchronising call), one with (kernel split)."""
    solver = pkg.CCSD(inp.h, inp.B, o, v, ndiis=6)
    for _ in range(2):
        solver.iterate()
    solver.triples()                                   # warm-up: function attributes, L2
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(solver.stream)
    en = solver.triples()
    e1.record(solver.stream)
    torch.cuda.synchronize()
    total_ms = e0.elapsed_time(e1)
    solver.enable_step_timing(True)
    solver.triples()
    tm = solver.triples_times()
    solver.close()
    del solver
    torch.cuda.empty_cache()
    vv, nt = ci.pair_count(v), o * (o - 1) * (o - 2) // 6
    cmac = nt * vv * v * 3 * (v + o)                   # unique i<j<k, rows a<b, K = 3v + 3o
    rf = pkg.real_flops_per_cmac()
    tf8 = 8.0 * cmac / (tm["w_gemm_ms"] * 1e-3) * 1e-12
    return {"seconds": round(total_ms * 1e-3, 4), "occupied_triples": nt, "w_gemm_ms": round(tm["w_gemm_ms"], 2),
            "energy_kernels_ms": round(tm["energy_ms"], 2), "w_gemm_tflops": round(tf8, 2),
            "w_gemm_frac_fp64_peak": round(tf8 * rf / 8.0 / peak_tflops, 4),
            "E(+T)": [en["+T"].real, en["+T"].imag], "E((T))": [en["(T)"].real, en["(T)"].imag],
            "E(-T)": [en["-T"].real, en["-T"].imag],
            "note": "one K-segmented DMMA GEMM (vv x v x (3v+3o)) per occupied triple i<j<k; fraction of peak on the "
                    "executed (3M) flops"}


def triples_sharded_bench(torch, pkg, inp, o, v, dist):
    """N > 1 only: the triples correction shared among the ranks (CCSD.triples_sharded: contiguous ranges of the
    occupied triples i<j<k, one all-reduce of six doubles).  Total work fixed -> strong scaling; seconds = max over ranks."""
    solver = pkg.CCSD(inp.h, inp.B, o, v, ndiis=6)
    for _ in range(2):
        solver.iterate()
    solver.triples_sharded()                           # warm-up
    torch.cuda.synchronize()
    dist.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(solver.stream)
    en = solver.triples_sharded()
    e1.record(solver.stream)
    torch.cuda.synchronize()
    sec = max_over_ranks(e0.elapsed_time(e1) * 1e-3, dist)
    nt = solver.triples_count()
    solver.close()
    del solver
    torch.cuda.empty_cache()
    return {"seconds": round(sec, 4), "ranks": dist.get_world_size(), "occupied_triples": nt, "scaling": "strong",
            "E(+T)": [en["+T"].real, en["+T"].imag], "E((T))": [en["(T)"].real, en["(T)"].imag],
            "E(-T)": [en["-T"].real, en["-T"].imag],
            "note": "each rank evaluates a contiguous range of the occupied triples (ccsd_triples_range); no data-path "
                    "collective, one all-reduce of six doubles"}


def direct_ladder_bench(torch, pkg, inp, o, v, steps=3, warmup=2):
    """Rank 4 of SURVEY 8(f), first half: the CCSD iteration with the integral-direct pp-ladder (<ab||cd> rebuilt from B
    every iteration, never stored)."""
    solver = pkg.CCSD(inp.h, inp.B, o, v, ndiis=6, direct_ladder=True)
    solver.enable_step_timing(True)
    ts = time_events(torch, solver.iterate, steps, warmup, solver.stream)
    st = solver.step_times()
    ws = solver.workspace_bytes
    solver.close()
    del solver
    torch.cuda.empty_cache()
    return {"s_per_iteration": round(statistics.median(ts) * 1e-3, 5), "pp_ladder_ms": round(st["pp_ladder"], 2),
            "workspace_gib": round(ws / 2 ** 30, 1), "steps": steps, "warmup": warmup}


def lambda_bench(torch, pkg, inp, o, v, steps=3, warmup=1):
    """NEXT-2 row of SURVEY 8(f): Lambda equations at the amplitudes after three CCSD iterations
    (the cost of a Lambda iteration does not depend on the convergence of T): Hbar build once, then timed iterations."""
    solver = pkg.CCSD(inp.h, inp.B, o, v, ndiis=6)
    for _ in range(3):
        solver.iterate()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(solver.stream)
    solver.lambda_init()
    e1.record(solver.stream)
    torch.cuda.synchronize()
    init_ms = e0.elapsed_time(e1)
    ts = time_events(torch, solver.lambda_iterate, steps, warmup, solver.stream)
    sn = solver.lambda_iterate()
    D = solver.density()
    tr = complex(torch.trace(D).item())
    ws = solver._lam_ws.numel()
    solver.close()
    del solver
    torch.cuda.empty_cache()
    return {"s_per_iteration": round(statistics.median(ts) * 1e-3, 5), "hbar_build_s": round(init_ms * 1e-3, 4),
            "steps": steps, "warmup": warmup, "step_norm_last": sn, "density_trace_abs": abs(tr),
            "workspace_gib": round(ws / 2 ** 30, 1),
            "note": "one permute + DMMA GEMM + signed permuted add per small term, packed-pair routes for the o^2 v^3 products; pp-ladder term on the packed "
                    "<ab||cd> with conjugated multipliers"}


def hbm_step_bytes(o: int, v: int, m: int, planes: bool = True, levels: dict | None = None) -> dict:
    """Algorithmic bytes of the HBM-bound steps of one iteration (16 B read + 16 B written per element a
    permutation moves; the update streams (2 + 2m) vectors at the least; m = pairs in the DIIS subspace).  levels: the solver's
    strassen_steps() (None / {}: plain products)."""
    oo, vv, ov = o * (o - 1) // 2, v * (v - 1) // 2, o * v
    nvec = ov + oo * vv
    levels = levels or {}
    moved = ov + oo * vv + 2 * ov * ov + v * oo * v + oo * v * v      # t1T, tau^T, Xm, T2r, tauc, t2hu
    extra = 0
    if planes:
        if "ring_gemm" not in levels:
            extra += 2 * ov * ov * 8                                  # planes of Xm, T2r (Strassen stacks carry their own)
        # Strassen stacks of tau for the ladder and C: tau read once per stack, 7 half-size / 49 quarter-size matrices (16 B) and
        # their planes (8 B) written
        used = {levels.get("pp_ladder", 0), levels.get("C_ovoo", 0)}
        if 1 in used:
            extra += oo * vv * 16 + 7 * ((oo + 1) // 2) * ((vv + 1) // 2) * 24
        if 2 in used:
            extra += oo * vv * 16 + 49 * ((oo + 3) // 4) * ((vv + 3) // 4) * 24
    return {"prep_permute": moved * 32 + extra,
            # Jacobi + Gram row in one pass (S, t and m-1 stored e read; e, u written), then sum_l c_l u_l (m read, 1 written)
            "update_diis": (2 * m + 4) * nvec * 16,
            "update_diis_floor": (2 * m + 2) * nvec * 16,
            # tau + its plane + energy in one pass: t2 and <ij||ab> read, tau (16 B) and plane (8 B) written
            "energy": oo * vv * (16 + 16 + 16 + (8 if planes else 0)) + ov * 32}


def iteration_bench(torch, pkg, cfg, inp, steps, warmup, peak, hbm_gbs, barrier=None, clock_index=None, e2e=False,
                    max_ranks=None, graph=1, strassen=1) -> dict:
    """W warm-up + exactly K timed ccsd_iterate of workload `cfg` the way a user runs them (residual replayed as a CUDA
    graph, no events inside), CUDA events on the solver's stream around the K steps; then a second pass of K iterations
    with the library's per-step events (direct launches) for the per-term table and the roofline launch."""
    o, v, L, _ = ci.CONFIGS[cfg]
    oo, vv, ov = ci.pair_count(o), ci.pair_count(v), o * v
    barrier = barrier or torch.cuda.synchronize
    pkg.launch_count(reset=True)
    t0 = time.perf_counter()
    solver = pkg.CCSD(inp.h, inp.B, o, v, ndiis=6, graph=graph, strassen=strassen)
    torch.cuda.synchronize()
    init_s = time.perf_counter() - t0
    init = solver.init_stats()
    e_mp2 = solver.energy()
    st = solver.stream
    for _ in range(warmup):
        solver.iterate()
    barrier()
    launches0 = pkg.launch_count()
    sampler = ClockSampler(clock_index) if clock_index is not None else None
    if sampler:
        sampler.start()
        time.sleep(0.25)
    t_wall0 = time.time()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(st)
    energies = []
    for _ in range(steps):
        energies.append(solver.iterate())
    e1.record(st)
    barrier()
    t_wall1 = time.time()
    ms_total = e0.elapsed_time(e1)
    launches = pkg.launch_count() - launches0
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    ms_total = max_over_ranks(ms_total, max_ranks)
    ms_per_step = ms_total / steps

    # ---- per-term pass: the library's own events between the steps (this switches the graph replay off) ----------
    solver.enable_step_timing(True)
    solver.iterate()
    step_acc, m_hist = {}, []
    done = warmup + steps + 1
    e0.record(st)
    for q in range(steps):
        solver.iterate()
        m_hist.append(min(6, done + q + 1))
        for k, x in solver.step_times().items():
            step_acc.setdefault(k, []).append(x)
    e1.record(st)
    torch.cuda.synchronize()
    ms_events = e0.elapsed_time(e1) / steps
    solver.enable_step_timing(False)
    fl = flops_per_iteration(o, v)
    ex = pkg.real_flops_per_cmac() / 8.0
    # a product that runs as one Strassen level (ccsd_options.strassen) EXECUTES 7/8 of the plain product's real flops
    strassen_steps = solver.strassen_steps()
    exk = {k: ex * (7.0 / 8.0) ** strassen_steps.get(k, 0) for k in fl}
    executed_total = fl["total"] * ex - sum(fl[k] * (ex - exk[k]) for k in strassen_steps)      # in 8-flop units x ex
    terms = {}
    for k, xs in step_acc.items():
        ms = statistics.median(xs)
        ent = {"ms": round(ms, 4)}
        if k in fl and ms > 0:
            ent["tflops"] = round(fl[k] / (ms * 1e-3) * 1e-12, 2)
            ent["frac_fp64_peak"] = round(fl[k] * exk[k] / (ms * 1e-3) * 1e-12 / peak, 4)
            if k in strassen_steps:
                ent["strassen_levels"] = strassen_steps[k]
        terms[k] = ent
    for k in ("prep_permute", "update_diis", "energy"):       # HBM-bound steps: algorithmic bytes / time
        gbs = [hbm_step_bytes(o, v, m, levels=strassen_steps)[k] / (x * 1e-3) * 1e-9
               for x, m in zip(step_acc[k], m_hist) if x > 0]
        if gbs:
            terms[k]["gbs"] = round(statistics.median(gbs), 1)
            terms[k]["frac_hbm"] = round(statistics.median(gbs) / hbm_gbs, 3)
    b = hbm_step_bytes(o, v, 6)
    terms["update_diis"]["vector_passes"] = 16
    terms["update_diis"]["vector_passes_floor"] = 14
    init_pack = None
    if init["pack_ms"] > 0:
        init_pack = {"pack_ms": round(init["pack_ms"], 3), "pack_gbs": round(init["packed_elems"] * 48 / (init["pack_ms"] * 1e-3) * 1e-9, 1),
                     "transpose_ms": round(init["transpose_ms"], 3),
                     "transpose_gbs": round(init["transposed_elems"] * 32 / (init["transpose_ms"] * 1e-3) * 1e-9, 1),
                     "gemm_ms": round(init["gemm_ms"], 3),
                     "note": "ccsd_init's build of the packed <ab||cd> (SURVEY 8(a) I2): slab GEMMs (ac|bd) over the auxiliary index, "
                             "slab transpositions (32 B per element), antisymmetrise-and-pack fills (two 16 B reads + one 16 B "
                             "write per packed element); device ms summed over the slabs"}
        init_pack["pack_frac_hbm"] = round(init_pack["pack_gbs"] / hbm_gbs, 3)
        init_pack["transpose_frac_hbm"] = round(init_pack["transpose_gbs"] / hbm_gbs, 3)
    out = {"workload": workload_string(cfg), "ms_per_step": ms_per_step, "s_per_iteration": round(ms_per_step * 1e-3, 6),
           "ms_per_step_with_step_events": round(ms_events, 4), "steps": steps, "warmup": warmup,
           "ideal_ms_at_peak": round(executed_total / peak * 1e-9, 4),
           "frac_of_ideal": round(executed_total / peak * 1e-9 / ms_per_step, 4),
           "executed_flops_per_iteration": executed_total, "strassen_steps": strassen_steps,
           "gpu_launches": launches, "gpu_launches_per_step": round(launches / steps, 1),
           "graph_replay": bool(st.cuda_stream != 0), "terms": terms, "init_seconds": round(init_s, 3), "init_pack": init_pack,
           "clocks": clocks,
           "energies": {"E_mp2_start": [e_mp2.real, e_mp2.imag], "E_last": [energies[-1][0].real, energies[-1][0].imag],
                        "step_norm_last": energies[-1][1]}}
    if e2e:
        # ---- end to end: amplitudes travel host(pinned) -> device -> host every step ------------------------------
        t1_d, t2_d = solver.get_amplitudes()
        t1_h = torch.empty(t1_d.shape, dtype=torch.complex128).pin_memory()
        t2_h = torch.empty(t2_d.shape, dtype=torch.complex128).pin_memory()
        t1_h.copy_(t1_d); t2_h.copy_(t2_d)

        def e2e_step():
            t1_d.copy_(t1_h, non_blocking=True)
            t2_d.copy_(t2_h, non_blocking=True)
            solver.set_amplitudes(t1_d, t2_d, reset_diis=False)
            solver.iterate()
            a1, a2 = solver.get_amplitudes()
            t1_h.copy_(a1, non_blocking=True)
            t2_h.copy_(a2, non_blocking=True)
            torch.cuda.current_stream().synchronize()

        e2e_step()
        barrier()
        tw = time.perf_counter()
        nsteps_e2e = max(1, min(steps, 5))
        for _ in range(nsteps_e2e):
            e2e_step()
        barrier()
        e2e_s = max_over_ranks((time.perf_counter() - tw) / nsteps_e2e, max_ranks)
        nvec_bytes = (ov + oo * vv) * 16
        out["e2e"] = {"value": e2e_s, "unit": "s/iteration", "h2d_bytes_per_step": nvec_bytes,
                      "d2h_bytes_per_step": nvec_bytes + 32, "steps": nsteps_e2e}
    solver.close()
    del solver
    torch.cuda.empty_cache()
    return out


def variant_sweep(torch, pkg, peak):
    """Profiling aid (--only-variants): the 3M tile variants of the DMMA GEMM on the shapes that decide the tile choice
    (DESIGN.md "The DMMA GEMM"): executed-flop fraction of the FP64 peak of ccsd_zgemm_nt(mode = 100 + variant)."""
    shapes = [("triples driver, 61 triples batched as rows", 50000, 224, 784, True, (11, 12, 15)),
              ("one triple", 24976, 224, 816, True, (11, 12, 15)),
              ("G_vv.t2", 125664, 224, 224, False, (5, 6, 14)),
              ("N = nocc product", 200000, 34, 224, False, (5, 6, 13)),
              ("pp-ladder cfg3", 24976, 561, 24976, True, (12, 15)),
              ("(ov)^3 cfg3", 7616, 7616, 7616, True, (12, 15)),
              ("pp-ladder cfg2", 12720, 276, 12720, True, (11, 12, 15))]
    out = []
    for name, M, N, K, planes, variants in shapes:
        g = torch.Generator(device="cuda").manual_seed(1)
        A = torch.view_as_complex(torch.randn((M, K, 2), generator=g, device="cuda", dtype=torch.float64))
        B = torch.view_as_complex(torch.randn((N, K, 2), generator=g, device="cuda", dtype=torch.float64))
        C = torch.zeros((M, N), dtype=torch.complex128, device="cuda")
        pl = (pkg.sum_plane(A), pkg.sum_plane(B)) if planes else None
        row = {"shape": name, "M": M, "N": N, "K": K, "planes": planes, "variants": {}}
        for v in variants:
            ts = time_events(torch, lambda: pkg.zgemm_nt(A, B, C=C, mode=100 + v, planes=pl), 5, 2)
            t = statistics.median(ts)
            row["variants"][str(v)] = {"ms": round(t, 3), "frac_fp64_peak": round(6.0 * M * N * K / (t * 1e-3) * 1e-12 / peak, 4)}
        row["picked"] = pkg.gemm_plan(M, N, K, 1, 0, planes)
        out.append(row)
        del A, B, C, pl
        torch.cuda.empty_cache()
    return out


def max_over_ranks(value: float, dist, device="cuda") -> float:
    """Multi-GPU numbers are the MAX over ranks (replicas-only path: no data-path collective exists)."""
    import torch
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def is_reporting_rank() -> bool:
    return int(os.environ.get("RANK", "0")) == 0


def run_ours(args) -> None:
    import torch
    import torch.distributed as dist
    import paper_2103_08473_b200 as pkg

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device; there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = args.config
    o, v, L, seed = ci.CONFIGS[cfg]
    oo, vv, ov = ci.pair_count(o), ci.pair_count(v), o * v
    if args.only_ladder and args.ladder_shape:
        o, v = (int(x) for x in args.ladder_shape.split(","))
        oo, vv = ci.pair_count(o), ci.pair_count(v)
        cfg = f"nocc={o} nvir={v}"
    if args.only_ov3:
        # profiling aid: the (ov)^3 product X[(a,i)][(j,b)] = sum_{(c,k)} H[(a,i)][(c,k)] T[(j,b)][(c,k)] of this workload's shape the
        # way ccsd_iterate runs it (operand stacks, ONE batched launch of the 7 / 49 products, result sum)
        pkg.load_library()
        gen = torch.Generator(device="cuda"); gen.manual_seed(seed)
        H = torch.view_as_complex(torch.randn((ov, ov, 2), generator=gen, device="cuda", dtype=torch.float64)).mul_(0.05)
        T = torch.view_as_complex(torch.randn((ov, ov, 2), generator=gen, device="cuda", dtype=torch.float64)).mul_(0.01)
        X = torch.zeros((ov, ov), dtype=torch.complex128, device="cuda")
        levels = {0: 0, 2: 1, 3: 2}.get(args.strassen, 2 if ov >= 3072 else (1 if ov >= 1024 else 0))
        if levels:
            ts = time_events(torch, lambda: pkg.zgemm_nt_strassen(H, T, C=X, levels=levels), args.steps, args.warmup)
        else:
            ts = time_events(torch, lambda: pkg.zgemm_nt(H, T, C=X), args.steps, args.warmup)
        t = statistics.median(ts)
        print(json.dumps({"metric": "ov3_product_call_ms", "value": t, "unit": "ms", "levels": levels,
                          "config": {"workload": f"{cfg} (ov)^3 product {ov}x{ov}x{ov}, {levels} Strassen level(s); the call includes "
                                                 "the binding's workspace allocation"}}))
        return
    if args.only_ladder:
        # profiling aid: just the pp-ladder launch of this workload's shape (same kernel, same launch configuration
        # as inside ccsd_iterate), W warm-ups + K timed launches
        pkg.load_library()
        gen = torch.Generator(device="cuda"); gen.manual_seed(seed)
        W = torch.view_as_complex(torch.randn((vv, vv, 2), generator=gen, device="cuda", dtype=torch.float64)).mul_(5e-3 / np.sqrt(2))
        tau = torch.view_as_complex(torch.randn((oo, vv, 2), generator=gen, device="cuda", dtype=torch.float64)).mul_(0.01 / np.sqrt(2))
        R = torch.zeros((oo, vv), dtype=torch.complex128, device="cuda")
        if args.strassen:
            # the form ccsd_iterate runs: one Strassen level.  This standalone call also stacks <ab||cd> (done once, by ccsd_init,
            # inside the solver), so ms_per_call is NOT the launch time; the batched gemm_dmma_kernel launch inside it is the
            # launch of the iteration (same kernel, same grid) -- this leg exists to capture that launch with ncu.
            # levels as ccsd_init chooses them for this shape (ccsd_lib.cu carve): two where ov >= 3072 and a quarter of oo >= 128
            levels = 2 if (o * v >= 3072 and (((oo + 1) // 2) + 1) // 2 >= 128) else 1
            if args.strassen in (2, 3):
                levels = args.strassen - 1
            ts = time_events(torch, lambda: pkg.zgemm_nt_strassen(W, tau, C=R, transposed_out=True, levels=levels),
                             args.steps, args.warmup)
            t = statistics.median(ts)
            print(json.dumps({"metric": "pp_ladder_strassen_call_ms", "value": t, "unit": "ms", "ms_per_call": t, "levels": levels,
                              "config": {"workload": f"{cfg} pp-ladder {vv}x{oo}x{vv}, {levels} Strassen level(s), both operand stacks "
                                                     "made inside the call"}}))
            return
        Ws, taus = pkg.sum_plane(W), pkg.sum_plane(tau)
        ts = time_events(torch, lambda: pkg.contract("pp_ladder_planes", o, v, [tau, W, taus, Ws], out=R),
                         args.steps, args.warmup)
        t = statistics.median(ts)
        print(json.dumps({"metric": "pp_ladder_tflops", "value": 8.0 * oo * vv * vv / (t * 1e-3) * 1e-12, "unit": "TFLOP/s",
                          "ms_per_launch": t, "config": {"workload": f"{cfg} pp-ladder {vv}x{oo}x{vv}"}}))
        return
    pkg.load_library()
    if args.only_transposes:
        # profiling aid: the transposes leg alone (o^2 v^2-shaped tensor of --config)
        print(json.dumps({"metric": "transpose_gbs", "unit": "GB/s", "config": {"workload": f"{cfg} o^2 v^2 complex128"},
                          "hbm_peak": measured_peaks(), "transposes": transpose_bench(torch, pkg, measured_peaks()["hbm_gbs"], o, v)}))
        return
    if args.only_variants:
        peak = pkg.measure_fp64_peak(4)
        print(json.dumps({"metric": "dmma_tile_variants", "unit": "fraction of FP64 peak (executed 3M flops)", "fp64_peak_tflops": peak,
                          "variants": {"5/11": "128x32", "6/12": "128x48", "13": "128x40", "14/15": "128x56", "11,12,15": "with sum planes"},
                          "sweep": variant_sweep(torch, pkg, peak)}))
        return
    inp = ci.make_config(cfg)                      # every replica solves the same synthetic problem
    if args.only_lambda:
        print(json.dumps({"metric": "lambda_seconds_per_iteration", "unit": "s", "config": {"workload": f"{cfg} Lambda"},
                          **lambda_bench(torch, pkg, inp, o, v)}))
        return
    if args.only_cc2:
        print(json.dumps({"metric": "cc2_seconds_per_iteration", "unit": "s", "config": {"workload": f"{cfg} CC2"},
                          **cc2_bench(torch, pkg, inp, o, v)}))
        return
    if args.only_direct:
        print(json.dumps({"metric": "direct_ladder_seconds_per_iteration", "unit": "s",
                          "config": {"workload": f"{cfg} CCSD, integral-direct pp-ladder"},
                          **direct_ladder_bench(torch, pkg, inp, o, v)}))
        return
    if args.only_triples:
        # profiling aid: ccsd_init, one iteration, then the perturbative triples of this workload (same launches as
        # the "triples" leg of the default run)
        peak = pkg.measure_fp64_peak(4)
        print(json.dumps({"metric": "triples_seconds", "unit": "s", "config": {"workload": f"{cfg} +T/(T)/-T"},
                          **triples_bench(torch, pkg, inp, o, v, peak)}))
        return
    peak = pkg.measure_fp64_peak(8) if rank == 0 else FP64_NOMINAL_TFLOPS
    peaks = measured_peaks()
    rf = pkg.real_flops_per_cmac()                                  # 6: the 3M kernels execute 3 real FMAs per complex MAC
    ex = rf / 8.0
    main = iteration_bench(torch, pkg, cfg, inp, args.steps, args.warmup, peak, peaks["hbm_gbs"], barrier=barrier,
                           clock_index=local, e2e=True, max_ranks=(dist if world > 1 else None), graph=args.graph,
                           strassen=args.strassen)
    trip_sharded = triples_sharded_bench(torch, pkg, inp, o, v, dist) if (world > 1 and not args.no_sweep) else None

    if not is_reporting_rank():
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the DMMA GEMM, measured on the pp-ladder launch) ------------------------
    fl = flops_per_iteration(o, v)
    ms_per_step = main["ms_per_step"]
    pp_ms = main["terms"]["pp_ladder"]["ms"]
    pp_tflops = fl["pp_ladder"] / (pp_ms * 1e-3) * 1e-12          # 8-flop (ZGEMM) convention
    pp_strassen = "pp_ladder" in main["strassen_steps"]
    ex_pp = ex * (7.0 / 8.0) ** main["strassen_steps"].get("pp_ladder", 0)     # one Strassen level: seven half-size products for eight
    pp_exec = pp_tflops * ex_pp
    gemm_steps = ("pp_ladder", "Hvovo_quad", "ring_gemm")
    gemm_ms = sum(main["terms"][k]["ms"] for k in gemm_steps)
    pp_levels = main["strassen_steps"].get("pp_ladder", 0)
    traffic = (NCU_TRAFFIC_BYTES_STRASSEN.get(pp_levels, {}) if pp_strassen else NCU_TRAFFIC_BYTES).get(cfg)
    traffic_source = (NCU_TRAFFIC_SOURCE.replace("r02_ncu_pp_ladder_cfg3.md", NCU_TRAFFIC_FILE_STRASSEN.get(pp_levels, "?"))
                      if pp_strassen else NCU_TRAFFIC_SOURCE)
    roofline = {"bound": "tensor", "kernel": "gemm_dmma_kernel<DmmaCfg<4,2,4,3,3M,planes>> (FP64 DMMA.8x8x4), pp-ladder launch" +
                          (": ONE batched launch of the 7 half-size / 49 quarter-size products of its Strassen level(s)" if pp_strassen else ""),
                "achieved": round(pp_exec, 3), "peak": round(peak, 3), "unit": "TFLOP/s",
                "frac": round(pp_exec / peak, 4), "traffic": traffic,
                "traffic_source": (traffic_source if traffic is not None else
                                   "no ncu --set full capture of this workload's launch on record"),
                "real_flops_per_complex_mac": 8.0 * ex_pp,
                "achieved_8flop_convention": round(pp_tflops, 3),
                "note": "unit = complex MAC over the packed ranges (oo*vv*vv per launch); achieved counts the real "
                        "flops the kernel EXECUTES per unit (6 with 3M; x 7/8 = 5.25 when the product runs as one Strassen "
                        "level) so that frac <= 1; on the ZGEMM 8-flop "
                        "convention the same launch is achieved_8flop_convention.  With the Strassen level launch_ms also "
                        "contains the pass that sums the seven products into S2 (HBM-bound, ~0.3 % of it); the operand "
                        "stacks are made outside it (<ab||cd>: once, in ccsd_init; tau: in prep_permute).  "
                        "launch_ms = median CUDA-event time of "
                        "the launch over the K iterations of the step-timed pass (direct launches, events between the "
                        "steps on the launching stream); `value` is timed without those events (graph replay)",
                "peak_source": "DMMA.8x8x4 issue-rate microbenchmark measured in this run (ccsd_measure_fp64_peak); "
                               f"nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = {FP64_NOMINAL_TFLOPS:.1f}; "
                               "MEASURED_PEAKS.json has no FP64 entry",
                "flops_per_launch": int(fl["pp_ladder"] * ex_pp), "flops_per_launch_8flop": fl["pp_ladder"],
                "launch_ms": round(pp_ms, 3),
                "share_of_step": round(pp_ms / main["ms_per_step_with_step_events"], 4),
                "three_big_gemms": {"ms": round(gemm_ms, 3),
                                    "share_of_step": round(gemm_ms / main["ms_per_step_with_step_events"], 4),
                                    "tflops": round(sum(fl[k] for k in gemm_steps) / (gemm_ms * 1e-3) * 1e-12, 2)}}

    torch.cuda.empty_cache()
    # the other BASELINE configs ride along (they cost milliseconds): s/iteration and the same per-term table
    others = {}
    if not args.no_sweep:
        for other in ("cfg1", "cfg2"):
            if other != cfg:
                r = iteration_bench(torch, pkg, other, ci.make_config(other), 10, 6, peak, peaks["hbm_gbs"])
                others[other] = {k: r[k] for k in ("workload", "s_per_iteration", "ms_per_step_with_step_events", "ideal_ms_at_peak",
                                                   "frac_of_ideal", "strassen_steps", "gpu_launches_per_step", "graph_replay", "terms", "energies")}
    conv = converge_bench(torch, pkg, inp, o, v) if not args.no_sweep else None
    cc2 = cc2_bench(torch, pkg, inp, o, v) if not args.no_sweep else None
    triples = triples_bench(torch, pkg, inp, o, v, peak) if not args.no_sweep else None
    lam = lambda_bench(torch, pkg, inp, o, v) if not args.no_sweep else None
    direct = direct_ladder_bench(torch, pkg, inp, o, v) if not args.no_sweep else None
    sweep = ladder_sweep(torch, pkg, peak) if not args.no_sweep else None
    yard = library_yardstick(torch, pkg, o, v, peak) if not args.no_sweep else None
    transposes = transpose_bench(torch, pkg, peaks["hbm_gbs"], o, v)
    cpu = oracle_baseline(cfg) if world == 1 else None
    cpu_sweep = oracle_ladder_sweep() if (world == 1 and not args.no_sweep) else None
    if sweep and cpu_sweep:
        for g, c in zip(sweep, cpu_sweep):
            g["cpu_oracle_seconds"] = c["seconds"]
            g["cpu_oracle"] = c

    line = {
        "metric": "ccsd_seconds_per_iteration", "value": ms_per_step * 1e-3, "unit": "s/iteration",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "complex128 (f64)",
        "data": "synthetic",
        "config": {"workload": workload_string(cfg), "replicas": world,
                   "l2": f"inputs larger than L2 (packed <ab||cd> = {vv * vv * 16 / 2 ** 30:.2f} GiB vs 126 MB L2); no flush needed",
                   "init_seconds": main["init_seconds"], "graph_replay": main["graph_replay"]},
        "iteration_tflops": round(fl["total"] / (ms_per_step * 1e-3) * 1e-12, 2),
        "iteration_frac_fp64_peak": round(main["executed_flops_per_iteration"] / (ms_per_step * 1e-3) * 1e-12 / peak, 4),
        "pp_ladder_tflops": round(pp_tflops, 2), "pp_ladder_frac_fp64_peak": round(pp_exec / peak, 4),
        "tflops_convention": f"8 real flop per complex MAC (ZGEMM); fractions of peak use the {rf} executed (x 7/8 for the "
                             "products that run as L Strassen levels: terms[].strassen_levels)",
        "ms_per_step_with_step_events": main["ms_per_step_with_step_events"],
        "roofline": roofline, "terms": main["terms"], "init_pack": main["init_pack"],
        "e2e": main["e2e"],
        "gpu_launches": main["gpu_launches"], "clocks": main["clocks"],
        "energies": main["energies"], "other_configs": others,
        "solve_to_convergence": conv, "cc2": cc2, "triples": triples, "triples_sharded": trip_sharded, "lambda": lam,
        "direct_ladder": direct, "ladder_sweep": sweep, "library_yardstick": yard, "transposes": transposes,
        "hbm_peak": peaks, "cpu_baseline": cpu,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg3", choices=["cfg0", "cfg1", "cfg2", "cfg3"])
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--graph", type=int, default=1, help="ccsd_options.graph of the main leg: 0 direct launches, 1 graph with parallel "
                                                          "branches, 3 serial graph (profiling aid)")
    ap.add_argument("--strassen", type=int, default=1, help="ccsd_options.strassen of the main leg: 1 (default) Strassen levels on "
                    "the four large contractions, 0 plain products, 2 one level only, 3 two levels everywhere (tests)")
    ap.add_argument("--only-ov3", action="store_true", help="profiling aid: the (ov)^3 product of --config's shape through "
                    "ccsd_zgemm_nt_strassen with the level count of the iteration (the batched launch of the ring / H^{ak}_{ci} terms)")
    ap.add_argument("--only-ladder", action="store_true", help="time only the pp-ladder launch of --config's shape")
    ap.add_argument("--ladder-shape", default="", help="with --only-ladder: 'nocc,nvir' of a BASELINE config-4 sweep shape")
    ap.add_argument("--only-lambda", action="store_true", help="time only the Lambda equations of --config")
    ap.add_argument("--only-triples", action="store_true", help="time only the perturbative triples of --config")
    ap.add_argument("--only-transposes", action="store_true", help="time only the 4-index transpositions")
    ap.add_argument("--only-cc2", action="store_true", help="time only the CC2 iteration of --config")
    ap.add_argument("--only-direct", action="store_true", help="time only the CCSD iteration with the integral-direct pp-ladder")
    ap.add_argument("--only-variants", action="store_true", help="time the 3M tile variants of the DMMA GEMM on the deciding shapes")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
