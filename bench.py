#!/usr/bin/env python
"""bench.py -- the VIPIR database scan on B200, measured.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--paper] [--modgemm] [--pipeline] [--only NAME]

Headline (BASELINE.json `metric`: "DB GB/s scanned & TOPS, % of HBM/INT8-TC roofline; 16 GiB u8
DB, batch 1/256"): one STEP is one pass of the whole hot path -- query-limb split + scan (one
fused kernel at batch 1), through the C ABI (vipir_dbmul) -- over one batch of synthetic queries against the
16 GiB u8 database of configs[2] (131072 x 131072, q = 2^32, batch 1).  `value` is GB of DB
scanned per second with all inputs resident in HBM; `e2e` is the same through vipir_dbmul_host
with the query in / the answer out of pinned HOST memory inside the timed region.

In the same JSON line (N = 1):
  "batched"   configs[3] (4 GiB, batch 256) on the tensor cores: sustained step (1 s settle) and burst, its own
              e2e through vipir_dbmul_host (64 MiB in, 64 MiB out per step), and a tensor roofline against the
              int8 MMA ceiling measured live (ceilings/ceilings.cu: a pure tcgen05.mma.kind::i8 loop, burst and
              sustained), with the nominal 4.5 POP/s and the 2 x measured-bf16 fractions beside it
  "configs"   every BASELINE.json config; each tensor-regime config as `ms_per_step` (sustained) and
              `ms_per_step_burst`
  "modgemm", "ntt"   the ring-packing kernels at the paper's 64 GiB hybrid shape for 32
              clients, each with its roofline (--modgemm adds 1 and 8 clients and the offline H transform)
  "cpu_baseline"   the oracle on the host cores: median of 100 passes over the first 8192 rows of the headline
              DB -- the sample and procedure --impl reference uses, so the two agree

The DB (16 GiB) is far larger than the 126 MB L2, so no L2 flush is needed between steps.
N > 1 (torchrun): the path shards by DB rows with no data-path collective (each
GPU holds a (D1/#GPU) x D0 partition; queries are broadcast) -- every rank scans its own
16 GiB row shard (weak scaling); value = all ranks' bytes / max-over-ranks device time.

--impl reference times the CPU oracle (oracle/, as it stands) on this box's host cores on a
bounded row sample of the same workload and prints the same JSON line with "impl": "reference".
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "db_scan_GBps_16GiB_u8_batch1"
UNIT = "GB/s"
SEED = 0
SETTLE_S = 1.0  # steady-state loop before a tensor-regime config is timed (the part settles at its ~1 kW cap)

# BASELINE.json configs (rows, cols, batch, db_bits, prime moduli?)
CONFIGS = {
    "C1_tiny_B1": (1024, 1024, 1, 8, False),
    "C2_1GiB_B1": (32768, 32768, 1, 8, False),
    "C3_16GiB_B1": (131072, 131072, 1, 8, False),
    "C3_16GiB_B8": (131072, 131072, 8, 8, False),
    "C4_4GiB_B256": (65536, 65536, 256, 8, False),
    "C5_rns_u16_B64x2": (32768, 32768, 64, 16, True),
    # configs[4] with the u16 DB held as its two byte-limb planes ("split into 2 u8 limbs"; vipir_db_split_u16,
    # offline): 8 int8 MACs per product and 4 limb columns per query vector instead of the byte view's 10 and 5
    "C5_rns_u16_B64x2_planes": (32768, 32768, 64, 16, True),
}
LIMB_PLANE_CONFIGS = {"C5_rns_u16_B64x2_planes"}
# --paper: the paper's own plain-SimplePIR runs (Table 2: B = 32 at 1/4/16/64 GiB,
# D0 ~ sqrt(D), H100 NVL) and SURVEY.md 8(f) NEXT-2 shapes of the same product; context, not configs
PAPER_CONFIGS = {
    "P_1GiB_B32": (32768, 32768, 32, 8, False),
    "P_4GiB_B32": (65536, 65536, 32, 8, False),
    "P_16GiB_B32": (131072, 131072, 32, 8, False),
    "P_64GiB_B32": (262144, 262144, 32, 8, False),
    "P_64GiB_B1": (262144, 262144, 1, 8, False),
    # throughput against batch size at a fixed DB (the paper's Fig 6 sweeps B = 1..32; B = 1, 8, 32 are above)
    "F6_16GiB_B2": (131072, 131072, 2, 8, False),
    "F6_16GiB_B4": (131072, 131072, 4, 8, False),
    "F6_16GiB_B16": (131072, 131072, 16, 8, False),
    "N2_hint_4GiB_B1280": (65536, 65536, 1280, 8, False),
    "N2_tall_64GiB_B1": (1 << 20, 65536, 1, 8, False),
    # DoublePIR / double-packing second folding, one client: (8N x D1) INT8 by D1 x (n+1) INT32
    "N2_fold2_4GiB_B1281": (32768, 131072, 1281, 8, False),
}
PAPER_QPS_H100 = {"P_1GiB_B32": 8244, "P_4GiB_B32": 2201, "P_16GiB_B32": 565, "P_64GiB_B32": 144}
HEADLINE = "C3_16GiB_B1"
BATCHED = "C4_4GiB_B256"


# ---- host-side helpers (also exercised by the gloo tests) -------------------------------------

def shard_rows(rank: int, world: int, rows_per_gpu: int):
    """Weak scaling over DB rows: rank r owns global rows [r*rows_per_gpu, (r+1)*rows_per_gpu)
    of a (world*rows_per_gpu) x cols database (row sharding)."""
    return rank * rows_per_gpu, (rank + 1) * rows_per_gpu


def aggregate(per_rank_ms, units_per_rank: float, steps: int):
    """Whole-job throughput: all ranks' units / the slowest rank's device time."""
    t_ms = max(per_rank_ms)
    total_units = units_per_rank * len(per_rank_ms) * steps
    return total_units / (t_ms * 1e-3), t_ms / steps


def measured_peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        d = json.loads(f.read_text())
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_burst": float(d["bf16_tflops"]),
                "bf16_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "source": "measured"}
    # fallback stated in B200_PROFILING.md
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "source": "fallback"}


def profiled_traffic(kernel: str):
    """dram bytes per launch of `kernel` from the committed ncu --set full capture, or None."""
    f = ROOT / "profiles" / "traffic.json"
    if f.exists():
        return json.loads(f.read_text()).get(kernel)
    return None


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.01):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        self.index, self.period = index, period_s
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    _NAMES = {
        0x0000000000000004: "sw_power_cap", 0x0000000000000008: "hw_slowdown",
        0x0000000000000020: "sw_thermal_slowdown", 0x0000000000000040: "hw_thermal_slowdown",
        0x0000000000000080: "hw_power_brake_slowdown", 0x0000000000000002: "applications_clocks_setting",
        0x0000000000000010: "sync_boost", 0x0000000000000100: "display_clocks_setting",
    }

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                r = self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for bit, name in self._NAMES.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


# ---- the CUDA arm ---------------------------------------------------------------------------

def time_events(fn, steps, warmup, stream):
    import torch
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        fn()
    e1.record(stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)  # ms for `steps` calls


def step_spread(fn, steps, stream):
    """Median and best single-step time (an event after every step; SURVEY.md 8(d) asks for both).  Reported beside the
    K-step total, which stays the value's basis."""
    import torch
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    ev[0].record(stream)
    for i in range(steps):
        fn()
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    t = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(steps))
    return {"median": t[len(t) // 2], "best": t[0], "worst": t[-1]}


def two_in_flight(rows, cols, batch, db_bits, moduli, layout, d_db, h_q, d_ref, steps):
    """A server that overlaps requests makes one plan per stream (include/vipir.h): two host threads, each with its own
    plan, stream and pinned buffers, call vipir_dbmul_host back to back against the same resident DB -- the copies of one
    request run beside the scan of the other.  Returns ms per request (all requests / the slower thread's device time,
    CUDA events on each thread's stream), after both threads have settled for a second."""
    import torch
    from paper_2606_11536_b200 import vipir
    T = h_q.shape[0]
    streams = [torch.cuda.Stream() for _ in range(2)]
    plans = [vipir.Plan(rows, cols, batch, db_bits, moduli, db_layout=layout) for _ in range(2)]
    bufs = [(h_q if i == 0 else h_q.clone().pin_memory(), torch.empty((T, batch, rows), dtype=torch.int32).pin_memory())
            for i in range(2)]
    ms = [0.0, 0.0]
    start = threading.Barrier(2)

    def worker(i):
        torch.cuda.set_device(d_db.device)
        with torch.cuda.stream(streams[i]):
            t_end = time.perf_counter() + SETTLE_S
            while time.perf_counter() < t_end:
                plans[i].host(d_db, bufs[i][0], bufs[i][1])
            start.wait()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(streams[i])
            for _ in range(steps):
                plans[i].host(d_db, bufs[i][0], bufs[i][1])
            e1.record(streams[i])
            streams[i].synchronize()
            ms[i] = e0.elapsed_time(e1)
    th = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    for i in range(2):
        if not torch.equal(bufs[i][1].cuda(), d_ref):
            raise RuntimeError("two requests in flight: an answer differs from vipir_dbmul's")
        plans[i].close()
    return max(ms) / (2 * steps)


MIN_WINDOW_MS = 100.0  # a step under 2 ms is timed over at least this long a window (the clock oscillates at the power cap)


def run_config(name, device_db, steps, warmup, peaks, with_e2e=False, row_offset_bytes=0, spread=False, exact_steps=False):
    """Times one config on the current device; returns a dict of measurements.  Every config that runs on the tensor
    cores is timed in the power-capped steady state (a 1 s settle loop first: `ms_per_step`, the number of record)
    and as a burst (`ms_per_step_burst`: the first steps after 0.5 s of idle).  Unless exact_steps (the headline: the
    contract's exactly-K steps), whatever takes under 2 ms per call is re-timed over a window of >= MIN_WINDOW_MS
    (`timed_steps` says how many calls that was), the step, the scan kernel and the splitter alike."""
    import torch
    from paper_2606_11536_b200 import inputs, vipir
    from paper_2606_11536_b200.inputs import device
    rows, cols, batch, db_bits, prime = (CONFIGS.get(name) or PAPER_CONFIGS[name])
    moduli = inputs.rns_primes(SEED) if prime else None
    kb = cols * db_bits // 8
    d_db = device_db[row_offset_bytes: row_offset_bytes + rows * kb].view(rows, kb)
    d_q = device.query(SEED, cols, batch, moduli)
    T = d_q.shape[0]
    d_a = torch.empty((T, batch, rows), dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream()
    out = {"rows": rows, "cols": cols, "batch": batch, "db_bits": db_bits, "moduli": moduli or "2^32"}
    layout = vipir.DB_ROW_MAJOR
    if name in LIMB_PLANE_CONFIGS:  # offline re-layout of the static DB, timed once and reported beside the step
        layout = vipir.DB_LIMB_PLANES
        d_planes = torch.empty_like(d_db)
        ms_prep = time_events(lambda: vipir.db_split_u16(d_db, d_planes, rows, cols), 1, 0, stream)
        out.update({"db_layout": "limb_planes", "ms_db_split_offline": ms_prep})
        d_db = d_planes

    def settle(fn, seconds=SETTLE_S):
        t_end = time.perf_counter() + seconds
        while time.perf_counter() < t_end:
            for _ in range(20):
                fn()
            torch.cuda.synchronize()

    with vipir.Plan(rows, cols, batch, db_bits, moduli, db_layout=layout) as plan:
        info = plan.info
        tensor = info["regime_name"] != "gemv"
        if tensor:
            plan(d_db, d_q, d_a)
            torch.cuda.synchronize()
            time.sleep(0.5)
            out["ms_per_step_burst"] = time_events(lambda: plan(d_db, d_q, d_a), 3, 0, stream) / 3
            settle(lambda: plan(d_db, d_q, d_a))
        def timed(fn):
            ms = time_events(fn, steps, warmup, stream) / steps
            n = steps
            if not exact_steps and ms < 2.0 and ms * steps < MIN_WINDOW_MS:
                n = int(MIN_WINDOW_MS / max(ms, 1e-3)) + 1
                ms = time_events(fn, n, 0, stream) / n
            return ms, n
        ms_step, out["timed_steps"] = timed(lambda: plan(d_db, d_q, d_a))
        if spread:  # headline config: spread of the single steps as well
            out["ms_step_spread"] = step_spread(lambda: plan(d_db, d_q, d_a), min(steps, 50), stream)
        # the dominant kernel alone (planes already in the workspace) and the splitter alone
        if info["launches"] == 1:   # GEMV with the split fused in: the step IS the scan kernel (same timed region)
            ms_scan = ms_step
        else:
            ms_scan, _ = timed(lambda: vipir.dbmul_scan(plan.handle, d_db, d_a))
        ms_split, _ = timed(lambda: vipir.split_limbs(plan.handle, d_q))
        if with_e2e:
            # the public host call (vipir_dbmul_host): query from pinned host memory in, answer in host memory out,
            # stream sync -- every step; the tensor regimes pipeline it over K slices (include/vipir.h)
            h_q = d_q.cpu().pin_memory()
            h_a = torch.empty((T, batch, rows), dtype=torch.int32).pin_memory()
            if tensor:
                settle(lambda: plan.host(d_db, h_q, h_a))
            for _ in range(warmup):
                plan.host(d_db, h_q, h_a)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(steps):
                plan.host(d_db, h_q, h_a)
            e1.record(stream)
            torch.cuda.synchronize()
            out["e2e_ms"] = e0.elapsed_time(e1) / steps
            out["h2d_bytes"] = h_q.numel() * 4
            out["d2h_bytes"] = h_a.numel() * 4
            # what the host link itself does on this box (one plain pinned copy each way), for context
            d_tmp = torch.empty_like(d_q)
            out["pcie_h2d_GBps"] = h_q.numel() * 4 / (time_events(lambda: d_tmp.copy_(h_q, non_blocking=True), 5, 2, stream) / 5) / 1e6
            out["pcie_d2h_GBps"] = h_q.numel() * 4 / (time_events(lambda: h_q.copy_(d_tmp, non_blocking=True), 5, 2, stream) / 5) / 1e6
            if not torch.equal(h_a.cuda(), d_a):
                raise RuntimeError(f"{name}: vipir_dbmul_host and vipir_dbmul disagree")
            if tensor:
                out["e2e_two_in_flight_ms"] = two_in_flight(rows, cols, batch, db_bits, moduli, layout, d_db, h_q, d_a, steps)
            del h_q, h_a, d_tmp
    db_bytes = rows * kb
    nq, lc = info["query_vectors"], info["limb_cols"]
    logical_ops = 2.0 * rows * cols * nq
    int8_ops = 2.0 * rows * kb * nq * lc  # what the tensor pipe executes (limb MACs)
    # what the method asks for: four query limbs x the DB element's byte limbs per product -- 4 int8
    # MACs for a u8 DB, 8 for u16; the byte view of a u16 DB executes 10
    method_ops = 2.0 * rows * cols * nq * 4 * (db_bits // 8)
    alg_bytes = db_bytes + 4 * cols * nq + 4 * rows * nq  # DB + query + answer
    out.update({
        "regime": info["regime_name"], "ms_per_step": ms_step, "ms_scan_kernel": ms_scan, "ms_split_kernel": ms_split,
        "db_GBps": db_bytes / ms_step / 1e6, "scan_kernel_GBps": alg_bytes / ms_scan / 1e6,
        "logical_TOPS": logical_ops / ms_step / 1e9, "int8_TOPS": int8_ops / ms_step / 1e9,
        "scan_kernel_int8_TOPS": int8_ops / ms_scan / 1e9,
        "frac_hbm_measured": alg_bytes / ms_scan / 1e6 / peaks["hbm_gbs"],
        "frac_hbm_nominal_8TBps": db_bytes / ms_step / 1e6 / 8000.0,
        "frac_int8_nominal_4500": int8_ops / ms_step / 1e9 / 4500.0,
        "plan": {k: info[k] for k in ("tile_cols", "mma_n", "m_tiles", "n_tiles", "n_chunks", "k_chunk_bytes", "stages",
                                       "grid", "smem_bytes", "launches")},
        "alg_bytes": alg_bytes, "int8_ops": int8_ops, "method_int8_ops": method_ops,
    })
    if tensor and peaks.get("mma_i8_sustained_TOPS"):
        # the scan kernel against the int8 MMA ceiling measured live in this run (ceilings.cu, sustained): the limb MACs
        # it executes, and the method's own (what the answer needs)
        ceil = peaks["mma_i8_sustained_TOPS"]
        out["frac_mma_ceiling_executed"] = int8_ops / ms_scan / 1e9 / ceil
        out["frac_mma_ceiling_method"] = method_ops / ms_scan / 1e9 / ceil
    del d_q, d_a
    return out


# ---- the parallel modular GEMMs of the ring-packing stage --------------------

MODGEMM_SHAPE = (3, 4096, 256, 1280)  # T = #RNS, NC = N, M = D_r, K = n: the 64 GiB hybrid protocol
MODGEMM_PRIMES = [536608769, 533463041, 531628033]  # < 2^29, = 1 mod 2^18


def run_modgemm(B, steps, warmup, peaks):
    """Out = H*C + (0|G) mod q_t at the paper's shape for B clients (ncols = 2B, gcols = B)."""
    import torch
    from paper_2606_11536_b200 import vipir
    from paper_2606_11536_b200.inputs import device, generator
    T, NC, M, K = MODGEMM_SHAPE
    ncols, gcols = 2 * B, B
    stream = torch.cuda.current_stream()
    d_H = device.modgemm_operand(SEED, generator.STREAM_MG_H, MODGEMM_PRIMES, NC, M * K)
    d_C = device.modgemm_operand(SEED, generator.STREAM_MG_C, MODGEMM_PRIMES, NC, ncols * K)
    d_G = device.modgemm_operand(SEED, generator.STREAM_MG_G, MODGEMM_PRIMES, NC, gcols * M)
    d_O = torch.empty((T, NC, ncols, M), dtype=torch.int32, device="cuda")
    with vipir.ModGemmPlan(T, NC, M, K, ncols, gcols, MODGEMM_PRIMES) as plan:
        ms_set_h = time_events(lambda: plan.set_h(d_H), 3, 1, stream) / 3   # offline step, reported apart
        del d_H
        info = plan.info
        # the step: ONE kernel (C split into limbs inside the products kernel); sustained like every tensor-touching leg
        t_end = time.perf_counter() + SETTLE_S
        while time.perf_counter() < t_end:
            for _ in range(10):
                plan(d_C, d_G, d_O)
            torch.cuda.synchronize()
        ms_step = time_events(lambda: plan(d_C, d_G, d_O), steps, warmup, stream) / steps
        # the two-kernel form (C limb planes written by a pre-pass), for comparison
        ms_split = time_events(lambda: vipir.modgemm_split_c(plan.handle, d_C), steps, warmup, stream) / steps
        ms_prod = time_events(lambda: vipir.modgemm_products(plan.handle, d_G, d_O), steps, warmup, stream) / steps
    macs = float(T) * NC * M * ncols * K
    out_bytes = 4.0 * T * NC * ncols * M
    c_bytes = 4.0 * T * NC * ncols * K   # raw words of C (fused) -- the same count as its four limb planes
    alg_bytes = info["h_limb_bytes"] + c_bytes + out_bytes + 4.0 * T * NC * gcols * M
    fused = bool(info["fused_split"])
    return {
        "workload": f"{T * NC} problems of {M} x {ncols} x {K} u32 mod q_t (B = {B} clients; H = {info['h_limb_bytes'] / 2**30:.1f} GiB)",
        "ms_per_step": ms_step, "fused_split": fused,
        "two_kernel_form": {"ms_products_kernel": ms_prod, "ms_split_c_kernel": ms_split},
        "ms_set_h_offline": ms_set_h,
        "modmac_T_per_s": macs / ms_step / 1e9, "int8_TOPS": 32.0 * macs / ms_step / 1e9,
        "H_GBps": info["h_limb_bytes"] / ms_step / 1e6,
        "roofline": {"bound": "hbm", "kernel": f"modgemm_i8_kernel<{info['cta_group']},{'true' if fused else 'false'}>",
                     "achieved": alg_bytes / ms_step / 1e6, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                     "frac": alg_bytes / ms_step / 1e6 / peaks["hbm_gbs"], "alg_bytes_per_launch": alg_bytes,
                     "ms_per_launch": ms_step,
                     "traffic": profiled_traffic("modgemm_i8_kernel_B%d" % B)},
        "plan": {k: info[k] for k in ("cta_group", "tile_cols", "mma_n", "m_tiles", "n_tiles", "n_chunks", "a_stages",
                                       "b_stages", "acc_stages", "smem_bytes", "grid", "launches")},
    }


def run_ntt(n_a, layout_name, steps, warmup):
    """Lift + forward NTT (N = 2^12, the 3 RNS primes) of n_a x 256 polynomials into G or H."""
    import torch
    from paper_2606_11536_b200 import vipir
    from paper_2606_11536_b200.inputs import device
    N, M, p_bits = 4096, MODGEMM_SHAPE[2], 18
    psi = [next(x for x in range(2, q) if pow(x, N, q) == q - 1) for q in MODGEMM_PRIMES]
    q_all = MODGEMM_PRIMES[0] * MODGEMM_PRIMES[1] * MODGEMM_PRIMES[2]
    scale = [(q_all >> p_bits) % q for q in MODGEMM_PRIMES] if layout_name == "G" else [1, 1, 1]
    layout = vipir.NTT_LAYOUT_G if layout_name == "G" else vipir.NTT_LAYOUT_H
    d_X = device.query(SEED, M * N, n_a)[0].view(torch.int32)
    d_X = (d_X >> (32 - p_bits)) & ((1 << p_bits) - 1)                  # words < 2^18, as after the fused switch
    T = len(MODGEMM_PRIMES)
    d_O = torch.empty((T, N, n_a, M) if layout_name == "G" else (T, N, M, n_a), dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream()
    with vipir.NttPlan(12, MODGEMM_PRIMES, psi, scale, p_bits) as plan:
        ms = time_events(lambda: plan(d_X, n_a, M, layout, d_O), steps, warmup, stream) / steps
        bad = plan.bad_input()
    polys = float(n_a) * M * T
    # ALU bound: N/2 * log2 N = 24576 Harvey butterflies per transform, against the butterfly rate of this part
    # measured live (ceilings.butterflies: the same butterfly on registers only, no shared memory, no global
    # traffic -- both integer pipes counted, whatever clock the part sustains)
    bf = polys * 24576
    ceil = butterfly_ceiling(MODGEMM_PRIMES[0])
    alg_bytes = 4.0 * n_a * M * N * (1 + T)
    return {"workload": f"{n_a} x {M} polynomials, N = 4096, {T} primes -> {layout_name}", "ms": ms, "bad_input": bad,
            "transforms_per_s": polys / ms * 1e3, "GBps_in_plus_out": alg_bytes / ms / 1e6,
            "roofline": {"bound": "alu", "kernel": "ntt_lift_kernel<12>", "achieved": bf / ms / 1e6,
                         "peak": ceil["G_butterflies_per_s"], "unit": "G butterflies/s (Harvey, INT32)",
                         "peak_source": "measured live: register-only butterfly loop (ceilings.cu), " + ceil["how"],
                         "frac": bf / ms / 1e6 / ceil["G_butterflies_per_s"],
                         "frac_of_derived_alu_pipe_peak": bf * 4 / ms * 1e3 / (148 * 64 * 1.965e9),
                         "traffic": profiled_traffic("ntt_lift_kernel_G_B32") if (n_a, layout_name) == (32, "G") else None}}


_BF_CEIL = {}


def butterfly_ceiling(q):
    """Harvey butterflies per second of the whole part, registers only (the ALU ceiling of the NTT's passes)."""
    if not _BF_CEIL:
        import torch
        from paper_2606_11536_b200 import ceilings
        stream = torch.cuda.current_stream()
        iters = 4096
        n = [0.0]

        def go():
            n[0] = ceilings.butterflies(iters, q)
        ms = time_events(go, 10, 3, stream) / 10
        _BF_CEIL.update({"G_butterflies_per_s": n[0] / ms / 1e6, "ms_per_launch": ms,
                         "how": f"{iters} x 32 butterflies per thread, 148 x 512 threads, 10 launches"})
    return _BF_CEIL


def mma_i8_ceiling():
    """The int8 tensor pipe alone (ceilings.cu: tcgen05.mma.cta_group::2.kind::i8 M256 N256 K32 back to back on
    operands resident in shared memory, every SM pair): as a burst after idle and sustained under the power cap."""
    import torch
    from paper_2606_11536_b200 import ceilings
    stream = torch.cuda.current_stream()
    iters = 6144   # x 4 MMAs x 128 clocks: ~1.7-2.2 ms per launch
    ops = [0.0]

    def go():
        ops[0] = ceilings.mma_i8(iters)
    go()
    torch.cuda.synchronize()
    time.sleep(0.5)
    ms_burst = time_events(go, 2, 0, stream) / 2
    t_end = time.perf_counter() + 2.0
    while time.perf_counter() < t_end:
        for _ in range(50):
            go()
        torch.cuda.synchronize()
    ms_sus = time_events(go, 50, 0, stream) / 50
    return {"burst_TOPS": ops[0] / ms_burst / 1e9, "sustained_TOPS": ops[0] / ms_sus / 1e9,
            "how": f"{iters} x 4 MMAs (M256 N256 K32, cta_group::2) per SM pair per launch; burst = 2 launches after "
                   "0.5 s idle, sustained = 50 launches after a 2 s loop; pseudo-random operand bytes in shared memory"}


def run_pipeline(B, steps, warmup, offline_hint=False):
    """The built chain at the paper's 64 GiB hybrid shape (N x D_r x D0 = 2^12 x 2^8 x 2^16):
    (1) scan of the 64 GiB DB for B clients with the fused 2^32 -> 2^18 switch, lift + NTT of its output into G,
    (3) H*C + (0|G) over the 15 GiB hint -- everything of the online server path except the expansion that
    produces C and the poly-HE folding (7)."""
    import torch
    from paper_2606_11536_b200 import vipir
    from paper_2606_11536_b200.inputs import device, generator
    T, NC, M, K = MODGEMM_SHAPE
    N, p_bits = NC, 18
    rows, cols = N * M, 1 << 16
    stream = torch.cuda.current_stream()
    d_db = device.db(SEED, rows, cols, 8)
    d_q = device.query(SEED, cols, B)
    d_a = torch.empty((1, B, rows), dtype=torch.int32, device="cuda")
    d_G = torch.empty((T, N, B, M), dtype=torch.int32, device="cuda")
    d_O = torch.empty((T, NC, 2 * B, M), dtype=torch.int32, device="cuda")
    d_C = device.modgemm_operand(SEED, generator.STREAM_MG_C, MODGEMM_PRIMES, NC, 2 * B * K)
    psi = [next(x for x in range(2, q) if pow(x, N, q) == q - 1) for q in MODGEMM_PRIMES]
    q_all = MODGEMM_PRIMES[0] * MODGEMM_PRIMES[1] * MODGEMM_PRIMES[2]
    scale = [(q_all >> p_bits) % q for q in MODGEMM_PRIMES]
    with vipir.Plan(rows, cols, B, 8, None, modswitch_bits=p_bits) as scan, \
            vipir.NttPlan(12, MODGEMM_PRIMES, psi, scale, p_bits) as ntt, \
            vipir.ModGemmPlan(T, NC, M, K, 2 * B, B, MODGEMM_PRIMES) as mg:
        # ---- offline phase: hint = DB x (D0 x n) public matrix, switched to 2^18, NTT along N -> H ----
        offline = {}
        if offline_hint:
            d_A = device.query(SEED + 1, cols, K)                                  # the public D0 x n matrix, [1][n][cols]
            d_hint = torch.empty((1, K, rows), dtype=torch.int32, device="cuda")
            with vipir.Plan(rows, cols, K, 8, None, modswitch_bits=p_bits) as hint_scan, \
                    vipir.NttPlan(12, MODGEMM_PRIMES, psi, [1, 1, 1], p_bits) as ntt_h:
                offline["ms_hint_scan"] = time_events(lambda: hint_scan(d_db, d_A, d_hint), 1, 1, stream)
                del d_A
                d_H = torch.empty((T, N, M, K), dtype=torch.int32, device="cuda")
                offline["ms_ntt_H"] = time_events(lambda: ntt_h(d_hint, K, M, vipir.NTT_LAYOUT_H, d_H), 1, 1, stream)
                del d_hint
        else:
            d_H = device.modgemm_operand(SEED, generator.STREAM_MG_H, MODGEMM_PRIMES, NC, M * K)
        offline["ms_set_h"] = time_events(lambda: mg.set_h(d_H), 1, 0, stream)
        torch.cuda.synchronize()
        del d_H
        torch.cuda.empty_cache()

        def step():
            scan(d_db, d_q, d_a)
            ntt(d_a, B, M, vipir.NTT_LAYOUT_G, d_G)
            mg(d_C, d_G, d_O)
        ms = time_events(step, steps, warmup, stream) / steps
        ms_scan = time_events(lambda: scan(d_db, d_q, d_a), steps, warmup, stream) / steps
        ms_ntt = time_events(lambda: ntt(d_a, B, M, vipir.NTT_LAYOUT_G, d_G), steps, warmup, stream) / steps
        ms_mg = time_events(lambda: mg(d_C, d_G, d_O), steps, warmup, stream) / steps
        bad = ntt.bad_input()
        regime = scan.info["regime_name"]
        n_kernels = scan.info["launches"] + 1 + mg.info["launches"]
    return {"workload": f"64 GiB u8 DB 2^20 x 2^16, B = {B}; N = 4096, D_r = 256, n = 1280, 3 RNS primes",
            "ms_per_batch": ms, "queries_per_s": B / ms * 1e3, "ms_scan": ms_scan, "ms_ntt_G": ms_ntt,
            "ms_modgemm": ms_mg, "scan_regime": regime, "kernels_per_batch": n_kernels, "ntt_bad_input": bad,
            "resident_GB": (rows * cols + 4.0 * T * NC * M * 1280) / 1e9, "offline": offline}


def oracle_passes(D, Q, passes, cores):
    """`passes` timed oracle.dbmul calls over the same sample; returns the per-pass seconds."""
    import oracle
    t = []
    for _ in range(passes):
        t0 = time.perf_counter()
        oracle.dbmul(D, Q, nthreads=cores)
        t.append(time.perf_counter() - t0)
    return t


CPU_PASSES = 100  # fixed: about 5-10 s of wall time on the sample below (1 GiB of DB per pass)


def cpu_baseline(sample_rows: int, device_db, cols: int):
    """The oracle, as it stands, on the host cores, on the first `sample_rows` rows of the headline workload (same
    bytes: copied back from the device-generated DB): CPU_PASSES passes, the median pass is the value.
    --impl reference times the same sample the same way (its value is the K-step total the contract asks for)."""
    import numpy as np
    import oracle
    from paper_2606_11536_b200 import inputs
    D = device_db[: sample_rows * cols].view(sample_rows, cols).cpu().numpy()
    Q = inputs.query(SEED, cols, 1)
    cores = os.cpu_count() or 1
    oracle_passes(D, Q, 3, cores)  # load + warm
    t = oracle_passes(D, Q, CPU_PASSES, cores)
    med = sorted(t)[len(t) // 2]
    # one thread, on the first 1024 rows (128 MiB) of the same sample (single- and all-thread times)
    t1 = sorted(oracle_passes(D[:1024], Q, 5, 1))[2]
    return {"value": D.size / med / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "value_from_total": len(t) * D.size / sum(t) / 1e9, "best_pass_GBps": D.size / min(t) / 1e9,
            "single_thread_GBps": D[:1024].size / t1 / 1e9,
            "sample": f"median of {len(t)} passes over the first {sample_rows} of 131072 rows x 131072 cols, batch 1 "
                      f"({D.size / 2**30:.0f} GiB of DB per pass), {sum(t):.2f} s wall on {cores} threads "
                      f"= {sum(t) * cores:.0f} core-seconds", "seconds": sum(t)}


def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2606_11536_b200 import build, vipir
    from paper_2606_11536_b200.inputs import device, generator

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    build.build()
    vipir.load()
    peaks = measured_peaks()

    if args.only:
        # one named config alone (a BASELINE.json config or a --paper shape), e.g. as the target of an ncu capture:
        # prints that config's measurements, not the bench line
        r_, c_, _, bits_, _ = CONFIGS.get(args.only) or PAPER_CONFIGS[args.only]
        buf = device.db(SEED, r_, c_, bits_).view(-1)
        torch.cuda.synchronize()
        print(json.dumps({"only": args.only, **run_config(args.only, buf, args.steps, args.warmup, peaks)}))
        return
    rows, cols, _, _, _ = CONFIGS[HEADLINE]
    # this rank's row shard of the (world*rows) x cols DB: same stream, offset by the shard's first byte
    r0, _ = shard_rows(rank, world, rows)
    nbytes = rows * cols
    alloc_bytes = max([nbytes] + [r * c * b // 8 for r, c, _, b, _ in PAPER_CONFIGS.values()]) if args.paper else nbytes
    buf = torch.empty(alloc_bytes, dtype=torch.uint8, device="cuda")
    lib = device._load()
    import ctypes
    key = generator.stream_key(SEED + 1000003 * rank, generator.STREAM_DB) if world > 1 else generator.stream_key(SEED, generator.STREAM_DB)
    rc = lib.vipir_inputs_fill_bytes(buf.data_ptr(), alloc_bytes, key, ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == 0
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- headline: timed region bracketed by barrier + synchronize, clocks sampled during it ----
    barrier()
    with ClockSampler(local_rank) as clk:
        head = run_config(HEADLINE, buf, args.steps, args.warmup, peaks, with_e2e=True, spread=True, exact_steps=True)
    barrier()
    times = [head["ms_per_step"] * args.steps]
    e2e_times = [head["e2e_ms"] * args.steps]
    if world > 1:
        t = torch.tensor([times[0], e2e_times[0]], dtype=torch.float64, device="cuda")
        gathered = [torch.zeros_like(t) for _ in range(world)]
        dist.all_gather(gathered, t)
        times = [float(g[0]) for g in gathered]
        e2e_times = [float(g[1]) for g in gathered]
    # read-only ceiling of this part, measured live on the same buffer (plain 128-bit loads, data discarded)
    ro_ms = time_events(lambda: device.read_only(buf[:nbytes]), 10, 3, torch.cuda.current_stream()) / 10
    read_only_gbs = nbytes / ro_ms / 1e6
    value, ms_per_step = aggregate(times, nbytes / 1e9, args.steps)
    e2e_value, _ = aggregate(e2e_times, nbytes / 1e9, args.steps)

    extra = {}
    cpu = None
    mma_ceil = None
    if rank == 0 and world == 1:
        mma_ceil = mma_i8_ceiling()
        peaks["mma_i8_sustained_TOPS"] = mma_ceil["sustained_TOPS"]
        # every BASELINE.json config rides along at N = 1 (a few seconds); --headline-only keeps just configs[2] and [3]
        for name in ([BATCHED] if args.headline_only else [n for n in CONFIGS if n != HEADLINE]):
            extra[name] = run_config(name, buf, args.steps, max(3, args.warmup), peaks, with_e2e=(name == BATCHED))
        if args.paper:
            # the read-only ceiling on the buffer each paper workload scans (the 64 GiB ones against 64 GiB of loads:
            # TLB reach and refresh are the part's, whatever they cost)
            ro = {}
            for label, nb in (("16GiB", 16 << 30), ("64GiB", 64 << 30)):
                if nb <= alloc_bytes:
                    ms = time_events(lambda: device.read_only(buf[:nb]), 5, 2, torch.cuda.current_stream()) / 5
                    ro[label] = nb / ms / 1e6
            extra["paper_read_only"] = {"GBps": ro, "how": "plain 128-bit loads over the first 16 / 64 GiB of the same buffer, 5 passes"}
            for name in PAPER_CONFIGS:
                extra[name] = run_config(name, buf, max(10, args.steps // 5), 3, peaks)
                r_, c_, _, bits_, _ = PAPER_CONFIGS[name]
                label = {16 << 30: "16GiB", 64 << 30: "64GiB"}.get(r_ * c_ * bits_ // 8)
                if label in ro:
                    extra[name]["read_only_ceiling_GBps"] = ro[label]
                    extra[name]["frac_of_read_only_ceiling"] = extra[name]["scan_kernel_GBps"] / ro[label]
                if name in PAPER_QPS_H100:
                    extra[name]["qps_batch32"] = 32.0 / (extra[name]["ms_per_step"] * 1e-3)
                    extra[name]["paper_qps_h100_nvl"] = PAPER_QPS_H100[name]
        cpu = cpu_baseline(args.cpu_sample_rows, buf, cols)
        # the ring-packing kernels at the paper's 64 GiB hybrid shape: B = 32 in the default line, the sweep on request
        if not args.headline_only or args.modgemm:
            mg_B = (1, 8, 32) if args.modgemm else (32,)
            extra["modgemm"] = {f"B{B}": run_modgemm(B, max(10, args.steps // 5), 3, peaks) for B in mg_B}
            extra["ntt"] = {"G_B32": run_ntt(32, "G", 300, 5)}  # ~0.4 ms per launch: a window above 100 ms
            if args.modgemm:
                extra["ntt"].update({"G_B1": run_ntt(1, "G", 50, 5), "H_n1280_offline": run_ntt(1280, "H", 3, 1)})
        if args.pipeline:
            del buf
            torch.cuda.empty_cache()
            extra["pipeline"] = {f"B{B}": run_pipeline(B, max(10, args.steps // 5), 3, offline_hint=(B == 1))
                                 for B in (1, 8, 32)}

    if rank == 0:
        b = extra.get(BATCHED)
        roofline = {"bound": "hbm", "kernel": "gemv_b1_kernel", "achieved": head["scan_kernel_GBps"],
                    "peak": peaks["hbm_gbs"], "peak_source": peaks["source"] + " copy bandwidth (MEASURED_PEAKS.json)"
                    if peaks["source"] == "measured" else "fallback 6650 GB/s (B200_PROFILING.md)",
                    "unit": "GB/s", "frac": head["frac_hbm_measured"],
                    "frac_of_nominal_8TBps": head["scan_kernel_GBps"] / 8000.0,
                    "read_only_ceiling_GBps": read_only_gbs,
                    "frac_of_read_only_ceiling": head["scan_kernel_GBps"] / read_only_gbs,
                    "ms_per_launch": head["ms_scan_kernel"], "alg_bytes_per_launch": head["alg_bytes"],
                    "traffic": profiled_traffic("gemv_b1_kernel")}
        e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": head["h2d_bytes"],
               "d2h_bytes_per_step": head["d2h_bytes"], "ms_per_step": head["e2e_ms"]}
        batched = None
        if b:
            sus = mma_ceil["sustained_TOPS"]
            batched = {
                "workload": "configs[3]: 4 GiB u8 DB 65536x65536, Q 65536x256 u32, q=2^32, 4 int8 limbs, K chunks <= 32768",
                "ms_per_step": b["ms_per_step"], "ms_per_step_burst": b["ms_per_step_burst"],
                "db_GBps": b["db_GBps"], "logical_TOPS": b["logical_TOPS"],
                "int8_TOPS": b["int8_TOPS"], "regime": b["regime"],
                "e2e": {"ms_per_step": b["e2e_ms"], "int8_TOPS": b["int8_ops"] / b["e2e_ms"] / 1e9,
                        "db_GBps": b["rows"] * b["cols"] / b["e2e_ms"] / 1e6,
                        "ratio_to_device_step": b["e2e_ms"] / b["ms_per_step"],
                        "two_requests_in_flight": {
                            "ms_per_request": b["e2e_two_in_flight_ms"],
                            "ratio_to_device_step": b["e2e_two_in_flight_ms"] / b["ms_per_step"],
                            "how": "two host threads, each with its own plan, stream and pinned buffers, calling "
                                   "vipir_dbmul_host back to back on the same resident DB"},
                        "h2d_bytes_per_step": b["h2d_bytes"], "d2h_bytes_per_step": b["d2h_bytes"],
                        "pcie_h2d_GBps": b["pcie_h2d_GBps"], "pcie_d2h_GBps": b["pcie_d2h_GBps"],
                        "how": "vipir_dbmul_host: H2D, limb split and scan pipelined over K slices, the answer "
                               "copied into mapped pinned host memory tile by tile; sustained (1 s settle)"},
                "roofline": {"bound": "tensor", "kernel": "gemm_i8_kernel<2,4,false>", "achieved": b["scan_kernel_int8_TOPS"],
                             "peak": sus, "unit": "TOP/s (int8)",
                             "peak_source": "measured live, sustained: pure tcgen05.mma.kind::i8 loop (ceilings.cu); "
                                            + mma_ceil["how"],
                             "frac": b["scan_kernel_int8_TOPS"] / sus,
                             "int8_mma_ceiling_TOPS": {"burst": mma_ceil["burst_TOPS"], "sustained": sus},
                             "achieved_burst": b["int8_ops"] / b["ms_per_step_burst"] / 1e9,
                             "frac_burst_of_burst_ceiling": b["int8_ops"] / b["ms_per_step_burst"] / 1e9 / mma_ceil["burst_TOPS"],
                             "frac_of_nominal_4500": b["scan_kernel_int8_TOPS"] / 4500.0,
                             "frac_of_2x_measured_sustained_bf16": b["scan_kernel_int8_TOPS"] / (2.0 * peaks["bf16_sustained"]),
                             "ms_per_launch": b["ms_scan_kernel"], "int8_ops_per_launch": b["int8_ops"],
                             "traffic": profiled_traffic("gemm_i8_kernel")},
            }
            # compact copies inside the two objects every record of this line keeps whole (`roofline`, `e2e`)
            br = batched["roofline"]
            roofline["batched"] = {
                "workload": "configs[3] 4 GiB u8, B = 256", "bound": "tensor", "kernel": br["kernel"],
                "achieved": br["achieved"], "peak": br["peak"], "unit": br["unit"],
                "peak_source": "int8 MMA ceiling measured live, sustained (ceilings.cu)", "frac": br["frac"],
                "frac_of_nominal_4500": br["frac_of_nominal_4500"], "ms_per_launch": br["ms_per_launch"],
                "ms_per_step": b["ms_per_step"], "ms_per_step_burst": b["ms_per_step_burst"], "traffic": br["traffic"]}
            e2e["batched"] = {
                "ms_per_step": b["e2e_ms"], "ratio_to_device_step": b["e2e_ms"] / b["ms_per_step"],
                "two_in_flight_ms": b["e2e_two_in_flight_ms"], "h2d_bytes_per_step": b["h2d_bytes"],
                "d2h_bytes_per_step": b["d2h_bytes"]}
            for key, cname in (("configs4_byte_view", "C5_rns_u16_B64x2"), ("configs4_limb_planes", "C5_rns_u16_B64x2_planes")):
                c = extra.get(cname)
                if c:
                    roofline[key] = {"bound": "tensor", "ms_per_step": c["ms_per_step"], "ms_per_launch": c["ms_scan_kernel"],
                                     "peak": sus, "unit": "TOP/s (int8)", "achieved_executed": c["scan_kernel_int8_TOPS"],
                                     "achieved_method": c["method_int8_ops"] / c["ms_scan_kernel"] / 1e9,
                                     "frac_executed": c["frac_mma_ceiling_executed"], "frac": c["frac_mma_ceiling_method"]}
        mg32 = extra.get("modgemm", {}).get("B32")
        if mg32:
            r = mg32["roofline"]
            roofline["modgemm_B32"] = {k: r[k] for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "ms_per_launch",
                                                          "traffic")}
        ntt32 = extra.get("ntt", {}).get("G_B32")
        if ntt32:
            r = ntt32["roofline"]
            roofline["ntt_G_B32"] = {"bound": r["bound"], "kernel": r["kernel"], "achieved": r["achieved"], "peak": r["peak"],
                                     "unit": r["unit"], "frac": r["frac"], "ms_per_launch": ntt32["ms"], "traffic": r["traffic"]}
        # key order: the per-config detail first, the objects of record last (a truncated tail of the line still holds them)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u8*u32->u32 (mod 2^32)", "data": "synthetic",
            "config": {"workload": "configs[2]: 16 GiB u8 DB 131072x131072 uniform, Q 131072x1 u32 uniform, q=2^32, "
                                   "seed 0; per GPU (row-sharded for N>1)",
                       "regime": head["regime"], "l2": "inputs (16 GiB) larger than L2; no flush",
                       "plan": head["plan"]},
        }
        if extra.get("paper_read_only"):
            line["paper_read_only_ceiling"] = extra.pop("paper_read_only")
        for key in ("modgemm", "ntt", "pipeline"):
            if key in extra:
                line[key] = extra.pop(key)
        if extra:
            drop = ("alg_bytes", "plan")
            line["configs"] = {n: {k: v for k, v in r.items() if k not in drop} for n, r in extra.items()}
            line["configs"][HEADLINE] = {k: v for k, v in head.items() if k not in drop}
        if batched:
            line["batched"] = batched
        line.update({
            "clocks": clk.summary(), "gpu_launches": head["plan"]["launches"] * args.steps,
            "ms_per_step_spread": head.get("ms_step_spread"),
            "cpu_baseline": cpu, "e2e": e2e, "roofline": roofline,
        })
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ---- the reference arm: the oracle on the host cores ---------------------------------------

def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np
    import oracle
    from paper_2606_11536_b200 import inputs
    rows, cols, _, _, _ = CONFIGS[HEADLINE]
    sample = args.ref_sample_rows
    cores = os.cpu_count() or 1
    oracle.build()
    D = inputs.db_rows(SEED, rows, cols, 8, 0, sample)
    Q = inputs.query(SEED, cols, 1)
    oracle_passes(D, Q, args.warmup, cores)
    t = oracle_passes(D, Q, args.steps, cores)
    dt = sum(t)
    value = D.size * args.steps / dt / 1e9
    desc = f"each step = first {sample} of 131072 rows x 131072 cols, batch 1 ({D.size / 2**20:.0f} MiB of DB)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
        "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u8*u32->u128 accumulate, % 2^32", "data": "synthetic",
        "config": {"workload": "configs[2] (16 GiB u8 DB, batch 1), bounded row sample: " + desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                         "median_pass_GBps": D.size / sorted(t)[len(t) // 2] / 1e9},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--headline-only", action="store_true", help="time only configs[2] (headline) and configs[3] (batched)")
    ap.add_argument("--paper", action="store_true", help="also time the paper's Table-2 shapes and NEXT-2 shapes (64 GiB DB)")
    ap.add_argument("--modgemm", action="store_true",
                    help="also time the ring-packing stage at the paper's 64 GiB shape: lift + NTT (G, H) and H*C+(0|G)")
    ap.add_argument("--pipeline", action="store_true",
                    help="also time the built chain scan -> NTT -> H*C+(0|G) at the paper's 64 GiB hybrid shape")
    ap.add_argument("--only", default=None, choices=sorted(list(CONFIGS) + list(PAPER_CONFIGS)),
                    help="time this one config alone and print its measurements (N = 1; not the bench line)")
    ap.add_argument("--cpu-sample-rows", type=int, default=8192)
    ap.add_argument("--ref-sample-rows", type=int, default=8192)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
