"""Planner tuning aid: time one shape of vipir_dbmul under VIPIR_TUNE_* plan-time overrides (csrc/vipir_api.cu).

    python -m paper_2606_11536_b200.tune_sweep CONFIG [SETTING ...]

CONFIG   a bench.py config name (C4_4GiB_B256, P_16GiB_B32, ...) or R<rows>x<cols>xB<batch> (u8 DB, q = 2^32)
SETTING  'K=V,K=V' -> VIPIR_TUNE_K=V for that plan ('-' = the planner's own choice); settings are timed round-robin,
         TUNE_SWEEP_REPS times (default 2), each after TUNE_SWEEP_SETTLE seconds (default 0.5) of back-to-back launches so
         that power-capped shapes are compared in steady state.  TUNE_SWEEP_PLANES=1: u16 DB held as limb planes.
Prints one JSON line per measurement: the scan kernel alone (vipir_dbmul_scan), or the whole call where that is one
launch.  The planner's constants and profiles/r01_tuning.md come from runs of this script; it holds no arithmetic of
the method.
"""
from __future__ import annotations

import json
import os
import sys
import time
from pathlib import Path


def main(argv):
    sys.path.insert(0, str(Path(__file__).resolve().parents[1]))
    import torch

    import bench
    from paper_2606_11536_b200 import inputs, vipir
    from paper_2606_11536_b200.inputs import device

    if len(argv) < 2:
        print(__doc__)
        return 2
    name, settings = argv[1], (argv[2:] or ["-"])
    if name.startswith("R"):
        r, c, b = name[1:].split("x")
        rows, cols, batch, db_bits, prime = int(r), int(c), int(b[1:]), 8, False
    else:
        rows, cols, batch, db_bits, prime = (bench.CONFIGS.get(name) or bench.PAPER_CONFIGS[name])
    moduli = inputs.rns_primes(0) if prime else None
    kb = cols * db_bits // 8
    d_db = device.db(0, rows, cols, db_bits)
    d_q = device.query(0, cols, batch, moduli)
    d_a = torch.empty((d_q.shape[0], batch, rows), dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream()
    layout = vipir.DB_ROW_MAJOR
    if os.environ.get("TUNE_SWEEP_PLANES"):
        planes = torch.empty_like(d_db)
        vipir.db_split_u16(d_db, planes, rows, cols)
        d_db, layout = planes, vipir.DB_LIMB_PLANES
    reps = int(os.environ.get("TUNE_SWEEP_REPS", "2"))
    settle = float(os.environ.get("TUNE_SWEEP_SETTLE", "0.5"))
    for rep in range(reps):
        for s in settings:
            keys = []
            if s != "-":
                for kv in s.split(","):
                    k, v = kv.split("=")
                    os.environ["VIPIR_TUNE_" + k] = v
                    keys.append("VIPIR_TUNE_" + k)
            try:
                with vipir.Plan(rows, cols, batch, db_bits, moduli, db_layout=layout) as plan:
                    info = plan.info
                    plan(d_db, d_q, d_a)
                    torch.cuda.synchronize()
                    one = info["launches"] == 1
                    fn = (lambda: plan(d_db, d_q, d_a)) if one else (lambda: vipir.dbmul_scan(plan.handle, d_db, d_a))
                    t_end = time.perf_counter() + settle
                    while time.perf_counter() < t_end:
                        for _ in range(10):
                            fn()
                        torch.cuda.synchronize()
                    ms = bench.time_events(fn, 30, 3, stream) / 30
                rec = {"cfg": name, "set": s, "rep": rep, "ms": round(ms, 4), "db_GBps": round(rows * kb / ms / 1e6, 1),
                       "int8_TOPS": round(2.0 * rows * kb * info["query_vectors"] * info["limb_cols"] / ms / 1e9, 1),
                       "plan": {k: info[k] for k in ("regime_name", "tile_cols", "mma_n", "m_tiles", "n_tiles", "n_chunks",
                                                     "stages", "smem_bytes", "m_sub", "grid")}}
            except vipir.VipirError as e:
                rec = {"cfg": name, "set": s, "err": str(e)[:200]}
            for k in keys:
                del os.environ[k]
            print(json.dumps(rec), flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv))
