"""Helpers for the GPU parity tests: run the C-ABI on torch device tensors, fetch results."""
from __future__ import annotations

import numpy as np

from paper_2606_11536_b200 import build, vipir


def ensure_built():
    build.build()


def run_dbmul(D_host: np.ndarray, Q_host: np.ndarray, moduli=None, regime=vipir.REGIME_AUTO, return_info=False,
              modswitch_bits=0, db_signed=False, db_layout=vipir.DB_ROW_MAJOR, tuning=None):
    """D_host rows x cols (u8/u16), Q_host [T][B][cols] u32 -> answer [T][B][rows] u32 via libvipir.
    db_layout = DB_LIMB_PLANES: the u16 DB is first re-laid out on the device by vipir_db_split_u16.
    tuning: explicit planner overrides (vipir_tuning fields)."""
    import torch
    ensure_built()
    D_host = np.ascontiguousarray(D_host)
    rows, cols = D_host.shape
    db_bits = 8 * D_host.dtype.itemsize
    Q_host = np.ascontiguousarray(Q_host, dtype=np.uint32)
    T, batch, _ = Q_host.shape
    d_db = torch.from_numpy(D_host.view(np.uint8).reshape(rows, -1)).cuda()
    d_q = torch.from_numpy(Q_host.view(np.int32)).cuda()
    d_a = torch.full((T, batch, rows), -1, dtype=torch.int32, device="cuda")  # poison
    if db_layout == vipir.DB_LIMB_PLANES:
        d_planes = torch.full_like(d_db, 0x5A)
        vipir.db_split_u16(d_db, d_planes, rows, cols)
        d_db = d_planes
    with vipir.Plan(rows, cols, batch, db_bits, moduli, regime, modswitch_bits, db_signed, db_layout, tuning) as plan:
        plan(d_db, d_q, d_a)
        torch.cuda.synchronize()
        info = plan.info
    out = d_a.cpu().numpy().view(np.uint32)
    return (out, info) if return_info else out


def run_dbmul_device(d_db, d_q, rows, cols, batch, db_bits, moduli=None, regime=vipir.REGIME_AUTO):
    """Same, inputs already on the device; returns (answer torch.int32 [T][B][rows], info)."""
    import torch
    ensure_built()
    T = 1 if not moduli else len(moduli)
    d_a = torch.full((T, batch, rows), -1, dtype=torch.int32, device="cuda")
    with vipir.Plan(rows, cols, batch, db_bits, moduli, regime) as plan:
        plan(d_db, d_q, d_a)
        torch.cuda.synchronize()
        info = plan.info
    return d_a, info
