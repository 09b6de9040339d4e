"""Build the native libraries in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_11536_b200.build [--force]

csrc/libvipir.so            the product: C ABI of include/vipir.h
inputs/libvipir_inputs.so   device twin of the seeded input generator (tests / bench only)
ceilings/libvipir_ceilings.so   measured ceilings for bench.py: pure int8 MMA loop, register-only butterflies
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC", "-shared"]

TARGETS = {
    PKG / "csrc" / "libvipir.so": {
        "src": [PKG / "csrc" / "vipir_api.cu"],
        "deps": sorted((PKG / "csrc").glob("*.cuh")) + [ROOT / "include" / "vipir.h"],
    },
    PKG / "inputs" / "libvipir_inputs.so": {
        "src": [PKG / "inputs" / "generator.cu"],
        "deps": [],
    },
    PKG / "ceilings" / "libvipir_ceilings.so": {
        "src": [PKG / "ceilings" / "ceilings.cu"],
        "deps": [PKG / "csrc" / "ptx.cuh", PKG / "csrc" / "gemm_i8_tcgen05.cuh", PKG / "csrc" / "ntt_lift.cuh"],
    },
}


def _stale(out: Path, inputs) -> bool:
    if not out.exists():
        return True
    t = out.stat().st_mtime
    return any(Path(f).stat().st_mtime > t for f in inputs)


def build(force: bool = False, verbose: bool = False) -> list[Path]:
    built = []
    for out, spec in TARGETS.items():
        inputs = list(spec["src"]) + list(spec["deps"])
        if force or _stale(out, inputs):
            tmp = out.with_name(out.name + f".tmp{os.getpid()}")
            cmd = [NVCC, *ARCH, *COMMON, "-o", str(tmp), *map(str, spec["src"])]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
                print(" ".join(cmd), flush=True)
            subprocess.run(cmd, check=True)
            os.replace(tmp, out)
            built.append(out)
    return built


if __name__ == "__main__":
    b = build(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print("built:", ", ".join(str(p.relative_to(ROOT)) for p in b) if b else "nothing (up to date)")
