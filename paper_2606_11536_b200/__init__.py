"""vipir-dbmul for B200: the VIPIR PIR server's database scan answer = D*Q mod q
(arxiv/paper_2606_11536) as hand-written sm_100a CUDA behind a
C-ABI library.  `vipir` is the thin ctypes binding; `inputs` the seeded input generators.

Importing this package loads nothing native; the first call into `vipir` loads
csrc/libvipir.so and raises if it is missing (there is no CPU fallback).
"""
__all__ = ["vipir", "inputs"]
