"""CPU oracle for the VIPIR database scan -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_2606_11536_b200``) never does, and this package never imports the product.
"""
from .vipir_oracle import (  # noqa: F401
    build,
    dbmul,
    dbmul_limbs,
    dbmul_signed,
    dbmul_bruteforce,
    modswitch,
    lib_path,
)
from .modgemm import modgemm, modgemm_bruteforce, modgemm_lazy  # noqa: F401  (NEXT-4)
from .ntt import ntt_lift, smallest_psi, LAYOUT_G, LAYOUT_H  # noqa: F401  (lift + NTT producing G and H)
