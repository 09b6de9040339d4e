"""Seeded synthetic input generators (host numpy twin + device CUDA twin).

Holds none of the method's arithmetic; serves the oracle's tests and the CUDA path's
tests / bench alike.  See generator.py for the definition.
"""
from .generator import (  # noqa: F401
    STREAM_DB,
    STREAM_QUERY,
    STREAM_MG_H,
    STREAM_MG_C,
    STREAM_MG_G,
    modgemm_operand,
    db_rows,
    query,
    residues,
    rns_primes,
    stream_key,
    uniform_bytes,
    words,
)
