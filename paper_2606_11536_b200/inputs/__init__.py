"""Seeded synthetic input generators (host numpy twin + device CUDA twin).

Holds none of the method's arithmetic; serves the oracle's tests and the CUDA path's
tests / bench alike.  See generator.py for the definition.
"""
from .generator import (  # noqa: F401
    STREAM_DB,
    STREAM_QUERY,
    db_rows,
    query,
    residues,
    rns_primes,
    stream_key,
    uniform_bytes,
    words,
)
