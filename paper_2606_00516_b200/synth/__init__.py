"""Seeded synthetic inputs (host numpy + device fill) and BASELINE.json-shaped batch descriptors.

A module of its own: it holds none of the method's arithmetic and is the only code the oracle's
tests and the CUDA path's tests/bench share.
"""
from . import gen, workloads  # noqa: F401
