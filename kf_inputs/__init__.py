"""Seeded synthetic inputs shared by the oracle's tests and the CUDA path's tests/bench.
Holds none of the method's arithmetic (see gen.py / workloads.py / gen_cuda.cu)."""
from . import gen, workloads  # noqa: F401
