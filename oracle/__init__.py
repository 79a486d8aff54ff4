"""TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain fp64 CPU oracle of the Kratos-polrad hot path (arxiv 2512.01283), in C
(`krp_oracle.c`), with a ctypes wrapper (`pyoracle.py`).  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this package.  It imports nothing from the CUDA package.
"""
from .pyoracle import (  # noqa: F401
    build, lib, OracleModel, OracleEvents, OracleStats, Observer, OracleZTable,
)
