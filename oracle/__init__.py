"""r360 oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see r360_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this package.
"""
from .binding import Oracle, OracleScene, build_oracle, load_oracle

__all__ = ["Oracle", "OracleScene", "build_oracle", "load_oracle"]
