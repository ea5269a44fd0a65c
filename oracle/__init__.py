"""TEST INFRASTRUCTURE: fp64 CPU oracle for the conserve_kv hot path.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  See oracle/oracle.c.
"""
from .oracle import (  # noqa: F401
    attention,
    build,
    gather,
    merge,
    place,
    pool_addr,
    pool_elems,
    provision,
    scatter,
    staging_elems,
    staging_message,
)
