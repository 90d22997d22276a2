"""TEST INFRASTRUCTURE ONLY: the fp64 CPU oracle of the ByteScale attention hot path.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the product package
``paper_2502_21231_b200`` and the product never imports it.
"""
from .attn import (attn_bwd, attn_fwd, bf16_to_f64, build, merge, rows_from_plan,  # noqa: F401
                   threads)
from .plan import plan as oracle_plan  # noqa: F401
from .assign import assign as oracle_assign  # noqa: F401
from .balance import balance as oracle_balance  # noqa: F401
