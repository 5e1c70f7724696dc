"""CPU oracle for the Hermite force/jerk hot path -- TEST INFRASTRUCTURE, not product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It does not import, and is not imported by, paper_1702_00440_b200's CUDA path.
"""
from .oracle import (  # noqa: F401
    HermiteOracle, build, pairsum, pairsum_longdouble, predict, correct, energy, next_block, block_init,
    block_update, initial_dt, num_threads, set_num_threads, DT_MAX, DT_MIN,
)
from . import lagrange  # noqa: F401,E402
from . import structure  # noqa: F401,E402
