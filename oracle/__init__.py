"""CPU oracle for the EA Metropolis + parallel-tempering hot path.

TEST INFRASTRUCTURE ONLY.  May be imported by tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs; never by the product
package (paper_1311_5582_b200), which in turn is never imported from here.
"""
from .ea_oracle import (Oracle, binder_ratio, build_oracle, correlation_length, philox4x32_10,
                        plane_correlation, round_trip_update)  # noqa: F401
