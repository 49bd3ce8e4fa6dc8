"""CPU oracle for the nematohydrodynamics hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this package.  It never imports paper_2503_06610_b200 and shares no code with it.
"""
from .nh_oracle import (Oracle, OracleError, molecular_field, director_rhs, elastic_stress,
                        elastic_force, viscous_stress, lc_force, frank3, num_threads)

__all__ = ["Oracle", "OracleError", "molecular_field", "director_rhs", "elastic_stress",
           "elastic_force", "viscous_stress", "lc_force", "frank3", "num_threads"]
