"""CPU oracle for the DP energy/force/virial path — TEST INFRASTRUCTURE, not part of the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It never imports paper_2004_11658_b200 and shares no code with it.
"""
from .dpo import Oracle  # noqa: F401
