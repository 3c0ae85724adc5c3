"""CPU oracle for the Horseshoe-Probit Gibbs sweep -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this package.  It never imports paper_1608_04329_b200 and shares no code with it.
"""
from .api import *  # noqa: F401,F403
