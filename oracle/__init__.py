"""CPU oracle of the TRED hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
See oracle/tred_oracle.py for the scope, citations and pins."""
from .tred_oracle import *  # noqa: F401,F403
from . import tred_oracle
