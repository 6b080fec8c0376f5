"""CPU oracle of the narrow-band level-set hot path — test infrastructure, not the product.

See oracle/ls_oracle.cpp for the algorithm (written from PAPER.md eq. 3-13) and
oracle/ls_oracle.py for the numpy/ctypes wrapper.
"""
from . import ls_oracle  # noqa: F401
