"""TEST INFRASTRUCTURE, NOT PRODUCT CODE -- FP64 CPU oracle (see oracle.py)."""
from .oracle import *  # noqa: F401,F403
