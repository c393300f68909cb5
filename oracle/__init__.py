"""ORACLE — test infrastructure only.  See oracle/oracle.py and oracle/dh_oracle.hpp."""
from .oracle import *  # noqa: F401,F403
from .oracle import build, params, num_threads, set_num_threads  # noqa: F401
