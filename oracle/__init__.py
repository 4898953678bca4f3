"""ORACLE -- test infrastructure, not the product.

Plain-C CPU restatement of the hot path (``lwe_oracle.c``) plus this ctypes
wrapper.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the product
(``paper_2606_01211_b200``) never does, and this package never imports the product.
"""
from .oracle import *  # noqa: F401,F403
