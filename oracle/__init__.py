"""CPU oracle for the PICSAR-QED hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the CUDA package.

``oracle.lib()`` returns the ctypes handle of ``libpicsarqed_oracle.so`` (built on demand
with g++ from ``picsarqed_oracle.cpp``); the thin numpy wrappers live in ``oracle.api``.
"""
from .build import build, lib_path  # noqa: F401
from .api import *  # noqa: F401,F403
