"""fp64 CPU oracle of the HCMS hot path -- test infrastructure, not product.

See :mod:`oracle.hcms_oracle`.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.
"""
from .hcms_oracle import *  # noqa: F401,F403
from . import hcms_oracle  # noqa: F401
