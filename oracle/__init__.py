"""oracle -- TEST INFRASTRUCTURE, NOT PRODUCT.

CPU oracle of the TPC clusterizer.
Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` /
``--impl reference`` legs of ``bench.py`` may import this package.  It shares
no code with ``paper_2511_17018_b200`` and never imports it.

* ``t1``  -- ctypes front end of ``tpcclus_oracle.c`` (plain C, single thread).
* ``t0_bruteforce`` -- pure-Python definitional formulation for tiny maps.
"""
from . import t1  # noqa: F401
