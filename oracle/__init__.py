"""CPU oracle for the OctaOctree query path — TEST INFRASTRUCTURE, never on the product path.

Two independent implementations of the same definition:
  * ``oracle.oo_oracle``   numpy float64, vectorised over queries, step by step (readable reference);
  * ``oracle.c``           plain C double (``oo_oracle.c``), one query at a time, OpenMP over queries
                           (the one that is timed as ``cpu_baseline``).
Only tests/, ``__graft_entry__.smoke()`` and bench.py's cpu_baseline / ``--impl reference`` legs may import this
package.  It imports nothing from ``paper_2606_08469_b200``.
"""
from . import oo_oracle  # noqa: F401
from . import c  # noqa: F401
