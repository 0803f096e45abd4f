"""CPU oracle (TEST INFRASTRUCTURE, not the product).

Thin ctypes binding over ``oracle/lbmref.c`` — a plain single-threaded fp64 C restatement of the
paper's time step (§II, App. A).  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package; it imports
nothing from ``paper_2605_30878_b200`` and shares no code with the CUDA path.
"""
from .ref import RefLBM, RefParams, build_oracle, lib  # noqa: F401
