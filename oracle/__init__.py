"""CPU oracle of the SdBG-construction hot path — TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package. It shares no code with ``paper_1409_7208_b200`` and never imports it.
"""
from .sdbg_oracle import Oracle, OracleResult, run_oracle, build_oracle_lib  # noqa: F401
