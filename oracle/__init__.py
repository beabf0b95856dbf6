"""CPU oracle for the coupled FDTD-LLG step -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares nothing with the CUDA
path (``paper_2103_12819_b200``) and never imports it.
"""
from .cpu_oracle import Oracle, build_oracle, constants, oracle_from_workload  # noqa: F401
