"""CPU oracle for the 2-D BGK-UGKS step (test infrastructure, NOT the product).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this package.  It shares no code with
``paper_1810_08137_b200`` and neither imports the other.
"""
from .binding import Oracle, build, lib  # noqa: F401
