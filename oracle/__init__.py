"""CPU oracle for the sequential Metropolis sweep (arXiv 1602.05716) -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_1602_05716_b200``) never does, and this package never imports the product.
"""
from .binding import Oracle, build_oracle, load_oracle, philox4x32_10, uniform_open01  # noqa: F401
