"""CPU oracle for the Fresnel plane-to-plane hot path -- TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs
of ``bench.py`` may import this package.  It shares no code with ``paper_1806_06467_b200``.
"""
