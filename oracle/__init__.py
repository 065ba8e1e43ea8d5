"""CPU oracle of the ODB group -> align -> collate path (test infrastructure, not the product).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  See ``odb_oracle.c`` for the arithmetic and its citations.
"""
