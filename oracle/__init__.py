"""CPU oracle for the RT-TDDFT time step of arXiv 2410.09189 (TEST INFRASTRUCTURE ONLY).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this package.  The product path (``paper_2410_09189_b200``) never does.
"""
