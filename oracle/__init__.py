"""anslin oracle — TEST INFRASTRUCTURE ONLY (plain CPU restatement of the paper's codec + GEMM).

Importable only from tests/, ``__graft_entry__.smoke()`` and bench.py's cpu_baseline /
``--impl reference`` legs.  The product package never imports it.
"""
