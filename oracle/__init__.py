"""ORACLE -- test infrastructure, not the product.

A plain, slow, fp64 CPU implementation of the PACI stage step and schedule, written from
/root/reference/PAPER.md.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
`cpu_baseline` / `--impl reference` legs may import it; it shares no code with
`paper_2606_07881_b200/` and never imports it.

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): see DESIGN.md "Oracle pins".
Unpinned: the training trajectory over many updates (no reference curve is reproducible
without OpenWebText) -- "parity unpinned" for that property only.
"""
