"""CPU oracle (FP64) for the FTLM hot path.  TEST INFRASTRUCTURE ONLY: only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import
anything under `oracle/`.  The product (`paper_2605_26261_b200/`) never does."""
