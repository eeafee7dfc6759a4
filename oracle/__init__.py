"""CPU oracle for the THC-RR-CCSD projected doubles residual and energy.

TEST INFRASTRUCTURE ONLY.  Nothing under `paper_2111_11473_b200/` imports this
package; only `tests/`, `__graft_entry__.smoke()` and the `cpu_baseline` /
`--impl reference` legs of `bench.py` may.  It shares no code with the CUDA path.

Tiers:
    bruteforce.py  T0   determinant-space <D| H exp(T2) |0>, needs no CC formula
    naive.py       T0b  literal nested loops over every summation index
    dense.py       T1   the oracle of record: dense t_ijab, explicit 4-index ERIs,
                        the closed-shell CCSD doubles residual at t1 = 0, projected
    rows.py        T2   semi-dense sampled rows for shapes where T1 does not fit
"""
