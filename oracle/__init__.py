"""CPU oracle for the Hubbard H*v + Lanczos hot path (TEST INFRASTRUCTURE ONLY).

tier 0  `hubbard_def`  — H from the operator definition, pure Python.
        `lanczos_ref`  — Algorithm 1 verbatim, numpy fp64.
tier 1  `ref` + `hubbard_ref.c` — matrix-free CPU restatement of the paper's CPU
        comparator; authority only through agreement with tier 0.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this package.  It imports nothing from
paper_1204_3425_b200/ and shares no code with it.
"""
