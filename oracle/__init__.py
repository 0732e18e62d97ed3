"""ORACLE package -- TEST INFRASTRUCTURE ONLY (see oracle/ref.py header).

`oracle.ref`   : definitional Python/fp64 form, for tiny inputs.
`oracle.cbind` : ctypes binding of oracle/tacg_oracle.c (plain C, fp64), for full
                 sizes and for bench.py's timed cpu_baseline.
Nothing here imports paper_2606_01007_b200.
"""
