"""CPU ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle/sv_oracle.cpp header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  The product (paper_2607_07816_b200) never does.

  oracle.sparse.SparseOracle   ctypes binding of sv_oracle.cpp (unordered_map simulator)
  oracle.dense                 dense 2^n simulator (numpy) that pins the sparse oracle
  oracle.build.build()         compiles sv_oracle.cpp with g++ (-ffp-contract=off)
"""
