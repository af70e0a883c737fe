"""B200-native batched Stratego environment step (arxiv 2511.07312 hot path).

`paper_2511_07312_b200.binding` is the thin Python binding over the C-ABI library
`libstrat.so` (include/strat.h).  `paper_2511_07312_b200.workloads` holds the seeded,
synthetic workload descriptions shared by the tests, the bench and the oracle checks;
it contains none of the method's arithmetic.  Importing this package loads nothing.
"""
