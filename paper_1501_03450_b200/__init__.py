"""gst -- B200-native spin-orbit tracking after arXiv:1501.03450 (GPUSPINTRACK).

`paper_1501_03450_b200.gst`       thin ctypes binding over the C-ABI library (include/gst.h)
`paper_1501_03450_b200.workloads` seeded synthetic lattices and bunches (BASELINE.json configs)
"""
