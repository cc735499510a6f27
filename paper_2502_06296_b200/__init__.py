"""B200-native Poisson + wall-normal Helmholtz hot path of arxiv/paper_2502_06296.

``binding``    thin ctypes binding of the C-ABI library (include/pz.h); argument marshalling only
``workloads``  seeded synthetic inputs of the BASELINE.json configurations (no method arithmetic)
"""
