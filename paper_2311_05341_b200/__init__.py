"""B200-native brute-force incoherent dedispersion (arXiv 2311.05341 hot path).

``binding`` is the thin ctypes face of the C-ABI library ``libdd.so`` (include/dd.h);
``workloads`` holds the seeded synthetic configs.  Nothing here imports ``oracle``.
"""
