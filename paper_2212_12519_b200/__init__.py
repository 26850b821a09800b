"""B200-native Joseph projector (after arxiv 2212.12519, "parallelproj").

``paper_2212_12519_b200.inputs``  seeded synthetic inputs (no projector arithmetic)
``paper_2212_12519_b200.binding`` thin ctypes binding over the C-ABI library (include/joseph_b200.h)
"""
