"""paper_1108_5882_b200 — B200-native hot path of the unbinned PWA likelihood (arXiv 1108.5882).

    from paper_1108_5882_b200 import binding   # ctypes front-end of libpwa.so (same names as pwa.h)
    from paper_1108_5882_b200 import inputs    # seeded synthetic input generator

`binding` raises ImportError if libpwa.so has not been built (python -m
paper_1108_5882_b200.build): there is no CPU fallback.
"""
