"""herald-b200: B200-native (sm_100a) per-block sparse-KV hot path of HERALD (arxiv/paper_2606_21633).

``paper_2606_21633_b200.herald``  thin ctypes binding over the C-ABI library (include/herald.h);
                                  importing it loads ``libherald.so`` and fails loudly if it is missing.
``paper_2606_21633_b200.synth``   seeded synthetic inputs (no method arithmetic).
``paper_2606_21633_b200.build``   nvcc build of the library for sm_100a.
"""
__all__ = ["herald", "synth", "build"]
