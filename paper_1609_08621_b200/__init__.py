"""pkdg-b200: B200-native gravity interaction-list evaluator (after PKDGRAV3, arXiv 1609.08621).

``paper_1609_08621_b200.binding`` is the thin ctypes layer over the C-ABI library
(``include/pkdg.h``); ``paper_1609_08621_b200.inputs`` is the seeded input generator
(harness).  Nothing here imports the oracle.
"""
__version__ = "0.1.0"
