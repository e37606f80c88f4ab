"""paper_2501_08261_b200 -- B200-native time-domain LISA response, TDI and likelihood.

``lib``   : ctypes binding of the C-ABI CUDA library (include/lisa_td.h).
``synth`` : seeded synthetic inputs of the five BASELINE.json configs (no method arithmetic).
``build`` : builds liblisa_td.so in-tree with nvcc for sm_100a.
"""
