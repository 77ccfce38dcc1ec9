"""B200-native fused deferred-collection hot path of SafeGPU (arXiv 1410.6685).

``paper_1410_6685_b200.sg``      ctypes binding of the C-ABI library (include/sg.h), same names.
``paper_1410_6685_b200.inputs``  seeded synthetic input generators (no method arithmetic).
``paper_1410_6685_b200.build``   nvcc build of csrc/ into libsafegpu.so (sm_100a).
"""
