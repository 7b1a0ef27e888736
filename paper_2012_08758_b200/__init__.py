"""B200-native hot path of arXiv 2012.08758: one 2N-RK3 step of isothermal resistive MHD.

The product is the C-ABI library (include/ac_mhd.h, csrc/) and its thin binding (binding.py).
inputs.py holds the seeded synthetic input generators only.
"""
