"""fp64 CPU oracle of the GMNN energy+force path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

See gmnn_oracle.c for the passages followed and gmnn_oracle.py for the ctypes face.
Nothing under paper_2505_22168_b200/ may import this package.
"""
