"""B200-native tensor transposition-and-update  B_Pi(i) <- alpha*A_i + beta*B_Pi(i)
(arXiv 1607.01249, Eq. 1).  The product is the C-ABI library ``libttc.so`` built from
``csrc/``; :mod:`paper_1607_01249_b200.ttc` is its thin ctypes binding (argument
marshalling only).  Nothing is loaded at package import; the binding fails loudly on
first use if the CUDA library has not been built."""
__version__ = "0.5.0"   # == the number in ttc_version() (tests/test_host_abi.py)
