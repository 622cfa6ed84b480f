"""B200-native hot path of the ABP/TAIGA synthetic diagnostic (arxiv/paper_2506_15812).

Sub-modules
-----------
workloads : seeded synthetic input generators (COMPASS-shaped Solov'ev fields, CDF tables,
            detector descriptors).  Holds none of the method's arithmetic; it is the only
            module shared by the CUDA path and the CPU oracle (``oracle/``).
taiga     : thin ctypes binding of the C ABI in ``include/taiga.h`` (``libtaiga.so``, hand
            written sm_100a CUDA).  Importing it fails loudly when the library is missing;
            there is no CPU fallback.

Nothing is imported eagerly so that ``workloads`` can be used without the CUDA library.
"""

__all__ = ["workloads", "sharding", "taiga"]
