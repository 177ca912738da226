"""paper_1307_5700_b200 -- B200-native hot path of the Medicina BEST-2 transient pipeline.

RFI clip -> multibeam brute-force incoherent dedispersion -> n-sigma detection, as
hand-written sm_100a CUDA behind the C ABI declared in ``include/mdsm.h``.  This package is a
thin ctypes binding with the same names; PyTorch is used by callers for device memory and
streams only.  There is no CPU fallback: importing :mod:`.binding` raises if ``libmdsm.so``
has not been built (``python paper_1307_5700_b200/build.py``).
"""
from .binding import *  # noqa: F401,F403
from .binding import __all__  # noqa: F401
