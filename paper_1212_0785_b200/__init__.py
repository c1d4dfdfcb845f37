"""paper_1212_0785_b200 — B200 (sm_100a) kernels for the SU(3) field operations of the HMC
molecular-dynamics step (arXiv:1212.0785), behind the C ABI of include/qcd.h.

`from paper_1212_0785_b200 import binding as qcd` gives the calls, named as in the header.
"""
from . import binding  # noqa: F401  (fails loudly if libqcdmd.so has not been built)
from .binding import *  # noqa: F401,F403
