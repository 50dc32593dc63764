"""B200-native ILE extrinsic-marginalised factored likelihood (arXiv 2210.07912, App. D / Eq. (1),(3)).

The product is the C-ABI library ``librift_ile.so`` (see ``include/rift_ile.h``); ``binding`` is the thin
Python layer of the same names, ``synth`` the seeded synthetic-input generators shared with the tests, ``ac_loop`` the round loop of the adaptive-cartesian
integrator over the sampler entry points of ``include/rift_ac.h``.
"""
from . import synth  # noqa: F401
from . import ac_loop  # noqa: F401
from . import gmm_loop  # noqa: F401
from .binding import *  # noqa: F401,F403
from .binding import lib, RiftError, LIB_PATH, EXPORTS  # noqa: F401
