"""B200-native macroparticle tracking (hot path of arXiv:1710.07350) behind the C ABI of include/elg.h.

    from paper_1710_07350_b200 import elg
    bl = elg.Beamline(elements, ring=False)
    b = elg.Bunch(coords_6xn, p0c_eV=1e9, charge_C=1e-9, beamline=bl)
    out = b.track(bl, n_turns=1, moments_every="turn")

Every step runs in the CUDA kernels of libelg.so; this package only marshals arguments.  PyTorch is
used for device memory and streams.  There is no CPU fallback: without the library or a CUDA device
the calls raise.
"""
from . import elg  # noqa: F401
from .build import build  # noqa: F401
