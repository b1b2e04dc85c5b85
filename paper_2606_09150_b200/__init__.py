"""paper_2606_09150_b200 — B200-native sparse causal chunk attention of Ultra Flash (arxiv/paper_2606_09150).

The product is the C-ABI library `libuf.so` (include/uf.h, include/uf_cmn.h, include/uf_static.h; CUDA sources in `csrc/`, built in-tree
by `build.py` for sm_100a).  This package is its thin ctypes binding: same call names, argument
marshalling only.  No CPU fallback exists; importing works without a GPU, every device call fails
loudly (UFError) without one.
"""
from . import binding  # noqa: F401
from .binding import *  # noqa: F401,F403
from .binding import __all__ as _binding_all
from . import cmn_binding  # noqa: F401
from .cmn_binding import *  # noqa: F401,F403
from .cmn_binding import __all__ as _cmn_all
from . import static_binding  # noqa: F401
from .static_binding import *  # noqa: F401,F403
from .static_binding import __all__ as _static_all
from .build import build  # noqa: F401

__all__ = list(_binding_all) + list(_cmn_all) + list(_static_all) + ["build", "binding", "cmn_binding", "static_binding"]
