"""libgpmap on one B200: exhaustive HP-model genotype-phenotype map enumeration (arXiv 2008.05612).

`gpmap` is the ctypes binding of the C-ABI library (include/gpmap.h); `build` compiles it in-tree for sm_100a.
"""
from . import build  # noqa: F401
from . import gpmap  # noqa: F401
