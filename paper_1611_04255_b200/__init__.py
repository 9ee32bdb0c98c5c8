"""B200-native Linear Pipeline (LP) collectives of arXiv 1611.04255.

The product is the C-ABI library ``liblp_b200.so`` (include/lp_collectives.h);
this package is its thin Python binding (``binding``) plus the seeded input
generators (``inputs``).  The CUDA library is loaded on first use and the
binding raises if it is missing: there is no CPU fallback.
"""
from . import inputs  # noqa: F401  (numpy only; holds none of the method's arithmetic)
