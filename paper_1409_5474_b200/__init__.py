"""B200-native direct-summation force library (arxiv/paper_1409_5474 hot path).

`binding` mirrors include/nb.h one to one; `Context` is a small convenience around it that owns a
context handle and allocates outputs with torch.  Nothing here computes: all arithmetic is in
libnb.so's sm_100a kernels (csrc/).  Importing fails loudly if the library has not been built.
"""
from . import binding
from .binding import *  # noqa: F401,F403  (the nb_* functions and status codes)
from .context import Context
from . import sharding

__all__ = ["binding", "Context", "sharding"] + [n for n in dir(binding) if n.startswith(("nb_", "NB"))]
