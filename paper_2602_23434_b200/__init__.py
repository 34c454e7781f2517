"""B200-native (sm_100a) Lagrangian-Particle hot path of arxiv/paper_2602_23434.

C ABI: include/lp.h, implemented by csrc/*.cu in liblp_b200.so.  `binding` mirrors the ABI
one-to-one; `LP` holds the torch tensors.  There is no CPU implementation in this package.
"""
from . import binding                       # noqa: F401
from .binding import LPError, make_config   # noqa: F401
from .lp import LP, config_from_workload    # noqa: F401
