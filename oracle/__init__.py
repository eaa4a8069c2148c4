"""TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front end of ``oracle/nbsdf_oracle.c`` (plain fp64 CPU definition of the
decoder hot path of arXiv 2406.17782).  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this.
Nothing here is shared with, imported by, or imports the CUDA package.
"""
from .binding import (  # noqa: F401
    QUERY_DTYPE, LIGHT_DTYPE, build, eval_queries, shade_frame, softplus, wrap,
    log_footprint, to_local, max_threads,
    pd_eval_queries, pd_shade_frame, oneblob, leaky, size01, inv_logmap, lerp_latent, encode_latent,
)
