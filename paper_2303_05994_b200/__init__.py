"""bsl6d-b200: the split 1-D advection sweep of the 6-D semi-Lagrangian Vlasov method of arXiv 2303.05994,
as hand-written sm_100a CUDA kernels behind a C ABI (include/bsl6d.h -> libbsl6d.so).

    from paper_2303_05994_b200 import create
    ctx = create(n, lo, dx, degree)         # bsl6d_create
    ctx.advect(f_in, f_out, dim, shift_source, dt)

Importing this package does not load the shared library; the first call does, and raises if it is missing.
"""
from .api import (Bsl6dError, Context, Grid, HostOp, LIB_PATH, Sweep, SYMBOLS, create, density_static, load_library,  # noqa: F401
                  version, OK, EINVAL, EALIAS, EUNSUPPORTED, ECUDA, ENOMEM, ESCRATCH, STATIC_SCRATCH_DOUBLES)
