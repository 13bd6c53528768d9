"""B200-native compressed-basis GMRES (arXiv 2009.12101): the Arnoldi-step hot path as hand-written
sm_100a kernels behind the C ABI of include/cbgmres.h.  See DESIGN.md."""
from .binding import (  # noqa: F401
    FORMATS,
    FORMAT_BYTES,
    FORMAT_CODE,
    EXPORTS,
    LIB_PATH,
    PROF_FAMILIES,
    CbgmresError,
    Solver,
    SolveResult,
    load_library,
    payload_dtype,
)
from . import model  # noqa: F401
