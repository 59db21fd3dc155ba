"""B200-native clover-Wilson QCD+QED Dirac solver with C* boundaries (arxiv 2502.02490 hot path).

Thin Python binding (argument marshalling only) over the C-ABI CUDA library ``libqxd.so``
(include/qxd.h).  PyTorch is used for device memory and streams only.  There is no CPU
fallback: importing works without a GPU, creating a context without the compiled library or
without CUDA raises.
"""
from .binding import (  # noqa: F401
    Qxd, QxdError, SolveInfo, load_library, library_path,
    QXD_F64, QXD_F32, QXD_F16, QXD_CGNE, QXD_BICGSTAB,
    QXD_OK, QXD_EINVAL, QXD_ESTATE, QXD_EWORKSPACE, QXD_ECUDA, QXD_ENOCONV,
)
