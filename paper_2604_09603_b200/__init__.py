"""B200-native (sm_100a) super-tree verify step of ECHO (arxiv 2604.09603).

`echo`      -- ctypes binding of the C-ABI library libecho.so (csrc/, include/echo.h)
`workloads` -- seeded synthetic inputs (no method arithmetic)
`build`     -- in-tree nvcc build of libecho.so
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "echo", "build"]
