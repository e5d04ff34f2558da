"""B200-native ViCoStream per-chunk LLM-ingestion hot path (arxiv/paper_2606_19849).

`vcs`    -- ctypes binding of the C ABI in include/vcs.h (libvcs.so, sm_100a kernels)
`stream` -- per-chunk driver: drop -> KV append -> bounded prefill; retrieval -> query prefill
`build`  -- in-tree nvcc build of libvcs.so
"""
from . import vcs  # noqa: F401
from .stream import QueryPath, VideoStream  # noqa: F401
