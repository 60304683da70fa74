"""foldcp-trimul: B200-native (sm_100a) triangle multiplicative update (arxiv 2603.14806 hot path).

The product is the C-ABI library libfoldcp_trimul.so (include/foldcp_trimul.h); this package holds
its CUDA sources (csrc/), the build step (build.py), a ctypes binding with the same entry points
(binding.py) and the seeded synthetic-input generators (synth.py).
"""
from . import binding, synth  # noqa: F401
from .binding import (BF16, F32, INCOMING, OUTGOING, FoldcpError, contract, finalize,  # noqa: F401
                      project, trimul, trimul_backward, workspace_bytes)
