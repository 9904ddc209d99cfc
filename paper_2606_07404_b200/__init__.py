"""B200-native routed-expert layer of the TQP method (arxiv 2606.07404): thin Python binding over libtqp.so.

Every step of the path runs in the hand-written CUDA kernels behind the C ABI (include/tqp.h); this package only
marshals arguments.  PyTorch is used for device memory and streams.  There is no CPU fallback: importing works
anywhere (so the ABI can be inspected), but creating a layer without the built library or an sm_100 GPU raises.
"""
from .binding import (TqpError, TqpLayer, TqSpace, abi_symbols, dispatch_noalloc, dispatch_noalloc_capacity, load_library, tq_levels, tq_rotation_qr,  # noqa: F401
                      workspace_bytes)
