"""B200 (sm_100a) MoE-chunk library of arxiv/paper_2606_11169: C-ABI in include/piper.h, CUDA kernels in
csrc/, and this thin ctypes binding (same names as the C-ABI).  No CPU path."""
from .binding import *  # noqa: F401,F403
from .binding import (ChunkArgs, Context, MoeDesc, PiperError, alloc_buffers, chunk_args, lib, make_desc)  # noqa: F401
