"""B200-native triangle attention with pair bias (fused forward/backward): Python binding of the
C-ABI library `libtri_attn.so` (see include/tri_attn.h and DESIGN.md)."""
from .binding import (BF16, ENDING, F32, STARTING, TriAttnError, bwd_workspace_bytes,  # noqa: F401
                      fwd_workspace_bytes, launch_count, uses_tensor_cores, load, profile_begin, profile_end, step_host_arena_bytes, tri_attn_bwd,
                      tri_attn_fwd, tri_attn_step_host, rows_fwd_workspace_bytes, rows_bwd_workspace_bytes,
                      tri_attn_rows_fwd, tri_attn_rows_bwd, noalloc_scratch_bytes, tri_attn_fwd_noalloc, tri_attn_dbias_reduce_scatter, tri_attn_bias_all_gather)
from .autograd import tri_attention  # noqa: F401,E402
