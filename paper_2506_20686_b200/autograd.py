"""torch.autograd front end of the C-ABI kernels: lets a PyTorch model call the fused operator and back-propagate through
it (the paper's kernels are used the same way from its training code).  Marshalling only: forward =
tri_attn_fwd, backward = tri_attn_bwd; nothing is computed here.  CUDA tensors only (there is no CPU path).

    O = tri_attention(Q, K, V, G, bias, mask=None, variant=STARTING)

Q, K, V, G: [B,N,H,N,d]; bias: [B,H,N,N] (same dtype); mask: [B,N,N] uint8 keep flags or None.  Gradients flow to Q, K, V,
G and bias (dBias is produced in fp32 by the kernels and cast to bias.dtype here, as autograd requires)."""
from __future__ import annotations

import torch

from . import binding


class _TriAttention(torch.autograd.Function):
    @staticmethod
    def forward(ctx, Q, K, V, G, bias, mask, variant):
        Q, K, V, G, bias = (t.contiguous() for t in (Q, K, V, G, bias))
        mask = None if mask is None else mask.contiguous()
        O, LSE = binding.tri_attn_fwd(Q, K, V, G, bias, mask, variant)
        ctx.save_for_backward(Q, K, V, G, bias, O, LSE) if mask is None else ctx.save_for_backward(Q, K, V, G, bias, O, LSE, mask)
        ctx.variant = variant
        return O

    @staticmethod
    def backward(ctx, dO):
        saved = ctx.saved_tensors
        Q, K, V, G, bias, O, LSE = saved[:7]
        mask = saved[7] if len(saved) > 7 else None
        dQ, dK, dV, dG, dBias = binding.tri_attn_bwd(dO.contiguous(), Q, K, V, G, bias, mask, O, LSE, ctx.variant)
        return dQ, dK, dV, dG, dBias.to(bias.dtype), None, None


def tri_attention(Q, K, V, G, bias, mask=None, variant=binding.STARTING):
    """O = sigmoid(G) * softmax_k(QK^T / sqrt(d) + bias + mask) V with gradients (see the module docstring)."""
    if not Q.is_cuda:
        raise binding.TriAttnError("tri_attention needs CUDA tensors (there is no CPU path)")
    return _TriAttention.apply(Q, K, V, G, bias, mask, variant)
