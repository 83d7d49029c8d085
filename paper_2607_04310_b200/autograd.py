"""torch.autograd bridge: the paper's implementation is a PyTorch module whose state gradients
come from autograd; this gives the same calling convention on top of the
CUDA path.  forward = psdf_eval (value and analytic witness gradient in ONE kernel launch),
backward = the chain rule with the stored gradient: no second pass over the obstacles.
Binding glue only: no PSDF arithmetic lives here.
"""
from __future__ import annotations

import torch

from . import psdf as _psdf


class _PsdfFunction(torch.autograd.Function):
    @staticmethod
    def forward(ctx, poses, scene):
        value, grad, _ = scene.eval(poses.detach().contiguous(), grad=True)
        ctx.save_for_backward(grad)
        return value

    @staticmethod
    def backward(ctx, grad_out):
        (grad,) = ctx.saved_tensors
        return grad_out.unsqueeze(1) * grad, None


class PSDF(torch.nn.Module):
    """phi(x, E) of eq.(6) for poses [N,3] = (x, y, theta) on the scene's device;
    differentiable w.r.t. the poses (at ties / kinks the gradient of one tied branch)."""

    def __init__(self, footprint, A, B, S, max_poses: int):
        super().__init__()
        self.scene = _psdf.Scene(footprint, A, B, S, max_poses)

    def update(self, A, B, S):
        """Perception update, same (M, E)."""
        self.scene.update(A, B, S)

    def forward(self, poses: torch.Tensor) -> torch.Tensor:
        assert poses.is_cuda and poses.dtype == torch.float32 and poses.shape[-1] == 3
        return _PsdfFunction.apply(poses, self.scene)
