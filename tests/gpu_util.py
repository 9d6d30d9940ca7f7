"""Helpers shared by the GPU parity tests: limb packing between oracle lists and device tensors."""
import numpy as np

from oracle.limbs import from_limbs, to_limbs


def polys_to_tensor(polys, L, device="cuda"):
    """polys: nested list [...][N] of Python ints -> int32 tensor [..., L, N] on the device (uint32 bit patterns)."""
    import torch

    def rec(x):
        if isinstance(x[0], (int, np.integer)):
            return to_limbs(x, L)
        return np.stack([rec(y) for y in x])

    arr = rec(polys)
    return torch.from_numpy(np.ascontiguousarray(arr).view(np.int32)).to(device)


def limbs_np_to_tensor(arr, device="cuda"):
    import torch
    return torch.from_numpy(np.ascontiguousarray(arr).view(np.int32)).to(device)


def tensor_to_np(t):
    return t.detach().cpu().numpy().view(np.uint32)


def tensor_to_polys(t):
    """int32 tensor [..., L, N] -> nested lists of Python ints [...][N]."""
    a = tensor_to_np(t)

    def rec(x):
        if x.ndim == 2:
            return from_limbs(x)
        return [rec(y) for y in x]

    return rec(a)


def coeff_from_limbs(a_np, k):
    """a_np: uint32 [L, N]; coefficient k as a Python int."""
    return sum(int(a_np[l, k]) << (32 * l) for l in range(a_np.shape[0]))
