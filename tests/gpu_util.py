"""Helpers of the -m gpu parity tests (CUDA path through the C ABI vs the CPU oracle)."""
import numpy as np
import pytest


def rel_l2(a, b):
    a = np.asarray(a).ravel()
    b = np.asarray(b).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def parity_mask(dims):
    """[T,Lz,Ly,Lx] int array of (x+y+z+t)&1."""
    lx, ly, lz, lt = dims
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    return (x + y + z + t) & 1


def tm():
    """Import the binding and require a CUDA device (no fallback: skip is NOT silent success --
    the gpu marker is only selected on a GPU box, where a missing device is an error)."""
    import torch
    import paper_1401_6750_b200 as tmod
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device; the CUDA path has no CPU fallback")
    return tmod


def to_np(t):
    return t.detach().cpu().numpy()
