"""Helpers for the GPU parity tests: move seeded boundary-layout numpy fields to the
device, through the C ABI binding, and back.  No arithmetic of the method here."""
import numpy as np
import torch

from paper_2001_05706_b200 import qcd

TOL = {8: 1e-12, 4: 2e-6}   # BASELINE.json north_star: per-field relative L2


def relerr(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


_ctx = None


def ctx():
    global _ctx
    if _ctx is None:
        _ctx = qcd.Context(0)
    return _ctx


def to_dev(a, precision):
    dt = {4: torch.float32, 8: torch.float64}[precision]
    return torch.from_numpy(np.ascontiguousarray(a)).to(device="cuda", dtype=dt).contiguous()


def pack(c, psi, dims, precision):
    """boundary numpy spinor -> internal device tensor (even block, odd block)."""
    return c.spinor_pack(to_dev(psi, precision), dims)


def unpack(c, internal, dims):
    return c.spinor_unpack(internal, dims).cpu().numpy().astype(np.float64)


def blocks(internal):
    """(even block, odd block) views of a full internal field."""
    h = internal.numel() // 2
    return internal[:h], internal[h:]


def parity_mask(dims):
    X, Y, Z, T = dims
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    return ((x + y + z + t) & 1)[..., None, None, None]
