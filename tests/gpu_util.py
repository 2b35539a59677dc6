"""Helpers for the -m gpu tests: marshalling between numpy (n, k) blocks and the binding's torch (k, n) views."""
import numpy as np


def to_dev(X):
    import torch
    return torch.from_numpy(np.ascontiguousarray(np.asarray(X, dtype=np.complex128).T)).cuda()


def to_host(T):
    return np.ascontiguousarray(T.cpu().numpy().T)


def pack(A, which):
    """dense numpy (N, N) -> packed device tiles (through the library's pack kernel)."""
    import paper_2504_10096_b200 as b
    N = A.shape[0]
    return b.bse_pack_from_dense(to_dev(A), N, which)   # to_dev gives the column-major image


def relerr(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)
