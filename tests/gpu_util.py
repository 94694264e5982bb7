"""Helpers for the -m gpu parity tests (CUDA path through the C ABI vs the CPU oracle)."""
import numpy as np


def f32(x):
    """a Python float that is exactly the fp32 value the C ABI receives"""
    return float(np.float32(x))


def make_ctx(mlp2, mlp3=None, ws_mb=2048, **kw):
    import paper_2505_08174_b200 as hh
    return hh.Context(mlp2, mlp3, workspace_bytes=ws_mb << 20, **kw)


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda()


def gpu_node_table(tr):
    order = np.lexsort((tr["hi"], tr["lo"]))
    return (np.stack([tr["lo"], tr["hi"], (tr["left"] < 0).astype(np.int64)], 1)[order], tr["bmin"][order], tr["bmax"][order])


def gpu_block_table(tr, tau, sigma):
    T = np.stack([tr["lo"][tau], tr["hi"][tau], tr["lo"][sigma], tr["hi"][sigma]], 1)
    return T[np.lexsort((T[:, 3], T[:, 2], T[:, 1], T[:, 0]))] if len(T) else T.reshape(0, 4)


def map_blocks_to_oracle(tr, tau, sigma, H):
    """index of each GPU admissible block in the oracle's P^G order (blocks identified by ranges, S-12)"""
    key = {}
    for g, (t, s) in enumerate(H.G):
        key[(int(H.lo[t]), int(H.hi[t]), int(H.lo[s]), int(H.hi[s]))] = g
    return np.array([key[(int(tr["lo"][t]), int(tr["hi"][t]), int(tr["lo"][s]), int(tr["hi"][s]))]
                     for t, s in zip(tau, sigma)], np.int64)
