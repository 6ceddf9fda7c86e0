"""Helpers for the -m gpu parity tests: the CUDA path (through the C ABI binding) next to the CPU oracle."""
import numpy as np
import torch

import pyoracle as po
from paper_2605_03563_b200 import binding as pb


def dev(a, dtype=torch.float64):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda", dtype=dtype).contiguous()


def host(t):
    return t.detach().cpu().numpy()


def make_pair(w, path=None):
    """(oracle, gpu handle) for a workload dict of paper_2605_03563_b200.workloads."""
    o = po.Oracle(w["shape"], w.get("spacing"), w.get("origin"), edges=w.get("edges"), coord=w.get("coord", 0),
                  order=w.get("order", 2), bc=w["bc"])
    g = pb.Poisson(w["shape"], w.get("spacing"), w.get("origin"), edges=w.get("edges"), coord=w.get("coord", 0),
                   order=w.get("order", 2), bc=w["bc"])
    if path is not None:
        g.set_option(pb.OPT_KERNEL_PATH, path)
    return o, g


def set_faces(o, g, faces):
    """Same ghost values on both sides; faces = list of 6 numpy arrays (or None)."""
    keep = []
    for f, a in enumerate(faces):
        if a is not None:
            o.set_ghost_face(f, a)
            keep.append(dev(a))
        else:
            keep.append(None)
    g.set_ghost_faces(keep)
    torch.cuda.synchronize()


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def pointwise_scaled(g_, c_, scale):
    """max |g - c| / scale, the C8 reading of 'pointwise relative difference'."""
    return float(np.max(np.abs(g_ - c_) / scale))


def stencil_scale(c, extra=None):
    """s_i = max(|c_i|, |c| over the 6 nearest neighbours[, extra_i]) — DESIGN.md tolerance metric C8."""
    a = np.abs(c)
    s = a.copy()
    for ax in range(3):
        for sh in (1, -1):
            s = np.maximum(s, np.roll(a, sh, axis=ax))
    if extra is not None:
        s = np.maximum(s, np.abs(extra))
    return np.maximum(s, 1e-300)
