"""Builds an oracle context and a CUDA context from the same seeded Workload (tests only)."""
import numpy as np

import oracle as orc
import paper_2602_08982_b200 as ws
import workloads as wl


def relerr(x, ref):
    x, ref = np.asarray(x), np.asarray(ref)
    d = np.max(np.abs(ref))
    return float(np.max(np.abs(x - ref)) / (d if d > 0 else 1.0))


def make_oracle(w, n_wf=None, **over):
    n_wf = w.n_wf if n_wf is None else n_wf
    o = orc.Oracle(w.mode, w.dims, w.dx, n_wf, **wl.context_kwargs(w, over))
    return wl.configure(o, w, n_wf)


def make_gpu(w, n_wf=None, **over):
    n_wf = w.n_wf if n_wf is None else n_wf
    g = ws.Context(w.mode, w.dims, w.dx, n_wf, **wl.context_kwargs(w, over))
    return wl.configure(g, w, n_wf)


def to_gpu(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def to_np(t):
    return t.detach().cpu().numpy()
