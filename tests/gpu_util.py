"""Helpers shared by the -m gpu tests: run the CUDA path through the C-ABI binding."""
import numpy as np
import torch

import paper_2204_08834_b200 as fl


def to_dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def plan_for(W):
    return fl.Plan(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2, bc_x=getattr(W, "bc_x", 0), bc_y=getattr(W, "bc_y", 0))


def gpu_step(W, plan=None):
    """returns numpy (u, v, w, p) after one flutas_projection_step on device copies of W's fields"""
    own = plan is None
    plan = plan or plan_for(W)
    d = [to_dev(a) for a in W.fields()]
    plan.projection_step(*d, W.dt)
    torch.cuda.synchronize()
    out = tuple(d[i].cpu().numpy() for i in (0, 1, 2, 4))
    assert np.array_equal(d[3].cpu().numpy(), W.phi) and np.array_equal(d[5].cpu().numpy(), W.p_old)
    if own:
        plan.destroy()
    return out


def rel_l2(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / nb if nb > 0 else np.linalg.norm(a - b)
