"""Helpers for the -m gpu tests: run the CUDA path (through the C ABI) on numpy inputs."""
import numpy as np

import paper_2603_20912_b200 as P


def gpu_ladder(L, t2, R0=None, sym=None, workspace_bytes=0, return_info=False, stream=None, debug=None):
    """sym=None: the plan's default (PPL_SYM_FULL from nvirt = 52 when its buffers fit, else PPL_SYM_PAIR_SA, else PPL_SYM_PAIR).
    debug: ppl_debug_opts_t fields by name (include/ppl.h)."""
    import torch

    x, v, _ = L.shape
    o = t2.shape[0]
    dev = torch.device("cuda:0")
    Ld = torch.from_numpy(L).to(dev)
    td = torch.from_numpy(t2).to(dev)
    Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device=dev) if R0 is None else torch.from_numpy(R0).to(dev)
    with P.Plan(o, v, x, workspace_bytes, debug=debug) as plan:
        if sym is not None:
            plan.set_symmetry(sym)
        info = plan.info()
        plan.apply(Ld, td, Rd, stream)
        torch.cuda.synchronize()
        R = Rd.cpu().numpy()
    return (R, info) if return_info else R


def relerr(got, want):
    m = np.abs(want).max()
    return float(np.abs(got - want).max() / (m if m > 0 else 1.0))
