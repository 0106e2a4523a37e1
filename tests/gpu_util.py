"""Helpers for the -m gpu tests: run a Workload through the C ABI (via the binding) and fetch numpy results."""
from __future__ import annotations

import numpy as np
import torch

from paper_1205_1222_b200 import binding


def run_gpu(wl, options=None, n_max=None, n_i_max=None, cap=None, ctx=None, want_pred=False, dtr=None, want_pot=False):
    """nb_create + nb_set_j + nb_regular_force (fused with the predictor) on cuda:0.  Returns (gpu dict of numpy
    arrays, launch info[, xp, vp])."""
    s = wl.state
    cap = wl.cap if cap is None else cap
    own = ctx is None
    if own:
        ctx = binding.Context(n_max or s.n, n_i_max or max(wl.n_i, 1), cap)
    for k, v in (options or {}).items():
        ctx.nb_set_option(k, v)
    ctx.set_state(s)
    dev = ctx.workspace.device
    i_idx = torch.from_numpy(np.ascontiguousarray(wl.i_idx, dtype=np.int32)).to(dev)
    r_s = torch.from_numpy(np.ascontiguousarray(wl.r_s, dtype=np.float64)).to(dev)
    out = ctx.alloc_outputs(wl.n_i)
    out["nbr_list"].fill_(-7)  # entries past the count must stay untouched
    if dtr is None and not want_pot:
        ctx.nb_regular_force(i_idx, r_s, s.t, out=out)
    else:  # the Listing-B2 variants: velocity criterion eq. (3) and / or potential
        dtr_t = None if dtr is None else torch.from_numpy(np.ascontiguousarray(dtr, dtype=np.float64)).to(dev)
        ctx.nb_regular_force_ex(i_idx, r_s, s.t, dtr=dtr_t, want_pot=want_pot, out=out)
    torch.cuda.synchronize()
    info = ctx.nb_last_launch_info()
    info["fixup_rows"] = ctx.nb_fixup_stats()["last"]  # rows the call recomputed in fp64 (fixup.cuh)
    gpu = {k: v.cpu().numpy() for k, v in out.items()}
    res = [gpu, info]
    if want_pred:
        xp, vp = ctx.nb_get_predicted()
        torch.cuda.synchronize()
        res += [xp.cpu().numpy(), vp.cpu().numpy()]
    if own:
        ctx.close()
    return tuple(res)
