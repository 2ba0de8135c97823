#!/usr/bin/env python
"""How the cost of 1,000 NLL+gradient evaluations (C1: 10^6 events, mass model) depends on how they are cut into
mf_nll_grad_points calls.  Consecutive calls overlap on the GPU (the kernel reads the parameter-only constants in place from a
pinned, device-mapped staging ring and waits for its predecessor only before it touches the shared scratch), so the sweep time
should not depend on the call size; MF_POINTS_COPY=1 restores the stream-ordered copy that serialises the calls.

    python paper_2505_12414_b200/examples/points_calls.py            # from the repository root, on a B200
"""
import json
import os
import sys

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import mf_datagen as dg  # noqa: E402
import paper_2505_12414_b200 as mf  # noqa: E402


def main():
    ctx = mf.Context(0)
    n, n_models = 1_000_000, 8
    models = [ctx.model_create(mf.MF_MASS_GAUSS_EXP, ctx.dataset_upload(dg.gen_mass(n, seed=1 + r), dg.MASS_LO, dg.MASS_HI))
              for r in range(n_models)]
    pts = np.ascontiguousarray(dg.gen_lambda_points(1000, 77, dg.MASS_TRUTH, 3 * dg.mass_sigma_stat(n)))
    out = torch.zeros((1000, 6), dtype=torch.float64, device="cuda")
    res = {}
    for per_call in (8, 20, 50, 100, 250, 500, 1000):
        def sweep(s):
            for p in range(0, 1000, per_call):
                models[s % n_models].nll_grad_points(pts[p:p + per_call], out[p].data_ptr())
        for s in range(5):
            sweep(s)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for s in range(20):
            sweep(s)
        e1.record()
        torch.cuda.synchronize()
        res[f"{per_call}_points_per_call"] = round(e0.elapsed_time(e1) / 20, 4)
    print(json.dumps({"ms_per_1000_evaluations": res, "copy_path": bool(os.environ.get("MF_POINTS_COPY"))}))


if __name__ == "__main__":
    main()
