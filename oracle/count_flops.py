"""Writes oracle/flop_model.json: the oracle's own operation count (add/sub/mul/min/max = 1,
div = 1, sqrt = 1; SURVEY.md §8(d) convention) per interior cell, for one RK3 step and for the
pieces of one RHS, as an exact cubic in 1/n for an n^3 periodic box (Taylor-Green input).

The counts come from the oracle run on its counting scalar type (ora_count_flops_*); they are
polynomial in 1/n because the work is (n+6)^3 cons->prim conversions, 3 n^2 (n+1) faces and n^3
cells; plus the count of one step of config 2 (channel) at full size.  Calls only oracle/ and the input generators.  Usage: python oracle/count_flops.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from oracle import ora  # noqa: E402
from paper_2406_19494_b200 import cases  # noqa: E402


def main():
    sizes = [8, 16, 32, 64]
    rows = {"step": [], "prim": [], "grad": [], "rhs": []}
    for n in sizes:
        c = cases.tgv(n)
        o = ora.Oracle(c)
        U = o.fill_halo(o.state())
        rows["step"].append(o.count_flops_step(o.state(), 1e-3) / c.cells)
        for key, what in (("prim", 1), ("grad", 2), ("rhs", 3)):
            rows[key].append(o.count_flops_part(U, what) / c.cells)
        print(n, {k: v[-1][3] for k, v in rows.items()}, flush=True)
    x = 1.0 / np.array(sizes, dtype=np.float64)
    V = np.vander(x, 4, increasing=True)
    model = {"convention": "add/sub/mul/min/max=1, div=1, sqrt=1; abs/sign/select=0",
             "basis": "c0 + c1/n + c2/n^2 + c3/n^3 per interior cell of an n^3 periodic box",
             "columns": ["basic", "div", "sqrt", "total"], "fit_sizes": sizes}
    for k, v in rows.items():
        model[k] = np.linalg.solve(V, np.array(v)).T.tolist()     # [column][coefficient]
    # config 2 (channel 192x128x128: walls, Sutherland viscosity, body force): counted at full size
    c = cases.channel()
    o = ora.Oracle(c)
    model["channel_step"] = (o.count_flops_step(o.state(), 1e-4) / c.cells).tolist()
    model["channel_dims"] = list(c.n)
    print("channel flops per cell-step:", model["channel_step"][3], flush=True)
    # the same step with the sixth-order dissipative flux (jf_set_visc_order(6))
    c.visc_order = 6
    o = ora.Oracle(c)
    model["channel_step_order6"] = (o.count_flops_step(o.state(), 1e-4) / c.cells).tolist()
    print("channel flops per cell-step, sixth-order dissipative flux:", model["channel_step_order6"][3], flush=True)
    with open(os.path.join(ROOT, "oracle", "flop_model.json"), "w") as f:
        json.dump(model, f, indent=1)
    print("asymptotic flops per cell-step:", model["step"][3][0])


if __name__ == "__main__":
    main()
