"""Per-class drift of the constants of motion along every ray: GPU fp32, GPU fp64 and the oracle side by side.

TEST INFRASTRUCTURE (it calls the oracle): BASELINE.json config C3 asks for "per-ray E, L_z, Q and null-norm drift
reported", SURVEY reading R12 for "per class ... for GPU and oracle side by side".  tests/test_gpu_drift.py asserts on
the numbers; run as a script on a B200 it prints the table of BASELINE.md section 5:

    python tests/drift_report.py [--json out.json]

Quantities, per ray, between the initial state and the stored final state, all evaluated in fp64 with the oracle's
(pinned) `invariants` and `metric`:
    dE    |E1 - E0| / |E0|                       E = -k_t
    dLz   |L1 - L0| / max(|L0|, 0.1)             L_z = k_phi            (floor: reading R14)
    dQ    |Q1 - Q0| / max(|Q0|, 0.1)             Carter's constant
    xi+1  |xi + 1| at the final state            the paper's own monitor, eq. (4): g k k / (g_tt k^t k^t)
    null  |g k k| / sum |g_mu_nu k^mu k^nu|      the null norm against the size of its terms (xi's denominator g_tt
                                                 changes sign at the ergosurface, where captured rays end)
Classes (each ray in exactly one): critical band = within 1 % of the Bardeen curve (north_star's exclusion); pole band =
polar turning point within asin(0.05) of the axis (R14); the rest by final status: escaped, captured.
"""
import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))      # run as a script: the repository root
import torch

import closed_forms as cf  # noqa: F401  (gpu_common needs it on the path)
import oracle as o
import paper_1303_5057_b200 as g
from gpu_common import edge_band, grid_pixels, pole_band, xi_eta_of
from paper_1303_5057_b200 import workloads as wl

CLASSES = ("escaped", "captured", "pole band", "critical band")
QUANT = ("dE", "dLz", "dQ", "xi+1", "null")


def drift(a, y0, y):
    """(n, 5) array of the quantities above."""
    inv0 = np.array([o.invariants(a, v) for v in y0])
    inv1 = np.array([o.invariants(a, v) for v in y])
    d = np.abs(inv1[:, :3] - inv0[:, :3]) / np.maximum(np.abs(inv0[:, :3]), 0.1)
    xi1, null = np.zeros(len(y)), np.zeros(len(y))
    for j, v in enumerate(y):
        if not np.all(np.isfinite(v)):
            xi1[j] = null[j] = np.inf
            continue
        gm = o.metric(a, v[1], v[2])
        k = v[4:8]
        terms = gm * np.outer(k, k)
        xi1[j] = abs(terms.sum() / (gm[0, 0] * k[0] * k[0]))
        null[j] = abs(terms.sum()) / np.abs(terms).sum()
    return np.column_stack([d, xi1, null])


def classes(a, inc, al, be, y0, status):
    xi, eta = xi_eta_of(a, y0)
    crit = edge_band(a, inc, al, be)
    pole = pole_band(a, xi, eta) & ~crit
    rest = ~crit & ~pole
    return {"escaped": rest & (status == g.ESCAPED), "captured": rest & (status == g.CAPTURED), "pole band": pole,
            "critical band": crit}


def _gather(batch, idx):
    ix = torch.from_numpy(idx.astype(np.int64)).to(batch.x.device)
    y = torch.cat([batch.x[ix], batch.k[ix]], dim=1).double().cpu().numpy()
    return y, batch.status[ix].cpu().numpy().astype(np.int32)


def samples():
    """(name, a, inc, W, sampled photon indices, their pixels, how to initialise a batch, oracle trace keywords)."""
    out = []
    for c, stride, off in ((wl.C1, 1, 0), (wl.C2, 8, 4), (wl.C3, 32, 16)):
        nx, ny, W = c["nx"], c["ny"], c["half_width"]
        cols = np.arange(off, nx, stride)
        idx = (cols[None, :] + nx * cols[:, None]).ravel().astype(np.uint64)
        al, be = grid_pixels(W, nx, ny)
        init = lambda b, c=c: g.gray_init_rays(b, c["a"], wl.R_OBS, c["inc_deg"], c["half_width"], c["nx"], c["ny"])
        out.append((c["name"], c["a"], c["inc_deg"], W, nx * ny, idx, al[idx.astype(np.int64)], be[idx.astype(np.int64)], init,
                    dict(nx=nx, ny=ny)))
    c = wl.C4
    n, m = 2 ** 24, 2 ** 14
    idx = np.arange(m, dtype=np.uint64) * np.uint64(n // m) + np.uint64(5)
    al, be = np.array([o.pixel_random(c["seed"], int(p), c["half_width"]) for p in idx]).T
    init = lambda b, c=c: g.gray_init_rays_random(b, c["a"], wl.R_OBS, c["inc_deg"], c["half_width"], c["seed"])
    out.append(("C4 (2^24)", c["a"], c["inc_deg"], c["half_width"], n, idx, al, be, init, dict(nx=0, ny=0, seed=c["seed"])))
    return out


def report():
    """{config: {impl: {class: {"n": rays, quantity: [median, max]}}}} for impl in gpu_f32, gpu_f64, oracle."""
    table = {}
    for name, a, inc, W, n, idx, al, be, init, okw in samples():
        rows = {}
        for impl, prec in (("gpu_f32", g.GRAY_F32), ("gpu_f64", g.GRAY_F64), ("oracle", None)):
            ref = o.trace(a, wl.R_OBS, inc, W, idx=idx, rule=o.STEP_EQ2, init_f32=(prec == g.GRAY_F32), threads=16, **okw)
            if prec is None:
                y0, y, st = ref["y0"], ref["y"], ref["status"]
            else:
                b = g.PhotonBatch(n, prec)
                init(b)
                y0, _ = _gather(b, idx)
                assert np.mean(y0 == ref["y0"]) > 0.999 or prec == g.GRAY_F64        # the same start as the oracle's
                g.gray_integrate(b, max_steps=wl.MAX_STEPS, params=g.StepParams(rule=g.STEP_EQ2))
                y, st = _gather(b, idx)
                del b
            d = drift(a, y0, y)
            rows[impl] = {}
            for cls, m in classes(a, inc, al, be, y0, st).items():
                fin = m & np.all(np.isfinite(d), axis=1)
                rows[impl][cls] = {"n": int(m.sum()), "bad": int((m & ~fin).sum())}
                for q, col in zip(QUANT, d.T):
                    rows[impl][cls][q] = [float(np.median(col[fin])), float(col[fin].max())] if fin.any() else [None, None]
        table[name] = rows
    return table


def markdown(table):
    fmt = lambda v: "—" if v[0] is None else f"{v[0]:.1e} / {v[1]:.1e}"
    lines = ["| config | class | rays | impl | " + " | ".join(QUANT) + " |", "|---|---|---|---|" + "---|" * len(QUANT)]
    for name, rows in table.items():
        for cls in CLASSES:
            for impl in ("gpu_f32", "gpu_f64", "oracle"):
                r = rows[impl][cls]
                if r["n"]:
                    lines.append(f"| {name} | {cls} | {r['n']} | {impl} | " + " | ".join(fmt(r[q]) for q in QUANT) + " |")
    return "\n".join(lines)


if __name__ == "__main__":
    t = report()
    if "--json" in sys.argv:
        with open(sys.argv[sys.argv.index("--json") + 1], "w") as f:
            json.dump(t, f, indent=1)
    print("median / max per class; rule eq. (2), h = 1/32, cap 20000 steps, no xi monitor")
    print(markdown(t))
