"""Helpers of the -m gpu parity tests: run the CUDA path through the C-ABI binding, the oracle beside it."""
import numpy as np
import torch

import closed_forms as cf
import oracle as o
import paper_1303_5057_b200 as g
from paper_1303_5057_b200 import workloads as wl


def gpu_state(batch):
    """(y[n, 8] float64, status[n], steps[n]) of a PhotonBatch, copied to the host."""
    torch.cuda.synchronize()
    y = torch.cat([batch.x, batch.k], dim=1).double().cpu().numpy()
    return y, batch.status.cpu().numpy().astype(np.int32), batch.steps.cpu().numpy().astype(np.int64) & 0xFFFFFFFF


def upload_state(batch, y0):
    """Put the oracle's initial states into a batch (rounded to the batch precision), status LIVE, steps 0."""
    t = torch.from_numpy(np.ascontiguousarray(y0)).to(batch.x.device).to(batch.x.dtype)
    batch.x.copy_(t[:, :4])
    batch.k.copy_(t[:, 4:])
    batch.status.zero_()
    batch.steps.zero_()


def grid_pixels(W, nx, ny):
    al = -W + (np.arange(nx) + 0.5) * 2 * W / nx
    be = -W + (np.arange(ny) + 0.5) * 2 * W / ny
    A, B = np.meshgrid(al, be)
    return A.ravel(), B.ravel()


def edge_band(a, inc, al, be, width=0.01):
    """True for pixels within `width` (relative) of the critical curve (SURVEY App. A.4 reading)."""
    rho_c = cf.bardeen_rho(a, inc, np.arctan2(be, al))
    return np.abs(np.hypot(al, be) / rho_c - 1) < width


def rel_err_final(y_gpu, y_ref):
    """Relative error of the final (r, theta, phi): |dr|/r, |dtheta|/max(theta,..), |dphi|/max(1,|phi|)."""
    d = np.abs(y_gpu[:, 1:4] - y_ref[:, 1:4])
    den = np.stack([np.abs(y_ref[:, 1]), np.maximum(np.abs(y_ref[:, 2]), 1e-2), np.maximum(np.abs(y_ref[:, 3]), 1.0)], 1)
    return (d / den).max(axis=1)


def xi_eta_of(a, y0):
    """(xi, eta) = (L_z / E, Q / E^2) of initial states, from the oracle's invariants."""
    inv = np.array([o.invariants(a, v) for v in y0])
    return inv[:, 1] / inv[:, 0], inv[:, 2] / inv[:, 0] ** 2


def exact_capture(a, xi, eta):
    return np.array([cf.captured_exact(a, x, e) for x, e in zip(xi, eta)])


POLE_SIN = 0.05


def pole_band(a, xi, eta):
    """Rays whose polar turning point lies within asin(POLE_SIN) ~ 2.9 deg of the spin axis (DESIGN.md reading
    R14): Boyer-Lindquist coordinates are singular there and an absolute rounding error in theta becomes a
    relative error delta/theta in k^phi; the paper treats this band separately."""
    return cf.sin_theta_min(a, xi, np.maximum(eta, 0.0)) < POLE_SIN
