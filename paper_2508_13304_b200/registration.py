"""The paper's first task as a loop over the library (PAPER.md :228-235, Eq.25): 2D/3D registration of one view by
Adam ascent on the NCC between the projection of a reference volume and the measured image.

Per iteration two asynchronous library calls on torch's current stream - `dfp_forward_fused_moments` (projection and
the three gradient moments in one traversal) and `dfp_ncc_pose_grad` (NCC and dNCC/dtheta on the device) - and one
28-byte read-back (NCC + 6 gradient components); the 6-parameter Adam update runs on the host, because the C ABI takes
poses as host arrays (the per-view set-up is done in fp64 on the host).  No projector arithmetic lives here.
"""
import numpy as np
import torch

from . import binding as _b

DEG = np.pi / 180.0


def register_view(geom, view, vol, target, theta0=None, max_iters=200, lr_mm=0.4, lr_rad=0.4 * DEG,
                  ncc_stop=0.999, dloss_stop=1e-5, betas=(0.9, 0.999), eps=1e-8):
    """Maximise NCC(A(M(theta)) vol, target) over theta = (t, gamma) from `theta0` (default 0, as in the paper).
    `view`: the gantry angle [1] (or one 12-number frame with FLAG_VIEW_FRAMES); `target`: cuda [1,nv,nu].
    Stop rule of PAPER.md :235: NCC > ncc_stop, or |NCC change| < dloss_stop over 5 consecutive iterations.
    Returns dict(theta, ncc, iterations, stop, history)."""
    g = _b.Geometry.of(geom)
    dev = vol.device
    theta = np.zeros(6) if theta0 is None else np.array(theta0, dtype=np.float64)
    lr = np.array([lr_mm] * 3 + [lr_rad] * 3)
    m, v = np.zeros(6), np.zeros(6)
    proj = torch.empty((1, g.nv, g.nu), dtype=torch.float32, device=dev)
    mom = torch.empty((1, 3, 6), dtype=torch.float32, device=dev)
    out = torch.empty(8, dtype=torch.float32, device=dev)                    # [ncc, pad, grad(6)]
    ws = torch.empty(_b.workspace_bytes(g, 1, _b.OP_FORWARD_FUSED), dtype=torch.uint8, device=dev)
    ws2 = torch.empty(_b.workspace_bytes(g, 1, _b.OP_NCC), dtype=torch.uint8, device=dev)
    host = torch.empty(8, dtype=torch.float32).pin_memory()
    hist, stop, calm, prev = [], "max_iters", 0, None
    it = 0
    for it in range(1, max_iters + 1):
        _b.forward_fused_moments(g, view, theta[None].astype(np.float32), vol, target, out_proj=proj, out_moments=mom, ws=ws)
        _b.ncc_pose_grad(g, proj, target, mom, out_ncc=out[0:1], out_grad=out[2:8].view(1, 6), ws=ws2)
        host.copy_(out, non_blocking=True)
        torch.cuda.current_stream(dev).synchronize()
        ncc, grad = float(host[0]), host[2:8].double().numpy()
        hist.append(ncc)
        if ncc > ncc_stop:
            stop = f"ncc>{ncc_stop}"
            break
        calm = calm + 1 if (prev is not None and abs(ncc - prev) < dloss_stop) else 0
        if calm >= 5:
            stop = f"dloss<{dloss_stop}"
            break
        prev = ncc
        m = betas[0] * m + (1 - betas[0]) * grad
        v = betas[1] * v + (1 - betas[1]) * grad * grad
        theta = theta + lr * (m / (1 - betas[0] ** it)) / (np.sqrt(v / (1 - betas[1] ** it)) + eps)     # ascent
    return {"theta": theta, "ncc": hist[-1], "iterations": it, "stop": stop, "history": hist}


def motion_compensated_backprojection(geom, views, proj, loss_fn, n_iters=80, lr_mm=0.1, lr_rad=0.1 * DEG, theta0=None,
                                      betas=(0.9, 0.999), eps=1e-12, callback=None):
    """The paper's second task as a loop over the library (PAPER.md :237-242, Eq.26): per-view rigid motion estimated by
    Adam descent on an image-sharpness loss of the (filtered) back-projection, 80 iterations, all views' 6 parameters
    at once and no trajectory regularisation.  Per iteration: `dfp_backproject` at the current poses, the caller's
    differentiable `loss_fn(volume) -> scalar` (torch; e.g. the gradient entropy) and its autograd gradient dL/dmu on
    the same stream, `dfp_backproject_pose_grad` with that upstream, one read-back of the [V, 6] gradient, Adam on the
    host.  `proj`: cuda [V, nv, nu] (already ramp-filtered for an FDK weight).  Returns dict(theta, losses)."""
    g = _b.Geometry.of(geom)
    dev = proj.device
    V = int(proj.shape[0])
    theta = np.zeros((V, 6)) if theta0 is None else np.array(theta0, dtype=np.float64)
    lr = np.array([lr_mm] * 3 + [lr_rad] * 3)
    m, v = np.zeros_like(theta), np.zeros_like(theta)
    vol = torch.empty((g.nz, g.ny, g.nx), dtype=torch.float32, device=dev)
    grad = torch.empty((V, 6), dtype=torch.float32, device=dev)
    ws = torch.empty(max(_b.workspace_bytes(g, V, _b.OP_BACKPROJECT), _b.workspace_bytes(g, V, _b.OP_BACKPROJECT_POSE_GRAD)),
                     dtype=torch.uint8, device=dev)
    host = torch.empty((V, 6), dtype=torch.float32).pin_memory()
    losses = []
    for it in range(1, n_iters + 1):
        th32 = theta.astype(np.float32)
        _b.backproject(g, views, th32, proj, out=vol, ws=ws)
        mu = vol.detach().requires_grad_(True)
        loss = loss_fn(mu)
        (up,) = torch.autograd.grad(loss, mu)
        _b.backproject_pose_grad(g, views, th32, proj, up.to(torch.float32).contiguous(), out=grad, ws=ws)
        host.copy_(grad, non_blocking=True)
        torch.cuda.current_stream(dev).synchronize()
        gr = host.double().numpy()
        losses.append(float(loss.detach()))
        if callback is not None:
            callback(it, theta, losses[-1])
        m = betas[0] * m + (1 - betas[0]) * gr
        v = betas[1] * v + (1 - betas[1]) * gr * gr
        theta = theta - lr * (m / (1 - betas[0] ** it)) / (np.sqrt(v / (1 - betas[1] ** it)) + eps)     # descent
    return {"theta": theta, "losses": losses}
