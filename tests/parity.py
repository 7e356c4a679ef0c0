"""Helpers shared by the GPU parity tests: the G17 error norm and tensor plumbing.
No arithmetic of the method lives here."""
import numpy as np
import torch

FORCE_TOL = 1e-12   # BASELINE.json north_star: forces within 1e-12 (norm-relative, G17)


def dev(x, dtype=torch.float64):
    return torch.as_tensor(np.ascontiguousarray(x), dtype=dtype).cuda().contiguous()


def host(x):
    return x.detach().cpu().numpy()


def g17_err(x_gpu, x_ref):
    """max over particles and components of |x_gpu - x_ref| / ||x_ref||_2 (per particle)."""
    x_gpu = np.asarray(x_gpu); x_ref = np.asarray(x_ref)
    nrm = np.linalg.norm(x_ref, axis=1, keepdims=True)
    assert np.all(nrm > 0), "zero reference norm: use the absolute bound instead"
    return float((np.abs(x_gpu - x_ref) / nrm).max())


def gpu_force(nb, pos, vel, accp, mass, eps, idx=None, split=0, jlanes=0):
    """One evaluation through the C-ABI: init, set a_pred, nb_force -> numpy (acc, jerk, snap)."""
    ctx = nb.nb_init(dev(pos), dev(vel), dev(mass), eps, 0.45, torch.cuda.current_stream())
    try:
        if accp is not None:
            nb.nb_set_pred_acc(ctx, dev(accp))
        nb.nb_set_tuning(ctx, split, jlanes)
        n = mass.shape[0] if idx is None else len(idx)
        out = [torch.full((n, 3), float("nan"), dtype=torch.float64, device="cuda") for _ in range(3)]
        nb.nb_force(ctx, None if idx is None else dev(idx, torch.int32), n, *out)
        torch.cuda.synchronize()
        launch = nb.nb_get_launch(ctx)
        return [host(o) for o in out], launch
    finally:
        nb.nb_free(ctx)
