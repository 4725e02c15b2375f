"""Helpers shared by the GPU parity tests: error metrics (reading R14) and the
tolerances BASELINE.json's north_star states."""
import numpy as np

# north_star: rho within 1e-12*max|rho| (fp64) / 1e-5*max|rho| (fp32); x, v within 1e-13 / 1e-6 relative
TOL_RHO = {"f64": 1e-12, "f32": 1e-5}
TOL_XV = {"f64": 1e-13, "f32": 1e-6}


def err_rho(rho_gpu, rho_ref):
    rho_ref = np.asarray(rho_ref, np.float64)
    return float(np.max(np.abs(np.asarray(rho_gpu, np.float64) - rho_ref)) / np.max(np.abs(rho_ref)))


def err_x(x_gpu, x_ref, L):
    """max |minimum-image(x_gpu - x_ref)| / L  (0 and L are the same point)."""
    d = np.asarray(x_gpu, np.float64) - np.asarray(x_ref, np.float64)
    d -= L * np.round(d / L)
    return float(np.max(np.abs(d)) / L) if d.size else 0.0


def err_v(v_gpu, v_ref, sigma_v=1.0):
    v_ref = np.asarray(v_ref, np.float64)
    if v_ref.size == 0:
        return 0.0
    return float(np.max(np.abs(np.asarray(v_gpu, np.float64) - v_ref)) / max(np.max(np.abs(v_ref)), sigma_v))


def to_dev(arrs, device="cuda"):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).to(device) for a in arrs]


def to_host(ts):
    return [t.cpu().numpy() for t in ts]
