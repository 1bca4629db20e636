"""Error metrics of reading A17 shared by the GPU parity tests and smoke()."""
import numpy as np

TOL_FP32 = 1e-4      # BASELINE.json north_star: "max relative error of 1e-4 in fp32"
TOL_TENSOR = 2e-3    # "... or 2e-3 (normalised by the Frobenius norm per channel) if tensor-core inputs are fp16"


def auto_power(vis):
    """vis [..., n_bl, 2, 2] -> per-input autocorrelation power [..., 2S] (index 2*station + pol)."""
    n_bl = vis.shape[-3]
    S = int((np.sqrt(8 * n_bl + 1) - 1) / 2)
    k = np.arange(S)
    diag = vis[..., k * (k + 1) // 2 + k, :, :]                      # [..., S, 2, 2]
    p = np.stack([diag[..., 0, 0].real, diag[..., 1, 1].real], axis=-1)  # [..., S, 2]
    return p.reshape(p.shape[:-2] + (2 * S,)), S


def err_fp32(vis_gpu, vis_ref):
    """max over elements of |dV| / sqrt(V_ii^pp V_kk^qq)  (autocorrelation-normalised, A17)."""
    p, S = auto_power(vis_ref)
    i_of = np.concatenate([np.arange(k + 1) for k in range(S)])
    k_of = np.concatenate([np.full(k + 1, k) for k in range(S)])
    worst = 0.0
    for pp in range(2):
        for qq in range(2):
            den = np.sqrt(np.abs(p[..., 2 * i_of + pp]) * np.abs(p[..., 2 * k_of + qq]))
            num = np.abs(vis_gpu[..., pp, qq] - vis_ref[..., pp, qq])
            with np.errstate(divide="ignore", invalid="ignore"):
                r = np.where(den > 0, num / den, np.where(num == 0, 0.0, np.inf))
            worst = max(worst, float(r.max()))
    return worst


def err_frobenius(vis_gpu, vis_ref):
    """max over (subband, channel) of ||dV||_F / ||V||_F over that channel's [n_bl][2][2] block."""
    d = np.abs(vis_gpu - vis_ref) ** 2
    n = np.abs(vis_ref) ** 2
    num = np.sqrt(d.sum(axis=(-1, -2, -3)))
    den = np.sqrt(n.sum(axis=(-1, -2, -3)))
    with np.errstate(divide="ignore", invalid="ignore"):
        r = np.where(den > 0, num / den, np.where(num == 0, 0.0, np.inf))
    return float(np.max(r))


def check(vis_gpu, vis_ref, mode_tensor: bool):
    """Returns (error, tolerance) in the metric of the mode."""
    if mode_tensor:
        return err_frobenius(vis_gpu, vis_ref), TOL_TENSOR
    return err_fp32(vis_gpu, vis_ref), TOL_FP32
