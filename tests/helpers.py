"""Shared helpers of the GPU parity tests (no method arithmetic)."""
import numpy as np

from oracle import oracle


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def host(t):
    return t.detach().cpu().numpy()


def orc_arch(a):
    return oracle.make_arch(a.kind, a.channels, a.fc, a.n_actions, a.in_c, a.in_h, a.in_w)


def close(got, ref, rtol, atol_rms=1.0, what=""):
    """|got - ref| <= rtol * max(|got|, |ref|) + rtol * atol_rms * RMS(ref)   (reading A15)."""
    got = np.asarray(got, np.float64); ref = np.asarray(ref, np.float64)
    assert got.shape == ref.shape, (what, got.shape, ref.shape)
    assert np.isfinite(got).all(), what
    tol = rtol * np.maximum(np.abs(got), np.abs(ref)) + rtol * atol_rms * np.sqrt(np.mean(ref ** 2) if ref.size else 0.0)
    err = np.abs(got - ref)
    bad = err > tol
    assert not bad.any(), f"{what}: {bad.sum()}/{bad.size} outside tolerance, worst err {err.max():.3e} (ref rms {np.sqrt(np.mean(ref**2)):.3e})"


def rel_l2(got, ref):
    ref = np.asarray(ref, np.float64); got = np.asarray(got, np.float64)
    return float(np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-30))




def close_bf16(got, ref, what="", rtol=2e-2):
    """CB_PREC_BF16_TC gate for network outputs (reading A15b): relative L2 error of the tensor <= 2e-2
    (north_star's number) and no element further than 2e-2 * max(|a|,|b|) + 8e-2 * RMS(ref) (outlier
    bound: ~6 sigma of the accumulated bf16 rounding noise derived in DESIGN.md section 3)."""
    got = np.asarray(got, np.float64); ref = np.asarray(ref, np.float64)
    assert got.shape == ref.shape and np.isfinite(got).all(), what
    e = rel_l2(got, ref)
    assert e <= rtol, f"{what}: relative L2 error {e:.3e} > {rtol}"
    close(got, ref, rtol, atol_rms=4.0, what=what)
