"""Error metrics and fixtures shared by the GPU parity tests (reading R24).

north_star: relative 1e-4 in fp32 mode; relative 2e-2 on states and 1e-2 on value estimates in
bf16 mode; resampling indices bit-exact given identical weights.  "Relative" is a per-tensor norm
ratio (element-wise relative error is meaningless for components that pass through zero).
"""
import numpy as np

TOL_FP32 = 1e-4
TOL_BF16_STATE = 2e-2
TOL_BF16_VALUE = 1e-2


def rel_l2(x, ref):
    x = np.asarray(x, np.float64)
    ref = np.asarray(ref, np.float64)
    den = np.linalg.norm(ref.ravel())
    return float(np.linalg.norm((x - ref).ravel()) / (den if den > 0 else 1.0))


def rel_inf(x, ref):
    x = np.asarray(x, np.float64)
    ref = np.asarray(ref, np.float64)
    den = np.max(np.abs(ref))
    return float(np.max(np.abs(x - ref)) / (den if den > 0 else 1.0))


def value_err(v, ref):
    """max_q |V - V_ref| / max(|V_ref|, mean_q |V_ref|)."""
    v = np.asarray(v, np.float64)
    ref = np.asarray(ref, np.float64)
    den = np.maximum(np.abs(ref), np.mean(np.abs(ref)))
    den = np.where(den > 0, den, 1.0)
    return float(np.max(np.abs(v - ref) / den))


def elem_err(x, ref):
    """max_i |x_i - ref_i| / max(|ref_i|, rms(ref)): element-wise, so that a wrong SMALL component cannot
    hide under a large one (the norm ratios above can); the rms floor keeps zero crossings meaningful."""
    x = np.asarray(x, np.float64)
    ref = np.asarray(ref, np.float64)
    rms = float(np.sqrt(np.mean(ref ** 2)))
    den = np.maximum(np.abs(ref), rms if rms > 0 else 1.0)
    return float(np.max(np.abs(x - ref) / den))


ELEM_FACTOR = 4.0  # element-wise bound = 4 x the north-star tolerance (a per-element error may exceed the norm ratio)


def assert_close(x, ref, tol, what=""):
    e2, ei, ee = rel_l2(x, ref), rel_inf(x, ref), elem_err(x, ref)
    assert e2 <= tol and ei <= tol, f"{what}: rel_l2={e2:.3e} rel_inf={ei:.3e} > {tol:.1e}"
    assert ee <= ELEM_FACTOR * tol, f"{what}: element-wise {ee:.3e} > {ELEM_FACTOR * tol:.1e}"


def t2n(t):
    return t.detach().float().cpu().numpy()
