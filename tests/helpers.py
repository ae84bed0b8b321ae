"""Shared test helpers (no method arithmetic beyond norms)."""
import numpy as np


def rel_fro(x, ref):
    """Relative Frobenius error per block, no floor (reading R14); returns the max over blocks."""
    x = np.asarray(x)
    ref = np.asarray(ref)
    if x.ndim == 2:
        x, ref = x[None], ref[None]
    x = x.reshape(-1, x.shape[-2], x.shape[-1])
    ref = ref.reshape(-1, ref.shape[-2], ref.shape[-1])
    if x.shape[0] == 0:
        return 0.0
    num = np.linalg.norm(x - ref, axis=(1, 2))
    den = np.linalg.norm(ref, axis=(1, 2))
    return float(np.max(num / den))
