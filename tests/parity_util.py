"""Helpers shared by the GPU parity tests (comparison logic only; no method arithmetic)."""
from __future__ import annotations

import numpy as np


def tri_index(n):
    """(i, j) arrays of the row-major lower triangle, b = i(i+1)/2 + j (reading R2)."""
    return np.tril_indices(n)


def f32_tolerance_check(vis_gpu, vis_ref, n_inputs, rel=1e-5):
    """north_star: |delta| <= 1e-5 * sqrt(|V_ii V_jj|) per visibility, V_ii/V_jj from the ORACLE
    (float64); if V_ii V_jj == 0 the difference must be exactly 0.  Returns max(err/scale)."""
    g = np.asarray(vis_gpu, dtype=np.float64)
    r = np.asarray(vis_ref, dtype=np.float64)
    assert g.shape == r.shape, (g.shape, r.shape)
    ii, jj = tri_index(n_inputs)
    diag = ii * (ii + 1) // 2 + ii
    auto_i = r[:, diag, 0]                       # [C][nb]: V_ii for the baseline's i
    auto_j = r[:, jj * (jj + 1) // 2 + jj, 0]
    scale = np.sqrt(np.abs(auto_i * auto_j))
    err = np.hypot(g[..., 0] - r[..., 0], g[..., 1] - r[..., 1])
    zero = scale == 0
    assert np.all(err[zero] == 0), "non-zero error where V_ii V_jj == 0"
    ratio = np.where(zero, 0.0, err / np.where(zero, 1.0, scale))
    worst = float(ratio.max()) if ratio.size else 0.0
    assert worst <= rel, f"float32 parity out of tolerance: max err/scale = {worst:.3e} > {rel}"
    # autocorrelations: imaginary part exactly zero (reading R9)
    assert np.all(g[:, np.unique(diag), 1] == 0), "Im V_ii must be exactly 0"
    return worst
