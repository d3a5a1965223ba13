"""Parity comparison rules (readings S14, S17) shared by the GPU tests."""
import numpy as np

MIP_REL = 1e-6       # north_star: MIP within 1e-6 relative error (scale-relative, S17)
EA_ABS = 1e-4        # north_star: emission-absorption RGBA within 1e-4 absolute per channel
ERT_BOUND = (1 - 0.99) + 1e-4
# S14: ERT-fragile pixels (some T_k within 1e-5 of the threshold) must be rarer than 0.5 % of hit pixels on the
# configs' TF_HAZE workloads, where few rays terminate.  Under TF_OPAQUE EVERY ray terminates, and the chance that
# one of its T_k lands within +-1e-5 of 0.01 is about 2e-5 / (0.01 alpha) ~ 0.5-1 % per ray (the oracle alone gives
# 0.1-0.6 % on the small test views), so those tests allow 2 %.  The GPU images are bit-identical to the oracle's
# anyway; the bound only guards the workload.
FRAGILE_FRAC_OPAQUE = 0.02


def check_mip(gpu: np.ndarray, ref: np.ndarray, data_scale: float):
    """Miss masks identical; |g-o| <= 1e-6 * max(|o|, R).  Returns stats."""
    assert gpu.shape == ref.shape
    miss_g, miss_o = np.isneginf(gpu), np.isneginf(ref)
    assert np.array_equal(miss_g, miss_o), f"miss masks differ on {(miss_g != miss_o).sum()} pixels"
    hit = ~miss_o
    err = np.abs(gpu[hit].astype(np.float64) - ref[hit].astype(np.float64))
    tol = MIP_REL * np.maximum(np.abs(ref[hit]).astype(np.float64), data_scale)
    bad = int((err > tol).sum())
    assert bad == 0, f"MIP: {bad} pixels beyond 1e-6 scale-relative, max err {err.max():.3e}"
    return {"pixels": int(hit.sum()), "bit_exact": float((gpu[hit] == ref[hit]).mean()) if hit.any() else 1.0,
            "max_abs": float(err.max()) if hit.any() else 0.0}


def check_ea(gpu: np.ndarray, ref: np.ndarray, fragile: np.ndarray | None = None, hit: np.ndarray | None = None,
             max_fragile_frac: float = 0.005):
    """max_c |g-o| <= 1e-4 on every non-fragile pixel; fragile pixels within the ERT bound and rare (S14)."""
    assert gpu.shape == ref.shape
    err = np.abs(gpu.astype(np.float64) - ref.astype(np.float64)).max(axis=-1)
    frag = np.zeros(err.shape, dtype=bool) if fragile is None else fragile
    bad = int((err[~frag] > EA_ABS).sum())
    assert bad == 0, f"EA: {bad} non-fragile pixels beyond 1e-4, max err {err[~frag].max():.3e}"
    if frag.any():
        assert err[frag].max() <= ERT_BOUND + 1e-4
        n_hit = int(hit.sum()) if hit is not None else err.size
        assert frag.sum() <= max_fragile_frac * max(n_hit, 1), "too many ERT-fragile pixels"
    return {"max_abs": float(err.max()), "bit_exact": float((gpu == ref).all(axis=-1).mean()),
            "fragile": int(frag.sum())}
