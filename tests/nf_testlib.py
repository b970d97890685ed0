"""Helpers shared by the GPU parity tests: run the CUDA path through the C-ABI binding, run the
oracle on the same float32 bits, and evaluate BASELINE.json's acceptance metric."""
import numpy as np
import torch

TOL_P999 = 1e-5   # |a_gpu - a_ref| / |a_ref| for 99.9 % of particles   (BASELINE.json north_star)
TOL_MAX = 1e-3    # ... and at the maximum


def u32(t: torch.Tensor) -> np.ndarray:
    return t.cpu().numpy().view(np.uint32)


def gpu_run(pos_cpu: torch.Tensor, cpd, L, eps, R=2, options=None, want_binning=False):
    import paper_2110_11398_b200 as nf
    pos = pos_cpu.cuda()
    with nf.Plan(cpd, L, eps, R) as plan:
        for k, v in (options or {}).items():
            plan.set_option(k, v)
        plan.bin(pos)
        acc = plan.accel()
        torch.cuda.synchronize()
        out = {"acc": acc.cpu().numpy().astype(np.float64), "stats": plan.stats()}
        if want_binning:
            out["binning"] = {k: u32(v) for k, v in plan.binning().items()}
    return out


def rel_errors(a_gpu: np.ndarray, a_ref: np.ndarray) -> np.ndarray:
    """Euclidean norm of the difference over the norm of the reference (reading C14).  Rows whose
    reference is exactly 0 (symmetric test inputs only, reading C13) are compared absolutely by the caller."""
    num = np.linalg.norm(a_gpu - a_ref, axis=1)
    den = np.linalg.norm(a_ref, axis=1)
    return num / np.where(den > 0, den, 1.0)


def assert_parity(a_gpu, a_ref, what=""):
    err = rel_errors(a_gpu, a_ref)
    assert np.all(np.isfinite(a_gpu)), f"{what}: non-finite GPU accelerations"
    p999 = np.quantile(err, 0.999) if len(err) else 0.0
    mx = err.max() if len(err) else 0.0
    assert p999 <= TOL_P999, f"{what}: 99.9 % quantile of rel. error {p999:.3e} > {TOL_P999}"
    assert mx <= TOL_MAX, f"{what}: max rel. error {mx:.3e} > {TOL_MAX}"
    return {"median": float(np.median(err)) if len(err) else 0.0, "p999": float(p999), "max": float(mx)}


def assert_binning_equal(b_gpu: dict, b_ref: dict):
    for k in ("cid", "count", "offset", "perm"):
        g, r = np.asarray(b_gpu[k], dtype=np.uint32), np.asarray(b_ref[k], dtype=np.uint32)
        assert g.shape == r.shape, (k, g.shape, r.shape)
        assert g.tobytes() == r.tobytes(), f"binning array {k!r} differs from the oracle"


def sample_sinks(count: np.ndarray, offset: np.ndarray, perm: np.ndarray, cpd: int, rng, n_random=2000,
                 n_heavy=20, per_heavy=200, n_void=50):
    """Sink sample for configs too large for a full oracle pass: random cells, the
    heaviest cells, the 8 corner cells and some face/edge cells (periodic wrap), the emptiest
    non-empty cells.  Returns sorted unique input indices."""
    C = cpd ** 3
    cells = set(rng.integers(0, C, n_random).tolist())
    order = np.argsort(count)
    cells.update(order[-n_heavy:].tolist())
    nonempty = order[count[order] > 0]
    cells.update(nonempty[:n_void].tolist())
    for cx in (0, cpd - 1):
        for cy in (0, cpd - 1):
            for cz in (0, cpd - 1):
                cells.add((cx * cpd + cy) * cpd + cz)
    for _ in range(50):
        c = rng.integers(0, cpd, 3)
        c[rng.integers(0, 3)] = rng.choice([0, 1, cpd - 2, cpd - 1])
        cells.add(int((c[0] * cpd + c[1]) * cpd + c[2]))
    sinks = []
    for c in cells:
        s = perm[offset[c]:offset[c + 1]]
        if len(s) > per_heavy:
            s = rng.choice(s, per_heavy, replace=False)
        sinks.append(np.asarray(s, dtype=np.int64))
    return np.unique(np.concatenate(sinks)) if sinks else np.zeros(0, np.int64)
