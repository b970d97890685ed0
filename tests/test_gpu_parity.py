"""GPU parity tests proper (-m gpu): the CUDA path, called through the C-ABI binding, against the
float64 oracle on the same seeded float32 inputs.  Binning and permutation bit-exact; accelerations
within BASELINE.json's tolerance (99.9 % of particles <= 1e-5, max <= 1e-3)."""
import os

import numpy as np
import pytest
import torch

import nf_inputs
from nf_testlib import (assert_binning_equal, assert_parity, gpu_run, rel_errors, sample_sinks, u32)

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def full_check(oracle_mod, pos_cpu, cpd, L, eps, R=2, options=None, what=""):
    out = gpu_run(pos_cpu, cpd, L, eps, R, options, want_binning=True)
    pos = pos_cpu.numpy()
    b = oracle_mod.bin_particles(pos, cpd, L)
    assert_binning_equal(out["binning"], b)
    ref = oracle_mod.accel(pos, cpd, L, eps, R, binning=b)
    st = assert_parity(out["acc"], ref, what)
    assert out["stats"]["interactions"] == oracle_mod.interactions(b["count"], cpd, R)
    return st, out


# ---------------------------------------------------------------- the five configs, small and full
def test_config1_full(oracle_mod):
    cfg = nf_inputs.config(1)
    st, out = full_check(oracle_mod, nf_inputs.generate(cfg), cfg.cpd, cfg.L, cfg.eps, cfg.R, what=cfg.name)
    print(cfg.name, st, out["stats"])


def test_config1_shuffled(oracle_mod):
    cfg = nf_inputs.config(1)
    pos = nf_inputs.generate(cfg)
    perm = torch.randperm(pos.shape[0], generator=torch.Generator().manual_seed(7))
    full_check(oracle_mod, pos[perm].contiguous(), cfg.cpd, cfg.L, cfg.eps, cfg.R, what="config1 shuffled")


@pytest.mark.parametrize("idx,n_side,cpd", [(2, 48, 12), (3, 40, 10), (4, 40, 10), (5, 40, 10)])
def test_scaled_configs_full(oracle_mod, idx, n_side, cpd):
    """Same recipes at sizes the oracle finishes in seconds; several tiles, ragged tails, heavy cells."""
    cfg = nf_inputs.scaled(idx, n_side, cpd)
    st, out = full_check(oracle_mod, nf_inputs.generate(cfg), cfg.cpd, cfg.L, cfg.eps, cfg.R, what=cfg.name)
    print(cfg.name, st)


@pytest.mark.parametrize("variant,fastpath", [(1, 1), (0, 0), (1, 0)])
def test_kernel_variants(oracle_mod, variant, fastpath):
    cfg = nf_inputs.scaled(4, 32, 8)
    full_check(oracle_mod, nf_inputs.generate(cfg), cfg.cpd, cfg.L, cfg.eps, cfg.R,
               options={"variant": variant, "fastpath": fastpath}, what=f"variant{variant} fast{fastpath}")


def sampled_check(oracle_mod, cfg, device="cpu"):
    pos_dev = nf_inputs.generate(cfg, device=device)
    pos_cpu = pos_dev.cpu()
    pos = pos_cpu.numpy()
    out = gpu_run(pos_cpu, cfg.cpd, cfg.L, cfg.eps, cfg.R, want_binning=True)
    b = oracle_mod.bin_particles(pos, cfg.cpd, cfg.L)
    assert_binning_equal(out["binning"], b)
    assert out["stats"]["interactions"] == oracle_mod.interactions(b["count"], cfg.cpd, cfg.R)
    rng = np.random.default_rng(cfg.seed)
    sinks = sample_sinks(b["count"], b["offset"], b["perm"], cfg.cpd, rng)
    ref = oracle_mod.accel(pos, cfg.cpd, cfg.L, cfg.eps, cfg.R, sinks=sinks, binning=b)
    st = assert_parity(out["acc"][sinks], ref, cfg.name + " (sampled)")
    # property that holds at any size: total force vanishes (pair antisymmetry), within FP32 bounds
    a = out["acc"]
    assert np.abs(a.sum(axis=0)).max() <= 2e-6 * np.abs(a).sum()
    print(cfg.name, "sampled sinks", len(sinks), st, out["stats"])


def full_size_full_oracle(oracle_mod, cfg):
    """EVERY particle of a full-size config against the oracle (full oracle on configs 1-3).  The maximum
    of BASELINE.json's rule is set by the most-cancelled particle of the whole set, which a sink sample does not bound."""
    pos_cpu = nf_inputs.generate(cfg)
    out = gpu_run(pos_cpu, cfg.cpd, cfg.L, cfg.eps, cfg.R, want_binning=True)
    pos = pos_cpu.numpy()
    b = oracle_mod.bin_particles(pos, cfg.cpd, cfg.L)
    assert_binning_equal(out["binning"], b)
    assert out["stats"]["interactions"] == oracle_mod.interactions(b["count"], cfg.cpd, cfg.R)
    ref = oracle_mod.accel(pos, cfg.cpd, cfg.L, cfg.eps, cfg.R, binning=b)
    st = assert_parity(out["acc"], ref, cfg.name + " (all particles)")
    a = out["acc"]
    assert np.abs(a.sum(axis=0)).max() <= 2e-6 * np.abs(a).sum()
    print(cfg.name, "ALL", len(ref), "particles", st, out["stats"])


def test_config2_full_size_full_oracle(oracle_mod):
    """1.85e10 pair interactions in float64: about 35 s of the box's 16 host cores."""
    full_size_full_oracle(oracle_mod, nf_inputs.config(2))


def test_config3_full_size_sampled(oracle_mod):
    sampled_check(oracle_mod, nf_inputs.config(3))


@pytest.mark.skipif(os.environ.get("NF_FULL_ORACLE") != "1", reason="1.41e11 float64 pair interactions (~4.5 min of 16 cores): NF_FULL_ORACLE=1; the result of the round-2 run is in DESIGN.md 5")
def test_config3_full_size_full_oracle(oracle_mod):
    full_size_full_oracle(oracle_mod, nf_inputs.config(3))


def test_config4_full_size_sampled(oracle_mod):
    sampled_check(oracle_mod, nf_inputs.config(4), device="cuda")


def test_config5_full_size_sampled(oracle_mod):
    """Production-size config (1024^3 particles, ~26 GB of positions + accelerations): binning bit-exact at
    full N, accelerations on the sink sample.  Needs ~60 GB of host memory for the oracle's arrays."""
    import psutil
    need = []
    if psutil.virtual_memory().available < 70 * 2 ** 30:
        need.append("70 GB of free host memory")
    if torch.cuda.mem_get_info()[0] < 120 * 2 ** 30:
        need.append("120 GB of free device memory")
    if need:
        # on the B200 box the production-size config must run: NF_REQUIRE_CONFIG5=1 turns the skip into a failure
        # (set by the round's GPU runs); elsewhere a smaller box skips visibly
        msg = "config 5 needs " + " and ".join(need)
        if os.environ.get("NF_REQUIRE_CONFIG5") == "1":
            pytest.fail(msg + " (NF_REQUIRE_CONFIG5=1)")
        pytest.skip(msg)
    cfg = nf_inputs.config(5)
    import paper_2110_11398_b200 as nf
    pos_dev = nf_inputs.generate(cfg, device="cuda")
    torch.cuda.empty_cache()
    pos = pos_dev.cpu().numpy()
    b = oracle_mod.bin_particles(pos, cfg.cpd, cfg.L)
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as plan:
        plan.bin(pos_dev)
        acc = plan.accel()
        torch.cuda.synchronize()
        stats = plan.stats()
        for k, v in plan.binning().items():            # one array at a time: 4.3 GB each
            assert u32(v).tobytes() == b[k].tobytes(), f"binning array {k!r} differs from the oracle"
            del v
    del pos_dev
    assert stats["interactions"] == oracle_mod.interactions(b["count"], cfg.cpd, cfg.R)
    rng = np.random.default_rng(cfg.seed)
    sinks = sample_sinks(b["count"], b["offset"], b["perm"], cfg.cpd, rng)
    ref = oracle_mod.accel(pos, cfg.cpd, cfg.L, cfg.eps, cfg.R, sinks=sinks, binning=b)
    a_s = acc[torch.from_numpy(sinks).cuda()].cpu().numpy().astype(np.float64)
    st = assert_parity(a_s, ref, cfg.name + " (sampled)")
    tot = acc.double().sum(0).abs().max().item() / acc.double().abs().sum().item()
    assert tot <= 2e-6
    print(cfg.name, "sampled sinks", len(sinks), st, stats)


# ---------------------------------------------------------------- closed forms through the GPU
def test_golden_two_body_gpu():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "two_body.txt")) if l.strip() and l[0] != "#"]
    for row in rows:
        cpd, R, eps = int(row[0]), int(row[1]), float(row[2])
        v = [float(t) for t in row[3:]]
        pos = torch.tensor([v[0:3], v[3:6]], dtype=torch.float32)
        a = gpu_run(pos, cpd, 1.0, eps, R)["acc"]
        exp = np.array(v[6:9])
        scale = max(np.abs(exp).max(), 1e-30)
        assert np.abs(a[0] - exp).max() <= 2e-6 * scale, (row, a)
        assert np.abs(a[1] + exp).max() <= 2e-6 * scale, (row, a)
        if not exp.any():
            assert not a.any()                       # exact zeros stay exact


def test_symmetric_lattice_gpu():
    """Reading C13: where the exact answer is 0, |a_gpu| <= 1e-5 * sum of pair-force magnitudes."""
    cpd = 8
    g = (np.stack(np.meshgrid(*[np.arange(cpd)] * 3, indexing="ij"), -1).reshape(-1, 3) + 0.5) / cpd
    a = gpu_run(torch.tensor(g, dtype=torch.float32), cpd, 1.0, 0.002, 2)["acc"]
    pair_sum = 124 * 64.0            # loose upper bound: 124 neighbours at >= 1/8
    assert np.abs(a).max() <= 1e-5 * pair_sum


# ---------------------------------------------------------------- degenerate and edge cases
def test_empty_and_single():
    import paper_2110_11398_b200 as nf
    with nf.Plan(7, 1.0, 0.01, 2) as p:
        p.bin(torch.zeros((0, 3), device="cuda"))
        assert p.accel().shape == (0, 3)
        p.bin(torch.tensor([[0.3, 0.9, 0.1]], device="cuda"))
        a = p.accel()
        torch.cuda.synchronize()
        assert a.shape == (1, 3) and not a.cpu().numpy().any()
        assert p.stats()["interactions"] == 1


def test_one_heavy_cell(oracle_mod):
    """All particles in one cell: many sink chunks, sources tiled through several pipeline stages."""
    g = torch.Generator().manual_seed(3)
    pos = (torch.rand((3001, 3), generator=g) * (1.0 / 6) * 0.999 + 2.0 / 6).to(torch.float32)
    full_check(oracle_mod, pos, 6, 1.0, 2e-3, 2, what="one heavy cell")


@pytest.mark.parametrize("cpd,eps", [(8, 0.004), (11, 0.002), (5, 0.03)])
def test_close_pairs_across_faces(oracle_mod, cpd, eps):
    """Pairs closer than eps_s that straddle cell faces, edges and corners (periodic ones included): the
    kernel may take the Newtonian body only for cells whose nearest face is farther than eps_s.
    Separations stay above 0.3 eps_s: the sink shift of a cross-face pair is rounded to 2^-24 cell widths
    (tolerance), which is 1e-5 of a separation of 0.006 cell widths."""
    rng = np.random.default_rng(cpd)
    m = 3000
    eps_s = 2.16 * eps
    base = rng.integers(0, cpd, (m, 3)).astype(np.float64) / cpd          # a cell corner
    free = rng.random((m, 3)) < 0.4                                         # axes along which the point is interior
    p = base + np.where(free, rng.random((m, 3)) / cpd, 0.0)                # on a face / edge / corner
    d = rng.normal(size=(m, 3))
    d *= (rng.random((m, 1)) * 0.65 + 0.3) * eps_s / np.linalg.norm(d, axis=1, keepdims=True)
    pos = np.concatenate([p - 0.5 * d, p + 0.5 * d, rng.random((2000, 3))]) % 1.0
    pos = pos.astype(np.float32)
    pos[pos >= 1.0] = 0.0
    for fast in (1, 0):
        full_check(oracle_mod, torch.from_numpy(pos), cpd, 1.0, eps, 2, options={"fastpath": fast},
                   what=f"close pairs across faces cpd{cpd} fast{fast}")


def test_coincident_particles(oracle_mod):
    g = torch.Generator().manual_seed(4)
    pos = torch.rand((500, 3), generator=g)
    pos = torch.cat([pos, pos[:100]]).contiguous()           # 100 exact duplicates
    full_check(oracle_mod, pos, 5, 1.0, 0.01, 2, what="coincident")
    full_check(oracle_mod, pos, 5, 1.0, 0.0, 2, what="coincident eps=0")


@pytest.mark.parametrize("cpd,R,eps,L", [(5, 2, 0.01, 1.0), (3, 1, 0.02, 1.0), (1, 0, 0.01, 1.0), (7, 3, 0.005, 1.0),
                                         (9, 4, 0.004, 1.0), (11, 5, 0.003, 1.0), (17, 8, 0.002, 1.0), (14, 6, 0.01, 3.0),
                                         (6, 0, 0.01, 1.0), (6, 2, 0.2, 1.0), (6, 2, 0.0, 1.0),
                                         (8, 2, 0.03, 7.5), (8, 2, 25.0, 2000.0), (16, 2, 1e-5, 2.0 ** -10)])
def test_parameter_sweep(oracle_mod, cpd, R, eps, L):
    """cpd = 2R+1 (every cell in every stencil), R = 0..8 (any R >= 0 with cpd >= 2R+1), eps = 0, eps_s larger than a cell (no fast
    path), non-unit and non-dyadic box sizes."""
    g = torch.Generator().manual_seed(cpd * 10 + R)
    pos = (torch.rand((4000, 3), generator=g, dtype=torch.float64) * L).to(torch.float32)
    pos[pos >= L] = 0.0
    full_check(oracle_mod, pos.contiguous(), cpd, L, eps, R, what=f"cpd{cpd} R{R} eps{eps} L{L}")


def test_adversarial_binning(oracle_mod):
    cpd = 7
    top = np.nextafter(np.float32(1.0), np.float32(0.0))
    faces = np.array([[k / cpd, (k + 1) / cpd, 0.0] for k in range(cpd)], dtype=np.float64)
    faces[faces >= 1.0] = top
    rng = np.random.default_rng(0)
    cases = {
        "faces": faces.astype(np.float32),
        "top": np.full((5, 3), top, np.float32),
        "zero": np.zeros((4, 3), np.float32),
        "mixed": np.concatenate([faces.astype(np.float32), rng.random((5000, 3), dtype=np.float32),
                                 np.full((300, 3), 0.3, np.float32)]),
    }
    for name, pos in cases.items():
        out = gpu_run(torch.from_numpy(pos), cpd, 1.0, 0.01, 2, want_binning=True)
        assert_binning_equal(out["binning"], oracle_mod.bin_particles(pos, cpd, 1.0))


def test_layout_is_lossless():
    """sorted cell-relative coordinates / scale + corner == input positions, exactly (host-side check of
    the Sterbenz argument in DESIGN.md); pad slots hold the dummy."""
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.config(1)
    pos = nf_inputs.generate(cfg)
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as p:
        p.bin(pos.cuda())
        b = {k: u32(v) for k, v in p.binning().items()}
        lay = p.layout()
    poff = u32(lay["poff"]).astype(np.int64)
    cnt = b["count"].astype(np.int64)
    assert np.array_equal(np.diff(poff), (cnt + 3) // 4 * 4)
    cid_sorted = np.repeat(np.arange(cfg.cpd ** 3), cnt)
    slot = np.repeat(poff[:-1], cnt) + (np.arange(len(cid_sorted)) - np.repeat(b["offset"][:-1].astype(np.int64), cnt))
    w = cfg.L / cfg.cpd
    p64 = pos.numpy().astype(np.float64)[b["perm"]]
    for d, (name, cidx) in enumerate(zip("xyz", [cid_sorted // cfg.cpd ** 2, (cid_sorted // cfg.cpd) % cfg.cpd, cid_sorted % cfg.cpd])):
        corner = (cidx.astype(np.float64) * w).astype(np.float32).astype(np.float64)
        rec = lay[name].cpu().numpy().astype(np.float64)[slot] / lay["scale"] + corner
        assert np.array_equal(rec, p64[:, d])
    real = np.zeros(poff[-1], bool)
    real[slot] = True
    assert np.all(lay["x"].cpu().numpy()[~real] == 2.0 ** 55)


@pytest.mark.parametrize("cpd,n", [(9, 40_000), (16, 100_001), (26, 8192), (63, 300_000), (90, 250_000), (125, 400_000),
                                   (203, 300_000), (255, 16_385)])
def test_binning_digit_widths(oracle_mod, cpd, n):
    """The sort takes 1-3 passes of 8-11 bit digits depending on cpd^3 (10 bits x 1 ... 8 bits x 3): binning arrays
    bit-exact against the oracle and the padded SoA layout lossless, on uniform positions with a block of
    particles in one cell (ties over many tiles) and ragged last tiles."""
    import paper_2110_11398_b200 as nf
    rng = np.random.default_rng(cpd * 1000 + 7)
    pos = rng.random((n, 3), dtype=np.float32)
    pos[n // 3: n // 3 + n // 5] = np.float32(0.5) + rng.random((n // 5, 3), dtype=np.float32) * np.float32(0.2 / cpd)
    pos = pos[rng.permutation(n)]
    ref = oracle_mod.bin_particles(pos, cpd, 1.0)
    with nf.Plan(cpd, 1.0, 1e-4, 2) as p:
        p.bin(torch.from_numpy(pos).cuda())
        b = {k: u32(v) for k, v in p.binning().items()}
        lay = p.layout()
        lay = {k: (v.cpu().numpy() if hasattr(v, "cpu") else v) for k, v in lay.items()}
    assert_binning_equal(b, ref)
    poff = lay["poff"].view(np.uint32).astype(np.int64)
    cnt = ref["count"].astype(np.int64)
    assert np.array_equal(np.diff(poff), (cnt + 3) // 4 * 4)
    cid_sorted = np.repeat(np.arange(cpd ** 3), cnt)
    slot = np.repeat(poff[:-1], cnt) + (np.arange(n) - np.repeat(ref["offset"][:-1].astype(np.int64), cnt))
    p64 = pos.astype(np.float64)[ref["perm"]]
    for d, (name, cidx) in enumerate(zip("xyz", [cid_sorted // cpd ** 2, (cid_sorted // cpd) % cpd, cid_sorted % cpd])):
        corner = (cidx.astype(np.float64) * (1.0 / cpd)).astype(np.float32).astype(np.float64)
        rec = lay[name].astype(np.float64)[slot] / lay["scale"] + corner
        assert np.array_equal(rec, p64[:, d]), name
        real = np.zeros(poff[-1], bool)
        real[slot] = True
        assert np.all(lay[name][:poff[-1]][~real] == 2.0 ** 55), name


def test_rebin_workspace_stream(oracle_mod):
    """nf_bin may be called repeatedly with new n; caller-lent workspace; non-default stream."""
    import paper_2110_11398_b200 as nf
    g = torch.Generator().manual_seed(9)
    with nf.Plan(6, 1.0, 0.004, 2) as p:
        ws = torch.empty(p.workspace_bytes(6000) + 256, dtype=torch.uint8, device="cuda")
        p.set_workspace(ws)
        s = torch.cuda.Stream()
        for n in (6000, 100, 3000):
            pos = torch.rand((n, 3), generator=g)
            with torch.cuda.stream(s):
                p.bin(pos.cuda())
                a = p.accel()
            s.synchronize()
            ref = oracle_mod.accel(pos.numpy(), 6, 1.0, 0.004, 2)
            assert_parity(a.cpu().numpy().astype(np.float64), ref, f"rebin n={n}")
        with pytest.raises(nf.NFError) as e:
            p.bin(torch.rand((100000, 3), device="cuda"))
        assert e.value.code == nf.binding.NF_ERR_NOMEM


def test_host_entry_points(oracle_mod):
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.scaled(1, 24, 6)
    pos = nf_inputs.generate(cfg).pin_memory()
    out = torch.empty_like(pos).pin_memory()
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as p:
        p.bin_host(pos)
        p.accel_host(out)
    ref = oracle_mod.accel(pos.numpy(), cfg.cpd, cfg.L, cfg.eps, cfg.R)
    assert_parity(out.numpy().astype(np.float64), ref, "host entry points")


def test_errors_gpu():
    import paper_2110_11398_b200 as nf
    B = nf.binding
    with nf.Plan(5, 1.0, 0.01, 2) as p:
        with pytest.raises(nf.NFError) as e:
            p.accel(torch.empty((3, 3), device="cuda"))
        assert e.value.code == B.NF_ERR_STATE
        for bad in (1.0, -1e-9, float("nan"), float("inf")):
            pos = torch.tensor([[0.5, 0.5, 0.5], [0.1, bad, 0.2]], device="cuda")
            with pytest.raises(nf.NFError) as e:
                p.bin(pos)
            assert e.value.code == B.NF_ERR_DOMAIN
            with pytest.raises(nf.NFError):
                p.accel(torch.empty((2, 3), device="cuda"))
        p.bin(torch.rand((10, 3), device="cuda"))      # the plan recovers
        p.accel()
        # the binding refuses output buffers that do not match the last binning (the C ABI would write out of bounds)
        with pytest.raises(ValueError):
            p.accel(torch.empty((9, 3), device="cuda"))
        with pytest.raises(ValueError):
            nf.nf_accel_kick(p._h, None, None, 0.1, torch.empty(5, device="cuda"))
        with pytest.raises(ValueError):
            nf.nf_accel_kick(p._h, None, torch.zeros((11, 3), device="cuda"), 0.1, None)
    # cpd < 2R+1 is the argument error, not R itself
    with pytest.raises(nf.NFError) as e:
        nf.Plan(10, 1.0, 0.01, 5)
    assert e.value.code == B.NF_ERR_ARG
    nf.Plan(11, 1.0, 0.01, 5).close()


# ---------------------------------------------------------------- fused kernel density estimate
TOL_RHO = 1e-5   # |rho_gpu - rho_ref| <= TOL_RHO * rho_ref for every particle (weights are O(1), rho >= 1)


def density_check(oracle_mod, pos_cpu, cpd, L, eps, b, R=2, options=None, sinks=None, what=""):
    import paper_2110_11398_b200 as nf
    pos = pos_cpu.numpy()
    with nf.Plan(cpd, L, eps, R) as plan:
        for k, v in (options or {}).items():
            plan.set_option(k, v)
        plan.bin(pos_cpu.cuda())
        acc, rho = plan.accel_density(b)
        acc0 = plan.accel()
        torch.cuda.synchronize()
    bn = oracle_mod.bin_particles(pos, cpd, L)
    ref_rho = oracle_mod.density(pos, cpd, L, b, R, sinks=sinks, binning=bn)
    ref_acc = oracle_mod.accel(pos, cpd, L, eps, R, sinks=sinks, binning=bn)
    g_rho = rho.cpu().numpy().astype(np.float64)
    g_acc = acc.cpu().numpy().astype(np.float64)
    if sinks is not None:
        g_rho, g_acc = g_rho[sinks], g_acc[sinks]
    err = np.abs(g_rho - ref_rho) / ref_rho
    assert err.max() <= TOL_RHO, f"{what}: density rel. error {err.max():.3e}"
    st = assert_parity(g_acc, ref_acc, what + " (accelerations of the fused pass)")
    # the force-only pass and the fused pass agree to rounding
    d = (acc - acc0).norm(dim=1) / acc0.norm(dim=1).clamp_min(1e-30)
    assert d.max().item() <= 1e-5
    return {"rho_max_err": float(err.max()), "rho_mean": float(ref_rho.mean()), **st}


def test_density_golden_gpu():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "density_two_body.txt")) if l.strip() and l[0] != "#"]
    import paper_2110_11398_b200 as nf
    for row in rows:
        cpd, R, b = int(row[0]), int(row[1]), float(row[2])
        v = [float(t) for t in row[3:]]
        pos = torch.tensor([v[0:3], v[3:6]], dtype=torch.float32)
        with nf.Plan(cpd, 1.0, 1e-6, R) as p:
            p.bin(pos.cuda())
            _, rho = p.accel_density(b)
        assert np.abs(rho.cpu().numpy() - v[6]).max() <= 1e-6, (row, rho)


@pytest.mark.parametrize("idx,n_side,cpd", [(1, 32, 9), (2, 48, 12), (4, 40, 10), (5, 40, 10)])
def test_density_scaled_configs(oracle_mod, idx, n_side, cpd):
    """b = 0.4 interparticle spacings on the config recipes, every particle compared."""
    cfg = nf_inputs.scaled(idx, n_side, cpd)
    st = density_check(oracle_mod, nf_inputs.generate(cfg), cfg.cpd, cfg.L, cfg.eps, 0.4 * cfg.L / cfg.n_side, cfg.R, what=cfg.name)
    print(cfg.name, st)


@pytest.mark.parametrize("cpd,R,bw,variant", [(6, 2, 1.5, 0), (6, 2, 2.0, 1), (5, 2, 0.3, 1), (7, 3, 0.999, 0), (3, 1, 1.0, 0),
                                             (8, 2, 0.05, 0)])
def test_density_radius_sweep(oracle_mod, cpd, R, bw, variant):
    """b from a small fraction of a cell up to R cell widths (kernel reaching every stencil cell), both kernel variants."""
    g = torch.Generator().manual_seed(cpd * 7 + R)
    pos = torch.rand((5000, 3), generator=g)
    st = density_check(oracle_mod, pos, cpd, 1.0, 0.004, bw / cpd, R, options={"variant": variant}, what=f"b={bw} cells")
    print(st)


def test_density_config3_full_size_sampled(oracle_mod):
    cfg = nf_inputs.config(3)
    pos = nf_inputs.generate(cfg)
    bn = oracle_mod.bin_particles(pos.numpy(), cfg.cpd, cfg.L)
    sinks = sample_sinks(bn["count"], bn["offset"], bn["perm"], cfg.cpd, np.random.default_rng(3), n_random=600)
    st = density_check(oracle_mod, pos, cfg.cpd, cfg.L, cfg.eps, 0.4 * cfg.L / cfg.n_side, cfg.R, sinks=sinks, what=cfg.name)
    print(cfg.name, "density, sampled sinks", len(sinks), st)


def test_density_errors_and_empty():
    import paper_2110_11398_b200 as nf
    B = nf.binding
    with nf.Plan(5, 1.0, 0.01, 2) as p:
        with pytest.raises(nf.NFError) as e:
            p.accel_density(0.05)
        assert e.value.code == B.NF_ERR_STATE
        p.bin(torch.rand((100, 3), device="cuda"))
        for bad in (0.0, -1.0, 0.41, float("nan")):             # R cell widths = 0.4
            with pytest.raises(nf.NFError) as e:
                p.accel_density(bad)
            assert e.value.code == B.NF_ERR_ARG
        p.bin(torch.zeros((0, 3), device="cuda"))
        a, r = p.accel_density(0.1)
        assert a.shape == (0, 3) and r.shape == (0,)


# ---------------------------------------------------------------- fused epilogue: kick + per-cell max |a| (NEXT 2)
def kick_check(oracle_mod, pos_cpu, cpd, L, eps, dt, R=2, v0=None, what=""):
    import paper_2110_11398_b200 as nf
    pos = pos_cpu.numpy()
    n = pos.shape[0]
    v0 = torch.zeros((n, 3)) if v0 is None else v0
    vel = v0.clone().cuda()
    with nf.Plan(cpd, L, eps, R) as plan:
        plan.bin(pos_cpu.cuda())
        acc, amax = plan.accel_kick(vel, dt)
        acc0 = plan.accel()
        vel2 = v0.clone().cuda()
        none_acc, amax2 = plan.accel_kick(vel2, dt, store_acc=False)           # accelerations not stored
        torch.cuda.synchronize()
    assert none_acc is None and torch.equal(vel, vel2) and torch.equal(amax, amax2)
    assert torch.equal(acc, acc0)                                              # the epilogue does not change the forces
    bn = oracle_mod.bin_particles(pos, cpd, L)
    a_ref = oracle_mod.accel(pos, cpd, L, eps, R, binning=bn)
    st = assert_parity(acc.cpu().numpy().astype(np.float64), a_ref, what)
    # kick: the velocity change against a_ref dt, same tolerance as the accelerations, plus the float32
    # rounding of the updated velocity (one FMA: half an ulp of v)
    v_ref = oracle_mod.kick(v0.numpy(), a_ref, dt)
    v_gpu = vel.cpu().numpy().astype(np.float64)
    num = np.linalg.norm(v_gpu - v_ref, axis=1)
    den = np.linalg.norm(a_ref * dt, axis=1)
    slack = 2.0 ** -23 * np.linalg.norm(v_ref, axis=1)
    ok = num <= 1e-5 * den + slack
    assert ok.mean() >= 0.999 and np.all(num <= 1e-3 * den + slack), f"{what}: kick"
    # per-cell maximum |a|
    m_ref = oracle_mod.cell_max_accel(a_ref, bn["cid"], cpd ** 3)
    m_gpu = amax.cpu().numpy().astype(np.float64)
    assert np.all((m_gpu == 0) == (bn["count"] == 0))
    nz = m_ref > 0
    err = np.abs(m_gpu[nz] - m_ref[nz]) / m_ref[nz]
    assert np.quantile(err, 0.999) <= 1e-5 and err.max() <= 1e-3, f"{what}: cell max {err.max():.3e}"
    return {"amax_max_err": float(err.max()), **st}


@pytest.mark.parametrize("idx,n_side,cpd", [(1, 32, 9), (2, 48, 12), (4, 40, 10), (5, 40, 10)])
def test_kick_scaled_configs(oracle_mod, idx, n_side, cpd):
    cfg = nf_inputs.scaled(idx, n_side, cpd)
    pos = nf_inputs.generate(cfg)
    g = torch.Generator().manual_seed(idx)
    v0 = torch.randn((cfg.n, 3), generator=g) * 50.0
    print(cfg.name, kick_check(oracle_mod, pos, cfg.cpd, cfg.L, cfg.eps, 1e-3, cfg.R, v0=v0, what=cfg.name))
    kick_check(oracle_mod, pos, cfg.cpd, cfg.L, cfg.eps, -0.25, cfg.R, what=cfg.name + " v0=0, dt<0")


def test_kick_golden_two_body_gpu():
    """a = +-256 x, dt = 2^-10: v_x changes by +-1/4 exactly; the cell maximum is 256, every other cell 0."""
    import paper_2110_11398_b200 as nf
    pos = torch.tensor([[0.53125, 0.5625, 0.5625], [0.59375, 0.5625, 0.5625]])
    vel = torch.tensor([[1.0, 2.0, 3.0], [-1.0, 0.5, 0.0]]).cuda()
    with nf.Plan(8, 1.0, 1e-6, 2) as p:
        p.bin(pos.cuda())
        _, amax = p.accel_kick(vel, 2.0 ** -10)
    v = vel.cpu().numpy()
    assert np.abs(v - np.array([[1.25, 2.0, 3.0], [-1.25, 0.5, 0.0]])).max() <= 1e-6
    m = amax.cpu().numpy()
    assert abs(m[(4 * 8 + 4) * 8 + 4] - 256.0) <= 1e-3 and np.count_nonzero(m) == 1


def test_kick_errors_and_empty():
    import paper_2110_11398_b200 as nf
    B = nf.binding
    with nf.Plan(5, 1.0, 0.01, 2) as p:
        with pytest.raises(nf.NFError) as e:
            nf.nf_accel_kick(p._h, None, torch.zeros((3, 3), device="cuda"), 0.1, None)
        assert e.value.code == B.NF_ERR_STATE
        p.bin(torch.rand((100, 3), device="cuda"))
        with pytest.raises(nf.NFError) as e:
            nf.nf_accel_kick(p._h, None, None, 0.1, None)
        assert e.value.code == B.NF_ERR_ARG
        with pytest.raises(nf.NFError) as e:
            p.accel_kick(torch.zeros((100, 3), device="cuda"), float("inf"))
        assert e.value.code == B.NF_ERR_ARG
        p.bin(torch.zeros((0, 3), device="cuda"))
        a, m = p.accel_kick(torch.zeros((0, 3), device="cuda"), 0.1)
        torch.cuda.synchronize()
        assert a.shape == (0, 3) and not m.cpu().numpy().any()


# ---------------------------------------------------------------- x-slab decomposition (NEXT 3), ranks emulated one after another
@pytest.mark.parametrize("idx,n_side,cpd,world,balanced", [(3, 40, 10, 2, False), (4, 40, 10, 3, True), (1, 32, 9, 4, True),
                                                           (2, 48, 5, 2, False), (4, 48, 12, 4, True), (5, 40, 10, 5, True)])
def test_slab_decomposition_matches_whole_box(oracle_mod, idx, n_side, cpd, world, balanced):
    """Each emulated rank bins its slabs plus the halo its peers would send (slabs.pack_for_peers: nf_slab_histogram +
    nf_slab_select on the device, the function halo_exchange ships) and computes its own sinks: bit-identical to the
    whole-box plan, interaction counts add up.  Ranges: equal slab counts, or balanced by the library's slab costs."""
    import paper_2110_11398_b200 as nf
    from paper_2110_11398_b200 import slabs
    cfg = nf_inputs.scaled(idx, n_side, cpd)
    pos = nf_inputs.generate(cfg)
    pos_d = pos.cuda()
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as plan:
        plan.set_option("window", 64)       # any window: equal on every plan
        plan.set_option("quad_vote", idx % 2)   # any instance of the direct kernel: equal on every plan (the automatic choice
        plan.bin(pos_d)                         # looks at the fullest cell a plan holds, which differs between the ranks)
        whole = plan.accel().cpu()
        total = plan.stats()["interactions"]
        cost = plan.slab_cost()
        assert sum(cost) == total                                      # the scheduler's exact cost, per slab
        parts = slabs.slab_partition(cfg.cpd, world, cost if balanced else None)
        sel = slabs.LibrarySelector(plan)
        b = oracle_mod.bin_particles(pos.numpy(), cfg.cpd, cfg.L)
        sl_ref = (b["cid"] // (cfg.cpd * cfg.cpd)).astype(np.int64)
        assert sel.histogram(pos_d) == np.bincount(sl_ref, minlength=cfg.cpd).tolist()
        owned, idx_owned = [], []
        for f, c in parts:
            o, i = plan.slab_select(pos_d, f, c, pos.shape[0], want_index=True)
            ref_i = np.nonzero(((sl_ref - f) % cfg.cpd) < c)[0]
            assert np.array_equal(i.cpu().numpy(), ref_i) and torch.equal(o.cpu(), pos[ref_i])      # stable, exact copies
            owned.append(o.contiguous())
            idx_owned.append(i.cpu())
        sends = [slabs.pack_for_peers(owned[q], cfg.cpd, cfg.R, q, world, parts, sel)[0] for q in range(world)]
    assert sum(c for _, c in parts) == cfg.cpd and all(c >= 1 for _, c in parts)
    got = torch.full_like(whole, float("nan"))
    inter = 0
    for r, (f, c) in enumerate(parts):
        local = torch.cat([owned[r]] + [sends[q][r] for q in range(world) if q != r]).contiguous()
        with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as plan:
            plan.set_sink_slabs(f, c)
            plan.set_option("window", 64)
            plan.set_option("quad_vote", idx % 2)
            plan.bin(local)
            acc = torch.full((local.shape[0], 3), 7.0, device="cuda")
            plan.accel(acc)
            torch.cuda.synchronize()
            inter += plan.stats()["interactions"]
            mine = plan.slab_cost()                                     # owned slabs only: the ranks' vectors add up
            assert all(mine[s] == (cost[s] if ((s - f) % cfg.cpd) < c else 0.0) for s in range(cfg.cpd))
        acc = acc.cpu()
        assert torch.all(acc[owned[r].shape[0]:] == 7.0)              # halo rows are not written
        got[idx_owned[r]] = acc[:owned[r].shape[0]]
    assert torch.equal(got, whole)
    assert inter == total
    ref = oracle_mod.accel(pos.numpy(), cfg.cpd, cfg.L, cfg.eps, cfg.R)
    assert_parity(got.numpy().astype(np.float64), ref, f"{cfg.name} in {world} slab ranges")
    if balanced:                                                       # the point of the cost partition: the slowest rank's share
        load = lambda pp: max(sum(cost[(f + i) % cfg.cpd] for i in range(c)) for f, c in pp)
        assert load(parts) <= load(slabs.slab_partition(cfg.cpd, world)) * (1 + 1e-12)


def test_sink_slab_errors():
    import paper_2110_11398_b200 as nf
    with nf.Plan(6, 1.0, 0.01, 2) as p:
        for bad in ((-1, 2), (6, 1), (0, 0), (0, 7)):
            with pytest.raises(nf.NFError) as e:
                p.set_sink_slabs(*bad)
            assert e.value.code == nf.binding.NF_ERR_ARG
        p.bin(torch.rand((50, 3), device="cuda"))
        p.set_sink_slabs(4, 3)                                        # wraps: slabs 4, 5, 0
        with pytest.raises(nf.NFError) as e:                          # the binning was invalidated
            p.accel()
        assert e.value.code == nf.binding.NF_ERR_STATE


# ---------------------------------------------------------------- Plummer comparison law (NEXT 4)
@pytest.mark.parametrize("idx,n_side,cpd,variant", [(1, 32, 9, 0), (4, 40, 10, 0), (5, 40, 10, 1)])
def test_plummer_softening(oracle_mod, idx, n_side, cpd, variant):
    cfg = nf_inputs.scaled(idx, n_side, cpd)
    pos = nf_inputs.generate(cfg)
    out = gpu_run(pos, cfg.cpd, cfg.L, cfg.eps, cfg.R, options={"softening": 1, "variant": variant})
    ref = oracle_mod.accel(pos.numpy(), cfg.cpd, cfg.L, cfg.eps, cfg.R, softening="plummer")
    print(cfg.name, "plummer", assert_parity(out["acc"], ref, cfg.name + " plummer"))
    spline = oracle_mod.accel(pos.numpy(), cfg.cpd, cfg.L, cfg.eps, cfg.R)
    assert rel_errors(out["acc"], spline).max() > 1e-4            # it really is a different law


def test_plummer_two_body_and_large_eps(oracle_mod):
    """3-4-5 case: |a| = 98.304; eps of several cell widths (no compact support: every stencil cell is softened)."""
    pos = torch.tensor([[0.5, 0.5625, 0.5625], [0.5 + 3 / 64, 0.5625, 0.5625]])
    a = gpu_run(pos, 8, 1.0, 1 / 16, 2, options={"softening": 1})["acc"]
    assert np.abs(a - np.array([[98.304, 0, 0], [-98.304, 0, 0]])).max() <= 2e-5
    g = torch.Generator().manual_seed(5)
    p = torch.rand((4000, 3), generator=g)
    for eps in (0.3, 0.0):
        out = gpu_run(p, 6, 1.0, eps, 2, options={"softening": 1})
        assert_parity(out["acc"], oracle_mod.accel(p.numpy(), 6, 1.0, eps, 2, softening="plummer"), f"plummer eps={eps}")


def test_bitwise_determinism():
    """No floating-point atomics anywhere: the summation order of a sink is fixed by the layout, not by which CTA picks
    its work unit, so repeated runs, the unit order (heavy_first) and re-binning give bit-identical accelerations."""
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.scaled(4, 48, 12)
    pos = nf_inputs.generate(cfg).cuda()
    outs = []
    for hf in (1, 0, 1):
        with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as p:
            p.set_option("heavy_first", hf)
            p.bin(pos)
            a1 = p.accel().clone()
            a2, rho = p.accel_density(0.4 * cfg.L / cfg.n_side)
            p.bin(pos)
            a3 = p.accel()
            torch.cuda.synchronize()
            assert torch.equal(a1, a3)
            outs.append((a1, a2.clone(), rho.clone()))
    for o in outs[1:]:
        assert all(torch.equal(x, y) for x, y in zip(o, outs[0]))


@pytest.mark.parametrize("idx,n_side,cpd", [(1, 32, 9), (4, 40, 10)])
def test_window_sizes(oracle_mod, idx, n_side, cpd):
    """Sinks per work unit ("window": multiples of 32 up to 256, 0 = the default 256): every choice within tolerance of the
    oracle, same interaction count, bit-identical for equal windows; bad values are rejected."""
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.scaled(idx, n_side, cpd)
    pos = nf_inputs.generate(cfg)
    ref = oracle_mod.accel(pos.numpy(), cfg.cpd, cfg.L, cfg.eps, cfg.R)
    counts, units = set(), {}
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as p:
        for w in (0, 32, 64, 96, 128, 224, 256, 64):
            p.set_option("window", w)
            p.bin(pos.cuda())
            a = p.accel().cpu()
            st = p.stats()
            counts.add(st["interactions"])
            assert_parity(a.numpy().astype(np.float64), ref, f"{cfg.name} window {w}")
            if w in units:
                assert torch.equal(units[w], a)
            units[w] = a
        with pytest.raises(nf.NFError):
            p.set_option("window", 48)
    assert len(counts) == 1


def test_config4_full_size_density_and_kick_sampled(oracle_mod):
    """The fused passes at the clustered production size (cells of 2.6e5 particles): density, kick and per-cell maxima on
    the sink sample, accelerations of the fused passes bit-identical to nf_accel."""
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.config(4)
    pos_dev = nf_inputs.generate(cfg, device="cuda")
    pos = pos_dev.cpu().numpy()
    b = oracle_mod.bin_particles(pos, cfg.cpd, cfg.L)
    sinks = sample_sinks(b["count"], b["offset"], b["perm"], cfg.cpd, np.random.default_rng(44), n_random=500, n_heavy=10, per_heavy=100)
    bw = 0.4 * cfg.L / cfg.n_side
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as plan:
        plan.bin(pos_dev)
        acc = plan.accel()
        acc_d, rho = plan.accel_density(bw)
        vel = torch.zeros_like(pos_dev)
        acc_k, amax = plan.accel_kick(vel, 2.0 ** -20)
        torch.cuda.synchronize()
    assert torch.equal(acc_k, acc) and torch.equal(vel, acc * 2.0 ** -20)
    assert (acc_d - acc).norm().item() <= 1e-6 * acc.norm().item()
    idx = torch.from_numpy(sinks).cuda()
    ref_rho = oracle_mod.density(pos, cfg.cpd, cfg.L, bw, cfg.R, sinks=sinks, binning=b)
    err = np.abs(rho[idx].cpu().numpy().astype(np.float64) - ref_rho) / ref_rho
    assert err.max() <= TOL_RHO, err.max()
    ref = oracle_mod.accel(pos, cfg.cpd, cfg.L, cfg.eps, cfg.R, sinks=sinks, binning=b)
    st = assert_parity(acc[idx].cpu().numpy().astype(np.float64), ref, cfg.name + " fused passes (sampled)")
    # per-cell maxima: exact maximum of the float32 norms the kernel wrote, for every cell
    norms = acc.double().norm(dim=1)
    cid = torch.from_numpy(b["cid"].astype(np.int64)).cuda()
    m_ref = torch.zeros(cfg.cpd ** 3, dtype=torch.float64, device="cuda").scatter_reduce_(0, cid, norms, "amax")
    assert torch.allclose(amax.double(), m_ref, rtol=2e-7, atol=0)
    print(cfg.name, "fused passes", st, "rho max err", float(err.max()), "rho max", float(ref_rho.max()))


# ---------------------------------------------------------------- per-particle source masses
@pytest.mark.parametrize("idx,n_side,cpd,options", [(1, 32, 9, {}), (4, 40, 10, {}), (4, 32, 8, {"variant": 1}),
                                                    (2, 48, 12, {"softening": 1}), (5, 40, 10, {"fastpath": 0})])
def test_masses_parity(oracle_mod, idx, n_side, cpd, options):
    """nf_set_masses: a_i = sum_j m_j d K against oracle.accel_mass (log-normal masses), same tolerance; unit masses
    through the mass kernel are bit-identical to the plain kernel; nf_bin and set_masses(None) return to m = 1."""
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.scaled(idx, n_side, cpd)
    pos = nf_inputs.generate(cfg)
    mass = nf_inputs.masses(cfg)
    soft = "plummer" if options.get("softening") else "spline"
    ref = oracle_mod.accel_mass(pos.numpy(), mass.numpy(), cfg.cpd, cfg.L, cfg.eps, cfg.R, softening=soft)
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as p:
        for k, v in options.items():
            p.set_option(k, v)
        p.bin(pos.cuda())
        unit = p.accel().cpu()
        p.set_masses(mass.cuda())
        a = p.accel().cpu()
        st = assert_parity(a.numpy().astype(np.float64), ref, f"{cfg.name} masses {options}")
        print(cfg.name, options, st)
        assert torch.equal(p.accel().cpu(), a)                              # deterministic
        p.set_masses(torch.ones(cfg.n, device="cuda"))
        assert torch.equal(p.accel().cpu(), unit)                           # k * 1 = k: the same bits as the plain kernel
        p.set_masses(mass.cuda())
        p.set_masses(None)
        assert torch.equal(p.accel().cpu(), unit)
        p.set_masses(mass.cuda())
        p.bin(pos.cuda())                                                   # a new binning starts with unit masses
        assert torch.equal(p.accel().cpu(), unit)


def test_masses_fused_passes_and_errors(oracle_mod):
    """Density and kick entry points with masses: forces bit-identical to nf_accel with the same masses, the density
    estimate unchanged by them (count-based); massless particles are test particles; state errors."""
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.scaled(4, 32, 8)
    pos = nf_inputs.generate(cfg)
    mass = nf_inputs.masses(cfg)
    mass[::5] = 0.0
    ref = oracle_mod.accel_mass(pos.numpy(), mass.numpy(), cfg.cpd, cfg.L, cfg.eps, cfg.R)
    b = 0.4 / cfg.n_side
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as p:
        p.n = cfg.n
        p.set_option("quad_vote", 0)        # one vote granularity in every entry point: then the forces agree bit for bit
        with pytest.raises(nf.NFError):
            p.set_masses(mass.cuda())                                       # before nf_bin
        p.bin(pos.cuda())
        _, rho_unit = p.accel_density(b)
        rho_unit = rho_unit.cpu()
        p.set_masses(mass.cuda())
        a = p.accel().cpu()
        assert_parity(a.numpy().astype(np.float64), ref, "masses with test particles")
        a2, rho = p.accel_density(b)
        # the fused density pass votes on max(eps_s, b) per four sources, the force-only pass on eps_s: a pair within 0.1 % of
        # eps_s may or may not take the spline's min (equal there to 1e-7), so the forces agree to rounding, not bit for bit
        assert ((a2.cpu() - a).norm(dim=1) <= 2e-6 * a.norm(dim=1)).all() and torch.equal(rho.cpu(), rho_unit)
        vel = torch.zeros((cfg.n, 3), device="cuda")
        a3, _ = p.accel_kick(vel, 0.5)
        assert torch.equal(a3.cpu(), a)
        assert torch.equal(vel.cpu(), a * 0.5)
        with pytest.raises(TypeError):
            p.set_masses(mass[:-1].cuda())
    with nf.Plan(4, 1.0, 0.01, 1) as p:                                     # n = 0
        p.bin(torch.zeros((0, 3), device="cuda"))
        p.set_masses(torch.zeros(0, device="cuda"))
        assert p.accel().shape == (0, 3)


@pytest.mark.parametrize("idx,device", [(3, "cpu"), (4, "cuda")])
def test_masses_full_size_sampled(oracle_mod, idx, device):
    """Masses at the full uniform and clustered sizes (the launch configuration bench.py times): accelerations of the
    sink sample against oracle.accel_mass, total momentum sum_i m_i a_i = 0 within FP32 bounds."""
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.config(idx)
    pos_dev = nf_inputs.generate(cfg, device=device).cuda()
    mass_dev = nf_inputs.masses(cfg, device=device).cuda()
    pos, mass = pos_dev.cpu().numpy(), mass_dev.cpu().numpy()
    b = oracle_mod.bin_particles(pos, cfg.cpd, cfg.L)
    sinks = sample_sinks(b["count"], b["offset"], b["perm"], cfg.cpd, np.random.default_rng(cfg.seed + 1), n_random=500,
                         n_heavy=10, per_heavy=100)
    ref = oracle_mod.accel_mass(pos, mass, cfg.cpd, cfg.L, cfg.eps, cfg.R, sinks=sinks, binning=b)
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as plan:
        plan.bin(pos_dev)
        plan.set_masses(mass_dev)
        acc = plan.accel()
        torch.cuda.synchronize()
    st = assert_parity(acc[torch.from_numpy(sinks).cuda()].cpu().numpy().astype(np.float64), ref, cfg.name + " masses (sampled)")
    ma = acc.double() * mass_dev.double()[:, None]
    assert float(ma.sum(0).abs().max()) <= 2e-6 * float(ma.abs().sum())
    print(cfg.name, "masses, sampled sinks", len(sinks), st)


@pytest.mark.parametrize("ns", [1, 31, 32, 33, 65, 96, 97, 129, 161, 193, 225, 255, 256, 257, 300])
def test_short_windows_share_stages(oracle_mod, ns):
    """One z-column holding `ns` particles next to a filled box: the column's windows have every number of sink groups
    (1..8), so the warps that share a window's stages come in all splits (8, 4, 2, 2, 1, ... with idle warps for 3, 5, 6, 7
    groups); results against the oracle and bit-identical between two runs (the partial sums are added in a fixed order)."""
    import paper_2110_11398_b200 as nf
    cpd, R, L = 6, 2, 1.0
    rng = np.random.default_rng(ns)
    col = rng.random((ns, 3)).astype(np.float32)
    col[:, 0] = (col[:, 0] + 2) / cpd                         # column (2, 3)
    col[:, 1] = (col[:, 1] + 3) / cpd
    rest = rng.random((3000, 3)).astype(np.float32)
    keep = ~((np.floor(rest[:, 0] * cpd) == 2) & (np.floor(rest[:, 1] * cpd) == 3))
    pos = torch.from_numpy(np.concatenate([col, rest[keep]]))
    eps = 0.01
    ref = oracle_mod.accel(pos.numpy(), cpd, L, eps, R)
    with nf.Plan(cpd, L, eps, R) as p:
        p.set_option("window", 256)                           # the column is one window of ns sinks (two from 257)
        p.bin(pos.cuda())
        a1 = p.accel().cpu()
        a2, rho = p.accel_density(0.05)
        a3 = p.accel().cpu()
    assert torch.equal(a1, a3) and torch.equal(a1, a2.cpu())
    assert_parity(a1.numpy().astype(np.float64), ref, f"column of {ns}")
    rho_ref = oracle_mod.density(pos.numpy(), cpd, L, 0.05, R)
    assert np.all(np.abs(rho.cpu().numpy() - rho_ref) <= 1e-5 * rho_ref)


# ---------------------------------------------------------------- incremental re-binning (nf_rebin)
def _drift(pos: torch.Tensor, L: float, cell: float, rms_cells: float, gen: torch.Generator, jump_frac: float = 0.0):
    """Seeded sub-cell displacements (the paper's particles drift much less than a cell per step), wrapped
    through the periodic faces; `jump_frac` of the particles additionally jump by up to two cells."""
    d = torch.randn(pos.shape, generator=gen, dtype=torch.float64) * (rms_cells * cell)
    if jump_frac > 0:
        who = torch.rand(pos.shape[0], generator=gen) < jump_frac
        d[who] += (torch.rand((int(who.sum()), 3), generator=gen, dtype=torch.float64) - 0.5) * 4 * cell
    q = torch.remainder(pos.double() + d, L).to(torch.float32)
    q[q >= L] = 0.0
    return q.contiguous()


def _rebin_check(oracle_mod, plan, pos, cfg, what, expect_path=None, fresh=True):
    import paper_2110_11398_b200 as nf
    plan.rebin(pos.cuda())
    acc = plan.accel()
    torch.cuda.synchronize()
    st = plan.stats()
    b = oracle_mod.bin_particles(pos.numpy(), cfg.cpd, cfg.L)
    assert_binning_equal({k: u32(v) for k, v in plan.binning().items()}, b)          # byte-equal to the oracle's definition
    assert st["interactions"] == oracle_mod.interactions(b["count"], cfg.cpd, cfg.R), what
    if expect_path is not None:
        assert st["rebin_path"] == expect_path, (what, st["rebin_path"], st["rebin_movers"])
    if fresh:                                                                       # same layout => same bits as a full nf_bin
        with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as p2:
            p2.bin(pos.cuda())
            acc2 = p2.accel()
            lay, lay2 = plan.layout(), p2.layout()
            for key in ("poff", "x", "y", "z"):
                assert torch.equal(lay[key], lay2[key]), (what, key)
            assert torch.equal(acc, acc2), what
    return acc, b, st


@pytest.mark.parametrize("idx,n_side,cpd", [(3, 40, 10), (4, 40, 10), (2, 48, 12), (1, 32, 9)])
def test_rebin_drift_steps(oracle_mod, idx, n_side, cpd):
    """k drift steps of seeded sub-cell displacements (face crossings, the periodic boundary, particles leaving the heavy
    cells of the clustered recipe): after every step nf_rebin equals nfo_bin byte for byte and the accelerations meet the
    tolerance (and are bit-identical to those of a fresh nf_bin)."""
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.scaled(idx, n_side, cpd)
    pos = nf_inputs.generate(cfg)
    gen = torch.Generator().manual_seed(900 + idx)
    cell = cfg.L / cfg.cpd
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as plan:
        plan.bin(pos.cuda())
        prev, seen = 0, 0
        for step, (rms, jump) in enumerate([(0.004, 0.0), (0.01, 0.0), (0.0, 0.0), (0.02, 0.002), (0.1, 0.0), (0.004, 0.0), (0.004, 0.0)]):
            pos = _drift(pos, cfg.L, cell, rms, gen, jump) if rms > 0 or jump > 0 else pos
            # more than 1/16 of the particles moved in the previous call: this one sorts from scratch (and counts no movers)
            # (a large drift may also overflow the per-cell arrival lists of the halo cells: either path is right then)
            path = 2 if prev > cfg.n // 16 else (None if rms >= 0.05 else 1)
            acc, b, st = _rebin_check(oracle_mod, plan, pos, cfg, f"{cfg.name} drift step {step}", expect_path=path)
            prev = st["rebin_movers"]
            if path == 1 and step == 2:
                assert st["rebin_movers"] == 0
            elif path == 1:
                assert 0 <= st["rebin_movers"] < cfg.n // 4
                seen += st["rebin_movers"]
            ref = oracle_mod.accel(pos.numpy(), cfg.cpd, cfg.L, cfg.eps, cfg.R, binning=b)
            assert_parity(acc.cpu().numpy().astype(np.float64), ref, f"{cfg.name} drift step {step}")
        assert seen > 0                                                # the merge path really moved particles


def test_rebin_fallbacks_and_errors(oracle_mod):
    """Everything moved (new random positions), one cell receiving more arrivals than the merge handles, the call after
    a step with many movers, errors: the result is always nfo_bin's."""
    import paper_2110_11398_b200 as nf
    B = nf.binding
    cfg = nf_inputs.scaled(3, 32, 8)
    pos = nf_inputs.generate(cfg)
    gen = torch.Generator().manual_seed(77)
    cell = cfg.L / cfg.cpd
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as plan:
        with pytest.raises(nf.NFError) as e:
            plan.rebin(pos.cuda())
        assert e.value.code == B.NF_ERR_STATE
        plan.bin(pos.cuda())
        with pytest.raises(ValueError):
            plan.rebin(pos[:100].cuda())                                   # another n: the binding refuses
        pos = torch.rand(pos.shape, generator=gen)                         # every particle somewhere else: sorted from scratch
        _rebin_check(oracle_mod, plan, pos, cfg, "teleport", expect_path=2)
        pos = _drift(pos, cfg.L, cell, 0.3, gen)                           # ~1/3 of the particles change cell: merge still exact
        _, _, st = _rebin_check(oracle_mod, plan, pos, cfg, "large drift")
        pos = _drift(pos, cfg.L, cell, 0.01, gen)                          # the call after many movers goes straight to the sort
        _rebin_check(oracle_mod, plan, pos, cfg, "after many movers", expect_path=2 if st["rebin_movers"] > cfg.n // 16 else 1)
        pos = _drift(pos, cfg.L, cell, 0.01, gen)
        _rebin_check(oracle_mod, plan, pos, cfg, "incremental again", expect_path=1)
        q = pos.clone()                                                    # 2000 particles collapse into one cell (> 512 arrivals)
        q[:2000] = torch.tensor([0.51, 0.52, 0.53]) + torch.rand((2000, 3), generator=gen) * 0.01
        _rebin_check(oracle_mod, plan, q.contiguous(), cfg, "collapse into one cell", expect_path=2)
        bad = q.clone()
        bad[5, 1] = float("nan")
        with pytest.raises(nf.NFError) as e:
            plan.rebin(bad.cuda())
        assert e.value.code == B.NF_ERR_DOMAIN
        with pytest.raises(nf.NFError) as e:                               # the binning is invalid after the error
            plan.accel()
        assert e.value.code == B.NF_ERR_STATE
        plan.bin(q.cuda())
        plan.set_sink_slabs(1, 3)                                          # options that change the units need a fresh nf_bin
        with pytest.raises(nf.NFError) as e:
            plan.rebin(q.cuda())
        assert e.value.code == B.NF_ERR_STATE
    with nf.Plan(5, 1.0, 0.01, 2) as plan:                                 # one particle, and none
        one = torch.tensor([[0.999, 0.5, 0.001]])
        plan.bin(one.cuda())
        plan.rebin(torch.tensor([[0.001, 0.5, 0.999]]).cuda())
        assert u32(plan.binning()["cid"]).tolist() == [0 * 25 + 2 * 5 + 4]
        assert torch.all(plan.accel() == 0)
        plan.bin(torch.empty((0, 3)).cuda())
        plan.rebin(torch.empty((0, 3)).cuda())


@pytest.mark.parametrize("seed", range(10))
def test_rebin_fuzz(oracle_mod, seed):
    """Random grids, distributions and drift amplitudes (none, tiny, a third of a cell, several cells), slab-restricted
    sinks, both kernel variants: three steps each against the oracle's binning, bit-identical to a fresh nf_bin."""
    import paper_2110_11398_b200 as nf
    from test_gpu_fuzz import KINDS, _positions
    rng = np.random.default_rng(4200 + seed)
    R = int(rng.integers(0, 4))
    cpd = int(rng.integers(2 * R + 1, 2 * R + 1 + rng.choice([1, 6, 20])))
    L = float(rng.choice([1.0, 0.125, 7.5]))
    n = int(rng.choice([1, 33, 3000, 20000, 60000]))
    pos = torch.from_numpy(_positions(rng, KINDS[seed % len(KINDS)], n, L))
    cell = L / cpd
    gen = torch.Generator().manual_seed(seed)
    with nf.Plan(cpd, L, 0.02 * cell, R) as plan:
        plan.set_option("variant", int(rng.integers(0, 2)))
        plan.bin(pos.cuda())
        for step in range(3):
            rms = float(rng.choice([0.0, 0.003, 0.03, 0.3, 1.5]))
            pos = _drift(pos, L, cell, rms, gen, jump_frac=float(rng.choice([0.0, 0.01])))
            plan.rebin(pos.cuda())
            acc = plan.accel()
            b = oracle_mod.bin_particles(pos.numpy(), cpd, L)
            assert_binning_equal({k: u32(v) for k, v in plan.binning().items()}, b)
            with nf.Plan(cpd, L, 0.02 * cell, R) as p2:
                p2.set_option("variant", 0)
                p2.bin(pos.cuda())
                lay, lay2 = plan.layout(), p2.layout()
                for key in ("poff", "x", "y", "z"):
                    assert torch.equal(lay[key], lay2[key]), (seed, step, key)
            assert plan.stats()["interactions"] == oracle_mod.interactions(b["count"], cpd, R)
            assert torch.isfinite(acc).all()


@pytest.mark.parametrize("idx,device", [(3, "cpu"), (4, "cuda")])
def test_rebin_full_size(oracle_mod, idx, device):
    """Config 3 / config 4 size: two drift steps at ~1 % movers, byte-equal to nfo_bin; prints the time of both paths."""
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.config(idx)
    pos = nf_inputs.generate(cfg, device=device).cpu()
    gen = torch.Generator().manual_seed(31 + idx)
    cell = cfg.L / cfg.cpd
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as plan:
        plan.bin(pos.cuda())
        ms_full = plan.stats()["ms_bin"]
        for step in range(2):
            pos = _drift(pos, cfg.L, cell, 0.004, gen)
            _, b, st = _rebin_check(oracle_mod, plan, pos, cfg, f"{cfg.name} rebin {step}", expect_path=1, fresh=(step == 1))
            print(f"{cfg.name}: nf_bin {ms_full:.3f} ms, nf_rebin {st['ms_bin']:.3f} ms with {st['rebin_movers']} movers "
                  f"({100.0 * st['rebin_movers'] / cfg.n:.2f} %)")


# ---------------------------------------------------------------- sparse windows: the flat loop of the direct kernel
@pytest.mark.parametrize("n,cpd,R,flat_below", [(8000, 10, 2, 22), (8000, 16, 2, 22), (6000, 20, 2, 22), (8000, 16, 2, 0), (20000, 12, 3, 1024),
                                                (30000, 9, 2, 1024), (3000, 25, 1, 22), (8000, 16, 2, 14)])
def test_sparse_flat_loop(oracle_mod, n, cpd, R, flat_below):
    """Windows with a handful of slots per cell walk a lane's stencil run in one flat loop (nf_set_option "flat_below"):
    8, 2 and 0.75 particles per cell with the default threshold, the same grid with the flat loop switched off, and dense
    grids FORCED onto the flat loop (threshold 1024) -- all against the oracle; voids and a clump in the same box."""
    g = torch.Generator().manual_seed(n + cpd)
    pos = torch.rand((n, 3), generator=g)
    pos[: n // 10] = 0.37 + 0.002 * torch.randn((n // 10, 3), generator=g)          # a clump: heavy cells next to sparse windows
    pos = torch.remainder(pos, 1.0).to(torch.float32).contiguous()
    pos[pos >= 1.0] = 0.0
    st, out = full_check(oracle_mod, pos, cpd, 1.0, 0.01 / cpd, R, options={"flat_below": flat_below}, what=f"flat n={n} cpd={cpd} R={R}")
    import paper_2110_11398_b200 as nf
    with nf.Plan(cpd, 1.0, 0.01 / cpd, R) as plan:                                   # fused passes on the same path
        plan.set_option("flat_below", flat_below)
        plan.bin(pos.cuda())
        acc, rho = plan.accel_density(0.4 / cpd)
        ref_rho = oracle_mod.density(pos.numpy(), cpd, 1.0, 0.4 / cpd, R)
        assert (np.abs(rho.cpu().numpy().astype(np.float64) - ref_rho) / ref_rho).max() <= 1e-5
        assert (acc.cpu().double().numpy() - out["acc"]).__abs__().max() <= 1e-5 * np.abs(out["acc"]).max()


@pytest.mark.parametrize("kind,n,cpd,R,flat_below", [
    ("uniform", 20000, 5, 2, 1024),      # cpd = 2R+1, one window spans the column: the run [-2, 6] has THREE periodic segments
    ("uniform", 2500, 7, 3, 1024),       # the same with R = 3 (run longer than the column)
    ("uniform", 60000, 6, 2, 1024),      # forced flat on dense cells: the run exceeds a stage, the producer falls back to the piece table
    ("columns", 3000, 300, 2, 22),       # ten columns of a 300^3 grid: one window spans 300 cells, above the 256 a lean stage describes
    ("columns", 2000, 250, 2, 22),       # 254-cell runs: the longest a lean stage takes, through both periodic faces
    ("faces", 6000, 24, 2, 22),          # particles crowded at z = 0 and z = L: every run of the face windows wraps
])
def test_lean_stages(oracle_mod, kind, n, cpd, R, flat_below):
    """Lean stages of the flat loop: the producer copies the padded offsets of a whole z-run instead of building
    a per-cell table.  Runs in one, two and three periodic segments, the two fallbacks to the piece table (more slots than a
    stage, more cells than a lean stage describes) and a mix of both in one unit -- each against the oracle, and against the
    stepped loop of the same binning (flat_below = 0; the FP32 chains are cut at different places, so not bit for bit)."""
    g = torch.Generator().manual_seed(7 * n + cpd)
    pos = torch.rand((n, 3), generator=g)
    if kind == "columns":
        cols = torch.randint(0, cpd, (10, 2), generator=g).float()
        pick = torch.randint(0, 10, (n,), generator=g)
        pos[:, 0] = (cols[pick, 0] + pos[:, 0]) / cpd
        pos[:, 1] = (cols[pick, 1] + pos[:, 1]) / cpd
    elif kind == "faces":
        pos[: n // 2, 2] = torch.remainder(0.02 * torch.randn(n // 2, generator=g), 1.0)
    pos = torch.remainder(pos, 1.0).to(torch.float32).contiguous()
    pos[pos >= 1.0] = 0.0
    eps = 0.01 / cpd
    st, out = full_check(oracle_mod, pos, cpd, 1.0, eps, R, options={"flat_below": flat_below}, what=f"lean {kind} n={n} cpd={cpd} R={R}")
    import paper_2110_11398_b200 as nf
    res = []
    for fb in (flat_below, 0):
        with nf.Plan(cpd, 1.0, eps, R) as plan:
            plan.set_option("flat_below", fb)
            plan.bin(pos.cuda())
            res.append(plan.accel().cpu().numpy())
    d = np.abs(res[0].astype(np.float64) - res[1]).max(axis=1)
    scale = np.abs(out["acc"]).max(axis=1) + 1e-300
    # both are within 1e-5 (99.9 %) / 1e-3 of the oracle; against each other the triangle inequality gives twice that
    assert np.quantile(d / scale, 0.999) <= 2e-5 and (d / scale).max() <= 2e-3, (np.quantile(d / scale, 0.999), (d / scale).max())


def test_flat_units_take_their_own_launch(oracle_mod):
    """nf_bin sorts the flat units (sparse windows) behind all the others and nf_accel runs the two groups as two launches of
    two kernel instances.  A box with a dense half and a sparse half: two launches, against the oracle, and bit
    for bit what ONE launch of the instance that holds both loops gives (heavy_first = 0: the list is not partitioned)."""
    import paper_2110_11398_b200 as nf
    g = torch.Generator().manual_seed(31)
    n, cpd = 60000, 20
    pos = torch.rand((n, 3), generator=g)
    pos[: n * 9 // 10, 0] *= 0.5                                  # nine tenths of the particles in the half x < 1/2
    pos = pos.to(torch.float32).contiguous()
    st, out = full_check(oracle_mod, pos, cpd, 1.0, 0.01 / cpd, 2, what="dense half + sparse half")
    assert out["stats"]["kernel_launches_accel"] == 2, out["stats"]
    one = gpu_run(pos, cpd, 1.0, 0.01 / cpd, 2, options={"heavy_first": 0})
    assert one["stats"]["kernel_launches_accel"] == 1, one["stats"]
    assert np.array_equal(one["acc"], out["acc"])
    # all flat, none flat: one launch each
    assert gpu_run(pos, cpd, 1.0, 0.01 / cpd, 2, options={"flat_below": 0})["stats"]["kernel_launches_accel"] == 1
    sparse = torch.rand((4000, 3), generator=g).to(torch.float32)
    assert gpu_run(sparse, 24, 1.0, 0.01 / 24, 2)["stats"]["kernel_launches_accel"] == 1
