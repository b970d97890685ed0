"""nf_slab_histogram_static: the entry point that allocates nothing (scratch in a static device array of the library,
include/nf.h) against the existing path nf_slab_histogram -- integer work, so the results must be EQUAL -- on two calls in
a row with different inputs (the shared array keeps the previous call's contents and the call must clear it).
Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _positions(n, L, seed, clump):
    g = torch.Generator().manual_seed(seed)
    p = torch.rand((n, 3), generator=g, dtype=torch.float64)
    if clump:                                           # most particles in two slabs: another histogram than the call before
        p[: (3 * n) // 4, 0] = 0.41 + 0.05 * torch.rand((3 * n) // 4, generator=g, dtype=torch.float64)
    p = (p * L).to(torch.float32)
    p[p >= L] = 0.0
    return p.contiguous()


@pytest.mark.parametrize("cpd,L", [(9, 1.0), (63, 7.5), (1024, 1.0)])
def test_static_scratch_matches_allocating_path(oracle_mod, cpd, L):
    import paper_2110_11398_b200 as nf
    with nf.Plan(cpd, L, 0.001 * L / cpd, 2) as plan:
        plan._use_current_stream()
        for call, (n, clump) in enumerate([(200_000, False), (50_001, True)]):      # two calls in a row, no nf_bin in between
            pos = _positions(n, L, 100 * cpd + call, clump)
            pos_d = pos.cuda()
            ref = nf.nf_slab_histogram(plan._h, pos_d, cpd)                          # the existing (allocating) path
            got = nf.nf_slab_histogram_static(plan._h, pos_d, cpd)
            assert got == ref, f"cpd {cpd} call {call}"
            assert sum(got) == n
            if cpd <= 63:                                                            # and both are the oracle's cell rule
                b = oracle_mod.bin_particles(pos.numpy(), cpd, L)
                assert got == np.bincount((b["cid"] // (cpd * cpd)).astype(np.int64), minlength=cpd).tolist()
        assert nf.nf_slab_histogram_static(plan._h, torch.empty((0, 3), device="cuda"), cpd) == [0] * cpd


def test_static_scratch_limit_and_errors():
    import paper_2110_11398_b200 as nf
    B = nf.binding
    pos = torch.rand((1000, 3), device="cuda")
    with nf.Plan(1025, 1.0, 1e-5, 2) as plan:                                        # one slab more than the static array holds
        plan._use_current_stream()
        with pytest.raises(nf.NFError) as e:
            nf.nf_slab_histogram_static(plan._h, pos, 1025)
        assert e.value.code == B.NF_ERR_ARG and "1024" in str(e.value)
        assert sum(nf.nf_slab_histogram(plan._h, pos, 1025)) == 1000                 # the allocating path takes it
    with nf.Plan(16, 1.0, 1e-3, 2) as plan:
        plan._use_current_stream()
        bad = pos.clone()
        bad[7, 0] = float("nan")
        with pytest.raises(nf.NFError) as e:
            nf.nf_slab_histogram_static(plan._h, bad, 16)
        assert e.value.code == B.NF_ERR_DOMAIN
        # the flag of the failed call does not leak into the next one
        assert nf.nf_slab_histogram_static(plan._h, pos, 16) == nf.nf_slab_histogram(plan._h, pos, 16)
