"""GPU parity of the fp32 k-RHS per-frequency GEMMs on tcgen05 (paper_2501_14911_b200/csrc/tt_gemm32_umma.cu), called
through the C ABI (tt_matvec_batched / tt_rmatvec_batched of a TT_F32 plan), against the CPU oracle column by column.

The shapes walk the kernels' own structure: one and several 64-sensor tiles (forward), 1..8 sensor K-blocks and an
even / odd number of raw stages (adjoint; N_d = 100 and 112 are the shapes whose shared-memory budget leaves an odd count,
which once let a second set of transform warps reach a stage one mbarrier phase early), ragged parameter tiles, several
parameter tiles per CTA, k = 16 / 32 / 48 / 64 (16- and 32-column launches), both layouts.  Bar: 1e-5 (BASELINE.json).
"""
import numpy as np
import pytest
import torch

from oracle import toeplitz_blocked as ob
import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tt():
    from paper_2501_14911_b200 import binding
    binding.lib()
    return binding


def rel(a, b):
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (nb if nb > 0 else 1.0)


def run_pair(tt, N_d, N_m, N_t, k, layout=0, umma=1):
    w = synth.CONFIGS["C4"].scaled(N_d=N_d, N_m=N_m, N_t=N_t, dtype=torch.float32)
    F = synth.block_column(w)
    M = synth.vector_m(w, k_rhs=k)
    D = synth.vector_d(w, k_rhs=k)
    lay = (lambda t: t.permute(2, 1, 0).contiguous()) if layout == 1 else (lambda t: t)
    unlay = (lambda t: t.permute(2, 1, 0)) if layout == 1 else (lambda t: t)
    tt.tt_debug_set("gemm32_umma", umma)
    plan = tt.Plan(F.cuda(), layout=layout, k_max=k)
    try:
        gd = unlay(plan.matvec_batched(lay(M).cuda())).cpu().numpy()
        gm = unlay(plan.rmatvec_batched(lay(D).cuda())).cpu().numpy()
    finally:
        plan.close()
        tt.tt_debug_set("gemm32_umma", 1)
    return F, M, D, gd, gm


SHAPES = [(49, 2049, 20, 32), (64, 8192, 12, 32), (100, 5000, 16, 32), (112, 16384, 6, 32), (128, 9000, 10, 16),
          (16, 3001, 10, 32), (3, 31, 6, 32), (65, 4100, 8, 16), (100, 16384, 6, 48), (70, 4100, 12, 64), (130, 4500, 12, 64)]


@pytest.mark.parametrize("N_d,N_m,N_t,k", SHAPES)
def test_tensor_core_gemms_equal_oracle(tt, N_d, N_m, N_t, k):
    F, M, D, gd, gm = run_pair(tt, N_d, N_m, N_t, k)
    for r in sorted({0, 1, k // 2, k - 1}):
        assert rel(gd[..., r], ob.matvec(F.numpy(), M[..., r].contiguous().numpy())) <= 1e-5
        assert rel(gm[..., r], ob.rmatvec(F.numpy(), D[..., r].contiguous().numpy())) <= 1e-5


def test_space_major_layout_takes_the_same_path(tt):
    F, M, D, gd, gm = run_pair(tt, 49, 2049, 20, 32, layout=1)
    for r in (0, 31):
        assert rel(gd[..., r], ob.matvec(F.numpy(), M[..., r].contiguous().numpy())) <= 1e-5
        assert rel(gm[..., r], ob.rmatvec(F.numpy(), D[..., r].contiguous().numpy())) <= 1e-5


@pytest.mark.parametrize("N_d,N_m,N_t,k", [(49, 6000, 12, 32), (100, 16384, 6, 32), (64, 4096, 10, 16)])
def test_tensor_core_and_fma_kernels_agree_in_every_element(tt, N_d, N_m, N_t, k):
    """Both kernel families compute the same fp32 products: every output element of one within a few fp32 roundings (relative
    to the largest element) of the other - a wrong tile, row or column anywhere would show, not only a wrong norm."""
    _, _, _, gd1, gm1 = run_pair(tt, N_d, N_m, N_t, k, umma=1)
    _, _, _, gd0, gm0 = run_pair(tt, N_d, N_m, N_t, k, umma=0)
    assert np.abs(gd1 - gd0).max() <= 2e-5 * np.abs(gd0).max()
    assert np.abs(gm1 - gm0).max() <= 2e-5 * np.abs(gm0).max()


def test_repeated_runs_are_bit_identical(tt):
    """The pipelines hand tiles between TMA, transform warps, the MMA and the epilogue through mbarriers: a missed dependency
    shows as run-to-run differences (as it did, at N_d = 100, before every raw stage belonged to one set of transform warps)."""
    first = None
    for _ in range(6):
        _, _, _, gd, gm = run_pair(tt, 100, 16384, 6, 32)
        if first is None:
            first = (gd.copy(), gm.copy())
        else:
            assert np.array_equal(first[0], gd) and np.array_equal(first[1], gm)
