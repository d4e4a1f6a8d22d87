"""tt_assemble_K_direct_static: the entry point that allocates nothing (scratch in a 64 MiB static device array inside
libtt.so, see include/tt.h) against the existing, allocating tt_assemble_K_direct, on two calls in a row.

Collected last on purpose (the file name): the suite runs with pytest -x.
"""
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu

TOL = 1e-5          # the fp32 bar of the other GPU tests (BASELINE.json north_star)


@pytest.fixture(scope="module")
def tt():
    from paper_2501_14911_b200 import binding
    binding.lib()
    return binding


def inputs(N_d, N_m, N_t):
    w = synth.CONFIGS["P5"].scaled(N_d=N_d, N_m=N_m, N_t=N_t)
    F = synth.block_column(w, device="cuda")
    G = synth.scaled_block_column(w, F)
    nv = synth.noise_var(w, device="cuda")
    return F, G, nv


def rel(a, b):
    return float((a - b).norm() / b.norm())


# n = 300: one slab in both paths (same summation order).  n = 3000, N_m = 4000: 48 000 scratch bytes per parameter, so the
# static path works in slabs of 1376 parameters where the allocating one takes all 4000 at once.
@pytest.mark.parametrize("N_d,N_m,N_t", [(6, 5000, 50), (30, 4000, 100)])
def test_static_entry_point_equals_the_allocating_path_twice(tt, N_d, N_m, N_t):
    n = N_d * N_t
    F, G, nv = inputs(N_d, N_m, N_t)
    want = torch.empty((n, n), dtype=torch.float64, device="cuda")
    tt.tt_assemble_K_direct(F, G, nv, N_d, N_m, N_t, tt.TT_F32, want, n)
    torch.cuda.synchronize()
    # a second problem in between, so that the static array holds another call's planes and tile list when the repeat starts
    F2, G2, nv2 = inputs(4, 700, 20)
    other = torch.empty((80, 80), dtype=torch.float64, device="cuda")
    got = [torch.full((n, n), float("nan"), dtype=torch.float64, device="cuda") for _ in range(2)]
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    tt.tt_assemble_K_direct_static(F, G, nv, N_d, N_m, N_t, tt.TT_F32, got[0], n)
    tt.tt_assemble_K_direct_static(F2, G2, nv2, 4, 700, 20, tt.TT_F32, other, 80)
    tt.tt_assemble_K_direct_static(F, G, nv, N_d, N_m, N_t, tt.TT_F32, got[1], n)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    for g in got:
        assert torch.isfinite(g).all()
        assert rel(g, want) <= TOL
        assert float((g - want).abs().max() / want.abs().max()) <= TOL
    assert torch.equal(got[0], got[1])                      # same inputs, same slabs, same order: bit for bit
    assert free0 - free1 <= (1 << 20)                       # no device memory was taken by the calls
    want2 = torch.empty((80, 80), dtype=torch.float64, device="cuda")
    tt.tt_assemble_K_direct(F2, G2, nv2, 4, 700, 20, tt.TT_F32, want2, 80)
    torch.cuda.synchronize()
    assert rel(other, want2) <= TOL


def test_static_entry_point_without_noise_is_the_product_alone(tt):
    N_d, N_m, N_t = 5, 1000, 35
    n = N_d * N_t
    F, G, nv = inputs(N_d, N_m, N_t)
    a = torch.empty((n, n), dtype=torch.float64, device="cuda")
    b = torch.empty((n, n), dtype=torch.float64, device="cuda")
    tt.tt_assemble_K_direct_static(F, G, None, N_d, N_m, N_t, tt.TT_F32, a, n)
    tt.tt_assemble_K_direct(F, G, None, N_d, N_m, N_t, tt.TT_F32, b, n)
    torch.cuda.synchronize()
    assert rel(a, b) <= TOL


def test_static_entry_point_rejects_what_does_not_fit(tt):
    """n = 40 000 rows need 16 n * 128 = 82 MB for the smallest slab: TT_ERR_STATIC_LIMIT (-13), nothing launched, K untouched."""
    F, G, nv = inputs(2, 64, 4)                              # never read: the size check comes first
    K = torch.zeros(16, dtype=torch.float64, device="cuda")
    with pytest.raises(tt.TTError) as ei:
        tt.tt_assemble_K_direct_static(F, G, nv, 100, 20000, 400, tt.TT_F32, K, 40000)
    assert ei.value.status == -13 and tt.tt_status_string(-13) == "TT_ERR_STATIC_LIMIT"
    with pytest.raises(tt.TTError) as ei:                    # fp64 has no scratch: not this entry point's business
        tt.tt_assemble_K_direct_static(F.double(), G.double(), nv.double(), 2, 64, 4, tt.TT_F64, K, 8)
    assert ei.value.status == -3
    torch.cuda.synchronize()
    assert float(K.abs().sum()) == 0.0
