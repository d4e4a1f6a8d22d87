"""The seeded input generators (harness): deterministic, sliceable, with the stated envelopes."""
import math

import numpy as np
import torch

import synth


def test_configs_match_baseline_json_shapes():
    c = synth.CONFIGS
    assert (c["C1"].N_d, c["C1"].N_m, c["C1"].N_t, c["C1"].seed) == (4, 64, 32, 0)
    assert (c["C2"].N_d, c["C2"].N_m, c["C2"].N_t, c["C2"].seed) == (64, 16384, 256, 1)
    assert (c["C3"].N_d, c["C3"].N_m, c["C3"].N_t, c["C3"].seed) == (100, 250000, 400, 2)
    assert (c["C4"].N_d, c["C4"].N_m, c["C4"].N_t, c["C4"].k_rhs) == (64, 65536, 512, 32)
    assert (c["C5"].N_d, c["C5"].N_m, c["C5"].N_t, c["C5"].seed) == (200, 100000, 400, 4)
    assert c["C3"].n_params == 100_000_000          # "about 1e8 params"
    assert c["C3"].dtype == torch.float32 and c["C2"].dtype == torch.float64


def test_deterministic_and_sliceable():
    w = synth.CONFIGS["C3"].scaled(N_d=5, N_m=300, N_t=6)
    F = synth.block_column(w)
    assert F.shape == (6, 5, 300) and F.dtype == torch.float32
    assert torch.equal(F, synth.block_column(w))
    sl = synth.block_column(w, k_range=(1, 4), s_range=(2, 3), p_range=(17, 200))
    assert torch.equal(sl, F[1:4, 2:3, 17:200])
    assert torch.equal(synth.block_column(w, chunk_elems=256), F)      # chunking does not change values
    m = synth.vector_m(w)
    assert m.shape == (6, 300) and torch.equal(m, synth.vector_m(w))
    assert not torch.equal(m[:, :5], synth.vector_d(w))
    M = synth.vector_m(w, k_rhs=3)
    assert M.shape == (6, 300, 3)


def test_normal_moments_and_envelopes():
    idx = torch.arange(400_000, dtype=torch.int64)
    z = synth.normal01(7, synth.TENSOR_M, idx).numpy()
    assert abs(z.mean()) < 0.01 and abs(z.std() - 1.0) < 0.01
    assert abs(np.mean(z ** 4) - 3.0) < 0.1
    u = synth.uniform01(7, synth.TENSOR_SCALE, idx).numpy()
    assert 0.0 < u.min() and u.max() < 1.0 and abs(u.mean() - 0.5) < 0.01
    # exp(-k/tau) decay and per-sensor scale in [0.5, 2] (C2 recipe)
    w = synth.CONFIGS["C2"].scaled(N_d=6, N_m=20000, N_t=65)
    F = synth.block_column(w).numpy()
    rms = np.sqrt((F ** 2).mean(axis=2))          # [k, s]
    ratio = rms[64] / rms[0]
    assert np.allclose(ratio, math.exp(-64 / 32.0), rtol=0.05)
    assert np.all(rms[0] > 0.45) and np.all(rms[0] < 2.1)
    # Gaussian bump (C3 recipe): energy concentrated within a few sigma of the sensor's centre
    w = synth.CONFIGS["C3"].scaled(N_d=3, N_m=4000, N_t=2)
    F = synth.block_column(w).double().numpy()
    for s in range(3):
        e = F[0, s] ** 2
        mu = int(np.argmax(np.convolve(e, np.ones(201) / 201, mode="same")))
        sigma = 0.05 * 4000
        near = e[max(0, mu - int(3 * sigma)): mu + int(3 * sigma)].sum()
        assert near / e.sum() > 0.99


def test_scaled_block_column_is_the_oracles_gstar_column():
    """synth.scaled_block_column (the device-side generator of the second block column at full size) against
    oracle/online_plain.gstar_block_column (G_k = F_k Gamma_s), bit for bit in both dtypes."""
    from oracle import online_plain as oo
    for dtype in (torch.float64, torch.float32):
        w = synth.CONFIGS["P5"].scaled(N_d=3, N_m=257, N_t=5, dtype=dtype)
        F = synth.block_column(w)
        ref = torch.from_numpy(oo.gstar_block_column(F.numpy(), synth.prior_gamma(w).numpy())).to(dtype)
        assert torch.equal(synth.scaled_block_column(w, F), ref)
