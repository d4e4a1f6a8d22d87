"""Inputs of the online-phase tests that are defined by the paper rather than drawn: the block column of G*.

G_k = F_k Gamma_s is formed by the ORACLE (oracle/online_plain.gstar_block_column) from the seeded F and
the seeded prior weights, rounded once to the workload's dtype, and the very same array is handed to both sides - the
oracle's formula is therefore on the GPU-parity path of every online test.  (At full size the tests and bench.py draw the
array on the device with synth.scaled_block_column, which tests/test_synth.py holds to this function bit for bit.)
"""
import torch

import synth


def gstar_column(w, F: torch.Tensor) -> torch.Tensor:
    from oracle import online_plain as oo
    g = synth.prior_gamma(w).numpy()
    return torch.from_numpy(oo.gstar_block_column(F.cpu().numpy(), g[: F.shape[2]])).to(w.dtype)
