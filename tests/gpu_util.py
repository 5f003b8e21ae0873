"""Helpers for the -m gpu parity tests: move a TInputs to the device."""
import numpy as np
import torch


def to_device(inp, device="cuda:0"):
    return [torch.from_numpy(np.ascontiguousarray(a)).to(device) for a in inp.arrays()]


def dims(inp):
    return inp.nocc, inp.nvir, inp.naux


# north_star tolerance: |dE| <= 1e-10 |E| + 1e-12 Eh
def e_tol(e):
    return 1e-10 * abs(e) + 1e-12
