"""Test-side assembly of the data streams: noise from sc_synth + injections from the ORACLE's template.
(No oracle input ever comes from the CUDA path.)"""
import numpy as np

import sc_synth as sy


def make_data(oracle, inp):
    """d_alpha = sum_i kappa_i h_alpha(theta_i) + n_alpha, kappa = rho / sqrt(<h|h>)  (O6, Eq. 3)."""
    cfg = oracle.make_config(inp["cfg"])
    dA, dE = inp["noise_A"].copy(), inp["noise_E"].copy()
    for inj in inp["injections"]:
        hA, hE, _ = oracle.template(cfg, inj["theta"])
        rho2 = oracle.inner(hA, hE, hA, hE, inp["S_A"], inp["S_E"], inp["df"])
        kappa = inj["rho"] / np.sqrt(rho2)
        dA += kappa * hA
        dE += kappa * hE
    return cfg, dA, dE


def gpu_handle(inp, dA, dE):
    import torch
    import paper_2408_13170_b200 as sc
    dev = torch.device("cuda:0")
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    return sc.Handle(inp["cfg"], torch.view_as_real(t(dA)).contiguous(), torch.view_as_real(t(dE)).contiguous(),
                     t(inp["S_A"]), t(inp["S_E"]))


def rel_err(got, want):
    got, want = np.asarray(got), np.asarray(want)
    return np.abs(got - want) / np.maximum(np.abs(want), 1e-300)
