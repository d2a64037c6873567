"""Helpers of the -m gpu parity tests: move a sagecal_inputs.Problem to the device and call the C ABI
(through the thin binding paper_1910_13908_b200).  No oracle code here."""
import numpy as np
import torch

import paper_1910_13908_b200 as sg


def dev(a, device="cuda:0"):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(device)


def host(t):
    return t.detach().cpu().numpy()


class per_baseline_form:
    """with per_baseline_form(): predictions use one phasor per (baseline, source) -- the arithmetic the fused RESID arm
    shares bit for bit -- instead of the station form (sagecal_predict_set_form)."""
    def __enter__(self):
        sg.predict_set_form(1)

    def __exit__(self, *exc):
        sg.predict_set_form(0)


def gpu_predict(prob, coh_format=sg.COH_FULL, precision=0, freqs=None):
    src = {k: dev(getattr(prob, k)) for k in ("src_l", "src_m", "src_I", "src_alpha", "src_Q", "src_U", "src_V")}
    return sg.predict_coherencies(prob.N, prob.T, prob.freqs if freqs is None else freqs, prob.f0, dev(prob.uvw),
                                  prob.cluster_offset, src["src_l"], src["src_m"], src["src_I"], src["src_alpha"],
                                  src["src_Q"], src["src_U"], src["src_V"], coh_format=coh_format, precision=precision)


def gpu_simulate(prob, coh_d, coh_format=sg.COH_FULL, noise=True):
    """V = sum_k J_true C_k J_true^H (+ the generator's noise), built by the CUDA path's own arithmetic."""
    vis0 = dev(prob.noise()) if noise else None
    return sg.corrupt_subtract(prob.N, prob.T, prob.F, coh_d, dev(prob.jones_true), vis0, sign=+1.0,
                               coh_format=coh_format)
