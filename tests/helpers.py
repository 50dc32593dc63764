"""Shared helpers of the GPU parity tests: build synthetic configs (coefficients of the injected point from
the ORACLE), create handles through the C-ABI binding, run the oracle on chosen samples."""
from __future__ import annotations

import numpy as np

from paper_2210_07912_b200 import synth


def oracle_geometry_fn(oracle, cfg, loc, resp, ml, mm):
    return lambda th: oracle.geometry_at(th, loc, resp, cfg.gmst, ml, mm, cfg.delta_t)


def build(oracle, cfg, n_points=None, noise=True):
    loc, resp = synth.detector_arrays(cfg)
    ml, mm = synth.mode_arrays(cfg)
    return synth.build_inputs(cfg, oracle_geometry_fn(oracle, cfg, loc, resp, ml, mm), n_points=n_points, noise=noise)


def create(binding, inp, precision, n_tau=None, points=None):
    cfg = inp.cfg
    sel = slice(None) if points is None else points
    Q, U, V = inp.Q[sel], inp.U[sel], inp.V[sel]
    return binding.rift_ile_create(inp.det_location, inp.det_response, cfg.gmst, inp.mode_l, inp.mode_m, Q.shape[0],
                                   cfg.n_t, cfg.delta_t, cfg.n_t if n_tau is None else n_tau, synth.D_REF_MPC, Q, U, V,
                                   precision=precision)


def oracle_eval(oracle, inp, point, params, n_tau=None):
    cfg = inp.cfg
    return oracle.eval_batch(inp.det_location, inp.det_response, cfg.gmst, inp.mode_l, inp.mode_m, cfg.delta_t,
                             synth.D_REF_MPC, inp.Q[point], inp.U[point], inp.V[point], params, n_tau=n_tau)


def rel_err(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return np.abs(a - b) / np.maximum(1.0, np.abs(b))
