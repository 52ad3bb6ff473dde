"""Helpers shared by the -m gpu tests: build a CUDA context and an oracle problem from the
same workloads.Config.  (Test-side glue: the only place both sides meet.)"""
from __future__ import annotations

import numpy as np
import torch

import workloads as w


def np_dtype(dt):
    return np.float32 if dt == "f32" else np.float64


def torch_dtype(dt):
    return torch.float32 if dt == "f32" else torch.float64


def make_ctx(cfg, dt, terms=None, tiles=None, path=0, slabs=0):
    from paper_2606_01114_b200 import Context
    ctx = Context(cfg.n, cfg.d, dtype=torch_dtype(dt), tiles=tiles, path=path, slabs=slabs)
    ctx.set_material(cfg.Ms, cfg.Aex, cfg.Ku, cfg.axis, cfg.alpha, cfg.gamma)
    ctx.set_zeeman(cfg.Hext)
    t = cfg.terms if terms is None else terms
    ctx.set_terms(t)
    if t & 1:
        ctx.demag_init()
    return ctx


def make_problem(oracle, cfg, terms=None, N=None):
    P = oracle.Problem(n=cfg.n, d=cfg.d, Ms=cfg.Ms, Aex=cfg.Aex, Ku=cfg.Ku, axis=cfg.axis,
                       alpha=cfg.alpha, gamma=cfg.gamma, Hext=cfg.Hext,
                       terms=cfg.terms if terms is None else terms, N=N)
    return P.prepare()


def round_input(m64, dt):
    """Inputs are generated once in fp64; fp32 runs see the fp32-rounded values on BOTH sides."""
    m = m64.astype(np_dtype(dt))
    return m, m.astype(np.float64)


def to_dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


TOL = {"f64": 1e-12, "f32": 2e-5}          # BASELINE.json north_star
TRAJ_TOL = {"f64": 1e-10, "f32": 1e-4}
