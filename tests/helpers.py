"""Shared test helpers (no method arithmetic)."""
import numpy as np
from oracle.nsc_oracle import Params, Oracle
from paper_1908_00587_b200 import synth


def params_of(cfg: dict, **over) -> Params:
    d = {k: cfg[k] for k in synth.PHYS_KEYS}
    d.update(over)
    return Params(**d)


def oracle_of(cfg: dict, dft="naive", solve="dense", real=np.float64, **over) -> Oracle:
    return Oracle(params_of(cfg, **over), dft=dft, solve=solve, real=real)


def nf_of(cfg):
    return 4 if cfg["Ra"] != 0.0 else 3
