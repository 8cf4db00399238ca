"""Shared test helpers: build an oracle Problem (and, on the GPU side, a library context) from a workload dict."""
import numpy as np


def oracle_problem(cfg, ref):
    from oracle.rhs import Problem
    return Problem(cfg["dim"], cfg["N"], cfg["X0"], cfg["EToV"], cfg.get("vertex_equiv"), cfg.get("EToB"),
                   cfg.get("pml_sigma"), RT=cfg["RT"], tau=cfg["tau"], q_inf=cfg.get("q_inf"),
                   motion_kind=cfg["motion_kind"], motion_params=cfg["motion_params"], ref=ref)


def rel_linf(a, b):
    """DESIGN.md R15: max |a-b| over everything, divided by max |b| over the whole state."""
    return float(np.abs(a - b).max() / np.abs(b).max())
