"""Shared test helpers: build an oracle Problem (and, on the GPU side, a library context) from a workload dict."""
import numpy as np

from workloads import configs, meshes


def oracle_problem(cfg, ref):
    from oracle.rhs import Problem
    return Problem(cfg["dim"], cfg["N"], cfg["X0"], cfg["EToV"], cfg.get("vertex_equiv"), cfg.get("EToB"),
                   cfg.get("pml_sigma"), RT=cfg["RT"], tau=cfg["tau"], q_inf=cfg.get("q_inf"),
                   motion_kind=cfg["motion_kind"], motion_params=cfg["motion_params"], ref=ref,
                   relax=cfg.get("relax", "collocation"))


def rel_linf(a, b):
    """DESIGN.md R15: max |a-b| over everything, divided by max |b| over the whole state."""
    return float(np.abs(a - b).max() / np.abs(b).max())


def submesh(cfg, EToE, samples, rings):
    """Workload dict restricted to ``samples`` plus ``rings`` layers of face neighbours (EToE from the oracle's
    connectivity).  Faces whose neighbour is outside the patch become far-field faces (tag 2), so the operator on
    the patch equals the full operator wherever the stencil stays inside: F on the samples needs 1 ring, stage
    state i of one SARK step needs i rings.  Returns (sub_cfg, patch_element_ids, position_of_samples_in_patch)."""
    samples = np.asarray(samples, dtype=np.int64)
    patch = np.unique(samples)
    for _ in range(rings):
        patch = np.unique(np.concatenate([patch, EToE[patch].ravel()]))
    inside = np.zeros(EToE.shape[0], dtype=bool)
    inside[patch] = True
    tags = np.where(inside[EToE[patch]], 0, 2).astype(np.int8)
    if cfg.get("EToB") is not None:
        orig = np.asarray(cfg["EToB"])[patch]
        tags = np.where(orig != 0, orig, tags).astype(np.int8)
    sub = dict(cfg)
    sub["EToV"] = np.ascontiguousarray(cfg["EToV"][patch])
    sub["EToB"] = tags
    sub["K"] = len(patch)
    if cfg.get("pml_sigma") is not None:
        sub["pml_sigma"] = np.ascontiguousarray(np.asarray(cfg["pml_sigma"])[patch])
    if cfg.get("q_inf") is None:
        sub["q_inf"] = np.zeros(cfg["Nf"])
    sub["q0"] = np.ascontiguousarray(cfg["q0"][patch])
    where = np.searchsorted(patch, samples)
    return sub, patch, where


def swimmer_small(lam, n=(12, 6, 6), lo=(-4.0, -3.0, -3.0), hi=(8.0, 3.0, 3.0)):
    """config 5 shape with a body fat enough to be resolved by a coarse grid (wall faces, far field, PML)."""
    cfg = configs.config5(lam, nx=n[0], ny=n[1], nz=n[2])
    X0, EToV, EToB, sigma = meshes.swimmer_box(n[0], n[1], n[2], half_height=1.2, half_width=1.2,
                                               lo=lo, hi=hi)
    cfg.update(X0=X0, EToV=EToV, EToB=EToB, pml_sigma=sigma)
    cfg["motion_params"] = cfg["motion_params"].copy()
    cfg["motion_params"][5] = 2.0                   # R_rigid: make the layer around the body move
    cfg["dt"] = configs.cfl_dt(3, 3, X0, EToV, cfg["RT"], 0.5, 0.2 * cfg["motion_params"][4])
    return configs._finish(cfg, lam)
