"""Writes tests/golden/oracle_fingerprints.txt: a few numbers of the ORACLE's own output on small seeded cases.

    python tests/golden/make_oracle_fingerprints.py

Calls only oracle/ and workloads/ (never the CUDA path).  The file is not a pin of the oracle against the paper (the
pins are tests/test_oracle_*.py); it is a tripwire: tests/test_oracle_fingerprints.py fails if a later change alters
the oracle's arithmetic, so that such a change has to be made knowingly (re-run this script and say in the commit
message which passage of PAPER.md or which DESIGN.md reading justifies it).
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import coords, forces, sark                      # noqa: E402
from oracle.operators import ReferenceElement                # noqa: E402
from oracle.rhs import Problem                               # noqa: E402
from workloads import configs                                # noqa: E402


def cases():
    """name -> (Problem factory arguments, cfg)."""
    r23, r33, r24 = ReferenceElement(2, 3), ReferenceElement(3, 3), ReferenceElement(2, 4)
    out = []
    for name, ref, cfg in (("cfg1_n4", r23, configs.config1(r23.lam, n=4)),
                           ("cfg4_n3_N3", r33, None),
                           ("cfg3_small", r24, configs.config3(r24.lam, ntheta=24, nr=8))):
        if cfg is None:
            cfg = configs.config4(r33.lam, n=3)
            cfg["N"] = 3
            cfg = configs._finish(cfg, r33.lam)
        out.append((name, ref, cfg))
    return out


def fingerprints():
    rows = []
    for name, ref, cfg in cases():
        rng = np.random.default_rng(199)
        q = cfg["q0"] * (1.0 + 1e-3 * rng.standard_normal(cfg["q0"].shape))
        for relax in ("collocation", "cubature"):
            P = Problem(cfg["dim"], cfg["N"], cfg["X0"], cfg["EToV"], cfg.get("vertex_equiv"), cfg.get("EToB"),
                        cfg.get("pml_sigma"), RT=cfg["RT"], tau=cfg["tau"], q_inf=cfg.get("q_inf"),
                        motion_kind=cfg["motion_kind"], motion_params=cfg["motion_params"], ref=ref, relax=relax)
            F = P.rhs(q, 0.21)
            F = F[0] if isinstance(F, tuple) else F
            w = np.cos(np.arange(F.size) * 0.37).reshape(F.shape)          # a fixed functional of the whole array
            rows.append((name, relax, "rhs", float((w * F).sum()), float(np.abs(F).max())))
            st, _ = sark.step_debug(P, q, 0.1, cfg["dt"])
            rows.append((name, relax, "step", float((w * st[-1]).sum()), float(np.abs(st[-1] - q).max())))
        P = Problem(cfg["dim"], cfg["N"], cfg["X0"], cfg["EToV"], cfg.get("vertex_equiv"), cfg.get("EToB"),
                    cfg.get("pml_sigma"), RT=cfg["RT"], tau=cfg["tau"], q_inf=cfg.get("q_inf"),
                    motion_kind=cfg["motion_kind"], motion_params=cfg["motion_params"], ref=ref)
        st, _, x1 = coords.step_debug(P, q, P.X0.copy(), 0.0, cfg["dt"])
        w = np.cos(np.arange(q.size) * 0.37).reshape(q.shape)
        rows.append((name, "collocation", "rk_coords", float((w * st[-1]).sum()), float(np.abs(x1 - P.X0).max())))
        Fp, Fv = forces.wall_force(P, q, 0.3)
        rows.append((name, "collocation", "wall_force", float(Fp.sum()), float(Fv.sum())))
    return rows


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_fingerprints.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_oracle_fingerprints.py from oracle/ only (no paper values, no CUDA values)\n")
        f.write("# case relax quantity value_a value_b\n")
        for name, relax, what, a, b in fingerprints():
            f.write("%s %s %s %.17e %.17e\n" % (name, relax, what, a, b))
    print(path)
