"""Host logic of the CUDA library, checked without a GPU (-m "not gpu").

  * libalegb.so loads and exports every symbol include/alegb.h declares
  * its reference element (built from a monomial basis in __float128) against the oracle's (Legendre + quadrature)
  * its face / node matching against the oracle's on every workload shape
  * mesh validation (BAD_MESH cases of SURVEY S4), argument validation
  * its SARK coefficients against tests/golden/sark_coefficients.txt (PAPER.md:L148 in 50-digit arithmetic)
  * no compute without a device: a host-only context fails loudly, there is no CPU fallback
"""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import mesh as omesh
from oracle import sark as osark
from workloads import configs, meshes

B = pytest.importorskip("paper_2607_00199_b200.binding")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "alegb.h")).read()
    declared = set(re.findall(r"\b(alegb_[a-z0-9_]+)\s*\(", header))
    assert len(declared) >= 20
    lib = ctypes.CDLL(B.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), "libalegb.so does not export %s" % name
    assert declared == set(B.EXPORTED), declared ^ set(B.EXPORTED)


@pytest.mark.parametrize("dim,N", [(d, n) for d in (2, 3) for n in (1, 2, 3, 4, 5)])
def test_reference_element_matches_oracle(dim, N, refs):
    ref = refs(dim, N)
    ctx = B.Context(dim, N, -1)
    assert (ctx.Np, ctx.Nfp, ctx.Nfaces, ctx.Nf) == (ref.Np, ref.Nfp, ref.Nfaces, 6 if dim == 2 else 10)
    ops, rr = ctx.alegb_get_operators(), ctx.alegb_get_reference()
    assert np.array_equal(rr["fmask"], ref.fmask)
    assert np.abs(rr["lam"] - ref.lam).max() < 5e-16
    for name, a in zip(("r", "s", "t"), range(dim)):
        assert np.abs(ops[name] - ref.x[:, a]).max() < 1e-15
    scale = max(np.abs(D).max() for D in ref.D)
    for name, a in zip(("Dr", "Ds", "Dt"), range(dim)):
        assert np.abs(ops[name] - ref.D[a]).max() < 2e-14 * scale
    assert np.abs(ops["LIFT"] - ref.LIFT).max() < 2e-14 * np.abs(ref.LIFT).max()
    assert np.abs(rr["w"] - ref.w).max() < 5e-15
    ctx.close()


@pytest.mark.parametrize("dim,N", [(2, 3), (2, 4), (3, 3), (3, 4)])
def test_library_operators_differentiate_and_lift_exactly(dim, N):
    """Pins the library's own matrices to the mathematics, not only to the oracle: D is exact on P_N, and
    J w^T LIFT(Fscale g) = sJ int_refface g with face weights summing to the reference face measure 2."""
    ctx = B.Context(dim, N, -1)
    ops, rr = ctx.alegb_get_operators(), ctx.alegb_get_reference()
    x = [ops["r"], ops["s"]] + ([ops["t"]] if dim == 3 else [])
    rng = np.random.default_rng(3)
    for _ in range(5):
        e = rng.integers(0, N + 1, size=dim)
        while e.sum() > N:
            e = rng.integers(0, N + 1, size=dim)
        p = np.prod([x[d] ** e[d] for d in range(dim)], axis=0)
        for a, name in enumerate(("Dr", "Ds", "Dt")[:dim]):
            ea = e.copy()
            if ea[a] == 0:
                exact = np.zeros_like(p)
            else:
                ea[a] -= 1
                exact = e[a] * np.prod([x[d] ** ea[d] for d in range(dim)], axis=0)
            assert np.abs(ops[name] @ p - exact).max() < 1e-12
    wl = rr["w"] @ ops["LIFT"]                       # face quadrature weights of each face
    for f in range(dim + 1):
        assert abs(wl[f * ctx.Nfp:(f + 1) * ctx.Nfp].sum() - 2.0) < 1e-13
    assert abs(rr["w"].sum() - (2.0 if dim == 2 else 4.0 / 3.0)) < 1e-14
    ctx.close()


def _cases():
    yield "cfg1", configs.config1(None)
    yield "cfg2", configs.config2(None, n=9)
    yield "cfg3", configs.config3(None, ntheta=16, nr=5)
    yield "cfg4", configs.config4(None, n=3)
    yield "cfg5", configs.config5(None, nx=8, ny=5, nz=5)


@pytest.mark.parametrize("name,cfg", list(_cases()), ids=[n for n, _ in _cases()])
def test_connectivity_matches_oracle(name, cfg, refs):
    ref = refs(cfg["dim"], cfg["N"])
    conn = omesh.connect(ref, cfg["EToV"], cfg.get("vertex_equiv"), cfg.get("EToB"))
    ctx = B.Context(cfg["dim"], cfg["N"], -1)
    ctx.alegb_mesh_upload(cfg["X0"], cfg["EToV"], cfg.get("vertex_equiv"), cfg.get("EToB"), cfg.get("pml_sigma"))
    ops = ctx.alegb_get_operators(with_maps=True)
    assert np.array_equal(ops["vmapM"], conn["vmapM"])
    assert np.array_equal(ops["vmapP"], conn["vmapP"])
    if cfg.get("pml_sigma") is not None:
        expect = np.nonzero(np.any(cfg["pml_sigma"] > 0, axis=1))[0]
        assert np.array_equal(ctx.alegb_pml_elements(), expect)
    ctx.close()


def test_bad_meshes_are_rejected():
    ctx = B.Context(2, 2, -1)
    X0, EToV, eq = meshes.periodic_square(2, 0.0, 1.0)          # periodic direction with 2 cells (S4)
    with pytest.raises(B.AlegbError) as e:
        ctx.alegb_mesh_upload(X0, EToV, eq)
    assert e.value.status == B.BAD_MESH
    X0, EToV, eq = meshes.periodic_square(3, 0.0, 1.0)
    with pytest.raises(B.AlegbError) as e:                      # boundary faces without tags
        ctx.alegb_mesh_upload(X0, EToV, None)
    assert e.value.status == B.BAD_MESH
    flipped = EToV.copy()
    flipped[0] = flipped[0][[0, 2, 1]]                          # negative Jacobian (L73)
    with pytest.raises(B.AlegbError) as e:
        ctx.alegb_mesh_upload(X0, flipped, eq)
    assert e.value.status == B.BAD_MESH and "Jacobian" in str(e.value)
    tags = np.ones((EToV.shape[0], 3), dtype=np.int8)           # a tag on an interior face
    with pytest.raises(B.AlegbError) as e:
        ctx.alegb_mesh_upload(X0, EToV, eq, tags)
    assert e.value.status == B.BAD_MESH
    bad = EToV.copy()
    bad[1, 1] = 10 ** 6
    with pytest.raises(B.AlegbError) as e:
        ctx.alegb_mesh_upload(X0, bad, eq)
    assert e.value.status == B.BAD_MESH
    ctx.alegb_mesh_upload(X0, EToV, eq)                         # and the good one passes
    assert ctx.K == 18
    ctx.close()


def test_argument_validation():
    with pytest.raises(B.AlegbError) as e:
        B.Context(4, 2, -1)
    assert e.value.status == B.INVALID_ARG
    with pytest.raises(B.AlegbError) as e:
        B.Context(3, 9, -1)
    assert e.value.status == B.UNSUPPORTED
    ctx = B.Context(2, 3, -1)
    with pytest.raises(B.AlegbError):
        ctx.alegb_set_params(-1.0, 1.0)
    with pytest.raises(B.AlegbError):
        ctx.alegb_set_motion(B.MOTION_SINES_PRODUCT, [0.1, 1.0])          # too few parameters
    with pytest.raises(B.AlegbError):
        ctx.alegb_set_motion(B.MOTION_PLUNGE_BLEND, [0.1, 1.0, 1.0, 2.0, 5.0, 0.0, 0.0])   # axis out of range
    with pytest.raises(B.AlegbError):
        ctx.alegb_set_motion(17, [])
    ctx.alegb_set_motion(B.MOTION_SINES_PRODUCT, [0.1, 1.0, 1.0, 1.0, 0.0, 0.0])
    for call in (lambda: ctx.alegb_set_relaxation(7), lambda: ctx.alegb_set_coordinate_mode(-1, 0.0)):
        with pytest.raises(B.AlegbError) as e:
            call()
        assert e.value.status == B.INVALID_ARG
    ctx.alegb_set_relaxation(B.RELAX_COLLOCATION)        # the default modes need no device
    ctx.alegb_set_coordinate_mode(B.COORDS_CLOSED_FORM, 0.0)
    ctx.alegb_set_geometry_overlap(False)
    ctx.close()


def test_no_cpu_fallback():
    """A context without a device must refuse every compute call (ALEGB_CUDA_ERROR), never compute on the host."""
    cfg = configs.config1(None)
    ctx = B.Context(2, 3, -1)
    ctx.alegb_mesh_upload(cfg["X0"], cfg["EToV"], cfg["vertex_equiv"])
    ctx.alegb_set_params(1.0, 1e-3)
    for call in (lambda: ctx.alegb_rhs(0.0, 16, 16, stream=0), lambda: ctx.alegb_step(16, 0.0, 1e-3, 1, stream=0),
                 lambda: ctx.alegb_geometry(0.0, stream=0), lambda: ctx.alegb_step_host(np.zeros(8), 0.0, 1e-3, 1),
                 lambda: ctx.alegb_profile_read(),
                 # the optional modes and the diagnostics have no host path either
                 lambda: ctx.alegb_set_relaxation(B.RELAX_CUBATURE), lambda: ctx.alegb_set_coordinate_mode(B.COORDS_RK, 0.0),
                 lambda: ctx.alegb_get_positions(16, stream=0), lambda: ctx.alegb_wall_forces(0.0, 16, 1, stream=0),
                 lambda: ctx.alegb_wall_forces_static(0.0, 16, 16, stream=0), lambda: ctx.alegb_measure_fp64_peak()):
        with pytest.raises(B.AlegbError) as e:
            call()
        assert e.value.status == B.CUDA_ERROR
    ctx.close()


def test_product_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_00199_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) in ("build", "__pycache__"):
            continue
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, re.M), fn
                assert "_work/" not in text, fn


# ------------------------------------------------------------------ SARK coefficients (R4-R6)
def _golden():
    rows = []
    for line in open(os.path.join(ROOT, "tests", "golden", "sark_coefficients.txt")):
        if line.strip() and not line.startswith("#"):
            rows.append([float(v) for v in line.split()])
    return rows


def test_sark_coefficients_against_golden():
    for g, a10, a20, a21, a30, a32, b0, b1, b3 in _golden():
        a, b = B.alegb_sark_coefficients(g)
        got = np.array([a[0], a[1], a[2], a[3], a[5], b[0], b[1], b[2], b[3]])
        want = np.array([a10, a20, a21, a30, a32, b0, b1, b1, b3])
        assert np.abs(got / want - 1.0).max() < 4e-16, (g, got, want)
        assert a[4] == 0.0


@pytest.mark.parametrize("gamma", [0.0, -1e-12, -1e-6, -1e-3, -0.04, -0.5, -0.999, -1.0, -1.999, -2.0, -2.5, -37.0, -1e3])
def test_sark_coefficients_against_oracle_and_identities(gamma):
    a, b = B.alegb_sark_coefficients(gamma)
    ao, bo = osark.coefficients(gamma)
    want = np.array([ao[1][0], ao[2][0], ao[2][1], ao[3][0], ao[3][1], ao[3][2]])
    assert np.abs(a - want).max() <= 4e-16 * np.abs(want).max()
    assert np.abs(b - np.array(bo)).max() <= 4e-16 * np.abs(bo).max()
    if gamma != 0.0:                                             # eq. 14 without the spurious 1/c_i (R5)
        phi = lambda z: np.expm1(z) / z
        assert abs(a[0] - 0.5 * phi(gamma / 2)) < 1e-15
        assert abs(a[1] + a[2] - 0.5 * phi(gamma / 2)) < 1e-15
        assert abs(a[3] + a[5] - phi(gamma)) < 1e-15
        assert abs(b.sum() - phi(gamma)) < 1e-15
    else:
        assert list(a) == [0.5, 0.0, 0.5, 0.0, 0.0, 1.0] and np.allclose(b, [1 / 6, 1 / 3, 1 / 3, 1 / 6], atol=0, rtol=1e-16)


@pytest.mark.parametrize("dim,N", [(2, 1), (2, 3), (2, 4), (2, 5), (3, 2), (3, 3), (3, 4), (3, 5)])
def test_cubature_matches_oracle_and_integrates_exactly(dim, N, refs):
    """NEXT-1: the library's own Gauss-Jacobi rule, I and P (host_ref.cpp, __float128, monomial
    basis) against the oracle's (scipy roots, product-Legendre basis), and against Dirichlet's closed-form integrals."""
    from math import factorial
    from oracle.cubature import Cubature
    from paper_2607_00199_b200 import binding as B
    ctx = B.Context(dim, N, -1)
    got = ctx.alegb_get_cubature()
    ref = refs(dim, N)
    cub = Cubature(ref)
    assert got["degree"] == 3 * N and got["Nc"] == cub.Nc
    # the two rules may order their points differently: sort both lexicographically
    def order(x):
        return np.lexsort(np.round(x.T[::-1], 12))
    og, oo = order(got["rst"].T), order(cub.x)
    assert np.abs(got["rst"].T[og] - cub.x[oo]).max() < 1e-14
    assert np.abs(got["w"][og] - cub.w[oo]).max() < 1e-15
    assert np.abs(got["I"][og] - cub.I[oo]).max() < 1e-12
    assert np.abs(got["P"][:, og] - cub.P[:, oo]).max() < 1e-12
    # closed form: sum_c w_c prod ((1+x_d)/2)^e_d = 2^dim prod e_d! / (sum e + dim)!
    x, w = got["rst"].T, got["w"]
    rng = np.random.default_rng(199)
    for _ in range(20):
        e = rng.multinomial(3 * N, np.ones(dim + 1) / (dim + 1))[:dim]
        exact = 2.0 ** dim * np.prod([factorial(int(v)) for v in e]) / factorial(int(e.sum()) + dim)
        assert abs(w @ np.prod(((1 + x) / 2) ** e, axis=1) - exact) < 1e-15
    ctx.close()
