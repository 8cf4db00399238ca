"""alegb_wall_forces_static: the wall-force integrals for callers that cannot allocate device memory.

Why the entry point exists.  Drag and lift are read every time step, so the call sits inside the
time loop.  alegb_wall_forces cudaMallocs its buffer of per-block partial sums the first time it runs, which is then
the middle of that loop.  An application that has handed the rest of the HBM to its own pool by then (a framework's
caching allocator, a solver's arena) gets out-of-memory from that cudaMalloc, and a loop that keeps several streams
busy pays a device-wide stall for it.  alegb_wall_forces_static keeps the partial sums in a fixed array inside the
library image (1024 blocks x 6 doubles = 48 KiB per GPU) and leaves the result in the caller's device buffer.

What is checked here, against the existing path (alegb_wall_forces) on the same inputs and with the tolerance of
test_wall_forces_match_oracle: two calls in a row with different states and times (the array is shared and keeps the
previous call's contents, which must not leak into the next result), two calls queued on one stream with no host
synchronisation between them, other grid sizes up to the limit, a mesh without tagged faces, and the rejection of a
grid that does not fit the array.  The static entry point is called BEFORE the existing one, so that in a fresh
process its once-per-device set-up (cudaGetSymbolAddress) is what runs first.

This file is named so that pytest collects it last: pytest -x stops at the first failure, and a failure here must
not hide the parity tests.
"""
import os
import re

import numpy as np
import pytest

from workloads import configs
from helpers import oracle_problem, swimmer_small

torch = pytest.importorskip("torch")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
MAX_BLOCKS = 1024          # ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS of include/alegb.h


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests must run on the B200 box")
    from paper_2607_00199_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def case(name, refs):
    if name == "cfg3":                                   # 2-D, moving wall + far field + layer
        ref = refs(2, 4); cfg = configs.config3(ref.lam, ntheta=24, nr=10)
    elif name == "cfg5":                                 # 3-D swimmer box
        ref = refs(3, 3); cfg = swimmer_small(ref.lam)
    else:                                                # cfg1: periodic, no tagged faces at all
        ref = refs(2, 3); cfg = configs.config1(ref.lam)
    return ref, cfg


def state(cfg, amp, seed):
    rng = np.random.default_rng(seed)
    return cfg["q0"] * (1.0 + amp * rng.standard_normal(cfg["q0"].shape))


def tolerances(cfg, ref, q, t):
    """The bound test_wall_forces_match_oracle uses: 1e-12 x wall area x RT x max|q| (pressure: max|q_1|)."""
    P = oracle_problem(cfg, ref)
    g = P.geometry(t)
    area = sum(2.0 * g["sJ"][P.EToB[:, f] == 1, f].sum() for f in range(ref.Nfaces))
    assert area > 0
    return 1e-12 * area * cfg["RT"] * np.abs(q[:, 0]).max(), 1e-12 * area * cfg["RT"] * np.abs(q).max()


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["cfg3", "cfg5"])
def test_static_wall_forces_equal_the_allocating_path_on_two_calls_in_a_row(name, refs, B):
    ref, cfg = case(name, refs)
    dim = cfg["dim"]
    ctx = B.context_from_config(cfg)
    qa, qb = state(cfg, 2e-2, 7), state(cfg, 5e-2, 11)
    ta, tb = 0.0, 0.4
    dqa, dqb = dev(qa), dev(qb)
    nan = float("nan")

    # two calls in a row, each waited for; the second must not see anything of the first
    Fa = torch.full((2 * dim,), nan, dtype=torch.float64, device="cuda")
    Fb = torch.full((2 * dim,), nan, dtype=torch.float64, device="cuda")
    ctx.alegb_wall_forces_static(ta, dqa, Fa)
    torch.cuda.synchronize()
    Fa1 = Fa.cpu().numpy().copy()
    ctx.alegb_wall_forces_static(tb, dqb, Fb)
    torch.cuda.synchronize()
    Fb1 = Fb.cpu().numpy().copy()

    # the existing path on the same inputs
    pa, va = ctx.alegb_wall_forces(ta, dqa, 1)
    pb, vb = ctx.alegb_wall_forces(tb, dqb, 1)
    tol_pa, tol_va = tolerances(cfg, ref, qa, ta)
    tol_pb, tol_vb = tolerances(cfg, ref, qb, tb)
    assert np.abs(pa).max() > 1e3 * tol_pa and np.abs(pa - pb).max() > 1e3 * tol_pa     # the two cases do differ
    for F, p, v, tp, tv in ((Fa1, pa, va, tol_pa, tol_va), (Fb1, pb, vb, tol_pb, tol_vb)):
        assert np.isfinite(F).all()
        assert np.abs(F[:dim] - p).max() <= tp and np.abs(F[dim:] - v).max() <= tv
        # nblocks = 0 is the grid of alegb_wall_forces: same kernels, same order of the sums, same bits
        assert np.array_equal(F[:dim], p) and np.array_equal(F[dim:], v)

    # the same two calls queued back to back on the current stream, no host synchronisation in between
    Fa.fill_(nan); Fb.fill_(nan)
    ctx.alegb_wall_forces_static(ta, dqa, Fa)
    ctx.alegb_wall_forces_static(tb, dqb, Fb)
    torch.cuda.synchronize()
    assert np.array_equal(Fa.cpu().numpy(), Fa1) and np.array_equal(Fb.cpu().numpy(), Fb1)

    # other grids: a ragged one, a single block (the whole array entry 0 only), the largest that fits; after the
    # 1024-block call the array is full of that call's sums and the 5-block call after it must still be right
    for nblocks in (37, 1, MAX_BLOCKS, 5):
        Fb.fill_(nan)
        ctx.alegb_wall_forces_static(tb, dqb, Fb, nblocks=nblocks)
        torch.cuda.synchronize()
        F = Fb.cpu().numpy()
        assert np.abs(F[:dim] - pb).max() <= tol_pb and np.abs(F[dim:] - vb).max() <= tol_vb, nblocks

    # a grid beyond the array is refused with the limit in the message, and nothing is written
    Fb.fill_(nan)
    with pytest.raises(B.AlegbError) as err:
        ctx.alegb_wall_forces_static(tb, dqb, Fb, nblocks=MAX_BLOCKS + 1)
    assert err.value.status == B.INVALID_ARG
    assert "ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS = %d" % MAX_BLOCKS in str(err.value) and str(MAX_BLOCKS + 1) in str(err.value)
    with pytest.raises(B.AlegbError):
        ctx.alegb_wall_forces_static(tb, dqb, Fb, nblocks=-1)
    torch.cuda.synchronize()
    assert torch.isnan(Fb).all()
    # ... and the context still works afterwards
    ctx.alegb_wall_forces_static(tb, dqb, Fb)
    torch.cuda.synchronize()
    assert np.array_equal(Fb.cpu().numpy(), Fb1)
    ctx.close()


@pytest.mark.gpu
def test_static_wall_forces_second_context_and_untagged_mesh(refs, B):
    """The array belongs to the device, not to a context: a second context that follows on the same stream gets its
    own right answer.  A mesh without tagged faces gives zeros, as alegb_wall_forces does."""
    ref3, cfg3 = case("cfg3", refs)
    ref1, cfg1 = case("cfg1", refs)
    c3, c1 = B.context_from_config(cfg3), B.context_from_config(cfg1)
    q3, q1 = dev(state(cfg3, 2e-2, 3)), dev(state(cfg1, 2e-2, 5))
    F3 = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    F1 = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    c3.alegb_wall_forces_static(0.2, q3, F3)
    c1.alegb_wall_forces_static(0.2, q1, F1)
    c3b = B.context_from_config(cfg3)
    F3b = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    c3b.alegb_wall_forces_static(0.2, q3, F3b)
    torch.cuda.synchronize()
    p, v = c3.alegb_wall_forces(0.2, q3, 1)
    assert np.array_equal(F3.cpu().numpy(), np.concatenate([p, v]))
    assert np.array_equal(F3b.cpu().numpy(), np.concatenate([p, v]))
    p1, v1 = c1.alegb_wall_forces(0.2, q1, 1)
    assert not p1.any() and not v1.any() and not F1.cpu().numpy().any()
    for c in (c3, c1, c3b):
        c.close()


def _function_body(src, name):
    """Text of the C/C++ function `name` (from its name up to the closing brace in column 0)."""
    m = re.search(r"^[^\n/]*\b%s\s*\([^;{]*\)\s*\{.*?^\}" % re.escape(name), src, re.S | re.M)
    assert m, name
    return m.group(0)


def test_static_entry_point_source_has_no_allocation_and_resolves_the_symbol():
    """Tripwire on the sources (no GPU): the entry point and what it calls in kernels.cu name no allocating runtime
    call, the scratch is a static aligned __device__ array of the stated size, and host code reaches it through
    cudaGetSymbolAddress with the return code looked at."""
    csrc = os.path.join(ROOT, "paper_2607_00199_b200", "csrc")
    api = open(os.path.join(csrc, "alegb_api.cu")).read()
    ker = open(os.path.join(csrc, "kernels.cu")).read()
    hdr = open(os.path.join(ROOT, "include", "alegb.h")).read()
    assert re.search(r"#define\s+ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS\s+%d\b" % MAX_BLOCKS, hdr)
    bodies = [_function_body(api, "alegb_wall_forces_static"), _function_body(api, "update_geometry"),
              _function_body(ker, "launch_wall_force_static"), _function_body(ker, "wall_force_static_scratch"),
              _function_body(ker, "launch_wall_force")]
    for body in bodies:
        for banned in ("cudaMalloc", "cudaFree", "dev_alloc", "dev_free", "cudaHostAlloc", "new ", "std::vector"):
            assert banned not in body, (banned, body[:80])
    assert "launch_wall_force_static" in bodies[0] and "wall_force_static_scratch" in bodies[2]
    assert re.search(r"static\s+__device__\s+__align__\(256\)\s+double\s+g_wall_force_partial\[kWallForceStaticBlocks \* 6\]", ker)
    assert re.search(r"e = cudaGetSymbolAddress\(\(void\*\*\)&p, g_wall_force_partial\);[^\n]*\n\s*if \(e != cudaSuccess\) return e;", bodies[3])
