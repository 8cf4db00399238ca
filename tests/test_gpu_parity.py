"""Parity of the CUDA path (through the C-ABI) with the CPU oracle, element by element, on the same seeded inputs.

Tolerances (BASELINE.json north_star; R15):
  stage states   max|q_gpu - q_orc| / max|q_orc| <= 1e-12 per stage, <= 1e-10 after 100 steps
  F(q, t)        |F_gpu - F_orc| <= 1e-12 * Fabs pointwise, Fabs = the oracle's sum of absolute values of all terms
  geometry       relative 1e-13
Everything here needs a GPU (-m gpu) and calls the library only through paper_2607_00199_b200.binding.
"""
import numpy as np
import pytest

from oracle import mesh as omesh
from oracle import motion as omotion
from oracle import physics, sark
from workloads import configs, meshes
from helpers import oracle_problem, rel_linf, submesh, swimmer_small

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_STAGE, TOL_100, TOL_F = 1e-12, 1e-10, 1e-12


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests must run on the B200 box")
    from paper_2607_00199_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def perturbed(cfg, amp=1e-3, seed=7):
    """Initial state with seeded element-wise noise, so that every face carries a jump."""
    rng = np.random.default_rng(seed)
    return cfg["q0"] * (1.0 + amp * rng.standard_normal(cfg["q0"].shape))


def make_case(name, refs):
    if name == "cfg1":
        ref = refs(2, 3); cfg = configs.config1(ref.lam)
    elif name == "cfg2":
        ref = refs(2, 4); cfg = configs.config2(ref.lam, n=12)
    elif name == "cfg3":
        ref = refs(2, 4); cfg = configs.config3(ref.lam, ntheta=24, nr=10)
    elif name == "cfg4":
        ref = refs(3, 4); cfg = configs.config4(ref.lam, n=4)
    elif name == "cfg5":
        ref = refs(3, 3); cfg = swimmer_small(ref.lam)
    elif name == "cfg5_tiny":
        ref = refs(3, 3); cfg = swimmer_small(ref.lam, n=(8, 4, 4), lo=(-2.0, -1.5, -1.5), hi=(4.0, 1.5, 1.5))
    elif name == "tri_N1":
        ref = refs(2, 1); cfg = configs.config2(ref.lam, n=7); cfg["N"] = 1; cfg = configs._finish(cfg, ref.lam)
    elif name == "tri_N5":
        ref = refs(2, 5); cfg = configs.config2(ref.lam, n=5); cfg["N"] = 5; cfg = configs._finish(cfg, ref.lam)
    elif name == "tet_N2":
        ref = refs(3, 2); cfg = configs.config4(ref.lam, n=3); cfg["N"] = 2; cfg = configs._finish(cfg, ref.lam)
    elif name == "tet_N5":
        ref = refs(3, 5); cfg = configs.config4(ref.lam, n=3); cfg["N"] = 5; cfg = configs._finish(cfg, ref.lam)
    else:
        raise KeyError(name)
    return ref, cfg


CASES = ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "tri_N1", "tri_N5", "tet_N2", "tet_N5"]
KERNELS = [1, 2]     # alegb_set_kernel: 1 = generic DFMA kernel, 2 = pipelined DMMA kernel


def make_ctx(B, cfg, kernel):
    ctx = B.context_from_config(cfg)
    try:
        ctx.alegb_set_kernel(kernel)
    except B.AlegbError as e:
        assert e.status == B.UNSUPPORTED and kernel == 2
        ctx.close()
        pytest.skip("no DMMA kernel for dim=%d N=%d (the generic kernel covers it)" % (cfg["dim"], cfg["N"]))
    return ctx


@pytest.mark.parametrize("name", CASES)
def test_geometry_matches_oracle(name, refs, B):
    ref, cfg = make_case(name, refs)
    P = oracle_problem(cfg, ref)
    ctx = B.context_from_config(cfg)
    dim, K = cfg["dim"], cfg["K"]
    for t in (0.0, 0.137, 0.77):
        vgeo = torch.empty(K, dim * dim + 1, dtype=torch.float64, device="cuda")
        sgeo = torch.empty(K, dim + 1, dim + 2, dtype=torch.float64, device="cuda")
        xv = torch.empty(cfg["X0"].shape, dtype=torch.float64, device="cuda")
        vv = torch.empty_like(xv)
        ctx.alegb_geometry(t, vgeo, sgeo, xv, vv)
        torch.cuda.synchronize()
        g = P.geometry(t)
        vgeo, sgeo = vgeo.cpu().numpy(), sgeo.cpu().numpy()
        assert np.abs(xv.cpu().numpy() - g["xv"]).max() <= 1e-14 * np.abs(g["xv"]).max()
        assert np.abs(vv.cpu().numpy() - g["vv"]).max() <= 1e-13 * max(np.abs(g["vv"]).max(), 1e-300)
        assert rel_linf(vgeo[:, -1], g["J"]) < 1e-13
        assert rel_linf(vgeo[:, :-1].reshape(K, dim, dim), g["Ginv"]) < 1e-13
        assert np.abs(sgeo[:, :, :dim] - g["nhat"]).max() < 1e-13
        assert rel_linf(sgeo[:, :, dim], g["sJ"]) < 1e-13
        assert rel_linf(sgeo[:, :, dim + 1], g["Fscale"]) < 1e-13
    ctx.close()


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("name", CASES)
def test_rhs_matches_oracle(name, kernel, refs, B):
    ref, cfg = make_case(name, refs)
    P = oracle_problem(cfg, ref)
    ctx = make_ctx(B, cfg, kernel)
    q = perturbed(cfg)
    dq, dF = dev(q), torch.empty(q.shape, dtype=torch.float64, device="cuda")
    for t in (0.0, 0.31):
        if P.sigma is None:
            ctx.alegb_rhs(t, dq, dF)
            torch.cuda.synchronize()
            F, Fabs = P.rhs(q, t, want_abs=True)
        else:
            rng = np.random.default_rng(11)
            aux = 1e-3 * rng.standard_normal((len(P.pml_elems), cfg["dim"]) + q.shape[1:])
            daux, dG = dev(aux), torch.empty(aux.shape, dtype=torch.float64, device="cuda")
            ctx.alegb_rhs_pml(t, dq, daux, dF, dG)
            torch.cuda.synchronize()
            F, G, Fabs = P.rhs(q, t, aux=aux, want_abs=True)
            assert np.array_equal(ctx.alegb_pml_elements(), P.pml_elems)
            # the auxiliary right-hand side has no Fabs of its own: its terms are a subset of F's
            assert np.abs(dG.cpu().numpy() - G).max() <= TOL_F * (Fabs[P.pml_elems].max() + np.abs(G).max())
        err = np.abs(dF.cpu().numpy() - F)
        floor = 1e-3 * Fabs.max()
        assert (err <= TOL_F * (Fabs + floor)).all(), (err / (Fabs + floor)).max()
        assert err.max() <= 1e-12 * np.abs(F).max()
    ctx.close()


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("name", CASES)
def test_stage_states_match_oracle(name, kernel, refs, B):
    """R19: the four stage states of one step (test_hundred_steps repeats this at step 100)."""
    ref, cfg = make_case(name, refs)
    P = oracle_problem(cfg, ref)
    ctx = make_ctx(B, cfg, kernel)
    q = perturbed(cfg)
    dt = cfg["dt"]
    st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_step_debug(dev(q), 0.05, dt, st)
    torch.cuda.synchronize()
    so, aux = sark.step_debug(P, q, 0.05, dt)
    for i in range(4):
        assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_STAGE
    if aux is not None:
        da = torch.empty(aux.shape, dtype=torch.float64, device="cuda")
        ctx.alegb_pml_get(da)
        torch.cuda.synchronize()
        assert np.abs(da.cpu().numpy() - aux).max() <= TOL_STAGE * max(np.abs(aux).max(), np.abs(q).max() * 1e-6)
    ctx.close()


@pytest.mark.parametrize("name,nsteps", [("cfg1", 100), ("cfg2", 100), ("cfg3", 100), ("cfg4", 100), ("cfg5_tiny", 100)])
def test_hundred_steps_match_oracle(name, nsteps, refs, B):
    ref, cfg = make_case(name, refs)
    P = oracle_problem(cfg, ref)
    ctx = B.context_from_config(cfg)
    q = perturbed(cfg, amp=1e-4)
    dt = cfg["dt"]
    dq = dev(q)
    ctx.alegb_step(dq, 0.0, dt, nsteps - 1)
    torch.cuda.synchronize()
    out = sark.step(P, q, 0.0, dt, nsteps - 1)
    qo, aux = out if isinstance(out, tuple) else (out, None)
    assert rel_linf(dq.cpu().numpy(), qo) <= TOL_100
    # stage states of step number `nsteps`, each side continuing from its own state
    st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_step_debug(dq, (nsteps - 1) * dt, dt, st)
    torch.cuda.synchronize()
    so, _ = sark.step_debug(P, qo, (nsteps - 1) * dt, dt, aux)
    for i in range(4):
        assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_100
    ctx.close()


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dim", [2, 3])
def test_free_stream_preserved_on_gpu(dim, kernel, refs, B):
    """GCL (Table 2): a uniform state stays uniform on the deforming mesh, every stage."""
    if dim == 2:
        ref = refs(2, 3); cfg = configs.config1(ref.lam); nsteps = 50
    else:
        ref = refs(3, 4); cfg = configs.config4(ref.lam, n=6); nsteps = 20
        u = np.broadcast_to([0.1, 0.05, -0.02], (cfg["K"], ref.Np, 3))
        cfg["q0"] = np.ascontiguousarray(np.transpose(configs.maxwellian(3, np.ones((cfg["K"], ref.Np)), u, 1.0), (0, 2, 1)))
    ctx = make_ctx(B, cfg, kernel)
    q0 = cfg["q0"]
    st = torch.empty((4,) + q0.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_step_debug(dev(q0), 0.13, cfg["dt"], st)
    torch.cuda.synchronize()
    assert np.abs(st.cpu().numpy() - q0[None]).max() < 1e-14
    dq = dev(q0)
    ctx.alegb_step(dq, 0.0, cfg["dt"], nsteps)
    torch.cuda.synchronize()
    assert np.abs(dq.cpu().numpy() - q0).max() < 1e-13
    xv = torch.empty(cfg["X0"].shape, dtype=torch.float64, device="cuda")
    ctx.alegb_geometry(0.25, d_xv=xv)
    torch.cuda.synchronize()
    assert np.abs(xv.cpu().numpy() - cfg["X0"]).max() > 0.02      # the mesh really moved
    ctx.close()


def test_uniform_relaxation_exact_on_gpu(refs, B):
    """R8 pin on the device: uniform non-equilibrium state, q4(t) = q4eq + (q4(0)-q4eq) e^{-t/tau} to round-off."""
    ref = refs(2, 3)
    cfg = configs.config1(ref.lam, n=4)
    ctx = B.context_from_config(cfg)
    qe = physics.equilibrium_state(2, np.array(1.0), np.array([0.1, 0.05]), 1.0)
    q0 = qe.copy(); q0[3:] += np.array([0.02, -0.01, 0.03])
    q = np.broadcast_to(q0[None, :, None], (cfg["K"], 6, ref.Np)).copy()
    dt, n = 0.4 * cfg["tau"], 25
    dq = dev(q)
    ctx.alegb_step(dq, 0.0, dt, n)
    torch.cuda.synchronize()
    exact = qe + (q0 - qe) * np.exp(-n * dt / cfg["tau"] * physics.stiff_mask(2))
    assert np.abs(dq.cpu().numpy() - exact[None, :, None]).max() < 5e-15
    ctx.close()


def test_collisionless_and_static(refs, B):
    """tau = inf (classic RK4, no relaxation) and no motion: both degenerate branches against the oracle."""
    ref = refs(2, 3)
    cfg = configs.config1(ref.lam, n=5)
    cfg["tau"] = float("inf"); cfg["motion_kind"] = 0; cfg["motion_params"] = None
    P = oracle_problem(cfg, ref)
    ctx = B.context_from_config(cfg)
    q = perturbed(cfg)
    st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_step_debug(dev(q), 0.0, cfg["dt"], st)
    torch.cuda.synchronize()
    so, _ = sark.step_debug(P, q, 0.0, cfg["dt"])
    for i in range(4):
        assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_STAGE
    ctx.close()


def test_user_motion_equals_builtin(refs, B):
    ref, cfg = make_case("cfg4", refs)
    P = oracle_problem(cfg, ref)
    t = 0.21
    xv, vv = omotion.vertices(cfg["motion_kind"], cfg["motion_params"], cfg["X0"], t)
    ctx = B.context_from_config(cfg)
    q = perturbed(cfg)
    dq, dF = dev(q), torch.empty(q.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_set_motion_user(dev(xv), dev(vv))
    ctx.alegb_rhs(123.0, dq, dF)                      # time is irrelevant for USER motion
    torch.cuda.synchronize()
    F, Fabs = P.rhs(q, t, want_abs=True)
    assert (np.abs(dF.cpu().numpy() - F) <= TOL_F * (Fabs + 1e-3 * Fabs.max())).all()
    ctx.close()


@pytest.mark.parametrize("kernel", KERNELS)
def test_single_element_and_ragged_batches(kernel, refs, B):
    """K = 1 (every face a far-field face) and K values around the kernel's batch sizes."""
    ref = refs(3, 3)
    X0 = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1.0]])
    q_inf = physics.equilibrium_state(3, np.array(1.0), np.array([0.1, 0.0, 0.05]), 1.0)
    for K in (1, 2, 11, 13, 25):
        XX = np.concatenate([X0 + np.array([3.0 * k, 0, 0]) for k in range(K)])
        EToV = np.arange(4 * K, dtype=np.int32).reshape(K, 4)
        EToB = np.full((K, 4), 2, dtype=np.int8)
        cfg = dict(dim=3, N=3, X0=XX, EToV=EToV, vertex_equiv=None, EToB=EToB, pml_sigma=None, RT=1.0, tau=1e-2,
                   q_inf=q_inf, motion_kind=2, motion_params=np.array([0.02, 1.0, 2.0, 0.3]), K=K, Np=20, Nf=10)
        rng = np.random.default_rng(K)
        q = q_inf[None, :, None] * (1.0 + 1e-2 * rng.standard_normal((K, 10, 20)))
        P = oracle_problem(cfg, ref)
        ctx = make_ctx(B, cfg, kernel)
        st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
        ctx.alegb_step_debug(dev(q), 0.1, 1e-3, st)
        torch.cuda.synchronize()
        so, _ = sark.step_debug(P, q, 0.1, 1e-3)
        for i in range(4):
            assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_STAGE
        ctx.close()


def test_streams_alignment_and_errors(refs, B):
    ref, cfg = make_case("cfg1", refs)
    ctx = B.context_from_config(cfg)
    q = perturbed(cfg)
    s = torch.cuda.Stream()
    dq = dev(q)
    a, b = dq.clone(), dq.clone()
    torch.cuda.synchronize()
    ctx.alegb_step(a, 0.0, cfg["dt"], 3)
    torch.cuda.synchronize()          # one context = one workspace: calls on different streams must not overlap
    with torch.cuda.stream(s):
        ctx.alegb_step(b, 0.0, cfg["dt"], 3, stream=s)
    torch.cuda.synchronize()
    assert torch.equal(a, b)                              # same kernels, same order: bit-identical
    n0 = ctx.alegb_launch_count()
    ctx.alegb_step(a, 0.0, cfg["dt"], 2)
    assert ctx.alegb_launch_count() - n0 >= 2 * 4         # at least one launch per stage
    buf = torch.empty(q.size + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(B.AlegbError) as e:
        ctx.alegb_step(buf.data_ptr() + 8, 0.0, cfg["dt"], 1)
    assert e.value.status == B.INVALID_ARG
    fresh = B.Context(2, 3, 0)
    with pytest.raises(B.AlegbError) as e:
        fresh.alegb_rhs(0.0, dq, a)
    assert e.value.status == B.NOT_READY
    fresh.close(); ctx.close()


def test_step_host_roundtrip(refs, B):
    ref, cfg = make_case("cfg2", refs)
    ctx = B.context_from_config(cfg)
    q = perturbed(cfg)
    dq = dev(q)
    ctx.alegb_step(dq, 0.0, cfg["dt"], 2)
    hq = torch.from_numpy(q.copy()).pin_memory()
    ctx.alegb_step_host(hq, 0.0, cfg["dt"], 2)
    assert np.array_equal(hq.numpy(), dq.cpu().numpy())
    ctx.close()


@pytest.mark.parametrize("name", ["cfg1", "cfg3", "cfg4"])
def test_graph_replay_is_bit_identical_to_direct_launches(name, refs, B):
    """alegb_step(nsteps >= 2) replays one captured CUDA graph per step with the stage times kept on the device
    (include/alegb.h: alegb_set_graph).  Same kernels, same arguments, same stage times => identical bits as the
    direct launches; also after t0 changes (no re-capture), after set_motion (re-capture) and on a user stream."""
    ref, cfg = make_case(name, refs)
    ctx = B.context_from_config(cfg)
    q = perturbed(cfg)
    dt = cfg["dt"]

    def run(graph, t0, nsteps, stream=None):
        ctx.alegb_set_graph(graph)
        ctx.alegb_pml_reset()
        dq = dev(q)
        n0 = ctx.alegb_launch_count()
        if stream is None:
            ctx.alegb_step(dq, t0, dt, nsteps)
        else:
            with torch.cuda.stream(stream):
                ctx.alegb_step(dq, t0, dt, nsteps)
            stream.synchronize()
        torch.cuda.synchronize()
        return dq.cpu().numpy(), ctx.alegb_launch_count() - n0

    direct, nd = run(False, 0.3, 5)
    replay, ng = run(True, 0.3, 5)
    assert np.array_equal(direct, replay)
    assert ng == nd + 5 + 1                      # one clock kernel per step + one clock set per call
    direct2, _ = run(False, 0.7, 3)
    replay2, _ = run(True, 0.7, 3)               # same graph, new t0 on the device
    assert np.array_equal(direct2, replay2) and not np.array_equal(direct2, direct)
    replay3, _ = run(True, 0.3, 5, torch.cuda.Stream())
    assert np.array_equal(direct, replay3)
    if cfg["motion_kind"] != 0:                  # changing the motion law invalidates the captured graph
        ctx.alegb_set_motion(0, [])
        still, _ = run(True, 0.3, 5)
        ref_still, _ = run(False, 0.3, 5)
        assert np.array_equal(still, ref_still) and not np.array_equal(still, direct)
    ctx.close()


@pytest.mark.parametrize("relax", ["collocation", "cubature"])
def test_full_size_throughput_config_sampled(relax, refs, B):
    """BASELINE.json configs[3] at full size (196,608 tets, N = 4), the launch configuration bench.py times
    (default mode, and bench.py --relax cubature).
    The oracle computes a sample of elements one patch at a time (helpers.submesh): F needs the face neighbours,
    stage state i needs i rings of them."""
    ref = refs(3, 4)
    cfg = configs.config4(ref.lam)
    assert cfg["K"] == 196608
    conn = omesh.connect(ref, cfg["EToV"], cfg["vertex_equiv"])
    ctx = B.context_from_config(cfg)
    cfg["relax"] = relax
    if relax == "cubature":
        ctx.alegb_set_relaxation(B.RELAX_CUBATURE)
    q = perturbed(cfg, amp=1e-4)
    cfg["q0"] = q
    dq = dev(q)
    dF = torch.empty_like(dq)
    t, dt = 0.2, cfg["dt"]
    ctx.alegb_rhs(t, dq, dF)
    st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_step_debug(dq, t, dt, st)
    torch.cuda.synchronize()
    rng = np.random.default_rng(5)
    samples = np.concatenate([[0, 1, cfg["K"] - 1, cfg["K"] - 2], rng.integers(0, cfg["K"], size=8)])
    Fg = dF[torch.from_numpy(samples).cuda()].cpu().numpy()
    sub, patch, where = submesh(cfg, conn["EToE"], samples, rings=1)
    F, Fabs = oracle_problem(sub, ref).rhs(sub["q0"], t, want_abs=True)
    assert (np.abs(Fg - F[where]) <= TOL_F * (Fabs[where] + 1e-3 * Fabs.max())).all()
    for s0 in samples[:6]:
        sub, patch, where = submesh(cfg, conn["EToE"], [s0], rings=4)
        so, _ = sark.step_debug(oracle_problem(sub, ref), sub["q0"], t, dt)
        for i in range(4):
            got = st[i, int(s0)].cpu().numpy()
            assert np.abs(got - so[i][where[0]]).max() <= TOL_STAGE * np.abs(so[i]).max()
    # property that holds at any size: the uniform state is a fixed point of the step on the deforming mesh
    u = np.broadcast_to([0.1, 0.05, -0.02], (cfg["K"], ref.Np, 3))
    q0 = np.ascontiguousarray(np.transpose(configs.maxwellian(3, np.ones((cfg["K"], ref.Np)), u, 1.0), (0, 2, 1)))
    dq = dev(q0)
    ctx.alegb_step(dq, 0.0, dt, 3)
    torch.cuda.synchronize()
    assert np.abs(dq.cpu().numpy() - q0).max() < 1e-13
    ctx.close()


# ------------------------------------------------------------------ NEXT-2: coordinates integrated by RK4 (L152, L233)
@pytest.mark.gpu
@pytest.mark.parametrize("name", ["cfg1", "cfg3", "cfg4"])
def test_rk_coordinates_stage_states_match_oracle(name, refs, B):
    """alegb_set_coordinate_mode(RK): stage states of one step from an advanced x_n, positions after several steps."""
    from oracle import coords
    ref, cfg = make_case(name, refs)
    P = oracle_problem(cfg, ref)
    q = perturbed(cfg)
    dt, t0 = cfg["dt"], 0.0
    ctx = B.context_from_config(cfg)
    ctx.alegb_set_coordinate_mode(B.COORDS_RK, t0)
    # two steps through alegb_step advance q and x_n; the oracle does the same
    dq = dev(q)
    ctx.alegb_step(dq, t0, dt, 2)
    dx = torch.empty(cfg["X0"].shape, dtype=torch.float64, device="cuda")
    ctx.alegb_get_positions(dx)
    torch.cuda.synchronize()
    if P.sigma is not None:
        qo, xo, auxo = coords.step(P, q, P.X0.copy(), t0, dt, 2)
    else:
        qo, xo = coords.step(P, q, P.X0.copy(), t0, dt, 2)
        auxo = None
    assert np.abs(dx.cpu().numpy() - xo).max() <= 1e-14 * max(1.0, np.abs(xo).max())
    assert rel_linf(dq.cpu().numpy(), qo) <= TOL_STAGE
    # the third step observed stage by stage; step_debug must leave x_n alone
    st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_step_debug(dq, t0 + 2 * dt, dt, st)
    dx2 = torch.empty_like(dx)
    ctx.alegb_get_positions(dx2)
    torch.cuda.synchronize()
    assert torch.equal(dx, dx2)
    so, _, _ = coords.step_debug(P, qo, xo, t0 + 2 * dt, dt, auxo)
    for i in range(4):
        assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_STAGE
    ctx.close()


@pytest.mark.gpu
def test_rk_coordinates_graph_replay_and_free_stream(refs, B):
    """Many steps through the captured graph equal the direct launches bit for bit, x_n included; a uniform state on
    the integrated mesh stays uniform (GCL, Table 2)."""
    ref, cfg = make_case("cfg1", refs)
    q0 = cfg["q0"]
    outs = []
    for graph in (1, 0):
        ctx = B.context_from_config(cfg)
        ctx.alegb_set_graph(graph)
        ctx.alegb_set_coordinate_mode(B.COORDS_RK, 0.0)
        dq = dev(q0)
        ctx.alegb_step(dq, 0.0, cfg["dt"], 25)
        dx = torch.empty(cfg["X0"].shape, dtype=torch.float64, device="cuda")
        ctx.alegb_get_positions(dx)
        torch.cuda.synchronize()
        outs.append((dq.cpu().numpy(), dx.cpu().numpy()))
        ctx.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    assert np.abs(outs[0][0] - q0).max() < 1e-13
    exact = omotion.vertices(cfg["motion_kind"], cfg["motion_params"], cfg["X0"], 25 * cfg["dt"])[0]
    assert np.abs(outs[0][1] - exact).max() < 1e-8             # follows the law to time-integration accuracy


@pytest.mark.gpu
def test_rk_coordinates_user_velocity(refs, B):
    """Motion kind USER in RK mode: a velocity constant in time moves the vertices linearly."""
    ref, cfg = make_case("cfg1", refs)
    rng = np.random.default_rng(199)
    xv = cfg["X0"].copy()
    vv = 0.05 * np.sin(np.pi * cfg["X0"][:, :1]) * np.sin(np.pi * cfg["X0"][:, 1:2]) * np.ones((1, 2))
    ctx = B.context_from_config(cfg)
    ctx.alegb_set_motion_user(dev(xv), dev(vv))
    ctx.alegb_set_coordinate_mode(B.COORDS_RK, 0.0)
    dq = dev(cfg["q0"])
    ctx.alegb_step(dq, 0.0, cfg["dt"], 10)
    dx = torch.empty(xv.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_get_positions(dx)
    torch.cuda.synchronize()
    assert np.abs(dx.cpu().numpy() - (xv + 10 * cfg["dt"] * vv)).max() < 1e-15
    assert np.abs(dq.cpu().numpy() - cfg["q0"]).max() < 1e-13       # free stream
    ctx.close()


# ------------------------------------------------------------------ NEXT-1: cubature-projected relaxation (L84-107, L197)
def _cubature_case(name, refs):
    ref, cfg = make_case(name, refs)
    cfg["relax"] = "cubature"
    return ref, cfg, oracle_problem(cfg, ref)


@pytest.mark.gpu
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "tri_N5", "tet_N2", "tet_N5"])
def test_cubature_rhs_matches_oracle(name, kernel, refs, B):
    ref, cfg, P = _cubature_case(name, refs)
    ctx = make_ctx(B, cfg, kernel)
    ctx.alegb_set_relaxation(B.RELAX_CUBATURE)
    q = perturbed(cfg, amp=3e-2)                     # large enough for the projection to differ from collocation
    dq, dF = dev(q), torch.empty(q.shape, dtype=torch.float64, device="cuda")
    t = 0.31
    ctx.alegb_rhs(t, dq, dF)
    torch.cuda.synchronize()
    out = P.rhs(q, t, want_abs=True)
    F, Fabs = out[0], out[-1]
    assert (np.abs(dF.cpu().numpy() - F) <= TOL_F * (Fabs + 1e-3 * Fabs.max())).all()
    # the mode is live: the collocated operator differs by far more than the tolerance
    ctx.alegb_set_relaxation(B.RELAX_COLLOCATION)
    dF2 = torch.empty_like(dF)
    ctx.alegb_rhs(t, dq, dF2)
    torch.cuda.synchronize()
    assert (dF2 - dF).abs().max().item() > 1e3 * TOL_F * Fabs.max()
    ctx.close()


@pytest.mark.gpu
def test_cubature_with_automatic_kernel_where_no_dmma_cubature_kernel_exists(refs, B):
    """3-D N=5 has neither a pipelined stage kernel nor a DMMA cubature kernel: the automatic selection
    (alegb_set_kernel(0), the default) must fall back to the generic kernels instead of failing."""
    ref, cfg, P = _cubature_case("tet_N5", refs)
    ctx = B.context_from_config(cfg)
    ctx.alegb_set_relaxation(B.RELAX_CUBATURE)
    q = perturbed(cfg, amp=3e-2)
    dq, dF = dev(q), torch.empty(q.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_rhs(0.31, dq, dF)
    torch.cuda.synchronize()
    out = P.rhs(q, 0.31, want_abs=True)
    F, Fabs = out[0], out[-1]
    assert (np.abs(dF.cpu().numpy() - F) <= TOL_F * (Fabs + 1e-3 * Fabs.max())).all()
    dq2 = dev(q)
    ctx.alegb_step(dq2, 0.0, cfg["dt"], 2)
    torch.cuda.synchronize()
    assert torch.isfinite(dq2).all().item()
    ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["cfg1", "cfg3", "cfg4"])
def test_cubature_stage_states_and_steps_match_oracle(name, refs, B):
    ref, cfg, P = _cubature_case(name, refs)
    ctx = B.context_from_config(cfg)
    ctx.alegb_set_relaxation(B.RELAX_CUBATURE)
    q = perturbed(cfg)
    st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_step_debug(dev(q), 0.1, cfg["dt"], st)
    torch.cuda.synchronize()
    so, _ = sark.step_debug(P, q, 0.1, cfg["dt"])
    for i in range(4):
        assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_STAGE
    # 20 steps through the captured graph (alegb_step_debug advanced the library's PML state: start it from zero)
    if P.sigma is not None:
        ctx.alegb_pml_reset()
    dq = dev(q)
    ctx.alegb_step(dq, 0.0, cfg["dt"], 20)
    torch.cuda.synchronize()
    qo = sark.step(P, q, 0.0, cfg["dt"], 20)
    qo = qo[0] if isinstance(qo, tuple) else qo
    assert rel_linf(dq.cpu().numpy(), qo) <= TOL_100
    ctx.close()


@pytest.mark.gpu
def test_cubature_free_stream_on_gpu(refs, B):
    ref, cfg = make_case("cfg1", refs)
    ctx = B.context_from_config(cfg)
    ctx.alegb_set_relaxation(B.RELAX_CUBATURE)
    dq = dev(cfg["q0"])
    ctx.alegb_step(dq, 0.0, cfg["dt"], 50)
    torch.cuda.synchronize()
    assert np.abs(dq.cpu().numpy() - cfg["q0"]).max() < 1e-13
    ctx.close()


# ------------------------------------------------------------------ measurement: the fp64 ceiling bench.py reports
@pytest.mark.gpu
def test_measured_fp64_peak_is_plausible(refs, B):
    """alegb_measure_fp64_peak: both microbenchmarks land near the figure derived from the unit counts
    (148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2 TFLOP/s) -- well above half of it (the chains do run on every SM and
    are not optimised away) and not above it by more than clock granularity allows."""
    ref, cfg = make_case("cfg1", refs)
    ctx = B.context_from_config(cfg)
    dmma, dfma = ctx.alegb_measure_fp64_peak()
    derived = 148 * 64 * 2 * 1.965e9 / 1e12
    assert 0.5 * derived < dmma < 1.1 * derived, (dmma, dfma)
    assert 0.5 * derived < dfma < 1.1 * derived, (dmma, dfma)
    ctx.close()


# ------------------------------------------------------------------ NEXT-3: wall-force integrals (L308, L369)
@pytest.mark.gpu
@pytest.mark.parametrize("name", ["cfg3", "cfg5", "cfg1"])
def test_wall_forces_match_oracle(name, refs, B):
    from oracle import forces
    ref, cfg = make_case(name, refs)
    P = oracle_problem(cfg, ref)
    q = perturbed(cfg, amp=2e-2)
    ctx = B.context_from_config(cfg)
    for t in (0.0, 0.4):
        Fp, Fv = ctx.alegb_wall_forces(t, dev(q), 1)
        Fp2, Fv2 = ctx.alegb_wall_forces(t, dev(q), 1)
        assert np.array_equal(Fp, Fp2) and np.array_equal(Fv, Fv2)          # deterministic
        op, ov = forces.wall_force(P, q, t)
        scale = max(np.abs(op).max(), np.abs(ov).max(), 1e-300)
        if name == "cfg1":                                                  # no wall faces
            assert not Fp.any() and not Fv.any() and not op.any()
        else:
            # absolute scale of the summed terms: the integral of |p| over the wall
            g = P.geometry(t)
            area = sum(2.0 * g["sJ"][P.EToB[:, f] == 1, f].sum() for f in range(ref.Nfaces))
            assert area > 0
            assert np.abs(Fp - op).max() <= 1e-12 * area * cfg["RT"] * np.abs(q[:, 0]).max()
            assert np.abs(Fv - ov).max() <= 1e-12 * area * cfg["RT"] * np.abs(q).max()
            assert scale > 0
    ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("name,where", [("cfg3", "all"), ("cfg5_tiny", "all"), ("cfg5_tiny", "every_other_quad")])
def test_layer_fusion_with_an_empty_or_interleaved_plain_list(name, where, refs, B):
    """The fused path splits the quads into a plain and a layer launch.  With damping on every element (a whole-domain
    sponge) the plain list is EMPTY and must not be launched at all (a NULL list means "every quad" to the kernel:
    the mesh would be swept twice and stage 2's in-place accumulator doubled); with the layer on every other quad the
    two lists interleave.  Stage states and auxiliary state of one step against the oracle, then five steps fused
    against the separate layer kernel."""
    ref, cfg = make_case(name, refs)
    cfg = dict(cfg)
    K, dim = cfg["EToV"].shape[0], cfg["dim"]
    sig = np.array(cfg["pml_sigma"], dtype=np.float64, copy=True)
    if where == "all":
        sig += 0.5
    else:
        sig[:] = 0.0
        sig[(np.arange(K) // 4) % 2 == 0] = (0.7, 0.0, 0.3)[:dim]
    cfg["pml_sigma"] = sig
    P = oracle_problem(cfg, ref)
    q, dt = perturbed(cfg), cfg["dt"]
    so, aux = sark.step_debug(P, q, 0.05, dt)
    out = {}
    for fused in (1, 0):
        ctx = B.context_from_config(cfg)
        ctx.alegb_set_layer_fusion(fused)
        assert ctx.alegb_pml_count() == (K if where == "all" else ((np.arange(K) // 4) % 2 == 0).sum())
        st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
        n0 = ctx.alegb_launch_count()
        ctx.alegb_step_debug(dev(q), 0.05, dt, st)
        nl = ctx.alegb_launch_count() - n0
        da = torch.empty(aux.shape, dtype=torch.float64, device="cuda")
        ctx.alegb_pml_get(da)
        torch.cuda.synchronize()
        for i in range(4):
            assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_STAGE, (fused, i)
        assert np.abs(da.cpu().numpy() - aux).max() <= TOL_STAGE * max(np.abs(aux).max(), np.abs(q).max() * 1e-6)
        dq = dev(q)
        ctx.alegb_pml_reset()
        ctx.alegb_step(dq, 0.0, dt, 5)
        ctx.alegb_pml_get(da)
        torch.cuda.synchronize()
        out[fused] = (dq, da.clone(), nl)
        ctx.close()
    if where == "all":
        assert out[1][2] < out[0][2]          # one stage launch per stage, not plain + layer
    for x, y in zip(out[1][:2], out[0][:2]):
        assert (x - y).abs().max().item() <= 1e-13 * max(y.abs().max().item(), 1e-300)


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["cfg1", "cfg3", "cfg4"])
def test_geometry_overlap_is_bit_identical(name, refs, B):
    """a1/a2 of stage i+1 beside the stage kernel of stage i (side stream, second geometry set): same bits as in-order
    launches, through the graph and through direct launches, closed-form and RK coordinates."""
    ref, cfg = make_case(name, refs)
    q = perturbed(cfg)
    outs = []
    for overlap, graph, rk in ((1, 1, 0), (0, 1, 0), (1, 0, 0), (0, 0, 0), (1, 1, 1), (0, 0, 1)):
        ctx = B.context_from_config(cfg)
        ctx.alegb_set_geometry_overlap(overlap)
        ctx.alegb_set_graph(graph)
        if rk:
            ctx.alegb_set_coordinate_mode(B.COORDS_RK, 0.0)
        dq = dev(q)
        ctx.alegb_step(dq, 0.0, cfg["dt"], 7)
        ctx.alegb_step(dq, 7 * cfg["dt"], cfg["dt"], 1)
        torch.cuda.synchronize()
        outs.append(dq.cpu().numpy())
        ctx.close()
    for o in outs[1:4]:
        assert np.array_equal(outs[0], o)
    assert np.array_equal(outs[4], outs[5])


@pytest.mark.gpu
@pytest.mark.parametrize("dim,N,n", [(3, 1, 12), (3, 2, 10), (3, 3, 10), (2, 1, 72), (2, 2, 64), (2, 3, 56)])
def test_low_orders_with_many_quads_per_cta(dim, N, n, refs, B):
    """Low orders have few work items per quad (NB = 1 at N = 1), so a consumer warp of the pipelined kernel owns an
    item only in every CW-th quad; with many quads per CTA this is the regime in which a warp that skipped the
    hand-over of the quads in between could pass an mbarrier parity wait two phases early (stale tile) or hang.
    Meshes large enough for >= 10 quads per CTA, all three kernels against the oracle."""
    ref = refs(dim, N)
    cfg = configs.config4(ref.lam, n=n) if dim == 3 else configs.config2(ref.lam, n=n)
    cfg["N"] = N
    cfg = configs._finish(cfg, ref.lam)
    assert cfg["K"] >= 148 * 4 * 10
    P = oracle_problem(cfg, ref)
    q = perturbed(cfg)
    F, Fabs = P.rhs(q, 0.2, want_abs=True)
    so, _ = sark.step_debug(P, q, 0.2, cfg["dt"])
    for kernel in KERNELS:
        ctx = B.context_from_config(cfg)
        try:
            ctx.alegb_set_kernel(kernel)
        except B.AlegbError:
            ctx.close()
            continue
        dq, dF = dev(q), torch.empty(q.shape, dtype=torch.float64, device="cuda")
        st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
        for rep in range(3):                                  # timing-dependent failures: a few repetitions
            ctx.alegb_rhs(0.2, dq, dF)
            ctx.alegb_step_debug(dq, 0.2, cfg["dt"], st)
            torch.cuda.synchronize()
            assert (np.abs(dF.cpu().numpy() - F) <= TOL_F * (Fabs + 1e-3 * Fabs.max())).all()
            for i in range(4):
                assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_STAGE
        ctx.close()


# ------------------------------------------------------------------ NEXT-2, general: stage data supplied by the caller
@pytest.mark.gpu
@pytest.mark.parametrize("name", ["cfg1", "cfg4"])
def test_user_stage_data_of_the_law_equal_the_builtin_modes_bit_for_bit(name, refs, B):
    """alegb_set_motion_user_stages fed with the law's own positions / velocities at the four stage times must give
    the bits of the built-in law, in closed-form mode and with RK-integrated coordinates (x_n included)."""
    ref, cfg = make_case(name, refs)
    q = perturbed(cfg)
    dt, t0, nsteps = cfg["dt"], 0.3, 3
    for rk in (0, 1):
        built = B.context_from_config(cfg)
        user = B.context_from_config(cfg)
        helper = B.context_from_config(cfg)                    # evaluates the law at the stage times
        if rk:
            built.alegb_set_coordinate_mode(B.COORDS_RK, t0)
        qa, qb = dev(q), dev(q)
        built.alegb_step(qa, t0, dt, nsteps)                   # three steps, through the captured graph
        nv = cfg["X0"].shape
        for n in range(nsteps):
            xv4 = torch.empty((4,) + nv, dtype=torch.float64, device="cuda")
            vv4 = torch.empty_like(xv4)
            for i, c in enumerate((0.0, 0.5, 0.5, 1.0)):
                helper.alegb_geometry((t0 + n * dt) + c * dt, d_xv=xv4[i], d_vv=vv4[i])
            torch.cuda.synchronize()
            user.alegb_set_motion_user_stages(xv4, vv4)
            if rk and n == 0:
                user.alegb_set_coordinate_mode(B.COORDS_RK, t0)   # x_n = the positions of entry 0
            user.alegb_step(qb, t0 + n * dt, dt, 1)
        torch.cuda.synchronize()
        assert torch.equal(qa, qb)
        if rk:
            xa = torch.empty(nv, dtype=torch.float64, device="cuda"); xb = torch.empty_like(xa)
            built.alegb_get_positions(xa); user.alegb_get_positions(xb)
            torch.cuda.synchronize()
            assert torch.equal(xa, xb)
        built.close(); user.close(); helper.close()


@pytest.mark.gpu
def test_user_stage_velocities_that_depend_on_the_positions_match_oracle(refs, B):
    """A rigid rotation of the whole (non-periodic view of the) mesh about its centre: v = Omega x (x - c) evaluated
    by the caller at its own RK stage positions (k_2 != k_3), RK coordinate mode.  Stage states and x_{n+1} against
    oracle/coords.py with the same four velocities; a uniform state stays uniform (GCL)."""
    from oracle import coords
    ref, cfg = make_case("cfg3", refs)                         # no periodic faces: a rotation is admissible
    P = oracle_problem(cfg, ref)
    om, cen = 20.0, np.array([0.5, 0.0])      # fast enough for k_2 - k_3 = O((om dt)^2) to be visible at the CFL step
    rot = lambda x: om * np.stack([-(x[:, 1] - cen[1]), x[:, 0] - cen[0]], axis=1)
    q = perturbed(cfg)
    dt, t0 = cfg["dt"], 0.0
    ctx = B.context_from_config(cfg)
    x = cfg["X0"].copy()
    dq = dev(q)
    qo, auxo = q, None
    for n in range(2):
        k1 = rot(x); k2 = rot(x + 0.5 * dt * k1); k3 = rot(x + 0.5 * dt * k2); k4 = rot(x + dt * k3)
        assert np.abs(k2 - k3).max() > 1e-9 * np.abs(k2).max()
        ks = np.stack([k1, k2, k3, k4])
        ctx.alegb_set_motion_user_stages(dev(np.stack([x] * 4)) if n == 0 else None, dev(ks))
        if n == 0:
            ctx.alegb_set_coordinate_mode(B.COORDS_RK, t0)
        st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
        ctx.alegb_step_debug(dq, t0 + n * dt, dt, st)          # observes the stages, leaves x_n and q alone
        ctx.alegb_pml_set(dev(auxo)) if auxo is not None else ctx.alegb_pml_reset()
        ctx.alegb_step(dq, t0 + n * dt, dt, 1)
        dx = torch.empty(x.shape, dtype=torch.float64, device="cuda")
        ctx.alegb_get_positions(dx)
        torch.cuda.synchronize()
        so, auxo, x = coords.step_debug(P, qo, x, t0 + n * dt, dt, auxo, stage_velocities=(k1, k2, k3, k4))
        for i in range(4):
            assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_STAGE
        qo = so[-1]
        assert rel_linf(dq.cpu().numpy(), qo) <= 2 * TOL_STAGE   # second step: each side continues from its own state
        assert np.abs(dx.cpu().numpy() - x).max() <= 1e-14 * np.abs(x).max()
    ctx.close()


# ------------------------------------------------------------------ a8 fused into the stage kernel
@pytest.mark.gpu
@pytest.mark.parametrize("name", ["cfg3", "cfg5", "cfg5_tiny"])
def test_layer_fusion_agrees_with_the_separate_layer_kernel(name, refs, B):
    """alegb_set_layer_fusion: the auxiliary fields advanced inside the pipelined stage kernel (default) against the
    separate layer kernel after it -- same equations (reading R12), F and G to round-off, ten steps of q and of the
    auxiliary state.  (Both paths are compared with the oracle by the other tests: the default is the fused one.)"""
    ref, cfg = make_case(name, refs)
    q = perturbed(cfg)
    rng = np.random.default_rng(11)
    out = {}
    for fused in (1, 0):
        ctx = B.context_from_config(cfg)
        ctx.alegb_set_layer_fusion(fused)
        Kpml = ctx.alegb_pml_count()
        assert Kpml > 0
        aux = 1e-3 * np.random.default_rng(11).standard_normal((Kpml, cfg["dim"]) + q.shape[1:])
        dq, dF = dev(q), torch.empty(q.shape, dtype=torch.float64, device="cuda")
        dG = torch.empty(aux.shape, dtype=torch.float64, device="cuda")
        n0 = ctx.alegb_launch_count()
        ctx.alegb_rhs_pml(0.3, dq, dev(aux), dF, dG)
        nl = ctx.alegb_launch_count() - n0
        ctx.alegb_pml_set(dev(aux))
        ctx.alegb_step(dq, 0.0, cfg["dt"], 10)
        da = torch.empty_like(dG)
        ctx.alegb_pml_get(da)
        torch.cuda.synchronize()
        out[fused] = (dF, dG, dq, da, nl)
        ctx.close()
    assert out[1][4] <= out[0][4]                              # the layer quads run through one (fused) launch
    for x, y in zip(out[1][:4], out[0][:4]):
        assert (x - y).abs().max().item() <= 1e-13 * max(y.abs().max().item(), 1e-300)
