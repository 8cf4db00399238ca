"""Parity at the sizes and in the launch configurations bench.py times (BASELINE.json configs at full size), and in
the steady state of the pipelined stage kernel's shared-memory ring (many quads per CTA, every element compared).

  * configs[1] (8,192 triangles) and configs[2] (60,000 triangles, wall + far field + PML ring): every element
    against the oracle at full size (F, four stage states, PML auxiliary state).
  * configs[3] (196,608 tetrahedra, N=4): F on >= 512 sampled elements spread over all 148 CTAs and all ring slots,
    stage states on 64 of them (oracle on patches, helpers.submesh); and EVERY element of the pipelined DMMA kernel
    against the generic DFMA kernel on the device (the generic kernel is itself compared with the oracle everywhere
    else) for F, the stage states and a few steps.
  * configs[4] (1.5 M tetrahedra, N=3, wall + far field + PML shell): sampled elements that include wall faces,
    far-field faces, layer elements, the first and the last quad.
  * 3-D N=4 with >= 17 quads per CTA (10,368 tetrahedra), every element, both kernels; and 100 steps with the ring
    wrapping many times (few CTAs through alegb_set_max_ctas).
Tolerances as in test_gpu_parity.py (north_star: 1e-12 per stage, 1e-10 after 100 steps; R15).
"""
import numpy as np
import pytest

from oracle import mesh as omesh
from oracle import sark
from workloads import configs
from helpers import oracle_problem, rel_linf, submesh

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
    rng = np.random.default_rng(seed)
    return cfg["q0"] * (1.0 + amp * rng.standard_normal(cfg["q0"].shape))


def check_rhs(Fg, F, Fabs):
    """DESIGN.md R15: pointwise against Fabs, with a floor of 1e-3 max Fabs (round-off of the largest entries that
    enter a node's sums through the dense operators)."""
    err = np.abs(Fg - F)
    floor = 1e-3 * Fabs.max()
    assert (err <= TOL_F * (Fabs + floor)).all(), (err / (Fabs + floor)).max()


# ---------------------------------------------------------------------------------- configs[1], configs[2]: everything
@pytest.mark.parametrize("index", [2, 3])
def test_full_size_2d_configs_every_element(index, refs, B):
    ref = refs(2, 4)
    cfg = configs.BY_INDEX[index](ref.lam)
    assert cfg["K"] == {2: 8192, 3: 60000}[index]
    P = oracle_problem(cfg, ref)
    q = perturbed(cfg)
    t, dt = 0.2, cfg["dt"]
    ctx = B.context_from_config(cfg)
    dq, dF = dev(q), torch.empty(q.shape, dtype=torch.float64, device="cuda")
    st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
    if P.sigma is None:
        ctx.alegb_rhs(t, dq, dF)
        F, Fabs = P.rhs(q, t, want_abs=True)
    else:
        rng = np.random.default_rng(11)
        aux = 1e-3 * rng.standard_normal((len(P.pml_elems), 2) + q.shape[1:])
        dG = torch.empty(aux.shape, dtype=torch.float64, device="cuda")
        ctx.alegb_rhs_pml(t, dq, dev(aux), dF, dG)
        F, G, Fabs = P.rhs(q, t, aux=aux, want_abs=True)
        assert len(P.pml_elems) > 1000 and np.array_equal(ctx.alegb_pml_elements(), P.pml_elems)
        assert np.abs(dG.cpu().numpy() - G).max() <= TOL_F * (Fabs[P.pml_elems].max() + np.abs(G).max())
        assert (cfg["EToB"] == 1).sum() == 300 and (cfg["EToB"] == 2).sum() == 300
    torch.cuda.synchronize()
    check_rhs(dF.cpu().numpy(), F, Fabs)
    ctx.alegb_pml_reset()
    ctx.alegb_step_debug(dq, t, dt, st)
    torch.cuda.synchronize()
    so, aux1 = sark.step_debug(P, q, t, dt)
    for i in range(4):
        assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_STAGE
    if aux1 is not None:
        da = torch.empty(aux1.shape, dtype=torch.float64, device="cuda")
        ctx.alegb_pml_get(da)
        torch.cuda.synchronize()
        assert np.abs(da.cpu().numpy() - aux1).max() <= TOL_STAGE * max(np.abs(aux1).max(), np.abs(q).max() * 1e-6)
    ctx.close()


# ---------------------------------------------------------------------------------- configs[3]: the throughput config
def spread_samples(K, n, num_ctas=148, slots=4, eg=4):
    """n element ids such that consecutive samples fall on consecutive CTAs (quad % num_ctas), cycle through the
    ring slots ((quad // num_ctas) % slots) and through the positions inside a quad; plus the first and last quad."""
    nquads = (K + eg - 1) // eg
    per_cta = nquads // num_ctas
    out = []
    for i in range(n):
        cta = i % num_ctas
        ql = (i // num_ctas * slots + i % slots + 5 * (i % 7)) % per_cta
        out.append(min(K - 1, eg * (ql * num_ctas + cta) + i % eg))
    out += [0, 1, 2, 3, K - 4, K - 3, K - 2, K - 1]
    return np.unique(np.array(out, dtype=np.int64))


def test_full_size_config4_sampled_over_all_ctas_and_slots(refs, B):
    ref = refs(3, 4)
    cfg = configs.config4(ref.lam)
    K = cfg["K"]
    assert K == 196608
    conn = omesh.connect(ref, cfg["EToV"], cfg["vertex_equiv"])
    ctx = B.context_from_config(cfg)
    q = perturbed(cfg, amp=1e-4)
    cfg["q0"] = q
    dq = dev(q)
    dF = torch.empty_like(dq)
    t, dt = 0.2, cfg["dt"]
    ctx.alegb_rhs(t, dq, dF)
    st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_step_debug(dq, t, dt, st)
    torch.cuda.synchronize()
    samples = spread_samples(K, 520)
    quads = samples // 4
    assert len(samples) >= 512 and len(set(quads % 148)) == 148 and len(set((quads // 148) % 4)) == 4
    Fg = dF[torch.from_numpy(samples).cuda()].cpu().numpy()
    sub, patch, where = submesh(cfg, conn["EToE"], samples, rings=1)
    F, Fabs = oracle_problem(sub, ref).rhs(sub["q0"], t, want_abs=True)
    check_rhs(Fg, F[where], Fabs[where])
    # stage state i needs i rings of neighbours: 64 samples (every slot, 64 different CTAs), one patch
    s64 = samples[:: len(samples) // 64][:64]
    assert len(set((s64 // 4 // 148) % 4)) == 4
    sub, patch, where = submesh(cfg, conn["EToE"], s64, rings=4)
    so, _ = sark.step_debug(oracle_problem(sub, ref), sub["q0"], t, dt)
    idx = torch.from_numpy(s64).cuda()
    for i in range(4):
        got = st[i][idx].cpu().numpy()
        assert np.abs(got - so[i][where]).max() <= TOL_STAGE * np.abs(so[i]).max()
    ctx.close()


@pytest.mark.parametrize("index", [4, 5])
def test_full_size_3d_configs_pipelined_equals_generic_kernel_on_every_element(index, refs, B):
    """No oracle cost: the generic DFMA kernel (a different implementation: one thread per node, operators as
    plain transposed matrices, no tensor cores, no ring) is compared with the oracle everywhere else; here it
    checks EVERY element of the pipelined DMMA kernel at full size, in the launch configuration bench.py times."""
    dim, N = (3, 4) if index == 4 else (3, 3)
    ref = refs(dim, N)
    cfg = configs.BY_INDEX[index](ref.lam)
    q = perturbed(cfg, amp=1e-4)
    t, dt = 0.2, cfg["dt"]
    res = {}
    for kernel in (1, 2):
        ctx = B.context_from_config(cfg)
        ctx.alegb_set_kernel(kernel)
        dq = dev(q)
        dF = torch.empty_like(dq)
        ctx.alegb_rhs(t, dq, dF)
        st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
        ctx.alegb_step_debug(dq, t, dt, st)
        ctx.alegb_pml_reset()
        ctx.alegb_step(dq, t, dt, 3)
        torch.cuda.synchronize()
        res[kernel] = (dF, st, dq)
        ctx.close()
    (F1, st1, q1), (F2, st2, q2) = res[1], res[2]
    fscale = F1.abs().max().item()
    # summation order differs (DMMA accumulates k in blocks of 4, the generic kernel in sequence): 1e-13 of the scale
    assert (F1 - F2).abs().max().item() <= 1e-13 * fscale * 10
    for i in range(4):
        assert (st1[i] - st2[i]).abs().max().item() <= 2e-13 * st1[i].abs().max().item()
    assert (q1 - q2).abs().max().item() <= 1e-12 * q1.abs().max().item()
    assert torch.isfinite(q2).all().item()


def test_full_size_config5_sampled(refs, B):
    """configs[4]: 1.5 M tetrahedra, N=3.  Samples: elements with a wall face, with a far-field face, inside the
    absorbing layer (several directions), the first and the last quad (the last one ragged if K % 4 != 0)."""
    ref = refs(3, 3)
    cfg = configs.config5(ref.lam)
    K = cfg["K"]
    assert K > 1_400_000
    conn = omesh.connect(ref, cfg["EToV"], None, cfg["EToB"])
    EToB, sigma = cfg["EToB"], cfg["pml_sigma"]
    wall = np.nonzero((EToB == 1).any(axis=1))[0]
    far = np.nonzero((EToB == 2).any(axis=1))[0]
    layer = np.nonzero((sigma > 0).any(axis=1))[0]
    corner = np.nonzero((sigma > 0).all(axis=1))[0]
    assert len(wall) >= 90 and len(far) > 1000 and len(layer) > 100000 and len(corner) > 0
    rng = np.random.default_rng(5)
    pick = lambda a, n: a[rng.integers(0, len(a), size=n)]
    samples = np.unique(np.concatenate([pick(wall, 24), pick(far, 24), pick(layer, 24), pick(corner, 8),
                                        rng.integers(0, K, size=40), [0, 1, 2, 3, K - 4, K - 3, K - 2, K - 1]]))
    ctx = B.context_from_config(cfg)
    assert ctx.alegb_workspace_bytes() > 8e9
    q = perturbed(cfg, amp=1e-3)
    cfg["q0"] = q
    dq = dev(q)
    dF = torch.empty_like(dq)
    t, dt = 0.6, cfg["dt"]
    Kpml = ctx.alegb_pml_count()
    assert Kpml == len(layer)
    rng = np.random.default_rng(11)
    aux = 1e-3 * rng.standard_normal((Kpml, 3, 10, ref.Np))
    daux = dev(aux)
    dG = torch.empty_like(daux)
    ctx.alegb_rhs_pml(t, dq, daux, dF, dG)
    torch.cuda.synchronize()
    sub, patch, where = submesh(cfg, conn["EToE"], samples, rings=1)
    Psub = oracle_problem(sub, ref)
    # the patch's layer elements in ascending order = the order of the oracle's compact auxiliary array
    pos_in_layer = np.searchsorted(layer, patch[Psub.pml_elems])
    assert np.array_equal(layer[pos_in_layer], patch[Psub.pml_elems])
    F, G, Fabs = Psub.rhs(sub["q0"], t, aux=aux[pos_in_layer], want_abs=True)
    Fg = dF[torch.from_numpy(samples).cuda()].cpu().numpy()
    check_rhs(Fg, F[where], Fabs[where])
    # auxiliary right-hand side on the sampled layer elements
    in_layer = np.isin(samples, layer)
    sl = samples[in_layer]
    gpos = np.searchsorted(layer, sl)
    Gg = dG[torch.from_numpy(gpos).cuda()].cpu().numpy()
    opos = np.searchsorted(patch[Psub.pml_elems], sl)
    assert len(sl) >= 24
    assert np.abs(Gg - G[opos]).max() <= TOL_F * (Fabs[where].max() + np.abs(G).max())
    # stage states of one step on >= 64 samples (4 rings each, one patch), auxiliary state from zero: wall, far field,
    # layer elements with one / two / three damped directions, elements just outside the layer, random ones, the
    # first and the last quad; and the auxiliary state after the step on the sampled layer elements
    nlive = (sigma > 0).sum(axis=1)
    one, two, three = (np.nonzero(nlive == k)[0] for k in (1, 2, 3))
    assert len(one) > 100000 and len(two) > 10000 and len(three) > 1000
    s64 = np.unique(np.concatenate([pick(wall, 12), pick(far, 12), pick(one, 12), pick(two, 12), pick(three, 8),
                                    rng.integers(0, K, size=8), [0, 1, 2, 3, K - 4, K - 3, K - 2, K - 1]]))
    assert len(s64) >= 64
    ctx.alegb_pml_reset()
    st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
    ctx.alegb_step_debug(dq, t, dt, st)
    da = torch.empty_like(daux)
    ctx.alegb_pml_get(da)
    torch.cuda.synchronize()
    sub, patch, where = submesh(cfg, conn["EToE"], s64, rings=4)
    Psub = oracle_problem(sub, ref)
    so, auxo = sark.step_debug(Psub, sub["q0"], t, dt)
    idx = torch.from_numpy(s64).cuda()
    for i in range(4):
        got = st[i][idx].cpu().numpy()
        assert np.abs(got - so[i][where]).max() <= TOL_STAGE * np.abs(so[i]).max()
    sl = s64[np.isin(s64, layer)]
    assert len(sl) >= 32
    got = da[torch.from_numpy(np.searchsorted(layer, sl)).cuda()].cpu().numpy()
    want = auxo[np.searchsorted(patch[Psub.pml_elems], sl)]
    # where sigma_d = 0 the auxiliary field never reaches q (it enters only as -sigma_d q~^d): compared where it can
    live = (sigma[sl] > 0)[:, :, None, None]
    assert np.abs((got - want) * live).max() <= TOL_STAGE * max(np.abs(auxo).max(), np.abs(q).max() * 1e-6)
    ctx.close()


# ---------------------------------------------------------------------------------- the ring in its steady state
def test_order4_3d_many_quads_per_cta_every_element(refs, B):
    """3-D N=4 (the instantiation bench.py times: 4 producer warps as one group, ring of 4, bar.sync hand-over) on
    10,368 tetrahedra = 2,592 quads = 17.5 quads per CTA, every element against the oracle, both kernels, three
    repetitions (timing-dependent failures)."""
    ref = refs(3, 4)
    cfg = configs.config4(ref.lam, n=12)
    assert cfg["K"] == 10368 and cfg["K"] // 4 >= 148 * 10
    P = oracle_problem(cfg, ref)
    q = perturbed(cfg)
    t, dt = 0.2, cfg["dt"]
    F, Fabs = P.rhs(q, t, want_abs=True)
    so, _ = sark.step_debug(P, q, t, dt)
    for kernel in (1, 2):
        ctx = B.context_from_config(cfg)
        ctx.alegb_set_kernel(kernel)
        dq, dF = dev(q), torch.empty(q.shape, dtype=torch.float64, device="cuda")
        st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
        for rep in range(3 if kernel == 2 else 1):
            dF.zero_(); st.zero_()
            ctx.alegb_rhs(t, dq, dF)
            ctx.alegb_step_debug(dq, t, dt, st)
            torch.cuda.synchronize()
            check_rhs(dF.cpu().numpy(), F, Fabs)
            for i in range(4):
                assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_STAGE
        ctx.close()


@pytest.mark.parametrize("dim,N,n", [(3, 4, 4), (3, 3, 4), (2, 4, 12)])
def test_hundred_steps_with_the_ring_wrapping(dim, N, n, refs, B):
    """100 steps with few CTAs (alegb_set_max_ctas), so that every CTA walks through many quads and every ring slot
    is reused many times per launch: 1, 5 and 16 CTAs give 96 / 20 / 6 quads per CTA on the 384-element 3-D mesh."""
    ref = refs(dim, N)
    cfg = configs.config4(ref.lam, n=n) if dim == 3 else configs.config2(ref.lam, n=n)
    cfg["N"] = N
    cfg = configs._finish(cfg, ref.lam)
    P = oracle_problem(cfg, ref)
    q = perturbed(cfg, amp=1e-4)
    dt, nsteps = cfg["dt"], 100
    qo = sark.step(P, q, 0.0, dt, nsteps - 1)
    so, _ = sark.step_debug(P, qo, (nsteps - 1) * dt, dt)
    for ctas in (1, 5, 16):
        ctx = B.context_from_config(cfg)
        ctx.alegb_set_kernel(2)
        ctx.alegb_set_max_ctas(ctas)
        dq = dev(q)
        ctx.alegb_step(dq, 0.0, dt, nsteps - 1)
        torch.cuda.synchronize()
        assert rel_linf(dq.cpu().numpy(), qo) <= TOL_100
        st = torch.empty((4,) + q.shape, dtype=torch.float64, device="cuda")
        ctx.alegb_step_debug(dq, (nsteps - 1) * dt, dt, st)
        torch.cuda.synchronize()
        for i in range(4):
            assert rel_linf(st[i].cpu().numpy(), so[i]) <= TOL_100
        ctx.close()


@pytest.mark.parametrize("dim,N", [(3, 3), (3, 4), (2, 4)])
def test_small_ring_wrapping_case(dim, N, refs, B):
    """The smallest case that wraps the ring several times (4 CTAs on a few hundred elements), one direct step and
    two graph-replayed steps with the a1/a2 side stream on, against the oracle.  This is also the case the
    compute-sanitizer runs of profiles/ use (racecheck / synccheck are 10-100x slower than a plain run)."""
    ref = refs(dim, N)
    cfg = configs.config4(ref.lam, n=4) if dim == 3 else configs.config2(ref.lam, n=12)
    cfg["N"] = N
    cfg = configs._finish(cfg, ref.lam)
    P = oracle_problem(cfg, ref)
    q = perturbed(cfg)
    dt = cfg["dt"]
    ctx = B.context_from_config(cfg)
    ctx.alegb_set_kernel(2)
    ctx.alegb_set_max_ctas(4)
    ctx.alegb_set_geometry_overlap(True)
    dq = dev(q)
    ctx.alegb_step(dq, 0.0, dt, 1)
    ctx.alegb_step(dq, dt, dt, 2)
    torch.cuda.synchronize()
    qo = sark.step(P, q, 0.0, dt, 3)
    assert rel_linf(dq.cpu().numpy(), qo) <= 3 * TOL_STAGE      # three steps, 1e-12 each
    ctx.close()
