"""GPU parity: the CUDA path (through the C ABI, include/wz.h) against the CPU oracle,
element by element on the same seeded inputs (SURVEY 8(d) thresholds):
  FFT / matvec: relative L2 error <= 1e-12 (complex128), <= 2e-5 (complex64);
  CG: true residual (recomputed by the ORACLE's M^dag M on the GPU's x) <= tol,
      iterations within +-2 of the oracle for complex128.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = {"c128": 1e-12, "c64": 2e-5}
NPDT = {"c128": np.complex128, "c64": np.complex64}

# lattices small enough for the oracle: several tiles, ragged/asymmetric extents
LATTICES = [(4, 4, 4, 4), (8, 8, 8, 8), (8, 4, 16, 8), (16, 16, 16, 16), (48, 24, 24, 24),
            (32, 8, 8, 8), (32, 16, 16, 16)]  # the last two: the paper's 8^3x32 and 16^3x32 (Tables V-VII)
# the lattices bench.py times (configs 4, 5b) and the paper's 32^3x64: one source, radix-2 oracle
BIG_LATTICES = [(32, 32, 32, 32), (64, 32, 32, 32), (64, 64, 64, 64)]


def rel(a, ref):
    return float(np.linalg.norm((a - ref).ravel()) / np.linalg.norm(ref.ravel()))


@pytest.fixture(scope="module")
def wz():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_1005_3276_b200 import wz as _wz

    _wz.lib()  # must load: no fallback
    return _wz


@pytest.fixture(scope="module")
def inp():
    from paper_1005_3276_b200 import inputs

    return inputs


def _fields(inp, dims, dtype, seed=7, sigma=0.4, nsrc=1):
    phi = inp.make_phi(seed, dims, sigma, NPDT[dtype])
    b = inp.make_sources(seed, nsrc, dims, NPDT[dtype])
    return phi, b


@pytest.mark.parametrize("dims", LATTICES)
@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("apbc", [True, False])
def test_fft4d_vs_oracle(wz, orc, inp, dims, dtype, apbc):
    if not wz.supported(dims, dtype):
        pytest.skip("no tile kernel")
    _, b = _fields(inp, dims, dtype, nsrc=2)
    plan = wz.Plan(dims, dtype, 2)
    d_b = torch.from_numpy(b).cuda()
    f = plan.fft4d(d_b, +1, apbc)
    ref = np.stack([orc.dft4d(b[j].astype(np.complex128), +1, apbc) for j in range(2)])
    assert rel(f.cpu().numpy(), ref) <= TOL[dtype]
    # inverse of the oracle's transform gives back b; also in place
    d_f = torch.from_numpy(ref.astype(NPDT[dtype])).cuda()
    plan.fft4d(d_f, -1, apbc, out=d_f)
    back = np.stack([orc.dft4d(ref[j].astype(NPDT[dtype]).astype(np.complex128), -1, apbc) for j in range(2)])
    assert rel(d_f.cpu().numpy(), back) <= TOL[dtype]
    # GPU round trip
    rt = plan.fft4d(f, -1, apbc)
    assert rel(rt.cpu().numpy(), b.astype(np.complex128)) <= 2 * TOL[dtype]


@pytest.mark.parametrize("dims", BIG_LATTICES)
@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("apbc", [True, False])
def test_fft4d_vs_oracle_bench_sizes(wz, orc, inp, dims, dtype, apbc):
    """The stand-alone transform in the launch configuration bench.py times (k_p01<FWD/INV> and
    k_p23<FFT, +-1> at 32^4 / 64^4, and the paper's 32^3x64), element by element against the oracle's
    radix-2 transform (steps a1, a2, a4, a5; Table V 883-890)."""
    if not wz.supported(dims, dtype):
        pytest.fail("bench lattices must be supported")
    b = inp.make_source(13, 0, dims, NPDT[dtype])
    plan = wz.Plan(dims, dtype, 1)
    d_b = torch.from_numpy(b).cuda()
    f = plan.fft4d(d_b, +1, apbc).cpu().numpy()
    ref = orc.dft4d(b.astype(np.complex128), +1, apbc)
    assert rel(f, ref) <= TOL[dtype]
    # inverse of (the rounded) oracle transform, in place
    refr = ref.astype(NPDT[dtype])
    d_f = torch.from_numpy(refr).cuda()
    plan.fft4d(d_f, -1, apbc, out=d_f)
    back = orc.dft4d(refr.astype(np.complex128), -1, apbc)
    assert rel(d_f.cpu().numpy(), back) <= TOL[dtype]


@pytest.mark.parametrize("dims", LATTICES)
@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("dagger", [False, True])
def test_apply_M_vs_oracle(wz, orc, inp, dims, dtype, dagger):
    if not wz.supported(dims, dtype):
        pytest.skip("no tile kernel")
    phi, b = _fields(inp, dims, dtype, nsrc=2)
    m, g, rho = 0.1 + 0.05j, 0.5 - 0.2j, 1.0  # complex m, g exercise the conjugations of Eq. 2.19
    plan = wz.Plan(dims, dtype, 2)
    out = plan.apply_M(torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda(), m, g, rho, dagger)
    ref = np.stack([orc.apply_M(phi.astype(np.complex128), b[j].astype(np.complex128), m, g, rho, dagger)
                    for j in range(2)])
    assert rel(out.cpu().numpy(), ref) <= TOL[dtype]


@pytest.mark.parametrize("dims", LATTICES)
@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("rho", [1.0, 0.7, 1.4])
def test_apply_MdagM_vs_oracle(wz, orc, inp, dims, dtype, rho):
    if not wz.supported(dims, dtype):
        pytest.skip("no tile kernel")
    if rho != 1.0 and dims[0] > 8:
        pytest.skip("rho sweep on the small lattices only")
    phi, b = _fields(inp, dims, dtype, nsrc=1)
    m, g = 0.05, 1.0
    plan = wz.Plan(dims, dtype, 1)
    out = plan.apply_MdagM(torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda(), m, g, rho)
    ref = orc.apply_MdagM(phi.astype(np.complex128), b[0].astype(np.complex128), m, g, rho)[None]
    assert rel(out.cpu().numpy(), ref) <= TOL[dtype]


def _solve_and_check(wz, orc, inp, cfg, nsrc=None, max_iter=50000):
    dims, dtype = cfg["dims"], cfg["dtype"]
    nsrc = nsrc or cfg["nsrc"]
    phi = inp.make_phi(cfg["seed"], dims, cfg["sigma"], NPDT[dtype])
    b = inp.make_sources(cfg["seed"], nsrc, dims, NPDT[dtype])
    plan = wz.Plan(dims, dtype, nsrc)
    x, infos = plan.cg_solve(torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda(), cfg["m"], cfg["g"],
                             cfg["rho"], cfg["tol"], max_iter)
    x = x.cpu().numpy()
    phi128 = phi.astype(np.complex128)
    out = []
    for j in range(nsrc):
        bj = b[j].astype(np.complex128)
        true_res = rel(orc.apply_MdagM(phi128, x[j], cfg["m"], cfg["g"], cfg["rho"]), bj)
        assert infos[j].converged
        assert true_res <= cfg["tol"], (j, true_res, infos[j])
        assert abs(infos[j].rel_residual_true - true_res) <= 0.05 * cfg["tol"]
        out.append((infos[j], true_res, phi128, bj))
    return out


@pytest.mark.parametrize("cfg_id", [1, 2])
def test_cg_complex128_configs(wz, orc, inp, cfg_id):
    cfg = inp.CONFIGS[cfg_id]
    (info, true_res, phi, b), = _solve_and_check(wz, orc, inp, cfg)
    xo, io = orc.cg(phi, b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 50000)
    assert io.converged
    # North star: +-2.  Enforced at config 1.  At config 2 the count at the stop is not determined to +-2 by
    # the method: the oracle's residual swings by +-30 % from one iteration to the next around tol, and
    # rounding-equivalent variants of the ORACLE ITSELF (naive or radix-2 DFT, blocked or pairwise dot products,
    # alpha from <p, M^dag M p> or from ||M p||^2) stop anywhere from 785 to 794 (reading G10, measured).
    # What the method does fix is pinned much harder by test_cg_trajectory_vs_oracle (x_k at 1e-10 while the two
    # trajectories have not yet separated); here: 1.5 % and the oracle must be at the threshold where the GPU stopped.
    delta = info.iterations - io.iterations
    print("config %s: iterations gpu=%d oracle=%d delta=%+d" % (cfg_id, info.iterations, io.iterations, delta))
    bound = 2 if cfg_id == 1 else max(2, int(0.015 * io.iterations))
    assert abs(delta) <= bound, (info.iterations, io.iterations)
    k = min(info.iterations, len(io.history) - 1)
    window = io.history[max(0, k - 2):k + 3]
    print("oracle residual history around the GPU's last iteration:", ["%.3e" % v for v in window])
    assert min(window) <= 2.0 * cfg["tol"]
    assert info.reliable_updates == 0


TRAJ_CASES = [
    # (name, dims, dtype, seed, sigma_phi, m, g)
    ("config 1", (4, 4, 4, 4), "c128", 1, 0.3, 0.1, 0.5),
    ("config 2", (8, 8, 8, 8), "c128", 2, 0.3, 0.05, 1.0),
    ("config 3 shape at 8^4, complex64", (8, 8, 8, 8), "c64", 3, 0.5, 0.02, 1.0),
    ("config 3, complex64", (16, 16, 16, 16), "c64", 3, 0.5, 0.02, 1.0),
    ("8^3x32 (paper lattice), complex128", (32, 8, 8, 8), "c128", 2, 0.3, 0.05, 1.0),
]


@pytest.mark.parametrize("case", TRAJ_CASES, ids=[c[0] for c in TRAJ_CASES])
def test_cg_trajectory_vs_oracle(wz, orc, inp, case):
    """The CG iterates themselves (steps a8-a10): after k = 1, 2, 5, 20 iterations the
    GPU's x_k and recursive residual against the oracle's, element by element, while rounding has not yet
    separated the two trajectories.  This pins alpha (from ||M p||^2 in pass C), beta, the x update applied
    one pass late and k_flush_x far harder than a final count can.  Two rounding-equivalent variants of the
    oracle itself agree to 1e-14 at k = 20 and differ by 3e-3 in x (40 % in the residual) at k = 100
    (G10), so k = 100 is only checked to be on the same convergence curve."""
    name, dims, dtype, seed, sig, m, g = case
    phi = inp.make_phi(seed, dims, sig, NPDT[dtype])
    b = inp.make_source(seed, 0, dims, NPDT[dtype])
    plan = wz.Plan(dims, dtype, 1)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b[None]).cuda()
    phi128, b128 = phi.astype(np.complex128), b.astype(np.complex128)
    tol_x = {"c128": 1e-10, "c64": 2e-5}[dtype]
    tol_r = {"c128": 1e-8, "c64": 1e-4}[dtype]
    for k in (1, 2, 5, 20, 100):
        x, infos = plan.cg_solve(d_phi, d_b, m, g, 1.0, 1e-30, k, raise_on_fail=False)
        if dtype == "c128":
            xo, io = orc.cg(phi128, b128, m, g, 1.0, 1e-30, k)
        else:
            xo, io = orc.cg_c64ru(phi128, b128, m, g, 1.0, 1e-30, k)
        dx = rel(x.cpu().numpy()[0], xo)
        dr = abs(infos[0].rel_residual_recursive - io.rel_residual_recursive) / io.rel_residual_recursive
        print("%s k=%d: |x_gpu - x_oracle|/|x_oracle| = %.2e, recursive residual gpu %.6e oracle %.6e (rel diff %.1e), RU %d/%d"
              % (name, k, dx, infos[0].rel_residual_recursive, io.rel_residual_recursive, dr,
                 infos[0].reliable_updates, io.reliable_updates))
        assert infos[0].iterations == io.iterations == k
        if k <= 20:
            scale = 1.0 if k <= 5 else 10.0  # rounding differences grow with k (complex64: one float ulp per update)
            assert dx <= tol_x * scale, (k, dx)
            assert dr <= tol_r * scale, (k, dr)
            assert infos[0].reliable_updates == io.reliable_updates
        else:
            assert dx <= 0.05 and dr <= 1.0, (k, dx, dr)


def test_cg_complex64_config3_all_sources(wz, orc, inp):
    """Config 3 as BASELINE.json states it: 16^4 complex64, four sources solved to 1e-6.  complex64 vectors +
    reliable updates (G9): bind on the true residual (recomputed by the oracle); every source's iteration
    count is compared with the oracle's O4' loop on the same source (G10: 5 %, +-2 is not expected) and
    must not be below the complex128 count by more than rounding noise."""
    cfg = inp.CONFIGS[3]
    res = _solve_and_check(wz, orc, inp, cfg)
    assert len(res) == 4
    for j, (info, true_res, phi, b) in enumerate(res):
        Xo, io = orc.cg_c64ru(phi, b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 50000)
        print("config 3 source %d: iters gpu=%d oracle(O4')=%d delta=%+d  RU gpu=%d oracle=%d  true residual %.3e"
              % (j, info.iterations, io.iterations, info.iterations - io.iterations, info.reliable_updates,
                 io.reliable_updates, true_res))
        assert io.converged
        assert info.reliable_updates >= 1
        assert abs(info.iterations - io.iterations) <= 0.05 * io.iterations
    # one source also against the complex128 loop: fewer iterations than exact-arithmetic-like CG would be a red flag
    info, _, phi, b = res[0]
    _, i128 = orc.cg(phi, b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 50000)
    print("config 3 source 0: complex128 oracle %d iterations" % i128.iterations)
    assert info.iterations >= 0.97 * i128.iterations


def test_cg_batch_of_sources_c64(wz, orc, inp):
    cfg = dict(inp.CONFIGS[3])
    cfg.update(dims=(8, 8, 8, 8), nsrc=3, m=0.05)
    res = _solve_and_check(wz, orc, inp, cfg)
    its = [r[0].iterations for r in res]
    # each source of the batch against a single-source solve of the same right-hand side
    dims = cfg["dims"]
    phi = torch.from_numpy(inp.make_phi(cfg["seed"], dims, cfg["sigma"], np.complex64)).cuda()
    b = torch.from_numpy(inp.make_sources(cfg["seed"], 3, dims, np.complex64)).cuda()
    plan = wz.Plan(dims, "c64", 1)
    for j in range(3):
        _, i1 = plan.cg_solve(phi, b[j:j + 1].contiguous(), cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 50000)
        assert i1[0].iterations == its[j] and min(its) > 10


def test_cg_max_iter_and_zero_source(wz, inp):
    cfg = inp.CONFIGS[2]
    dims = cfg["dims"]
    phi = torch.from_numpy(inp.make_phi(2, dims, 0.3)).cuda()
    b = torch.from_numpy(inp.make_source(2, 0, dims)).cuda()
    plan = wz.Plan(dims, "c128", 1)
    with pytest.raises(wz.WZError) as e:
        plan.cg_solve(phi, b, cfg["m"], cfg["g"], 1.0, 1e-10, 5)
    assert e.value.status == wz.WZ_ENOTCONVERGED
    x, infos = plan.cg_solve(phi, b, cfg["m"], cfg["g"], 1.0, 1e-10, 5, raise_on_fail=False)
    assert infos[0].iterations == 5 and not infos[0].converged and infos[0].rel_residual_true > 1e-10
    x, infos = plan.cg_solve(phi, torch.zeros_like(b), cfg["m"], cfg["g"], 1.0, 1e-10, 100)
    assert infos[0].converged and infos[0].iterations == 0 and float(x.abs().max()) == 0.0


def test_errors(wz, inp):
    dims = (4, 4, 4, 4)
    plan = wz.Plan(dims, "c128", 1)
    phi = torch.from_numpy(inp.make_phi(1, dims, 0.3)).cuda()
    b = torch.from_numpy(inp.make_source(1, 0, dims)).cuda()
    with pytest.raises(wz.WZError) as e:
        plan.apply_M(phi, b, 0.1, 0.5, 1.0, False, out=b)  # in == out
    assert e.value.status == wz.WZ_EINVAL
    with pytest.raises(wz.WZError) as e:
        plan.apply_MdagM(phi, b, 0.1, 0.5, 2.5)  # rho outside (0, 2)
    assert e.value.status == wz.WZ_EINVAL
    with pytest.raises(wz.WZError) as e:
        plan.fft4d(torch.stack([b, b]), +1, True)  # nbatch > max_batch
    assert e.value.status == wz.WZ_EINVAL
    with pytest.raises(wz.WZError) as e:
        wz.Plan((5, 4, 4, 4), "c128", 1)  # T odd
    assert e.value.status == wz.WZ_EINVAL
    with pytest.raises(wz.WZError) as e:
        wz.Plan((10, 4, 4, 4), "c128", 1)
    assert e.value.status == wz.WZ_EUNSUPPORTED


def test_fft_constant_phi_closed_form(wz, inp):
    """P5 on the GPU at a size the oracle does not run: constant phi = phi0 gives
    M^dag M = (d^2(p) + |w|^2) 1 in momentum space, so
    F[M^dag M psi] = (d^2 + |w|^2) F[psi]; checked with the GPU FFT on 32^4 complex64
    against d^2 computed here in numpy from Eq. (3.1)/(4.2)."""
    dims = (32, 32, 32, 32)
    if not wz.supported(dims, "c64"):
        pytest.skip("no tile kernel")
    m, g, rho, phi0 = 0.01, 1.5, 1.0, 0.3 - 0.2j
    b = inp.make_source(4, 0, dims, np.complex64)
    plan = wz.Plan(dims, "c64", 1)
    d_b = torch.from_numpy(b).cuda()
    d_phi = torch.full(dims, phi0, dtype=torch.complex64, device="cuda")
    q = plan.apply_MdagM(d_phi, d_b, m, g, rho)
    fq = plan.fft4d(q, +1, True).cpu().numpy().astype(np.complex128)
    fb = plan.fft4d(d_b, +1, True).cpu().numpy().astype(np.complex128)
    p = [2 * np.pi * (np.arange(L) + (0.5 if mu == 0 else 0.0)) / L for mu, L in enumerate(dims)]
    P = np.meshgrid(*p, indexing="ij")
    S2 = sum(np.sin(x) ** 2 for x in P)
    Mw = rho - 2 * sum(np.sin(x / 2) ** 2 for x in P)
    s = np.sqrt(Mw ** 2 + S2)
    c = np.where(Mw >= 0, 2 * rho / (s + Mw + (Mw < 0)), 2 * rho * (s - Mw) / S2)
    d2 = c ** 2 * S2
    w = m + 2 * g * np.complex128(np.complex64(phi0))
    ref = (d2 + abs(w) ** 2)[None] * fb
    assert rel(fq, ref) <= 2e-5


# ---- full-size checks (BASELINE.json configs 4 and 5), in the launch configuration bench.py times ----

@pytest.mark.parametrize("dims,dtype", [((32, 32, 32, 32), "c64"), ((32, 32, 32, 32), "c128"),
                                        ((64, 64, 64, 64), "c64"), ((64, 64, 64, 64), "c128")])
def test_full_size_MdagM_vs_oracle(wz, orc, inp, dims, dtype):
    """One M^dag M at 32^4 / 64^4 against the oracle (radix-2 route), element by element."""
    if not wz.supported(dims, dtype):
        pytest.fail("configs 4 and 5b must be supported")
    cfg = inp.CONFIGS[4 if dims[0] == 32 else "5b"]
    phi = inp.make_phi(cfg["seed"], dims, cfg["sigma"], NPDT[dtype])
    b = inp.make_source(cfg["seed"], 0, dims, NPDT[dtype])
    plan = wz.Plan(dims, dtype, 1)
    out = plan.apply_MdagM(torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda(), cfg["m"], cfg["g"], cfg["rho"])
    out = out.cpu().numpy()
    del plan
    ref = orc.apply_MdagM(phi.astype(np.complex128), b.astype(np.complex128), cfg["m"], cfg["g"], cfg["rho"])
    assert rel(out, ref) <= TOL[dtype]


def test_config4_batched_solve_true_residual(wz, orc, inp):
    """Config 4 as bench.py runs it: 12 sources in lock step to 1e-6.  Every source must
    converge; for a sample of sources the ORACLE recomputes the true residual of the GPU's x."""
    cfg = inp.CONFIGS[4]
    dims, nsrc = cfg["dims"], cfg["nsrc"]
    phi = inp.make_phi(cfg["seed"], dims, cfg["sigma"], np.complex64)
    b = inp.make_sources(cfg["seed"], nsrc, dims, np.complex64)
    plan = wz.Plan(dims, "c64", nsrc)
    x, infos = plan.cg_solve(torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda(), cfg["m"], cfg["g"],
                             cfg["rho"], cfg["tol"], 100000)
    assert all(i.converged for i in infos)
    assert all(i.rel_residual_true <= cfg["tol"] for i in infos)
    its = [i.iterations for i in infos]
    print("config 4 iterations per source:", its, "reliable updates:", [i.reliable_updates for i in infos])
    assert max(its) < 1.2 * min(its)  # same operator, same spectrum: counts differ by a few per cent
    phi128 = phi.astype(np.complex128)
    for j in (0, nsrc - 1):
        xj = x[j].cpu().numpy()
        res = rel(orc.apply_MdagM(phi128, xj, cfg["m"], cfg["g"], cfg["rho"]), b[j].astype(np.complex128))
        assert res <= cfg["tol"], (j, res)
        assert abs(res - infos[j].rel_residual_true) <= 0.02 * cfg["tol"]


def test_batched_solve_equals_single_solves(wz, inp):
    """Lock-step batching does not couple the sources: same iteration counts and the same x,
    bit for bit, as solving each source alone (fixed-order reductions per source)."""
    cfg = inp.CONFIGS[3]
    dims = cfg["dims"]
    phi = torch.from_numpy(inp.make_phi(cfg["seed"], dims, cfg["sigma"], np.complex64)).cuda()
    b = torch.from_numpy(inp.make_sources(cfg["seed"], 3, dims, np.complex64)).cuda()
    plan = wz.Plan(dims, "c64", 3)
    xb, ib = plan.cg_solve(phi, b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 400, raise_on_fail=False)
    for j in range(3):
        xs, i1 = plan.cg_solve(phi, b[j:j + 1].contiguous(), cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 400,
                               raise_on_fail=False)
        assert i1[0].iterations == ib[j].iterations == 400
        assert i1[0].reliable_updates == ib[j].reliable_updates
        assert torch.equal(xs[0], xb[j])


@pytest.mark.parametrize("key", ["5a", "5b"])
def test_config5_solve_true_residual(wz, orc, inp, key):
    """Config 5 (48x24^3 mixed radix 2/3, and 64^4): one Gaussian source solved to 1e-6 in
    complex64 with reliable updates; the ORACLE recomputes the true residual of the GPU's x
    (naive-DFT route at 48x24^3, radix-2 route at 64^4)."""
    cfg = inp.CONFIGS[key]
    dims = cfg["dims"]
    phi = inp.make_phi(cfg["seed"], dims, cfg["sigma"], np.complex64)
    b = inp.make_source(cfg["seed"], 0, dims, np.complex64)
    plan = wz.Plan(dims, "c64", 1)
    x, infos = plan.cg_solve(torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda(), cfg["m"], cfg["g"],
                             cfg["rho"], cfg["tol"], 200000)
    info = infos[0]
    print("config %s: iterations %d, reliable updates %d, true residual %.3e"
          % (key, info.iterations, info.reliable_updates, info.rel_residual_true))
    assert info.converged and info.rel_residual_true <= cfg["tol"] and info.reliable_updates >= 1
    xh = x.cpu().numpy()
    del plan, x
    res = rel(orc.apply_MdagM(phi.astype(np.complex128), xh, cfg["m"], cfg["g"], cfg["rho"]),
              b.astype(np.complex128))
    assert res <= cfg["tol"], res
    assert abs(res - info.rel_residual_true) <= 0.02 * cfg["tol"]


# ---- NEXT-1: free-inverse preconditioning ----

@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 4, 16, 8), (16, 16, 16, 16), (48, 24, 24, 24)])
@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_M0inv_and_MtdagMt_vs_oracle(wz, orc, inp, dims, dtype):
    phi, b = _fields(inp, dims, dtype, nsrc=2)
    m, g, rho = 0.3 + 0.1j, 0.4 - 0.2j, 1.0
    plan = wz.Plan(dims, dtype, 2)
    d_b, d_phi = torch.from_numpy(b).cuda(), torch.from_numpy(phi).cuda()
    b128, phi128 = b.astype(np.complex128), phi.astype(np.complex128)
    for dagger in (False, True):
        out = plan.apply_M0inv(d_b, m, rho, dagger).cpu().numpy()
        ref = np.stack([orc.apply_M0inv(dims, b128[j], m, rho, dagger) for j in range(2)])
        assert rel(out, ref) <= TOL[dtype]
    out = plan.apply_MtdagMt(d_phi, d_b, m, g, rho).cpu().numpy()
    ref = np.stack([orc.apply_Mtilde(phi128, orc.apply_Mtilde(phi128, b128[j], m, g, rho), m, g, rho, dagger=True)
                    for j in range(2)])
    assert rel(out, ref) <= TOL[dtype]


@pytest.mark.parametrize("dims,dtype,tol", [((8, 8, 8, 8), "c128", 1e-12), ((8, 8, 8, 8), "c64", 1e-6),
                                            ((16, 16, 16, 16), "c64", 1e-6)])
def test_cg_pc_weak_coupling_like_table_VI(wz, orc, inp, dims, dtype, tol):
    """Table VI regime (m = 1, g = 1/5): the preconditioned solve converges in 8 (1e-6) to 15 (1e-12)
    iterations; counts within +-2 of the oracle's, true residual of the ORIGINAL system recomputed
    by the oracle."""
    m, g, rho = 1.0, 0.2, 1.0
    phi = inp.make_phi(5, dims, 0.5, NPDT[dtype])
    b = inp.make_sources(5, 2, dims, NPDT[dtype])
    plan = wz.Plan(dims, dtype, 2)
    x, infos = plan.cg_solve(torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda(), m, g, rho, tol, 2000,
                             precondition=True)
    x = x.cpu().numpy()
    phi128 = phi.astype(np.complex128)
    for j in range(2):
        bj = b[j].astype(np.complex128)
        xo, io = orc.cg_pc(phi128, bj, m, g, rho, tol, 2000)
        true_res = rel(orc.apply_MdagM(phi128, x[j], m, g, rho), bj)
        print("pc %s %s: iterations gpu=%d oracle=%d true residual %.2e (oracle %.2e)"
              % (dims, dtype, infos[j].iterations, io.iterations, true_res, io.rel_residual_true))
        assert infos[j].converged and io.converged
        assert abs(infos[j].iterations - io.iterations) <= 2
        assert infos[j].iterations <= 25
        assert abs(true_res - infos[j].rel_residual_true) <= 0.05 * max(true_res, tol)
        assert true_res <= 20 * tol  # original-system residual: same order as the preconditioned one
        assert rel(x[j], xo) <= (1e-9 if dtype == "c128" else 1e-4)


def test_cg_pc_strong_coupling_config2(wz, orc, inp):
    """Config 2 parameters (g sigma = 0.3, m = 0.05): preconditioning still has to give the same x."""
    cfg = inp.CONFIGS[2]
    dims = cfg["dims"]
    phi = inp.make_phi(cfg["seed"], dims, cfg["sigma"])
    b = inp.make_source(cfg["seed"], 0, dims)
    plan = wz.Plan(dims, "c128", 1)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    x0, i0 = plan.cg_solve(d_phi, d_b, cfg["m"], cfg["g"], 1.0, 1e-10, 20000)
    x1, i1 = plan.cg_solve(d_phi, d_b, cfg["m"], cfg["g"], 1.0, 1e-10, 20000, precondition=True)
    print("config 2: plain %d iterations, preconditioned %d" % (i0[0].iterations, i1[0].iterations))
    res = rel(orc.apply_MdagM(phi, x1.cpu().numpy(), cfg["m"], cfg["g"], 1.0), b)
    assert i1[0].converged and res <= 1e-7
    assert rel(x1.cpu().numpy(), x0.cpu().numpy()) <= 1e-6


# ---- NEXT-4: locality probe ----

@pytest.mark.parametrize("dims,dtype", [((16, 16, 16, 16), "c128"), ((16, 16, 16, 16), "c64"), ((8, 4, 16, 8), "c128")])
def test_locality_profile_vs_oracle(wz, orc, dims, dtype):
    plan = wz.Plan(dims, dtype, 1)
    for spin in (0, 3):
        f = np.array(plan.locality_profile(spin))
        fo, psio = orc.locality_profile(dims, spin)
        assert f.shape == fo.shape
        assert f[0] <= (1e-12 if dtype == "c128" else 1e-5)          # Fig. 1: f(0) = 0
        assert np.max(np.abs(f[1:] - fo[1:]) / fo[1:]) <= (1e-11 if dtype == "c128" else 1e-4)
    eta = torch.zeros((4,) + tuple(dims), dtype=plan.tdtype, device="cuda")
    eta[2, 0, 0, 0, 0] = 1.0
    psi = plan.apply_Dslash(eta).cpu().numpy()
    assert rel(psi, orc.locality_profile(dims, 2)[1]) <= TOL[dtype]


# ---- NEXT-2 (first step): shifted system (Eq. 7.13) ----

@pytest.mark.parametrize("dims,dtype,tol", [((8, 8, 8, 8), "c128", 1e-10), ((8, 4, 16, 8), "c128", 1e-10),
                                            ((8, 8, 8, 8), "c64", 1e-6), ((16, 16, 16, 16), "c64", 1e-6)])
def test_cg_shift_vs_oracle(wz, orc, inp, dims, dtype, tol):
    """(M^dag M + sigma) x = b over a ladder of shifts: iteration counts within +-2 of the oracle's
    (1% for long solves), solution against the oracle's, true residual of the SHIFTED system
    recomputed by the oracle; iterations fall as sigma grows."""
    m, g, rho = 0.05, 1.0, 1.0
    phi = inp.make_phi(6, dims, 0.3, NPDT[dtype])
    b = inp.make_sources(6, 2, dims, NPDT[dtype])
    plan = wz.Plan(dims, dtype, 2)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    phi128 = phi.astype(np.complex128)
    its = []
    for sigma in (0.01, 1.0, 100.0):
        x, infos = plan.cg_solve(d_phi, d_b, m, g, rho, tol, 20000, sigma=sigma)
        x = x.cpu().numpy()
        for j in range(2):
            bj = b[j].astype(np.complex128)
            # complex64 plans follow reading G9: compare with the oracle's complex64 + reliable-update loop
            if dtype == "c128":
                xo, io = orc.cg_shift(phi128, bj, m, g, sigma, rho, tol, 20000)
            else:
                xo, io = orc.cg_c64ru(phi128, bj, m, g, rho, tol, 20000, sigma=sigma)
            true_res = rel(orc.apply_MdagM(phi128, x[j], m, g, rho) + sigma * x[j], bj)
            print("shift %g %s %s: iterations gpu=%d oracle=%d true residual %.2e"
                  % (sigma, dims, dtype, infos[j].iterations, io.iterations, true_res))
            assert infos[j].converged and io.converged
            # G10: near the stop the oracle's residual hovers within +-30 % of tol for several iterations
            # (measured here at sigma = 1: 1.31, 1.41, 1.28, 1.44, 0.93 x tol), and its own count moves with
            # the OpenMP thread count (492 on one box, 491 on the next; GPU 496 on both): bind complex128 at
            # max(2, 2 %) AND require the oracle to be at the threshold where the GPU stopped
            bound = max(2, io.iterations // 50) if dtype == "c128" else max(2, io.iterations // 20)
            assert abs(infos[j].iterations - io.iterations) <= bound
            if dtype == "c128":
                k = min(infos[j].iterations, len(io.history) - 1)
                assert min(io.history[max(0, k - 2):k + 3]) <= 2.0 * tol
            assert true_res <= tol * (1.0 + 1e-3)
            assert abs(true_res - infos[j].rel_residual_true) <= 0.05 * tol
            assert rel(x[j], xo) <= (1e-7 if dtype == "c128" else 5e-4)
        its.append(infos[0].iterations)
    assert its[0] > its[1] > its[2]


def test_cg_shift_zero_is_plain_solve_and_errors(wz, inp):
    dims = (8, 8, 8, 8)
    phi = inp.make_phi(6, dims, 0.3)
    b = inp.make_sources(6, 1, dims)
    plan = wz.Plan(dims, "c128", 1)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    x0, i0 = plan.cg_solve(d_phi, d_b, 0.05, 1.0, 1.0, 1e-10, 20000)
    x1, i1 = plan.cg_solve(d_phi, d_b, 0.05, 1.0, 1.0, 1e-10, 20000, sigma=0.0)
    assert i0[0].iterations == i1[0].iterations and torch.equal(x0, x1)
    with pytest.raises(wz.WZError) as e:
        plan.cg_solve(d_phi, d_b, 0.05, 1.0, 1.0, 1e-10, 100, sigma=-1.0)
    assert e.value.status == wz.WZ_EINVAL


# ---- NEXT-2 (second step): preconditioned shifted system and the rational sum
#      (Eq. 7.14; 877-892 Eq. 7.6-7.7; 948-950 cutoff rule; Table VII) ----

@pytest.mark.parametrize("dims,dtype,tol", [((8, 8, 8, 8), "c128", 1e-10), ((8, 4, 16, 8), "c128", 1e-12),
                                            ((8, 8, 8, 8), "c64", 1e-6), ((16, 16, 16, 16), "c64", 1e-6),
                                            ((48, 24, 24, 24), "c64", 1e-6)])
def test_cg_shift_pc_vs_oracle(wz, orc, inp, dims, dtype, tol):
    """Eq. 7.14 at weak coupling (m = 1, g = 1/5) over a ladder of shifts: iteration counts against the
    oracle's literal composition (+-2; 5 % for complex64, G10), solution, and the true residual of the
    shifted ORIGINAL system (M^dag M + sigma) x = b recomputed by the oracle."""
    m, g, rho = 1.0, 0.2, 1.0
    phi = inp.make_phi(8, dims, 0.5, NPDT[dtype])
    b = inp.make_sources(8, 2, dims, NPDT[dtype])
    plan = wz.Plan(dims, dtype, 2)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    phi128 = phi.astype(np.complex128)
    nchk = 1 if dims[0] == 48 else 2  # the oracle's naive DFT at 48x24^3 takes ~13 s per solve: one source there
    for sigma in (0.01, 1.0, 100.0):
        x, infos = plan.cg_solve(d_phi, d_b, m, g, rho, tol, 2000, precondition=True, sigma=sigma)
        x = x.cpu().numpy()
        for j in range(nchk):
            bj = b[j].astype(np.complex128)
            xo, io = orc.cg_shift_pc(phi128, bj, m, g, sigma, rho, tol, 2000)
            true_res = rel(orc.apply_MdagM(phi128, x[j], m, g, rho) + sigma * x[j], bj)
            print("shift-pc %g %s %s: iterations gpu=%d oracle=%d true residual %.2e (oracle %.2e)"
                  % (sigma, dims, dtype, infos[j].iterations, io.iterations, true_res, io.rel_residual_true))
            assert infos[j].converged and io.converged
            bound = 2 if dtype == "c128" else max(2, io.iterations // 20)
            assert abs(infos[j].iterations - io.iterations) <= bound
            assert abs(true_res - infos[j].rel_residual_true) <= 0.05 * max(true_res, tol)
            assert true_res <= 20 * tol
            assert rel(x[j], xo) <= (1e-8 if dtype == "c128" else 1e-4)


def test_cg_shift_pc_special_cases_and_errors(wz, orc, inp):
    cfg = inp.CONFIGS[2]
    dims = cfg["dims"]
    phi = inp.make_phi(cfg["seed"], dims, cfg["sigma"])
    b = inp.make_sources(cfg["seed"], 1, dims)
    plan = wz.Plan(dims, "c128", 1)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    # sigma = 0 is the preconditioned solve, bit for bit
    x0, i0 = plan.cg_solve(d_phi, d_b, 1.0, 0.2, 1.0, 1e-10, 2000, precondition=True)
    x1, i1 = plan.cg_solve(d_phi, d_b, 1.0, 0.2, 1.0, 1e-10, 2000, precondition=True, sigma=0.0)
    assert i0[0].iterations == i1[0].iterations and torch.equal(x0, x1)
    # strong coupling (config 2): Eq. 7.14 and Eq. 7.13 have the same solution
    xa, ia = plan.cg_solve(d_phi, d_b, cfg["m"], cfg["g"], 1.0, 1e-10, 20000, sigma=0.5)
    xb, ib = plan.cg_solve(d_phi, d_b, cfg["m"], cfg["g"], 1.0, 1e-10, 20000, precondition=True, sigma=0.5)
    print("config 2, sigma 0.5: plain %d iterations, preconditioned %d" % (ia[0].iterations, ib[0].iterations))
    assert ib[0].converged and rel(xb.cpu().numpy(), xa.cpu().numpy()) <= 1e-7
    # g = 0, sigma = 0: the operator is the identity, one iteration
    _, i2 = plan.cg_solve(d_phi, d_b, 1.0, 0.0, 1.0, 1e-10, 100, precondition=True, sigma=0.0)
    assert i2[0].iterations == 1
    for kw in (dict(sigma=-1.0, precondition=True), dict(sigma=float("nan"), precondition=True)):
        with pytest.raises(wz.WZError) as e:
            plan.cg_solve(d_phi, d_b, 1.0, 0.2, 1.0, 1e-10, 100, **kw)
        assert e.value.status == wz.WZ_EINVAL
    with pytest.raises(wz.WZError) as e:  # M0 must be invertible
        plan.cg_solve(d_phi, d_b, 0.0, 0.2, 1.0, 1e-10, 100, precondition=True, sigma=1.0)
    assert e.value.status == wz.WZ_EINVAL


@pytest.mark.parametrize("dims,dtype,tol", [((8, 8, 8, 8), "c128", 1e-12), ((16, 16, 16, 16), "c64", 1e-6)])
def test_rational_apply_vs_oracle(wz, orc, inp, dims, dtype, tol):
    """Eq. 7.6 with d = 20 shifts at Table VII's parameters (m = 1, g = 0.1), preconditioned up to
    beta = 100: the sum against the oracle's, per-shift iteration counts against the oracle's, and the
    paper's caps (under 100 iterations per problem in single, under 200 in double precision)."""
    m, g, rho = 1.0, 0.1, 1.0
    phi = inp.make_phi(9, dims, 0.5, NPDT[dtype])
    eta = inp.make_sources(9, 2, dims, NPDT[dtype])
    a0, al, be = inp.rational_ladder(20, 1e-2, 1e3)
    plan = wz.Plan(dims, dtype, 2)
    out, infos = plan.rational_apply(torch.from_numpy(phi).cuda(), torch.from_numpy(eta).cuda(), m, g, a0, al, be,
                                     rho, tol, 1000)
    out = out.cpu().numpy()
    phi128 = phi.astype(np.complex128)
    cap = 200 if dtype == "c128" else 100
    total = 0
    for j in range(2):
        ref, oinfos = orc.rational_apply(phi128, eta[j].astype(np.complex128), m, g, a0, al, be, rho, tol, 1000)
        assert rel(out[j], ref) <= (1e-10 if dtype == "c128" else 2e-6)
        for i in range(20):
            gi, oi = infos[i][j], oinfos[i]
            assert gi.converged and oi.converged and gi.iterations < cap
            if dtype == "c128" or be[i] <= 100.0:  # plain complex64 solves follow G9's loop, not this oracle's
                assert abs(gi.iterations - oi.iterations) <= max(2, oi.iterations // 20), (i, gi.iterations, oi.iterations)
            total += gi.iterations
    print("rational sum %s %s: %d iterations over 20 shifts x 2 sources" % (dims, dtype, total))
    # the plain branch alone and the preconditioned branch alone give the same sum
    out_np, _ = plan.rational_apply(torch.from_numpy(phi).cuda(), torch.from_numpy(eta).cuda(), m, g, a0, al, be,
                                    rho, tol, 5000, pc_cutoff=-1.0)
    assert rel(out_np.cpu().numpy(), out) <= (1e-9 if dtype == "c128" else 1e-5)


def test_rational_apply_edge_cases(wz, inp):
    dims = (4, 4, 4, 4)
    phi = inp.make_phi(9, dims, 0.5)
    eta = inp.make_sources(9, 1, dims)
    plan = wz.Plan(dims, "c128", 1)
    d_phi, d_eta = torch.from_numpy(phi).cuda(), torch.from_numpy(eta).cuda()
    out, infos = plan.rational_apply(d_phi, d_eta, 1.0, 0.1, 0.75, [], [], 1.0, 1e-10, 100)  # no shifts: alpha0 eta
    assert infos == [] and rel(out.cpu().numpy(), 0.75 * eta) <= 1e-15
    with pytest.raises(wz.WZError) as e:
        plan.rational_apply(d_phi, d_eta, 1.0, 0.1, 0.0, [1.0], [-2.0], 1.0, 1e-10, 100)
    assert e.value.status == wz.WZ_EINVAL


# ---- NEXT-3: mixed precision to double-precision tolerances ----

@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (16, 16, 16, 16)])
def test_mixed_precision_solve_to_double_tolerance(wz, orc, inp, dims):
    """single precision 'could however be used for a mixed precision conjugate gradient'.
    A WZ_C64 plan iterates in complex64 and corrects with complex128 reliable updates (reading G9), so it
    reaches the double-precision tolerance 1e-10: true residual recomputed by the oracle, solution against
    the complex128 oracle, iteration count against the oracle's complex64 + reliable-update loop (5 %)."""
    m, g, rho, tol = 0.05, 1.0, 1.0, 1e-10
    phi = inp.make_phi(2, dims, 0.3, np.complex64)
    b = inp.make_sources(2, 1, dims, np.complex64)
    plan = wz.Plan(dims, "c64", 1)
    x, infos = plan.cg_solve(torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda(), m, g, rho, tol, 50000)
    x = x.cpu().numpy()[0]
    phi128, b128 = phi.astype(np.complex128), b[0].astype(np.complex128)
    Xo, io = orc.cg_c64ru(phi128, b128, m, g, rho, tol, 50000)
    xd, idb = orc.cg(phi128, b128, m, g, rho, tol, 50000)
    true_res = rel(orc.apply_MdagM(phi128, x, m, g, rho), b128)
    print("mixed precision %s: iterations gpu=%d (reliable updates %d) oracle c64ru=%d (%d) oracle c128=%d true residual %.2e"
          % (dims, infos[0].iterations, infos[0].reliable_updates, io.iterations, io.reliable_updates, idb.iterations, true_res))
    assert infos[0].converged and io.converged
    assert true_res <= tol * (1.0 + 1e-3)
    assert abs(infos[0].iterations - io.iterations) <= max(2, io.iterations // 20)
    assert rel(x, xd) <= 1e-8 and rel(x, Xo) <= 1e-8


# ---- the NEXT kernels in the launch configuration bench.py times (32^4 complex64: P23_MULTPC, fwdcg_s / endcg_s
#      with the (x2,x3) volume compiled in) against the oracle (Tables VI, VII) ----

def test_pc_and_shifted_solves_at_32x4_vs_oracle(wz, orc, inp):
    dims = (32, 32, 32, 32)
    phi = inp.make_phi(4, dims, 0.5, np.complex64)
    b = inp.make_sources(4, 1, dims, np.complex64)
    plan = wz.Plan(dims, "c64", 1)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    phi128, b128 = phi.astype(np.complex128), b[0].astype(np.complex128)
    tol = 1e-6
    # Table VI parameters: 8 iterations in single precision (tests/golden/table_VI_pc_iterations.txt)
    x, infos = plan.cg_solve(d_phi, d_b, 1.0, 0.2, 1.0, tol, 500, precondition=True)
    xo, io = orc.cg_pc(phi128, b128, 1.0, 0.2, 1.0, tol, 500)
    print("32^4 pc: iterations gpu=%d oracle=%d, true residual gpu %.2e oracle %.2e"
          % (infos[0].iterations, io.iterations, infos[0].rel_residual_true, io.rel_residual_true))
    assert infos[0].converged and io.converged and abs(infos[0].iterations - io.iterations) <= 2
    assert 6 <= infos[0].iterations <= 10
    assert rel(x.cpu().numpy()[0], xo) <= 1e-4
    # Table VII parameters (m = 1, g = 0.1): Eq. 7.14 below the cutoff, Eq. 7.13 above it
    for sigma, pc in ((0.5, True), (20.0, True), (300.0, False)):
        x, infos = plan.cg_solve(d_phi, d_b, 1.0, 0.1, 1.0, tol, 2000, precondition=pc, sigma=sigma)
        if pc:
            xo, io = orc.cg_shift_pc(phi128, b128, 1.0, 0.1, sigma, 1.0, tol, 2000)
        else:
            xo, io = orc.cg_c64ru(phi128, b128, 1.0, 0.1, 1.0, tol, 2000, sigma=sigma)
        xg = x.cpu().numpy()[0]
        true_res = rel(orc.apply_MdagM(phi128, xg, 1.0, 0.1, 1.0) + sigma * xg, b128)
        print("32^4 sigma=%g pc=%d: iterations gpu=%d oracle=%d true residual %.2e"
              % (sigma, pc, infos[0].iterations, io.iterations, true_res))
        assert infos[0].converged and io.converged
        assert abs(infos[0].iterations - io.iterations) <= max(2, io.iterations // 20)
        assert infos[0].iterations < 100  # under 100 iterations per problem in single precision
        assert abs(true_res - infos[0].rel_residual_true) <= 0.05 * max(true_res, tol)
        assert true_res <= (20 * tol if pc else tol * (1 + 1e-3))
        assert rel(xg, xo) <= 1e-4


@pytest.mark.parametrize("dims", [(32, 8, 8, 8), (32, 16, 16, 16)])
@pytest.mark.parametrize("dtype,tol,want", [("c64", 1e-6, 8), ("c128", 1e-12, 15)])
def test_paper_lattices_table_VI(wz, orc, inp, dims, dtype, tol, want):
    """The paper's own lattices 8^3x32 and 16^3x32 at Table VI's parameters (m = 1, g = 1/5, Gaussian b;
    PAPER.md:935-944): the preconditioned solve takes the 8 (single) / 15 (double) iterations the paper
    prints (tests/golden/table_VI_pc_iterations.txt), the plain solve is compared with the oracle's."""
    m, g, rho = 1.0, 0.2, 1.0
    phi = inp.make_phi(5, dims, 0.5, NPDT[dtype])
    b = inp.make_sources(5, 1, dims, NPDT[dtype])
    plan = wz.Plan(dims, dtype, 1)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    phi128, b128 = phi.astype(np.complex128), b[0].astype(np.complex128)
    x, infos = plan.cg_solve(d_phi, d_b, m, g, rho, tol, 2000, precondition=True)
    xo, io = orc.cg_pc(phi128, b128, m, g, rho, tol, 2000)
    print("%s %s pc: iterations gpu=%d oracle=%d (Table VI: %d)" % (dims, dtype, infos[0].iterations, io.iterations, want))
    assert infos[0].converged and abs(infos[0].iterations - io.iterations) <= 2
    assert abs(infos[0].iterations - want) <= 1
    assert rel(x.cpu().numpy()[0], xo) <= (1e-9 if dtype == "c128" else 1e-4)
    # plain solve: the paper needed 830-1800 iterations at these parameters with its phi ensemble
    x, infos = plan.cg_solve(d_phi, d_b, m, g, rho, tol, 20000)
    if dtype == "c128":
        xo, io = orc.cg(phi128, b128, m, g, rho, tol, 20000)
    else:
        xo, io = orc.cg_c64ru(phi128, b128, m, g, rho, tol, 20000)
    xg = x.cpu().numpy()[0]
    true_res = rel(orc.apply_MdagM(phi128, xg, m, g, rho), b128)
    print("%s %s plain: iterations gpu=%d oracle=%d true residual %.2e" % (dims, dtype, infos[0].iterations, io.iterations, true_res))
    assert infos[0].converged and true_res <= tol * (1 + 1e-3)
    assert abs(infos[0].iterations - io.iterations) <= max(2, int(0.05 * io.iterations))


def test_paper_lattice_32x3x64_MdagM(wz, orc, inp):
    """32^3x64, the largest lattice of Tables V-VII: one M^dag M in both precisions against the oracle."""
    dims = (64, 32, 32, 32)
    for dtype in ("c64", "c128"):
        phi = inp.make_phi(5, dims, 0.5, NPDT[dtype])
        b = inp.make_source(5, 0, dims, NPDT[dtype])
        plan = wz.Plan(dims, dtype, 1)
        out = plan.apply_MdagM(torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda(), 1.0, 0.2, 1.0).cpu().numpy()
        del plan
        ref = orc.apply_MdagM(phi.astype(np.complex128), b.astype(np.complex128), 1.0, 0.2, 1.0)
        assert rel(out, ref) <= TOL[dtype]


# ---- config 4 source 0 against the oracle's full solve (SURVEY 8(d) "Oracle timed beside it") ----

def _read_golden_solve(name):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    vals, hist = {}, []
    with open(path) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            w = line.split()
            if w[0] == "history":
                hist.append((int(w[1]), float(w[2])))
            else:
                vals[w[0]] = float(w[1])
    return vals, hist


def test_config4_source0_vs_oracle_full_solve(wz, inp):
    """The headline workload's iteration count and residual history against the oracle's O4' loop run to
    convergence on the same source (tests/golden/config4_src0_oracle.txt, written by
    tests/golden/make_config4_src0.py from oracle/ alone): count within 5 % (G10), and the GPU's residual
    history lies on the oracle's convergence curve."""
    vals, hist = _read_golden_solve("config4_src0_oracle.txt")
    assert vals["converged"] == 1 and vals["rel_residual_true"] <= 1e-6
    cfg = inp.CONFIGS[4]
    dims = cfg["dims"]
    phi = inp.make_phi(cfg["seed"], dims, cfg["sigma"], np.complex64)
    b = inp.make_sources(cfg["seed"], 1, dims, np.complex64)
    plan = wz.Plan(dims, "c64", 1)
    x, infos = plan.cg_solve(torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda(), cfg["m"], cfg["g"], cfg["rho"],
                             cfg["tol"], 100000)
    info = infos[0]
    n_or = int(vals["iterations"])
    print("config 4 source 0: iterations gpu=%d oracle=%d (%+.2f %%), reliable updates gpu=%d oracle=%d"
          % (info.iterations, n_or, 100.0 * (info.iterations - n_or) / n_or, info.reliable_updates,
             int(vals["reliable_updates"])))
    assert info.converged and info.rel_residual_true <= cfg["tol"]
    assert abs(info.iterations - n_or) <= 0.05 * n_or
    assert abs(info.reliable_updates - vals["reliable_updates"]) <= 3
    # history shape: at the iterations the host sampled, log10 of the residual against the oracle's curve
    # (interpolated in log space between its stored points); both oscillate by +-30 % per iteration, and the
    # curves shift against each other by the few per cent the counts differ
    ks = np.array([k for k, _ in hist], dtype=np.float64)
    lr = np.log10(np.array([r for _, r in hist]))
    gh = plan.cg_history(0)
    assert len(gh) > 100
    dev = []
    for k, r in gh:
        if k < 50 or k > 0.9 * min(info.iterations, n_or) or r <= 0:
            continue
        dev.append(abs(np.log10(r) - np.interp(k, ks, lr)))
    dev = np.array(dev)
    print("history: %d samples, median |dlog10| %.3f, max %.3f" % (len(dev), np.median(dev), dev.max()))
    assert np.median(dev) <= 0.15 and dev.max() <= 0.6


# ---- CUDA graph replay of the iteration chunks (north star iii) and host-side argument checks ----

@pytest.mark.parametrize("dims,dtype", [((8, 8, 8, 8), "c128"), ((16, 16, 16, 16), "c64")])
def test_graph_replay_equals_stream_launches(wz, inp, dims, dtype):
    phi = torch.from_numpy(inp.make_phi(3, dims, 0.5, NPDT[dtype])).cuda()
    b = torch.from_numpy(inp.make_sources(3, 2, dims, NPDT[dtype])).cuda()
    plan = wz.Plan(dims, dtype, 2)
    tol = 1e-10 if dtype == "c128" else 1e-6
    res = {}
    plan.cg_solve(phi, b, 0.05, 1.0, 1.0, tol, 8, raise_on_fail=False)  # the plan's first solve also builds its c(p) table (one launch)
    for on in (True, False, True):
        plan.set_graph(on)
        plan.reset_launch_count()
        x, infos = plan.cg_solve(phi, b, 0.05, 1.0, 1.0, tol, 100000)
        res.setdefault(on, []).append((x.clone(), [(i.iterations, i.reliable_updates, i.rel_residual_true) for i in infos],
                                       plan.launch_count))
    (xg, ig, lg), (xg2, ig2, lg2) = res[True]
    (xs, is_, ls), = res[False]
    assert ig == is_ == ig2 and torch.equal(xg, xs) and torch.equal(xg, xg2)
    assert lg == ls == lg2 and lg >= 5 * max(i[0] for i in ig)  # replayed launches are counted
    # other arguments -> a new capture, same results as stream launches
    plan.set_graph(True)
    xa, ia = plan.cg_solve(phi, b, 0.05, 1.0, 1.0, tol, 100000, sigma=0.5)
    plan.set_graph(False)
    xb, ib = plan.cg_solve(phi, b, 0.05, 1.0, 1.0, tol, 100000, sigma=0.5)
    assert torch.equal(xa, xb) and [i.iterations for i in ia] == [i.iterations for i in ib]
    h = plan.cg_history(1)
    assert h[0][0] > 0 and h[-1][0] == ib[1].iterations and h[-1][1] <= tol * 1.01
    assert all(h[i][0] < h[i + 1][0] for i in range(len(h) - 1))


def test_binding_rejects_mismatched_buffers(wz, inp):
    dims = (4, 4, 4, 4)
    plan = wz.Plan(dims, "c128", 3)
    phi = torch.from_numpy(inp.make_phi(1, dims, 0.3)).cuda()
    b3 = torch.from_numpy(inp.make_sources(1, 3, dims)).cuda()
    one = torch.empty_like(b3[0])
    with pytest.raises(ValueError):
        plan.fft4d(b3, +1, True, out=one)  # three spinors in, room for one out
    with pytest.raises(ValueError):
        plan.apply_M(phi, b3, 0.1, 0.5, 1.0, False, out=one)
    with pytest.raises(ValueError):
        plan.cg_solve(phi, b3, 0.1, 0.5, out=torch.empty_like(one))
    with pytest.raises(ValueError):
        plan.fft4d(b3.cpu(), +1, True)
    b1 = b3[:1].contiguous()
    with pytest.raises(wz.WZError) as e:  # x must not alias b
        plan.cg_solve(phi, b1, 0.1, 0.5, out=b1)
    assert e.value.status == wz.WZ_EINVAL
    with pytest.raises(wz.WZError) as e:
        plan.rational_apply(phi, b1, 0.1, 0.5, 0.0, [1.0], [1.0], out=b1)
    assert e.value.status == wz.WZ_EINVAL


def test_second_device(wz, orc, inp):
    """A plan on cuda:1 in a process that already used cuda:0 (the twiddle tables are per-device constant
    memory): FFT and M^dag M against the oracle.  Needs two GPUs."""
    if torch.cuda.device_count() < 2:
        pytest.skip("one GPU")
    dims = (8, 8, 8, 8)
    phi, b = _fields(inp, dims, "c128")
    wz.Plan(dims, "c128", 1, "cuda:0").fft4d(torch.from_numpy(b).to("cuda:0"), +1, True)
    plan = wz.Plan(dims, "c128", 1, "cuda:1")
    d_b, d_phi = torch.from_numpy(b).to("cuda:1"), torch.from_numpy(phi).to("cuda:1")
    assert torch.cuda.current_device() == 0
    f = plan.fft4d(d_b, +1, True).cpu().numpy()
    assert rel(f, orc.dft4d(b[0], +1, True)[None]) <= 1e-12
    q = plan.apply_MdagM(d_phi, d_b, 0.05, 1.0, 1.0).cpu().numpy()
    assert rel(q[0], orc.apply_MdagM(phi, b[0], 0.05, 1.0, 1.0)) <= 1e-12
    with pytest.raises(ValueError):
        plan.fft4d(torch.from_numpy(b).to("cuda:0"), +1, True)


# ---- NEXT-2, second half: multi-shift CG (oracle O8; Eq. 7.6-7.7, 927-931 Eq. 7.13) ----

@pytest.mark.parametrize("dims,dtype,tol", [((8, 8, 8, 8), "c128", 1e-10), ((8, 4, 16, 8), "c128", 1e-12),
                                            ((8, 8, 8, 8), "c64", 1e-6), ((16, 16, 16, 16), "c64", 1e-6)])
def test_cg_multishift_vs_oracle(wz, orc, inp, dims, dtype, tol):
    """All shifts from one Krylov space: per shift the iteration at which it froze against the oracle's
    multi-shift loop (complex128; complex64 plans add their polishing iterations, so only a lower bound
    there), the solution against the oracle's, and the true residual of (M^dag M + sigma_i) x_i = b
    recomputed by the oracle.  Shifts unsorted on purpose (the base system is the smallest, wherever it is)."""
    m, g, rho = 0.05, 1.0, 1.0
    sigmas = [1.0, 0.01, 100.0, 0.0, 1e4]
    phi = inp.make_phi(6, dims, 0.3, NPDT[dtype])
    b = inp.make_sources(6, 2, dims, NPDT[dtype])
    plan = wz.Plan(dims, dtype, 2)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    plan.reset_launch_count()
    x, infos = plan.cg_solve_multishift(d_phi, d_b, m, g, sigmas, rho, tol, 20000)
    launches = plan.launch_count
    x = x.cpu().numpy()
    phi128 = phi.astype(np.complex128)
    for j in range(2):
        bj = b[j].astype(np.complex128)
        Xo, io, mv = orc.cg_multishift(phi128, bj, m, g, sigmas, rho, tol, 20000)
        for i, sigma in enumerate(sigmas):
            gi = infos[i][j]
            true_res = rel(orc.apply_MdagM(phi128, x[i, j], m, g, rho) + sigma * x[i, j], bj)
            print("multishift %s %s sigma=%g: iterations gpu=%d (+polish RU %d) oracle=%d true residual %.2e"
                  % (dims, dtype, sigma, gi.iterations, gi.reliable_updates, io[i].iterations, true_res))
            assert gi.converged and io[i].converged
            assert abs(true_res - gi.rel_residual_true) <= 0.05 * tol
            if dtype == "c128":
                assert true_res <= tol * 1.05
                assert abs(gi.iterations - io[i].iterations) <= max(2, int(0.015 * io[i].iterations))
                assert rel(x[i, j], Xo[i]) <= 1e-7
            else:
                assert true_res <= tol * (1 + 1e-3)
                assert gi.iterations >= io[i].iterations - max(2, int(0.05 * io[i].iterations))
                assert rel(x[i, j], Xo[i]) <= 5e-4
    # one matvec per base iteration: far fewer launches than five separate solves
    base_its = max(infos[3][j].iterations for j in range(2))
    assert launches < 12 * base_its + 2000


def test_cg_multishift_single_shift_and_errors(wz, inp):
    dims = (8, 8, 8, 8)
    phi = inp.make_phi(6, dims, 0.3)
    b = inp.make_sources(6, 1, dims)
    plan = wz.Plan(dims, "c128", 1)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    x0, i0 = plan.cg_solve(d_phi, d_b, 0.05, 1.0, 1.0, 1e-10, 20000, sigma=0.5)
    x1, i1 = plan.cg_solve_multishift(d_phi, d_b, 0.05, 1.0, [0.5], 1.0, 1e-10, 20000)
    assert i1[0][0].iterations == i0[0].iterations and torch.equal(x1[0], x0)  # the base system IS wz_cg_solve_shift
    for bad in ([], [-1.0], [0.1] * 33):
        with pytest.raises(wz.WZError) as e:
            plan.cg_solve_multishift(d_phi, d_b, 0.05, 1.0, bad, 1.0, 1e-10, 100)
        assert e.value.status == wz.WZ_EINVAL
    x2, i2 = plan.cg_solve_multishift(d_phi, d_b, 0.05, 1.0, [0.5, 2.0], 1.0, 1e-10, 7, raise_on_fail=False)
    assert i2[0][0].iterations == 7 and not i2[0][0].converged and not i2[1][0].converged


@pytest.mark.parametrize("dims,dtype,tol", [((8, 8, 8, 8), "c128", 1e-12), ((16, 16, 16, 16), "c64", 1e-6)])
def test_rational_apply_multishift_vs_oracle(wz, orc, inp, dims, dtype, tol):
    """Eq. 7.6 with the shifts above the cutoff from one multi-shift solve (and all of them with pc_cutoff < 0):
    the sum against the oracle's one-solve-per-shift sum and against the library's own per-shift mode."""
    m, g, rho = 1.0, 0.1, 1.0
    phi = inp.make_phi(9, dims, 0.5, NPDT[dtype])
    eta = inp.make_sources(9, 2, dims, NPDT[dtype])
    a0, al, be = inp.rational_ladder(20, 1e-2, 1e3)
    plan = wz.Plan(dims, dtype, 2)
    d_phi, d_eta = torch.from_numpy(phi).cuda(), torch.from_numpy(eta).cuda()
    phi128 = phi.astype(np.complex128)
    ref = np.stack([orc.rational_apply(phi128, eta[j].astype(np.complex128), m, g, a0, al, be, rho, tol, 1000)[0]
                    for j in range(2)])
    bound = 1e-10 if dtype == "c128" else 2e-6
    for cutoff in (100.0, -1.0):
        out, infos = plan.rational_apply(d_phi, d_eta, m, g, a0, al, be, rho, tol, 5000, pc_cutoff=cutoff, multishift=True)
        assert all(i.converged for row in infos for i in row)
        assert rel(out.cpu().numpy(), ref) <= bound
        its = [max(i.iterations for i in row) for row in infos]
        print("rational multishift %s %s cutoff %g: iterations per shift %s" % (dims, dtype, cutoff, its))


# ---- every solver path once on the two smallest lattices.  compute-sanitizer is closed on
#      this GPU pool (profiles/r02_sanitizer.md), so the test carries its own checks: the caller's output
#      buffers sit between canary regions (out-of-bounds writes), and every solve is repeated and must
#      reproduce bit for bit (a race in the ticket-counter reductions, the deferred x update or the in-place
#      p / r rewrites would show up as run-to-run differences) ----

def _guarded(shape, dtype, pad=4096):
    """A tensor of `shape` carved out of a larger allocation with canaries on both sides."""
    n = int(np.prod(shape))
    buf = torch.full((n + 2 * pad,), 7.25 - 1.5j, dtype=dtype, device="cuda")
    return buf[pad:pad + n].view(shape), buf, pad


def _canaries_intact(buf, pad):
    v = torch.tensor(7.25 - 1.5j, dtype=buf.dtype, device=buf.device)
    return bool((buf[:pad] == v).all() and (buf[-pad:] == v).all())


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 8, 8, 8)])
def test_small_solves_all_paths(wz, orc, inp, dims):
    m, g, rho = 0.1, 0.5, 1.0
    for dtype, tol in (("c128", 1e-10), ("c64", 1e-6)):
        phi = inp.make_phi(1, dims, 0.3, NPDT[dtype])
        b = inp.make_sources(1, 2, dims, NPDT[dtype])
        phi128 = phi.astype(np.complex128)
        plan = wz.Plan(dims, dtype, 2)
        d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
        cases = {"plain": {}, "pc": {"precondition": True}, "shift": {"sigma": 0.3},
                 "shift_pc": {"precondition": True, "sigma": 0.3}}
        for graph in (True, False):
            plan.set_graph(graph)
            for name, kw in cases.items():
                xg, xbuf, pad = _guarded(b.shape, torch.complex128)
                x, infos = plan.cg_solve(d_phi, d_b, m, g, rho, tol, 5000, out=xg, **kw)
                assert _canaries_intact(xbuf, pad), (dtype, name)
                x2, infos2 = plan.cg_solve(d_phi, d_b, m, g, rho, tol, 5000, **kw)
                assert torch.equal(x, x2) and [i.iterations for i in infos] == [i.iterations for i in infos2]
                sigma = kw.get("sigma", 0.0)
                for j in range(2):
                    xj = x[j].cpu().numpy()
                    res = rel(orc.apply_MdagM(phi128, xj, m, g, rho) + sigma * xj, b[j].astype(np.complex128))
                    assert infos[j].converged and res <= (20 * tol if "pc" in name else tol * (1 + 1e-3)), (dtype, name, res)
                if dtype == "c64" and name == "plain":
                    assert infos[0].reliable_updates >= 1
        xg, xbuf, pad = _guarded((3,) + b.shape, torch.complex128)
        x, infos = plan.cg_solve_multishift(d_phi, d_b, m, g, [0.0, 0.3, 30.0], rho, tol, 5000, out=xg)
        assert _canaries_intact(xbuf, pad)
        x2, _ = plan.cg_solve_multishift(d_phi, d_b, m, g, [0.0, 0.3, 30.0], rho, tol, 5000)
        assert torch.equal(x, x2)
        assert all(i.converged and i.rel_residual_true <= tol * (1 + 1e-3) for row in infos for i in row)
        a0, al, be = inp.rational_ladder(4, 1e-1, 1e2)
        out, _ = plan.rational_apply(d_phi, d_b, m, g, a0, al, be, rho, tol, 5000)
        out2, _ = plan.rational_apply(d_phi, d_b, m, g, a0, al, be, rho, tol, 5000, multishift=True)
        assert rel(out2.cpu().numpy(), out.cpu().numpy()) <= (1e-8 if dtype == "c128" else 1e-4)
        fg, fbuf, pad = _guarded(b.shape, plan.tdtype)
        f = plan.fft4d(d_b, +1, True, out=fg)
        qg, qbuf, qpad = _guarded(b.shape, plan.tdtype)
        plan.apply_MdagM(d_phi, d_b, m, g, rho, out=qg)
        assert _canaries_intact(fbuf, pad) and _canaries_intact(qbuf, qpad)
        assert rel(plan.fft4d(f, -1, True).cpu().numpy(), b.astype(np.complex128)) <= 2 * TOL[dtype]
        assert len(plan.locality_profile(0)) == 1 + sum(d // 2 for d in dims)


# ---- NEXT-3: defect correction, complex64 inner / complex128 outer (oracle O9) ----

@pytest.mark.parametrize("dims,inner_tol", [((8, 8, 8, 8), 1e-3), ((16, 16, 16, 16), 1e-3), ((8, 8, 8, 8), 1e-1)])
def test_cg_dc_vs_oracle(wz, orc, inp, dims, inner_tol):
    """complex64 inner solves restarted inside a complex128 outer loop, to the double-precision tolerance
    1e-10: the same number of outer corrections as the oracle's loop, inner iterations within 5 % (G10),
    true residual recomputed by the oracle, solution against the complex128 oracle; and side by side
    with the reliable-update route of wz_cg_solve to the same tolerance."""
    m, g, rho, tol = 0.05, 1.0, 1.0, 1e-10
    phi = inp.make_phi(2, dims, 0.3, np.complex64)
    b = inp.make_sources(2, 2, dims, np.complex64)
    plan = wz.Plan(dims, "c64", 2)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    x, infos = plan.cg_solve_dc(d_phi, d_b, m, g, rho, tol, inner_tol, 200000)
    xr, iru = plan.cg_solve(d_phi, d_b, m, g, rho, tol, 200000)
    x = x.cpu().numpy()
    phi128 = phi.astype(np.complex128)
    for j in range(2):
        bj = b[j].astype(np.complex128)
        Xo, io = orc.cg_dc(phi128, bj, m, g, rho, tol, inner_tol, 200000)
        true_res = rel(orc.apply_MdagM(phi128, x[j], m, g, rho), bj)
        print("dc %s inner_tol %g: inner iterations gpu=%d oracle=%d, outer gpu=%d oracle=%d, true residual %.2e; "
              "reliable-update route: %d iterations" % (dims, inner_tol, infos[j].iterations, io.iterations,
                                                          infos[j].reliable_updates, io.reliable_updates, true_res,
                                                          iru[j].iterations))
        assert infos[j].converged and io.converged
        assert true_res <= tol * (1 + 1e-3) and abs(true_res - infos[j].rel_residual_true) <= 0.05 * tol
        assert abs(infos[j].reliable_updates - io.reliable_updates) <= 1
        assert abs(infos[j].iterations - io.iterations) <= max(2, int(0.05 * io.iterations))
        assert rel(x[j], Xo) <= 1e-7
    with pytest.raises(wz.WZError) as e:
        wz.Plan(dims, "c128", 1).cg_solve_dc(d_phi.to(torch.complex128), d_b[:1].to(torch.complex128), m, g)
    assert e.value.status == wz.WZ_EINVAL
    with pytest.raises(wz.WZError) as e:
        plan.cg_solve_dc(d_phi, d_b, m, g, rho, tol, 1.5)
    assert e.value.status == wz.WZ_EINVAL


def test_M0inv_at_64x4_complex128(wz, orc, inp):
    """The free inverse where a CTA of the contiguous pass holds only one component pair (64x64 complex128
    planes): off-diagonal launch + accumulating diagonal launch (P23_DIAGPC) against the oracle, both signs."""
    dims = (64, 64, 64, 64)
    b = inp.make_source(5, 0, dims)
    plan = wz.Plan(dims, "c128", 1)
    d_b = torch.from_numpy(b).cuda()
    m = 0.3 + 0.1j
    for dagger in (False, True):
        out = plan.apply_M0inv(d_b, m, 1.0, dagger).cpu().numpy()
        ref = orc.apply_M0inv(dims, b, m, 1.0, dagger)
        assert rel(out, ref) <= TOL["c128"]


# ---- NEXT-3, third form: binary16 storage of the inner solver's vectors (oracle O10) ----

@pytest.mark.parametrize("dims,m,sig,seed", [((8, 8, 8, 8), 0.05, 0.3, 2), ((16, 16, 16, 16), 0.02, 0.5, 3)])
def test_cg_dc_half_storage_vs_oracle(wz, orc, inp, dims, m, sig, seed):
    """Defect correction with t, chi, r, p stored in binary16: true residual recomputed by the oracle <= tol, the
    solution against the complex128 oracle, outer corrections and inner iterations against the oracle's O10 loop
    (a MODEL with fewer roundings: it rounds r, p, chi; the kernels also round the FFT temporary between passes),
    and the first inner solve step by step: the recursive residual after k iterations against O10's."""
    g, rho, tol, itol = 1.0, 1.0, 1e-6, 1e-1
    phi = inp.make_phi(seed, dims, sig, np.complex64)
    b = inp.make_sources(seed, 2, dims, np.complex64)
    plan = wz.Plan(dims, "c64", 2)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    x, infos = plan.cg_solve_dc(d_phi, d_b, m, g, rho, tol, itol, 100000, half_storage=True)
    x64, i64 = plan.cg_solve_dc(d_phi, d_b, m, g, rho, tol, 1e-3, 100000)
    x = x.cpu().numpy()
    phi128 = phi.astype(np.complex128)
    for j in range(2 if dims[0] == 8 else 1):  # one oracle solve at 16^4 (a minute each)
        bj = b[j].astype(np.complex128)
        Xo, io = orc.cg_dc_f16(phi128, bj, m, g, rho, tol, itol, 100000)
        xd, _ = orc.cg(phi128, bj, m, g, rho, 1e-10, 100000)
        true_res = rel(orc.apply_MdagM(phi128, x[j], m, g, rho), bj)
        print("half storage %s: inner iterations gpu=%d oracle(O10)=%d, outer gpu=%d oracle=%d, true residual %.2e; complex64 "
              "defect correction: %d iterations" % (dims, infos[j].iterations, io.iterations, infos[j].reliable_updates,
                                                    io.reliable_updates, true_res, i64[j].iterations))
        assert infos[j].converged and io.converged
        assert true_res <= tol * (1 + 1e-3) and abs(true_res - infos[j].rel_residual_true) <= 0.05 * tol
        assert abs(infos[j].reliable_updates - io.reliable_updates) <= 1
        assert abs(infos[j].iterations - io.iterations) <= 0.2 * io.iterations  # measured: 1 % at 8^4, 2-12 % at 16^4
        assert rel(x[j], xd) <= 1e-3 and rel(x[j], Xo) <= 1e-3  # kappa * tol
    # the first inner solve (first outer step, loose inner tolerance): count of iterations to inner_tol
    _, ik = plan.cg_solve_dc(d_phi, d_b[:1].contiguous(), m, g, rho, 0.5, itol, 100000, half_storage=True)
    _, ok_ = orc.cg_dc_f16(phi128, b[0].astype(np.complex128), m, g, rho, 0.5, itol, 100000)
    print("first inner solve: gpu %d iterations, oracle %d" % (ik[0].iterations, ok_.iterations))
    # (the residual swings by tens of per cent per iteration, so the FIRST crossing of inner_tol moves: 71 vs 86 at 8^4)
    assert ik[0].reliable_updates == ok_.reliable_updates == 1
    assert abs(ik[0].iterations - ok_.iterations) <= max(4, 0.3 * ok_.iterations)
    assert ik[0].rel_residual_true <= 1.3 * itol and ok_.rel_residual_true <= 1.3 * itol


def test_cg_dc_half_storage_errors(wz, inp):
    dims = (8, 4, 16, 8)  # no binary16-storage kernels for this lattice
    phi = torch.from_numpy(inp.make_phi(2, dims, 0.3, np.complex64)).cuda()
    b = torch.from_numpy(inp.make_sources(2, 1, dims, np.complex64)).cuda()
    with pytest.raises(wz.WZError) as e:
        wz.Plan(dims, "c64", 1).cg_solve_dc(phi, b, 0.05, 1.0, 1.0, 1e-6, 1e-1, 100, half_storage=True)
    assert e.value.status == wz.WZ_EUNSUPPORTED


@pytest.mark.parametrize("dims,m,sig,seed", [((8, 8, 8, 8), 0.05, 0.3, 2), ((16, 16, 16, 16), 0.02, 0.5, 3)])
def test_cg_half_storage_reliable_updates_vs_oracle(wz, orc, inp, dims, m, sig, seed):
    """binary16 storage with complex128 reliable updates and rescaling (wz_cg_solve_half against oracle O11): true
    residual recomputed by the oracle, iterations and updates against O11 (10 %) and against the complex64
    solver on the same sources, solution against the complex128 oracle; and the trajectory: the recursive residual
    after k = 1, 2, 5, 20 iterations against O11's (both sides round r, p, chi to binary16; the kernels also round
    the FFT temporary, so agreement is at the 1e-3 level, not bit for bit)."""
    g, rho, tol = 1.0, 1.0, 1e-6
    phi = inp.make_phi(seed, dims, sig, np.complex64)
    b = inp.make_sources(seed, 2, dims, np.complex64)
    plan = wz.Plan(dims, "c64", 2)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b).cuda()
    x, infos = plan.cg_solve(d_phi, d_b, m, g, rho, tol, 100000, half_storage=True)
    x2, infos2 = plan.cg_solve(d_phi, d_b, m, g, rho, tol, 100000, half_storage=True)
    assert torch.equal(x, x2) and [i.iterations for i in infos] == [i.iterations for i in infos2]  # run-to-run
    _, i64 = plan.cg_solve(d_phi, d_b, m, g, rho, tol, 100000)
    x = x.cpu().numpy()
    phi128 = phi.astype(np.complex128)
    for j in range(2 if dims[0] == 8 else 1):  # one oracle solve at 16^4 (a minute each)
        bj = b[j].astype(np.complex128)
        Xo, io = orc.cg_f16ru(phi128, bj, m, g, rho, tol, 100000)
        xd, _ = orc.cg(phi128, bj, m, g, rho, 1e-10, 100000)
        true_res = rel(orc.apply_MdagM(phi128, x[j], m, g, rho), bj)
        print("half storage + reliable updates %s: iterations gpu=%d oracle(O11)=%d, updates gpu=%d oracle=%d, true residual %.2e; "
              "complex64 solver: %d iterations" % (dims, infos[j].iterations, io.iterations, infos[j].reliable_updates,
                                                    io.reliable_updates, true_res, i64[j].iterations))
        assert infos[j].converged and io.converged
        assert true_res <= tol * (1 + 1e-3) and abs(true_res - infos[j].rel_residual_true) <= 0.05 * tol
        # measured: +2 % at 8^4, +4 ... +6 % at 16^4 (the kernels round the FFT temporary between passes, the model does not)
        assert abs(infos[j].iterations - io.iterations) <= max(2, 0.10 * io.iterations)
        assert abs(infos[j].reliable_updates - io.reliable_updates) <= 3
        assert infos[j].iterations <= 1.2 * i64[j].iterations
        assert rel(x[j], xd) <= 1e-3 and rel(x[j], Xo) <= 1e-3  # kappa * tol
    b0 = d_b[:1].contiguous()
    for k in (1, 2, 5, 20):
        _, ik = plan.cg_solve(d_phi, b0, m, g, rho, 1e-30, k, half_storage=True, raise_on_fail=False)
        _, ok_ = orc.cg_f16ru(phi128, b[0].astype(np.complex128), m, g, rho, 1e-30, k)
        dr = abs(ik[0].rel_residual_recursive - ok_.rel_residual_recursive) / ok_.rel_residual_recursive
        print("k=%d: recursive residual gpu %.5e oracle %.5e (rel diff %.1e)" % (k, ik[0].rel_residual_recursive,
                                                                                   ok_.rel_residual_recursive, dr))
        assert ik[0].iterations == ok_.iterations == k and dr <= 5e-3
    with pytest.raises(ValueError):
        plan.cg_solve(d_phi, d_b, m, g, rho, tol, 100, half_storage=True, precondition=True)


def test_config5a_half_storage_true_residual(wz, orc, inp):
    """Config 5a (48x24^3, mixed radix 2/3) by the binary16-storage solver with reliable updates: the ORACLE recomputes
    the true residual of the returned x; iteration count next to the complex64 solver's."""
    cfg = inp.CONFIGS["5a"]
    dims = cfg["dims"]
    phi = inp.make_phi(cfg["seed"], dims, cfg["sigma"], np.complex64)
    b = inp.make_source(cfg["seed"], 0, dims, np.complex64)
    plan = wz.Plan(dims, "c64", 1)
    d_phi, d_b = torch.from_numpy(phi).cuda(), torch.from_numpy(b[None]).cuda()
    x, infos = plan.cg_solve(d_phi, d_b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 400000, half_storage=True)
    _, i64 = plan.cg_solve(d_phi, d_b, cfg["m"], cfg["g"], cfg["rho"], cfg["tol"], 400000)
    print("config 5a, binary16 storage: %d iterations, %d updates (complex64 solver: %d, %d), true residual %.3e"
          % (infos[0].iterations, infos[0].reliable_updates, i64[0].iterations, i64[0].reliable_updates,
             infos[0].rel_residual_true))
    assert infos[0].converged and infos[0].rel_residual_true <= cfg["tol"]
    # the iteration overhead of binary16 storage grows with the condition number: +8 % at 8^4, +10 % at 16^4, +14 % at 32^4,
    # +36 % here (18108 against 13345; lambda_max 1.8e5, m = 0.005)
    assert infos[0].iterations <= 1.5 * i64[0].iterations
    xh = x.cpu().numpy()[0]
    res = rel(orc.apply_MdagM(phi.astype(np.complex128), xh, cfg["m"], cfg["g"], cfg["rho"]), b.astype(np.complex128))
    assert res <= cfg["tol"] and abs(res - infos[0].rel_residual_true) <= 0.02 * cfg["tol"]


def test_source_blocks_do_not_change_results(wz, inp):
    """wz_plan_set_block: sources advanced block by block instead of all in lock step give the same x, bit for bit
    (the sources are independent solves with per-source reductions), with and without graph replay."""
    dims = (16, 16, 16, 16)
    phi = torch.from_numpy(inp.make_phi(3, dims, 0.5, np.complex64)).cuda()
    b = torch.from_numpy(inp.make_sources(3, 5, dims, np.complex64)).cuda()
    plan = wz.Plan(dims, "c64", 5)
    x0, i0 = plan.cg_solve(phi, b, 0.02, 1.0, 1.0, 1e-6, 600, raise_on_fail=False)
    for blk, graph in ((2, True), (3, False), (1, True), (0, True)):
        plan.set_block(blk)
        plan.set_graph(graph)
        x1, i1 = plan.cg_solve(phi, b, 0.02, 1.0, 1.0, 1e-6, 600, raise_on_fail=False)
        assert torch.equal(x0, x1), (blk, graph)
        assert [i.iterations for i in i0] == [i.iterations for i in i1]
        assert [i.reliable_updates for i in i0] == [i.reliable_updates for i in i1]
