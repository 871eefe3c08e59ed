"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json's: max relative error per moment
field <= 1e-12 (fp64) / 2e-5 (fp32); droplets: sign(phi) agreement >= 99.99 %.
Error norm (reading C17): max|gpu - oracle| / max|oracle| per field; a field whose
oracle maximum is below 1e-6 of its group's (u, P-diagonal, P-off-diagonal) uses the group's."""
import numpy as np
import pytest

from paper_2301_01622_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lbwp():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2301_01622_b200 import build as lbuild
    from paper_2301_01622_b200 import lbwp as mod
    lbuild.build()
    return mod


from parity_norms import TOL, parity_errors, report, sign_agreement  # noqa: E402  (tests/ is on sys.path)


def run_gpu(lbwp, cfg, m0, steps, kernel="auto", scheme="moments"):
    with lbwp.Lbwp(m0, lattice=cfg["lattice"], dtype=cfg["dtype"], ncomp=cfg["ncomp"], tau=cfg["tau"],
                   A=cfg["A"], beta=cfg["beta"], kernel=kernel, scheme=scheme) as sim:
        sim.step(steps)
        out = sim.moments_host()
        assert sim.steps_done == steps
    return out


def run_oracle(oracle, cfg, m0, steps, pop=False):
    fn = oracle.pop_run if pop else oracle.run
    return fn(m0, lattice=cfg["lattice"], ncomp=cfg["ncomp"], tau=cfg["tau"], nsteps=steps, A=cfg["A"],
              beta=cfg["beta"])


def check(lbwp, oracle, cfg, steps, kernel="auto", scheme="moments", tol=None):
    m0 = wl.as_dtype(cfg["moments"], cfg["dtype"])
    got = run_gpu(lbwp, cfg, m0, steps, kernel, scheme)
    ref = run_oracle(oracle, cfg, m0, steps, pop=(scheme == "populations"))
    assert np.isfinite(got).all()
    errs, _raw = report("%s/%s/%s/%d steps" % (cfg["name"], kernel, scheme, steps), got, ref, cfg["ncomp"], cfg["dtype"])
    assert errs.max() <= (tol or TOL[cfg["dtype"]]), (cfg["name"], kernel, errs)
    return got, ref


# ---- config 1: D3Q27, 32^3, fp64, tau=0.8, Taylor-Green, 100 steps ------------------------
@pytest.mark.parametrize("kernel", ["tma", "march", "gather"])
def test_config1_taylor_green_fp64(lbwp, oracle, kernel):
    check(lbwp, oracle, wl.config1(), 100, kernel=kernel)


# ---- config 2 at a ragged size spanning several tiles with a tail, both lattices/dtypes ----
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("lattice", [19, 27])
@pytest.mark.parametrize("kernel", ["auto", "gather"])
def test_config2_ragged(lbwp, oracle, dtype, lattice, kernel):
    cfg = dict(name="config2_ragged", moments=wl.noisy_solenoidal(0, shape=(45, 38, 41)), lattice=lattice,
               ncomp=1, tau=0.6, A=0.0, beta=0.0, dtype=dtype)
    check(lbwp, oracle, cfg, 60, kernel=kernel)


# ---- the TMA kernel: tiles in x and y, ragged z chunks, thin boxes (wrap planes coincide) ------
@pytest.mark.parametrize("dtype,shape", [("f32", (128, 24, 37)), ("f32", (64, 8, 1)), ("f32", (64, 16, 2)),
                                         ("f32", (192, 40, 3)), ("f64", (64, 24, 21)), ("f64", (32, 8, 1)),
                                         ("f64", (96, 16, 2))])
@pytest.mark.parametrize("steps", [1, 2, 25])
@pytest.mark.parametrize("lattice", [27, 19])
def test_tma_kernel_shapes(lbwp, oracle, dtype, shape, steps, lattice):
    cfg = dict(name="tma%d_%s_%s" % (lattice, dtype, "x".join(map(str, shape))),
               moments=wl.noisy_solenoidal(0, shape=shape), lattice=lattice, ncomp=1, tau=0.6, A=0.0, beta=0.0,
               dtype=dtype)
    check(lbwp, oracle, cfg, steps, kernel="tma")


def test_tma_tau_one_and_restart(lbwp, oracle):
    """tau = 1 makes the stored S-form independent of Pi (pin P6): lbwp_moments must still return the
    pre-collision Pi of the current step; set_moments restarts the step counter and the t = 0 export."""
    shape = (64, 16, 9)
    m0 = wl.as_dtype(wl.noisy_solenoidal(0, shape=shape), "f64")
    m0[4:] += 1e-3 * np.random.default_rng(5).uniform(-1, 1, m0[4:].shape)   # off-equilibrium Pi
    with lbwp.Lbwp(m0, lattice=27, dtype="f64", tau=1.0, kernel="tma") as sim:
        assert sim.kernel_name == "tma27_f64"
        assert np.array_equal(sim.moments_host(), m0)
        sim.step(3)
        got = sim.moments_host()
        ref = oracle.run(m0, lattice=27, tau=1.0, nsteps=3)
        assert parity_errors(got, ref, 1, "f64").max() <= 1e-12
        sim.set_moments(got)
        assert sim.steps_done == 0 and np.array_equal(sim.moments_host(), got)
        sim.step(2)
        ref5 = oracle.run(got, lattice=27, tau=1.0, nsteps=2)
        assert parity_errors(sim.moments_host(), ref5, 1, "f64").max() <= 1e-12


# ---- config 2 itself: 128^3, tau=0.6, 1000 steps, fp32 and fp64 (BASELINE.json).  Both runs start from the same
#      fp32-representable state (the recipe rounded to fp32, which fp64 holds exactly), so one oracle run of 1000
#      steps (about two minutes on the box's host cores) serves both.
@pytest.fixture(scope="module")
def config2_reference(oracle):
    cfg = wl.config2(128, "f32")
    m0 = wl.as_dtype(cfg["moments"], "f32")
    return cfg, m0, oracle.run(m0, lattice=27, ncomp=1, tau=cfg["tau"], nsteps=1000)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config2_128_1000_steps(lbwp, config2_reference, dtype):
    cfg, m0, ref = config2_reference
    cfg = dict(cfg, dtype=dtype)
    got = run_gpu(lbwp, cfg, m0.astype(np.float64) if dtype == "f64" else m0, 1000)
    errs, _ = report("config2_128/%s/1000 steps" % dtype, got, ref, 1, dtype)
    assert errs.max() <= TOL[dtype], errs


# ---- two-component colour gradient (reading C6): config-3 geometry scaled to 48^3 ----------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("lattice", [19, 27])
def test_config3_scaled_droplets(lbwp, oracle, dtype, lattice):
    cfg = wl.config3(48)
    cfg.update(dtype=dtype, lattice=lattice)
    got, ref = check(lbwp, oracle, cfg, 200)
    assert sign_agreement(got, ref) >= 0.9999


# ---- the two-component TMA paths (fused: csrc/lbwp_tma2g.cuh; split collide / stream: csrc/lbwp_tma2.cuh): several tiles, ragged z chunk,
#      thin box, tau != 1 (non-equilibrium Pi matters), droplets crossing the periodic boundary -------------
@pytest.mark.parametrize("dtype,shape", [("f32", (64, 24, 20)), ("f32", (128, 16, 37)), ("f32", (64, 8, 2)),
                                         ("f64", (32, 24, 20)), ("f64", (64, 16, 5))])
@pytest.mark.parametrize("steps,tau", [(1, 1.0), (30, 0.7)])
@pytest.mark.parametrize("lattice,kernel", [(27, "tma"), (27, "tma_split"), (19, "tma"), (19, "tma_split")])
def test_tma_two_component(lbwp, oracle, dtype, shape, steps, tau, lattice, kernel):
    nx, ny, nz = shape
    tg = wl.taylor_green(0, shape=shape)
    m = wl.droplets(0, [(0.3 * nx, 0.5 * ny, 0.5 * nz), (0.95 * nx, 0.1 * ny, 0.6 * nz)], 0.3 * min(ny, nx),
                    [0.03, -0.03], background_u=[tg[1], tg[2], tg[3]], shape=shape)
    cfg = dict(name="tma2_q%d_%s_%s" % (lattice, dtype, "x".join(map(str, shape))), moments=m, lattice=lattice, ncomp=2,
               tau=tau, A=0.01, beta=0.7, dtype=dtype)
    m0 = wl.as_dtype(m, dtype)
    split = kernel == "tma_split"
    with lbwp.Lbwp(m0, lattice=lattice, dtype=dtype, ncomp=2, tau=tau, A=0.01, beta=0.7, kernel=kernel) as sim:
        assert sim.kernel_name == "tma%d_%s_c2%s" % (lattice, dtype, "split" if split else "")
        assert sim.launches_per_step == (2 if split else 1)      # fused: ONE kernel per time step
        back = sim.moments_host()          # t = 0: the input, up to the j = rho u round trip
        assert np.abs(back.astype(np.float64) - m0).max() <= (3e-7 if dtype == "f32" else 1e-15)
    got, ref = check(lbwp, oracle, cfg, steps, kernel=kernel)
    assert sign_agreement(got, ref) >= 0.9999


# ---- comparison kernel vs its own mini-oracle (population-storing pull BGK) ----------------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("lattice", [19, 27])
def test_population_kernel(lbwp, oracle, dtype, lattice):
    cfg = dict(name="pop", moments=wl.noisy_solenoidal(0, shape=(37, 30, 33)), lattice=lattice, ncomp=1,
               tau=0.6, A=0.0, beta=0.0, dtype=dtype)
    check(lbwp, oracle, cfg, 40, scheme="populations")
    check(lbwp, oracle, cfg, 0, scheme="populations")


# ---- two-component comparison kernel (one population set per colour) vs its mini-oracle:
#      ragged box, droplet crossing the periodic boundary, tau != 1, sign(phi) ---------------------------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("lattice", [19, 27])
def test_population_kernel_two_component(lbwp, oracle, dtype, lattice):
    shape = (37, 30, 33)
    nx, ny, nz = shape
    tg = wl.taylor_green(0, shape=shape)
    m = wl.droplets(0, [(0.3 * nx, 0.5 * ny, 0.5 * nz), (0.95 * nx, 0.1 * ny, 0.6 * nz)], 0.25 * min(ny, nx),
                    [0.03, -0.03], background_u=[tg[1], tg[2], tg[3]], shape=shape)
    cfg = dict(name="pop2", moments=m, lattice=lattice, ncomp=2, tau=0.7, A=0.01, beta=0.7, dtype=dtype)
    m0 = wl.as_dtype(m, dtype)
    with lbwp.Lbwp(m0, lattice=lattice, dtype=dtype, ncomp=2, tau=0.7, A=0.01, beta=0.7, scheme="populations") as sim:
        assert sim.kernel_name == "pop_pull%d_%s_c2" % (lattice, dtype)
        assert sim.launches_per_step == 3
    check(lbwp, oracle, cfg, 0, scheme="populations")
    check(lbwp, oracle, cfg, 1, scheme="populations")
    got, ref = check(lbwp, oracle, cfg, 40, scheme="populations")
    assert sign_agreement(got, ref) >= 0.9999


# ---- edge cases: degenerate boxes, zero steps, set_moments, library-owned buffers ----------
@pytest.mark.parametrize("shape", [(1, 1, 1), (1, 7, 3), (3, 1, 33), (2, 2, 65), (5, 9, 1)])
@pytest.mark.parametrize("kernel", ["auto", "gather"])
def test_degenerate_boxes(lbwp, oracle, shape, kernel):
    rng = np.random.default_rng(11)
    nz, ny, nx = shape
    rho = 1.0 + 0.05 * rng.uniform(-1, 1, shape)
    u = [0.03 * rng.uniform(-1, 1, shape) for _ in range(3)]
    m = wl.pack1(rho, u)
    m[4:] += 0.01 * rng.uniform(-1, 1, (6, nz, ny, nx))
    cfg = dict(name=f"box{shape}", moments=m, lattice=27, ncomp=1, tau=0.7, A=0.0, beta=0.0, dtype="f64")
    check(lbwp, oracle, cfg, 5, kernel=kernel)


def test_zero_steps_and_round_trip(lbwp):
    cfg = wl.config2(24, "f32")
    m0 = wl.as_dtype(cfg["moments"], "f32")
    with lbwp.Lbwp(m0, lattice=27, dtype="f32", tau=0.6, use_torch_buffers=False) as sim:
        sim.step(0)
        a = sim.moments_host()
        # import/export only shifts by 1 and 1/3: at most one rounding of the shifted value
        assert np.abs(a - m0).max() <= 1.2e-7
        sim.step(3)
        b = sim.moments_host()
        c = sim.moments().cpu().numpy()       # device destination, same values, state untouched
        assert np.array_equal(b, c)
        sim.set_moments(m0)
        assert sim.steps_done == 0
        sim.step(3)
        assert np.array_equal(sim.moments_host(), b)   # deterministic


@pytest.mark.parametrize("ncomp", [1, 2])
def test_checkpoint_resume(lbwp, ncomp):
    """The moments are the complete state: lbwp_moments -> lbwp_init continues the run.  The TMA path
    stores collided moments internally, so a resume re-collides the exported ones: equal up to rounding, not bit for bit."""
    shape = (64, 16, 12)
    if ncomp == 1:
        m0 = wl.noisy_solenoidal(0, shape=shape)
    else:
        m0 = wl.droplets(0, [(20, 8, 6), (50, 3, 4)], 5, [0.03, -0.03], shape=shape)
    kw = dict(lattice=27, dtype="f64", ncomp=ncomp, tau=0.7, A=0.01, beta=0.7)
    with lbwp.Lbwp(m0, **kw) as sim:
        assert sim.kernel_name.startswith("tma27")
        sim.step(8)
        straight = sim.moments_host()
    with lbwp.Lbwp(m0, **kw) as sim:
        sim.step(4)
        mid = sim.moments_host()
    with lbwp.Lbwp(mid, **kw) as sim:
        sim.step(4)
        resumed = sim.moments_host()
    assert np.abs(resumed - straight).max() <= 1e-13


def test_device_input_and_errors(lbwp):
    import torch
    cfg = wl.config1()
    m0 = torch.from_numpy(wl.as_dtype(cfg["moments"], "f64")).cuda()
    with lbwp.Lbwp(m0, lattice=27, dtype="f64", tau=0.8) as sim:
        sim.step(2)
        assert sim.launches_per_step == 1 and "27" in sim.kernel_name
        with pytest.raises(lbwp.LbwpError):
            sim.step(-1)
    with pytest.raises(lbwp.LbwpError):
        lbwp.Lbwp(m0, lattice=27, dtype="f64", tau=0.4)


# ---- the sizes and launch configurations bench.py times, element by element against the oracle: 256^3 and 512^3
#      fp32, 2 steps (512^3: 4096 work items in 16 z chunks; about 15 s and 35 GB of host memory for the oracle) ----
@pytest.mark.parametrize("n", [256, 512])
def test_bench_size(lbwp, oracle, n):
    check(lbwp, oracle, wl.sweep_case(n, 27, 1, "f32"), 2)


def test_invariants_512(lbwp):
    import torch
    n = 512
    k = 2 * np.pi / n
    x = torch.arange(n, device="cuda", dtype=torch.float64)
    ux = 0.01 * torch.sin(k * x)[None, None, :] * torch.cos(k * x)[None, :, None] * torch.ones(n, 1, 1, device="cuda", dtype=torch.float64)
    uy = -0.01 * torch.cos(k * x)[None, None, :] * torch.sin(k * x)[None, :, None] * torch.ones(n, 1, 1, device="cuda", dtype=torch.float64)
    m0 = torch.empty((10, n, n, n), dtype=torch.float32, device="cuda")
    m0[0] = 1.0
    m0[1], m0[2], m0[3] = ux.float(), uy.float(), 0.0
    m0[4], m0[5], m0[6] = 1 / 3 + m0[1] ** 2, 1 / 3 + m0[2] ** 2, 1 / 3
    m0[7], m0[8], m0[9] = m0[1] * m0[2], 0.0, 0.0
    del ux, uy
    with lbwp.Lbwp(m0, lattice=27, dtype="f32", tau=0.8) as sim:
        mass0 = m0[0].double().sum().item()
        px0 = (m0[0].double() * m0[1].double()).sum().item()
        sim.step(20)
        out = sim.moments(out=m0)
        mass1 = out[0].double().sum().item()
        px1 = (out[0].double() * out[1].double()).sum().item()
        amp = out[1].abs().max().item()
    assert abs(mass1 - mass0) / mass0 < 1e-7          # Eq. 1 summed over the periodic box
    assert abs(px1 - px0) < 1e-7 * n ** 3 * 0.01
    # Taylor-Green decay exp(-2 nu k^2 t), nu = cs^2 (tau - 1/2) = 0.1
    assert abs(amp / 0.01 - np.exp(-2 * 0.1 * k * k * 20)) < 1e-4


# ---- lbwp_diagnostics: the fused reduction against the oracle's, after a few steps;
#      masses / momentum / mean to the rounding of the state, probe densities element-wise, node count exactly up to
#      the nodes whose density sits within rounding of the threshold -------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("scheme", ["moments", "populations"])
def test_diagnostics(lbwp, oracle, dtype, scheme):
    cfg = wl.config3(64)
    m0 = wl.as_dtype(cfg["moments"], dtype)
    probes = [(16, 32, 32), (32, 32, 32), (63, 0, 5)]
    kw = dict(lattice=27, ncomp=2, tau=0.9, A=0.01, beta=0.7)
    with lbwp.Lbwp(m0, dtype=dtype, scheme=scheme, **kw) as sim:
        sim.step(20)
        got = sim.diagnostics(0.5, probes)
        state = sim.moments_host()
    ref = (oracle.pop_run if scheme == "populations" else oracle.run)(m0, nsteps=20, **kw)
    want = oracle.diagnostics(ref, ncomp=2, threshold=0.5, probes=probes)
    tol = TOL[dtype]
    n = 64 ** 3
    for k in (0, 1):
        assert abs(got["mass"][k] - want["mass"][k]) <= tol * want["mass"][k]
    assert np.abs(np.array(got["momentum"]) - want["momentum"]).max() <= tol * n * 0.05
    assert abs(got["rho_mean_above"] - want["rho_mean_above"]) <= 10 * tol
    assert abs(got["rho_max"] - want["rho_max"]) <= 10 * tol
    assert np.abs(np.array(got["probe_rho"]) - want["probe_rho"]).max() <= 10 * tol
    near = int((np.abs(ref[0] - 0.5) < 1e-4).sum())                      # nodes that rounding may move across 0.5
    assert abs(got["count_above"] - want["count_above"]) <= near
    # and it is exactly the reduction of what lbwp_moments returns
    own = oracle.diagnostics(state, ncomp=2, threshold=0.5, probes=probes)
    assert got["count_above"] == own["count_above"] and got["probe_rho"] == own["probe_rho"]
    assert abs(got["mass"][0] - own["mass"][0]) <= 1e-9 * own["mass"][0]


def test_diagnostics_errors(lbwp):
    m0 = wl.as_dtype(wl.config1()["moments"], "f64")
    with lbwp.Lbwp(m0, dtype="f64", tau=0.8) as sim:
        d = sim.diagnostics(0.5)
        assert d["count_above"] == 32 ** 3 and abs(d["rho_mean_above"] - 1.0) < 1e-15 and d["mass"][1] == 0.0
        with pytest.raises(lbwp.LbwpError):
            sim.diagnostics(0.5, [(32, 0, 0)])


# ---- near-contact repulsion (Eq. 10; readings C20-C24): two drops pressed against
#      each other with the force on, against the oracle; the force must act (the run differs from A_h = 0) and the
#      momentum it injects is antisymmetric between the drops ------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("lattice", [19, 27])
def test_near_contact_force(lbwp, oracle, dtype, lattice):
    n, R, gap = 40, 9.0, 2.0
    d = 2 * R + gap
    m = wl.droplets(n, [(n / 2 - d / 2, n / 2, n / 2 - 2), (n / 2 + d / 2, n / 2, n / 2 + 2)], R, [0.03, -0.03], shape=(n, 36, 33))
    m0 = wl.as_dtype(m, dtype)
    kw = dict(lattice=lattice, tau=0.8, A=0.01, beta=0.7)
    steps = 25
    with lbwp.Lbwp(m0, dtype=dtype, ncomp=2, A_h=0.02, h_c=4.0, **kw) as sim:
        assert sim.kernel_name == "gather%d_%s_c2" % (lattice, dtype) and sim.launches_per_step == 3
        sim.step(steps)
        got = sim.moments_host()
    ref = oracle.run_nc(m0, nsteps=steps, A_h=0.02, h_c=4.0, **kw)
    errs, _ = report("near_contact_q%d/%s/%d steps" % (lattice, dtype, steps), got, ref, 2, dtype)
    assert errs.max() <= TOL[dtype], errs
    assert sign_agreement(got, ref) >= 0.9999
    off = oracle.run(m0, ncomp=2, nsteps=steps, **kw)
    assert np.abs(ref - off).max() > 1e-3                    # the repulsion changed the collision
    with pytest.raises(lbwp.LbwpError):                      # not built into the split TMA form
        lbwp.Lbwp(wl.as_dtype(wl.config3(64)["moments"], dtype), dtype=dtype, ncomp=2, A_h=0.02, kernel="tma_split", **kw)


# the same force behind the fused two-component TMA kernel (a fix-up pass on the collided moments, lbwp_contact.cuh):
# a box the tiles divide, the drops pressed against each other across tile, chunk and periodic boundaries
# nz = 38: the fix-up pass's boxes of four planes overhang the grid; h_c = 6: its walk leaves the shared-memory tile, so
# the kernel variant that reads rA from global memory runs
@pytest.mark.parametrize("nz,h_c", [(36, 4.0), (38, 4.0), (36, 6.0)])
@pytest.mark.parametrize("lattice", [19, 27])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_near_contact_force_fused(lbwp, oracle, dtype, lattice, nz, h_c):
    shape = (64, 40, nz)
    nx, ny, nz = shape
    R, gap = 9.0, 2.0
    d = 2 * R + gap
    # the film between the drops lies on the periodic x boundary (ghost columns) and on a tile boundary in y
    centres = [(nx - d / 2, 16.0, nz / 2 - 2), (d / 2, 16.0, nz / 2 + 2)]
    m = wl.droplets(0, centres, R, [0.03, -0.03], shape=shape)
    m0 = wl.as_dtype(m, dtype)
    kw = dict(lattice=lattice, tau=0.8, A=0.01, beta=0.7)
    steps = 25
    with lbwp.Lbwp(m0, dtype=dtype, ncomp=2, A_h=0.02, h_c=h_c, **kw) as sim:
        assert sim.kernel_name == "tma%d_%s_c2" % (lattice, dtype) and sim.launches_per_step == 3
        sim.step(steps)
        got = sim.moments_host()
        sim.step(1)                                          # lbwp_moments after a further step: the export path
        got1 = sim.moments_host()
    ref = oracle.run_nc(m0, nsteps=steps, A_h=0.02, h_c=h_c, **kw)
    errs, _ = report("near_contact_fused_q%d/%s/%d steps" % (lattice, dtype, steps), got, ref, 2, dtype)
    assert errs.max() <= TOL[dtype], errs
    assert sign_agreement(got, ref) >= 0.9999
    ref1 = oracle.run_nc(ref, nsteps=1, A_h=0.02, h_c=h_c, **kw)
    assert parity_errors(got1, ref1, 2, dtype).max() <= TOL[dtype]
    off = oracle.run(m0, ncomp=2, nsteps=steps, **kw)
    assert np.abs(ref - off).max() > 1e-3                    # the repulsion changed the collision
    with lbwp.Lbwp(m0, dtype=dtype, ncomp=2, A_h=0.02, h_c=h_c, kernel="gather", **kw) as sim:   # and the generic path agrees
        sim.step(steps)
        gen = sim.moments_host()
    assert parity_errors(got, gen.astype(np.float64), 2, dtype).max() <= TOL[dtype]


# the moments stay the complete state with the force on: lbwp_moments -> lbwp_set_moments on the same context (the import
# re-collides and runs the fix-up pass on buffer 0, whose layout differs from buffer 1's in the x-paired fp32 kernel)
@pytest.mark.parametrize("dtype,tol", [("f64", 1e-12), ("f32", 2e-5)])
def test_near_contact_restart(lbwp, dtype, tol):
    shape = (64, 40, 38)
    nx, ny, nz = shape
    R, gap = 9.0, 2.0
    d = 2 * R + gap
    m = wl.droplets(0, [(nx - d / 2, 16.0, nz / 2 - 2), (d / 2, 16.0, nz / 2 + 2)], R, [0.03, -0.03], shape=shape)
    m0 = wl.as_dtype(m, dtype)
    kw = dict(lattice=19, dtype=dtype, ncomp=2, tau=0.8, A=0.01, beta=0.7, A_h=0.02, h_c=4.0)
    with lbwp.Lbwp(m0, **kw) as sim:
        assert sim.kernel_name == "tma19_%s_c2" % dtype
        sim.step(9)
        straight = sim.moments_host().astype(np.float64)
        sim.set_moments(m0)
        sim.step(5)                                          # odd: the state sits in buffer 1 when it is exported
        mid = sim.moments_host()
        sim.set_moments(mid)
        assert sim.steps_done == 0
        sim.step(4)
        resumed = sim.moments_host().astype(np.float64)
    assert np.abs(resumed - straight).max() <= tol * np.abs(straight).max()
