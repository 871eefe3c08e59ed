"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json's: max relative error per moment
field <= 1e-12 (fp64) / 2e-5 (fp32); droplets: sign(phi) agreement >= 99.99 %.
Error norm (reading C17): max|gpu - oracle| / max|oracle| per field; a field whose
oracle maximum is below 1e-6 of its group's (u, P-diagonal, P-off-diagonal) uses the group's."""
import os

import numpy as np
import pytest

from paper_2301_01622_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}


@pytest.fixture(scope="module")
def lbwp():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2301_01622_b200 import build as lbuild
    from paper_2301_01622_b200 import lbwp as mod
    lbuild.build()
    return mod


EPS = {"f64": 2.0 ** -53, "f32": 2.0 ** -24}   # unit roundoff of the state / arithmetic type


def moment_field_errors(got, ref, ncomp):
    """BASELINE.json's norm: max relative error per MOMENT FIELD of H = [rho, u_a, P_ab]
    (PAPER.md:39): max over nodes and components of |gpu - oracle| / max over nodes and
    components of |oracle|, for the densities, the velocity vector and the pressure tensor."""
    off = ncomp - 1
    out = []
    for g in (range(0, ncomp), range(off + 1, off + 4), range(off + 4, off + 10)):
        num = max(np.abs(got[k].astype(np.float64) - ref[k]).max() for k in g)
        out.append(num / max(np.abs(ref[k]).max() for k in g))
    return np.array(out)


def field_errors(got, ref, ncomp, dtype="f64"):
    """Stricter, per stored COMPONENT (reading C17): max|gpu - oracle| / max|oracle|
    of that component alone, after discounting the rounding floor of the sums Eq. 1-3 themselves:
      * the fp64 oracle adds populations of size w_i*rho, so any component is only known to
        64*2^-53*max|group| absolute (group = densities, u, P-diagonal; off-diagonals share the
        diagonal's terms) -- P_xy ~ 1e-5 in config 1 is a small difference of O(1/54) terms;
      * in the state precision, P_ab sums populations whose odd part is 3 w_i rho c.u, so its
        absolute rounding floor is 4*eps*max|rho u| (matters for fp32 Taylor-Green, where
        max|P_xy| = u0^2/4 = 2.5e-5 is 400 times smaller than max|rho u| = 1e-2).
    A component identically ~0 (u_z in config 1) is scaled by its group's maximum."""
    off = ncomp - 1
    groups = [list(range(0, ncomp)), [off + 1, off + 2, off + 3], [off + 4, off + 5, off + 6],
              [off + 7, off + 8, off + 9]]
    rho = ref[:ncomp].sum(axis=0)
    jmax = max(np.abs(rho * ref[off + 1 + a]).max() for a in range(3))
    errs = np.zeros(ref.shape[0])
    for gi, g in enumerate(groups):
        gmax = max(np.abs(ref[k]).max() for k in g)
        unit = groups[2] if gi == 3 else g
        floor = 64 * EPS["f64"] * max(np.abs(ref[k]).max() for k in unit)
        if gi >= 2:
            floor += 4 * EPS[dtype] * jmax
        for k in g:
            s = np.abs(ref[k]).max()
            if s < 1e-6 * gmax:
                s = gmax
            d = np.abs(got[k].astype(np.float64) - ref[k]).max()
            errs[k] = max(d - floor, 0.0) / s
    return errs


def parity_errors(got, ref, ncomp, dtype):
    """Both norms; every parity test gates on both at BASELINE.json's tolerance."""
    return np.concatenate([moment_field_errors(got, ref, ncomp), field_errors(got, ref, ncomp, dtype)])


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
    errs = parity_errors(got, ref, cfg["ncomp"], cfg["dtype"])
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


# ---- config 2 itself: 128^3, tau=0.6, fp32 and fp64.  The oracle runs at a few MLUPS, so the
#      default run takes 40 steps at 128^3 and the full 1000 steps at 64^3 (same recipe, same
#      error-growth horizon); LBWP_FULL_CONFIGS=1 runs the 1000 steps at 128^3 as BASELINE states.
FULL = os.environ.get("LBWP_FULL_CONFIGS", "0") == "1"


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config2_128(lbwp, oracle, dtype):
    check(lbwp, oracle, wl.config2(128, dtype), 1000 if FULL else 40)


def test_config2_1000_steps_fp32(lbwp, oracle):
    check(lbwp, oracle, wl.config2(64, "f32"), 1000)


# ---- two-component colour gradient (reading C6): config-3 geometry scaled to 48^3 ----------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("lattice", [19, 27])
def test_config3_scaled_droplets(lbwp, oracle, dtype, lattice):
    cfg = wl.config3(48)
    cfg.update(dtype=dtype, lattice=lattice)
    got, ref = check(lbwp, oracle, cfg, 200)
    phi_g = got[0].astype(np.float64) - got[1]
    phi_r = ref[0] - ref[1]
    agree = np.mean(np.sign(phi_g) == np.sign(phi_r))
    assert agree >= 0.9999


# ---- the two-component TMA path (split collide / stream, csrc/lbwp_tma2.cuh): several tiles, ragged z chunk,
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
        assert sim.launches_per_step == 2
        back = sim.moments_host()          # t = 0: the input, up to the j = rho u round trip
        assert np.abs(back.astype(np.float64) - m0).max() <= (3e-7 if dtype == "f32" else 1e-15)
    got, ref = check(lbwp, oracle, cfg, steps, kernel=kernel)
    agree = np.mean(np.sign(got[0].astype(np.float64) - got[1]) == np.sign(ref[0] - ref[1]))
    assert agree >= 0.9999


# ---- config 3 itself (128^3, fp32, tau=1, A=0.01, beta=0.7).  The drops touch between steps 100 and 200 and the
#      rupture of the film between them amplifies any perturbation by 1e4-1e5 (measured: the fp64 kernel goes from
#      7e-14 to 4e-10 against the fp64 oracle, three independent fp32 kernels from 3e-6 to 0.1-0.18, and 0.06 apart from
#      each other: profiles/r01_config3_divergence.md).  BASELINE's fp32 tolerance is therefore gated up to the contact;
#      after it (LBWP_FULL_CONFIGS=1: all 2000 steps) the gates are what an fp32 trajectory can keep: colour masses, the
#      sign of the phase field on >= 99.9 % of the nodes, bounded fields.  The fp64 run of the same configuration must
#      stay within 2e-5 and 100 % sign agreement through the collision (next test). ---
def test_config3_full_size(lbwp, oracle):
    cfg = wl.config3(128)
    m0 = wl.as_dtype(cfg["moments"], "f32")
    kw = dict(lattice=27, ncomp=2, tau=cfg["tau"], A=cfg["A"], beta=cfg["beta"])
    pre = 100 if FULL else 40
    with lbwp.Lbwp(m0, dtype="f32", **kw) as sim:
        sim.step(pre)
        got = sim.moments_host()
        ref = oracle.run(m0, nsteps=pre, **kw)
        assert parity_errors(got, ref, 2, "f32").max() <= TOL["f32"]
        assert np.mean(np.sign(got[0].astype(np.float64) - got[1]) == np.sign(ref[0] - ref[1])) >= 0.9999
        if not FULL:
            return
        sim.step(2000 - pre)
        got = sim.moments_host().astype(np.float64)
    ref = oracle.run(ref, nsteps=2000 - pre, **kw)
    assert np.isfinite(got).all() and np.abs(got[2:5]).max() < 0.2
    for k in (0, 1):                                   # each colour's mass (Eq. 1 summed over the box)
        assert abs(got[k].sum() - m0[k].astype(np.float64).sum()) <= 2e-5 * m0[k].astype(np.float64).sum()
    assert np.mean(np.sign(got[0] - got[1]) == np.sign(ref[0] - ref[1])) >= 0.999
    print("config3 after 2000 steps, fp32 vs fp64 oracle:", parity_errors(got, ref, 2, "f32"))


def test_config3_long_run_fp64(lbwp, oracle):
    """Same configuration in fp64, through the collision (300 steps; 2000 with LBWP_FULL_CONFIGS=1): the kernel differs
    from the oracle only in the order of its additions, and even that is amplified to 1e-6 (never beyond 2e-5)."""
    cfg = wl.config3(128)
    m0 = wl.as_dtype(cfg["moments"], "f32").astype(np.float64)
    kw = dict(lattice=27, ncomp=2, tau=cfg["tau"], A=cfg["A"], beta=cfg["beta"])
    steps = 2000 if FULL else 300
    with lbwp.Lbwp(m0, dtype="f64", **kw) as sim:
        sim.step(steps)
        got = sim.moments_host()
    ref = oracle.run(m0, nsteps=steps, **kw)
    assert parity_errors(got, ref, 2, "f64").max() <= 2e-5
    assert np.mean(np.sign(got[0] - got[1]) == np.sign(ref[0] - ref[1])) == 1.0


# ---- config 4 (256^3 off-axis collision, fp32): its 4000 steps are hours of oracle time, so the full-size box is
#      checked over its first steps (12; 100 with LBWP_FULL_CONFIGS=1) in the launch configuration bench.py times ----
def test_config4_full_size_first_steps(lbwp, oracle):
    cfg = wl.config4(256)
    got, ref = check(lbwp, oracle, cfg, 100 if FULL else 12)
    agree = np.mean(np.sign(got[0].astype(np.float64) - got[1]) == np.sign(ref[0] - ref[1]))
    assert agree >= 0.9999


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
    agree = np.mean(np.sign(got[0].astype(np.float64) - got[1]) == np.sign(ref[0] - ref[1]))
    assert agree >= 0.9999


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


# ---- full bench size, launch configuration bench.py times: 256^3 fp32, 2 steps vs oracle,
#      and invariants at 512^3 (conservation; the oracle cannot finish 512^3 in seconds) -----
def test_bench_size_256(lbwp, oracle):
    cfg = wl.sweep_case(256, 27, 1, "f32")
    m0 = wl.as_dtype(cfg["moments"], "f32")
    got = run_gpu(lbwp, cfg, m0, 2)
    ref = run_oracle(oracle, cfg, m0, 2)
    assert parity_errors(got, ref, 1, "f32").max() <= TOL["f32"]


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
