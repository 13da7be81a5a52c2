"""Parity of the CUDA path (through the C ABI) with the fp64 CPU oracle, element by element on the same
seeded inputs.  Needs a B200: run with -m gpu.

Tolerances (BASELINE.json north_star; definitions DESIGN.md "Tolerances"), per field array, BOTH norms asserted:
  fp64 fields after 20 steps : strict  max_x |gpu - oracle| / max_x |oracle| <= 1e-12
                               R14     max_x |gpu - oracle| / max(1, max_x |oracle|) <= 1e-12
  fp32 fields after 20 steps : strict  max_x |gpu - oracle| <= 2e-4                          (north_star, absolute)
                               R14     max_x |gpu - oracle| / max(1, max_x |oracle|) <= 2e-4
  (the one exception to the strict fp32 bound is config 3's physics, s = 1 in the matter era, where eps grows to ~30 in
   20 steps and 2e-4 absolute is below fp32 resolution of the field itself: SURVEY 8(c) "Config consequences of G3")
  winding                    : bit-exact on identical snapshots (produced by the oracle, uploaded with ahs_set_fields)
  <v^2> sums                 : fp64 1e-10 relative, fp32 2e-5 relative to sum |K Lag|, sum |G Lag|
  Gauss residual             : at roundoff of the storage type on both paths
"""
import json
import math
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-4}


@pytest.fixture(scope="module", autouse=True)
def oracle_on_all_cores(oracle):
    """The oracle's results do not depend on its thread count (test_oracle_is_independent_of_the_thread_count)."""
    oracle.set_threads(0)
    yield
    oracle.set_threads(1)


def record(test, **kw):
    """Observed maxima: printed (pytest -s) and, if AHS_PARITY_LOG names a file, appended to it as JSON lines."""
    line = json.dumps(dict(test=test, **kw))
    print(line)
    path = os.environ.get("AHS_PARITY_LOG")
    if path:
        with open(path, "a") as f:
            f.write(line + "\n")


@pytest.fixture(scope="module")
def ahs():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1809_00995_b200 import binding
    binding.load()
    return binding


def field_errors(got, ref):
    """R14 norm per field array: max |d| / max(1, max |oracle|)."""
    return [np.abs(got[k] - ref[k]).max() / max(1.0, np.abs(ref[k]).max()) for k in range(10)]


def strict_errors(got, ref, prec):
    """north_star's norms as stated: fp64 max |d| / max |oracle| (relative), fp32 max |d| (absolute)."""
    out = []
    for k in range(10):
        d, m = np.abs(got[k] - ref[k]).max(), np.abs(ref[k]).max()
        out.append(d if prec == "f32" else (d / m if m > 0 else (0.0 if d == 0 else np.inf)))
    return out


def assert_fields(test, got, ref, prec, names, strict=True, tol=None, **ctx):
    tol = TOL[prec] if tol is None else tol
    r14, st = field_errors(got, ref), strict_errors(got, ref, prec)
    record(test, prec=prec, strict_asserted=strict, max_r14=max(r14), max_strict=max(st),
           strict_per_field={n: float("%.3g" % e) for n, e in zip(names, st)}, **ctx)
    for k in range(10):
        assert r14[k] <= tol, (names[k], "R14", r14[k], ctx)
        if strict:
            assert st[k] <= tol, (names[k], "strict", st[k], ctx)


def oracle_params(O, sim):
    q = dict(sim.params)
    q.pop("seed")
    return O.Params(**q)


def check_diag(O, p, sim, prec, snap, n):
    """Diagnostics on an identical snapshot.  `snap` comes from the ORACLE side (never from the CUDA path); it is
    uploaded with ahs_set_fields (fp32 storage: the test rounds it to fp32 first so both sides see the same values)."""
    if prec == "f32":
        snap = snap.astype(np.float32).astype(np.float64)
    sim.set_fields(snap, n)
    d = sim.diagnostics()
    r = O.diagnostics(p, snap, n)
    assert d["step"] == n and d["tau"] == pytest.approx(p.tau0 + n * p.dt, rel=1e-15)
    assert d["n_pierced"] == r["n_pierced"] and d["sum_abs_w"] == r["sum_abs_w"]          # bit-exact
    assert d["L"] == pytest.approx(r["L"], rel=1e-14)
    assert (math.isinf(d["xi"]) and math.isinf(r["xi"])) or d["xi"] == pytest.approx(r["xi"], rel=1e-14)
    K, G, Lg = O.site_fields(p, snap, n)
    rel = 1e-10 if prec == "f64" else 2e-5
    assert abs(d["v2_num"] - r["v2_num"]) <= rel * np.abs(K * Lg).sum() + 1e-300
    assert abs(d["v2_den"] - r["v2_den"]) <= rel * np.abs(G * Lg).sum() + 1e-300
    assert abs(d["mean_lagrangian"] - r["mean_lagrangian"]) <= rel * np.abs(Lg).mean() + 1e-300
    Vp = O.site_fields4(p, snap, n)[3]                       # potential-weighted estimator and xi_L
    floor = 1e-18 * Vp.size * max(1.0, G.max(), K.max())     # |phi| = sigma exactly (IC): Vp is rounding noise, ~1e-32
    assert abs(d["v2v_num"] - r["v2v_num"]) <= rel * (K * Vp).sum() + floor
    assert abs(d["v2v_den"] - r["v2v_den"]) <= rel * (G * Vp).sum() + floor
    if r["mean_lagrangian"] < -1e-3 * np.abs(Lg).mean():
        assert d["xi_L"] == pytest.approx(r["xi_L"], rel=50 * rel)
    # equation-of-state estimator (Eq. 12): the two Lagrangian-weighted sums, relative to their absolute sums
    K6, G6, L6, V6, El, Bm = O.site_fields6(p, snap, n)
    rho, prs = K6 + G6 + V6 + El + Bm, K6 - G6 / 3 - V6 + (El + Bm) / 3
    # observed errors of the sums, in units of the absolute sums they are compared against (bar: `rel`)
    ratio = lambda err, scale: float("%.3g" % (abs(err) / scale)) if scale > 0 else 0.0
    record("check_diag", prec=prec, N=int(snap.shape[-1]), kernel=sim.kernel_kind, bar=rel,
           v2_num=ratio(d["v2_num"] - r["v2_num"], np.abs(K * Lg).sum()), v2_den=ratio(d["v2_den"] - r["v2_den"], np.abs(G * Lg).sum()),
           lagrangian=ratio(d["mean_lagrangian"] - r["mean_lagrangian"], np.abs(Lg).mean()),
           eos_num=ratio(d["eos_num"] - r["eos_num"], np.abs(prs * L6).sum()), eos_den=ratio(d["eos_den"] - r["eos_den"], np.abs(rho * L6).sum()))
    assert abs(d["eos_num"] - r["eos_num"]) <= rel * np.abs(prs * L6).sum() + 1e-300
    assert abs(d["eos_den"] - r["eos_den"]) <= rel * np.abs(rho * L6).sum() + 1e-300
    if abs(r["eos_den"]) > 0.05 * np.abs(rho * L6).sum():
        assert d["v2_omega"] == pytest.approx(r["v2_omega"], rel=200 * rel, abs=200 * rel)
    eps_m = 2.3e-16 if prec == "f64" else 6e-8
    gscale = max(1.0, r["gauss_rhs_rms"], np.abs(snap[7:10]).max())
    assert abs(d["gauss_max"] - r["gauss_max"]) <= 64 * eps_m * gscale
    assert d["gauss_rhs_rms"] == pytest.approx(r["gauss_rhs_rms"], rel=1e-5, abs=1e-30)
    assert d["nonfinite"] == r["nonfinite"] == 0
    return d, r


def rounded(f, prec):
    return f.astype(np.float32).astype(np.float64) if prec == "f32" else f


# ---------------------------------------------------------------------------------------------------------
# initial condition
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec,N", [("f64", 32), ("f32", 32), ("f32", 128), ("f64", 64)])
@pytest.mark.parametrize("ic", ["random_phase", "gaussian"])
def test_initial_condition_matches_oracle(ahs, oracle, prec, N, ic):
    seed = 180900995
    with ahs.Simulation(N=N, precision=prec, seed=seed, ic=ic, sigma=1.1) as sim:
        got = sim.get_fields()
    p = oracle.Params(N=N, sigma=1.1)
    ref = oracle.initial_condition(p, seed, oracle.IC_GAUSSIAN if ic == "gaussian" else oracle.IC_RANDOM_PHASE)
    assert not got[2:].any()
    if prec == "f32":
        ref32 = ref.astype(np.float32).astype(np.float64)
        # fp64 sincos on the device may differ from glibc by an ulp of fp64 -> at most 1 ulp of fp32 after rounding
        assert np.abs(got[:2] - ref32[:2]).max() <= 2.0 ** -23 * max(1.0, np.abs(ref[:2]).max())
        assert np.mean(got[:2] == ref32[:2]) > 0.999
    else:
        assert np.abs(got[:2] - ref[:2]).max() <= 4e-16 * max(1.0, np.abs(ref[:2]).max())


# ---------------------------------------------------------------------------------------------------------
# fields after 20 steps from an identical uploaded snapshot (north_star)
# ---------------------------------------------------------------------------------------------------------
CASES = [
    # N, precision, m, s, kernel
    (32, "f64", 1.0, 1.0, "generic"),     # config 1
    (32, "f32", 1.0, 0.0, "generic"),
    (20, "f64", 2.0, 0.5, "generic"),     # ragged: N not a multiple of the block size, several blocks
    (36, "f32", 2.0, 0.0, "generic"),
    (64, "f64", 1.0, 1.0, "auto"),
    (128, "f32", 1.0, 0.0, "auto"),       # config 2 / 4 physics, one fp32 tile wide (row-copy staging)
    (128, "f32", 2.0, 1.0, "auto"),       # config 3 physics (matter, s=1), 20 steps are inside the stable window
    (192, "f64", 1.0, 0.0, "auto"),       # three fp64 tiles in x: left-edge, interior and right-edge tiles of the TMA path
    (128, "f64", 1.0, 1.0, "auto"),       # config 5 physics, two fp64 tiles in x
    (256, "f32", 1.0, 0.0, "auto"),       # two fp32 tiles in x: left- and right-edge tiles of the TMA path, z-chunks of 16
    (384, "f32", 1.0, 0.0, "auto"),       # three fp32 tiles in x: left-edge, interior and right-edge TMA tiles
]
# strict fp32 bound not applicable (see the module docstring): eps ~ 30 after 20 steps
STRICT_EXEMPT = {(128, "f32", 2.0, 1.0)}


@pytest.mark.parametrize("N,prec,m,s,kernel", CASES)
def test_fields_after_20_steps(ahs, oracle, N, prec, m, s, kernel):
    from paper_1809_00995_b200 import synthetic
    nsteps = 20                           # north_star's 20 steps; the oracle (all cores) needs ~0.05 us per site-update
    with ahs.Simulation(N=N, precision=prec, m=m, s=s, ic="none", kernel=kernel) as sim:
        p = oracle_params(oracle, sim)
        ref = rounded(oracle.initial_condition(p, synthetic.SEED_PRIMARY), prec)   # the oracle's IC, uploaded
        sim.set_fields(ref, 0)
        sim.step(nsteps)
        got = sim.get_fields()
        assert sim.step_count == nsteps
        oracle.step(p, ref, 0, nsteps)
        assert_fields("fields_after_20_steps", got, ref, prec, oracle.FIELD_NAMES, strict=(N, prec, m, s) not in STRICT_EXEMPT,
                      N=N, m=m, s=s, kernel=sim.kernel_kind, nsteps=nsteps)
        # Gauss's law on the device trajectory itself
        d = sim.diagnostics()
        assert d["gauss_max"] <= (1e-12 if prec == "f64" else 2e-5) * max(1.0, d["gauss_rhs_rms"])
        check_diag(oracle, p, sim, prec, ref, nsteps)


@pytest.mark.parametrize("N,prec,kernel", [(24, "f64", "generic"), (24, "f32", "generic"), (64, "f64", "auto"), (128, "f32", "auto")])
def test_step_from_generic_snapshot(ahs, oracle, N, prec, kernel):
    """All ten fields non-zero (theta, eps, Pi of order 0.3): exercises every term of Eqs. 4-5 from step one."""
    from paper_1809_00995_b200 import synthetic
    f0 = synthetic.random_snapshot(N, seed=77)
    if prec == "f32":
        f0 = f0.astype(np.float32).astype(np.float64)
    nsteps = 3
    with ahs.Simulation(N=N, precision=prec, m=1.0, s=1.0, ic="none", kernel=kernel, tau0=2.0) as sim:
        p = oracle_params(oracle, sim)
        sim.set_fields(f0, step=7)
        assert np.array_equal(sim.get_fields(), f0)                 # round trip is exact
        np.testing.assert_allclose(sim.coefficients(7), oracle.coeffs(p, 7), rtol=1e-14)
        sim.step(nsteps)
        got = sim.get_fields()
        ref = oracle.step(p, f0.copy(), 7, nsteps)
        assert_fields("step_from_generic_snapshot", got, ref, prec, oracle.FIELD_NAMES, tol=1e-13 if prec == "f64" else 2e-5,
                      N=N, kernel=sim.kernel_kind, nsteps=nsteps)
        check_diag(oracle, p, sim, prec, ref, 7 + nsteps)


def test_march_and_generic_kernels_agree_on_device(ahs):
    """The two CUDA implementations are independent code: they must agree to rounding at sizes the oracle cannot reach."""
    # 512^3 fp32 / 256^3 fp64: four tiles in x, so left-edge, interior and right-edge tiles of the TMA path all occur
    for prec, N, tol in (("f32", 256, 2e-5), ("f64", 128, 1e-13), ("f32", 512, 2e-5), ("f64", 256, 1e-13)):
        with ahs.Simulation(N=N, precision=prec, kernel="auto", seed=5) as a, \
             ahs.Simulation(N=N, precision=prec, kernel="generic", seed=5) as b:
            if a.kernel_kind != "march":
                pytest.skip("z-marching kernel not available for this size")
            a.step(10); b.step(10)
            fa, fb = a.get_fields_native(), b.get_fields_native()
            for k in range(10):
                assert np.abs(fa[k] - fb[k]).max() <= tol * max(1.0, np.abs(fb[k]).max()), k
            da, db = a.diagnostics(), b.diagnostics()
            assert da["n_pierced"] > 0
            if np.array_equal(fa, fb):
                assert da["n_pierced"] == db["n_pierced"]
            # the two diagnostics implementations on ONE snapshot (the marching handle's): integers equal, sums to rounding
            b.set_fields_native(fa, step=10)
            db = b.diagnostics()
            assert (da["n_pierced"], da["sum_abs_w"]) == (db["n_pierced"], db["sum_abs_w"])
            rel = 1e-5 if prec == "f32" else 1e-11
            for key in ("v2_num", "v2_den", "v2v_num", "v2v_den", "mean_lagrangian", "gauss_rhs_rms"):
                assert da[key] == pytest.approx(db[key], rel=rel, abs=rel * abs(db["v2_den"]) if key.startswith("v2") else 0), key
            assert abs(da["gauss_max"] - db["gauss_max"]) <= (1e-5 if prec == "f32" else 1e-13) * max(1.0, db["gauss_rhs_rms"])


# ---------------------------------------------------------------------------------------------------------
# config 1 in full: 100 steps, diagnostics every 10 (literal reading finite to step ~80; also tau_ref = 11)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("tau_ref,last", [(0.0, 60), (11.0, 100)])
def test_config1_series(ahs, oracle, tau_ref, last):
    """Both paths run config 1 side by side from the oracle's IC; the series of diagnostics must agree."""
    from paper_1809_00995_b200 import synthetic
    kw = dict(N=32, precision="f64", m=1.0, s=1.0, tau_ref=tau_ref)
    with ahs.Simulation(ic="none", **kw) as sim, ahs.Simulation(ic="none", **kw) as probe:
        p = oracle_params(oracle, sim)
        ref = oracle.initial_condition(p, synthetic.SEED_PRIMARY)
        sim.set_fields(ref, 0)
        for n in range(0, last + 1, 10):
            if n:
                sim.step(10)
                oracle.step(p, ref, n - 10, 10)
            d = sim.diagnostics()                               # the device's own trajectory
            ro = oracle.diagnostics(p, ref, n)                  # the oracle's own trajectory
            assert d["n_pierced"] == ro["n_pierced"]
            assert d["xi"] == pytest.approx(ro["xi"], rel=1e-12)
            assert d["gauss_max"] < 1e-12 * max(1.0, d["gauss_rhs_rms"])
            K, G, Lg = oracle.site_fields(p, ref, n)
            assert abs(d["v2_num"] - ro["v2_num"]) <= 1e-8 * np.abs(K * Lg).sum() + 1e-300
            assert abs(d["v2_den"] - ro["v2_den"]) <= 1e-8 * np.abs(G * Lg).sum() + 1e-300
            check_diag(oracle, p, probe, "f64", ref, n)         # identical snapshot: bit-exact winding
            if n <= 20:
                assert max(field_errors(sim.get_fields(), ref)) <= 1e-12


def test_config1_literal_reading_goes_nonfinite_and_is_reported(ahs):
    """DESIGN.md R3: config 1 read literally (a = tau) leaves the leapfrog stability region before step 100."""
    with ahs.Simulation(N=32, precision="f64", m=1.0, s=1.0, seed=1) as sim:
        sim.step(60)
        assert sim.diagnostics()["nonfinite"] == 0
        sim.step(60)
        d = sim.diagnostics()
        f = sim.get_fields()
        assert d["nonfinite"] == 1 or np.abs(f[0:2]).max() > 1e3
        if d["nonfinite"]:
            with pytest.raises(ahs.AhsError) as e:
                sim.diagnostics(allow_nonfinite=False)
            assert e.value.code == ahs.AHS_ERR_NONFINITE


# ---------------------------------------------------------------------------------------------------------
# invariants on the device path itself (properties that hold at any size)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec,N", [("f64", 32), ("f32", 128)])
def test_vacuum_and_string_pair(ahs, oracle, prec, N):
    with ahs.Simulation(N=N, precision=prec, ic="none", m=1.0, s=1.0) as sim:
        f = np.zeros((10, N, N, N)); f[0] = 1.0
        sim.set_fields(f, 0)
        sim.step(5)
        assert np.array_equal(sim.get_fields(), f)                # the vacuum stays the vacuum, bitwise
        d = sim.diagnostics()
        assert d["n_pierced"] == 0 and math.isinf(d["xi"]) and d["gauss_max"] == 0.0
    M = 16 if N == 32 else N
    if prec == "f64":
        M = 16
    z, y, x = np.meshgrid(np.arange(M), np.arange(M), np.arange(M), indexing="ij")
    th = np.arctan2(y - (M / 2 - 0.5), x - (M / 4 - 0.5)) - np.arctan2(y - (M / 2 - 0.5), x - (3 * M / 4 - 0.5))
    f = np.zeros((10, M, M, M)); f[0] = np.cos(th); f[1] = np.sin(th)
    with ahs.Simulation(N=M, precision=prec, ic="none") as sim:
        sim.set_fields(f, 0)
        d = sim.diagnostics()
        assert d["n_pierced"] == 2 * M and d["sum_abs_w"] == 2 * M       # north_star: exactly 2N pierced plaquettes
        assert d["L"] == pytest.approx(math.pi / 6 * 0.5 * 2 * M)


@pytest.mark.parametrize("prec,N", [("f64", 32), ("f32", 64)])
def test_gauge_transformation_leaves_diagnostics_unchanged(ahs, oracle, prec, N):
    from paper_1809_00995_b200 import synthetic
    with ahs.Simulation(N=N, precision=prec, ic="none", m=1.0, s=0.0) as sim:
        p = oracle_params(oracle, sim)
        f = oracle.step(p, oracle.initial_condition(p, 3), 0, 30)
        sim.set_fields(f, 30)
        d0 = sim.diagnostics()
        al = synthetic.gauge_angles(N, seed=9)
        g = f.copy()
        c, s_ = np.cos(al), np.sin(al)
        g[0], g[1] = f[0] * c - f[1] * s_, f[0] * s_ + f[1] * c
        g[2], g[3] = f[2] * c - f[3] * s_, f[2] * s_ + f[3] * c
        for i in range(3):
            g[4 + i] = f[4 + i] + (np.roll(al, -1, axis=2 - i) - al)
        sim.set_fields(g, 30)
        d1 = sim.diagnostics()
        if prec == "f64":
            assert d1["n_pierced"] == d0["n_pierced"] and d0["n_pierced"] > 0
            assert d1["v2"] == pytest.approx(d0["v2"], rel=1e-9)
        else:
            # fp32 storage rounds the transformed fields: counts may move by a few ties, sums by ~1e-5
            assert abs(int(d1["n_pierced"]) - int(d0["n_pierced"])) <= 1e-4 * d0["n_pierced"] + 2
            assert d1["v2"] == pytest.approx(d0["v2"], rel=2e-3)


@pytest.mark.parametrize("N,prec,kernel", [(48, "f32", "generic"), (128, "f32", "auto"), (128, "f64", "auto")])
def test_long_run_series_vs_oracle(ahs, oracle, N, prec, kernel):
    """north_star: long-run xi(tau) and <v^2> agree within 2 % (GPU trajectory vs the fp64 oracle's own trajectory from the
    same initial condition, config-2 physics: radiation era, s = 0), to tau = 33, diagnostics every 20 steps.  The 128^3 cases run
    the z-marching kernels (kernel="auto"), i.e. the kernels bench.py times.  <v^2>_L is a ratio with a sign-indefinite
    weight (R16): the 2 % criterion is applied to it where |den| is well away from 0, and to <v^2>_V always."""
    nsteps, every = 320, 20
    with ahs.Simulation(N=N, precision=prec, ic="none", m=1.0, s=0.0, kernel=kernel) as sim:
        if kernel == "auto":
            assert sim.kernel_kind == "march"
        p = oracle_params(oracle, sim)
        ref = rounded(oracle.initial_condition(p, 11), prec)
        sim.set_fields(ref, 0)
        series = []
        for n in range(every, nsteps + 1, every):
            sim.step(every)
            oracle.step(p, ref, n - every, every)
            d = sim.diagnostics()
            r = oracle.diagnostics(p, ref, n)
            K, G, Lg = oracle.site_fields(p, ref, n)
            den_ok = abs(r["v2_den"]) > 0.05 * np.abs(G * Lg).sum()
            series.append(dict(n=n, xi=(d["xi"], r["xi"]), n_pierced=(d["n_pierced"], r["n_pierced"]), v2_V=(d["v2_V"], r["v2_V"]),
                               v2_L=(d["v2"], r["v2"]), den_ok=bool(den_ok), gauss=d["gauss_max"]))
            assert d["xi"] == pytest.approx(r["xi"], rel=0.02), series
            assert abs(int(d["n_pierced"]) - int(r["n_pierced"])) <= 0.02 * r["n_pierced"], series
            assert d["v2_V"] == pytest.approx(r["v2_V"], rel=0.02), series
            if den_ok:
                assert d["v2"] == pytest.approx(r["v2"], rel=0.02), series
            assert d["gauss_max"] < (5e-5 if prec == "f32" else 1e-12) * max(1.0, d["gauss_rhs_rms"]), series
        got = sim.get_fields()
        err = field_errors(got, ref)
        rel = lambda a, b: abs(a - b) / abs(b)
        record("long_run_series", N=N, prec=prec, kernel=sim.kernel_kind, nsteps=nsteps, max_field_err_r14=max(err),
               max_dphi=float(np.abs(got[:2] - ref[:2]).max()),
               max_rel_xi=max(rel(*x["xi"]) for x in series), max_rel_v2_V=max(rel(*x["v2_V"]) for x in series),
               max_rel_v2_L_where_den_ok=max([rel(*x["v2_L"]) for x in series if x["den_ok"]] or [0.0]),
               n_pierced_equal_at=sum(x["n_pierced"][0] == x["n_pierced"][1] for x in series), calls=len(series))
        # no chaotic divergence -- fp32 arithmetic drifts from fp64 by ~1e-4 in phi over 160-320 steps
        assert max(err) < (5e-3 if prec == "f32" else 1e-10), err


def test_native_transfer_and_device_pointers(ahs):
    import torch
    N = 32
    with ahs.Simulation(N=N, precision="f32", seed=2) as sim:
        sim.step(3)
        a = sim.get_fields_native()
        assert a.dtype == np.float32 and np.array_equal(a.astype(np.float64), sim.get_fields())
        pinned = torch.empty((10, N, N, N), dtype=torch.float32).pin_memory()
        sim.get_fields_native(pinned.data_ptr())
        assert np.array_equal(pinned.numpy(), a)
        sim.set_fields_native(pinned.data_ptr(), step=3)
        assert np.array_equal(sim.get_fields_native(), a)
        sim.step(1)
        sim.set_fields_native(pinned.data_ptr(), step=3, wait=False)      # ahs_set_fields_native_async: ordered on the handle's stream
        sim.step(2)
        b = sim.get_fields_native()
        sim.set_fields_native(a, step=3)
        sim.step(2)
        assert sim.step_count == 5 and np.array_equal(sim.get_fields_native(), b)
        sim.set_fields_native(a, step=3)
        ptr = sim.field_device_ptr(0)
        assert ptr != 0 and ptr % 256 == 0
        st, tau, nl = sim.state()
        assert st == 3 and tau == pytest.approx(1.3) and nl >= 4
    # the plain north_star constructor: library-owned memory, default stream
    h = ahs.create(32, 0.5, 0.1, 2.0, 1.0, 1.0, 1.0, 0.0, 1.0, 5)
    lib = ahs.load()
    import ctypes as C
    assert lib.ahs_step(C.c_void_p(h), 2) == 0
    L, v2, g = C.c_double(), C.c_double(), C.c_double()
    assert lib.ahs_diagnostics(C.c_void_p(h), C.byref(L), C.byref(v2), C.byref(g)) == 0
    assert L.value > 0 and g.value < 1e-5
    ahs.destroy_raw(h)


def test_create_rejects_bad_arguments(ahs):
    for kw in (dict(N=2), dict(N=32, dt=0.0), dict(N=32, tau0=0.01, m=1.0), dict(N=32, precision="f32", kernel="march")):
        with pytest.raises(ahs.AhsError):
            ahs.Simulation(**kw)


@pytest.mark.parametrize("prec,N", [("f64", 64), ("f32", 128)])
def test_winding_bit_exact_when_links_sit_next_to_ties(ahs, oracle, prec, N):
    """The marching diagnostics kernel decides rint() from fp32 phases and falls back to fp64 when a link is within
    4e-6 (1 + |t|) turns of a half-integer.  Here a third of the links are PUT next to a tie, at
    distances from 1e-12 to 1e-4 turns on either side, so fast path, fallback and the boundary between them are all
    hit; the count must still equal the oracle's fp64 decision, integer for integer."""
    rng = np.random.default_rng(20260101 + N)
    f = np.zeros((10, N, N, N))
    ph = rng.uniform(-np.pi, np.pi, (N, N, N))
    mod = 1.0 + 0.3 * rng.standard_normal((N, N, N))
    f[0], f[1] = mod * np.cos(ph), mod * np.sin(ph)
    f = rounded(f, prec)
    arg = np.arctan2(f[1], f[0])
    for i, ax in enumerate((2, 1, 0)):                      # direction i = x, y, z <-> numpy axis 2, 1, 0
        d = np.roll(arg, -1, axis=ax) - arg
        turns = rng.integers(-2, 3, (N, N, N)) + 0.5
        off = rng.choice([-1.0, 1.0], (N, N, N)) * 10.0 ** rng.uniform(-12, -4, (N, N, N))
        near = d - 2 * np.pi * (turns + off)                # (d - theta) / 2 pi = turns + off
        plain = 0.3 * rng.standard_normal((N, N, N))
        f[4 + i] = np.where(rng.random((N, N, N)) < 1 / 3, near, plain)
    f = rounded(f, prec)
    p = oracle.Params(N=N, m=1.0, s=0.0)
    for kernel in ("auto", "generic"):
        with ahs.Simulation(N=N, precision=prec, m=1.0, s=0.0, ic="none", kernel=kernel) as sim:
            sim.set_fields(f, 0)
            d = sim.diagnostics()
        r = oracle.diagnostics(p, f, 0)
        assert r["n_pierced"] > N ** 3 // 10
        assert (d["n_pierced"], d["sum_abs_w"]) == (r["n_pierced"], r["sum_abs_w"]), kernel


# ---------------------------------------------------------------------------------------------------------
# full size (BASELINE.json configs[3]: 1024^3 fp32, the launch configuration bench.py times), sampled outputs
# ---------------------------------------------------------------------------------------------------------
class _DeviceArray:
    """Zero-copy view of a live field (ahs_field_device_ptr) for torch.as_tensor."""

    def __init__(self, ptr, N, typestr):
        self.__cuda_array_interface__ = {"shape": (N, N, N), "typestr": typestr, "data": (ptr, False), "version": 2}


def _gather_window(sim, origin, B):
    import torch
    N = sim.N
    typestr = "<f4" if sim.dtype == np.float32 else "<f8"
    ix = [torch.as_tensor((np.arange(o, o + B) % N), device="cuda") for o in origin]
    out = np.empty((10, B, B, B))
    for k in range(10):
        t = torch.as_tensor(_DeviceArray(sim.field_device_ptr(k), N, typestr), device="cuda")
        out[k] = t[ix[2][:, None, None], ix[1][None, :, None], ix[0][None, None, :]].double().cpu().numpy()
    return out


def test_full_size_1024_sampled_windows_and_closed_forms(ahs, oracle):
    """configs[3] at full size, north_star's 20 steps, in the launch configuration bench.py times.  (1) Sampled outputs:
    the oracle generates the initial condition of small windows of the 1024^3 lattice from the Philox specification
    (aho_ic_window), steps each window 20 times as a periodic 56^3 lattice and is compared on the 16^3 interior that the
    wrong wrap cannot have reached (one site per step, halo 20) -- interiors sit on tile corners of the march (x multiple
    of 128, y multiple of 4), on its z-chunk boundaries (z multiple of 64) and on the periodic corner of the lattice, so
    interior, left-edge and right-edge TMA tiles and the y-edge row-copy tiles are all sampled.  Strict norm: max |d| <= 2e-4.
    (2) Properties that hold at any size: closed forms of the diagnostics on the random-phase initial condition, Gauss's
    law at fp32 roundoff after stepping."""
    import torch
    N, nsteps, halo, inner = 1024, 20, 20, 16
    free, _ = torch.cuda.mem_get_info()
    if free < ahs.required_bytes(N, "f32") + (2 << 30):
        pytest.skip("needs %.0f GB of free device memory" % (ahs.required_bytes(N, "f32") / 1e9))
    seed, B = 180900995, inner + 2 * halo
    with ahs.Simulation(N=N, precision="f32", m=1.0, s=0.0, seed=seed) as sim:
        assert sim.kernel_kind == "march"
        d0 = sim.diagnostics()
        sites = float(N) ** 3
        # i.i.d. uniform phases: a plaquette is pierced with probability 1/3; with theta = Pi = eps = 0 and |phi| = sigma,
        # Lag = -G, G = (1/dx^2) sum_i 2 (1 - cos D_i) with D_i i.i.d. uniform: E G = 24, E G^2 = 672 at dx = 0.5
        assert abs(d0["n_pierced"] / (3 * sites) - 1 / 3) < 1e-4
        assert d0["v2_num"] == 0.0 and d0["gauss_max"] == 0.0 and d0["nonfinite"] == 0
        assert d0["mean_lagrangian"] == pytest.approx(-24.0, rel=1e-3)
        assert d0["v2_den"] / sites == pytest.approx(-672.0, rel=2e-3)
        sim.step(nsteps)
        rng = np.random.default_rng(5)
        # first site of each compared 16^3 interior
        interiors = [(-8, -8, -8), (128 - 8, 4 - 8, 64 - 8), (512 - 2, 700 + 1, 128 - 6), (1024 - 128 - 5, 1024 - 4 - 6, 960),
                     (896 - 8, 512 - 8, 1024 - 64 - 8), (-8, 300, 448 - 8)]
        interiors += [tuple(int(v) for v in rng.integers(0, N, 3)) for _ in range(4)]
        pw = oracle.Params(N=B, m=1.0, s=0.0)
        sl = slice(halo, halo + inner)
        worst = np.zeros(10)
        for io in interiors:
            origin = tuple(v - halo for v in io)
            ref = rounded(oracle.initial_condition_window(pw, seed, N, origin), "f32")
            oracle.step(pw, ref, 0, nsteps)
            got = _gather_window(sim, origin, B)
            for k in range(10):
                d = np.abs(got[k][sl, sl, sl] - ref[k][sl, sl, sl]).max()
                worst[k] = max(worst[k], d)
                assert d <= TOL["f32"], (io, oracle.FIELD_NAMES[k], d)                                          # strict: absolute
                assert d / max(1.0, np.abs(ref[k][sl, sl, sl]).max()) <= TOL["f32"], (io, oracle.FIELD_NAMES[k], d)   # R14
        record("full_size_1024_windows", nsteps=nsteps, windows=len(interiors), inner=inner, halo=halo, max_strict=float(worst.max()),
               strict_per_field={n: float("%.3g" % e) for n, e in zip(oracle.FIELD_NAMES, worst)})
        d = sim.diagnostics()
        assert d["nonfinite"] == 0 and d["step"] == nsteps
        assert d["gauss_max"] <= 2e-5 * max(1.0, d["gauss_rhs_rms"])


def test_full_size_512_fp64_sampled_windows(ahs, oracle):
    """configs[4] (512^3 fp64, m = 1, s = 1, the configuration bench.py --lattice 512 --precision f64 times) at full size, north_star's
    20 steps: sampled windows as in the 1024^3 test (the oracle steps each window as a periodic 56^3 lattice from the Philox initial
    condition of that window; compared on the 16^3 interior the wrong wrap cannot have reached).  Interiors sit on tile corners of the
    fp64 march (x multiple of 64, y multiple of 4), on its z-chunk boundaries (z multiple of 32) and on the periodic corner.  Strict
    norm: max |d| / max |oracle| <= 1e-12 over the interior, per field array; then the diagnostics' closed forms and Gauss's law."""
    N, nsteps, halo, inner = 512, 20, 20, 16
    seed, B = 180900995, inner + 2 * halo
    with ahs.Simulation(N=N, precision="f64", m=1.0, s=1.0, seed=seed) as sim:
        assert sim.kernel_kind == "march"
        sim.step(nsteps)
        rng = np.random.default_rng(9)
        interiors = [(-8, -8, -8), (64 - 8, 4 - 8, 32 - 8), (256 - 2, 300 + 1, 96 - 6), (512 - 64 - 5, 512 - 4 - 6, 480),
                     (448 - 8, 256 - 8, 512 - 32 - 8), (-8, 200, 224 - 8)]
        interiors += [tuple(int(v) for v in rng.integers(0, N, 3)) for _ in range(2)]
        pw = oracle.Params(N=B, m=1.0, s=1.0)
        sl = slice(halo, halo + inner)
        worst = np.zeros(10)
        for io in interiors:
            origin = tuple(v - halo for v in io)
            ref = oracle.initial_condition_window(pw, seed, N, origin)
            oracle.step(pw, ref, 0, nsteps)
            got = _gather_window(sim, origin, B)
            for k in range(10):
                d = np.abs(got[k][sl, sl, sl] - ref[k][sl, sl, sl]).max() / np.abs(ref[k][sl, sl, sl]).max()
                worst[k] = max(worst[k], d)
                assert d <= TOL["f64"], (io, oracle.FIELD_NAMES[k], d)
        record("full_size_512_fp64_windows", nsteps=nsteps, windows=len(interiors), inner=inner, halo=halo, max_strict=float(worst.max()),
               strict_per_field={n: float("%.3g" % e) for n, e in zip(oracle.FIELD_NAMES, worst)})
        d = sim.diagnostics()
        assert d["nonfinite"] == 0 and d["step"] == nsteps
        assert d["gauss_max"] <= 1e-12 * max(1.0, d["gauss_rhs_rms"])


def test_config3_gaussian_ic_fields_after_20_steps(ahs, oracle):
    """BASELINE config 3 as configured except for the size: fp32, matter era (m = 2), true equations (s = 1), literal a = (tau/tau0)^m,
    GAUSSIAN initial condition (amplitudes from 0 to ~3 sigma, not |phi| = sigma) -- the whole 128^3 lattice against the oracle after
    north_star's 20 steps, from the oracle's Gaussian IC uploaded to the device.  R14 norm asserted; the strict absolute norm is
    recorded and bounded by 2e-4 x the field's own maximum (eps grows to ~30 in these 20 steps, SURVEY 8(c) 'Config consequences of
    G3': 2e-4 absolute is below one fp32 ulp of such a value)."""
    N, nsteps = 128, 20
    with ahs.Simulation(N=N, precision="f32", m=2.0, s=1.0, ic="none") as sim:
        p = oracle_params(oracle, sim)
        ref = rounded(oracle.initial_condition(p, 180900995, kind=oracle.IC_GAUSSIAN), "f32")
        assert np.abs(np.hypot(ref[0], ref[1]) - 1.0).max() > 0.5          # not the random-phase IC
        sim.set_fields(ref, 0)
        sim.step(nsteps)
        got = sim.get_fields()
        oracle.step(p, ref, 0, nsteps)
        assert_fields("config3_gaussian_128", got, ref, "f32", oracle.FIELD_NAMES, strict=False, N=N, m=2.0, s=1.0, kernel=sim.kernel_kind, nsteps=nsteps)
        d = sim.diagnostics()
        assert d["gauss_max"] <= 2e-5 * max(1.0, d["gauss_rhs_rms"])
        check_diag(oracle, p, sim, "f32", ref, nsteps)


def test_full_size_512_config3_sampled_windows(ahs, oracle):
    """configs[2] (BASELINE config 3) as configured and at full size: 512^3 fp32, m = 2, s = 1, a = (tau/tau0)^m read literally, the
    DEVICE's own Gaussian initial condition (ahs_ic.cu), 20 steps.  Sampled windows as in the 1024^3 test: the oracle generates the
    Gaussian IC of each 56^3 window from the Philox specification (aho_ic_window, kind 1), steps it 20 times as a small periodic
    lattice and is compared on the 16^3 interior the wrong wrap cannot have reached.  Interiors sit on tile corners of the fp32 march
    (x multiple of 128, y multiple of 4), on z-chunk boundaries and on the periodic corner.  R14 norm asserted (max |d| /
    max(1, max |oracle|) <= 2e-4); the strict absolute maximum is recorded."""
    N, nsteps, halo, inner = 512, 20, 20, 16
    seed, B = 180900995, inner + 2 * halo
    with ahs.Simulation(N=N, precision="f32", m=2.0, s=1.0, ic="gaussian", seed=seed) as sim:
        assert sim.kernel_kind == "march"
        sim.step(nsteps)
        rng = np.random.default_rng(13)
        interiors = [(-8, -8, -8), (128 - 8, 4 - 8, 32 - 8), (256 - 2, 300 + 1, 96 - 6), (512 - 128 - 5, 512 - 4 - 6, 480),
                     (384 - 8, 256 - 8, 512 - 16 - 8), (-8, 200, 224 - 8)]
        interiors += [tuple(int(v) for v in rng.integers(0, N, 3)) for _ in range(2)]
        pw = oracle.Params(N=B, m=2.0, s=1.0)
        sl = slice(halo, halo + inner)
        worst, worst_r14 = np.zeros(10), np.zeros(10)
        for io in interiors:
            origin = tuple(v - halo for v in io)
            ref = rounded(oracle.initial_condition_window(pw, seed, N, origin, kind=oracle.IC_GAUSSIAN), "f32")
            oracle.step(pw, ref, 0, nsteps)
            got = _gather_window(sim, origin, B)
            for k in range(10):
                d = np.abs(got[k][sl, sl, sl] - ref[k][sl, sl, sl]).max()
                r14 = d / max(1.0, np.abs(ref[k][sl, sl, sl]).max())
                worst[k], worst_r14[k] = max(worst[k], d), max(worst_r14[k], r14)
                assert r14 <= TOL["f32"], (io, oracle.FIELD_NAMES[k], d, r14)
        record("full_size_512_config3_windows", nsteps=nsteps, windows=len(interiors), inner=inner, halo=halo, max_r14=float(worst_r14.max()),
               max_strict=float(worst.max()), strict_per_field={n: float("%.3g" % e) for n, e in zip(oracle.FIELD_NAMES, worst)})
        d = sim.diagnostics()
        assert d["nonfinite"] == 0 and d["step"] == nsteps and d["n_pierced"] > 0
        assert d["gauss_max"] <= 2e-5 * max(1.0, d["gauss_rhs_rms"])


@pytest.mark.parametrize("prec,N", [("f32", 256), ("f64", 128)])
def test_repeated_diagnostics_are_bit_identical(ahs, prec, N):
    """The diagnostics march hands phases round inside a warp through shared memory (fp32) and re-fills its stage ring from whichever warp
    releases a slot last: 100 calls on one snapshot must return the same record bit for bit (integer counts; fp64 sums in a fixed order
    for a fixed launch shape), under both staging modes.  A race in either mechanism would show as a count or a sum that moves."""
    with ahs.Simulation(N=N, precision=prec, seed=5) as sim:
        sim.step(15)
        for staging in (ahs.AHS_STAGING_TENSOR, ahs.AHS_STAGING_ROWS):
            sim.set_option(ahs.AHS_OPT_STAGING, staging)
            first = sim.diagnostics()
            assert first["n_pierced"] > 0 and first["nonfinite"] == 0
            for _ in range(100):
                d = sim.diagnostics()
                assert all(d[k] == first[k] or (d[k] != d[k] and first[k] != first[k]) for k in first), [k for k in first if d[k] != first[k]]


def test_long_window_is_deterministic_and_keeps_gauss_law(ahs):
    """Regression for a shared-memory race of the marching step kernel (profiles/HISTORY.md, "r2 race"): a tensor / bulk copy
    issued right after __syncthreads() could overwrite a stage other warps were still reading -- about one corrupted
    site per 500 launches at 512^3, visible as a Gauss-law violation of 1e-2 and as run-to-run differences.  Two runs of
    60 back-to-back launches must agree bit for bit and keep Gauss's law at fp32 roundoff."""
    import hashlib
    out = []
    for _ in range(2):
        with ahs.Simulation(N=512, precision="f32", m=1.0, s=0.0, seed=180900995) as sim:
            sim.step(60)
            d = sim.diagnostics()
            out.append((hashlib.md5(sim.get_fields_native().tobytes()).hexdigest(), d["n_pierced"], d["v2_num"], d["gauss_max"]))
            assert d["gauss_max"] <= 2e-5 * max(1.0, d["gauss_rhs_rms"]), d
    assert out[0] == out[1]


def test_chunk_starts_under_stress_are_bit_identical(ahs):
    """The hand-over of the prologue's stages to the copy engine at every z-chunk start (profiles/HISTORY.md, "r2 race"): 1000 launches at
    256^3 with 128 chunks per tile -- a chunk start every second plane, 3.4e7 hand-overs per run, 64 x the default shape's -- in both
    staging modes.  A stage overwritten while a slower warp still reads it corrupts a site; the fields must instead equal the
    default launch shape's bit for bit (they do not depend on where the chunk boundaries fall) and Gauss's law must hold."""
    import hashlib
    N, nsteps = 256, 1000
    digests = {}
    for name, opts in (("default", {}), ("128 chunks, tensor maps", {ahs.AHS_OPT_STEP_CHUNKS: 128}),
                       ("128 chunks, row copies", {ahs.AHS_OPT_STEP_CHUNKS: 128, ahs.AHS_OPT_STAGING: ahs.AHS_STAGING_ROWS}),
                       ("85 chunks (uneven), tensor maps", {ahs.AHS_OPT_STEP_CHUNKS: 85})):
        with ahs.Simulation(N=N, precision="f32", m=1.0, s=0.0, seed=180900995) as sim:
            for k, v in opts.items():
                sim.set_option(k, v)
            sim.step(nsteps)
            d = sim.diagnostics()
            assert d["nonfinite"] == 0 and d["gauss_max"] <= 2e-5 * max(1.0, d["gauss_rhs_rms"]), (name, d)
            digests[name] = (hashlib.md5(sim.get_fields_native().tobytes()).hexdigest(), d["n_pierced"])
    assert len(set(digests.values())) == 1, digests


def test_c_B_parameter_reaches_the_weight(ahs, oracle):
    """ahs_params.c_B (R2) and c_E (R21): the factors on the plaquette sum and on the electric term of Eq. 2 enter the Lagrangian
    weight only; c_B = 0.5 is Eq. 2 as printed, c_E = (dt/dx)^2 = 0.04 the rescaling of E that L44 states."""
    from paper_1809_00995_b200 import synthetic
    for prec, N, kernel in (("f64", 64, "auto"), ("f32", 128, "auto"), ("f64", 24, "generic")):
        f = rounded(synthetic.random_snapshot(N, seed=5), prec)
        for cB, cE in ((0.5, 1.0), (1.0, 1.0), (1.0, 0.04), (0.5, 0.04)):
            p = oracle.Params(N=N, m=1.0, s=0.0, c_B=cB, c_E=cE)
            with ahs.Simulation(N=N, precision=prec, m=1.0, s=0.0, ic="none", c_B=cB, c_E=cE, kernel=kernel) as sim:
                sim.set_fields(f, 4)
                d = sim.diagnostics()
            r = oracle.diagnostics(p, f, 4)
            K, G, Lg = oracle.site_fields(p, f, 4)
            rel = 1e-10 if prec == "f64" else 2e-5
            assert abs(d["v2_num"] - r["v2_num"]) <= rel * np.abs(K * Lg).sum()
            assert abs(d["mean_lagrangian"] - r["mean_lagrangian"]) <= rel * np.abs(Lg).mean()
            assert d["n_pierced"] == r["n_pierced"] and d["v2v_num"] == pytest.approx(r["v2v_num"], rel=rel)
            assert d["v2_omega"] == pytest.approx(r["v2_omega"], rel=100 * rel)


# ---------------------------------------------------------------------------------------------------------
# tuning options (ahs_set_option), several handles, the non-finite flag
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec,N", [("f32", 256), ("f64", 128)])
def test_options_change_the_launch_shape_not_the_result(ahs, prec, N):
    """Every accepted value of ahs_set_option: row-copy staging instead of tensor-map TMA, and z-chunk counts from one chunk
    per tile to chunks of 2 and 3 planes (uneven: 100 and 37 do not divide N), which multiplies the chunk starts where the
    march hands its first stages over to the copy engine.  Fields must be bit-identical to the default launch shape
    (each site's arithmetic does not depend on the tiling); the integer counts equal; the fp64 sums equal to reduction order."""
    with ahs.Simulation(N=N, precision=prec, seed=21) as ref:
        ref.step(6)
        want, dref = ref.get_fields_native(), ref.diagnostics()
    settings = [{ahs.AHS_OPT_STAGING: ahs.AHS_STAGING_ROWS}, {ahs.AHS_OPT_STEP_CHUNKS: 1, ahs.AHS_OPT_DIAG_CHUNKS: 1},
                {ahs.AHS_OPT_STEP_CHUNKS: 100, ahs.AHS_OPT_DIAG_CHUNKS: 37}, {ahs.AHS_OPT_STEP_CHUNKS: N // 2, ahs.AHS_OPT_DIAG_CHUNKS: N // 4},
                {ahs.AHS_OPT_STAGING: ahs.AHS_STAGING_ROWS, ahs.AHS_OPT_STEP_CHUNKS: 37, ahs.AHS_OPT_DIAG_CHUNKS: 5},
                {ahs.AHS_OPT_STEP_PDL: 1}, {ahs.AHS_OPT_STEP_PDL: 1, ahs.AHS_OPT_STEP_CHUNKS: 100, ahs.AHS_OPT_STAGING: ahs.AHS_STAGING_ROWS}]
    for opts in settings:
        with ahs.Simulation(N=N, precision=prec, seed=21) as sim:
            for k, v in opts.items():
                sim.set_option(k, v)
            sim.step(6)
            assert np.array_equal(sim.get_fields_native(), want), opts
            d = sim.diagnostics()
            assert (d["n_pierced"], d["sum_abs_w"], d["nonfinite"]) == (dref["n_pierced"], dref["sum_abs_w"], 0), opts
            for key in ("v2_num", "v2_den", "v2v_num", "v2v_den", "mean_lagrangian", "gauss_rhs_rms"):
                assert d[key] == pytest.approx(dref[key], rel=1e-11, abs=1e-11 * abs(dref["v2_den"])), (opts, key)
            assert d["gauss_max"] == dref["gauss_max"], opts
    with ahs.Simulation(N=N, precision=prec) as sim:
        for bad in ((99, 0), (ahs.AHS_OPT_STAGING, 2), (ahs.AHS_OPT_STEP_CHUNKS, N + 1), (ahs.AHS_OPT_DIAG_CHUNKS, -1), (ahs.AHS_OPT_DIAG_TRIG, 2), (ahs.AHS_OPT_STEP_PDL, 2)):
            with pytest.raises(ahs.AhsError) as e:
                sim.set_option(*bad)
            assert e.value.code == ahs.AHS_ERR_INVALID_ARG


@pytest.mark.parametrize("N", [128, 256])
def test_diag_trig_option_both_settings_against_the_oracle(ahs, oracle, N):
    """AHS_OPT_DIAG_TRIG: the sums of Eqs. 2, 9, 10, 12 on an fp32 lattice with the special-function unit's sine / cosine (default)
    and with the polynomial routines, each against the oracle on the same snapshot with the SAME bar (check_diag; 2e-5 of the
    absolute sums).  Observed (recorded): ~1.5e-7 and ~1e-8.  The winding count and the Gauss residual do not depend on the
    setting; an fp64 lattice ignores it bit for bit."""
    O = oracle
    with ahs.Simulation(N=N, precision="f32", seed=77) as sim:
        p = oracle_params(O, sim)
        snap = O.initial_condition(p, seed=77)
        O.step(p, snap, 0, 12)
        got = {}
        for name, v in (("hardware", ahs.AHS_TRIG_HARDWARE), ("polynomial", ahs.AHS_TRIG_POLYNOMIAL)):
            sim.set_option(ahs.AHS_OPT_DIAG_TRIG, v)
            got[name], r = check_diag(O, p, sim, "f32", snap, 12)
        h, q = got["hardware"], got["polynomial"]
        assert (h["n_pierced"], h["sum_abs_w"], h["gauss_max"]) == (q["n_pierced"], q["sum_abs_w"], q["gauss_max"])
        assert h["v2_num"] != q["v2_num"]                       # (the two settings really are two code paths)
        for key in ("v2_num", "v2_den", "eos_num", "eos_den"):
            assert abs(q[key] - r[key]) <= 2e-7 * abs(r["v2_den"]), key     # the polynomials stay at the 1e-8 level
    with ahs.Simulation(N=128, precision="f64", seed=77) as sim:
        sim.step(3)
        a = sim.diagnostics()
        sim.set_option(ahs.AHS_OPT_DIAG_TRIG, ahs.AHS_TRIG_POLYNOMIAL)
        b = sim.diagnostics()
        assert all(b[k] == a[k] or (a[k] != a[k] and b[k] != b[k]) for k in a)      # (xi_L is NaN while the mean Lagrangian is > 0)


def test_two_handles_on_two_streams_interleaved(ahs):
    """Distinct handles are independent (include/ahs.h): two replicas on two streams, their steps and asynchronous
    diagnostics interleaved from one host thread, give what each gives alone."""
    import torch
    N = 256
    alone = []
    for seed in (1, 2):
        with ahs.Simulation(N=N, precision="f32", seed=seed) as sim:
            sim.step(8)
            alone.append((sim.diagnostics(), sim.get_fields_native()))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    sims = []
    for seed, st in zip((1, 2), streams):
        with torch.cuda.stream(st):
            sims.append(ahs.Simulation(N=N, precision="f32", seed=seed))
    assert sims[0].stream_handle != sims[1].stream_handle
    for _ in range(4):
        for sim in sims:
            sim.step(1)
        for sim in sims:
            sim.diagnostics_launch()
        for sim in reversed(sims):
            sim.step(1)
    got = [sim.diagnostics_fetch() for sim in sims]          # the record of the LAST launch (step 7)
    for sim, (d_alone, f_alone), g in zip(sims, alone, got):
        assert g["step"] == 7
        d = sim.diagnostics()
        assert d["step"] == 8 and d["n_pierced"] == d_alone["n_pierced"] and d["v2_num"] == d_alone["v2_num"]
        assert np.array_equal(sim.get_fields_native(), f_alone)
        sim.destroy()


@pytest.mark.parametrize("prec,N,kernel", [("f32", 128, "auto"), ("f32", 128, "generic"), ("f64", 64, "auto"), ("f64", 24, "generic")])
def test_nonfinite_flag_means_a_stored_value_is_not_finite(ahs, oracle, prec, N, kernel):
    """include/ahs.h: `nonfinite` is about the ten stored arrays, on both diagnostics implementations and on the oracle: a NaN
    or an infinity in any one of them sets it; a finite value whose square overflows the storage type does not."""
    from paper_1809_00995_b200 import synthetic
    base = rounded(synthetic.random_snapshot(N, seed=8), prec)
    p = oracle.Params(N=N, m=1.0, s=0.0)
    rng = np.random.default_rng(0)
    with ahs.Simulation(N=N, precision=prec, m=1.0, s=0.0, ic="none", kernel=kernel) as sim:
        for k in range(10):
            f = base.copy()
            z, y, x = (int(v) for v in rng.integers(0, N, 3))
            f[k, z, y, x] = np.nan if k % 2 else np.inf
            sim.set_fields(f, 0)
            assert sim.diagnostics()["nonfinite"] == 1, oracle.FIELD_NAMES[k]
            if k in (0, 5, 9):
                assert oracle.diagnostics(p, f, 0)["nonfinite"] == 1
        big = 1e20 if prec == "f32" else 1e160
        for k in (0, 2, 7):
            f = base.copy()
            f[k, N // 2, 1, N - 1] = big
            sim.set_fields(f, 0)
            d = sim.diagnostics()
            assert d["nonfinite"] == 0 and not math.isfinite(d["mean_lagrangian"]), oracle.FIELD_NAMES[k]
            assert oracle.diagnostics(p, f, 0)["nonfinite"] == 0
        sim.set_fields(base, 0)
        assert sim.diagnostics()["nonfinite"] == 0


def test_table4_script_runs_through_the_library(ahs):
    """paper_1809_00995_b200/table4.py (the s = 0 rows of the paper's Table 4) on a 128^3 box, one seed per era:
    far too small to be in scaling, so only sanity is asserted -- finite numbers, the mean string separation growing at a rate of
    the paper's order (0.3), velocities between 0 and 1, Gauss's law at fp32 roundoff."""
    from paper_1809_00995_b200 import table4
    N = 128
    steps = int(round(N * 0.5 / 2 / 0.1))
    for m in (1.0, 2.0):
        r = table4.run(N, m, seed=1, steps=steps - steps % 10, every=10, fit_from=16.0, precision="f32", c_B=0.0, c_E=0.0)
        assert all(math.isfinite(v) for v in r.values()), r
        assert 0.2 < r["xi_dot"] < 0.5 and 0.15 < r["xi_L_dot"] < 0.6, r
        assert 0.0 < r["v2_V"] < 1.0 and 0.0 < r["v2_omega"] < 1.0, r
        assert r["gauss_max"] < 1e-4, r


# ---------------------------------------------------------------------------------------------------------
# z-slab decomposition (ahs_group): every slab on THIS GPU -- the same kernels, peer stores and event
# ordering as across GPUs, launched one after another (nothing waits on the device)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec,N,slabs", [("f32", 256, (1, 2, 4, 8)), ("f64", 128, (2, 4)), ("f32", 128, (2, 32))])
def test_slab_group_reproduces_the_single_lattice_bit_for_bit(ahs, prec, N, slabs):
    """A lattice cut into P z-slabs with ghost planes kept current by the step kernel's stores into the neighbours' memory must
    evolve exactly like the whole lattice on one handle: fields bit for bit (every site's arithmetic is the same), winding counts
    exactly, fp64 sums to the order of the final reduction, Gauss's law at roundoff across the slab faces."""
    nsteps = 12
    with ahs.Simulation(N=N, precision=prec, m=1.0, s=0.0, seed=77) as ref:
        ic = ref.get_fields_native()
        ref.step(nsteps)
        want, dref = ref.get_fields_native(), ref.diagnostics()
    for P in slabs:
        with ahs.Group(N=N, nslabs=P, precision=prec, m=1.0, s=0.0, seed=77) as g:
            assert np.array_equal(g.get_fields_native(), ic), P                       # the same Philox initial condition, slab by slab
            g.step(5)
            d5 = g.diagnostics()
            g.step(nsteps - 5)
            got, d = g.get_fields_native(), g.diagnostics()
            assert np.array_equal(got, want), (P, [int((got[k] != want[k]).sum()) for k in range(10)])
            assert d["step"] == nsteps and d5["step"] == 5
            assert (d["n_pierced"], d["sum_abs_w"], d["nonfinite"]) == (dref["n_pierced"], dref["sum_abs_w"], 0), P
            for key in ("v2_num", "v2_den", "v2v_num", "v2v_den", "eos_num", "eos_den", "mean_lagrangian", "gauss_rhs_rms"):
                assert d[key] == pytest.approx(dref[key], rel=1e-11, abs=1e-11 * abs(dref["v2_den"])), (P, key)
            assert d["gauss_max"] == dref["gauss_max"], P


def test_slab_group_from_uploaded_fields_and_options(ahs, oracle):
    """ahs_group_set_fields_native fills the ghost planes from the neighbours; then 20 steps against the ORACLE (all ten fields
    non-zero from the start), with a chunk count that does not divide the slab and row-copy staging on one of the runs."""
    from paper_1809_00995_b200 import synthetic
    N, nsteps = 128, 20
    f0 = synthetic.random_snapshot(N, seed=31).astype(np.float32)
    p = oracle.Params(N=N, m=2.0, s=0.0, tau0=2.0)
    ref = oracle.step(p, f0.astype(np.float64), 3, nsteps)
    for P, opts in ((4, {}), (2, {ahs.AHS_OPT_STEP_CHUNKS: 7, ahs.AHS_OPT_DIAG_CHUNKS: 3}), (8, {ahs.AHS_OPT_STAGING: ahs.AHS_STAGING_ROWS})):
        with ahs.Group(N=N, nslabs=P, precision="f32", m=2.0, s=0.0, tau0=2.0, ic="none") as g:
            for k, v in opts.items():
                g.set_option(k, v)
            g.set_fields_native(f0, step=3)
            assert np.array_equal(g.get_fields_native(), f0)
            g.step(nsteps)
            got = g.get_fields_native().astype(np.float64)
            assert_fields("slab_group_vs_oracle", got, ref, "f32", oracle.FIELD_NAMES, N=N, slabs=P, nsteps=nsteps)
            d = g.diagnostics()
            r = oracle.diagnostics(p, got, 3 + nsteps)                                   # the oracle on the group's own snapshot
            assert (d["n_pierced"], d["sum_abs_w"]) == (r["n_pierced"], r["sum_abs_w"])
            K, G, Lg = oracle.site_fields(p, got, 3 + nsteps)
            assert abs(d["v2_num"] - r["v2_num"]) <= 2e-5 * np.abs(K * Lg).sum()
            assert abs(d["gauss_max"] - r["gauss_max"]) <= 64 * 6e-8 * max(1.0, r["gauss_rhs_rms"], np.abs(got[7:10]).max())
    with pytest.raises(ahs.AhsError):
        ahs.Group(N=N, nslabs=3)                                                          # must divide N
    with pytest.raises(ahs.AhsError):
        ahs.Group(N=N, nslabs=2, devices=[0, 99])


def test_slab_handles_are_driven_through_their_group(ahs):
    """A slab's handle (ahs_group_slab) takes options and reports state, but stepping it, measuring it or touching its fields on its
    own would leave the group's buffers and ghost planes out of step: those calls return AHS_ERR_STATE and change nothing.  Chunk
    counts are bounded by the planes the slab owns, not by N."""
    import ctypes as C
    N, P = 128, 2
    lib = ahs.load()
    with ahs.Simulation(N=N, precision="f32", seed=5) as ref, ahs.Group(N=N, nslabs=P, precision="f32", seed=5) as g:
        h = C.c_void_p(lib.ahs_group_slab(g._g, 1))
        d = ahs.ahs_diag()
        buf = np.zeros((10, N, N, N), dtype=np.float32)
        assert lib.ahs_step(h, 1) == ahs.AHS_ERR_STATE and "ahs_group" in ahs.last_error()
        assert lib.ahs_diagnostics_launch(h) == ahs.AHS_ERR_STATE
        assert lib.ahs_diagnostics_ex(h, C.byref(d)) == ahs.AHS_ERR_STATE
        assert lib.ahs_diagnostics_fetch(h, C.byref(d)) == ahs.AHS_ERR_STATE
        assert lib.ahs_get_fields_native(h, buf.ctypes.data) == ahs.AHS_ERR_STATE
        assert lib.ahs_set_fields_native(h, buf.ctypes.data, 0) == ahs.AHS_ERR_STATE
        assert lib.ahs_set_option(h, ahs.AHS_OPT_STEP_CHUNKS, N // P + 1) == ahs.AHS_ERR_INVALID_ARG     # 64 planes per slab
        assert lib.ahs_set_option(h, ahs.AHS_OPT_DIAG_CHUNKS, N // P + 1) == ahs.AHS_ERR_INVALID_ARG
        assert lib.ahs_set_option(h, ahs.AHS_OPT_STEP_CHUNKS, N // P) == ahs.AHS_OK
        st = C.c_int64(-1)
        assert lib.ahs_get_state(h, C.byref(st), None, None) == ahs.AHS_OK and st.value == 0             # none of the refused calls stepped it
        ref.step(6)
        g.step(3)
        g.diagnostics()
        g.step(3)
        assert np.array_equal(g.get_fields_native(), ref.get_fields_native())
    with pytest.raises(ahs.AhsError) as e:
        ahs.Group(N=2048, nslabs=1)                                # refused before any memory is asked for
    assert "at least 2 slabs" in str(e.value)


@pytest.mark.parametrize("prec,N,P", [("f32", 256, 4), ("f64", 128, 2)])
def test_slab_group_exchange_by_copies_is_bit_identical(ahs, prec, N, P):
    """AHS_EXCHANGE_COPIES -- what two GPUs without peer access to one another get: the faces travel by cudaMemcpyPeerAsync behind the
    step instead of the kernel's own stores.  Same bar: the single lattice bit for bit, also when the mode changes in mid-run."""
    with ahs.Simulation(N=N, precision=prec, m=1.0, s=0.0, seed=21) as ref, ahs.Group(N=N, nslabs=P, precision=prec, m=1.0, s=0.0, seed=21) as g:
        assert g.copied_faces == 0                                   # one GPU: every face by the kernel's stores
        g.set_exchange(ahs.AHS_EXCHANGE_COPIES)
        assert g.copied_faces == 2 * P
        ref.step(7)
        g.step(4)
        d4 = g.diagnostics()
        g.step(3)
        assert d4["step"] == 4 and np.array_equal(g.get_fields_native(), ref.get_fields_native())
        g.set_exchange(ahs.AHS_EXCHANGE_STORES)
        assert g.copied_faces == 0
        ref.step(5)
        g.step(5)
        assert np.array_equal(g.get_fields_native(), ref.get_fields_native())
        d, dref = g.diagnostics(), ref.diagnostics()
        assert (d["n_pierced"], d["sum_abs_w"], d["gauss_max"]) == (dref["n_pierced"], dref["sum_abs_w"], dref["gauss_max"])
        with pytest.raises(ahs.AhsError):
            g.set_exchange(2)


def _device_count():
    import torch
    return torch.cuda.device_count()


def test_slab_group_on_several_devices_bit_for_bit(ahs):
    """The path a one-GPU box never reaches: slabs on different GPUs (peer access between neighbours, the step kernel's stores into
    the neighbours' ghost planes over NVLink, events waited for across devices, the per-device shared-memory attribute).  Same bar
    as on one GPU: the single lattice bit for bit."""
    ndev = _device_count()
    if ndev < 2:
        pytest.skip("needs at least 2 CUDA devices, this box has %d: the multi-device slab path stays unmeasured here" % ndev)
    N, nsteps = 256, 12
    with ahs.Simulation(N=N, precision="f32", m=1.0, s=0.0, seed=77) as ref:
        ref.step(nsteps)
        want, dref = ref.get_fields_native(), ref.diagnostics()
    for P, devices in ((2, [0, 1]), (4, [d % ndev for d in range(4)]), (ndev, list(range(ndev)))):
        if N % P:
            continue
        with ahs.Group(N=N, nslabs=P, devices=devices, precision="f32", m=1.0, s=0.0, seed=77) as g:
            if P == 4:
                g.set_exchange(ahs.AHS_EXCHANGE_COPIES)             # the path of GPUs without peer access, across real devices
            g.step(5)
            d5 = g.diagnostics()
            g.step(nsteps - 5)
            got, d = g.get_fields_native(), g.diagnostics()
            assert np.array_equal(got, want), (devices, [int((got[k] != want[k]).sum()) for k in range(10)])
            assert d5["step"] == 5 and (d["n_pierced"], d["sum_abs_w"], d["nonfinite"]) == (dref["n_pierced"], dref["sum_abs_w"], 0), devices
            assert d["v2_num"] == pytest.approx(dref["v2_num"], rel=1e-11) and d["gauss_max"] == dref["gauss_max"], devices


def test_handles_on_two_devices_driven_from_one_thread(ahs):
    """include/ahs.h: a handle belongs to the device that was current when it was created, and every later call switches to that
    device for its own duration -- one host thread drives handles on several GPUs without calling cudaSetDevice itself."""
    import torch
    if _device_count() < 2:
        pytest.skip("needs at least 2 CUDA devices, this box has %d" % _device_count())
    kw = dict(N=128, precision="f32", m=1.0, s=0.0, seed=11)
    home = torch.cuda.current_device()
    with torch.cuda.device(1):
        far = ahs.Simulation(**kw)
    near = ahs.Simulation(**kw)
    try:
        for _ in range(3):                                          # interleaved, never switching devices here
            near.step(2)
            far.step(2)
        dn, df = near.diagnostics(), far.diagnostics()
        assert torch.cuda.current_device() == home
        assert np.array_equal(near.get_fields_native(), far.get_fields_native())
        assert dn == df
    finally:
        far.destroy()
        near.destroy()


@pytest.mark.parametrize("prec,N,kernel", [("f64", 64, "auto"), ("f32", 128, "auto"), ("f64", 20, "generic")])
def test_s_schedule_matches_oracle(ahs, oracle, prec, N, kernel):
    """ahs_set_s_schedule: core growth (s = -1), a linear ramp, then the true equations (s = 1), 30 steps
    across all three against the oracle; coefficients on the ramp to 1e-14; Gauss's law at roundoff on the device trajectory (it
    only holds if every coupling takes s at its own time level); diagnostics on the oracle's snapshot."""
    sched = ((1.0, -1.0), (2.0, -1.0), (3.0, 1.0))
    with ahs.Simulation(N=N, precision=prec, m=1.0, s=0.25, ic="none", kernel=kernel) as sim:
        sim.set_s_schedule(sched)
        p = oracle.Params(N=N, m=1.0, s=0.25, s_schedule=sched)
        for n in (3, 14, 17, 25):
            np.testing.assert_allclose(sim.coefficients(n), oracle.coeffs(p, n), rtol=1e-14)
        ref = rounded(oracle.initial_condition(p, 9), prec)
        sim.set_fields(ref, 0)
        sim.step(30)
        got = sim.get_fields()
        oracle.step(p, ref, 0, 30)
        assert_fields("s_schedule", got, ref, prec, oracle.FIELD_NAMES, tol=1e-12 if prec == "f64" else 2e-4, N=N, kernel=sim.kernel_kind, nsteps=30)
        d = sim.diagnostics()
        assert d["gauss_max"] <= (1e-12 if prec == "f64" else 2e-5) * max(1.0, d["gauss_rhs_rms"])
        check_diag(oracle, p, sim, prec, ref, 30)
        sim.set_s_schedule(())                                                       # back to the constant s
        np.testing.assert_allclose(sim.coefficients(14), oracle.coeffs(oracle.Params(N=N, m=1.0, s=0.25), 14), rtol=1e-14)
        with pytest.raises(ahs.AhsError):
            sim.set_s_schedule(((2.0, 0.0), (1.0, 1.0)))
