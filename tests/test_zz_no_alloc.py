"""ahs_diagnostics_static: the diagnostics entry point for callers that cannot allocate.

Some users of libahs hold their ten field arrays on the GPU themselves and call in from a place where device memory may not be
asked for: a production run that has filled HBM (a cudaMalloc hours into the run can fail), an analysis hook inside another
framework's step loop (the framework's caching allocator owns the free memory, and cudaMalloc / cudaFree stall every stream of the
device), a latency-critical loop.  For them the library has one call that allocates nothing: the reduction's scratch records sit in a
fixed 444.25 KiB array inside libahs.so (one per GPU, shared by all calls, keeping the last call's contents).

What is checked here, through the C ABI, against the EXISTING path (a handle's ahs_diagnostics_ex) on the same device arrays:
  * two calls in a row (the second starts from the scratch the first left behind) each agree with the handle's result -- counts
    exactly, sums within the bars test_gpu_parity.check_diag uses (1e-10 on fp64 lattices, 2e-5 on fp32 ones, of the sum of the
    absolute values of the terms, which the oracle supplies: the Lagrangian-weighted sums cancel heavily); against a handle on the
    same one-thread-per-site kernel the record is equal bit for bit, as include/ahs.h promises;
  * a small lattice right after a large one reads none of the large one's leftover records;
  * the free device memory does not move across a call once the first call on the device has been made;
  * sizes beyond the stated maximum and pointers that are not device memory are refused with a message, before anything is launched.

This file sorts after every other test file on purpose: `pytest -x` stops at the first failure, and a failure in this add-on must not
hide the parity tests.  It passes alone in a fresh process (it then makes the device's first call itself) and after the others.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

BAR = {"f64": 1e-10, "f32": 2e-5}          # the bars of check_diag (tests/test_gpu_parity.py)
EPS = {"f64": 2.3e-16, "f32": 6e-8}
SUMS = ("v2_num", "v2_den", "mean_lagrangian", "v2v_num", "v2v_den", "eos_num", "eos_den")


@pytest.fixture(scope="module")
def ahs():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1809_00995_b200 import binding
    binding.load()
    return binding


def static_diagnostics(ahs, sim, prec):
    """The new entry point on the live device arrays of `sim` (no copy), on the handle's stream so that it runs behind its steps."""
    ptrs = [sim.field_device_ptr(k) for k in range(10)]
    q = {k: v for k, v in sim.params.items() if k not in ("seed", "N")}
    return ahs.diagnostics_static(ptrs, sim.N, sim.step_count, precision=prec, stream=sim.stream_handle, **q)


def scales(O, sim, snap, n):
    """What check_diag measures the sums' errors against: the sums of the absolute values of their terms, from the oracle's per-site
    fields of the same snapshot (the scales only -- the values compared are the two CUDA paths')."""
    q = dict(sim.params)
    q.pop("seed")
    K, G, Lg, Vp, El, Bm = O.site_fields6(O.Params(**q), snap.astype(np.float64), n)
    rho, prs = K + G + Vp + El + Bm, K - G / 3 - Vp + (El + Bm) / 3
    return dict(v2_num=np.abs(K * Lg).sum(), v2_den=np.abs(G * Lg).sum(), mean_lagrangian=np.abs(Lg).mean(), v2v_num=(K * Vp).sum(),
                v2v_den=(G * Vp).sum(), eos_num=np.abs(prs * Lg).sum(), eos_den=np.abs(rho * Lg).sum(), eps=np.abs(snap[7:10]).max())


def assert_agree(got, ref, prec, scale):
    bar = BAR[prec]
    assert got["step"] == ref["step"] and got["tau"] == ref["tau"]
    assert got["n_pierced"] == ref["n_pierced"] and got["sum_abs_w"] == ref["sum_abs_w"]          # integers: exactly
    assert got["L"] == ref["L"] and got["xi"] == ref["xi"]
    for k in SUMS:
        assert abs(got[k] - ref[k]) <= bar * scale[k] + 1e-300, (k, got[k], ref[k], scale[k])
    for k in ("v2", "v2_V"):
        assert got[k] == pytest.approx(ref[k], rel=200 * bar, abs=200 * bar), k
    if abs(ref["eos_den"]) > 0.05 * scale["eos_den"]:                                           # else a ratio of cancelled sums
        assert got["v2_omega"] == pytest.approx(ref["v2_omega"], rel=200 * bar, abs=200 * bar)
    assert abs(got["gauss_max"] - ref["gauss_max"]) <= 64 * EPS[prec] * max(1.0, ref["gauss_rhs_rms"], scale["eps"])
    assert got["gauss_rhs_rms"] == pytest.approx(ref["gauss_rhs_rms"], rel=1e-5, abs=1e-30)
    assert got["nonfinite"] == ref["nonfinite"] == 0


@pytest.mark.parametrize("prec,N", [("f32", 128), ("f64", 64)])
def test_two_calls_in_a_row_agree_with_the_handle_path(ahs, oracle, prec, N):
    oracle.set_threads(0)
    kw = dict(N=N, precision=prec, seed=1809, m=1.0, s=0.0)
    with ahs.Simulation(kernel="auto", **kw) as sim, ahs.Simulation(kernel="generic", ic="none", **kw) as gen:
        assert sim.kernel_kind == "march" and gen.kernel_kind == "generic"
        sim.step(10)
        first = static_diagnostics(ahs, sim, prec)            # call 1 (the device's very first when this file runs alone)
        sim.step(10)
        second = static_diagnostics(ahs, sim, prec)           # call 2: the array still holds call 1's records
        again = static_diagnostics(ahs, sim, prec)            # and once more on the same snapshot
        assert again == second                                # bit for bit: nothing of an earlier call leaks into a later one
        snap20 = sim.get_fields_native()
        ref_march = sim.diagnostics()                         # existing path, z-marching kernel
        assert ref_march["n_pierced"] > 0                     # a network is there: the comparison is not 0 == 0
        assert_agree(second, ref_march, prec, scales(oracle, sim, snap20, 20))
        gen.set_fields_native(snap20, step=20)
        ref_generic = gen.diagnostics()                       # existing path, the same one-thread-per-site kernel
        assert static_diagnostics(ahs, gen, prec) == ref_generic == second
        # call 1 against the existing path on ITS snapshot: replay the first ten steps
        with ahs.Simulation(kernel="auto", **kw) as replay:
            replay.step(10)
            snap10 = replay.get_fields_native()
            assert_agree(first, replay.diagnostics(), prec, scales(oracle, replay, snap10, 10))
            gen.set_fields_native(snap10, step=10)
            assert gen.diagnostics() == first


def test_small_lattice_after_a_large_one_reads_only_its_own_records(ahs):
    with ahs.Simulation(N=128, precision="f32", seed=7, kernel="generic") as big, ahs.Simulation(N=16, precision="f32", seed=8, kernel="generic") as small:
        big.step(5)
        small.step(5)
        d_big = static_diagnostics(ahs, big, "f32")           # 4736 block records written
        d_small = static_diagnostics(ahs, small, "f32")       # 32 blocks: records 32..4735 are the large lattice's leftovers
        assert d_small == small.diagnostics() and d_big == big.diagnostics()
        assert d_small["n_pierced"] != d_big["n_pierced"]


def test_a_call_allocates_no_device_memory(ahs):
    import torch
    with ahs.Simulation(N=64, precision="f32", seed=3, kernel="generic") as sim:
        sim.step(3)
        static_diagnostics(ahs, sim, "f32")                   # set-up call: code and array are on the GPU after this
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        for _ in range(3):
            static_diagnostics(ahs, sim, "f32")
        assert torch.cuda.mem_get_info()[0] == free_before


def test_sizes_beyond_the_maximum_and_foreign_pointers_are_refused(ahs):
    import torch
    assert ahs.AHS_STATIC_SCRATCH_BYTES == 96 * (ahs.AHS_STATIC_MAX_RECORDS + 1) + 160 == 454912
    x = torch.zeros(16 ** 3, dtype=torch.float32, device="cuda")
    ten = [x] * 10
    ahs.diagnostics_static(ten, 16, 0)                         # ten readable arrays of the right size: accepted
    for bad_N in (ahs.AHS_STATIC_MAX_N + 1, 2 * ahs.AHS_STATIC_MAX_N, 3):
        with pytest.raises(ahs.AhsError) as e:
            ahs.diagnostics_static(ten, bad_N, 0)              # refused on N alone: the arrays are never touched
        assert e.value.code == ahs.AHS_ERR_INVALID_ARG and str(ahs.AHS_STATIC_MAX_N) in str(e.value)
    host = np.zeros(16 ** 3, dtype=np.float32)
    for bad in (ten[:9] + [0], ten[:4] + [host.ctypes.data] + ten[5:]):
        with pytest.raises(ahs.AhsError) as e:
            ahs.diagnostics_static(bad, 16, 0)
        assert e.value.code == ahs.AHS_ERR_INVALID_ARG and "fields10" in str(e.value)
    with pytest.raises(ahs.AhsError):
        ahs.diagnostics_static(ten, 16, -1)
