"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerances (BASELINE.json north_star): relative L2 error on psi and on the
detector image <= 1e-11 for fp64 contexts and <= 1e-4 for fp32 contexts.  For fp32 the truth is the
oracle run in double on the same float-rounded inputs (V, mask, psi0, coefficients).
"""
import os

import numpy as np
import pytest

import oracle
from oracle import OracleRun
from workloads import make_config, random_state, random_potential, PERIODIC, DIRICHLET

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-11, "f32": 1e-4}
TWOPASS, FUSED = 1, 2


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / nb) if nb > 0 else float(np.linalg.norm(a))


def make_ctx(nx, ny, nz, batch, dx, dt, dtype, **kw):
    from paper_2401_07416_b200 import Tdse
    return Tdse(nx, ny, nz, batch, dx, dt, 1.0, 1.0, dtype, **kw)


def oracle_for(w, entry, steps):
    return OracleRun.from_workload(w, entry=entry, dtype="f64",
                                   round_to="f32" if w.dtype == "f32" else None).step(steps)


# ------------------------------------------------------------------------------------------
# S0 / S1: potential builder and packet init
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("idx,shape", [(0, (24, 20, 28)), (1, (40, 36, 48)), (3, (36, 40, 44)), (4, (48, 40, 56))])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_potential_and_packet_match_oracle(idx, shape, dtype):
    from paper_2401_07416_b200 import Tdse
    w = make_config(idx, n=shape, batch=2 if idx == 3 else 1, dtype=dtype)
    t = Tdse.from_workload(w)
    for b in range(w.batch):
        o = OracleRun.from_workload(w, entry=b, dtype="f64", round_to="f32" if dtype == "f32" else None)
        V = t.read_potential(b)
        R, I = t.read_psi(b)
        if dtype == "f64":
            assert np.max(np.abs(V - o.V64)) <= 1e-13 * max(1.0, np.max(np.abs(o.V64)))
            assert rel_l2(R, o.R) < 1e-14 and rel_l2(I, o.I) < 1e-14
        else:
            # one rounding of a double result that may differ in its last bits: at most 1 ulp
            ulp = np.spacing(np.abs(o.V).astype(np.float32)).astype(np.float64)
            assert np.all(np.abs(V.astype(np.float64) - o.V) <= ulp)
            assert rel_l2(R, o.R) < 1e-7 and rel_l2(I, o.I) < 1e-7
        assert V.min() >= w.vmin and V.max() <= w.vmax
    t.close()


# ------------------------------------------------------------------------------------------
# S2-S5: the recurrence on raw seeded states, every boundary combination, awkward sizes
# ------------------------------------------------------------------------------------------
BCS = [(PERIODIC, PERIODIC, DIRICHLET), (DIRICHLET, DIRICHLET, DIRICHLET), (PERIODIC, PERIODIC, PERIODIC),
       (DIRICHLET, PERIODIC, PERIODIC), (PERIODIC, DIRICHLET, DIRICHLET)]
SHAPES = [(72, 40, 37), (64, 64, 16), (8, 6, 5), (136, 70, 21), (4, 3, 2)]
VARIANTS = [(TWOPASS, 1), (FUSED, 1), (FUSED, 2)]


def fused_eligible(nx, ny, dtype):
    """include/tdse.h, tdse_set_option("kernel"): 16-byte rows, even ny, domain at least as wide as two frames."""
    return nx % (4 if dtype == "f32" else 2) == 0 and ny % 2 == 0 and nx >= 8 and ny >= 8


@pytest.mark.parametrize("kernel,tblock", VARIANTS)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape,bc", list(zip(SHAPES, BCS)) + [((40, 24, 30), BCS[2]), ((40, 24, 30), BCS[1]),
                                                               ((8, 8, 5), BCS[2]), ((8, 8, 3), BCS[4])])
def test_recurrence_matches_oracle_on_random_states(kernel, tblock, dtype, shape, bc):
    nx, ny, nz = shape
    if kernel == FUSED and not fused_eligible(nx, ny, dtype):
        # forcing the fused kernel on a shape it does not take must fail loudly, not fall back
        t = make_ctx(nx, ny, nz, 1, 0.25, 0.004, dtype)
        t.set_option("kernel", FUSED)
        t.set_potential_grid(0, np.zeros((nz, ny, nx), dtype=t.np_dtype))
        t.set_state(0, np.ones((nz, ny, nx), dtype=t.np_dtype), np.ones((nz, ny, nx), dtype=t.np_dtype))
        from paper_2401_07416_b200 import TdseError, TDSE_EINVAL
        with pytest.raises(TdseError) as ei:
            t.step(1)
        assert ei.value.code == TDSE_EINVAL
        t.close()
        return
    dx, dt, steps, batch = 0.25, 0.004, 23, 2
    absorb = min(4, nz // 3)
    t = make_ctx(nx, ny, nz, batch, dx, dt, dtype)
    t.set_boundary(*bc, absorb, absorb, 0.07, 2)
    t.set_option("kernel", kernel)
    t.set_option("tblock", tblock)
    k_det = min(3, nz - 1)
    t.set_detector(k_det, 5, 8)
    ora = []
    for b in range(batch):
        V = random_potential(100 + b, (nz, ny, nx), -30.0, 5.0)
        R0, I0 = random_state(200 + b, (nz, ny, nx))
        t.set_potential_grid(b, V.astype(t.np_dtype))
        t.set_state(b, R0.astype(t.np_dtype), I0.astype(t.np_dtype))
        o = OracleRun(nx, ny, nz, dx, dt, bc=bc, absorb_lo=absorb, absorb_hi=absorb, strength=0.07,
                      round_to="f32" if dtype == "f32" else None)
        o.set_potential_grid(V).set_state(R0, I0).set_detector(k_det, 5)
        ora.append(o.step(steps))
    t.step(steps)
    assert t.get_info("kernel") == kernel and t.get_info("steps") == steps
    for b in range(batch):
        R, I = t.read_psi(b)
        D, tr = t.detector_read(b)
        tol = TOL[dtype]
        assert rel_l2(R, ora[b].R) < tol and rel_l2(I, ora[b].I) < tol
        assert len(tr) == 4 and rel_l2(D, ora[b].D) < tol and rel_l2(tr, ora[b].trace) < tol
    t.close()


@pytest.mark.parametrize("seed", [101, 102, 103])
def test_randomised_configurations_every_kernel_variant(seed):
    """Seeded random draws of everything at once -- shape (fused-eligible or not), batch, boundary flags, absorber
    widths, anisotropic spacing, step count split over two calls, sampling period, detector plane, and for the fused
    kernel the z chunking, prefetch depth and dependent-launch overlap -- each run through the two-pass kernel and
    the fused kernel with T = 1 and T = 2 and compared with the oracle."""
    from paper_2401_07416_b200 import Tdse
    rng = np.random.default_rng(seed)
    for case in range(8):
        dtype = "f64" if rng.random() < 0.5 else "f32"
        vw = 2 if dtype == "f64" else 4
        nx = int(rng.integers(2, 40)) * vw if rng.random() < 0.8 else int(rng.integers(3, 90))
        ny = int(rng.integers(4, 60)) * 2 if rng.random() < 0.8 else int(rng.integers(3, 90))
        nz = int(rng.integers(2, 70))
        batch = int(rng.integers(1, 4))
        bc = tuple(int(x) for x in rng.integers(0, 2, 3))
        alo, ahi = int(rng.integers(0, max(1, nz // 3))), int(rng.integers(0, max(1, nz // 3)))
        steps, every, k_det = int(rng.integers(1, 14)), int(rng.integers(1, 6)), int(rng.integers(0, nz))
        dx = 0.2
        dy, dz = dx * (1.0 + 0.3 * rng.random()), dx * (1.0 - 0.3 * rng.random())
        dt = 0.4 / (2.0 * (1 / dx ** 2 + 1 / dy ** 2 + 1 / dz ** 2) + 50.0)
        V = [random_potential(seed * 1000 + case * 10 + b, (nz, ny, nx), -50.0, 0.0) for b in range(batch)]
        S = [random_state(seed * 2000 + case * 10 + b, (nz, ny, nx)) for b in range(batch)]
        oracles = []
        for b in range(batch):
            o = OracleRun(nx, ny, nz, dx, dt, bc=bc, absorb_lo=alo, absorb_hi=ahi, strength=0.06, power=2,
                          round_to="f32" if dtype == "f32" else None, dy=dy, dz=dz)
            o.set_potential_grid(V[b]).set_state(*S[b]).set_detector(k_det, every)
            oracles.append(o.step(steps))
        variants = [(TWOPASS, 1, 1)]
        if fused_eligible(nx, ny, dtype):
            variants += [(FUSED, 1, 1), (FUSED, 2, 1), (FUSED, 2, 0)]
        for kernel, T, pdl in variants:
            t = Tdse(nx, ny, nz, batch, dx, dt, 1.0, 1.0, dtype)
            t.set_spacing(dy, dz)
            t.set_boundary(bc[0], bc[1], bc[2], alo, ahi, 0.06, 2)
            for b in range(batch):
                t.set_potential_grid(b, V[b].astype(t.np_dtype))
                t.set_state(b, S[b][0].astype(t.np_dtype), S[b][1].astype(t.np_dtype))
            t.set_detector(k_det, every, 32)
            t.set_option("kernel", kernel); t.set_option("tblock", T); t.set_option("pdl", pdl)
            if kernel == FUSED and rng.random() < 0.5:
                t.set_option("z_chunks", int(rng.integers(1, 6)))
            if kernel == FUSED and rng.random() < 0.5:
                t.set_option("prefetch", int(rng.integers(1, 3)))
            first = int(rng.integers(0, steps + 1))
            t.step(first); t.step(steps - first)
            what = (seed, case, dtype, (nx, ny, nz), batch, bc, (alo, ahi), steps, every, k_det, kernel, T, pdl)
            for b in range(batch):
                R, I = t.read_psi(b)
                D, tr = t.detector_read(b)
                o = oracles[b]
                assert len(tr) == len(o.trace) == steps // every, what
                assert rel_l2(R, o.R) < TOL[dtype] and rel_l2(I, o.I) < TOL[dtype], what
                if len(tr):
                    assert rel_l2(D, o.D) < TOL[dtype] and rel_l2(tr, o.trace) < TOL[dtype], what
            t.close()


@pytest.mark.parametrize("kernel,tblock", VARIANTS)
def test_step_counts_split_across_calls_and_odd_sampling_period(kernel, tblock):
    """n steps in one call == the same steps in uneven pieces; `every` odd forces T=1 launches in between."""
    w = make_config(1, n=(40, 32, 48), steps=0)
    from paper_2401_07416_b200 import Tdse
    a, b = Tdse.from_workload(w), Tdse.from_workload(w)
    for t in (a, b):
        t.set_option("kernel", kernel); t.set_option("tblock", tblock)
        t.set_detector(7, 3, 32)
    a.step(31)
    for n in (1, 2, 5, 0, 7, 16):
        b.step(n)
    Ra, Ia = a.read_psi(0); Rb, Ib = b.read_psi(0)
    Da, ta = a.detector_read(0); Db, tb = b.detector_read(0)
    assert len(ta) == len(tb) == 10
    assert np.array_equal(Da, Db) and np.array_equal(ta, tb)
    if kernel == TWOPASS or tblock == 1:
        assert np.array_equal(Ra, Rb) and np.array_equal(Ia, Ib)     # same arithmetic, same order
    else:
        assert rel_l2(Ra, Rb) < 1e-13 and rel_l2(Ia, Ib) < 1e-13     # T=2 vs T=1 launches regroup nothing either
    o = OracleRun.from_workload(w)
    o.set_detector(7, 3).step(31)
    assert rel_l2(Ra, o.R) < 1e-11 and rel_l2(Da, o.D) < 1e-11 and rel_l2(ta, o.trace) < 1e-11
    a.close(); b.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_dependent_launch_overlap_changes_nothing(dtype):
    """The fused kernel is launched with programmatic stream serialization (the next launch's CTAs become resident
    while the previous one drains).  Many back-to-back launches on a grid of a few CTAs, with detector samples, reads and a
    host-side mask change in between, must give bit-identical results with the overlap switched off, and match the oracle."""
    w = make_config(1, n=(40, 32, 24), steps=0).with_(dtype=dtype)
    from paper_2401_07416_b200 import Tdse
    res = []
    for pdl in (1, 0):
        t = Tdse.from_workload(w)
        t.set_option("kernel", FUSED); t.set_option("pdl", pdl)
        t.set_detector(5, 4, 64)
        t.step(121)                                   # 60 T=2 launches + T=1 tails around the samples
        mid = t.read_psi(0)
        t.step(2); t.step(1); t.step(36)
        res.append((mid, t.read_psi(0), t.detector_read(0)))
        t.close()
    for x, y in zip(res[0], res[1]):
        assert np.array_equal(x[0], y[0]) and np.array_equal(x[1], y[1])
    o = OracleRun.from_workload(w, dtype="f64", round_to="f32" if dtype == "f32" else None)
    o.set_detector(5, 4).step(160)
    tol = TOL[dtype]
    (R, I), (D, tr) = res[0][1], res[0][2]
    assert rel_l2(R, o.R) < tol and rel_l2(I, o.I) < tol and rel_l2(D, o.D) < tol and rel_l2(tr, o.trace) < tol


def test_identical_entries_give_bitwise_identical_results_at_any_batch_position():
    w = make_config(3, n=(64, 48, 40), batch=1, steps=0)
    from paper_2401_07416_b200 import Tdse
    w5 = w.with_(batch=5, atoms=[w.atoms[0]] * 5)
    t = Tdse.from_workload(w5)
    t.step(24)
    R0, I0 = t.read_psi(0)
    D0, tr0 = t.detector_read(0)
    for b in (1, 4):
        R, I = t.read_psi(b)
        D, tr = t.detector_read(b)
        assert np.array_equal(R, R0) and np.array_equal(I, I0) and np.array_equal(D, D0) and np.array_equal(tr, tr0)
    t.close()


def test_fused_and_twopass_agree_and_conserve_the_visscher_norm():
    w = make_config(0, n=(48, 40, 56), steps=0)
    from paper_2401_07416_b200 import Tdse
    out = {}
    for kernel in (TWOPASS, FUSED):
        t = Tdse.from_workload(w)
        t.set_option("kernel", kernel)
        q0 = t.norm(0)
        t.step(200)
        q1 = t.norm(0)
        assert abs(q1[0] - q0[0]) / q0[0] < 1e-12          # conserved exactly by the scheme (no mask in cfg 0)
        out[kernel] = t.read_psi(0)
        t.close()
    assert rel_l2(out[FUSED][0], out[TWOPASS][0]) < 1e-12
    o = OracleRun.from_workload(w)
    assert abs(o.norm()[0] - q0[0]) / q0[0] < 1e-13


# ------------------------------------------------------------------------------------------
# the BASELINE configurations (reduced grid / full steps where the oracle finishes in seconds)
# ------------------------------------------------------------------------------------------
# per-cell guard beside the rel-L2 bound (a single wrong seam cell of a 512^3 grid moves the rel-L2 by < 1e-4):
# max |error| over all cells, relative to max |psi| (for the image: to max D)
CELL_TOL = {"f64": 1e-10, "f32": 1e-3}


def max_abs_rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    scale = float(np.max(np.abs(b)))
    return float(np.max(np.abs(a - b))) / scale if scale > 0 else float(np.max(np.abs(a)))


def _run_config(w, steps, entries=None):
    from paper_2401_07416_b200 import Tdse
    t = Tdse.from_workload(w)
    t.step(steps)
    worst = 0.0
    for b in (entries if entries is not None else range(w.batch)):
        R, I = t.read_psi(b)
        D, tr = t.detector_read(b)
        o = oracle_for(w, b, steps)
        errs = (rel_l2(R, o.R), rel_l2(I, o.I), rel_l2(D, o.D), rel_l2(tr, o.trace))
        worst = max(worst, *errs)
        assert len(tr) == len(o.trace) == steps // w.every
        cell = max(max_abs_rel(R, o.R), max_abs_rel(I, o.I), max_abs_rel(D, o.D))
        assert cell < CELL_TOL[w.dtype], "entry %d: per-cell error %.3e" % (b, cell)
    info = (t.get_info("kernel"), t.get_info("tblock"))
    t.close()
    return worst, info


def test_config0_full_size_full_steps():
    w = make_config(0)
    worst, info = _run_config(w, w.steps)
    assert info == (FUSED, 1)       # 64^3: chunks of a few planes, the launcher's cost model takes one step per pass
    assert worst < 1e-11


def test_config1_full_size_full_steps():
    w = make_config(1)
    worst, info = _run_config(w, w.steps)
    assert info == (FUSED, 2)
    assert worst < 1e-11


def test_config2_reduced_grid():
    w = make_config(2, n=(64, 64, 128), steps=800)
    worst, _ = _run_config(w, w.steps)
    assert worst < 1e-4


def test_config3_reduced_batch_and_grid():
    w = make_config(3, n=(64, 64, 64), batch=6, steps=600)
    worst, _ = _run_config(w, w.steps, entries=(0, 3, 5))
    assert worst < 1e-4


def test_config4_reduced_grid_fp32_vs_fp64_detector_agreement():
    from paper_2401_07416_b200 import Tdse
    imgs = {}
    for dtype in ("f32", "f64"):
        w = make_config(4, n=(64, 64, 96), dtype=dtype, steps=400, batch=2)
        worst, _ = _run_config(w, w.steps)
        assert worst < TOL[dtype]
        t = Tdse.from_workload(w)
        t.step(w.steps)
        imgs[dtype] = t.detector_read(1)[0]
        t.close()
    assert rel_l2(imgs["f32"], imgs["f64"]) < 1e-4


# ------------------------------------------------------------------------------------------
# the stated step counts (BJ north star: "after the stated step counts"): the float recurrence is compared with the
# fp64 oracle on the same rounded inputs after ALL steps of the configuration, so the tolerance covers the error
# growth over 8000 / 4000 / 2000 steps and not only the first few hundred
# ------------------------------------------------------------------------------------------
def test_config2_reduced_grid_full_step_count():
    w = make_config(2, n=(64, 64, 128))
    assert w.steps == 8000 and w.dtype == "f32"
    worst, info = _run_config(w, w.steps)
    assert info == (FUSED, 2) and worst < 1e-4


def test_config3_full_grid_full_step_count_sampled_entries():
    """The bench workload itself: 64 x 128^3 f32, all 4000 steps, entries 0 and 63 against the oracle."""
    w = make_config(3)
    assert (w.batch, w.nx, w.ny, w.nz, w.dtype, w.steps) == (64, 128, 128, 128, "f32", 4000)
    worst, info = _run_config(w, w.steps, entries=(0, 63))
    assert info == (FUSED, 2) and worst < 1e-4


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config4_reduced_grid_full_step_count(dtype):
    w = make_config(4, n=(64, 64, 96), dtype=dtype, batch=1)
    assert w.steps == 2000
    worst, info = _run_config(w, w.steps)
    assert info == (FUSED, 2) and worst < TOL[dtype]


@pytest.mark.skipif(bool(os.environ.get("TDSE_SKIP_FULL_PARITY")), reason="TDSE_SKIP_FULL_PARITY set (minutes of oracle time)")
@pytest.mark.parametrize("idx,dtype", [(2, "f32"), (4, "f64"), (4, "f32")])
def test_full_size_full_step_count(idx, dtype):
    """cfg 2 (256 x 256 x 512 f32, 8000 steps) and cfg 4 (384^3 f64 and 512^3 f32, 2000 steps, entry 0) at
    BASELINE.json's full size and step count, every cell compared (rel-L2 and per-cell); prints the errors for the
    evidence file (profiles/r02_full_size_parity.md).  The oracle needs minutes of host time per case (OpenMP);
    TDSE_SKIP_FULL_PARITY=1 leaves these three out of a quick local run."""
    import time
    from paper_2401_07416_b200 import Tdse
    w = make_config(idx, dtype=dtype, batch=1) if idx == 4 else make_config(idx)
    t0 = time.time()
    t = Tdse.from_workload(w)
    t.step(w.steps)
    R, I = t.read_psi(0)
    D, tr = t.detector_read(0)
    info = (t.get_info("kernel"), t.get_info("tblock"))
    t.close()
    t1 = time.time()
    o = oracle_for(w, 0, w.steps)
    t2 = time.time()
    e_psi = max(rel_l2(R, o.R), rel_l2(I, o.I))
    e_det = max(rel_l2(D, o.D), rel_l2(tr, o.trace))
    e_cell = max(max_abs_rel(R, o.R), max_abs_rel(I, o.I), max_abs_rel(D, o.D))
    print("full-size parity cfg%d %s %dx%dx%d, %d steps: rel-L2 psi %.3e, detector image/trace %.3e, per-cell %.3e "
          "(kernel %s; GPU %.0f s, oracle %.0f s on %d threads)"
          % (idx, dtype, w.nx, w.ny, w.nz, w.steps, e_psi, e_det, e_cell, info, t1 - t0, t2 - t1, oracle.max_threads()))
    assert info == (FUSED, 2)
    assert e_psi < TOL[dtype] and e_det < TOL[dtype] and e_cell < CELL_TOL[dtype]


# ------------------------------------------------------------------------------------------
# BASELINE.json's full sizes, in the launch configuration bench.py times (tile, z chunks, batch): a few steps,
# compared element by element with the oracle on sampled entries
# ------------------------------------------------------------------------------------------
def test_config3_full_batch_full_grid_sampled_entries():
    """64 x 128^3 f32: the bench workload; entries 0, 31, 63 against the oracle after 24 steps (2 detector samples),
    and the launch shape is the one bench.py reports."""
    w = make_config(3, steps=24)
    assert (w.batch, w.nx, w.ny, w.nz, w.dtype) == (64, 128, 128, 128, "f32")
    worst, info = _run_config(w, w.steps, entries=(0, 31, 63))
    assert info == (FUSED, 2) and worst < 1e-4


def test_config2_full_grid_few_steps():
    w = make_config(2, steps=40)
    assert (w.nx, w.ny, w.nz, w.dtype) == (256, 256, 512, "f32")
    worst, info = _run_config(w, w.steps)
    assert info == (FUSED, 2) and worst < 1e-4


@pytest.mark.parametrize("dtype,n", [("f32", 512), ("f64", 384)])
def test_config4_full_grids_seeded_state(dtype, n):
    """512^3 f32 / 384^3 f64 with the cfg-4 boundary set-up, seeded potential and state (the atom-list build at this
    size is covered at reduced size: on the CPU it alone would take minutes), 6 steps, every cell compared."""
    nx = ny = nz = n
    dx = 0.15
    dt = 0.5 / (6.0 / dx ** 2 + 200.0)
    t = make_ctx(nx, ny, nz, 1, dx, dt, dtype)
    t.set_boundary(PERIODIC, PERIODIC, DIRICHLET, 16, 16, 0.05, 2)
    t.set_detector(10, 3, 4)
    V = random_potential(41, (nz, ny, nx), -200.0, 0.0)
    R0, I0 = random_state(42, (nz, ny, nx))
    t.set_potential_grid(0, V.astype(t.np_dtype))
    t.set_state(0, R0.astype(t.np_dtype), I0.astype(t.np_dtype))
    o = OracleRun(nx, ny, nz, dx, dt, bc=(PERIODIC, PERIODIC, DIRICHLET), absorb_lo=16, absorb_hi=16, strength=0.05,
                  round_to="f32" if dtype == "f32" else None)
    o.set_potential_grid(V).set_state(R0, I0).set_detector(10, 3)
    del V, R0, I0
    t.step(6)
    o.step(6)
    assert (t.get_info("kernel"), t.get_info("tblock")) == (FUSED, 1)      # 6 = 2 + 1 (sample) + 2 + 1 (sample)
    R, I = t.read_psi(0)
    tol = TOL[dtype]
    assert rel_l2(R, o.R) < tol and rel_l2(I, o.I) < tol
    # per-cell bound as well: no tile, chunk seam or frame image may be off while the norm hides it
    scale = float(np.max(np.abs(o.R)))
    assert np.max(np.abs(R.astype(np.float64) - o.R)) < (1e-9 if dtype == "f64" else 1e-3) * scale
    D, tr = t.detector_read(0)
    assert len(tr) == 2 and rel_l2(D, o.D) < tol and rel_l2(tr, o.trace) < tol
    t.close()


def test_flat_offsets_beyond_2_31_elements_per_array():
    """Maximum sizes: 18 entries of 512^3 f32 make every array 2.49e9 stored elements (9.3 GiB), so the last entries sit
    beyond element 2^31 and byte 2^33.  All entries get the same seeded state: entry 0 is compared with the oracle cell by
    cell, entries 16 and 17 (both beyond 2^31 elements) must be bit-identical to it, and so must their detector outputs."""
    import torch
    from workloads import random_state, random_potential
    n, batch = 512, 18
    assert 15 * (n + 8) * (n + 8) * n < 2 ** 31 < 16 * (n + 8) * (n + 8) * n
    dx = 0.15
    dt = 0.5 / (6.0 / dx ** 2 + 200.0)
    t = make_ctx(n, n, n, batch, dx, dt, "f32")
    t.set_boundary(PERIODIC, PERIODIC, DIRICHLET, 16, 16, 0.05, 2)
    t.set_detector(10, 3, 4)
    V = random_potential(43, (n, n, n), -200.0, 0.0)
    R0, I0 = random_state(44, (n, n, n))
    dev = [torch.from_numpy(a.astype(np.float32)).cuda() for a in (V, R0, I0)]
    t.set_potential_grid(-1, dev[0])
    t.set_state(-1, dev[1], dev[2])
    torch.cuda.synchronize()
    del dev
    o = OracleRun(n, n, n, dx, dt, bc=(PERIODIC, PERIODIC, DIRICHLET), absorb_lo=16, absorb_hi=16, strength=0.05,
                  round_to="f32")
    o.set_potential_grid(V).set_state(R0, I0).set_detector(10, 3)
    del V, R0, I0
    t.step(6)
    o.step(6)
    assert t.get_info("kernel") == FUSED
    R, I = t.read_psi(0)
    D, tr = t.detector_read(0)
    assert rel_l2(R, o.R) < 1e-4 and rel_l2(I, o.I) < 1e-4 and rel_l2(D, o.D) < 1e-4 and rel_l2(tr, o.trace) < 1e-4
    for b in (16, 17):
        Rb, Ib = t.read_psi(b)
        Db, trb = t.detector_read(b)
        assert np.array_equal(Rb, R) and np.array_equal(Ib, I) and np.array_equal(Db, D) and np.array_equal(trb, tr)
    t.close()


@pytest.mark.skipif(bool(os.environ.get("TDSE_SKIP_FULL_PARITY")), reason="TDSE_SKIP_FULL_PARITY set (minutes of oracle time)")
def test_detector_plane_in_the_rounding_noise_is_no_worse_than_the_float_oracle():
    """The geometry DESIGN.md reading 19 retired (round 1's literal cfg 4: packet at 0.3 Lz, slab top at 0.6 Lz, detector plane
    k = 10), kept as a noise-floor case on a 64 x 64 x 512 column that preserves the distances along z: the plane sits 5.4 sigma
    behind the packet and sees, within 2000 steps, only the Gaussian tail (1e-12 of the peak density) and the float rounding
    noise the packet radiates.  The 1e-4 image tolerance cannot be met there by ANY float code -- the oracle's own float
    instantiation misses its fp64 run by 5.7e-3 -- so the claim tested is: the GPU's image error is within 2x of that floor,
    while psi itself still meets 1e-4."""
    from paper_2401_07416_b200 import Tdse
    from workloads.configs import fcc111_slab
    w = make_config(4, n=(64, 64, 512), dtype="f32", batch=1)
    lx, ly, lz = w.nx * w.dx, w.ny * w.dx, w.nz * w.dx
    pk = dict(w.packet)
    pk["z0"] = 0.3 * lz
    w = w.with_(atoms=[fcc111_slab(lx, ly, 0.6 * lz, 4)], packet=pk, k_det=10)
    assert (pk["z0"] - w.k_det * w.dx) / pk["sigma"] > 5.0 and w.steps == 2000
    t = Tdse.from_workload(w)
    t.step(w.steps)
    R, I = t.read_psi(0)
    D, tr = t.detector_read(0)
    t.close()
    o64 = OracleRun.from_workload(w, dtype="f64", round_to="f32").step(w.steps)
    o32 = OracleRun.from_workload(w, dtype="f32").step(w.steps)
    e_gpu, e_orc = rel_l2(D, o64.D), rel_l2(o32.D, o64.D)
    print("noise-floor plane: image rel-L2 GPU f32 vs oracle f64 %.3e, oracle f32 vs oracle f64 %.3e; psi GPU %.3e, oracle f32 %.3e"
          % (e_gpu, e_orc, rel_l2(R, o64.R), rel_l2(o32.R, o64.R)))
    assert e_orc > 1e-4                                   # the float floor itself is above the tolerance here
    assert e_gpu <= 2.0 * e_orc
    assert rel_l2(R, o64.R) < 1e-4 and rel_l2(I, o64.I) < 1e-4


@pytest.mark.skipif(bool(os.environ.get("TDSE_SKIP_FULL_PARITY")), reason="TDSE_SKIP_FULL_PARITY set (minutes of oracle time)")
@pytest.mark.parametrize("dtype,batch", [("f64", 48), ("f32", 40)])
def test_config4_at_the_batch_that_fills_hbm_first_and_last_entry(dtype, batch):
    """BASELINE.json configs[4] is the batch "scaled to fill most of the 180 GB": 40 x 512^3 f32 / 48 x 384^3 f64 are
    111 / 113 GB of workspace, the launch shape (grid size, wave count, entry offsets far beyond 2^31 elements) of the
    fill-HBM runs BASELINE.md quotes.  SURVEY.md section 8(d): the oracle runs entries 0 and batch-1, the rest is covered
    by position invariance.  Entry 0 is the undisplaced slab, entry batch-1 a thermally displaced one (seed 4000 + b,
    workloads/configs.py); both are compared with the oracle in every cell after 20 steps (two detector samples), with
    the per-cell guard; entry 17 is a planted copy of entry batch-1 and must equal it bit for bit."""
    import torch
    from paper_2401_07416_b200 import Tdse
    w = make_config(4, dtype=dtype, batch=batch, steps=20)
    assert (w.nx, w.batch, w.every) == (512 if dtype == "f32" else 384, batch, 10)
    assert w.seeds[0] is None and w.seeds[batch - 1] == 4000 + batch - 1
    atoms = list(w.atoms)
    atoms[17] = atoms[batch - 1].copy()
    w = w.with_(atoms=atoms)
    t = Tdse.from_workload(w)
    assert t.workspace.numel() > 100e9
    t.step(w.steps)
    assert (t.get_info("kernel"), t.get_info("tblock")) == (FUSED, 2)
    out = {b: t.read_psi(b) + t.detector_read(b) for b in (0, 17, batch - 1)}
    t.close()
    del t
    torch.cuda.empty_cache()                      # hand the 110 GB back before the next test's context
    for x17, xl in zip(out[17], out[batch - 1]):
        assert np.array_equal(x17, xl)
    for b in (0, batch - 1):
        R, I, D, tr = out[b]
        o = oracle_for(w, b, w.steps)
        assert len(tr) == len(o.trace) == 2
        errs = (rel_l2(R, o.R), rel_l2(I, o.I), rel_l2(D, o.D), rel_l2(tr, o.trace))
        cell = max(max_abs_rel(R, o.R), max_abs_rel(I, o.I), max_abs_rel(D, o.D))
        print("fill-HBM parity cfg4 %s %d x %d^3, entry %d, %d steps: rel-L2 R %.3e I %.3e D %.3e trace %.3e, per-cell %.3e"
              % (dtype, batch, w.nx, b, w.steps, *errs, cell))
        assert max(errs) < TOL[dtype] and cell < CELL_TOL[dtype], "entry %d" % b
    assert not np.array_equal(out[0][0], out[batch - 1][0])        # the displaced entry really differs


# ------------------------------------------------------------------------------------------
# frame-mode detector and pairwise dissimilarity (eq 16)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("include_t0", [True, False])
def test_frames_and_dissimilarity_match_oracle(dtype, include_t0):
    from paper_2401_07416_b200 import Tdse, TdseError, TDSE_EINVAL, TDSE_ESTATE
    w = make_config(3, n=(40, 36, 44), batch=10, steps=46, dtype=dtype)    # 10 entries: a full 8x8 pair tile + ragged ones
    w = w.with_(every=5)
    t = Tdse.from_workload(w)
    with pytest.raises(TdseError) as e:                    # frame mode is off
        t.dissimilarity(0, 1)
    assert e.value.code == TDSE_ESTATE
    nfr = w.steps // w.every + (1 if include_t0 else 0)
    t.set_frames(nfr + 3, include_t0)
    t.step(17)
    t.step(w.steps - 17)                                   # split across calls, not aligned with the sampling period
    assert t.get_info("nframes") == nfr
    tol = TOL[dtype]
    ora, gpu = [], []
    for b in range(w.batch):
        o = OracleRun.from_workload(w, entry=b, dtype="f64", round_to="f32" if dtype == "f32" else None)
        o.set_frames(True, include_t0).step(w.steps)
        fr = t.frames_read(b)
        assert fr.shape == (nfr, w.ny, w.nx) and len(o.frames) == nfr
        for s in range(nfr):
            assert rel_l2(fr[s], o.frames[s]) < tol
        D, tr = t.detector_read(b)
        first = 1 if include_t0 else 0
        assert rel_l2(fr[first:].sum(axis=0), D) < 1e-14   # the accumulated image is the sum of the kept frames
        assert np.allclose(w.dx ** 2 * fr[first:].sum(axis=(1, 2)), tr, rtol=1e-12)
        ora.append(np.array(o.frames)); gpu.append(fr)
    s0, s1 = 2, nfr - 2
    d = t.dissimilarity(s0, s1)
    assert d.shape == (10, 10) and np.array_equal(d, d.T) and np.all(np.diag(d) == 0.0)
    for k in range(w.batch):
        for j in range(k + 1, w.batch):
            # the reduction alone (same frames in, different summation order): rounding level
            assert abs(d[k, j] - oracle.dissimilarity(gpu[k], gpu[j], w.dx ** 2, s0, s1)) <= 1e-12 * d[k, j]
            # end to end against the oracle's own trajectories
            want = oracle.dissimilarity(ora[k], ora[j], w.dx ** 2, s0, s1)
            assert abs(d[k, j] - want) <= 10 * tol * want
    with pytest.raises(TdseError) as e:
        t.dissimilarity(0, nfr)                            # window beyond the frames kept
    assert e.value.code == TDSE_EINVAL
    with pytest.raises(TdseError) as e:
        t.frames_read(0, nfr - 1, 2)
    assert e.value.code == TDSE_EINVAL
    t.close()


# ------------------------------------------------------------------------------------------
# the paper's own boundary set-up: periodic on all three axes with an absorbing layer at one z face only
# ("100 planes appended below the cell")
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel,tblock", VARIANTS)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_fully_periodic_with_one_face_absorber(kernel, tblock, dtype):
    nx, ny, nz = 40, 24, 36
    dx, dt, steps, batch = 0.25, 0.004, 31, 2
    t = make_ctx(nx, ny, nz, batch, dx, dt, dtype)
    t.set_boundary(PERIODIC, PERIODIC, PERIODIC, 0, 9, 0.07, 2)
    t.set_option("kernel", kernel)
    t.set_option("tblock", tblock)
    t.set_detector(nz - 2, 4, 8)                    # detector plane inside the layer, next to the periodic seam
    ora = []
    for b in range(batch):
        V = random_potential(300 + b, (nz, ny, nx), -30.0, 5.0)
        R0, I0 = random_state(400 + b, (nz, ny, nx))
        t.set_potential_grid(b, V.astype(t.np_dtype))
        t.set_state(b, R0.astype(t.np_dtype), I0.astype(t.np_dtype))
        o = OracleRun(nx, ny, nz, dx, dt, bc=(PERIODIC,) * 3, absorb_lo=0, absorb_hi=9, strength=0.07,
                      round_to="f32" if dtype == "f32" else None)
        o.set_potential_grid(V).set_state(R0, I0).set_detector(nz - 2, 4)
        ora.append(o.step(steps))
    assert np.all(ora[0].M[: nz - 9] == 1.0) and ora[0].M[-1] < 1.0      # one face only
    t.step(steps)
    tol = TOL[dtype]
    for b in range(batch):
        R, I = t.read_psi(b)
        D, tr = t.detector_read(b)
        assert rel_l2(R, ora[b].R) < tol and rel_l2(I, ora[b].I) < tol
        assert rel_l2(D, ora[b].D) < tol and rel_l2(tr, ora[b].trace) < tol
    t.close()


# ------------------------------------------------------------------------------------------
# anisotropic mesh (c_x != c_y != c_z)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel,tblock", VARIANTS)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_anisotropic_mesh_matches_oracle(kernel, tblock, dtype):
    # the paper's mesh ratios: 35.4/240 : 40.9/240 : 70/420 Angstrom, here in bohr-sized numbers
    w = make_config(1, n=(40, 36, 48), steps=37, dtype=dtype)
    w = w.with_(dy=w.dx * 40.9 / 35.4, dz=w.dx * (70.0 / 420.0) / (35.4 / 240.0), every=6)
    from paper_2401_07416_b200 import Tdse
    t = Tdse.from_workload(w)
    t.set_option("kernel", kernel)
    t.set_option("tblock", tblock)
    o = OracleRun.from_workload(w, entry=0, dtype="f64", round_to="f32" if dtype == "f32" else None)
    assert o.dy == w.dy and o.dz == w.dz and len({o.coef[0], o.coef[1], o.coef[2]}) == 3
    # S0 / S1 on the anisotropic mesh
    V = t.read_potential(0)
    R, I = t.read_psi(0)
    if dtype == "f64":
        assert np.max(np.abs(V - o.V64)) <= 1e-13 * max(1.0, np.max(np.abs(o.V64)))
        assert rel_l2(R, o.R) < 1e-14 and rel_l2(I, o.I) < 1e-14
    else:
        assert np.all(np.abs(V.astype(np.float64) - o.V) <= np.spacing(np.abs(o.V).astype(np.float32)).astype(np.float64))
        assert rel_l2(R, o.R) < 1e-7 and rel_l2(I, o.I) < 1e-7
    t.step(w.steps)
    o.step(w.steps)
    assert t.get_info("kernel") == kernel
    tol = TOL[dtype]
    R, I = t.read_psi(0)
    D, tr = t.detector_read(0)
    assert rel_l2(R, o.R) < tol and rel_l2(I, o.I) < tol
    assert rel_l2(D, o.D) < tol and rel_l2(tr, o.trace) < tol          # trace carries dx*dy
    qv, qp = t.norm(0)
    ov, op = o.norm()
    assert abs(qv - ov) < 10 * tol * abs(ov) and abs(qp - op) < 10 * tol * abs(op)   # norms carry dx*dy*dz
    t.close()


# ------------------------------------------------------------------------------------------
# unit-cell potential tiled and interpolated on the device
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_potential_cell_matches_oracle(dtype):
    import torch
    rng = np.random.default_rng(9)
    cell = -5.0 * rng.random((9, 7, 6))
    nx, ny, nz, dx, dy, dz = 44, 38, 30, 0.17, 0.21, 0.19
    a, org = (1.9, 2.3, 4.0), (0.3, -0.7, 1.0)
    t = make_ctx(nx, ny, nz, 2, dx, 0.001, dtype)
    t.set_spacing(dy, dz)
    t.set_boundary(PERIODIC, PERIODIC, DIRICHLET)
    t.set_potential_cell(0, cell, a, org, -4.0, -0.5)                                    # host cell
    t.set_potential_cell(1, torch.from_numpy(cell).cuda(), a, org, -4.0, -0.5)           # device cell
    want = oracle.potential_cell(nx, ny, nz, dx, cell, a, org, -4.0, -0.5, dy, dz)
    for b in range(2):
        V = t.read_potential(b)
        # the mesh coordinate i*dx - x0 may be fused into one FMA on the device: last-bit differences in the
        # interpolation weights, continuous in the result
        if dtype == "f64":
            assert np.max(np.abs(V - want)) <= 1e-13 * np.max(np.abs(want))
        else:
            assert np.all(np.abs(V.astype(np.float64) - want) <= np.spacing(np.abs(want).astype(np.float32)).astype(np.float64))
    assert want.min() == -4.0 and want.max() == -0.5   # both clamps are exercised
    t.close()


# ------------------------------------------------------------------------------------------
# edge cases and error behaviour of the boundary
# ------------------------------------------------------------------------------------------
def test_call_order_and_stability_errors():
    from paper_2401_07416_b200 import Tdse, TdseError, TDSE_ESTATE, TDSE_EUNSTABLE, TDSE_EINVAL
    t = make_ctx(16, 16, 16, 1, 0.2, 0.004, "f64")
    with pytest.raises(TdseError) as e:
        t.step(1)
    assert e.value.code == TDSE_ESTATE
    with pytest.raises(TdseError) as e:
        t.set_wavepacket(0, 1.6, 1.6, 1.6, 0.5, 0, 0, 1.0)
    assert e.value.code == TDSE_ESTATE
    t.set_potential(0, np.zeros((0, 6)), -1.0, 0.0)
    with pytest.raises(TdseError) as e:
        t.step(1)
    assert e.value.code == TDSE_ESTATE
    t.set_wavepacket(0, 1.6, 1.6, 1.6, 0.5, 0, 0, 1.0)
    t.step(0)
    t.step(3)
    with pytest.raises(TdseError) as e:
        t.set_potential(3, np.zeros((0, 6)), -1.0, 0.0)
    assert e.value.code == TDSE_EINVAL
    with pytest.raises(TdseError) as e:
        t.set_boundary(0, 0, 5)
    assert e.value.code == TDSE_EINVAL
    t.close()
    # dt past the sufficient bound 2 / (6/dx^2 + max|V|)
    u = make_ctx(8, 8, 8, 1, 0.2, 1.01 * 0.04 / 3.0, "f64")
    u.set_potential(0, np.zeros((0, 6)), 0.0, 0.0)
    R0, I0 = random_state(99, (8, 8, 8))
    u.set_state(0, R0, I0)
    with pytest.raises(TdseError) as e:
        u.step(1)
    assert e.value.code == TDSE_EUNSTABLE
    u.set_option("allow_unstable", 1)
    u.step(400)                                   # blow-up just past dt_c = dx^2/3, as the oracle pin
    R, _ = u.read_psi(0)
    o = OracleRun(8, 8, 8, 0.2, 1.01 * 0.04 / 3.0, bc=(PERIODIC,) * 3).set_potential_grid(np.zeros((8, 8, 8)))
    o.set_state(R0, I0).step(400)
    assert np.linalg.norm(R) / np.linalg.norm(R0) > 1e20
    assert rel_l2(R, o.R) < 1e-9
    u.close()


def test_three_array_workspace_runs_twopass_only():
    from paper_2401_07416_b200 import Tdse, TdseError, TDSE_EINVAL
    w = make_config(0, n=(24, 24, 24), steps=0)
    t = Tdse.from_workload(w, pingpong=False)
    assert t.get_info("pingpong") == 0
    t.step(10)
    assert t.get_info("kernel") == TWOPASS
    t.set_option("kernel", FUSED)
    with pytest.raises(TdseError) as e:
        t.step(1)
    assert e.value.code == TDSE_EINVAL
    R, I = t.read_psi(0)
    o = OracleRun.from_workload(w).step(10)
    assert rel_l2(R, o.R) < 1e-12
    t.close()


def test_odd_nx_falls_back_to_twopass_under_auto():
    from paper_2401_07416_b200 import Tdse
    w = make_config(1, n=(23, 17, 19), steps=0)
    t = Tdse.from_workload(w)
    t.step(12)
    assert t.get_info("kernel") == TWOPASS
    R, I = t.read_psi(0)
    D, tr = t.detector_read(0)
    o = OracleRun.from_workload(w).step(12)
    assert rel_l2(R, o.R) < 1e-12 and rel_l2(I, o.I) < 1e-12 and rel_l2(D, o.D) < 1e-12
    t.close()


def test_user_stream_and_device_resident_inputs():
    import torch
    from paper_2401_07416_b200 import Tdse
    w = make_config(3, n=(32, 32, 32), batch=2, steps=0)
    s = torch.cuda.Stream()
    t = Tdse(w.nx, w.ny, w.nz, w.batch, w.dx, w.dt, 1.0, 1.0, w.dtype, stream=s)
    t.set_boundary(*w.bc, w.absorb_lo, w.absorb_hi, w.strength, w.power)
    dev_atoms = [torch.from_numpy(a).to("cuda") for a in w.atoms]
    torch.cuda.synchronize()
    for b in range(w.batch):
        t.set_potential_device(b, dev_atoms[b], w.atoms[b].shape[0], w.vmin, w.vmax, w.rcut)
    p = w.packet
    t.set_wavepacket(-1, p["x0"], p["y0"], p["z0"], p["sigma"], p["kx"], p["ky"], p["kz"], 0.0)
    t.set_detector(w.k_det, 10, 4)
    t.step(40)
    s.synchronize()
    img_ptr, tr_ptr, ms = t.detector_device()
    assert img_ptr and tr_ptr and ms == 4
    for b in range(w.batch):
        R, I = t.read_psi(b)
        D, tr = t.detector_read(b)
        o = oracle_for(w, b, 40)
        assert rel_l2(R, o.R) < 1e-4 and rel_l2(D, o.D) < 1e-4 and rel_l2(tr, o.trace) < 1e-4
    t.close()


# ------------------------------------------------------------------------------------------
# call order, devices, buffers (host-side logic of the library)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel,tblock", VARIANTS)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("first,then", [((PERIODIC, PERIODIC, DIRICHLET), (DIRICHLET, DIRICHLET, DIRICHLET)),
                                        ((DIRICHLET, DIRICHLET, DIRICHLET), (PERIODIC, PERIODIC, PERIODIC)),
                                        ((PERIODIC, DIRICHLET, PERIODIC), (DIRICHLET, PERIODIC, DIRICHLET))])
def test_boundary_flags_changed_after_the_data_was_loaded(kernel, tblock, dtype, first, then):
    """tdse_set_boundary after tdse_set_state / tdse_set_potential_grid: the fused kernel takes its x/y neighbours from
    the storage frames, which were filled under the old flags and must follow the new ones (include/tdse.h)."""
    nx, ny, nz, dx, dt, steps = 40, 24, 18, 0.25, 0.004, 9
    t = make_ctx(nx, ny, nz, 1, dx, dt, dtype)
    t.set_boundary(*first, 3, 3, 0.07, 2)
    t.set_option("kernel", kernel)
    t.set_option("tblock", tblock)
    V = random_potential(300, (nz, ny, nx), -30.0, 5.0)
    R0, I0 = random_state(301, (nz, ny, nx))
    t.set_potential_grid(0, V.astype(t.np_dtype))
    t.set_state(0, R0.astype(t.np_dtype), I0.astype(t.np_dtype))
    t.set_boundary(*then, 3, 3, 0.07, 2)
    t.set_detector(2, 3, 4)
    t.step(steps)
    o = OracleRun(nx, ny, nz, dx, dt, bc=then, absorb_lo=3, absorb_hi=3, strength=0.07,
                  round_to="f32" if dtype == "f32" else None)
    o.set_potential_grid(V).set_state(R0, I0).set_detector(2, 3).step(steps)
    R, I = t.read_psi(0)
    D, tr = t.detector_read(0)
    tol = TOL[dtype]
    assert t.get_info("kernel") == kernel
    assert rel_l2(R, o.R) < tol and rel_l2(I, o.I) < tol and rel_l2(D, o.D) < tol and rel_l2(tr, o.trace) < tol
    t.close()


def test_atoms_many_periods_outside_the_box_with_a_cutoff():
    """The pair test takes the nearest image over any number of periods; the brick culling of the builder must keep
    the same atoms (an atom three box lengths outside a periodic axis is as close as its image inside)."""
    from paper_2401_07416_b200 import Tdse
    w = make_config(4, n=(48, 40, 56), batch=1, dtype="f64")
    lx, ly = w.nx * w.dx, w.ny * w.dx
    atoms = w.atoms[0].copy()
    atoms[::3, 0] += 3.0 * lx
    atoms[1::3, 1] -= 2.0 * ly
    w2 = w.with_(atoms=[atoms], rcut=3.0)
    t = Tdse.from_workload(w2)
    V = t.read_potential(0)
    t.close()
    o = OracleRun.from_workload(w2, entry=0, dtype="f64")
    o_in = OracleRun.from_workload(w.with_(rcut=3.0), entry=0, dtype="f64")
    assert np.max(np.abs(V - o.V64)) <= 1e-13 * max(1.0, np.max(np.abs(o.V64)))
    assert np.max(np.abs(o.V64 - o_in.V64)) <= 1e-9 * np.max(np.abs(o_in.V64))     # the shifted list is the same crystal


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("rcut", [0.0, 3.07])     # not a multiple of dx: with an atom ON a grid point, cells at lattice distances
def test_screening_lengths_far_below_the_mesh_and_denormal(dtype, rcut):   # (12, 16, 0) dx = 20 dx would sit exactly on the cutoff, where keep / skip hangs on the last bit of r^2
    """exp(-r/screen) with screen = 1e-8 (x = -1e10) and a denormal screen (1/screen = inf, x = -inf) underflows to 0 in
    the definition (include/tdse.h; libm in the oracle).  The builder's table exp must do the same instead of wrapping
    its integer exponent or producing inf - inf: those atoms contribute nothing, the others are unaffected."""
    from paper_2401_07416_b200 import Tdse
    w = make_config(4, n=(48, 40, 56), batch=1, dtype=dtype)
    atoms = w.atoms[0].copy()
    atoms[:, 0:3] += np.array([0.0123, 0.0077, 0.0031]) * w.dx     # no screened atom sits exactly on a grid point (r = 0)
    atoms[0::4, 5] = 1e-8          # column 5 = screen
    atoms[1::4, 5] = 5e-324        # smallest denormal
    atoms[2::4, 5] = 2e-3          # x around -1e3 .. -1e4: below -746, inside the int range
    atoms[3, 0:3] = (7 * w.dx, 5 * w.dx, 9 * w.dx)     # an unscreened-range atom exactly on a grid point stays finite
    w2 = w.with_(atoms=[atoms], rcut=rcut)
    t = Tdse.from_workload(w2)
    V = t.read_potential(0)
    t.close()
    o = OracleRun.from_workload(w2, entry=0, dtype="f64", round_to="f32" if dtype == "f32" else None)
    assert np.all(np.isfinite(V))
    if dtype == "f64":
        assert np.max(np.abs(V - o.V64)) <= 1e-13 * max(1.0, np.max(np.abs(o.V64)))
    else:
        ulp = np.spacing(np.abs(o.V).astype(np.float32)).astype(np.float64)
        assert np.all(np.abs(V.astype(np.float64) - o.V) <= ulp)
    assert np.ptp(o.V64) > 0.1                                       # the remaining quarter of the atoms still shapes V


def test_set_detector_keeps_the_trace_buffer_and_survives_a_failed_allocation():
    from paper_2401_07416_b200 import Tdse, TdseError, TDSE_ENOMEM
    w = make_config(0, n=(24, 24, 24), steps=0, batch=64)
    t = Tdse.from_workload(w)
    t.set_detector(5, 2, 6)
    _, tr0, ms0 = t.detector_device()
    t.step(4)
    t.set_detector(7, 2, 6)                        # same max_samples: same buffer, counters reset
    _, tr1, ms1 = t.detector_device()
    assert tr0 == tr1 and ms0 == ms1 == 6 and t.get_info("nsamples") == 0
    with pytest.raises(TdseError) as e:
        t.set_detector(7, 2, 2 ** 31 - 1)          # 64 entries x 16 GiB of doubles: beyond any device
    assert e.value.code == TDSE_ENOMEM
    _, tr2, ms2 = t.detector_device()
    assert tr2 == tr1 and ms2 == 6                 # the previous set-up is still in force
    t.step(4)
    D, tr = t.detector_read(0)
    o = OracleRun.from_workload(w).step(4).set_detector(7, 2).step(4)      # set_detector resets image, trace and counter only
    assert len(tr) == 2 and rel_l2(D, o.D) < 1e-12 and rel_l2(tr, o.trace) < 1e-12
    t.close()


def test_contexts_on_two_devices_in_one_process():
    """cudaFuncSetAttribute is per device and every call must run on its context's device whatever is current."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    from paper_2401_07416_b200 import Tdse
    w = make_config(1, n=(32, 32, 40), steps=0)
    ctxs = [Tdse.from_workload(w, device="cuda:%d" % d) for d in (0, 1)]
    torch.cuda.set_device(0)
    for t in ctxs:
        t.step(20)
    o = OracleRun.from_workload(w).step(20)
    for t in ctxs:
        assert t.get_info("kernel") == FUSED
        R, I = t.read_psi(0)
        assert rel_l2(R, o.R) < 1e-11 and rel_l2(I, o.I) < 1e-11
        t.close()
    assert torch.cuda.current_device() == 0


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("idx,shape,batch", [(3, (36, 40, 44), 5), (3, (128, 24, 20), 3), (4, (48, 40, 56), 3), (2, (40, 36, 48), 2)])
def test_batched_potential_build_is_bit_identical_to_one_entry_at_a_time(idx, shape, batch, dtype):
    """tdse_set_potential_batch (one launch, shared substrate prefix summed once, host or device lists) against
    tdse_set_potential entry by entry: the same list-order fp64 sums, so every bit agrees; entry 0 and the last entry
    against the oracle as well.  Shapes cover both cells-per-thread variants (nx >= 128) and the cutoff variant (cfg 4)."""
    import torch
    from paper_2401_07416_b200 import Tdse
    w = make_config(idx, n=shape, batch=batch, dtype=dtype)
    if idx == 4:
        w = w.with_(atoms=[w.atoms[0]] + [np.concatenate([w.atoms[0][:9], a[9:]]) for a in w.atoms[1:]])   # shared prefix of 9 atoms together with the cutoff
    cat = np.ascontiguousarray(np.concatenate(w.atoms, axis=0))
    off = np.concatenate([[0], np.cumsum([a.shape[0] for a in w.atoms])]).astype(np.int32)
    ref = make_ctx(w.nx, w.ny, w.nz, batch, w.dx, w.dt, dtype)
    ref.set_boundary(*w.bc, w.absorb_lo, w.absorb_hi, w.strength, w.power)
    for b in range(batch):
        ref.set_potential(b, w.atoms[b], w.vmin, w.vmax, w.rcut)
    Vref = [ref.read_potential(b) for b in range(batch)]
    ref.close()
    for on_device in (False, True):
        t = make_ctx(w.nx, w.ny, w.nz, batch, w.dx, w.dt, dtype)
        t.set_boundary(*w.bc, w.absorb_lo, w.absorb_hi, w.strength, w.power)
        lists = torch.from_numpy(cat).cuda() if on_device else cat
        t.set_potential_batch(lists, off, w.vmin, w.vmax, w.rcut)
        for b in range(batch):
            assert np.array_equal(t.read_potential(b), Vref[b]), (on_device, b)
        # the framed storage too: the step kernel reads V through its periodic images
        p = w.packet
        t.set_wavepacket(-1, p["x0"], p["y0"], p["z0"], p["sigma"], p["kx"], p["ky"], p["kz"], 0.0)
        t.step(6)
        R, _ = t.read_psi(batch - 1)
        o = oracle_for(w, batch - 1, 6)
        assert rel_l2(R, o.R) < TOL[dtype]
        t.close()
    for b in (0, batch - 1):
        o = OracleRun.from_workload(w, entry=b, dtype="f64", round_to="f32" if dtype == "f32" else None)
        if dtype == "f64":
            assert np.max(np.abs(Vref[b] - o.V64)) <= 1e-13 * max(1.0, np.max(np.abs(o.V64)))
        else:
            ulp = np.spacing(np.abs(o.V).astype(np.float32)).astype(np.float64)
            assert np.all(np.abs(Vref[b].astype(np.float64) - o.V) <= ulp)


@pytest.mark.parametrize("tblock", [1, 2])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape,bc,batch", [((72, 40, 37), BCS[0], 2), ((136, 70, 21), BCS[3], 1), ((64, 64, 16), BCS[1], 3),
                                            ((128, 128, 40), BCS[2], 2), ((40, 24, 5), BCS[4], 1), ((132, 66, 9), BCS[2], 1),
                                            ((64, 32, 12), BCS[2], 2), ((8, 8, 6), BCS[2], 1)])
def test_iteration_barrier_variants_are_bit_identical(tblock, dtype, shape, bc, batch):
    """tdse_set_option("variant"): the fused kernel with the per-plane block barrier (2) and with the split arrive / wait
    mbarrier (1) do the same arithmetic in the same order -- every bit of psi and of the detector output must agree, over
    several z chunks and launches; 0 lets the launcher pick (the split barrier on single-wave f64 grids)."""
    nx, ny, nz = shape
    dx, dt, steps = 0.25, 0.004, 14
    out = []
    variants = (2, 1, 0)
    for variant in variants:
        t = make_ctx(nx, ny, nz, batch, dx, dt, dtype)
        t.set_boundary(*bc, min(4, nz // 3), min(4, nz // 3), 0.07, 2)
        t.set_option("kernel", FUSED)
        t.set_option("tblock", tblock)
        t.set_option("variant", variant)
        t.set_detector(min(3, nz - 1), 4, 8)
        for b in range(batch):
            V = random_potential(500 + b, (nz, ny, nx), -30.0, 5.0)
            R0, I0 = random_state(600 + b, (nz, ny, nx))
            t.set_potential_grid(b, V.astype(t.np_dtype))
            t.set_state(b, R0.astype(t.np_dtype), I0.astype(t.np_dtype))
        t.step(steps)
        out.append([t.read_psi(b) + t.detector_read(b) for b in range(batch)])
        t.close()
    for v, res in zip(variants[1:], out[1:]):
        for b in range(batch):
            for x0, x1 in zip(out[0][b], res[b]):
                assert np.array_equal(x0, x1), "variant %s, entry %d" % (v, b)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("include_t0,ring_slots,pinned", [(True, 2, True), (False, 3, True), (True, 5, False)])
def test_streamed_frames_equal_the_flat_frame_mode_bit_for_bit(dtype, include_t0, ring_slots, pinned):
    """tdse_set_frame_stream (device ring of a few sample slots, one asynchronous copy per slot into a host buffer) keeps
    the frames tdse_set_frames keeps, every bit, with many more frames than ring slots; the accumulated image and the trace
    do not change; frames beyond the capacity are dropped; and a second trajectory after a reset starts at frame 0 again."""
    from paper_2401_07416_b200 import Tdse, TdseError, TDSE_ESTATE
    w = make_config(3, n=(40, 36, 44), batch=3, steps=57, dtype=dtype).with_(every=3)
    nfr = w.steps // w.every + (1 if include_t0 else 0)
    flat = Tdse.from_workload(w)
    flat.set_frames(nfr, include_t0)
    flat.step(w.steps)
    want = [flat.frames_read(b) for b in range(w.batch)]
    want_det = [flat.detector_read(b) for b in range(w.batch)]
    flat.close()

    t = Tdse.from_workload(w)
    with pytest.raises(TdseError) as e:
        t.frames_sync()
    assert e.value.code == TDSE_ESTATE
    cap = nfr - 2                                          # the last two frames do not fit
    t.set_frame_stream(cap, ring_slots, include_t0, pinned=pinned)
    t.step(20)
    t.step(w.steps - 20)
    got = t.frames_sync()
    assert got.shape == (w.batch, cap, w.ny, w.nx) and t.get_info("nframes") == nfr
    for b in range(w.batch):
        assert np.array_equal(got[b], want[b][:cap])
        D, tr = t.detector_read(b)
        assert np.array_equal(D, want_det[b][0]) and np.array_equal(tr, want_det[b][1])
    with pytest.raises(TdseError) as e:                    # the frames are not on the device in this mode
        t.dissimilarity(0, 1)
    assert e.value.code == TDSE_ESTATE
    # a second trajectory: same packet again, frames restart at slot 0
    p = w.packet
    t.set_wavepacket(-1, p["x0"], p["y0"], p["z0"], p["sigma"], p["kx"], p["ky"], p["kz"], p["amplitude"])
    t.step(w.steps)
    again = t.frames_sync()
    for b in range(w.batch):
        assert np.array_equal(again[b], want[b][:cap])
    t.set_frame_stream(0, 0)                               # off
    t.close()


# ------------------------------------------------------------------------------------------
# the paper's own mesh as ONE pass: unit-cell potential resampled onto 240 x 240 x (420 + 100)
# anisotropic cells, periodic on all axes with the 100-plane absorber at the bottom, packet moving down, a frame every
# 20 steps streamed to the host, then eq (16) between the configurations
# ------------------------------------------------------------------------------------------
def _paper_ctx(m, **kw):
    from paper_2401_07416_b200 import Tdse
    t = Tdse(m.nx, m.ny, m.nz, m.batch, m.dx, m.dt, m.mass, m.hbar, m.dtype, **kw)
    t.set_spacing(m.dy, m.dz)
    t.set_boundary(*m.bc, m.absorb_lo, m.absorb_hi, m.strength, m.power)
    for b in range(m.batch):
        t.set_potential_cell(b, m.unit_cells[b], m.cell_edges, m.cell_origin, m.vmin, m.vmax)
    p = m.packet
    t.set_wavepacket(-1, p["x0"], p["y0"], p["z0"], p["sigma"], p["kx"], p["ky"], p["kz"], p["amplitude"])
    return t


def _paper_oracle(m, b):
    o = OracleRun(m.nx, m.ny, m.nz, m.dx, m.dt, m.mass, m.hbar, "f64", m.bc, m.absorb_lo, m.absorb_hi, m.strength, m.power,
                  round_to="f32" if m.dtype == "f32" else None, dy=m.dy, dz=m.dz)
    o.set_potential_cell(m.unit_cells[b], m.cell_edges, m.cell_origin, m.vmin, m.vmax)
    o.set_wavepacket(**m.packet)
    o.set_detector(m.k_det, m.every)
    return o.set_frames(True, True)


@pytest.mark.parametrize("n,steps,dtype", [((48, 32, 84), 200, "f64"), ((48, 32, 84), 200, "f32"), (None, 300, "f32")])
def test_paper_mesh_whole_pass_matches_oracle(n, steps, dtype):
    """n = None is the full 240 x 240 x 520 mesh: nx = 240 is 3.75 of the fused kernel's 64-wide f32 tiles and ny = 240 is 7.5 of
    its 32 rows, so the ragged last tile column and row run at the size the paper uses.  Entries 0 and batch-1 against the
    oracle: V, psi, image, trace and every streamed frame; the device-frame run must reproduce the streamed frames bit for
    bit, and d_kj from it must match eq (16) evaluated by the oracle on the oracle's own frames."""
    from workloads import paper_mesh
    m = paper_mesh(batch=3, steps=steps, n=n, dtype=dtype)
    tol = TOL[dtype]
    nfr = steps // m.every + 1
    t = _paper_ctx(m)
    t.set_detector(m.k_det, m.every, nfr)
    t.set_frame_stream(nfr, 3, True)
    t.step(steps)
    got = t.frames_sync().copy()
    assert got.shape == (m.batch, nfr, m.ny, m.nx)
    if n is None:
        assert (t.get_info("kernel"), t.get_info("tblock"), t.get_info("tile_x"), t.get_info("tile_y")) == (FUSED, 2, 64, 32)
    ora = {}
    for b in (0, m.batch - 1):
        o = _paper_oracle(m, b)
        V = t.read_potential(b)
        if dtype == "f64":
            assert np.max(np.abs(V - o.V64)) <= 1e-13 * max(1.0, np.max(np.abs(o.V64)))
        else:
            assert np.all(np.abs(V.astype(np.float64) - o.V) <= np.spacing(np.abs(o.V).astype(np.float32)).astype(np.float64))
        o.step(steps)
        R, I = t.read_psi(b)
        D, tr = t.detector_read(b)
        errs = (rel_l2(R, o.R), rel_l2(I, o.I), rel_l2(D, o.D), rel_l2(tr, o.trace))
        cell = max(max_abs_rel(R, o.R), max_abs_rel(I, o.I), max_abs_rel(D, o.D))
        fr_err = max(rel_l2(got[b][s], o.frames[s]) for s in range(nfr))
        print("paper mesh %s %dx%dx%d entry %d, %d steps: rel-L2 R %.3e I %.3e D %.3e trace %.3e frames %.3e, per-cell %.3e"
              % (dtype, m.nx, m.ny, m.nz, b, steps, *errs, fr_err, cell))
        assert max(errs) < tol and cell < CELL_TOL[dtype] and fr_err < tol and len(o.frames) == nfr
        ora[b] = np.array(o.frames)
    # the same trajectories with the frames kept on the device, then eq (16)
    t.set_frames(nfr, True)
    p = m.packet
    t.set_wavepacket(-1, p["x0"], p["y0"], p["z0"], p["sigma"], p["kx"], p["ky"], p["kz"], p["amplitude"])
    t.step(steps)
    for b in range(m.batch):
        assert np.array_equal(t.frames_read(b), got[b])
    d = t.dissimilarity(1, nfr - 1)
    want = oracle.dissimilarity(ora[0], ora[m.batch - 1], m.dx * m.dy, 1, nfr - 1)
    assert want > 0 and abs(d[0, m.batch - 1] - want) <= 10 * tol * want
    t.close()


def _random_ctx(nx, ny, nz, batch, dtype, seed):
    t = make_ctx(nx, ny, nz, batch, 0.25, 0.004, dtype)
    t.set_boundary(PERIODIC, PERIODIC, DIRICHLET, 2, 2, 0.07, 2)
    for b in range(batch):
        V = random_potential(seed + b, (nz, ny, nx), -30.0, 5.0)
        R0, I0 = random_state(seed + 100 + b, (nz, ny, nx))
        t.set_potential_grid(b, V.astype(t.np_dtype))
        t.set_state(b, R0.astype(t.np_dtype), I0.astype(t.np_dtype))
    return t


@pytest.mark.parametrize("pinned", [True, False])
def test_streamed_frames_ring_of_two_sampled_every_step_on_large_planes(pinned):
    """The hard case for slot reuse: a sample after EVERY step, only two ring slots, 2 MiB per entry and frame (512 x 512),
    so the step that comes back to a slot finds its copy-out still under way (always with a pageable host buffer, where
    the copies serialise; usually with a pinned one).  The detector launch that follows the wait on the slot's event is
    a plain stream-ordered launch (no programmatic dependent launch), and every frame must equal the flat mode's."""
    nx, ny, nz, batch, steps = 512, 512, 12, 2, 24
    flat = _random_ctx(nx, ny, nz, batch, "f32", 900)
    flat.set_detector(5, 1, steps)
    flat.set_frames(steps + 1, True)
    flat.step(steps)
    want = [flat.frames_read(b) for b in range(batch)]
    flat.close()
    t = _random_ctx(nx, ny, nz, batch, "f32", 900)
    t.set_detector(5, 1, steps)
    t.set_frame_stream(steps + 1, 2, True, pinned=pinned)
    t.step(steps)
    got = t.frames_sync()
    assert got.shape == (batch, steps + 1, ny, nx)
    for b in range(batch):
        assert np.array_equal(got[b], want[b]), "entry %d" % b
    t.close()


def test_streamed_frames_with_a_host_pitch_beyond_the_2d_copy_limit():
    """capacity * ny * nx * 8 bytes = 257 * 8 MiB > 2^31 - 1 (cudaDevAttrMaxPitch): the strided 2-D copy cannot carry that
    pitch, so a slot leaves as one copy per entry.  Same frames as the flat mode, at the right places of the host buffer
    (only the few frames taken are ever touched in the 4 GiB pageable buffer)."""
    nx, ny, nz, batch, steps, cap = 1024, 1024, 8, 2, 3, 257
    flat = _random_ctx(nx, ny, nz, batch, "f32", 950)
    flat.set_detector(3, 1, steps)
    flat.set_frames(steps + 1, True)
    flat.step(steps)
    want = [flat.frames_read(b) for b in range(batch)]
    flat.close()
    t = _random_ctx(nx, ny, nz, batch, "f32", 950)
    t.set_detector(3, 1, steps)
    t.set_frame_stream(cap, 2, True, pinned=False)
    t.step(steps)
    got = t.frames_sync()
    assert got.shape == (batch, steps + 1, ny, nx)
    for b in range(batch):
        assert np.array_equal(got[b], want[b]), "entry %d" % b
    t.close()


def test_batch_build_and_frame_stream_argument_errors_and_empty_lists():
    """Host-side checks of the two round-2 calls: bad offsets / NULL / too few ring slots fail with TDSE_EINVAL and leave the
    context usable; entries with an empty atom list get V = clamp(0) (or just the shared prefix when every list is short)."""
    import ctypes as C
    from paper_2401_07416_b200 import Tdse, TdseError, TDSE_EINVAL
    w = make_config(3, n=(32, 32, 24), batch=3, dtype="f64")
    t = make_ctx(w.nx, w.ny, w.nz, 3, w.dx, w.dt, "f64")
    t.set_boundary(*w.bc, 2, 2, 0.05, 2)
    atoms = np.ascontiguousarray(np.concatenate(w.atoms[:2]))
    n0, n1 = w.atoms[0].shape[0], w.atoms[1].shape[0]
    for bad in ([0, n0, n0 - 1, n0 + n1], [-1, n0, n0, n0 + n1]):
        with pytest.raises(TdseError) as e:
            t.set_potential_batch(atoms, bad, w.vmin, w.vmax)
        assert e.value.code == TDSE_EINVAL
    with pytest.raises(TdseError) as e:
        t.set_potential_batch(atoms, [0, n0, n0, n0 + n1], 1.0, -1.0)      # vmin > vmax
    assert e.value.code == TDSE_EINVAL
    # entry 1 has no atoms at all
    t.set_potential_batch(atoms, [0, n0, n0, n0 + n1], w.vmin, w.vmax)
    assert np.array_equal(t.read_potential(1), np.zeros((w.nz, w.ny, w.nx)))
    for b, lst in ((0, w.atoms[0]), (2, w.atoms[1])):
        o = OracleRun(w.nx, w.ny, w.nz, w.dx, w.dt, bc=w.bc).set_potential_atoms(lst, w.vmin, w.vmax)
        assert np.max(np.abs(t.read_potential(b) - o.V64)) <= 1e-13 * max(1.0, np.max(np.abs(o.V64)))
    # frame stream: needs a buffer and >= 2 slots
    buf = np.zeros((3, 4, w.ny, w.nx))
    dp = C.POINTER(C.c_double)
    assert t.L.tdse_set_frame_stream(t._h, buf.ctypes.data_as(dp), 4, 1, 1) == TDSE_EINVAL
    assert t.L.tdse_set_frame_stream(t._h, None, 4, 2, 1) == TDSE_EINVAL
    assert t.L.tdse_set_frame_stream(t._h, buf.ctypes.data_as(dp), -1, 2, 1) == TDSE_EINVAL
    # still usable: pageable host buffer given directly through the C ABI, 2 slots for 4 frames
    p = w.packet
    t.set_wavepacket(-1, p["x0"], p["y0"], p["z0"], p["sigma"], p["kx"], p["ky"], p["kz"], 0.0)
    t.set_detector(3, 2, 8)
    assert t.L.tdse_set_frame_stream(t._h, buf.ctypes.data_as(dp), 4, 2, 1) == 0
    t.step(6)
    n = C.c_int(0)
    assert t.L.tdse_frames_sync(t._h, C.byref(n)) == 0 and n.value == 4
    assert np.all(buf.sum(axis=(2, 3)) > 0)
    assert t.L.tdse_set_frame_stream(t._h, None, 0, 0, 1) == 0      # off again before the buffer goes
    t.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape,bc,batch", [((72, 40, 37), BCS[0], 2), ((136, 70, 21), BCS[2], 1), ((64, 32, 9), BCS[1], 3),
                                            ((128, 128, 24), BCS[2], 1), ((8, 8, 5), BCS[3], 2)])
def test_nothing_is_written_outside_the_workspace(shape, bc, batch, dtype):
    """Guard bands on both sides of a caller-owned workspace (and between its five arrays there is none to spare: they are
    contiguous) stay untouched through potential build, packet init, fused steps of both temporal blocks and the two-pass
    kernel: the kernels advance store addresses from below the first plane of a chunk and must never dereference them there."""
    import ctypes as C
    import torch
    from paper_2401_07416_b200 import binding as B
    nx, ny, nz = shape
    L = B.load()
    code = B.TDSE_F32 if dtype == "f32" else B.TDSE_F64
    nbytes = L.tdse_workspace_bytes(nx, ny, nz, batch, code, 1)
    guard = 1 << 20
    buf = torch.full((nbytes + 2 * guard,), 0xA5, dtype=torch.uint8, device="cuda")
    assert (buf.data_ptr() + guard) % 256 == 0
    h = C.c_void_p()
    assert L.tdse_create(C.byref(h), nx, ny, nz, batch, 0.25, 0.004, 1.0, 1.0, code) == 0
    assert L.tdse_bind(h, buf.data_ptr() + guard, nbytes, None) == 0
    assert L.tdse_set_boundary(h, *bc, 2, 2, 0.07, 2) == 0
    atoms = B.atoms_array(np.array([[nx * 0.1, ny * 0.1, nz * 0.1, 3.0, 0.2, 0.6], [0.3, 0.2, 0.1, 2.0, 0.1, 0.0]]))
    assert L.tdse_set_potential(h, -1, atoms[0], atoms[1], -50.0, 0.0, 0.0) == 0
    assert L.tdse_set_wavepacket(h, -1, nx * 0.12, ny * 0.12, nz * 0.1, 1.0, 0.0, 0.0, 1.0, 0.0) == 0
    assert L.tdse_set_detector(h, 1, 3, 8) == 0
    for kernel, tblock in ((2, 2), (2, 1), (1, 1)):
        if kernel == 2 and not fused_eligible(nx, ny, dtype):
            continue
        assert L.tdse_set_option(h, b"kernel", kernel) == 0 and L.tdse_set_option(h, b"tblock", tblock) == 0
        for variant in (1, 2):
            assert L.tdse_set_option(h, b"variant", variant) == 0
            assert L.tdse_step(h, 7) == 0
    torch.cuda.synchronize()
    assert bool((buf[:guard] == 0xA5).all()) and bool((buf[guard + nbytes:] == 0xA5).all())
    L.tdse_destroy(h)
