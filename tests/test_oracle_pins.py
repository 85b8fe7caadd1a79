"""Pins for the CPU oracle (oracle/) against what the paper and the mathematics fix.

None of these retype the oracle's loops: each one reaches the same result by a different
route (dense spectral decomposition, FFT, exact matrix exponential, continuum closed forms,
textbook constants, values printed in PAPER.md) so that a dropped term, wrong sign, wrong
index or transposed boundary flag fails at least one of them.  SURVEY.md section 8(c).
"""
import json
import math
import os

import numpy as np
import pytest

import oracle
from oracle import OracleRun
from workloads import make_config, random_state, random_potential, PERIODIC, DIRICHLET

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


# ---------------------------------------------------------------------------------------
# independent dense construction of A = dt H / hbar on tiny grids (textbook Kronecker sum)
# ---------------------------------------------------------------------------------------
def d2_matrix(n, bc):
    D = np.zeros((n, n))
    for i in range(n):
        D[i, i] -= 2.0
        for nb in (i - 1, i + 1):
            if 0 <= nb < n:
                D[i, nb] += 1.0
            elif bc == PERIODIC:
                D[i, nb % n] += 1.0
    return D


def dense_A(nx, ny, nz, bc, c, cv, V):
    """A f = -c (d2x + d2y + d2z) f + cv V f on the flat index (k*ny + j)*nx + i."""
    Ix, Iy, Iz = np.eye(nx), np.eye(ny), np.eye(nz)
    lap = (np.kron(np.kron(d2_matrix(nz, bc[2]), Iy), Ix)
           + np.kron(np.kron(Iz, d2_matrix(ny, bc[1])), Ix)
           + np.kron(np.kron(Iz, Iy), d2_matrix(nx, bc[0])))
    return -c * lap + cv * np.diag(np.asarray(V, dtype=np.float64).ravel())


def leapfrog_modes(a, r0, i0, n):
    """Per spectral mode: (r, i)^{n} = M^n (r, i)^0, M = [[1-a^2, a], [-a, 1]]."""
    r = np.empty_like(r0)
    i = np.empty_like(i0)
    for m in range(a.size):
        Mn = np.linalg.matrix_power(np.array([[1.0 - a[m] ** 2, a[m]], [-a[m], 1.0]]), n)
        r[m], i[m] = Mn @ np.array([r0[m], i0[m]])
    return r, i


TINY = [
    ((5, 4, 6), (PERIODIC, DIRICHLET, PERIODIC)),
    ((4, 5, 3), (DIRICHLET, PERIODIC, DIRICHLET)),
    ((3, 3, 7), (PERIODIC, PERIODIC, PERIODIC)),
    ((6, 2, 4), (DIRICHLET, DIRICHLET, DIRICHLET)),
    ((2, 5, 3), (PERIODIC, PERIODIC, DIRICHLET)),   # n = 2 periodic: both neighbours are the same cell
]


@pytest.mark.parametrize("shape,bc", TINY)
def test_recurrence_vs_dense_spectral_closed_form(shape, bc):
    nx, ny, nz = shape
    dx, dt = 0.3, 0.01
    V = random_potential(11, (nz, ny, nx), -3.0, 1.0)
    R0, I0 = random_state(12, (nz, ny, nx))
    o = OracleRun(nx, ny, nz, dx, dt, bc=bc).set_potential_grid(V).set_state(R0, I0)
    n = 300
    o.step(n)
    c, _, _, cv = oracle.coefficients(dx, dt, 1.0, 1.0)
    a, U = np.linalg.eigh(dense_A(nx, ny, nz, bc, c, cv, V))
    assert np.max(np.abs(a)) < 2.0
    r, i = leapfrog_modes(a, U.T @ R0.ravel(), U.T @ I0.ravel(), n)
    assert rel_l2(o.R, U @ r) < 1e-12
    assert rel_l2(o.I, U @ i) < 1e-12


def test_recurrence_vs_fft_closed_form_periodic_free():
    nx, ny, nz = 32, 24, 40
    dx, dt = 0.25, 0.008
    R0, I0 = random_state(5, (nz, ny, nx))
    o = OracleRun(nx, ny, nz, dx, dt, bc=(PERIODIC,) * 3)
    o.set_potential_grid(np.zeros((nz, ny, nx))).set_state(R0, I0)
    n = 200
    o.step(n)
    c = oracle.coefficients(dx, dt, 1.0, 1.0)[0]
    kz, ky, kx = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    a = 4.0 * c * (np.sin(np.pi * kx / nx) ** 2 + np.sin(np.pi * ky / ny) ** 2 + np.sin(np.pi * kz / nz) ** 2)
    theta = 2.0 * np.arcsin(a / 2.0)
    # M^n = (sin n th / sin th) M - (sin (n-1) th / sin th) 1   (Cayley-Hamilton, det M = 1, tr M = 2 cos th)
    with np.errstate(invalid="ignore", divide="ignore"):
        s1 = np.where(theta > 0, np.sin(n * theta) / np.sin(theta), n)
        s0 = np.where(theta > 0, np.sin((n - 1) * theta) / np.sin(theta), n - 1)
    r0h, i0h = np.fft.fftn(R0), np.fft.fftn(I0)
    rh = (s1 * (1 - a ** 2) - s0) * r0h + s1 * a * i0h
    ih = -s1 * a * r0h + (s1 - s0) * i0h
    assert rel_l2(o.R, np.fft.ifftn(rh).real) < 1e-12
    assert rel_l2(o.I, np.fft.ifftn(ih).real) < 1e-12


def test_matches_exact_propagator_second_order_and_staggered_start():
    """R^n ~ Re psi(n dt), I^{n-1/2} ~ Im psi((n-1/2) dt), psi(t) = exp(-i H t/hbar) psi0 (eq 1)."""
    nx, ny, nz = 5, 4, 6
    bc = (PERIODIC, DIRICHLET, DIRICHLET)
    dx = 0.4
    V = random_potential(3, (nz, ny, nx), -2.0, 0.5)
    R0, J0 = random_state(4, (nz, ny, nx))
    errs = []
    t_end = 0.3
    for n in (100, 200, 400):
        dt = t_end / n
        coef = oracle.coefficients(dx, dt, 1.0, 1.0)
        Ih = oracle.stagger(bc, coef, V, R0, J0)
        o = OracleRun(nx, ny, nz, dx, dt, bc=bc).set_potential_grid(V).set_state(R0, Ih)
        o.step(n)
        a, U = np.linalg.eigh(dense_A(nx, ny, nz, bc, coef[0], coef[3], V))   # a = dt * E / hbar
        r0, j0 = U.T @ R0.ravel(), U.T @ J0.ravel()
        re = U @ (r0 * np.cos(a * n) + j0 * np.sin(a * n))
        im = U @ (j0 * np.cos(a * (n - 0.5)) - r0 * np.sin(a * (n - 0.5)))
        errs.append(max(rel_l2(o.R, re), rel_l2(o.I, im)))
    assert errs[0] < 2e-3
    assert 3.6 < errs[0] / errs[1] < 4.4
    assert 3.6 < errs[1] / errs[2] < 4.4


def test_naive_unstaggered_start_is_worse():
    """Guards the sign of the half-step shift: I^{-1/2} = J0 + A R0 / 2, not J0 and not J0 - A R0 / 2."""
    nx, ny, nz = 5, 4, 6
    bc = (PERIODIC, DIRICHLET, DIRICHLET)
    dx, n, t_end = 0.4, 200, 0.3
    dt = t_end / n
    V = random_potential(3, (nz, ny, nx), -2.0, 0.5)
    R0, J0 = random_state(4, (nz, ny, nx))
    coef = oracle.coefficients(dx, dt, 1.0, 1.0)
    a, U = np.linalg.eigh(dense_A(nx, ny, nz, bc, coef[0], coef[3], V))
    r0, j0 = U.T @ R0.ravel(), U.T @ J0.ravel()
    re = U @ (r0 * np.cos(a * n) + j0 * np.sin(a * n))
    Ih = oracle.stagger(bc, coef, V, R0, J0)
    e = {}
    for name, start in (("stagger", Ih), ("naive", J0), ("wrong_sign", 2 * J0 - Ih)):
        o = OracleRun(nx, ny, nz, dx, dt, bc=bc).set_potential_grid(V).set_state(R0, start)
        e[name] = rel_l2(o.step(n).R, re)
    assert e["stagger"] < 0.2 * e["naive"] < 0.2 * e["wrong_sign"] * 2


def test_visscher_norm_conserved_without_mask_and_decays_with_mask():
    nx, ny, nz = 12, 10, 16
    bc = (PERIODIC, PERIODIC, DIRICHLET)
    V = random_potential(7, (nz, ny, nx), -20.0, 0.0)
    R0, I0 = random_state(8, (nz, ny, nx))
    o = OracleRun(nx, ny, nz, 0.2, 0.003, bc=bc).set_potential_grid(V).set_state(R0, I0)
    q0 = o.norm()[0]
    qs = [o.step(50).norm() for _ in range(8)]
    assert max(abs(q[0] - q0) for q in qs) / abs(q0) < 1e-13
    # the paper's density R^2 + I^2 is NOT conserved exactly: it oscillates at O(a)
    assert max(abs(q[1] - qs[0][1]) for q in qs) / abs(q0) > 1e-6
    m = OracleRun(nx, ny, nz, 0.2, 0.003, bc=bc, absorb_lo=4, absorb_hi=4, strength=0.05)
    m.set_potential_grid(np.zeros_like(V)).set_state(R0, I0)
    last = m.norm()[0]
    for _ in range(6):
        q = m.step(20).norm()[0]
        assert q < last
        last = q


def mask_table(nz, w_lo, w_hi, strength, power):
    """M[k] of DESIGN.md reading 6 (forward Euler on the quadratic CAP of eq (10)), written out here
    independently of oracle.mask: xi = fractional depth into the layer, M = 1 - strength * xi^power."""
    M = np.ones(nz)
    for k in range(nz):
        if w_lo > 0 and k < w_lo:
            M[k] = 1.0 - strength * ((w_lo - k) / w_lo) ** power
        if w_hi > 0 and k > nz - 1 - w_hi:
            M[k] = 1.0 - strength * ((k - (nz - 1 - w_hi)) / w_hi) ** power
    return M


ABSORBER_CASES = [
    # shape, bc, absorb_lo, absorb_hi, strength, power
    ((4, 3, 8), (PERIODIC, PERIODIC, DIRICHLET), 3, 2, 0.30, 2),     # both z faces, different widths (cfg 1-4 layout)
    ((3, 5, 7), (PERIODIC, PERIODIC, PERIODIC), 4, 0, 0.25, 2),      # the paper's own set-up: periodic z, one-face CAP
    ((5, 2, 6), (DIRICHLET, PERIODIC, DIRICHLET), 0, 3, 0.40, 3),    # high face only, cubic profile
    ((6, 6, 6), (DIRICHLET, DIRICHLET, PERIODIC), 2, 2, 0.20, 2),    # nx = ny = nz: an M[j]-for-M[k] slip still shows
]


@pytest.mark.parametrize("shape,bc,w_lo,w_hi,strength,power", ABSORBER_CASES)
def test_absorber_inside_the_step_vs_dense_linear_map(shape, bc, w_lo, w_hi, strength, power):
    """Where and how often the mask multiplies (readings 6-7; eq (10)).  One full step is
    the linear map  I' = D_M (I - A R),  R' = D_M (R + A I'),  D_M = diag(M[k]) -- the mask acts on the freshly
    updated field in BOTH half-steps, new = M (old + stencil).  Build that map densely with numpy from the
    independent dense_A and mask_table, raise it to the n-th power, compare with the oracle stepping cell by cell.
    A mask applied in one half-step only, M*old + stencil, or M indexed by the wrong axis each miss by > 1e-3."""
    nx, ny, nz = shape
    N = nx * ny * nz
    dx, dt = 0.3, 0.01
    V = random_potential(31, (nz, ny, nx), -3.0, 1.0)
    R0, I0 = random_state(32, (nz, ny, nx))
    n = 37
    o = OracleRun(nx, ny, nz, dx, dt, bc=bc, absorb_lo=w_lo, absorb_hi=w_hi, strength=strength, power=power)
    o.set_potential_grid(V).set_state(R0, I0).step(n)
    c, _, _, cv = oracle.coefficients(dx, dt, 1.0, 1.0)
    A = dense_A(nx, ny, nz, bc, c, cv, V)
    DM = np.diag(np.repeat(mask_table(nz, w_lo, w_hi, strength, power), ny * nx))   # flat index (k*ny + j)*nx + i
    E, Z = np.eye(N), np.zeros((N, N))
    half_I = np.block([[E, Z], [-DM @ A, DM]])          # (R, I) -> (R, I')      eq (9) then mask
    half_R = np.block([[DM, DM @ A], [Z, E]])           # (R, I') -> (R', I')    eq (8) then mask
    S = np.linalg.matrix_power(half_R @ half_I, n)
    want = S @ np.concatenate([R0.ravel(), I0.ravel()])
    assert rel_l2(o.R, want[:N]) < 1e-12
    assert rel_l2(o.I, want[N:]) < 1e-12
    # the plausible mis-readings really are different maps on this input (so the bound above discriminates)
    alt_one_half = np.linalg.matrix_power(half_R @ np.block([[E, Z], [-A, E]]), n)       # mask in eq (8) only
    alt_old_only = np.linalg.matrix_power(np.block([[DM, A], [Z, E]]) @ np.block([[E, Z], [-A, DM]]), n)   # M*old + stencil
    for alt in (alt_one_half, alt_old_only):
        assert rel_l2((alt @ np.concatenate([R0.ravel(), I0.ravel()]))[:N], want[:N]) > 1e-3


@pytest.mark.parametrize("shape,bc,w_lo,w_hi,strength,power", ABSORBER_CASES)
def test_norms_with_absorber_vs_dense_linear_map(shape, bc, w_lo, w_hi, strength, power):
    """oracle_norm's look-ahead carries the mask (readings 6-7): I^{n+1/2} is what the next
    eq (9) half-step WOULD store, D_M (I - A R), so
        q_visscher = dV ( R.R + (D_M (I - A R)).I ),     q_paper = dV ( R.R + I.I ).
    Built densely from dense_A and mask_table (neither is the oracle's code) on a state that has been stepped into the
    absorber.  Dropping M from the look-ahead, or using it squared, each miss by > 1e-4 on these inputs."""
    nx, ny, nz = shape
    dx, dt = 0.3, 0.01
    V = random_potential(41, (nz, ny, nx), -3.0, 1.0)
    R0, I0 = random_state(42, (nz, ny, nx))
    o = OracleRun(nx, ny, nz, dx, dt, bc=bc, absorb_lo=w_lo, absorb_hi=w_hi, strength=strength, power=power)
    o.set_potential_grid(V).set_state(R0, I0).step(5)
    c, _, _, cv = oracle.coefficients(dx, dt, 1.0, 1.0)
    A = dense_A(nx, ny, nz, bc, c, cv, V)
    m = np.repeat(mask_table(nz, w_lo, w_hi, strength, power), ny * nx)
    R, I = np.asarray(o.R, dtype=np.float64).ravel(), np.asarray(o.I, dtype=np.float64).ravel()
    look = I - A @ R
    dV = dx ** 3
    want_v = dV * (R @ R + (m * look) @ I)
    want_p = dV * (R @ R + I @ I)
    qv, qp = o.norm()
    assert abs(qv - want_v) <= 1e-13 * abs(want_v)
    assert abs(qp - want_p) <= 1e-13 * abs(want_p)
    for alt in (dV * (R @ R + look @ I), dV * (R @ R + (m * m * look) @ I)):     # no mask / mask twice
        assert abs(alt - want_v) > 1e-4 * abs(want_v)


def test_stationary_eigenvector_has_constant_visscher_density():
    nx, ny, nz = 4, 3, 5
    bc = (DIRICHLET, PERIODIC, DIRICHLET)
    dx, dt = 0.5, 0.02
    V = random_potential(21, (nz, ny, nx), -4.0, 0.0)
    c, _, _, cv = oracle.coefficients(dx, dt, 1.0, 1.0)
    a, U = np.linalg.eigh(dense_A(nx, ny, nz, bc, c, cv, V))
    m = 2
    v = U[:, m].reshape(nz, ny, nx)
    o = OracleRun(nx, ny, nz, dx, dt, bc=bc).set_potential_grid(V).set_state(v, 0.5 * a[m] * v)
    expect = v ** 2 * (1.0 - a[m] ** 2 / 4.0)
    for n in (7, 40, 111):
        o.set_state(v, 0.5 * a[m] * v).step(n)
        Rn, Iminus = o.R.copy(), o.I.copy()
        o.step(1)
        Iplus = o.I
        assert np.max(np.abs(Rn * Rn + Iplus * Iminus - expect)) < 1e-14


def test_harmonic_oscillator_ground_state_is_stationary():
    """V = r^2/2 (m = omega = hbar = 1); continuum ground state pi^(-3/4) exp(-r^2/2)."""
    n, dx = 40, 0.3                      # box half-width 5.85 >= 5.8
    ctr = (n - 1) / 2 * dx
    ax = np.arange(n) * dx - ctr
    z, y, x = np.meshgrid(ax, ax, ax, indexing="ij")
    V = 0.5 * (x * x + y * y + z * z)
    dt = 0.008
    o = OracleRun(n, n, n, dx, dt).set_potential_grid(V)
    o.set_wavepacket(ctr, ctr, ctr, 1.0, 0.0, 0.0, 0.0)          # sigma = 1: exp(-r^2/2)
    E0 = 1.5 - 3.0 * dx * dx / 32.0                              # discrete-Laplacian shift of the level
    rho0 = o.R ** 2 + o.I ** 2
    c = n // 2
    r_c0 = o.R[c, c, c]
    worst, phase_err = 0.0, 0.0
    steps_per = 40
    for s in range(1, 14):                                       # ~ one period 2 pi / E0 = 4.2
        o.step(steps_per)
        t = s * steps_per * dt
        rho = o.R ** 2 + o.I ** 2
        worst = max(worst, float(np.max(np.abs(rho - rho0)) / rho0.max()))
        phase_err = max(phase_err, abs(o.R[c, c, c] / r_c0 - math.cos(E0 * t)))
    assert worst < 6e-2
    assert phase_err < 2e-2
    # and a wrong sign of the V term would not be stationary at all
    bad = OracleRun(n, n, n, dx, dt).set_potential_grid(-V)
    bad.set_wavepacket(ctr, ctr, ctr, 1.0, 0.0, 0.0, 0.0)
    bad.step(200)
    assert np.max(np.abs(bad.R ** 2 + bad.I ** 2 - rho0)) / rho0.max() > 0.3


def free_gaussian(x, y, z, t, r0, sigma, k0):
    """Continuum solution of eq (2) with V = 0 (hbar = m = 1) for the packet of eq (3)."""
    tau = t / sigma ** 2
    dx_, dy_, dz_ = x - r0[0] - k0[0] * t, y - r0[1] - k0[1] * t, z - r0[2] - k0[2] * t
    N = (math.pi * sigma ** 2) ** -0.75
    env = N * (1 + 1j * tau) ** -1.5 * np.exp(-(dx_ ** 2 + dy_ ** 2 + dz_ ** 2) / (2 * sigma ** 2 * (1 + 1j * tau)))
    ph = k0[0] * (x - r0[0]) + k0[1] * (y - r0[1]) + k0[2] * (z - r0[2]) - 0.5 * (k0[0] ** 2 + k0[1] ** 2 + k0[2] ** 2) * t
    return env * np.exp(1j * ph)


def _free_gaussian_error(dx, dt, t_end):
    lx, ly, lz = 10.0, 10.0, 12.0
    nx, ny, nz = int(round(lx / dx)), int(round(ly / dx)), int(round(lz / dx))
    r0 = ((nx - 1) / 2 * dx, (ny - 1) / 2 * dx, 5.0)
    k0 = (0.0, 0.5, 2.0)
    o = OracleRun(nx, ny, nz, dx, dt).set_potential_grid(np.zeros((nz, ny, nx)))
    o.set_wavepacket(r0[0], r0[1], r0[2], 1.0, *k0)
    n = int(round(t_end / dt))
    o.step(n)
    z, y, x = np.meshgrid(np.arange(nz) * dx, np.arange(ny) * dx, np.arange(nx) * dx, indexing="ij")
    eR = rel_l2(o.R, free_gaussian(x, y, z, n * dt, r0, 1.0, k0).real)
    eI = rel_l2(o.I, free_gaussian(x, y, z, (n - 0.5) * dt, r0, 1.0, k0).imag)
    # centroid of the density moves toward +z and +y (sign of the phase in eq (3))
    rho = o.R ** 2 + o.I ** 2
    zc = float((rho * z).sum() / rho.sum())
    yc = float((rho * y).sum() / rho.sum())
    return max(eR, eI), zc - r0[2], yc - r0[1]


def test_free_gaussian_spreading_matches_closed_form_second_order_in_dx():
    e1, dz1, dy1 = _free_gaussian_error(0.2, 0.004, 0.5)
    e2, dz2, dy2 = _free_gaussian_error(0.1, 0.001, 0.5)
    assert e1 < 6e-2 and e2 < 1.5e-2
    assert 3.3 < e1 / e2 < 4.7
    # numerical group velocity sin(k dx)/dx (hbar = m = 1)
    assert abs(dz2 - 0.5 * math.sin(2.0 * 0.1) / 0.1) < 5e-3
    assert abs(dy2 - 0.5 * math.sin(0.5 * 0.1) / 0.1) < 5e-3


def test_blow_up_just_past_the_stability_bound():
    """V = 0, periodic, even n: a_max = 12 c exactly, so dt_c = m dx^2 / (3 hbar)."""
    n, dx = 8, 0.2
    dtc = dx * dx / 3.0
    R0, I0 = random_state(99, (n, n, n))
    out = {}
    for f in (0.99, 1.01):
        o = OracleRun(n, n, n, dx, f * dtc, bc=(PERIODIC,) * 3)
        o.set_potential_grid(np.zeros((n, n, n))).set_state(R0, I0).step(400)
        out[f] = float(np.linalg.norm(o.R) / np.linalg.norm(R0))
    assert out[0.99] < 50.0
    assert out[1.01] > 1e20


# ---------------------------------------------------------------------------------------
# potential builder, mask, packet, detector
# ---------------------------------------------------------------------------------------
def test_potential_single_atom_closed_form_superposition_and_clamp():
    nx, ny, nz, dx = 9, 7, 8, 0.4
    bc = (DIRICHLET,) * 3
    a1 = np.array([[1.3, 0.9, 1.7, 3.0, 0.2, 0.7]])
    a2 = np.array([[2.2, 2.0, 0.4, 1.5, 0.05, 0.0]])          # unscreened
    V1 = oracle.potential(nx, ny, nz, dx, bc, a1, -1e9, 1e9)
    V2 = oracle.potential(nx, ny, nz, dx, bc, a2, -1e9, 1e9)
    V12 = oracle.potential(nx, ny, nz, dx, bc, np.concatenate([a1, a2]), -1e9, 1e9)
    z, y, x = np.meshgrid(np.arange(nz) * dx, np.arange(ny) * dx, np.arange(nx) * dx, indexing="ij")
    r = np.sqrt((x - 1.3) ** 2 + (y - 0.9) ** 2 + (z - 1.7) ** 2)
    assert np.allclose(V1, -3.0 * np.exp(-r / 0.7) / np.sqrt(r * r + 0.2), rtol=1e-14, atol=0)
    r = np.sqrt((x - 2.2) ** 2 + (y - 2.0) ** 2 + (z - 0.4) ** 2)
    assert np.allclose(V2, -1.5 / np.sqrt(r * r + 0.05), rtol=1e-14, atol=0)
    assert np.allclose(V12, V1 + V2, rtol=1e-14, atol=0)
    Vc = oracle.potential(nx, ny, nz, dx, bc, np.concatenate([a1, a2]), -2.5, -0.6)
    assert Vc.min() == -2.5 and Vc.max() == -0.6
    assert np.array_equal(Vc, np.clip(V12, -2.5, -0.6))
    assert V12.min() < -2.5 and V12.max() > -0.6


def test_potential_periodic_nearest_image_and_cutoff():
    nx, ny, nz, dx = 10, 8, 6, 0.5
    bc = (PERIODIC, PERIODIC, DIRICHLET)
    a = np.array([[0.3, 3.6, 1.1, 2.0, 0.1, 0.9]])
    V = oracle.potential(nx, ny, nz, dx, bc, a, -1e9, 0.0)
    for sx, sy in ((nx * dx, 0.0), (0.0, -ny * dx), (2 * nx * dx, ny * dx)):
        b = a.copy(); b[0, 0] += sx; b[0, 1] += sy
        assert np.allclose(oracle.potential(nx, ny, nz, dx, bc, b, -1e9, 0.0), V, rtol=1e-12, atol=0)
    # z is Dirichlet: true distance, a shift by Lz changes V
    b = a.copy(); b[0, 2] += nz * dx
    assert not np.allclose(oracle.potential(nx, ny, nz, dx, bc, b, -1e9, 0.0), V, rtol=1e-3)
    # nearest image really is the nearest: brute force over 3x3 images
    z, y, x = np.meshgrid(np.arange(nz) * dx, np.arange(ny) * dx, np.arange(nx) * dx, indexing="ij")
    r2 = np.full(V.shape, np.inf)
    for ix in (-1, 0, 1):
        for iy in (-1, 0, 1):
            r2 = np.minimum(r2, (x - 0.3 - ix * nx * dx) ** 2 + (y - 3.6 - iy * ny * dx) ** 2 + (z - 1.1) ** 2)
    assert np.allclose(V, -2.0 * np.exp(-np.sqrt(r2) / 0.9) / np.sqrt(r2 + 0.1), rtol=1e-13, atol=0)
    Vcut = oracle.potential(nx, ny, nz, dx, bc, a, -1e9, 0.0, rcut=1.5)
    assert np.array_equal(Vcut != 0.0, np.sqrt(r2) <= 1.5)
    assert np.array_equal(Vcut[Vcut != 0.0], V[Vcut != 0.0])


def test_config0_potential_value_next_to_the_centre():
    w = make_config(0)
    V = oracle.potential(w.nx, w.ny, w.nz, w.dx, w.bc, w.atoms[0], w.vmin, w.vmax)
    # the atom sits between grid points: the 8 nearest points are at (0.1, 0.1, 0.1) from it
    assert abs(V[31, 31, 31] - (-1.0 / math.sqrt(3 * 0.1 ** 2 + 0.5))) < 1e-14
    assert abs(V[32, 31, 32] - V[31, 31, 31]) < 1e-14
    assert V.min() >= -50.0 and V.max() <= 0.0
    assert abs(w.dt - 0.5 / (6.0 / 0.04 + 1.0 / math.sqrt(0.5))) < 1e-18
    assert abs(w.dt - 3.3022e-3) < 1e-7


def test_mask_invariants():
    M = oracle.mask(64, 16, 24, 0.05, 2)
    assert np.all(M[16:64 - 24] == 1.0)
    assert M[0] == 1.0 - 0.05 and M[63] == 1.0 - 0.05
    assert np.all(np.diff(M[:17]) > 0) and np.all(np.diff(M[39:]) < 0)
    assert abs(M[8] - (1 - 0.05 * 0.25)) < 1e-16           # xi = 1/2, quadratic
    assert abs(oracle.mask(64, 16, 24, 0.05, 3)[8] - (1 - 0.05 * 0.125)) < 1e-16
    assert np.all(oracle.mask(10, 0, 0) == 1.0)


def test_wavepacket_normalisation_direction_and_envelope():
    n, dx, s = 48, 0.25, 1.0
    ctr = (n - 1) / 2 * dx
    R0, J0 = oracle.wavepacket(n, n, n, dx, ctr, ctr, ctr, s, 0.0, 0.0, 1.7)
    assert abs((R0 ** 2 + J0 ** 2).sum() * dx ** 3 - 1.0) < 1e-6          # N = (pi s^2)^(-3/4)
    # envelope exp(-r^2 / 2 s^2) on psi: |psi|^2 has variance s^2/2 per axis
    z = np.arange(n) * dx - ctr
    rho_z = (R0 ** 2 + J0 ** 2).sum(axis=(1, 2))
    assert abs((rho_z * z * z).sum() / rho_z.sum() - 0.5 * s * s) < 1e-4
    # phase advances along +z for kz > 0: psi(z+dz)/psi(z) has argument +kz*dz
    c = n // 2
    ratio = (R0[c + 1, c, c] + 1j * J0[c + 1, c, c]) / (R0[c, c, c] + 1j * J0[c, c, c])
    assert abs(np.angle(ratio) - 1.7 * dx) < 1e-12
    Ra, Ja = oracle.wavepacket(n, n, n, dx, ctr, ctr, ctr, s, 0.0, 0.0, 1.7, amplitude=2.0)
    assert abs(np.hypot(Ra, Ja).max() - 2.0 * math.exp(-3 * (dx / 2) ** 2 / 2)) < 1e-12


def test_detector_identities():
    w = make_config(0, n=(20, 18, 24), steps=60)
    o = OracleRun.from_workload(w)
    o.set_detector(5, 10)
    imgs = []
    for _ in range(6):
        o.step(10)
        imgs.append(o.R[5] ** 2 + o.I[5] ** 2)
    assert len(o.trace) == 6
    assert np.allclose(o.D, np.sum(imgs, axis=0), rtol=1e-14, atol=0)
    assert np.allclose(o.trace, [im.sum() * w.dx ** 2 for im in imgs], rtol=1e-13, atol=0)
    assert abs(o.D.sum() - sum(o.trace) / w.dx ** 2) / o.D.sum() < 1e-13
    # counter is global: 7 + 3 steps samples once, at step 10
    p = OracleRun.from_workload(w)
    p.set_detector(5, 10)
    p.step(7); assert len(p.trace) == 0
    p.step(3); assert len(p.trace) == 1 and abs(p.trace[0] - o.trace[0]) < 1e-15


def test_f32_instantiation_tracks_f64():
    w = make_config(1, n=(24, 24, 32), steps=300)
    o64 = OracleRun.from_workload(w, dtype="f64", round_to="f32").step(300)
    o32 = OracleRun.from_workload(w, dtype="f32").step(300)
    assert o32.R.dtype == np.float32
    assert rel_l2(o32.R, o64.R) < 2e-5 and rel_l2(o32.I, o64.I) < 2e-5
    assert rel_l2(o32.D, o64.D) < 2e-5


def test_openmp_is_bit_identical_to_serial():
    w = make_config(1, n=(16, 20, 24), steps=40)
    oracle.set_threads(1)
    a = OracleRun.from_workload(w).step(40)
    oracle.set_threads(max(2, min(4, oracle.max_threads())))
    b = OracleRun.from_workload(w).step(40)
    oracle.set_threads(oracle.max_threads())
    assert np.array_equal(a.R, b.R) and np.array_equal(a.I, b.I) and np.array_equal(a.D, b.D)


# ---------------------------------------------------------------------------------------
# values printed in the paper
# ---------------------------------------------------------------------------------------
def test_paper_time_step_and_coefficients():
    g = json.load(open(os.path.join(GOLDEN, "paper_values.json")))
    si = g["si_constants"]
    ts = g["time_step_attoseconds"]
    spac = [L * 1e-10 / n for L, n in zip(ts["domain_angstrom"], ts["mesh"])]
    dt = oracle.paper_time_step(*spac, si["electron_mass_kg"], si["hbar_Js"])
    assert round(dt / 1e-18, ts["printed_digits"]) == ts["value"]              # 0.38 as
    # the other printed domain (40.9 A in x) would NOT give 0.38 as
    alt = oracle.paper_time_step(40.9e-10 / 240, 40.9e-10 / 240, 70e-10 / 420, si["electron_mass_kg"], si["hbar_Js"])
    assert round(alt / 1e-18, 2) != ts["value"]
    # eq (11) makes the coefficient of PAPER.md:87 exactly 1/10 on the finest axis
    cx, cy, cz, cv = oracle.coefficients(spac[0], dt, si["electron_mass_kg"], si["hbar_Js"], spac[1], spac[2])
    assert abs(cx - 0.1) < 1e-15 and cy < cx and cz < cx
    assert abs(cv - dt / si["hbar_Js"]) == 0.0
    # eq (4) is the de Broglie wavelength: 12.2643 / sqrt(E[eV]) Angstrom (textbook constant)
    lam = oracle.paper_wavelength(60.0 * si["eV_J"], si["electron_mass_kg"], si["hbar_Js"])
    assert abs(lam / 1e-10 - si["de_broglie_angstrom_sqrt_eV"] / math.sqrt(60.0)) < 2e-5
    assert 140 * 140 * (420 + g["cap_planes"]["value"]) == g["mesh_points_small"]["value"]


# ---------------------------------------------------------------------------------------
# frame-mode detector and trajectory dissimilarity (eq 16)
# ---------------------------------------------------------------------------------------
def test_frames_against_fft_closed_form_and_accumulated_image():
    """Frames are (R^s)^2 + (I^{s-1/2})^2 on the plane at s = 0, h, 2h, ...: pinned with the discrete-exact
    Fourier solution of the free periodic recurrence (independent of the oracle), and with the identities
    sum_{s>=1} frame_s = accumulated image, trace_s = dx^2 sum(frame_s)."""
    nx, ny, nz = 16, 12, 20
    dx, dt, h, k_det = 0.25, 0.008, 7, 5
    R0, I0 = random_state(11, (nz, ny, nx))
    o = OracleRun(nx, ny, nz, dx, dt, bc=(PERIODIC,) * 3)
    o.set_potential_grid(np.zeros((nz, ny, nx))).set_state(R0, I0).set_detector(k_det, h).set_frames(True, True)
    o.step(10).step(20)          # split across calls, not aligned with h
    assert len(o.frames) == 1 + 30 // h
    c = oracle.coefficients(dx, dt, 1.0, 1.0)[0]
    kz, ky, kx = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    a = 4.0 * c * (np.sin(np.pi * kx / nx) ** 2 + np.sin(np.pi * ky / ny) ** 2 + np.sin(np.pi * kz / nz) ** 2)
    theta = 2.0 * np.arcsin(a / 2.0)
    r0h, i0h = np.fft.fftn(R0), np.fft.fftn(I0)
    for f, n in enumerate(range(0, 31, h)):
        if n == 0:
            R, I = R0, I0
        else:
            with np.errstate(invalid="ignore", divide="ignore"):
                s1 = np.where(theta > 0, np.sin(n * theta) / np.sin(theta), n)
                s0 = np.where(theta > 0, np.sin((n - 1) * theta) / np.sin(theta), n - 1)
            R = np.fft.ifftn((s1 * (1 - a ** 2) - s0) * r0h + s1 * a * i0h).real
            I = np.fft.ifftn(-s1 * a * r0h + (s1 - s0) * i0h).real
        assert rel_l2(o.frames[f], R[k_det] ** 2 + I[k_det] ** 2) < 1e-12
    assert rel_l2(sum(o.frames[1:]), o.D) < 1e-15
    assert np.allclose([dx * dx * f.sum() for f in o.frames[1:]], o.trace, rtol=1e-14)
    # without the t = 0 frame the list starts at s = h
    p = OracleRun(nx, ny, nz, dx, dt, bc=(PERIODIC,) * 3)
    p.set_potential_grid(np.zeros((nz, ny, nx))).set_state(R0, I0).set_detector(k_det, h).set_frames(True, False).step(30)
    assert len(p.frames) == 30 // h and np.array_equal(p.frames[0], o.frames[1])


def test_dissimilarity_closed_forms_and_metric_properties():
    """eq (16): closed forms that do not go through the oracle -- proportional trajectories, disjoint supports,
    shifted Gaussians on a fine plane -- and the metric axioms (identity, symmetry, triangle inequality)."""
    rng = np.random.default_rng(3)
    ns, ny, nx, dA = 9, 10, 14, 0.15 ** 2
    pattern = rng.random((ny, nx))
    a, b = rng.random(ns) + 0.5, rng.random(ns) + 0.5
    fa, fb = a[:, None, None] * pattern, b[:, None, None] * pattern
    s0, s1 = 2, 7
    # proportional frames: d = mean_s |a_s - b_s| * sqrt(dA * sum(pattern^2))
    want = np.mean(np.abs(a - b)[s0:s1 + 1]) * math.sqrt(dA * float((pattern ** 2).sum()))
    assert abs(oracle.dissimilarity(fa, fb, dA, s0, s1) - want) < 1e-14 * want
    # disjoint supports: the cross term vanishes, d = mean_s sqrt(dA (|rho_k|^2 + |rho_j|^2))
    left, right = np.zeros((ns, ny, nx)), np.zeros((ns, ny, nx))
    left[:, :, : nx // 2] = rng.random((ns, ny, nx // 2))
    right[:, :, nx // 2:] = rng.random((ns, ny, nx - nx // 2))
    want = np.mean([math.sqrt(dA * float((left[s] ** 2).sum() + (right[s] ** 2).sum())) for s in range(s0, s1 + 1)])
    assert abs(oracle.dissimilarity(left, right, dA, s0, s1) - want) < 1e-14 * want
    # two unit Gaussians of width w a distance delta apart (continuum closed form below)
    n, L, w, delta = 256, 16.0, 1.0, 1.3
    x = (np.arange(n) + 0.5) * L / n
    X, Y = np.meshgrid(x, x)
    g1 = np.exp(-((X - 8.0) ** 2 + (Y - 8.0) ** 2) / (2 * w * w))
    g2 = np.exp(-((X - 8.0 - delta) ** 2 + (Y - 8.0) ** 2) / (2 * w * w))
    # int g1^2 = pi w^2, int g1 g2 = pi w^2 exp(-delta^2/(4 w^2))  =>  int (g1-g2)^2 = 2 pi w^2 (1 - exp(-delta^2/(4 w^2)))
    want = math.sqrt(2.0 * math.pi * w * w * (1.0 - math.exp(-delta * delta / (4 * w * w))))
    got = oracle.dissimilarity(g1[None], g2[None], (L / n) ** 2, 0, 0)
    assert abs(got - want) < 1e-10 * want      # the trapezoid-like sum of a smooth, decayed integrand is spectrally accurate
    # metric axioms on random trajectories
    t = [rng.random((ns, ny, nx)) for _ in range(3)]
    d = lambda p, q: oracle.dissimilarity(t[p], t[q], dA, 0, ns - 1)
    assert d(0, 0) == 0.0 and d(0, 1) == d(1, 0) and d(0, 2) <= d(0, 1) + d(1, 2)
    # scaling: rho -> alpha rho scales d by alpha
    assert abs(oracle.dissimilarity(3.0 * t[0], 3.0 * t[1], dA, 0, ns - 1) - 3.0 * d(0, 1)) < 1e-13


# ---------------------------------------------------------------------------------------
# anisotropic mesh (c_x != c_y != c_z; the paper's own mesh is 35.4/240 x 40.9/240 x 70/420 A)
# ---------------------------------------------------------------------------------------
def test_anisotropic_recurrence_vs_dense_and_fft_closed_forms():
    # tiny mixed-BC grid: dense A with one coefficient per axis, built here with numpy
    nx, ny, nz = 5, 4, 6
    bc = (PERIODIC, DIRICHLET, PERIODIC)
    dx, dy, dz, dt = 0.4, 0.3, 0.55, 0.004
    V = random_potential(21, (nz, ny, nx), -3.0, 1.0)
    R0, I0 = random_state(22, (nz, ny, nx))
    o = OracleRun(nx, ny, nz, dx, dt, bc=bc, dy=dy, dz=dz).set_potential_grid(V).set_state(R0, I0)
    n = 150
    o.step(n)
    cx, cy, cz, cv = oracle.coefficients(dx, dt, 1.0, 1.0, dy, dz)
    assert cx != cy != cz
    Ix, Iy, Iz = np.eye(nx), np.eye(ny), np.eye(nz)
    A = (-cz * np.kron(np.kron(d2_matrix(nz, bc[2]), Iy), Ix) - cy * np.kron(np.kron(Iz, d2_matrix(ny, bc[1])), Ix)
         - cx * np.kron(np.kron(Iz, Iy), d2_matrix(nx, bc[0])) + cv * np.diag(V.ravel()))
    a, U = np.linalg.eigh(A)
    r, i = leapfrog_modes(a, U.T @ R0.ravel(), U.T @ I0.ravel(), n)
    assert rel_l2(o.R, U @ r) < 1e-12 and rel_l2(o.I, U @ i) < 1e-12
    # medium periodic free grid: Fourier symbol a = sum_d 4 c_d sin^2(pi kappa_d / n_d)
    nx, ny, nz = 16, 12, 20
    R0, I0 = random_state(23, (nz, ny, nx))
    o = OracleRun(nx, ny, nz, dx, dt, bc=(PERIODIC,) * 3, dy=dy, dz=dz)
    o.set_potential_grid(np.zeros((nz, ny, nx))).set_state(R0, I0).set_detector(3, 10)
    n = 120
    o.step(n)
    kz, ky, kx = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    a = 4.0 * (cx * np.sin(np.pi * kx / nx) ** 2 + cy * np.sin(np.pi * ky / ny) ** 2 + cz * np.sin(np.pi * kz / nz) ** 2)
    theta = 2.0 * np.arcsin(a / 2.0)
    with np.errstate(invalid="ignore", divide="ignore"):
        s1 = np.where(theta > 0, np.sin(n * theta) / np.sin(theta), n)
        s0 = np.where(theta > 0, np.sin((n - 1) * theta) / np.sin(theta), n - 1)
    r0h, i0h = np.fft.fftn(R0), np.fft.fftn(I0)
    R = np.fft.ifftn((s1 * (1 - a ** 2) - s0) * r0h + s1 * a * i0h).real
    I = np.fft.ifftn(-s1 * a * r0h + (s1 - s0) * i0h).real
    assert rel_l2(o.R, R) < 1e-12 and rel_l2(o.I, I) < 1e-12
    # the trace carries the plane's area element dx*dy, the norms the volume element dx*dy*dz
    assert abs(o.trace[-1] - dx * dy * float((R[3] ** 2 + I[3] ** 2).sum())) < 1e-12 * o.trace[-1]
    qv, qp = o.norm()
    assert abs(qp - dx * dy * dz * float((R ** 2 + I ** 2).sum())) < 1e-12 * qp


def test_anisotropic_potential_and_packet_closed_forms():
    nx, ny, nz, dx, dy, dz = 12, 10, 14, 0.3, 0.2, 0.45
    atom = np.array([[1.1, 0.7, 2.9, 3.0, 0.2, 0.8]])
    V = oracle.potential(nx, ny, nz, dx, (DIRICHLET,) * 3, atom, -1e9, 0.0, dy=dy, dz=dz)
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    r = np.sqrt((i * dx - 1.1) ** 2 + (j * dy - 0.7) ** 2 + (k * dz - 2.9) ** 2)
    assert np.allclose(V, -3.0 * np.exp(-r / 0.8) / np.sqrt(r * r + 0.2), rtol=1e-13)
    # nearest image uses the box lengths n_d * d_d of each axis
    Vp = oracle.potential(nx, ny, nz, dx, (PERIODIC,) * 3, atom, -1e9, 0.0, dy=dy, dz=dz)
    shifted = atom + np.array([[nx * dx, -ny * dy, 2 * nz * dz, 0, 0, 0]])
    assert np.allclose(Vp, oracle.potential(nx, ny, nz, dx, (PERIODIC,) * 3, shifted, -1e9, 0.0, dy=dy, dz=dz), rtol=1e-12)
    R0, J0 = oracle.wavepacket(nx, ny, nz, dx, 1.5, 1.0, 3.0, 0.9, 0.3, -0.4, 1.1, 2.0, dy=dy, dz=dz)
    G = 2.0 * np.exp(-((i * dx - 1.5) ** 2 + (j * dy - 1.0) ** 2 + (k * dz - 3.0) ** 2) / (2 * 0.81))
    phi = 0.3 * (i * dx - 1.5) - 0.4 * (j * dy - 1.0) + 1.1 * (k * dz - 3.0)
    assert np.allclose(R0, G * np.cos(phi), atol=1e-14) and np.allclose(J0, G * np.sin(phi), atol=1e-14)


# ---------------------------------------------------------------------------------------
# unit-cell potential tiled and interpolated onto the mesh (reading 24)
# ---------------------------------------------------------------------------------------
def test_potential_cell_interpolation_closed_forms():
    mx, my, mz, ax, ay, az = 6, 5, 7, 1.8, 2.0, 3.0
    hx, hy, hz = ax / mx, ay / my, az / (mz - 1)
    kk, jj, ii = np.meshgrid(np.arange(mz), np.arange(my), np.arange(mx), indexing="ij")
    nx, ny, nz, dx, dy, dz = 20, 18, 16, 0.17, 0.23, 0.21
    org = (0.05, -0.3, 0.4)
    K, J, I = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    X, Y, Z = I * dx - org[0], J * dy - org[1], K * dz - org[2]
    big = 1e30
    # (a) a cell that is linear in z only is reproduced exactly, with the nearest plane beyond the cell
    V = oracle.potential_cell(nx, ny, nz, dx, 2.0 + 0.5 * kk * hz, (ax, ay, az), org, -big, big, dy, dz)
    assert np.allclose(V, 2.0 + 0.5 * np.clip(Z, 0.0, az), rtol=0, atol=1e-13)
    # (b) a periodic function sampled on a fine cell: the error obeys the linear-interpolation bound h^2 max|f''|/8
    #     per axis, and the result is exactly periodic in x, y
    f = lambda x, y, z: np.cos(2 * np.pi * x / ax) * np.sin(2 * np.pi * y / ay) * (1.0 + 0.3 * z)
    fine = 8
    kk2, jj2, ii2 = np.meshgrid(np.arange(mz), np.arange(my * fine), np.arange(mx * fine), indexing="ij")
    cell = f(ii2 * hx / fine, jj2 * hy / fine, kk2 * hz)
    V = oracle.potential_cell(nx, ny, nz, dx, cell, (ax, ay, az), org, -big, big, dy, dz)
    want = f(X, Y, np.clip(Z, 0.0, az))
    h2 = max((hx / fine) ** 2 * (2 * np.pi / ax) ** 2, (hy / fine) ** 2 * (2 * np.pi / ay) ** 2) / 8.0 * 2.0
    assert np.max(np.abs(V - want)) <= 1.3 * (1.0 + 0.3 * az) * h2      # interpolation error bound of linear interpolation
    shifted = oracle.potential_cell(nx, ny, nz, dx, cell, (ax, ay, az), (org[0] + 3 * ax, org[1] - 2 * ay, org[2]), -big, big, dy, dz)
    assert np.allclose(V, shifted, rtol=0, atol=1e-12)
    # (c) at mesh points that coincide with cell nodes the node value comes back; a constant cell stays constant; clamp
    Vn = oracle.potential_cell(mx * 2, my * 2, mz, hx, np.arange(mz * my * mx, dtype=float).reshape(mz, my, mx),
                               (ax, ay, az), (0.0, 0.0, 0.0), -big, big, hy, hz)
    assert np.allclose(Vn[:, :my, :mx], np.arange(mz * my * mx).reshape(mz, my, mx), atol=1e-9)
    assert np.allclose(Vn[:, my:, mx:], Vn[:, :my, :mx], atol=1e-9)                      # the supercell repeats
    Vc = oracle.potential_cell(nx, ny, nz, dx, np.full((mz, my, mx), -3.5), (ax, ay, az), org, -2.0, 0.0, dy, dz)
    assert np.all(Vc == -2.0)
