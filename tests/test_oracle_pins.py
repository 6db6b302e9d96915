"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: every expected value is a closed form, an
invariant, a brute-force recomputation written differently (numpy all-pairs), or the paper's worked example.
"""
import numpy as np
import pytest

from conftest import golden
from lsm_inputs import FIXED, MOVE, config1, triangular_lattice, two_phase_spring_params, blob_image
from lsm_inputs.generators import SQ3_2
from oracle.olsm import OracleSim


def _two_particles(x1, k, r0, rc, dt, gamma=0.0, m=1.0, fix0=True, sample_every=0):
    x = np.array([[0.0, 0.0], [x1, 0.0]])
    s = OracleSim(x, [0], [1], [k], [r0], [rc], dt, gamma, mass=m, sample_every=sample_every)
    if fix0:
        s.set_boundary(0, [0], FIXED)
    return s


def test_P1_paper_oscillator_example():
    """fixed end + free end, closed-form Verlet trajectory and analytic ODE solution."""
    g = golden("paper_sho_example.txt")
    s = _two_particles(g["x0"], g["k"], g["r0"], 100.0, g["dt"], m=g["m"])
    th = np.arccos(1.0 - g["k"] * g["dt"] ** 2 / (2.0 * g["m"]))
    w = np.sqrt(g["k"] / g["m"])
    err_cf, err_an = 0.0, 0.0
    for n in range(1, int(g["n_steps"]) + 1):
        s.step(1)
        x, v = s.read_state()
        assert x[0, 0] == 0.0 and x[0, 1] == 0.0 and x[1, 1] == 0.0
        amp = g["x0"] - g["r0"]
        err_cf = max(err_cf, abs(x[1, 0] - (g["r0"] + amp * np.cos(n * th))))
        if n % int(g["output_every"]) == 0:
            err_an = max(err_an, abs(x[1, 0] - (g["r0"] + amp * np.cos(w * n * g["dt"]))))
    assert err_cf <= 1e-11
    assert err_an <= 2e-4            # "accurate ... without error accumulation" (L127)
    assert abs(x[1, 0] - 5.804755697) < 1e-8


def test_P1_velocity_closed_form():
    """Full-step velocity of velocity Verlet on a linear spring: v_n = -(A sin(theta)/dt) sin(n theta)."""
    k, r0, dt = 1e-4, 10.0, 1.0
    s = _two_particles(15.0, k, r0, 100.0, dt)
    th = np.arccos(1.0 - k * dt * dt / 2.0)
    for n in range(1, 400):
        s.step(1)
        _, v = s.read_state()
        assert abs(v[1, 0] + 5.0 * np.sin(th) / dt * np.sin(n * th)) < 1e-12


def test_P2_two_free_particles_reduced_mass():
    """Period 2 pi sqrt(m_red/k) (north_star closed form): separation = r0 + A cos(n theta2), COM at rest."""
    k, r0, dt, m = 1e-4, 10.0, 1.0, 1.0
    s = _two_particles(15.0, k, r0, 100.0, dt, fix0=False, m=m)
    mred = m / 2.0
    th2 = np.arccos(1.0 - (k / mred) * dt * dt / 2.0)
    assert abs(2 * np.pi / th2 * dt - 2 * np.pi * np.sqrt(mred / k)) < 2e-3 * 444.288   # discrete vs continuous period
    for n in range(1, 1001):
        s.step(1)
        x, v = s.read_state()
        assert abs((x[1, 0] - x[0, 0]) - (r0 + 5.0 * np.cos(n * th2))) <= 1e-11
        assert abs(0.5 * (x[1, 0] + x[0, 0]) - 7.5) <= 1e-12
        assert abs(v[0, 0] + v[1, 0]) <= 1e-15


@pytest.mark.parametrize("eps", [1e-3, 1e-5])
def test_P3_affine_uniaxial_stress_state(eps):
    """Young's modulus 2k/sqrt(3) and Poisson's ratio 1/3 of the triangular lattice (north_star), exact finite-strain
    forms: under x -> x(1-eps/3), y -> y(1+eps) interior forces vanish and each interior top-row particle carries
    f_y = -2 k (L - r0)/L * (sqrt3/2)(1+eps) r0 with L = r0 sqrt((1-eps/3)^2/4 + 3(1+eps)^2/4)."""
    nx = ny = 64
    kk = 1.7
    x, si, sj, site, kind = triangular_lattice(nx, ny)
    xa = x * np.array([1.0 - eps / 3.0, 1.0 + eps])
    M = si.size
    s = OracleSim(xa, si, sj, np.full(M, kk), np.ones(M), np.full(M, 2.0), 0.01)
    f = s.read_forces()
    row, col = site // nx, site % nx
    interior = (row > 0) & (row < ny - 1) & (col > 0) & (col < nx - 1)
    L = np.sqrt((1 - eps / 3) ** 2 / 4 + 3 * (1 + eps) ** 2 / 4)
    fmag_d = kk * (L - 1.0)          # force magnitude of one diagonal spring
    # Poisson's ratio 1/3: lateral contraction eps/3 leaves interior particles force-free to first order; the exact
    # residual is second order in eps and cancels by symmetry -> zero to rounding
    # (rounding: coordinates up to 64 carry ulp 1.4e-14, so differences carry that absolute error times k)
    assert np.abs(f[interior]).max() <= 8 * np.finfo(float).eps * np.abs(xa).max() * kk < 1e-7 * fmag_d
    top_int = (row == ny - 1) & (col > 0) & (col < nx - 1)
    fy_expect = -2.0 * fmag_d / L * SQ3_2 * (1 + eps)
    assert np.allclose(f[top_int, 1], fy_expect, rtol=1e-9 / max(eps / 1e-5, 1), atol=0)
    # E = 2k/sqrt3 per unit thickness: stress per unit width / strain -> 2k/sqrt3 as eps -> 0
    E_lat = -fy_expect / eps
    assert abs(E_lat / (2 * kk / np.sqrt(3)) - 1) < 2 * eps
    # energy (Eq. 1): n_h horizontal springs stretched by -eps/3, n_d diagonal springs of length L
    n_h, n_d = ny * (nx - 1), (ny - 1) * (2 * nx - 1)
    assert (kind == 0).sum() == n_h and (kind != 0).sum() == n_d
    U, _ = s.read_energy()
    U_expect = 0.5 * kk * (n_h * (eps / 3) ** 2 + n_d * (L - 1.0) ** 2)
    assert abs(U[0] / U_expect - 1) < 1e-9


def _random_state(nx, ny, seed, amp=0.05):
    x, si, sj, site, kind = triangular_lattice(nx, ny)
    rng = np.random.default_rng(seed)
    x = x + rng.uniform(-amp, amp, x.shape)
    M = si.size
    k = rng.uniform(0.5, 2.0, M)
    r0 = rng.uniform(0.9, 1.1, M)
    return x, si, sj, k, r0


def test_P4_zero_net_force_and_torque():
    x, si, sj, k, r0 = _random_state(24, 20, 1)
    s = OracleSim(x, si, sj, k, r0, np.full(si.size, 5.0), 0.01)
    f = s.read_forces()
    # scale: sum of |contributions|
    d = x[sj] - x[si]
    r = np.linalg.norm(d, axis=1)
    scale = 2 * np.sum(np.abs(k * (r - r0)))
    assert np.abs(f.sum(axis=0)).max() <= 1e-13 * scale
    torque = np.sum(x[:, 0] * f[:, 1] - x[:, 1] * f[:, 0])
    assert abs(torque) <= 1e-13 * scale * np.abs(x).max()


@pytest.mark.parametrize("nx,ny", [(4, 3), (8, 8), (5, 7)])
def test_P5_brute_force_all_pairs(nx, ny):
    """O(N^2) recomputation: every particle pair whose INITIAL distance is r0 (within 1e-9) is a spring."""
    x0, si, sj, _, _ = triangular_lattice(nx, ny)
    N = x0.shape[0]
    rng = np.random.default_rng(nx * 100 + ny)
    x = x0 + rng.uniform(-0.08, 0.08, x0.shape)
    kk = 1.3
    s = OracleSim(x, si, sj, np.full(si.size, kk), np.ones(si.size), np.full(si.size, 9.0), 0.01)
    f = s.read_forces()
    fb = np.zeros_like(x)
    npairs = 0
    for a in range(N):
        for b in range(N):
            if a == b or abs(np.hypot(*(x0[a] - x0[b])) - 1.0) > 1e-9:
                continue
            npairs += 1
            rab = np.hypot(*(x[a] - x[b]))
            fb[a] += -kk * (rab - 1.0) * (x[a] - x[b]) / rab      # Eq. 2 as printed (L55)
    assert npairs == 2 * si.size
    assert np.abs(f - fb).max() <= 1e-14


def test_P6_energy_conservation_and_scaling():
    """gamma=0, grips FIXED, 1 % affine pre-stretch released: |dE/E0| < 1e-8 over 10^4 steps at dt = 1e-3;
    fluctuation scales as dt^2 (halving dt divides it by 4)."""
    nx = ny = 32
    x, si, sj, site, _ = triangular_lattice(nx, ny)
    row = site // nx
    M = si.size
    xa = x * np.array([1.0, 1.01])
    def run(dt, nsteps, every):
        s = OracleSim(xa, si, sj, np.ones(M), np.ones(M), np.full(M, 2.0), dt)
        s.set_boundary(0, np.flatnonzero(row == 0), FIXED)
        s.set_boundary(1, np.flatnonzero(row == ny - 1), FIXED)
        U, KE = s.read_energy(); E0 = U[0] + KE[0]; dev = 0.0
        for _ in range(nsteps // every):
            s.step(every)
            U, KE = s.read_energy()
            dev = max(dev, abs(U[0] + KE[0] - E0) / E0)
        return dev
    d1 = run(1e-3, 10000, 100)
    assert d1 < 1e-8
    d_a, d_b = run(0.02, 2000, 10), run(0.01, 4000, 20)
    assert 3.6 < d_a / d_b < 4.4


def test_P6_momentum_conservation_free_lattice():
    x, si, sj, k, r0 = _random_state(16, 16, 7)
    rng = np.random.default_rng(3)
    v = rng.normal(0, 0.01, x.shape)
    s = OracleSim(x, si, sj, k, r0, np.full(si.size, 9.0), 0.01, v=v)
    p0 = v.sum(axis=0)
    s.step(2000)
    _, v1 = s.read_state()
    assert np.abs(v1.sum(axis=0) - p0).max() <= 1e-13


def test_P7_strict_greater_than_dyadic():
    """Q1: r == rc exactly survives; all numbers dyadic so every operation is exact."""
    x = np.array([[0.0, 0.0], [1.0, 0.0]])
    s = OracleSim(x, [0], [1], [1.0], [1.0], [1.0 + 2.0 ** -3], 1.0)
    s.set_boundary(0, [0], FIXED)
    s.set_boundary(1, [1], MOVE, [2.0 ** -10, 0.0])
    s.step(128)
    xx, _ = s.read_state()
    assert xx[1, 0] == 1.125
    b, bs, nb = s.read_broken()
    assert nb == 0 and not b[0] and bs[0] == -1
    assert s.read_forces()[1, 0] == -0.125 / 1.125 * 1.125       # -k (r - r0) (x1-x0)/r
    s.step(1)
    b, bs, nb = s.read_broken()
    assert nb == 1 and b[0] and bs[0] == 129
    assert np.all(s.read_forces() == 0.0)


def test_P8_irreversible_breakage():
    """Q2/Q3/Q18: once broken, force and energy stay zero even when r drops below rc again."""
    x = np.array([[0.0, 0.0], [1.0, 0.0]])
    s = OracleSim(x, [0], [1], [1.0], [1.0], [1.25], 1.0, sample_every=1)
    s.set_boundary(0, [0], FIXED)
    s.set_boundary(1, [1], MOVE, [0.0625, 0.0])
    s.step(6)                                  # r = 1.375 > 1.25 -> broke at step 5 (1.3125)
    b, bs, nb = s.read_broken()
    assert nb == 1 and bs[0] == 5
    s.set_boundary(1, [1], MOVE, [-0.0625, 0.0])
    s.step(6)                                  # back to r = 1.0
    xx, _ = s.read_state()
    assert xx[1, 0] == 1.0
    assert np.all(s.read_forces() == 0.0)
    U, _ = s.read_energy()
    assert U[0] == 0.0
    h = s.read_stress()
    assert list(h["n_broken"][:, 0]) == [0, 0, 0, 0, 1, 1, 1, 1, 1, 1, 1, 1]
    assert np.all(h["U"][4:, 0] == 0.0) and h["U"][3, 0] == 0.5 * 0.25 ** 2


def test_P9_time_reversibility():
    """PAPER.md:L76 claims time reversibility: n steps, v -> -v, n steps returns to the start."""
    x, si, sj, k, r0 = _random_state(16, 16, 11, amp=0.03)
    s = OracleSim(x, si, sj, k, r0, np.full(si.size, 9.0), 0.01)
    s.step(1000)
    x1, v1 = s.read_state()
    s2 = OracleSim(x1, si, sj, k, r0, np.full(si.size, 9.0), 0.01, v=-v1)
    s2.step(1000)
    x2, v2 = s2.read_state()
    assert np.abs(x2 - x).max() <= 1e-10
    assert np.abs(v2).max() <= 1e-10


def test_P10_force_is_minus_grad_U():
    x, si, sj, k, r0 = _random_state(8, 8, 5)
    rc = np.full(si.size, 9.0)
    f = OracleSim(x, si, sj, k, r0, rc, 0.01).read_forces()
    h = 1e-6
    rng = np.random.default_rng(0)
    for _ in range(24):
        p, c = rng.integers(x.shape[0]), rng.integers(2)
        xp, xm = x.copy(), x.copy()
        xp[p, c] += h; xm[p, c] -= h
        Up = OracleSim(xp, si, sj, k, r0, rc, 0.01).read_energy()[0][0]
        Um = OracleSim(xm, si, sj, k, r0, rc, 0.01).read_energy()[0][0]
        assert abs(-(Up - Um) / (2 * h) - f[p, c]) <= 1e-7 * max(1.0, abs(f[p, c]))


def test_P12_damping_closed_form():
    """Q7: with c = gamma dt/m the step reduces to u_{n+2} - (2 - c - w^2 dt^2) u_{n+1} + (1 - c) u_n = 0."""
    m = k = r0 = 1.0
    dt, gamma, u0 = 0.01, 0.01, 0.05
    s = _two_particles(r0 + u0, k, r0, 10.0, dt, gamma=gamma, m=m)
    c, w2 = gamma * dt / m, k / m * dt * dt
    rho = np.sqrt(1 - c)
    cphi = (2 - c - w2) / (2 * rho)
    phi = np.arccos(cphi)
    A, u1 = u0, u0 * (1 - w2 / 2)
    B = (u1 / rho - A * cphi) / np.sin(phi)
    err = 0.0
    for blk in range(100):
        s.step(100)
        n = (blk + 1) * 100
        x, _ = s.read_state()
        err = max(err, abs((x[1, 0] - r0) - rho ** n * (A * np.cos(n * phi) + B * np.sin(n * phi))))
    assert err <= 1e-11
    assert abs(rho ** 10000 - np.exp(-gamma * 100.0 / (2 * m))) < 2e-5


def test_boundary_reaction_and_sampling_static():
    """Reaction sums R_g = sum of spring forces on the group's particles (north_star item 4): static affine state,
    R_top,y = -R_bot,y = sum over top-row particles of the closed-form per-particle force (edge particles differ)."""
    nx = ny = 16
    eps = 1e-3
    x, si, sj, site, _ = triangular_lattice(nx, ny)
    xa = x * np.array([1.0 - eps / 3, 1.0 + eps])
    M = si.size
    row = site // nx
    s = OracleSim(xa, si, sj, np.ones(M), np.ones(M), np.full(M, 2.0), 1e-3, gamma=0.0, sample_every=1)
    s.set_boundary(0, np.flatnonzero(row == 0), FIXED)
    s.set_boundary(1, np.flatnonzero(row == ny - 1), FIXED)
    s.step(1)
    h = s.read_stress()
    L = np.sqrt((1 - eps / 3) ** 2 / 4 + 3 * (1 + eps) ** 2 / 4)
    n_diag_top = 2 * nx - 1                      # diagonal/vertical springs hanging from the top row
    fy = -(L - 1.0) / L * SQ3_2 * (1 + eps)
    # the interior moved by O(eps^2 dt^2): reaction equals the static value to ~1e-9 relative
    assert abs(h["R"][0, 0, 1, 1] / (n_diag_top * fy) - 1) < 1e-6
    assert abs(h["R"][0, 0, 0, 1] / (-n_diag_top * fy) - 1) < 1e-6
    assert h["step"][0] == 1


def test_batched_equals_individual():
    """Batched layout (a9): a disjoint union evolves each specimen exactly as it evolves alone."""
    from lsm_inputs import config4, single_specimen
    pb = config4(B=3, n=16)
    sb = OracleSim.from_problem(pb, sample_every=50)
    sb.step(200)
    xb, vb = sb.read_state()
    hb = sb.read_stress()
    for b in range(3):
        p1 = single_specimen(b, 16)
        s1 = OracleSim.from_problem(p1, sample_every=50)
        s1.step(200)
        x1, v1 = s1.read_state()
        sl = slice(pb.particle_offsets[b], pb.particle_offsets[b + 1])
        assert np.array_equal(xb[sl], x1) and np.array_equal(vb[sl], v1)
        h1 = s1.read_stress()
        assert np.array_equal(hb["U"][:, b], h1["U"][:, 0]) and np.array_equal(hb["R"][:, b], h1["R"][:, 0])


def test_config1_reference_values():
    """SURVEY.md S2 (an independent numpy scratch run of config 1 at survey time): no breakage in 10^4 steps,
    sigma_top = 1.742e-2, sigma_bot = 2.208e-2, U = 0.7073, KE = 0.0278 at step 10^4."""
    p = config1()
    s = OracleSim.from_problem(p)
    s.step(10000)
    h = s.read_stress()
    assert h["n_broken"][-1, 0] == 0
    assert abs(-h["R"][-1, 0, 1, 1] / p.meta["W0"] - 1.742e-2) < 5e-6
    assert abs(h["R"][-1, 0, 0, 1] / p.meta["W0"] - 2.208e-2) < 5e-6
    assert abs(h["U"][-1, 0] - 0.7073) < 5e-5 and abs(h["KE"][-1, 0] - 0.0278) < 5e-5


def test_generators_match_paper_shapes():
    g = golden("paper_table1_table2.txt")
    lo, hi = g["t2_springs_min"] / g["t2_particles_min"], g["t2_springs_max"] / g["t2_particles_max"]
    p = config1()
    assert p.M == 64 * 63 + 63 * 127 == 12033
    assert lo - 0.1 < p.M / p.N < 3.0                      # Table 2: M/N = 2.885 .. 2.941
    deg = np.bincount(np.concatenate([p.spring_i, p.spring_j]), minlength=p.N)
    assert deg.max() == 6 and (deg == 6).sum() == 3844     # "six springs"
    d = np.linalg.norm(p.x[p.spring_j] - p.x[p.spring_i], axis=1)
    assert np.abs(d - 1.0).max() < 1e-14
    # Table 1: rc/r0 between 1.01 and 1.10; the synthetic configs stay in a comparable range
    assert 1.0 < g["t1_stiff_rc"] / g["t1_stiff_r0"] < p.rc[0] / p.r0[0] + 1e-12 <= g["t1_soft_rc"] / g["t1_soft_r0"] + 1e-12


# ---------------------------------------------------------------- P13: per-particle virial stress (Eq. 7)
@pytest.mark.parametrize("eps", [1e-3, 2e-2])
def test_P13_virial_equals_cauchy_stress_in_affine_state(eps):
    """In a homogeneous static state the virial stress of an interior particle, divided by its (deformed) cell area,
    is the Cauchy stress: sigma_yy = the top row's reaction per unit deformed width (P3's closed form), sigma_xx = 0
    (Poisson's ratio 1/3: the lateral contraction eps/3 is exactly the stress-free one to first order; the residual is
    the second-order term given below), sigma_xy = 0 by symmetry."""
    nx = ny = 32
    kk = 1.7
    x, si, sj, site, kind = triangular_lattice(nx, ny)
    xa = x * np.array([1.0 - eps / 3.0, 1.0 + eps])
    M = si.size
    s = OracleSim(xa, si, sj, np.full(M, kk), np.ones(M), np.full(M, 2.0), 0.01)
    S = s.read_virial()
    row, col = site // nx, site % nx
    interior = (row > 0) & (row < ny - 1) & (col > 0) & (col < nx - 1)
    ax, ay = 1.0 - eps / 3.0, 1.0 + eps
    L = np.sqrt(ax ** 2 / 4 + 3 * ay ** 2 / 4)
    g_d, g_h = kk * (L - 1.0) / L, kk * (ax - 1.0) / ax          # k (r - r0)/r of a diagonal / a horizontal spring
    cell = ax * SQ3_2 * ay                                        # deformed area per particle
    # closed forms: 4 diagonal springs with d = (+-ax/2, +-sqrt3/2 ay), 2 horizontal springs with d = (+-ax, 0)
    syy = 0.5 * 4 * g_d * (SQ3_2 * ay) ** 2
    sxx = 0.5 * (4 * g_d * (ax / 2) ** 2 + 2 * g_h * ax ** 2)
    assert np.allclose(S[interior, 1], syy, rtol=1e-11)
    # sxx is a cancellation of terms of size syy; coordinates up to 32 carry ulp 7e-15, so each bond length does too
    noise = 8 * np.finfo(float).eps * np.abs(xa).max() * kk
    assert np.abs(S[interior, 0] - sxx).max() <= noise < 1e-9 * syy
    assert np.abs(S[interior, 2]).max() <= noise
    # sigma_yy = reaction of the top row per unit deformed width (the force f_y of P3 over the spacing ax)
    f = s.read_forces()
    top_int = (row == ny - 1) & (col > 0) & (col < nx - 1)
    assert np.allclose(S[interior, 1] / cell, -f[top_int, 1].mean() / ax, rtol=1e-11)
    # Poisson's ratio 1/3: sigma_xx vanishes to first order in eps (it is O(eps^2) of sigma_yy's O(eps))
    assert abs(sxx) <= 2.0 * eps * syy


def test_P13_virial_kinetic_term_and_sum_rule():
    """Kinetic term -m v(x)v on a free particle without springs; and sum over particles of the static virial = sum
    over springs of g d(x)d (each spring gives half to either end): trace = sum_s k (r - r0) r, brute force."""
    x = np.array([[0.0, 0.0], [3.0, 0.0]])
    v = np.array([[0.5, -2.0], [0.0, 0.0]])
    s = OracleSim(x, [0], [1], 0.0, 1.0, 10.0, 0.01, v=v, mass=np.array([3.0, 1.0]))
    S = s.read_virial()
    assert np.allclose(S[0], [-3.0 * 0.25, -3.0 * 4.0, -3.0 * 0.5 * -2.0]) and np.all(S[1] == 0.0)
    xs, si, sj, k, r0 = _random_state(7, 6, seed=5)
    s = OracleSim(xs, si, sj, k, r0, np.full(si.size, 9.0), 0.01)
    S = s.read_virial()
    d = xs[sj] - xs[si]
    r = np.sqrt((d ** 2).sum(axis=1))
    g = k * (r - r0) / r
    assert np.allclose(S[:, 0].sum(), (g * d[:, 0] ** 2).sum(), rtol=1e-12)
    assert np.allclose(S[:, 2].sum(), (g * d[:, 0] * d[:, 1]).sum(), rtol=1e-11, atol=1e-14)
    assert np.allclose((S[:, 0] + S[:, 1]).sum(), (k * (r - r0) * r).sum(), rtol=1e-12)


# ---------------------------------------------------------------- P15: Lagrangian strain field, Eq. 8 (L150, L156), reading Q21
def _green_lagrange(F):
    F = np.asarray(F, dtype=float)
    E = 0.5 * (F.T @ F - np.eye(F.shape[0]))
    return np.array([E[0, 0], E[1, 1], E[0, 1]]) if F.shape[0] == 2 else np.array([E[0, 0], E[1, 1], E[2, 2], E[0, 1], E[1, 2], E[2, 0]])


def test_P15_strain_of_a_homogeneous_deformation_is_green_lagrange():
    """x -> F x + t with a NON-symmetric F (stretch + shear + rotation part): the local affine fit recovers F at every
    particle that has two independent bonds -- interior, edge and corner alike -- so eps = (F^T F - I)/2 everywhere.
    F F^T (a transposed J), F^T F without the 1/2, the small-strain (F + F^T)/2 - I: all differ from it by > 1e-2."""
    nx, ny = 9, 7
    x, si, sj, site, _ = triangular_lattice(nx, ny)
    F = np.array([[1.25, 0.5], [0.125, 0.875]])
    s = OracleSim(x, si, sj, 1.0, 1.0, 10.0, 0.01)
    s.write_state(x @ F.T + np.array([3.0, -2.0]))
    E, ok = s.read_strain()
    want = _green_lagrange(F)
    assert ok.all() and np.abs(E - want).max() <= 1e-13
    wrong = [_green_lagrange(F.T), 2 * want, np.array([F[0, 0] - 1, F[1, 1] - 1, 0.5 * (F[0, 1] + F[1, 0])])]
    assert min(np.abs(w - want).max() for w in wrong) > 1e-2
    # rigid motion: rotation by 0.7 rad + translation -> zero strain
    c, sn = np.cos(0.7), np.sin(0.7)
    s.write_state(x @ np.array([[c, -sn], [sn, c]]).T + np.array([-1.0, 4.0]))
    E, ok = s.read_strain()
    assert ok.all() and np.abs(E).max() <= 1e-14
    # the reference is the configuration given at create, not the last written state: undeformed again -> 0 (V V^-1 rounds)
    s.write_state(x)
    assert np.abs(s.read_strain()[0]).max() <= 1e-15


@pytest.mark.parametrize("eps", [1e-3, 1e-6])
def test_P15_small_strain_limit_of_the_uniaxial_state(eps):
    """P3's affine state x * (1 - eps/3, 1 + eps) (Poisson's ratio 1/3): e_yy = eps + eps^2/2, e_xx = -eps/3 + eps^2/18,
    e_xy = 0; to first order the symmetric displacement gradient (eps_yy = eps, eps_xx = -eps/3)."""
    x, si, sj, site, _ = triangular_lattice(16, 12)
    s = OracleSim(x * np.array([1.0 - eps / 3.0, 1.0 + eps]), si, sj, 1.0, 1.0, 2.0, 0.01)
    assert np.abs(s.read_strain()[0]).max() <= 1e-15            # created in that state: it IS the reference
    s = OracleSim(x, si, sj, 1.0, 1.0, 2.0, 0.01)
    s.write_state(x * np.array([1.0 - eps / 3.0, 1.0 + eps]))
    E, ok = s.read_strain()
    assert ok.all()
    assert np.abs(E[:, 1] - (eps + eps ** 2 / 2)).max() <= 1e-14 and np.abs(E[:, 0] - (-eps / 3 + eps ** 2 / 18)).max() <= 1e-14
    assert np.abs(E[:, 2]).max() <= 1e-14
    assert np.abs(E[:, 1] - eps).max() <= eps ** 2 and np.abs(E[:, 0] + eps / 3).max() <= eps ** 2


def test_P15_least_squares_against_numpy_and_bond_selection():
    """(a) a NON-affine displacement: per particle, J from numpy's lstsq (SVD) on the stacked bond vectors d0 J ~ d (the
    row-vector form of Shimizu et al.), eps = (J J^T - I)/2 -- another routine, the paper's own index order;
    (b) only bonds alive now count: a neighbour whose spring has broken (r > rc) does not enter the fit;
    (c) fewer than two independent bonds (none, one, two collinear): flagged, reported as 0, never NaN."""
    x, si, sj, site, _ = triangular_lattice(8, 6)
    rng = np.random.default_rng(21)
    s = OracleSim(x, si, sj, 1.0, 1.0, 10.0, 0.01)
    xc = x @ np.array([[1.1, 0.2], [-0.1, 0.95]]).T + rng.uniform(-0.05, 0.05, x.shape)
    s.write_state(xc)
    E, ok = s.read_strain()
    assert ok.all()
    for p in range(x.shape[0]):
        nb = np.concatenate([sj[si == p], si[sj == p]])
        J = np.linalg.lstsq(x[nb] - x[p], xc[nb] - xc[p], rcond=None)[0]
        G = 0.5 * (J @ J.T - np.eye(2))
        assert np.abs(E[p] - [G[0, 0], G[1, 1], G[0, 1]]).max() <= 1e-13
    # (b) centre 0 with neighbours 1, 2 (moved by F1) and 3 (torn away: its spring breaks at create + write_state)
    F1 = np.array([[1.5, 0.25], [0.0, 0.75]])
    x4 = np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 1.0], [-1.0, -1.0], [5.0, 5.0], [6.0, 5.0], [7.0, 5.0], [9.0, 9.0]])
    si4, sj4 = [0, 0, 0, 4, 5], [1, 2, 3, 5, 6]
    s = OracleSim(x4, si4, sj4, 1.0, np.array([1.0, 1.0, np.sqrt(2.0), 1.0, 1.0]), np.array([9.0, 9.0, 2.0, 9.0, 9.0]), 0.01)
    x4c = x4 @ F1.T
    x4c[3] = [-4.0, -4.0]                                           # |d| = 5.66 > rc = 2: broken
    x4c[4:7] = x4[4:7] * 1.5                                        # a collinear chain, stretched
    s.write_state(x4c)
    assert s.read_broken()[0].tolist() == [False, False, True, False, False]
    E, ok = s.read_strain()
    assert ok.tolist() == [True, False, False, False, False, False, False, False]
    assert np.abs(E[0] - _green_lagrange(F1)).max() <= 1e-15        # from bonds 0-1 and 0-2 alone
    assert np.all(E[1:] == 0.0) and np.isfinite(E).all()            # one bond (1, 2, 4, 6), none (3, 7), two collinear (5)


def test_P15_strain_3d():
    """D = 3: a non-symmetric homogeneous F on a cubic network with face diagonals -> (F^T F - I)/2 in the order
    {xx, yy, zz, xy, yz, zx}; a rotation about a skew axis -> 0; a plain cubic network's corner (3 orthogonal bonds) is
    still full rank, a particle with bonds in one plane only is flagged."""
    from lsm_inputs import cubic_lattice_3d
    x, si, sj, r0 = cubic_lattice_3d(4, 3, 5)
    F = np.array([[1.25, 0.5, 0.0], [0.125, 0.875, 0.25], [-0.25, 0.0, 1.5]])
    s = OracleSim(x, si, sj, 1.0, r0, 10.0 * r0, 0.01)
    s.write_state(x @ F.T + np.array([1.0, 2.0, 3.0]))
    E, ok = s.read_strain()
    assert ok.all() and np.abs(E - _green_lagrange(F)).max() <= 1e-13
    assert np.abs(_green_lagrange(F.T) - _green_lagrange(F)).max() > 1e-2
    n = np.array([1.0, 2.0, 2.0]) / 3.0
    K = np.array([[0, -n[2], n[1]], [n[2], 0, -n[0]], [-n[1], n[0], 0]])
    R = np.eye(3) + np.sin(0.9) * K + (1 - np.cos(0.9)) * K @ K
    s.write_state(x @ R.T)
    assert np.abs(s.read_strain()[0]).max() <= 1e-14
    xs, si2, sj2, r02 = cubic_lattice_3d(2, 2, 1, diagonals=False)   # a single square in the plane z = 0
    s = OracleSim(xs, si2, sj2, 1.0, r02, 10.0 * r02, 0.01)
    s.write_state(xs * 1.1)
    E, ok = s.read_strain()
    assert not ok.any() and np.all(E == 0.0)


# ---------------------------------------------------------------- P14: the oracle's D = 3 branch (the paper's listing is 3-D, L93-L97)
def test_P14_3d_oscillator_along_a_skew_axis_and_invariants():
    """(a) P1's worked example rotated onto the axis (1,2,2)/3: the 3-D trajectory must be the 1-D closed form along
    that axis (velocity Verlet commutes with rotations); (b) zero net force and torque, F = -grad U by central
    differences, on a perturbed cubic network with face diagonals; (c) uniform stretch of a plain cubic network:
    every interior particle force-free, each face particle pulled back by k (stretch - 1) r0 per bond."""
    from lsm_inputs import cubic_lattice_3d
    n = np.array([1.0, 2.0, 2.0]) / 3.0
    k, r0, dt, m = 1e-4, 10.0, 1.0, 1.0
    x = np.array([[0.0, 0.0, 0.0], 15.0 * n])
    s = OracleSim(x, [0], [1], k, r0, 100.0, dt)
    s.set_boundary(0, [0], FIXED)
    theta = np.arccos(1.0 - k * dt * dt / (2 * m))
    for nstep in (1, 10, 250, 1000):
        s.step(nstep - s.current_step)
        xs, _ = s.read_state()
        assert np.abs(xs[1] - (r0 + 5.0 * np.cos(nstep * theta)) * n).max() <= 1e-11
    # (b)
    xs, si, sj, r0s = cubic_lattice_3d(4, 3, 5)
    rng = np.random.default_rng(3)
    xs = xs + rng.uniform(-0.05, 0.05, xs.shape)
    ks = rng.uniform(0.5, 2.0, si.size)
    s = OracleSim(xs, si, sj, ks, r0s, np.full(si.size, 9.0), 0.01)
    f = s.read_forces()
    scale = np.abs(f).sum()
    assert np.abs(f.sum(axis=0)).max() <= 1e-13 * scale and np.abs(np.cross(xs, f).sum(axis=0)).max() <= 1e-12 * scale
    U0 = s.read_energy()[0][0]
    d = xs[sj] - xs[si]
    assert np.isclose(U0, (0.5 * ks * (np.sqrt((d ** 2).sum(axis=1)) - r0s) ** 2).sum(), rtol=1e-13)
    h = 1e-6
    for p, c in ((7, 0), (20, 1), (33, 2)):
        up = []
        for sgn in (+1, -1):
            xq = xs.copy(); xq[p, c] += sgn * h
            up.append(OracleSim(xq, si, sj, ks, r0s, np.full(si.size, 9.0), 0.01).read_energy()[0][0])
        assert abs(-(up[0] - up[1]) / (2 * h) - f[p, c]) <= 1e-7 * np.abs(f).max()
    # (c)
    nx = 5
    xs, si, sj, r0s = cubic_lattice_3d(nx, nx, nx, diagonals=False)
    lam, kk = 1.01, 1.7
    s = OracleSim(xs * lam, si, sj, kk, r0s, np.full(si.size, 9.0), 0.01)
    f = s.read_forces()
    g = np.round(xs).astype(int)
    interior = np.all((g > 0) & (g < nx - 1), axis=1)
    assert np.abs(f[interior]).max() <= 1e-14
    face = (g[:, 0] == nx - 1) & np.all((g[:, 1:] > 0) & (g[:, 1:] < nx - 1), axis=1)
    assert np.allclose(f[face, 0], -kk * (lam - 1.0), rtol=1e-12) and np.abs(f[face, 1:]).max() <= 1e-14


def test_P13_virial_3d_uniform_stretch_and_sum_rule():
    """3-D virial: a plain cubic network stretched uniformly by lam has, at every interior particle, the diagonal virial
    S_cc = 1/2 * 2 bonds * k (lam - 1) r0 * lam r0 per axis = the Cauchy stress k (lam-1)/(lam r0) x the cell volume
    lam^3; off-diagonals 0.  Sum rule on a perturbed network with diagonals: sum_p tr S_p = sum_s k (r - r0) r."""
    from lsm_inputs import cubic_lattice_3d
    nx, lam, kk = 5, 1.02, 1.7
    xs, si, sj, r0s = cubic_lattice_3d(nx, nx, nx, diagonals=False)
    s = OracleSim(xs * lam, si, sj, kk, r0s, np.full(si.size, 9.0), 0.01)
    S = s.read_virial()
    g = np.round(xs).astype(int)
    interior = np.all((g > 0) & (g < nx - 1), axis=1)
    assert S.shape == (xs.shape[0], 6)
    assert np.allclose(S[interior, :3], kk * (lam - 1.0) * lam, rtol=1e-12) and np.abs(S[interior, 3:]).max() <= 1e-14
    sigma = S[interior, 0] / lam ** 3                       # virial / deformed cell volume
    assert np.allclose(sigma, kk * (lam - 1.0) / lam ** 2, rtol=1e-12)   # = bond force k (lam-1) over the face area lam^2
    xs, si, sj, r0s = cubic_lattice_3d(4, 5, 3)
    rng = np.random.default_rng(9)
    xs = xs + rng.uniform(-0.05, 0.05, xs.shape)
    ks = rng.uniform(0.5, 2.0, si.size)
    v = rng.normal(0, 0.1, xs.shape)
    S = OracleSim(xs, si, sj, ks, r0s, np.full(si.size, 9.0), 0.01, v=v, mass=2.0).read_virial()
    d = xs[sj] - xs[si]; r = np.sqrt((d ** 2).sum(axis=1))
    assert np.isclose(S[:, :3].sum(), (ks * (r - r0s) * r).sum() - 2.0 * (v ** 2).sum(), rtol=1e-12)
    assert np.isclose(S[:, 4].sum(), (ks * (r - r0s) / r * d[:, 1] * d[:, 2]).sum() - 2.0 * (v[:, 1] * v[:, 2]).sum(), rtol=1e-11)


def test_P11_summation_order_sensitivity_budget():
    """P11: what the GPU tolerances rest on.  The same config-1 run with the spring list permuted, the
    endpoints swapped at random and the particles renumbered differs from the original only by rounding: after 10^4
    steps |dx|, |dv| stay below 1e-11 (survey scratch: 4e-13, 7e-13), three orders inside north_star's 1e-9."""
    from lsm_inputs import config1, shuffle_ids
    p = config1()
    q = shuffle_ids(p, 12)
    a = OracleSim.from_problem(p); a.step(10000)
    b = OracleSim.from_problem(q); b.step(10000)
    xa, va = a.read_state(); xb, vb = b.read_state()
    perm = q.meta["perm"]                     # new particle id -> old particle id
    assert a.read_broken()[2] == 0 and b.read_broken()[2] == 0
    dx, dv = np.abs(xb - xa[perm]).max(), np.abs(vb - va[perm]).max()
    assert 0 < dx <= 1e-11 and dv <= 1e-11


# ---------------------------------------------------------------- mass != 1 (Eq. 4 a = F/m; per-type masses, L88)
def test_P1_oscillator_with_mass_4():
    """P1's closed form with m = 4: theta = arccos(1 - k dt^2 / (2 m)); a wrong `fd*m` (or a dropped 1/m) changes the
    period by a factor 4 (2) and fails at 1e-11.  The sampled KE = 1/2 m v^2 with the closed-form full-step velocity."""
    k, r0, dt, m, A = 1e-4, 10.0, 1.0, 4.0, 5.0
    s = _two_particles(r0 + A, k, r0, 100.0, dt, m=m, sample_every=1)
    th = 2.0 * np.arcsin(np.sqrt(k * dt * dt / (4.0 * m)))     # = arccos(1 - k dt^2 / (2 m)), well conditioned at small angles
    for n in range(1, 1501):
        s.step(1)
        x, v = s.read_state()
        assert abs(x[1, 0] - (r0 + A * np.cos(n * th))) <= 1e-11
        assert abs(v[1, 0] + A * np.sin(th) / dt * np.sin(n * th)) <= 1e-12
    h = s.read_stress()
    n = np.arange(1, 1501)
    ke = 0.5 * m * (A * np.sin(th) / dt * np.sin(n * th)) ** 2
    assert np.abs(h["KE"][:, 0] - ke).max() <= 1e-13 * ke.max()
    U, KE = s.read_energy()
    assert abs(KE[0] - ke[-1]) <= 1e-13 * ke.max()


def test_P2_two_free_particles_unequal_masses():
    """Two free particles with m0 = 3, m1 = 0.5 (a per-particle mass ARRAY): the separation follows the closed form
    with the reduced mass m0 m1/(m0 + m1); the mass-weighted centre of mass stays put; each particle moves by its
    mass share; sampled KE = 1/2 m_red v_rel^2 with the closed-form relative velocity."""
    k, r0, dt, A = 1e-4, 10.0, 1.0, 5.0
    m0, m1 = 3.0, 0.5
    x = np.array([[0.0, 0.0], [r0 + A, 0.0]])
    s = OracleSim(x, [0], [1], [k], [r0], [100.0], dt, mass=np.array([m0, m1]), sample_every=1)
    mred = m0 * m1 / (m0 + m1)
    th = 2.0 * np.arcsin(np.sqrt((k / mred) * dt * dt / 4.0))  # = arccos(1 - (k/m_red) dt^2 / 2)
    com0 = (m1 * (r0 + A)) / (m0 + m1)
    for n in range(1, 1001):
        s.step(1)
        xx, vv = s.read_state()
        sep = xx[1, 0] - xx[0, 0]
        assert abs(sep - (r0 + A * np.cos(n * th))) <= 1e-11
        assert abs((m0 * xx[0, 0] + m1 * xx[1, 0]) / (m0 + m1) - com0) <= 1e-12
        assert abs(m0 * vv[0, 0] + m1 * vv[1, 0]) <= 1e-15
        # particle 1 carries the share m0/(m0+m1) of the relative motion
        assert abs((xx[1, 0] - (r0 + A)) - m0 / (m0 + m1) * (sep - (r0 + A))) <= 1e-11
    h = s.read_stress()
    n = np.arange(1, 1001)
    vrel = -A * np.sin(th) / dt * np.sin(n * th)
    ke = 0.5 * mred * vrel ** 2
    assert np.abs(h["KE"][:, 0] - ke).max() <= 1e-12 * ke.max()


def test_P12_damping_with_mass_2():
    """P12's recurrence with m = 2: c = gamma dt / m, w^2 = k/m.  Pins that the damping force is divided by m exactly
    once (gamma has units mass/time, Q7)."""
    m, k, r0 = 2.0, 1.0, 1.0
    dt, gamma, u0 = 0.01, 0.03, 0.05
    s = _two_particles(r0 + u0, k, r0, 10.0, dt, gamma=gamma, m=m)
    c, w2 = gamma * dt / m, k / m * dt * dt
    rho = np.sqrt(1 - c)
    cphi = (2 - c - w2) / (2 * rho)
    phi = np.arccos(cphi)
    A, u1 = u0, u0 * (1 - w2 / 2)
    B = (u1 / rho - A * cphi) / np.sin(phi)
    for blk in range(50):
        s.step(100)
        n = (blk + 1) * 100
        x, _ = s.read_state()
        assert abs((x[1, 0] - r0) - rho ** n * (A * np.cos(n * phi) + B * np.sin(n * phi))) <= 1e-11


# ---------------------------------------------------------------- kinematic particles (Q6) and olsm_write_state
def test_kinematic_velocity_is_du_over_dt_and_carries_no_KE():
    """Q6: a MOVE particle reports v = du/dt (also right after set_boundary, before any step), a FIXED one v = 0, and
    neither enters KE; the virial's kinetic term uses that stored velocity."""
    dt = 0.25
    x = np.array([[0.0, 0.0], [1.0, 0.0], [5.0, 5.0]])
    v = np.array([[9.0, 9.0], [7.0, 7.0], [0.5, -1.0]])
    s = OracleSim(x, [0], [1], 0.0, 1.0, 10.0, dt, v=v, mass=np.array([1.0, 2.0, 4.0]), sample_every=1)
    s.set_boundary(0, [0], FIXED)
    s.set_boundary(1, [1], MOVE, [0.125, -0.5])
    _, vv = s.read_state()
    assert np.array_equal(vv[0], [0.0, 0.0]) and np.array_equal(vv[1], [0.5, -2.0]) and np.array_equal(vv[2], [0.5, -1.0])
    assert s.read_energy()[1][0] == 0.5 * 4.0 * (0.25 + 1.0)          # only the free particle
    S = s.read_virial()
    assert np.array_equal(S[1], [-2.0 * 0.25, -2.0 * 4.0, -2.0 * 0.5 * -2.0])
    s.step(3)
    xx, vv = s.read_state()
    assert np.array_equal(xx[1], [1.375, -1.5]) and np.array_equal(vv[1], [0.5, -2.0]) and np.array_equal(xx[0], [0.0, 0.0])
    assert np.array_equal(xx[2], [5.0 + 3 * dt * 0.5, 5.0 - 3 * dt])   # free flight (k = 0)
    assert np.all(s.read_stress()["KE"][:, 0] == 0.5 * 4.0 * 1.25)


def test_write_state_restarts_on_the_closed_form():
    """olsm_write_state: (a) writing the closed-form state (x_n, v_n) of P1's oscillator into a handle that has already
    run somewhere else continues ON the closed form (forces are refreshed from the written positions -- with a stale
    f the very next kick is wrong -- and v is taken as the full-step velocity); (b) a MOVE particle takes the written
    position as its new origin and restarts its step count there: after j more steps it sits at written + j du exactly
    (dyadic du) -- a missing n0 reset or origin re-snapshot is off by (steps before the write) * du."""
    k, r0, dt, A = 1e-4, 10.0, 1.0, 5.0
    th = 2.0 * np.arcsin(np.sqrt(k * dt * dt / 4.0))           # = arccos(1 - k dt^2 / 2)
    n0 = 137
    xn = r0 + A * np.cos(n0 * th)
    vn = -A * np.sin(th) / dt * np.sin(n0 * th)
    du = np.array([2.0 ** -7, -2.0 ** -9])
    #            fixed end   oscillator      a MOVE particle tied to nothing (k irrelevant: own spring has k = 0)
    x = np.array([[0.0, 0.0], [r0 + 1.0, 0.0], [40.0, 3.0], [41.0, 3.0]])
    s = OracleSim(x, [0, 2], [1, 3], [k, 0.0], [r0, 1.0], [100.0, 100.0], dt)
    s.set_boundary(0, [0], FIXED)
    s.set_boundary(1, [2], MOVE, du)
    s.step(61)                                                   # somewhere else: step counter 61, group origin at step 0
    xw = np.array([[0.0, 0.0], [xn, 0.0], [50.0, -2.0], [41.0, 3.0]])
    vw = np.array([[0.0, 0.0], [vn, 0.0], [123.0, 456.0], [0.0, 0.0]])   # the written v of a kinematic particle is ignored
    s.write_state(xw, vw)
    f = s.read_forces()
    assert abs(f[1, 0] + k * (xn - r0)) <= 1e-18 and f[0, 0] == -f[1, 0]
    _, vv = s.read_state()
    assert np.array_equal(vv[2], du / dt)
    for j in range(1, 401):
        s.step(1)
        xx, vv = s.read_state()
        assert abs(xx[1, 0] - (r0 + A * np.cos((n0 + j) * th))) <= 1e-11
        assert abs(vv[1, 0] + A * np.sin(th) / dt * np.sin((n0 + j) * th)) <= 1e-12
        assert np.array_equal(xx[2], [50.0 + j * du[0], -2.0 + j * du[1]])
        assert np.array_equal(xx[0], [0.0, 0.0])


def test_set_boundary_mid_run_keeps_the_held_force():
    """Redefining a group between two steps changes memberships and origins only: the total force fd = f - gamma v held
    from the last force evaluation (Q7: damping with the velocity held at force time) still feeds the next first half
    kick of every particle that stays free.  Closed form: P12's damped oscillator keeps following its recurrence when
    an unrelated MOVE group is reversed in the middle of the run."""
    m = k = r0 = 1.0
    dt, gamma, u0 = 0.01, 0.05, 0.05
    x = np.array([[0.0, 0.0], [r0 + u0, 0.0], [10.0, 0.0], [11.0, 0.0]])
    s = OracleSim(x, [0, 2], [1, 3], [k, 0.0], [r0, 1.0], [10.0, 10.0], dt, gamma=gamma)
    s.set_boundary(0, [0], FIXED)
    s.set_boundary(1, [2], MOVE, [2.0 ** -10, 0.0])
    c, w2 = gamma * dt / m, k / m * dt * dt
    rho = np.sqrt(1 - c)
    cphi = (2 - c - w2) / (2 * rho)
    phi = np.arccos(cphi)
    A, u1 = u0, u0 * (1 - w2 / 2)
    B = (u1 / rho - A * cphi) / np.sin(phi)
    for n in range(1, 2001):
        s.step(1)
        if n == 777:
            s.set_boundary(1, [2], MOVE, [-2.0 ** -10, 0.0])      # reversal: origin = current position, n0 = 777
        if n == 1200:
            s.set_boundary(1, [], MOVE, [0.0, 0.0])               # release: particle 2 flies on freely with v = du/dt
        xx, vv = s.read_state()
        assert abs((xx[1, 0] - r0) - rho ** n * (A * np.cos(n * phi) + B * np.sin(n * phi))) <= 1e-12
        if n <= 777:
            assert xx[2, 0] == 10.0 + n * 2.0 ** -10
        elif n <= 1200:
            assert xx[2, 0] == 10.0 + (2 * 777 - n) * 2.0 ** -10
    # released at step 1200 with v = -2^-10/dt, then damped free flight (k = 0): v_{n+1} = v_n (1 - c/2 ... ) per Q7:
    # kick1: v += hdt*(-gamma v_held)/m, kick2 likewise with the half-step velocity -> checked as monotone decay here
    assert -2.0 ** -10 / dt < vv[2, 0] < 0.0 and xx[2, 0] < 10.0 + (2 * 777 - 1200) * 2.0 ** -10


def test_threaded_variant_is_bit_equal_to_the_serial_loop():
    """olsm_set_threads (the all-cores timing leg of bench.py): same arithmetic per spring, same ascending-spring-id
    summation per particle -> x, v, f, broken set, break steps and the sampled history must all be BIT-equal to the
    serial reference loop through a fracture run; also in a batch, in 3-D, and when switching back and forth."""
    from lsm_inputs import config2, config4, cubic_lattice_3d
    p = config2(n=48, seed=11, n_blobs=24, du_y=6e-4)
    p.sample_every = 50
    a = OracleSim.from_problem(p); b = OracleSim.from_problem(p)
    b.set_threads(4)
    # the threaded -> serial switch falls BETWEEN two sample steps (samples every 50), and U is read right after it and again
    # at the next sample: a serial evaluation must not be overwritten by the per-spring energies of the last threaded one
    a.step(1470); b.step(1470); b.set_threads(1); a.step(10); b.step(10)
    assert np.array_equal(a.read_energy()[0], b.read_energy()[0]) and np.array_equal(a.read_energy()[1], b.read_energy()[1])
    a.step(2520); b.step(520); b.set_threads(3); b.step(2000)
    assert a.read_broken()[2] > 10
    for u, w in zip(a.read_state() + (a.read_forces(),) + a.read_broken()[:2], b.read_state() + (b.read_forces(),) + b.read_broken()[:2]):
        assert np.array_equal(u, w)
    ha, hb = a.read_stress(), b.read_stress()
    for key in ha:
        assert np.array_equal(ha[key], hb[key]), key
    assert np.array_equal(a.read_energy()[0], b.read_energy()[0]) and np.array_equal(a.read_virial(), b.read_virial())
    pb = config4(B=3, n=16)
    a = OracleSim.from_problem(pb, sample_every=50); b = OracleSim.from_problem(pb, sample_every=50)
    b.set_threads(8)
    a.step(300); b.step(300)
    assert np.array_equal(a.read_state()[0], b.read_state()[0]) and np.array_equal(a.read_stress()["U"], b.read_stress()["U"])
    x, si, sj, r0 = cubic_lattice_3d(5, 4, 6)
    x = x + np.random.default_rng(1).uniform(-0.05, 0.05, x.shape)
    a = OracleSim(x, si, sj, 1.0, r0, 1.04 * r0, 0.02); b = OracleSim(x, si, sj, 1.0, r0, 1.04 * r0, 0.02)
    b.set_threads(4)
    a.step(200); b.step(200)
    assert a.read_broken()[2] > 0 and np.array_equal(a.read_broken()[1], b.read_broken()[1])
    assert np.array_equal(a.read_state()[0], b.read_state()[0]) and np.array_equal(a.read_state()[1], b.read_state()[1])
