"""Pins for the fp64 oracle (oracle/rad_oracle.c) -- CPU only.

The paper prints no worked numerical example for the radiation detector (PAPER.md has
no equation for it), so every pin is a closed form, an invariant or a
brute force, as BASELINE.json north_star prescribes ("zero output for unaccelerated
straight-line motion; cyclotron lines at harmonics of w_c for helical motion; exact
linearity in particle weights and superposition across particles and steps; brute-force
agreement on tiny inputs").  Pin numbers follow SURVEY.md section 8(c).
Each pin is chosen so that a plausible slip (dropped dt, wrong sign of the phase, wrong
power of (1 - beta.n), transposed cross product, metres vs c) fails at least one of them.
"""
import numpy as np
import pytest
from scipy import special

C = 299792458.0


def _run(oracle_mod, dirs, omega, dt, steps, t0=0.0, scale=1.0, bins=None):
    """steps: iterable of (step_index, state list)."""
    o = oracle_mod.Oracle(dirs, omega, dt, t0=t0, scale=scale, bins=bins)
    for t, st in steps:
        o.accumulate_step(t, *st)
    return o


def _const_state(r0, beta, bdot, w=1.0, dtype=np.float64):
    vals = list(r0) + list(beta) + list(bdot) + [w]
    return [np.array([v], dtype=dtype) for v in vals]


DIRS = np.array([[1.0, 0.0, 0.0], [0.0, 0.0, 2.0], [0.3, -0.5, 0.8], [-0.6, 0.64, 0.48],
                 [0.1, 0.2, -0.97]])
UNIT = DIRS / np.linalg.norm(DIRS, axis=1, keepdims=True)
OMEGA = np.array([3.0e14, 1.0e15, 2.7e15, 8.1e15, 3.3e16])
DT = 2.0e-17


# ------------------------------------------------------------------------------ P1 zero
def test_p1_unaccelerated_motion_gives_exact_zero(oracle_mod):
    rng = np.random.default_rng(1)
    n = 50
    beta = rng.uniform(-0.5, 0.5, (3, n))
    r0 = rng.uniform(0, 1e-5, (3, n))
    steps = []
    for t in range(7):
        r = r0 + C * beta * t * DT
        steps.append((t, [r[0], r[1], r[2], beta[0], beta[1], beta[2],
                          np.zeros(n), np.zeros(n), np.zeros(n), rng.uniform(0.5, 2, n)]))
    o = _run(oracle_mod, DIRS, OMEGA, DT, steps)
    assert np.all(o.A == 0.0)
    assert np.all(o.spectrum() == 0.0)


# ----------------------------------------------------------- P2 / P3 Dirichlet kernel
def _dirichlet(x, T):
    """sin(T x/2)/sin(x/2)."""
    return np.sin(T * x / 2.0) / np.sin(x / 2.0)


@pytest.mark.parametrize("t0", [0.0, 3.7e-16])
def test_p2_p3_static_particle_dirichlet_kernel(oracle_mod, t0):
    r0 = np.array([1.3e-6, -2.1e-6, 0.7e-6])
    b = np.array([2.0e12, -1.0e12, 0.5e12])
    w, T = 1.7, 23
    st = _const_state(r0, (0, 0, 0), b, w)
    o = _run(oracle_mod, DIRS, OMEGA, DT, [(t, st) for t in range(T)], t0=t0)
    A = o.amplitude()
    S = o.spectrum()
    for i, n in enumerate(UNIT):
        ndb = n @ b
        vec = n * ndb - b                       # n x (n x b), written as BAC-CAB
        for j, om in enumerate(OMEGA):
            dk = _dirichlet(om * DT, T)
            # P2: magnitude
            s_ref = w ** 2 * (b @ b - ndb ** 2) * DT ** 2 * dk ** 2
            assert S[i, j] == pytest.approx(s_ref, rel=1e-9)
            # P3: complex amplitude incl. sign of the phase, t0 and n.r/c
            ph = np.exp(1j * om * (t0 - (n @ r0) / C)) * np.exp(1j * om * (T - 1) * DT / 2.0)
            a_ref = w * DT * vec * ph * dk
            assert np.allclose(A[i, j], a_ref, rtol=1e-9, atol=1e-12 * np.abs(a_ref).max())


# --------------------------------------------------------- P4 Doppler-shifted Dirichlet
def test_p4_uniform_motion_with_constant_betadot_doppler(oracle_mod):
    r0 = np.array([0.4e-6, 0.9e-6, -0.3e-6])
    beta = np.array([0.31, -0.12, 0.22])
    b = np.array([-1.0e12, 3.0e12, 2.0e12])
    w, T = 0.8, 31
    steps = [(t, _const_state(r0 + C * beta * t * DT, beta, b, w)) for t in range(T)]
    S = _run(oracle_mod, DIRS, OMEGA, DT, steps).spectrum()
    for i, n in enumerate(UNIT):
        d = 1.0 - n @ beta
        vec = (n - beta) * (n @ b) - b * d     # BAC-CAB of n x ((n-beta) x b)
        for j, om in enumerate(OMEGA):
            dk = _dirichlet(om * d * DT, T)    # Doppler: w' = w (1 - n.beta)
            s_ref = w ** 2 * (vec @ vec) / d ** 4 * DT ** 2 * dk ** 2
            assert S[i, j] == pytest.approx(s_ref, rel=2e-9)


# ------------------------------------------------------------ P5 two-particle interference
def test_p5_two_displaced_particles_interfere(oracle_mod):
    r0 = np.array([0.2e-6, 0.1e-6, 0.5e-6])
    dr = np.array([0.37e-6, -0.81e-6, 0.29e-6])
    b = np.array([1.0e12, 2.0e12, -0.7e12])
    T = 9
    one = [(t, _const_state(r0, (0, 0, 0), b)) for t in range(T)]
    two_state = [np.array([r0[0], r0[0] + dr[0]]), np.array([r0[1], r0[1] + dr[1]]),
                 np.array([r0[2], r0[2] + dr[2]])] + [np.zeros(2)] * 3 + \
                [np.full(2, b[0]), np.full(2, b[1]), np.full(2, b[2]), np.ones(2)]
    S1 = _run(oracle_mod, DIRS, OMEGA, DT, one).spectrum()
    S2 = _run(oracle_mod, DIRS, OMEGA, DT, [(t, two_state) for t in range(T)]).spectrum()
    for i, n in enumerate(UNIT):
        for j, om in enumerate(OMEGA):
            fac = 4.0 * np.cos(om * (n @ dr) / (2.0 * C)) ** 2
            assert S2[i, j] == pytest.approx(S1[i, j] * fac, rel=1e-9, abs=1e-14 * S1.max())


# ------------------------------------------------------- P6 linearity and superposition
def _random_steps(rng, n, T, dtype=np.float64):
    out = []
    for t in range(T):
        st = [rng.uniform(0, 5e-6, n) for _ in range(3)] + \
             [rng.uniform(-0.4, 0.4, n) for _ in range(3)] + \
             [rng.uniform(-3e12, 3e12, n) for _ in range(3)] + [rng.uniform(0.5, 2.0, n)]
        out.append((t, [a.astype(dtype) for a in st]))
    return out


def test_p6_linearity_superposition_split_permutation(oracle_mod):
    rng = np.random.default_rng(6)
    steps = _random_steps(rng, 40, 5)
    base = _run(oracle_mod, DIRS, OMEGA, DT, steps)
    A0, S0 = base.amplitude(), base.spectrum()
    # weights scaled by lambda: A -> lambda A, S -> lambda^2 S
    lam = 3.0
    scaled = [(t, st[:9] + [lam * st[9]]) for t, st in steps]
    o = _run(oracle_mod, DIRS, OMEGA, DT, scaled)
    assert np.allclose(o.amplitude(), lam * A0, rtol=1e-13, atol=0)
    assert np.allclose(o.spectrum(), lam ** 2 * S0, rtol=1e-12)
    # particle set split into two calls with the same step_index; and two detectors summed
    o = oracle_mod.Oracle(DIRS, OMEGA, DT, scale=1.0)
    oa = oracle_mod.Oracle(DIRS, OMEGA, DT, scale=1.0)
    ob = oracle_mod.Oracle(DIRS, OMEGA, DT, scale=1.0)
    for t, st in steps:
        o.accumulate_step(t, *[a[:17] for a in st])
        o.accumulate_step(t, *[a[17:] for a in st])
        oa.accumulate_step(t, *[a[:17] for a in st])
        ob.accumulate_step(t, *[a[17:] for a in st])
    tol = 1e-12 * np.abs(A0).max()
    assert np.allclose(o.amplitude(), A0, rtol=0, atol=tol)
    assert np.allclose(oa.amplitude() + ob.amplitude(), A0, rtol=0, atol=tol)
    # permutation of particles and order of steps
    perm = rng.permutation(40)
    o = _run(oracle_mod, DIRS, OMEGA, DT, [(t, [a[perm] for a in st]) for t, st in steps[::-1]])
    assert np.allclose(o.amplitude(), A0, rtol=0, atol=tol)
    # bin subset == same bins of the full run, bit for bit; other bins untouched
    bins = np.array([0, 7, 13, 24])
    sub = _run(oracle_mod, DIRS, OMEGA, DT, steps, bins=bins)
    full = base.A.reshape(-1, 3, 2)
    assert np.array_equal(sub.A.reshape(-1, 3, 2)[bins], full[bins])
    mask = np.ones(full.shape[0], bool)
    mask[bins] = False
    assert np.all(sub.A.reshape(-1, 3, 2)[mask] == 0.0)


def test_p6_f32_state_is_promoted_value_for_value(oracle_mod):
    rng = np.random.default_rng(66)
    steps32 = _random_steps(rng, 20, 3, dtype=np.float32)
    steps64 = [(t, [a.astype(np.float64) for a in st]) for t, st in steps32]
    a32 = _run(oracle_mod, DIRS, OMEGA, DT, steps32).A
    a64 = _run(oracle_mod, DIRS, OMEGA, DT, steps64).A
    assert np.array_equal(a32, a64)


# ------------------------------------------------------- P7 cyclotron (Schott) harmonics
@pytest.mark.parametrize("beta_par", [0.0, 0.05, -0.3])
def test_p7_cyclotron_lines_match_schott_formula(oracle_mod, beta_par):
    """Single helical electron, M whole gyro-periods, integer steps per period: at
    w_m = m w_c / (1 - beta_par cos th) the raw |A|^2 equals
    (2 pi M m)^2 / D^2 [ bp^2 J_m'(x)^2 + ((cos th - beta_par)/sin th)^2 J_m(x)^2 ],
    x = m bp sin th / D  (Schott / Bekefi; SURVEY.md pin P7)."""
    wc, bp, M, spp = 1.0e14, 0.1, 3, 40
    dt = 2.0 * np.pi / wc / spp
    phi0, r0 = 0.83, np.array([0.3e-6, -0.2e-6, 0.6e-6])
    rho = C * bp / wc
    steps = []
    for t in range(M * spp):
        ph = wc * t * dt + phi0
        r = r0 + np.array([rho * (np.sin(ph) - np.sin(phi0)),
                           rho * (-np.cos(ph) + np.cos(phi0)), C * beta_par * t * dt])
        steps.append((t, _const_state(r, (bp * np.cos(ph), bp * np.sin(ph), beta_par),
                                      (-wc * bp * np.sin(ph), wc * bp * np.cos(ph), 0.0))))
    for theta, az in [(0.4, 0.3), (1.1, -2.0), (np.pi / 2, 1.0), (2.5, 0.1)]:
        n = np.array([np.sin(theta) * np.cos(az), np.sin(theta) * np.sin(az), np.cos(theta)])
        D = 1.0 - beta_par * np.cos(theta)
        ms = np.arange(1, 5)
        om = ms * wc / D
        S = _run(oracle_mod, n[None, :], om, dt, steps).spectrum()[0]
        x = ms * bp * np.sin(theta) / D
        ref = (2 * np.pi * M * ms) ** 2 / D ** 2 * (
            bp ** 2 * special.jvp(ms, x) ** 2
            + ((np.cos(theta) - beta_par) / np.sin(theta)) ** 2 * special.jv(ms, x) ** 2)
        assert np.allclose(S, ref, rtol=1e-9)


def test_p7_off_harmonic_frequencies_are_dark(oracle_mod):
    """Between the lines (w = (m+1/2) w_c, whole number of periods M even) the sum over
    periods cancels: |A|^2 is many orders below the neighbouring line."""
    wc, bp, M, spp = 1.0e14, 0.1, 4, 40
    dt = 2.0 * np.pi / wc / spp
    rho = C * bp / wc
    steps = []
    for t in range(M * spp):
        ph = wc * t * dt
        steps.append((t, _const_state((rho * np.sin(ph), -rho * np.cos(ph), 0.0),
                                      (bp * np.cos(ph), bp * np.sin(ph), 0.0),
                                      (-wc * bp * np.sin(ph), wc * bp * np.cos(ph), 0.0))))
    n = np.array([[np.sin(1.0), 0.0, np.cos(1.0)]])
    S = _run(oracle_mod, n, np.array([1.0, 1.5, 2.0, 2.5]) * wc, dt, steps).spectrum()[0]
    assert S[1] < 1e-20 * S[0] and S[3] < 1e-20 * S[2]


# --------------------------------------------------------------------- P8 brute force
def test_p8_bruteforce_numpy_complex128(oracle_mod):
    rng = np.random.default_rng(8)
    T, N = 6, 12
    steps = _random_steps(rng, N, T)
    t0 = 1.1e-16
    o = _run(oracle_mod, DIRS, OMEGA, DT, steps, t0=t0)
    ref = np.zeros((len(DIRS), len(OMEGA), 3), dtype=np.complex128)
    for t, st in steps:
        r, be, bd, w = np.stack(st[0:3], 1), np.stack(st[3:6], 1), np.stack(st[6:9], 1), st[9]
        for i, n in enumerate(UNIT):
            for k in range(N):
                vec = np.cross(n, np.cross(n - be[k], bd[k]))
                a = w[k] * vec / (1.0 - be[k] @ n) ** 2
                tret = t0 + t * DT - (n @ r[k]) / C
                ref[i] += a[None, :] * np.exp(1j * OMEGA * tret)[:, None] * DT
    assert np.allclose(o.amplitude(), ref, rtol=0, atol=1e-12 * np.abs(ref).max())
    assert np.allclose(o.spectrum(), (np.abs(ref) ** 2).sum(-1), rtol=1e-11)


def test_p8_bruteforce_mpmath_tiny(oracle_mod):
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 40
    rng = np.random.default_rng(88)
    steps = _random_steps(rng, 2, 3)
    dirs, om = DIRS[2:4], OMEGA[3:5]          # the large-phase bins
    o = _run(oracle_mod, dirs, om, DT, steps)
    for i, nraw in enumerate(dirs):
        nn = [mp.mpf(float(v)) for v in nraw]
        nrm = mp.sqrt(sum(v * v for v in nn))
        n = [v / nrm for v in nn]
        for j, w_j in enumerate(om):
            acc = [mp.mpc(0)] * 3
            for t, st in steps:
                for k in range(2):
                    r, be, bd = ([mp.mpf(float(st[c + o3][k])) for c in range(3)] for o3 in (0, 3, 6))
                    wk = mp.mpf(float(st[9][k]))
                    d = 1 - sum(be[c] * n[c] for c in range(3))
                    g = [n[c] - be[c] for c in range(3)]
                    inner = [g[1] * bd[2] - g[2] * bd[1], g[2] * bd[0] - g[0] * bd[2],
                             g[0] * bd[1] - g[1] * bd[0]]
                    outer = [n[1] * inner[2] - n[2] * inner[1], n[2] * inner[0] - n[0] * inner[2],
                             n[0] * inner[1] - n[1] * inner[0]]
                    tau = mp.mpf(t) * mp.mpf(DT) - sum(n[c] * r[c] for c in range(3)) / mp.mpf(C)
                    ph = mp.expj(mp.mpf(float(w_j)) * tau)
                    for c in range(3):
                        acc[c] += wk * mp.mpf(DT) * outer[c] / d ** 2 * ph
            got = o.amplitude()[i, j]
            scale = max(abs(complex(a)) for a in acc)
            for c in range(3):
                assert abs(got[c] - complex(acc[c])) <= 1e-11 * scale


# ------------------------------------------------------------------------ P9 SI constant
def test_p9_default_scale_is_e2_over_16pi3eps0c(oracle_mod):
    assert oracle_mod.default_scale() == pytest.approx(1.949313784587704e-38, rel=1e-9)
    # scale == 0 selects it
    st = _const_state((0, 0, 0), (0, 0, 0), (1e12, 0, 0))
    s_default = _run(oracle_mod, DIRS, OMEGA, DT, [(0, st)], scale=0.0).spectrum()
    s_unit = _run(oracle_mod, DIRS, OMEGA, DT, [(0, st)], scale=1.0).spectrum()
    assert np.allclose(s_default, s_unit * 1.949313784587704e-38, rtol=1e-9)


# ----------------------------------------------------------------- P10 Larmor / Parseval
def test_p10_frequency_integral_matches_angular_power(oracle_mod):
    """int_0^inf S dw = pi * sum_t |n x ((n-beta) x betadot)|^2/(1-beta.n)^5 dt  (raw scale=1),
    the retarded-time power law (Jackson 14.38): pins the (1-beta.n) powers jointly with P4."""
    wc, bp, bz, M, spp = 1.0e14, 0.3, 0.2, 4, 1024
    dt = 2.0 * np.pi / wc / spp
    rho = C * bp / wc
    n = np.array([np.sin(0.9) * np.cos(0.4), np.sin(0.9) * np.sin(0.4), np.cos(0.9)])
    steps, power = [], 0.0
    for t in range(M * spp):
        ph = wc * t * dt
        be = np.array([bp * np.cos(ph), bp * np.sin(ph), bz])
        bd = np.array([-wc * bp * np.sin(ph), wc * bp * np.cos(ph), 0.0])
        r = np.array([rho * np.sin(ph), -rho * np.cos(ph), C * bz * t * dt])
        steps.append((t, _const_state(r, be, bd)))
        d = 1.0 - be @ n
        vec = (n - be) * (n @ bd) - bd * d
        power += (vec @ vec) / d ** 5 * dt
        if t == 0:
            jump2 = (vec @ vec) / d ** 6       # |a(tau)|^2 at the window edge, a(tau)=vec/d^3
    # dense linear grid well past the highest significant harmonic; lines have width
    # ~ w_c/M, resolved with w_c/(16 M) spacing
    om = np.arange(1, 16 * M * 40 + 1) * (wc / (16.0 * M))
    S = _run(oracle_mod, n[None, :], om, dt, steps).spectrum()[0]
    dw = om[1] - om[0]
    # the rectangular time window gives |A|^2 a (|J0|^2+|J1|^2)/w^2 tail (J = jump of the
    # observer-time signal at either edge; equal by periodicity): add it beyond the grid
    integral = np.sum(S) * dw + 2.0 * jump2 / (om[-1] + 0.5 * dw)
    assert integral == pytest.approx(np.pi * power, rel=2e-4)


# ------------------------------------------------- P11 per-region detectors (NEXT-2)
def _region_case(rng, T=4, sizes=(5, 0, 9, 1, 7)):
    off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    return off, _random_steps(rng, int(off[-1]), T)


def test_p11_regions_sum_to_the_global_detector_and_are_independent(oracle_mod):
    """A_r = the sum over the particles of region r: (i) sum_r A_r = A of all particles,
    (ii) an empty region is exactly zero, (iii) region r equals a plain detector fed only
    region r's particles, (iv) changing the particles of one region leaves the others alone,
    (v) the total spectrum is |sum_r A_r|^2, not sum_r |A_r|^2."""
    rng = np.random.default_rng(11)
    off, steps = _region_case(rng)
    R = len(off) - 1
    ro = oracle_mod.RegionOracle(R, DIRS, OMEGA, DT, t0=2e-17, scale=1.0)
    for t, st in steps:
        ro.accumulate_step(t, off, *st)
    glob = _run(oracle_mod, DIRS, OMEGA, DT, steps, t0=2e-17)
    A = ro.amplitude()
    scale = np.abs(glob.amplitude()).max()
    assert np.allclose(A.sum(0), glob.amplitude(), rtol=0, atol=1e-13 * scale)
    assert np.all(ro.A[1] == 0.0)
    for r in range(R):
        sub = [(t, [a[off[r]:off[r + 1]] for a in st]) for t, st in steps]
        assert np.array_equal(A[r], _run(oracle_mod, DIRS, OMEGA, DT, sub, t0=2e-17).amplitude())
    assert np.allclose(ro.spectrum_total(), glob.spectrum(), rtol=1e-11)
    assert not np.allclose(ro.spectrum().sum(0), glob.spectrum(), rtol=1e-3)
    # (iv)
    steps2 = [(t, [a.copy() for a in st]) for t, st in steps]
    for t, st in steps2:
        st[6][off[2]:off[3]] *= -3.0
    ro2 = oracle_mod.RegionOracle(R, DIRS, OMEGA, DT, t0=2e-17, scale=1.0)
    for t, st in steps2:
        ro2.accumulate_step(t, off, *st)
    for r in (0, 1, 3, 4):
        assert np.array_equal(ro2.A[r], ro.A[r])
    assert not np.allclose(ro2.A[2], ro.A[2])


def test_p11_regions_bruteforce_masked_numpy(oracle_mod):
    """Independent formulation: one pass over ALL particles with a region-membership mask
    (no slicing), numpy complex128; offsets[0] > 0 and a tail beyond offsets[-1] are skipped."""
    rng = np.random.default_rng(111)
    T, N = 3, 20
    steps = _random_steps(rng, N, T)
    off = np.array([2, 6, 6, 13, 17], dtype=np.int64)          # particles 0,1 and 17..19 in no region
    R = len(off) - 1
    rid = np.full(N, -1)
    for r in range(R):
        rid[off[r]:off[r + 1]] = r
    ro = oracle_mod.RegionOracle(R, DIRS, OMEGA, DT, scale=1.0)
    ref = np.zeros((R, len(DIRS), len(OMEGA), 3), dtype=np.complex128)
    for t, st in steps:
        ro.accumulate_step(t, off, *st)
        r_, be, bd, w = np.stack(st[0:3], 1), np.stack(st[3:6], 1), np.stack(st[6:9], 1), st[9]
        for i, n in enumerate(UNIT):
            vec = np.cross(n, np.cross(n - be, bd))                       # [N,3]
            a = w[:, None] * vec / (1.0 - be @ n)[:, None] ** 2
            ph = np.exp(1j * OMEGA[None, :] * (t * DT - (r_ @ n) / C)[:, None])   # [N,W]
            for r in range(R):
                m = (rid == r).astype(float)
                ref[r, i] += np.einsum("k,kc,kw->wc", m, a, ph) * DT
    assert np.allclose(ro.amplitude(), ref, rtol=0, atol=1e-12 * np.abs(ref).max())
    assert np.allclose(ro.spectrum(), (np.abs(ref) ** 2).sum(-1), rtol=1e-11, atol=0)


def test_p11_regions_bin_subset_and_f32(oracle_mod):
    rng = np.random.default_rng(112)
    off, steps = _region_case(rng, T=2)
    steps32 = [(t, [a.astype(np.float32) for a in st]) for t, st in steps]
    R = len(off) - 1
    full = oracle_mod.RegionOracle(R, DIRS, OMEGA, DT, scale=1.0)
    bins = np.array([1, len(OMEGA) + 2, 3 * len(OMEGA) - 1], dtype=np.int64)
    sub = oracle_mod.RegionOracle(R, DIRS, OMEGA, DT, scale=1.0, bins=bins)
    for t, st in steps32:
        full.accumulate_step(t, off, *st)
        sub.accumulate_step(t, off, *st)
    Sf, Ss = full.spectrum().reshape(R, -1), sub.spectrum().reshape(R, -1)
    assert np.array_equal(Sf[:, bins], Ss[:, bins])
    mask = np.ones(Sf.shape[1], bool); mask[bins] = False
    assert np.all(Ss[:, mask] == 0.0)
    # fp32 state is promoted value for value
    steps64 = [(t, [a.astype(np.float64) for a in st]) for t, st in steps32]
    f64 = oracle_mod.RegionOracle(R, DIRS, OMEGA, DT, scale=1.0)
    for t, st in steps64:
        f64.accumulate_step(t, off, *st)
    assert np.array_equal(f64.A, full.A)


# ------------------------------------------------- P12 spatial window (NEXT-3, reading W1)
def _win_np(kind, u):
    inside = (u >= 0.0) & (u <= 1.0)
    val = 1.0 - np.abs(2.0 * u - 1.0) if kind == "triangle" else 0.54 - 0.46 * np.cos(2.0 * np.pi * u)
    return np.where(inside, val, 0.0)


@pytest.mark.parametrize("kind,u,expect", [("triangle", 0.25, 0.5), ("triangle", 0.5, 1.0), ("triangle", 0.9, 0.2),
                                            ("hamming", 0.5, 1.0), ("hamming", 0.25, 0.54), ("hamming", 0.0, 0.08),
                                            ("triangle", 1.0000001, 0.0), ("hamming", -1e-9, 0.0)])
def test_p12_window_value_scales_the_dirichlet_kernel(oracle_mod, kind, u, expect):
    """Static particle (pin P2) inside a box window along x only: |A|^2 = W(u)^2 x the Dirichlet
    kernel; w1 has the textbook values (triangle 1-|2u-1|, Hamming 0.54-0.46 cos 2 pi u), and a
    particle outside the box contributes exactly nothing."""
    L, o = 4e-6, -1e-6
    r0 = (o + u * L, 7e-7, -3e-7)
    b = np.array([1.0e13, -2.0e13, 0.5e13])
    T = 9
    steps = [(t, _const_state(r0, (0, 0, 0), b, w=1.7)) for t in range(T)]
    win = (kind, (o, 0.0, 0.0), (L, 0.0, -1.0))            # y, z: extent <= 0 -> not windowed
    ow = oracle_mod.Oracle(DIRS, OMEGA, DT, scale=1.0, window=win)
    for t, st in steps:
        ow.accumulate_step(t, *st)
    S0 = _run(oracle_mod, DIRS, OMEGA, DT, steps).spectrum()
    if expect == 0.0:
        assert np.all(ow.A == 0.0)
    else:
        assert np.allclose(ow.spectrum(), expect ** 2 * S0, rtol=1e-9 if u != 0.0 else 1e-6)
        n = UNIT[2]
        x = OMEGA * DT / 2
        closed = (1.7 * expect) ** 2 * (b @ b - (n @ b) ** 2) * DT ** 2 * (np.sin(T * x) / np.sin(x)) ** 2
        assert np.allclose(ow.spectrum()[2], closed, rtol=1e-8)


def test_p12_window_equals_reweighting_and_none_is_identity(oracle_mod):
    """Windowed oracle == plain oracle fed w * W(r) computed here in numpy (product over the
    windowed axes, positions of each step); type none / zero extents are the identity."""
    rng = np.random.default_rng(12)
    steps = _random_steps(rng, 40, 3)
    o, L = np.array([-2e-6, -1e-6, -4e-6]), np.array([5e-6, 3e-6, 0.0])   # some particles fall outside
    for kind in ("triangle", "hamming"):
        ow = oracle_mod.Oracle(DIRS, OMEGA, DT, scale=1.0, window=(kind, o, L))
        steps_rw = []
        for t, st in steps:
            ow.accumulate_step(t, *st)
            W = np.ones(40)
            for c in range(2):
                W = W * _win_np(kind, (st[c] - o[c]) / L[c])
            steps_rw.append((t, st[:9] + [st[9] * W]))
        ref = _run(oracle_mod, DIRS, OMEGA, DT, steps_rw)
        assert np.allclose(ow.A, ref.A, rtol=0, atol=1e-13 * np.abs(ref.A).max())
        assert 0 < np.count_nonzero(_win_np(kind, (steps[0][1][0] - o[0]) / L[0]) == 0.0) < 40
    plain = _run(oracle_mod, DIRS, OMEGA, DT, steps)
    for win in (("none", o, L), ("triangle", o, np.zeros(3))):
        ow = oracle_mod.Oracle(DIRS, OMEGA, DT, scale=1.0, window=win)
        for t, st in steps:
            ow.accumulate_step(t, *st)
        assert np.array_equal(ow.A, plain.A)
    # per-region oracle takes the same window
    off = np.array([0, 15, 40], dtype=np.int64)
    ro = oracle_mod.RegionOracle(2, DIRS, OMEGA, DT, scale=1.0, window=("hamming", o, L))
    ow = oracle_mod.Oracle(DIRS, OMEGA, DT, scale=1.0, window=("hamming", o, L))
    for t, st in steps:
        ro.accumulate_step(t, off, *st)
        ow.accumulate_step(t, *st)
    assert np.allclose(ro.A.sum(0), ow.A, rtol=0, atol=1e-13 * np.abs(ow.A).max())


# ------------------------------------------------- P13 Nyquist limiter (NEXT-3, reading N1)
def test_p13_nyquist_static_particle_loses_exactly_the_undersampled_bins(oracle_mod):
    """beta = 0 (1 - beta.n = 1): bins with w dt >= pi nu vanish exactly, the others keep the
    Dirichlet closed form; nu = 0 and a huge nu leave everything in place."""
    b = np.array([1.0e13, -2.0e13, 0.5e13])
    T = 7
    steps = [(t, _const_state((1e-7, 2e-7, 3e-7), (0, 0, 0), b)) for t in range(T)]
    plain = _run(oracle_mod, DIRS, OMEGA, DT, steps).spectrum()
    nu = 0.1                                                   # pi nu / dt = 1.57e16 rad/s
    cut = OMEGA * DT >= np.pi * nu
    assert cut.tolist() == [False, False, False, False, True]
    o = oracle_mod.Oracle(DIRS, OMEGA, DT, scale=1.0, nyquist=nu)
    for t, st in steps:
        o.accumulate_step(t, *st)
    S = o.spectrum()
    assert np.all(S[:, cut] == 0.0) and np.array_equal(S[:, ~cut], plain[:, ~cut])
    x = OMEGA * DT / 2
    closed = (b @ b - (UNIT[3] @ b) ** 2) * DT ** 2 * (np.sin(T * x) / np.sin(x)) ** 2
    assert np.allclose(S[3, ~cut], closed[~cut], rtol=1e-9)
    for nu_off in (0.0, 1e9):
        o2 = oracle_mod.Oracle(DIRS, OMEGA, DT, scale=1.0, nyquist=nu_off)
        for t, st in steps:
            o2.accumulate_step(t, *st)
        assert np.array_equal(o2.spectrum(), plain)
    # the limiter setting of one oracle object does not leak into the next call of another
    assert np.array_equal(_run(oracle_mod, DIRS, OMEGA, DT, steps).spectrum(), plain)


def test_p13_nyquist_cutoff_is_doppler_shifted_by_direction(oracle_mod):
    """Particle moving with beta = 0.9 x: towards the observer (n = +x) 1 - beta.n = 0.1, so the
    cut-off frequency pi nu / (dt (1 - beta.n)) is 19x higher than for n = -x.  Kept bins equal
    pin P4's closed form, and a second, static particle is limited by its own factor only."""
    beta = np.array([0.9, 0.0, 0.0])
    b = np.array([0.0, 3.0e13, 1.0e13])
    r0 = np.array([1e-7, -2e-7, 0.5e-7])
    T, nu = 6, 0.05
    dirs = np.array([[1.0, 0, 0], [-1.0, 0, 0], [0, 1.0, 0]])
    mov = [(t, _const_state(r0 + beta * C * t * DT, beta, b)) for t in range(T)]
    o = oracle_mod.Oracle(dirs, OMEGA, DT, scale=1.0, nyquist=nu)
    for t, st in mov:
        o.accumulate_step(t, *st)
    S = o.spectrum()
    for i, n in enumerate(dirs):
        d = 1.0 - beta @ n
        cut = OMEGA * DT * d >= np.pi * nu
        vec = np.cross(n, np.cross(n - beta, b))
        xp = OMEGA * d * DT / 2
        closed = (vec @ vec) / d ** 4 * DT ** 2 * (np.sin(T * xp) / np.sin(xp)) ** 2
        assert np.all(S[i, cut] == 0.0)
        assert np.allclose(S[i, ~cut], closed[~cut], rtol=1e-8)
    assert np.count_nonzero(S[0]) > np.count_nonzero(S[1])        # forward keeps more bins than backward
    # add a static particle: where the mover is cut, the sum equals the static particle alone
    both = [(t, [np.concatenate([a, s]) for a, s in zip(st, _const_state(-r0, (0, 0, 0), 2 * b))]) for t, st in mov]
    stat = [(t, _const_state(-r0, (0, 0, 0), 2 * b)) for t in range(T)]
    ob = oracle_mod.Oracle(dirs, OMEGA, DT, scale=1.0, nyquist=nu)
    os_ = oracle_mod.Oracle(dirs, OMEGA, DT, scale=1.0, nyquist=nu)
    for (t, s2), (_, s1) in zip(both, stat):
        ob.accumulate_step(t, *s2)
        os_.accumulate_step(t, *s1)
    cut_mov = OMEGA * DT * 1.9 >= np.pi * nu                     # direction -x
    assert np.allclose(ob.spectrum()[1, cut_mov], os_.spectrum()[1, cut_mov], rtol=1e-12)


# ---------------------------------------------- P14 macro-particle form factor (reading FF1)
# g_k(n, w) = sqrt(w_k + (w_k^2 - w_k) F^2(n, w)); the pins below fix everything the
# mathematics fixes about it: both limits, the interpolation between them in closed form for two
# shapes, the direction dependence, and the order "form factor first, window after".
def _ff_run(oracle_mod, dirs, omega, dt, steps, form_factor, **kw):
    o = oracle_mod.Oracle(dirs, omega, dt, scale=1.0, form_factor=form_factor, **kw)
    for t, st in steps:
        o.accumulate_step(t, *st)
    return o


def _ff_steps(rng, n, T, wmax=None):
    steps = []
    w = np.ones(n) if wmax is None else 10.0 ** rng.uniform(0, np.log10(wmax), n)
    for t in range(T):
        st = [rng.uniform(0, 2e-6, n) for _ in range(3)] + [rng.uniform(-0.4, 0.4, n) for _ in range(3)] \
            + [rng.normal(0, 1e13, n) for _ in range(3)] + [w]
        steps.append((t, st))
    return steps


@pytest.mark.parametrize("ff", [("gaussian", (3e-8, 1e-8, 2e-8)), ("cic", (5e-8, 5e-8, 5e-8)),
                                ("incoherent", (0, 0, 0))])
def test_p14_unit_weight_is_the_identity_bit_for_bit(oracle_mod, ff):
    """w = 1: g = sqrt(1 + 0 * F^2) = 1 exactly, whatever the shape."""
    steps = _ff_steps(np.random.default_rng(141), 40, 3)
    a = _ff_run(oracle_mod, DIRS, OMEGA, DT, steps, ff)
    b = _run(oracle_mod, DIRS, OMEGA, DT, steps)
    assert np.array_equal(a.A, b.A)


@pytest.mark.parametrize("ff", [("gaussian", (0, 0, 0)), ("cic", (0, 0, 0))])
def test_p14_point_particle_limit_is_the_coherent_sum(oracle_mod, ff):
    """Zero size: F = 1, g = sqrt(w^2) = w -> today's fully coherent sum (amplitude linear in w)."""
    steps = _ff_steps(np.random.default_rng(142), 30, 2, wmax=1e4)
    a = _ff_run(oracle_mod, DIRS, OMEGA, DT, steps, ff)
    b = _run(oracle_mod, DIRS, OMEGA, DT, steps)
    assert np.abs(a.A - b.A).max() <= 1e-13 * np.abs(b.A).max()


def test_p14_incoherent_limit_intensity_is_linear_in_the_weight(oracle_mod):
    """F = 0: one macro-particle of weight w radiates w times (not w^2 times) one particle; the
    same at huge size for the Gaussian shape (F underflows to 0)."""
    rng = np.random.default_rng(143)
    (t, st), = _ff_steps(rng, 1, 1)
    S1 = _run(oracle_mod, DIRS, OMEGA, DT, [(0, st)]).spectrum()
    for wgt in (4.0, 1234.5):
        stw = st[:9] + [np.array([wgt])]
        Sw = _ff_run(oracle_mod, DIRS, OMEGA, DT, [(0, stw)], ("incoherent", (0, 0, 0))).spectrum()
        assert np.allclose(Sw, wgt * S1, rtol=1e-13)
        Sg = _ff_run(oracle_mod, DIRS, OMEGA, DT, [(0, stw)], ("gaussian", (1.0, 1.0, 1.0))).spectrum()
        assert np.allclose(Sg, wgt * S1, rtol=1e-13)
        Sc = _run(oracle_mod, DIRS, OMEGA, DT, [(0, stw)]).spectrum()      # coherent, for contrast
        assert np.allclose(Sc, wgt ** 2 * S1, rtol=1e-13)


def test_p14_gaussian_shape_times_dirichlet_closed_form(oracle_mod):
    """Static macro-particle, constant betadot b, T steps (pin P2's set-up):
    S = g^2 (|b|^2 - (n.b)^2) dt^2 sin^2(wT dt/2)/sin^2(w dt/2), g^2 = w + (w^2 - w) exp(-sum_c (w n_c s_c/c)^2)
    with an ANISOTROPIC Gaussian, so the value depends on the direction through n_c s_c."""
    T, wgt = 17, 250.0
    b = np.array([2.0e12, -1.0e12, 3.0e12])
    sig = np.array([4.0e-8, 1.0e-8, 2.5e-8])
    st = _const_state([1e-7, 2e-7, -1e-7], [0, 0, 0], b, w=wgt)
    o = _ff_run(oracle_mod, DIRS, OMEGA, DT, [(t, st) for t in range(T)], ("gaussian", sig))
    S = o.spectrum()
    saw_intermediate = False
    for i, n in enumerate(UNIT):
        for j, om in enumerate(OMEGA):
            F2 = np.exp(-np.sum((om * n * sig / C) ** 2))
            g2 = wgt + (wgt ** 2 - wgt) * F2
            expect = g2 * (b @ b - (n @ b) ** 2) * DT ** 2 * _dirichlet(om * DT, T) ** 2
            assert S[i, j] == pytest.approx(expect, rel=1e-11)
            saw_intermediate |= 0.05 < F2 < 0.95
    assert saw_intermediate           # the grid really samples the transition, not only the two limits


def test_p14_cic_shape_first_zero_and_textbook_values(oracle_mod):
    """CIC (triangular) shape of cell size D along x, observed along x: F = sinc^2(w D / 2c).
    At w D / 2c = pi the shape factor vanishes (fully incoherent, g^2 = w); at pi/2 it is
    (2/pi)^2, F^2 = (2/pi)^4; at 0+ it is 1."""
    wgt, D = 100.0, 6.0e-8
    n = np.array([[1.0, 0.0, 0.0]])
    om = np.array([2e-6 * C / D, np.pi * C / D, 2 * np.pi * C / D])               # x = w D/2c = 1e-6, pi/2, pi
    b = np.array([0.0, 1.0e12, 0.0])
    st = _const_state([0, 0, 0], [0, 0, 0], b, w=wgt)
    dt = 1e-19
    S = _ff_run(oracle_mod, n, om, dt, [(0, st)], ("cic", (D, 7 * D, 9 * D))).spectrum()[0]   # y, z sizes: n_y = n_z = 0
    base = (b @ b) * dt ** 2
    assert S[0] == pytest.approx(wgt ** 2 * base, rel=1e-10)
    assert S[1] == pytest.approx((wgt + (wgt ** 2 - wgt) * (2 / np.pi) ** 4) * base, rel=1e-12)
    assert S[2] == pytest.approx(wgt * base, rel=1e-9)      # sin(pi) ~ 1e-16: F^2 ~ 1e-64


def test_p14_bruteforce_numpy_with_window(oracle_mod):
    """Independent numpy complex128 evaluation of the whole sum with g_k(n, w) and a window:
    the form factor acts on the macro weight, the window multiplies afterwards."""
    rng = np.random.default_rng(145)
    n_p, T = 12, 3
    steps = _ff_steps(rng, n_p, T, wmax=1e3)
    size = np.array([2e-8, 3e-8, 1e-8])
    win = ("triangle", (0.0, 0.0, 0.0), (2e-6, 0.0, 2e-6))
    for kind in ("gaussian", "cic"):
        o = _ff_run(oracle_mod, DIRS, OMEGA, DT, steps, (kind, size), window=win)
        A = np.zeros((len(UNIT), len(OMEGA), 3), dtype=np.complex128)
        for t, st in steps:
            r, be, bd, w = np.stack(st[0:3], 1), np.stack(st[3:6], 1), np.stack(st[6:9], 1), st[9]
            u = r / np.array([2e-6, 1.0, 2e-6])
            Wn = (1 - np.abs(2 * u[:, 0] - 1)) * (1 - np.abs(2 * u[:, 2] - 1))
            for i, n in enumerate(UNIT):
                d = 1 - be @ n
                vec = np.cross(n, np.cross(n - be, bd))
                tau = t * DT - r @ n / C
                for j, om in enumerate(OMEGA):
                    if kind == "gaussian":
                        F = np.exp(-0.5 * np.sum((om * n * size / C) ** 2))
                    else:
                        F = np.prod(np.sinc(om * n * size / (2 * C) / np.pi) ** 2)
                    g = np.sqrt(w + (w * w - w) * F * F)
                    A[i, j] += ((g * Wn * DT / d ** 2 * np.exp(1j * om * tau))[:, None] * vec).sum(0)
        assert np.abs(o.amplitude() - A).max() <= 1e-12 * np.abs(A).max()


def test_p14_regions_and_bad_arguments(oracle_mod):
    rng = np.random.default_rng(146)
    steps = _ff_steps(rng, 20, 2, wmax=50)
    ff = ("gaussian", (2e-8, 2e-8, 2e-8))
    off = np.array([0, 7, 7, 20])
    ro = oracle_mod.RegionOracle(3, DIRS, OMEGA, DT, scale=1.0, form_factor=ff)
    for t, st in steps:
        ro.accumulate_step(t, off, *st)
    whole = _ff_run(oracle_mod, DIRS, OMEGA, DT, steps, ff)
    assert np.abs(ro.A.sum(axis=0) - whole.A).max() <= 1e-13 * np.abs(whole.A).max()
    assert np.allclose(ro.spectrum_total(), whole.spectrum(), rtol=1e-12)
    with pytest.raises(KeyError):
        oracle_mod.Oracle(DIRS, OMEGA, DT, form_factor=("box", (1, 1, 1)))
