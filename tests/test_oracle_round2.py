"""Pins of the oracle functions added in round 2 (CPU only, -m "not gpu"): per-event C^-1 with a position-dependent
sigma_z, the exact theta-integrated kernel (8(f4)), the direct-reconstruction histogram (8(f2)) and the
counter-based event generator (8(f4)).  As in test_oracle_pins.py no test retypes an oracle formula: expected values
come from the detector forward model, closed forms, published known answers, invariants and the independent numpy
generator of paper_1502_07478_b200.synth."""
import math
import os

import numpy as np
import pytest

from paper_1502_07478_b200 import synth
from test_oracle_pins import R, L, forward, laplace_from_forward_model

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


@pytest.fixture
def eta(oracle):
    oracle.set_sigma_z_edge(0.1)
    yield 0.1
    oracle.set_sigma_z_edge(0.0)
    oracle.set_gamma(0.0)
    oracle.set_exact_kernel(0)


# ------------------------------------------------------------------------------------------------------
# sigma_z(z~u, z~d): PAPER.md:124, reading R22
# ------------------------------------------------------------------------------------------------------
def test_sigma_z_is_lowest_at_the_centre_and_ten_percent_higher_at_the_edge(oracle, eta):
    """"on the order of 10% from the center (lowest) to the edge (highest)"."""
    sz = 10.0
    assert oracle.sigma_z_at(0.0, L, sz) == sz
    assert oracle.sigma_z_at(0.5 * L, L, sz) == pytest.approx(1.1 * sz, rel=1e-15)
    assert oracle.sigma_z_at(-0.5 * L, L, sz) == pytest.approx(1.1 * sz, rel=1e-15)
    assert oracle.sigma_z_at(0.9 * L, L, sz) == pytest.approx(1.1 * sz, rel=1e-15)        # smeared past the strip end: edge value
    zs = np.linspace(0, 0.5 * L, 50)
    v = np.array([oracle.sigma_z_at(z, L, sz) for z in zs])
    assert (np.diff(v) > 0).all() and (v >= sz).all()
    assert [oracle.sigma_z_at(z, L, sz) for z in (-30, -120)] == [oracle.sigma_z_at(z, L, sz) for z in (30, 120)]
    oracle.set_sigma_z_edge(0.0)
    assert oracle.sigma_z_at(200.0, L, sz) == sz                                           # the paper's constant case


def test_cinv_is_eq12_with_each_strips_own_sigma_z(oracle, eta):
    gamma = 0.2 / (math.sqrt(2) * 10 * 40)
    oracle.set_gamma(gamma)
    C = oracle.cinv(200.0, -50.0, L, 10.0, 40.0)
    su, sd = oracle.sigma_z_at(200.0, L, 10.0), oracle.sigma_z_at(-50.0, L, 10.0)
    assert su > sd > 10.0
    want = np.array([[1 / su**2, 0, gamma], [0, 1 / sd**2, -gamma], [gamma, -gamma, 1 / 40.0**2]])   # Eq. 12
    assert np.allclose(C, want, rtol=1e-15, atol=0)
    assert np.all(np.linalg.eigvalsh(C) > 0)


def test_kernel_with_per_event_matrix_is_the_saddle_point_of_the_forward_model(oracle, eta):
    """Eq. 7 with C^-1 = diag(1/sigma_z(z~u)^2, 1/sigma_z(z~d)^2, 1/sigma_dl^2) (+ gamma) against the second-order Laplace
    value built from the forward model with that matrix.  With unequal first two entries the (y - R) and (y + R)
    components of a and o no longer combine to y^2 + R^2: a sign or an index error there fails this pin."""
    rng = np.random.default_rng(23)
    for sz, sdl in [(10, 40), (5, 20), (20, 80)]:
        for frac in (0.0, 0.3):
            gamma = frac / (math.sqrt(2.0) * 1.1 * sz * sdl)
            oracle.set_gamma(gamma)
            worst, moved = 0.0, 0.0
            for _ in range(80):
                ev = forward(rng.uniform(-220, 220), rng.uniform(-150, 150), rng.uniform(-0.5, 0.5))
                ev = ev + rng.normal(size=3) * np.array([sz, sz, sdl])
                tan_t, y_t, z_t = oracle.eq2(*ev, R)
                y, z = y_t + rng.uniform(-1.4, 1.4) * sdl, z_t + rng.uniform(-2, 2) * sz
                C = oracle.cinv(ev[0], ev[1], L, sz, sdl)
                want = laplace_with_matrix(ev, y, z, C)
                got = oracle.kernel_c(y, z, tan_t, y_t, z_t, R, C, 2.0)
                worst = max(worst, abs(got / want - 1.0))
                moved = max(moved, abs(laplace_from_forward_model(ev, y, z, sz, sdl, gamma=gamma) / want - 1.0))
                b = forward(y, z, math.atan(tan_t)) - ev
                assert abs(b @ C @ b - oracle.bCb_c(y - y_t, z - z_t, tan_t, C)) < 1e-8
            assert worst < 2e-7, (sz, sdl, frac, worst)
            assert moved > 1e-2                    # the position dependence moves the kernel far beyond the pin's resolution


def laplace_with_matrix(ev, y, z, Cinv):
    """laplace_from_forward_model (test_oracle_pins.py) for an arbitrary inverse covariance matrix."""
    theta_t = math.atan((ev[0] - ev[1]) / (2.0 * R))
    h = 1e-3
    e0 = forward(y, z, theta_t)
    ep, em = forward(y, z, theta_t + h), forward(y, z, theta_t - h)
    ep2, em2 = forward(y, z, theta_t + 2 * h), forward(y, z, theta_t - 2 * h)
    a = (-ep2 + 8 * ep - 8 * em + em2) / (12 * h)
    o = 0.5 * (-ep2 + 16 * ep - 30 * e0 + 16 * em - em2) / (12 * h * h)
    b = e0 - np.asarray(ev, float)
    D = a @ Cinv @ a + 2.0 * (o @ Cinv @ b)
    expo = -0.5 * (b @ Cinv @ b - (b @ Cinv @ a) ** 2 / D)
    return math.sqrt(np.linalg.det(Cinv)) / (2.0 * math.pi) ** 1.5 * math.sqrt(2.0 * math.pi / D) * math.exp(expo) / math.pi


@pytest.mark.parametrize("tan_t", [0.0, 0.3, -0.55])
def test_bbox_of_the_per_event_ellipse(oracle, eta, tan_t):
    """App. B for a general matrix: the half extents are the largest |dy|, |dz| on b C^-1 b = 9 (brute boundary scan)."""
    C = oracle.cinv(230.0, -40.0, L, 10.0, 40.0)
    hy, hz = oracle.bbox_half_extents_c(tan_t, C)
    phi = np.linspace(0, 2 * math.pi, 20001)
    best_y = best_z = 0.0
    for c, s in zip(np.cos(phi), np.sin(phi)):
        r = 3.0 / math.sqrt(oracle.bCb_c(c, s, tan_t, C))       # the form is quadratic: scale the direction onto the ellipse
        best_y, best_z = max(best_y, abs(r * c)), max(best_z, abs(r * s))
    assert best_y == pytest.approx(hy, rel=1e-6) and best_z == pytest.approx(hz, rel=1e-6)


def test_mlem_with_position_dependent_sigma_z_equals_dense_eq3(oracle, eta):
    """Listing 1 with per-event matrices against a dense transcription of Eq. 3 whose P comes from kernel_c (pinned above)."""
    n_y, n_z, pixel, sz, sdl = 12, 10, 14.0, 10.0, 40.0
    cfg = synth.CONFIGS["cfg1"]
    ev = synth.generate_events(cfg.phantom, 50, R, L, sz, sdl, seed=9) * np.float32(0.5)
    ev[:, :2] += np.float32(120.0)                              # hits away from the strip centre: sigma_u != sigma_d
    rho = np.random.default_rng(1).uniform(0.5, 2.0, (n_y, n_z))
    ys = (np.arange(n_y) - 0.5 * (n_y - 1)) * pixel
    zs = (np.arange(n_z) - 0.5 * (n_z - 1)) * pixel
    s = oracle.sensitivity_image(R, L, n_y, n_z, pixel).ravel()
    P = np.zeros((len(ev), n_y * n_z))
    for j, e in enumerate(ev.astype(np.float64)):
        tan_t, y_t, z_t = oracle.eq2(*e, R)
        C = oracle.cinv(e[0], e[1], L, sz, sdl)
        for iy, y in enumerate(ys):
            for iz, z in enumerate(zs):
                if oracle.bCb_c(y - y_t, z - z_t, tan_t, C) <= 9.0:
                    P[j, iy * n_z + iz] = oracle.kernel_c(y, z, tan_t, y_t, z_t, R, C)
    denom = P @ (s * rho.ravel())
    ok = denom > 0
    want = rho.ravel() * (P[ok] / denom[ok, None]).sum(axis=0)
    want[s <= 0] = 0
    for brute in (False, True):
        got, ne, ns = oracle.mlem_iterate(ev, R, L, sz, sdl, n_y, n_z, pixel, rho, brute=brute)
        assert ne == int((P > 0).sum()) and ns == int((~ok).sum())
        assert np.max(np.abs(got.ravel() - want)) <= 1e-12 * want.max()
    oracle.set_sigma_z_edge(0.0)
    base, _, _ = oracle.mlem_iterate(ev, R, L, sz, sdl, n_y, n_z, pixel, rho)
    assert np.max(np.abs(base.ravel() - want)) > 1e-3 * want.max()          # eta = 0.1 is visible in the image


# ------------------------------------------------------------------------------------------------------
# exact kernel: the integral Eq. 7 approximates
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("y,z,Z", [(0.0, 0.0, 250.0), (100.0, 50.0, 250.0), (-150.0, -120.0, 600.0)])
def test_exact_kernel_integrates_to_the_box_probability(oracle, y, z, Z):
    """For every theta the normal density factorises (gamma = 0), so int P_exact de~ over the box |z_u~|, |z_d~| <= Z (all
    dl~) is  int dtheta/pi  Pr(|z_u(theta) + n_u| <= Z) Pr(|z_d(theta) + n_d| <= Z)  with Gaussian n: error functions,
    no kernel involved.  (For sigma_z -> 0 this is s(y, z) of Eq. 4 with L = 2Z; the smeared box edges cost ~2 % at
    Z = 250.)  A wrong prefactor, Jacobian or forward model fails by far more than the 0.3 % allowed."""
    from scipy.special import erf

    sz, sdl, hz, hl = 10.0, 40.0, 5.0 if Z < 300 else 10.0, 20.0       # steps <= sigma: the sums converge like exp(-2 pi^2 sigma^2 / h^2)
    zs = np.arange(-Z + hz / 2, Z, hz)
    dls = np.arange(-2 * abs(y) * 1.6 - 6 * sdl, 2 * abs(y) * 1.6 + 6 * sdl, hl)
    zu, zd, dl = np.meshgrid(zs, zs, dls, indexing="ij")
    ev = np.stack([zu.ravel(), zd.ravel(), dl.ravel()], axis=1)
    P = oracle.kernel_exact_events(ev, y, z, R, L, sz, sdl, n_theta=1501)
    total = P.sum() * hz * hz * hl
    th = np.linspace(-0.5 * math.pi + 1e-7, 0.5 * math.pi - 1e-7, 400001)
    e = forward(y, z, th)

    def inside(c):
        return 0.5 * (erf((Z - c) / (math.sqrt(2) * sz)) - erf((-Z - c) / (math.sqrt(2) * sz)))

    f = inside(e[0]) * inside(e[1])
    want = float(np.sum(0.5 * (f[1:] + f[:-1]) * np.diff(th)) / math.pi)
    assert abs(want / oracle.sensitivity(y, z, R, 2 * Z) - 1.0) < 0.03          # Eq. 4 up to the edge smearing
    assert abs(total / want - 1.0) < 3e-3


def test_exact_kernel_is_what_eq7_approximates(oracle):
    """Inside the 3-sigma ellipse Eq. 7 stays within ~1 % rms of the integral (4.2e-3 rms at 10 / 40);
    the values of SURVEY.md's worked example (tests/golden/worked_example.txt, last column) are reproduced."""
    ev = np.array([120.0, -60.0, -80.0])
    C = oracle.cinv(ev[0], ev[1], L, 10.0, 40.0)
    tan_t, y_t, z_t = oracle.eq2(*ev, R)
    gold = {(50.0, 40.0): 1.63479146e-07, (20.0, 30.0): 1.00792074e-07, (95.0, 50.0): 3.24243572e-09, (-10.0, 20.0): 4.32257629e-09,
            (40.0, 60.0): 1.56112432e-09}
    for (y, z), want in gold.items():
        assert oracle.kernel_exact(y, z, ev, R, C, 200001) == pytest.approx(want, rel=2e-8)
        assert oracle.kernel_exact(y, z, ev, R, C, 4001) == pytest.approx(want, rel=1e-6)     # converged long before
    assert oracle.kernel_exact(y_t, z_t, ev, R, C, 200001) == pytest.approx(1.90594985e-07, rel=2e-8)
    rng = np.random.default_rng(5)
    rel = []
    for _ in range(200):
        e = forward(rng.uniform(-200, 200), rng.uniform(-150, 150), rng.uniform(-0.5, 0.5)) + rng.normal(size=3) * np.array([10, 10, 40])
        t, yt, zt = oracle.eq2(*e, R)
        y, z = yt + rng.uniform(-1.4, 1.4) * 40, zt + rng.uniform(-2, 2) * 10
        if oracle.bCb(y - yt, z - zt, t, 10, 40) > 9:
            continue
        rel.append(oracle.kernel(y, z, t, yt, zt, R, 10, 40) / oracle.kernel_exact(y, z, e, R, oracle.cinv(e[0], e[1], L, 10, 40), 8001) - 1)
    assert 1e-3 < np.sqrt(np.mean(np.square(rel))) < 1e-2


def test_mlem_in_exact_mode_uses_the_integral(oracle):
    cfg = synth.CONFIGS["cfg1"]
    n_y, n_z, pixel = 10, 10, 16.0
    ev = synth.generate_events(cfg.phantom, 25, R, L, 10.0, 40.0, seed=4) * np.float32(0.4)
    rho = np.random.default_rng(2).uniform(0.5, 2.0, (n_y, n_z))
    ys = (np.arange(n_y) - 0.5 * (n_y - 1)) * pixel
    zs = (np.arange(n_z) - 0.5 * (n_z - 1)) * pixel
    s = oracle.sensitivity_image(R, L, n_y, n_z, pixel).ravel()
    P = np.zeros((len(ev), n_y * n_z))
    for j, e in enumerate(ev.astype(np.float64)):
        tan_t, y_t, z_t = oracle.eq2(*e, R)
        C = oracle.cinv(e[0], e[1], L, 10.0, 40.0)
        for iy, y in enumerate(ys):
            for iz, z in enumerate(zs):
                if oracle.bCb(y - y_t, z - z_t, tan_t, 10.0, 40.0) <= 9.0:
                    P[j, iy * n_z + iz] = oracle.kernel_exact(y, z, e, R, C, 3001)
    denom = P @ (s * rho.ravel())
    want = rho.ravel() * (P / denom[:, None]).sum(axis=0)
    try:
        oracle.set_exact_kernel(3001)
        got, ne, ns = oracle.mlem_iterate(ev, R, L, 10.0, 40.0, n_y, n_z, pixel, rho)
    finally:
        oracle.set_exact_kernel(0)
    assert ns == 0 and ne == int((P > 0).sum())
    assert np.max(np.abs(got.ravel() - want)) <= 1e-12 * want.max()
    eq7, _, _ = oracle.mlem_iterate(ev, R, L, 10.0, 40.0, n_y, n_z, pixel, rho)
    d = np.max(np.abs(eq7.ravel() - want)) / want.max()
    assert 1e-6 < d < 2e-2                      # the approximation is visible and small


# ------------------------------------------------------------------------------------------------------
# direct reconstruction histogram (Eq. 2 + binning, Fig. 4b)
# ------------------------------------------------------------------------------------------------------
def test_direct_histogram_puts_noise_free_events_into_the_emitting_pixel(oracle):
    """Eq. 2 inverts Eq. 1, so an unsmeared event is counted in the pixel that contains its emission
    point (points within 1e-3 pixel of a pixel border are left out: the events are rounded to fp32)."""
    cfg = synth.CONFIGS["fig4"]
    ev, truth = synth.noise_free_events(20000, cfg.R, cfg.L, seed=3, y_max=0.45 * cfg.n_y * cfg.pixel)
    fy = truth[:, 0] / cfg.pixel + 0.5 * (cfg.n_y - 1) + 0.5
    fz = truth[:, 1] / cfg.pixel + 0.5 * (cfg.n_z - 1) + 0.5
    safe = (np.abs(fy - np.round(fy)) > 1e-3) & (np.abs(fz - np.round(fz)) > 1e-3)
    inside = (fy >= 0) & (fy < cfg.n_y) & (fz >= 0) & (fz < cfg.n_z)
    want = np.zeros((cfg.n_y, cfg.n_z), dtype=np.uint32)
    np.add.at(want, (np.floor(fy[safe & inside]).astype(int), np.floor(fz[safe & inside]).astype(int)), 1)
    got, outside = oracle.direct_histogram(ev[safe].astype(np.float32), cfg.R, cfg.n_y, cfg.n_z, cfg.pixel)
    assert (got == want).all() and outside == int((safe & ~inside).sum())
    assert int(got.sum()) + outside == int(safe.sum())


def test_direct_pixel_coords_invert_the_forward_model(oracle):
    """jo_direct_pixel_coords is Eq. 2 in fp64 plus the grid convention: for unsmeared events of the forward model (synth:
    Eq. 1 and the strip geometry, no Eq. 2) it returns the emission point in pixels from the lower grid edge - up to the
    rounding of the events to fp32 (|z| <= 250 mm, |dl| <= 600 mm: <= 3e-5 mm, 1e-5 pixel of 4 mm) - and the histogram is
    its floor; a wrong sign, a swapped axis or a half-pixel shift fail here."""
    from types import SimpleNamespace

    fig4 = synth.CONFIGS["fig4"]
    cfg = SimpleNamespace(R=fig4.R, L=fig4.L, n_y=25, n_z=40, pixel=4.0)   # smaller than the emission region: some points fall outside
    ev, truth = synth.noise_free_events(5000, cfg.R, cfg.L, seed=9, y_max=0.45 * fig4.n_y * fig4.pixel)
    ev32 = ev.astype(np.float32)
    c = oracle.direct_pixel_coords(ev32, cfg.R, cfg.n_y, cfg.n_z, cfg.pixel)
    ys = (np.arange(cfg.n_y) - 0.5 * (cfg.n_y - 1)) * cfg.pixel          # pixel centres as the header defines them
    zs = (np.arange(cfg.n_z) - 0.5 * (cfg.n_z - 1)) * cfg.pixel
    want_y = (truth[:, 0] - (ys[0] - 0.5 * cfg.pixel)) / cfg.pixel       # distance from the lower edge of pixel row 0
    want_z = (truth[:, 1] - (zs[0] - 0.5 * cfg.pixel)) / cfg.pixel
    assert np.max(np.abs(c[:, 0] - want_y)) < 2e-5 and np.max(np.abs(c[:, 1] - want_z)) < 2e-5
    inside = (c[:, 0] >= 0) & (c[:, 0] < cfg.n_y) & (c[:, 1] >= 0) & (c[:, 1] < cfg.n_z)
    assert 0.1 * len(c) < inside.sum() < 0.9 * len(c)                    # both cases occur
    want = np.zeros((cfg.n_y, cfg.n_z), dtype=np.uint32)
    np.add.at(want, (np.floor(c[inside, 0]).astype(int), np.floor(c[inside, 1]).astype(int)), 1)
    got, outside = oracle.direct_histogram(ev32, cfg.R, cfg.n_y, cfg.n_z, cfg.pixel)
    assert (got == want).all() and outside == int((~inside).sum())
    bad = np.array([[np.nan, 0, 0], [0, np.inf, 0], [0, 0, -np.inf]], dtype=np.float32)
    assert np.isnan(oracle.direct_pixel_coords(bad, cfg.R, cfg.n_y, cfg.n_z, cfg.pixel)).all()


def test_direct_histogram_conventions(oracle):
    n_y, n_z, px = 4, 6, 8.0                       # 1 / pixel is exact in fp32: the borders below are decided exactly
    # an event with z_u = z_d = z and dl = -2y reconstructs to (y, z) exactly (theta~ = 0)
    def at(y, z):
        return [z, z, -2.0 * y]
    ev = np.array([at(-12.0, -20.0), at(12.0, 20.0), at(-16.0, 0.0), at(15.999, 23.999), at(16.0, 0.0), at(0.0, 24.0), at(0.0, -24.001),
                   [np.nan, 0, 0], [0, np.inf, 0]], dtype=np.float32)
    h, outside = oracle.direct_histogram(ev, 450.0, n_y, n_z, px)
    assert h[0, 0] == 1 and h[3, 5] == 2           # centres of the corner pixels; just inside the upper corner
    assert h[0, 3] == 1                            # y = -16 is the closed lower edge of row 0
    assert h.sum() == 4 and outside == 5           # upper edges are open; NaN / inf never count
    h2, _ = oracle.direct_histogram(ev[:2], 450.0, n_y, n_z, px, hist=h)          # increments
    assert h2 is h and h[0, 0] == 2


def test_direct_histogram_of_smeared_events_is_a_blurred_phantom(oracle):
    """Fig. 4b: the direct reconstruction already shows the phantom, blurred by the detector resolution."""
    cfg = synth.CONFIGS["fig4"]
    ev = synth.config_events(cfg, n=200_000)
    h, outside = oracle.direct_histogram(ev, cfg.R, cfg.n_y, cfg.n_z, cfg.pixel)
    assert h.sum() + outside == len(ev) and outside < 0.05 * len(ev)
    ys = (np.arange(cfg.n_y) - 0.5 * (cfg.n_y - 1)) * cfg.pixel
    zs = (np.arange(cfg.n_z) - 0.5 * (cfg.n_z - 1)) * cfg.pixel
    truth = synth.phantom_intensity(cfg.phantom, *np.meshgrid(ys, zs, indexing="ij"))
    s = oracle.sensitivity_image(cfg.R, cfg.L, cfg.n_y, cfg.n_z, cfg.pixel)
    assert np.corrcoef(h.ravel(), (truth * s).ravel())[0, 1] > 0.6


# ------------------------------------------------------------------------------------------------------
# event generator (Philox4x32-10 per event slot)
# ------------------------------------------------------------------------------------------------------
def test_philox_known_answers(oracle):
    """Known-answer vectors of Philox4x32-10 (tests/golden/philox4x32_10_kat.txt)."""
    n = 0
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if len(line) == 10:
            w = [int(x, 16) for x in line]
            assert oracle.philox4x32_10(w[0:4], w[4:6]) == w[6:10]
            n += 1
    assert n == 3


def test_generator_slots_do_not_depend_on_how_they_are_asked_for(oracle):
    cfg = synth.CONFIGS["cfg2"]
    args = (cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl)
    a = oracle.generate_events(cfg.phantom, 5000, *args, seed=11)
    b = oracle.generate_events(cfg.phantom, 1234, *args, seed=11, first=2000)
    assert (a[2000:3234] == b).all()
    assert not (oracle.generate_events(cfg.phantom, 100, *args, seed=12) == a[:100]).all()
    assert np.isfinite(a).all()
    assert len(np.unique(a[:, 0])) > 0.99 * len(a)            # slots are different events (fp32 values may collide by chance)


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "fig4"])
def test_generator_matches_the_numpy_recipe_statistically(oracle, name):
    """The same recipe as synth.generate_events with another random stream: first two moments of every
    column within 5 standard errors, and the 2-D distribution of the reconstructed points (chi-square of the two
    direct-reconstruction histograms on a coarse grid)."""
    cfg = synth.CONFIGS[name]
    n = 400_000
    got = oracle.generate_events(cfg.phantom, n, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, seed=3).astype(np.float64)
    ref = synth.config_events(cfg, n=n).astype(np.float64)
    for c in range(3):
        sd = ref[:, c].std()
        assert abs(got[:, c].mean() - ref[:, c].mean()) < 5 * sd * math.sqrt(2.0 / n)
        m4 = np.mean((ref[:, c] - ref[:, c].mean()) ** 4)
        assert abs(got[:, c].var() - ref[:, c].var()) < 5 * math.sqrt(2.0 * (m4 - sd**4) / n)
    assert abs(np.corrcoef(got[:, 0], got[:, 1])[0, 1] - np.corrcoef(ref[:, 0], ref[:, 1])[0, 1]) < 0.01
    ny, nz, px = 16, 20, cfg.pixel * cfg.n_y / 16
    ha, _ = oracle.direct_histogram(got.astype(np.float32), cfg.R, ny, nz, px)
    hb, _ = oracle.direct_histogram(ref.astype(np.float32), cfg.R, ny, nz, px)
    ha, hb = ha.ravel().astype(float), hb.ravel().astype(float)
    m = (ha + hb) >= 40
    chi2 = float(np.sum((ha[m] - hb[m]) ** 2 / (ha[m] + hb[m])))
    dof = int(m.sum()) - 1
    assert chi2 < dof + 5 * math.sqrt(2 * dof), (chi2, dof)


def test_generator_smearing_and_acceptance(oracle):
    """With sigma = 0 every event is an exact detected LOR: both hits on the strips, Eq. 1 satisfied, the emission point
    (recovered with Eq. 2) inside the phantom; with sigma > 0 the residuals to those are N(0, sigma)."""
    cfg = synth.CONFIGS["cfg2"]
    exact = oracle.generate_events(cfg.phantom, 50_000, cfg.R, cfg.L, 0.0, 0.0, seed=5).astype(np.float64)
    assert (np.abs(exact[:, :2]) <= 0.5 * cfg.L + 1e-3).all()
    t = (exact[:, 0] - exact[:, 1]) / (2 * cfg.R)
    y = -0.5 * exact[:, 2] / np.sqrt(1 + t * t)
    z = 0.5 * (exact[:, 0] + exact[:, 1]) + y * t
    assert (synth.phantom_intensity(cfg.phantom, y * (1 - 1e-6), z * (1 - 1e-6)) > 0).mean() > 0.999
    smeared = oracle.generate_events(cfg.phantom, 50_000, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, seed=5).astype(np.float64)
    d = smeared - exact                         # same slots, same attempts: only the smearing differs
    for c, sig in enumerate((cfg.sigma_z, cfg.sigma_z, cfg.sigma_dl)):
        assert abs(d[:, c].mean()) < 5 * sig / math.sqrt(len(d)) and d[:, c].std() == pytest.approx(sig, rel=0.02)
    assert abs(np.corrcoef(d[:, 0], d[:, 1])[0, 1]) < 0.02 and abs(np.corrcoef(d[:, 0], d[:, 2])[0, 1]) < 0.02
    theta = np.arctan(t)
    hist, _ = np.histogram(theta, bins=8, range=(-0.25, 0.25))     # well inside the angular acceptance of the phantom
    assert hist.min() > 0.8 * hist.max()        # uniform in theta where the acceptance does not cut
