"""Pins of the fp64 CPU oracle against what the paper and the mathematics fix (CPU only, -m "not gpu").

None of these tests retypes an oracle formula.  Each one reaches the expected value by another road:
the detector forward model (Eq. 1 / Fig. 1 geometry) differentiated or integrated numerically,
Monte-Carlo acceptance, closed forms, invariants of Eq. 3, a dense-matrix transcription of Eq. 3, or the
worked example that SURVEY.md section 8(c) derived before any code existed (tests/golden/).
"""
import math
import os

import numpy as np
import pytest

from paper_1502_07478_b200 import synth

R, L = 450.0, 500.0
GOLD = os.path.join(os.path.dirname(__file__), "golden", "worked_example.txt")


# ------------------------------------------------------------------------------------------------------
# independent helpers: the detector forward model e(y, z, theta) (PAPER.md:52-55 and Fig. 1 geometry)
# ------------------------------------------------------------------------------------------------------
def forward(y, z, theta, R=R):
    """Exact measurement (z_u, z_d, dl) of an emission at (y, z) along in-plane angle theta."""
    return np.array([z + (R - y) * np.tan(theta), z - (R + y) * np.tan(theta), -2.0 * y / np.cos(theta)])


def gauss3(e_meas, e_exact, sz, sdl):
    """Normalised 3-D Gaussian density N(e_meas; e_exact, diag(sz^2, sz^2, sdl^2))."""
    d = np.asarray(e_meas).reshape(3, -1) - np.asarray(e_exact).reshape(3, -1)
    chi2 = (d[0] / sz) ** 2 + (d[1] / sz) ** 2 + (d[2] / sdl) ** 2
    return np.exp(-0.5 * chi2) / ((2.0 * math.pi) ** 1.5 * sz * sz * sdl)


def exact_theta_integral(ev, y, z, sz, sdl, R=R, n=200001):
    """P_exact(e~ | y, z) = int dtheta/pi N(e~; e(y, z, theta), C) over (-pi/2, pi/2) (R15), trapezoid."""
    th = np.linspace(-0.5 * math.pi + 1e-9, 0.5 * math.pi - 1e-9, n)
    f = gauss3(np.asarray(ev, float).reshape(3, 1), forward(y, z, th, R), sz, sdl)
    return float(np.sum(0.5 * (f[1:] + f[:-1]) * np.diff(th)) / math.pi)


def cinv_eq12(sz, sdl, gamma=0.0):
    """Eq. 12 as printed."""
    return np.array([[1 / sz**2, 0.0, gamma], [0.0, 1 / sz**2, -gamma], [gamma, -gamma, 1 / sdl**2]])


def laplace_from_forward_model(ev, y, z, sz, sdl, R=R, gamma=0.0):
    """Second-order saddle-point value of the theta integral, built ONLY from the forward model:
    expand e(theta) = e(theta~) + a d + o d^2 with a, o from central differences (no Eq. 8-10 typed in),
    keep terms to d^2 in the exponent and do the Gaussian integral over d analytically."""
    theta_t = math.atan((ev[0] - ev[1]) / (2.0 * R))
    h = 1e-3
    e0 = forward(y, z, theta_t, R)
    ep, em = forward(y, z, theta_t + h, R), forward(y, z, theta_t - h, R)
    ep2, em2 = forward(y, z, theta_t + 2 * h, R), forward(y, z, theta_t - 2 * h, R)
    a = (-ep2 + 8 * ep - 8 * em + em2) / (12 * h)                       # d e / d theta, O(h^4)
    o = 0.5 * (-ep2 + 16 * ep - 30 * e0 + 16 * em - em2) / (12 * h * h)  # 1/2 d2 e / d theta2, O(h^4)
    b = e0 - np.asarray(ev, float)
    Cinv = cinv_eq12(sz, sdl, gamma)
    D = a @ Cinv @ a + 2.0 * (o @ Cinv @ b)
    expo = -0.5 * (b @ Cinv @ b - (b @ Cinv @ a) ** 2 / D)
    norm = math.sqrt(np.linalg.det(Cinv)) / (2.0 * math.pi) ** 1.5       # Gaussian density prefactor
    return norm * math.sqrt(2.0 * math.pi / D) * math.exp(expo) / math.pi


def read_golden():
    sections, cur = {}, None
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("["):
            cur = line.strip("[]")
            sections[cur] = []
        else:
            sections[cur].append(line.split())
    return sections


# ------------------------------------------------------------------------------------------------------
# Eq. 1 / Eq. 2
# ------------------------------------------------------------------------------------------------------
def test_eq2_inverts_eq1_on_noise_free_events(oracle):
    """the direct reconstruction reproduces exact emission points (R1-R3)."""
    ev, tr = synth.noise_free_events(2000, R, L, seed=3)
    for (zu, zd, dl), (y, z, t) in zip(ev, tr):
        tan_t, y_t, z_t = oracle.eq2(zu, zd, dl, R)
        assert abs(tan_t - t) < 1e-12
        assert abs(y_t - y) < 1e-10 and abs(z_t - z) < 1e-10


def test_eq1_matches_lor_geometry(oracle):
    """Eq. 1 with the hit points on the LOR equals -2y/cos(theta) (distance difference along the line)."""
    rng = np.random.default_rng(0)
    for _ in range(200):
        y, z, th = rng.uniform(-300, 300), rng.uniform(-200, 200), rng.uniform(-0.5, 0.5)
        zu, zd, dl = forward(y, z, th)
        assert abs(oracle.eq1_delta_l(y, z, zu, zd, R) - dl) < 1e-10


def test_eq2_worked_example(oracle):
    g = dict((k, float(v)) for k, v in read_golden()["eq2"])
    tan_t, y_t, z_t = oracle.eq2(120.0, -60.0, -80.0, 450.0)
    assert abs(tan_t - g["tan_theta"]) < 1e-12
    assert abs(y_t - g["y_t"]) < 1e-9 and abs(z_t - g["z_t"]) < 1e-9


def test_eq2_wrong_sign_or_factor_would_fail(oracle):
    """Plausible mistakes (second printed forms of Eq. 2, R2) are off by many mm."""
    zu, zd, dl = forward(80.0, -30.0, 0.3)
    _, y_t, z_t = oracle.eq2(zu, zd, dl, R)
    assert abs(y_t - 80.0) < 1e-10 and abs(z_t + 30.0) < 1e-10
    y_printed = 2 * R * dl / math.sqrt(abs(zu - zd) + 4 * R * R)   # PAPER.md:61 second form, as printed
    assert abs(y_printed - 80.0) > 50.0


# ------------------------------------------------------------------------------------------------------
# Eq. 4 sensitivity
# ------------------------------------------------------------------------------------------------------
def test_sensitivity_closed_form_centre(oracle):
    assert abs(oracle.sensitivity(0.0, 0.0, R, L) - (2.0 / math.pi) * math.atan(L / (2 * R))) < 1e-15
    assert abs(oracle.sensitivity(0.0, 0.0, R, L) - 0.3228289344) < 1e-10


@pytest.mark.parametrize("y,z", [(100.0, 0.0), (0.0, 150.0), (-160.0, 160.0), (200.0, -248.75), (-255.5, 249.5)])
def test_sensitivity_vs_monte_carlo_acceptance(oracle, y, z):
    """Eq. 4 is the fraction of in-plane angles (uniform on (-pi/2, pi/2)) whose LOR hits both strips."""
    rng = np.random.default_rng(42)
    n = 2_000_000
    th = rng.uniform(-0.5 * math.pi, 0.5 * math.pi, n)
    zu, zd, _ = forward(y, z, th)
    acc = np.mean((np.abs(zu) <= 0.5 * L) & (np.abs(zd) <= 0.5 * L))
    s = oracle.sensitivity(y, z, R, L)
    assert abs(s - acc) < 5.0 * math.sqrt(max(acc, 1e-4) / n) + 1e-5


def test_sensitivity_golden_and_clamp(oracle):
    for y, z, s_eq4, _mc in read_golden()["sensitivity"]:
        assert abs(oracle.sensitivity(float(y), float(z), R, L) - float(s_eq4)) < 2e-6
    assert oracle.sensitivity(0.0, 255.5, R, L) == 0.0            # Eq. 4 is -0.0078 there (R13)
    img = oracle.sensitivity_image(R, L, 512, 512, 1.0)
    assert img.min() == 0.0 and (img[:, :6] == 0).all() and (img[:, -6:] == 0).all() and (img[:, 6:-6] > 0).all()


def test_sensitivity_symmetries(oracle):
    img = oracle.sensitivity_image(R, L, 64, 64, 5.0)
    assert np.allclose(img, img[::-1, :], atol=1e-15) and np.allclose(img, img[:, ::-1], atol=1e-15)
    # layout: row-major, z fastest, centred grid
    assert abs(img[10, 20] - oracle.sensitivity((10 - 31.5) * 5.0, (20 - 31.5) * 5.0, R, L)) < 1e-15


# ------------------------------------------------------------------------------------------------------
# b C^-1 b and Appendix B
# ------------------------------------------------------------------------------------------------------
def test_bCb_equals_residual_of_forward_model(oracle):
    """b = e(y, z, theta~) - e~ and b C^-1 b its Mahalanobis norm, via the forward model."""
    rng = np.random.default_rng(1)
    for _ in range(300):
        sz, sdl = rng.uniform(4, 20), rng.uniform(15, 90)
        ev = forward(rng.uniform(-200, 200), rng.uniform(-150, 150), rng.uniform(-0.5, 0.5))
        ev = ev + rng.normal(size=3) * np.array([sz, sz, sdl])
        tan_t, y_t, z_t = oracle.eq2(*ev, R)
        y, z = y_t + rng.uniform(-60, 60), z_t + rng.uniform(-40, 40)
        b = forward(y, z, math.atan(tan_t)) - ev
        want = (b[0] / sz) ** 2 + (b[1] / sz) ** 2 + (b[2] / sdl) ** 2
        assert abs(oracle.bCb(y - y_t, z - z_t, tan_t, sz, sdl) - want) < 1e-9 * max(1.0, want)


@pytest.mark.parametrize("tan_t,sz,sdl", [(0.0, 10, 40), (0.2, 10, 40), (-0.55, 5, 20), (0.4, 20, 80)])
def test_bbox_circumscribes_ellipse(oracle, tan_t, sz, sdl):
    """B.2 against a brute-force boundary scan of b C^-1 b = 9 and against the marginal-std closed form."""
    h_y, h_z = oracle.bbox_half_extents(tan_t, sz, sdl)
    phi = np.linspace(0, 2 * math.pi, 400001)
    r = np.array([3.0 / math.sqrt(oracle.bCb(math.cos(p), math.sin(p), tan_t, sz, sdl)) for p in phi[::40]])
    # refine around the maxima with the full scan, vectorised through the quadratic form's homogeneity
    q_unit = np.array([oracle.bCb(1, 0, tan_t, sz, sdl), oracle.bCb(0, 1, tan_t, sz, sdl),
                       oracle.bCb(1, 1, tan_t, sz, sdl)])
    A, B = q_unit[0], q_unit[1]
    C = 0.5 * (q_unit[2] - A - B)
    rr = 3.0 / np.sqrt(A * np.cos(phi) ** 2 + 2 * C * np.cos(phi) * np.sin(phi) + B * np.sin(phi) ** 2)
    assert np.allclose(rr[::40], r, rtol=1e-12)
    assert abs(np.max(rr * np.cos(phi)) - h_y) < 1e-6 * h_y
    assert abs(np.max(rr * np.sin(phi)) - h_z) < 1e-6 * h_z
    cos_t = 1.0 / math.sqrt(1 + tan_t**2)
    sin_t = tan_t * cos_t
    assert abs(h_y - 3 * 0.5 * sdl * cos_t) < 1e-9                # 3 x std of y~ = -dl~ cos(theta)/2
    assert abs(h_z - 3 * math.sqrt(sz**2 / 2 + sdl**2 * sin_t**2 / 4)) < 1e-9


def test_bbox_worked_example(oracle):
    g = dict((k, float(v)) for k, v in read_golden()["appendix_b"])
    h_y, h_z = oracle.bbox_half_extents(0.2, 10.0, 40.0)
    assert abs(h_y - g["h_y"]) < 1e-7 and abs(h_z - g["h_z"]) < 1e-7


# ------------------------------------------------------------------------------------------------------
# kernel, Eq. 7-12
# ------------------------------------------------------------------------------------------------------
def test_kernel_is_the_saddle_point_of_the_forward_model(oracle):
    """Eq. 7 (with a = d e/d theta, R5, and K = det^(1/2)(C^-1) / 2 pi^2, R4) equals the second-order
    Laplace value of int dtheta/pi N(e~; e(theta), C) computed from the forward model alone; a dropped
    term, a wrong sign in o/a/b, k=1 instead of 2 or the printed 1/2pi prefactor all fail this."""
    rng = np.random.default_rng(7)
    worst = 0.0
    for sz, sdl in [(10, 40), (5, 20), (20, 80)]:
        for _ in range(150):
            ev = forward(rng.uniform(-220, 220), rng.uniform(-150, 150), rng.uniform(-0.5, 0.5))
            ev = ev + rng.normal(size=3) * np.array([sz, sz, sdl])
            tan_t, y_t, z_t = oracle.eq2(*ev, R)
            y, z = y_t + rng.uniform(-1.4, 1.4) * sdl, z_t + rng.uniform(-2, 2) * sz
            want = laplace_from_forward_model(ev, y, z, sz, sdl)
            got = oracle.kernel(y, z, tan_t, y_t, z_t, R, sz, sdl, 2.0)
            worst = max(worst, abs(got / want - 1.0))
            # the printed third component of a (k=1) is distinguishable at this precision for off-axis pixels
    assert worst < 2e-7, worst


def test_kernel_with_gamma_is_the_saddle_point_of_the_forward_model(oracle):
    """Eq. 7 with the general C^-1 of Eq. 12 (gamma != 0) against the same forward-model Laplace value
    with the full 3x3 matrix; a gamma term with the wrong sign, on the wrong pair of components or dropped from one of
    the three quadratic forms fails.  b C^-1 b (B.3, the 3-sigma ellipse) does not depend on gamma: b1 = b2."""
    rng = np.random.default_rng(17)
    try:
        for sz, sdl in [(10, 40), (5, 20), (20, 80)]:
            for frac in (0.3, -0.3, 0.6):
                gamma = frac / (math.sqrt(2.0) * sz * sdl)          # positive definite for |frac| < 1
                oracle.set_gamma(gamma)
                assert oracle.get_gamma() == gamma
                worst, moved = 0.0, 0.0
                for _ in range(60):
                    ev = forward(rng.uniform(-220, 220), rng.uniform(-150, 150), rng.uniform(-0.5, 0.5))
                    ev = ev + rng.normal(size=3) * np.array([sz, sz, sdl])
                    tan_t, y_t, z_t = oracle.eq2(*ev, R)
                    y, z = y_t + rng.uniform(-1.4, 1.4) * sdl, z_t + rng.uniform(-2, 2) * sz
                    want = laplace_from_forward_model(ev, y, z, sz, sdl, gamma=gamma)
                    got = oracle.kernel(y, z, tan_t, y_t, z_t, R, sz, sdl, 2.0)
                    worst = max(worst, abs(got / want - 1.0))
                    moved = max(moved, abs(laplace_from_forward_model(ev, y, z, sz, sdl) / want - 1.0))
                    b = forward(y, z, math.atan(tan_t)) - ev
                    assert abs(b @ cinv_eq12(sz, sdl, gamma) @ b - oracle.bCb(y - y_t, z - z_t, tan_t, sz, sdl)) < 1e-8
                assert worst < 2e-7, (sz, sdl, frac, worst)
                assert moved > 1e-2          # gamma changes the kernel by far more than the pin's resolution
    finally:
        oracle.set_gamma(0.0)


def test_kernel_k1_differs_from_k2_measurably(oracle):
    ev = np.array([120.0, -60.0, -80.0])
    tan_t, y_t, z_t = oracle.eq2(*ev, R)
    p2 = oracle.kernel(50, 40, tan_t, y_t, z_t, R, 10, 40, 2.0)
    p1 = oracle.kernel(50, 40, tan_t, y_t, z_t, R, 10, 40, 1.0)
    want = laplace_from_forward_model(ev, 50.0, 40.0, 10.0, 40.0)
    assert abs(p2 / want - 1) < 2e-7 and abs(p1 / want - 1) > 5e-6


def test_kernel_close_to_exact_theta_integral(oracle):
    """Eq. 7 approximates the theta-integrated Gaussian: ~1 % inside the 3-sigma ellipse."""
    rng = np.random.default_rng(11)
    rel = []
    for _ in range(60):
        sz, sdl = 10.0, 40.0
        ev = forward(rng.uniform(-200, 200), rng.uniform(-150, 150), rng.uniform(-0.45, 0.45))
        ev = ev + rng.normal(size=3) * np.array([sz, sz, sdl])
        tan_t, y_t, z_t = oracle.eq2(*ev, R)
        y, z = y_t + rng.uniform(-40, 40), z_t + rng.uniform(-15, 15)
        if oracle.bCb(y - y_t, z - z_t, tan_t, sz, sdl) > 9:
            continue
        rel.append(oracle.kernel(y, z, tan_t, y_t, z_t, R, sz, sdl) / exact_theta_integral(ev, y, z, sz, sdl) - 1)
    rel = np.array(rel)
    assert len(rel) > 30 and np.sqrt(np.mean(rel**2)) < 1e-2 and np.max(np.abs(rel)) < 5e-2


def test_kernel_worked_example(oracle):
    g = read_golden()
    tan_t, y_t, z_t = oracle.eq2(120.0, -60.0, -80.0, 450.0)
    for row in g["kernel"]:
        y = y_t if row[0] == "y_t" else float(row[0])
        z = z_t if row[1] == "z_t" else float(row[1])
        q, inside, p_k2, p_k1, p_exact = float(row[2]), int(row[3]), float(row[8]), float(row[9]), float(row[10])
        assert abs(oracle.bCb(y - y_t, z - z_t, tan_t, 10, 40) - q) < 1e-7
        assert (oracle.bCb(y - y_t, z - z_t, tan_t, 10, 40) <= 9.0) == bool(inside)
        assert abs(oracle.kernel(y, z, tan_t, y_t, z_t, 450, 10, 40, 2.0) / p_k2 - 1) < 2e-8
        assert abs(oracle.kernel(y, z, tan_t, y_t, z_t, 450, 10, 40, 1.0) / p_k1 - 1) < 2e-8
        assert abs(exact_theta_integral([120.0, -60.0, -80.0], y, z, 10, 40, 450.0) / p_exact - 1) < 1e-6


@pytest.mark.parametrize("y,z,Z,want", [(0.0, 0.0, 250.0, 0.32283), (100.0, 50.0, 250.0, 0.26996),
                                        (-150.0, -120.0, 600.0, 0.49363)])
def test_kernel_integrates_to_sensitivity_over_measurement_space(oracle, y, z, Z, want):
    """int P de~ over |z_u~|,|z_d~| <= Z, all dl~  ~=  s(y, z) evaluated with L = 2Z (-> 1 as Z -> inf),
    up to edge smearing O(sigma_z / Z) (north_star: "P integrating to ~1 over measurement space")."""
    sz, sdl, hz, hl = 10.0, 40.0, 4.0, 8.0
    zs = np.arange(-Z + hz / 2, Z, hz)
    dls = np.arange(-2 * abs(y) * 1.6 - 6 * sdl, 2 * abs(y) * 1.6 + 6 * sdl, hl)
    zu, zd, dl = np.meshgrid(zs, zs, dls, indexing="ij")
    ev = np.stack([zu.ravel(), zd.ravel(), dl.ravel()], axis=1)
    P, inside = oracle.kernel_events(ev, y, z, R, sz, sdl)
    total = P.sum() * hz * hz * hl
    s_box = oracle.sensitivity(y, z, R, 2 * Z)
    assert abs(s_box - want) < 1e-4
    assert abs(total / s_box - 1.0) < 0.025
    cut = P[inside].sum() * hz * hz * hl                            # 3-sigma truncation keeps 1 - exp(-4.5)
    assert abs(cut / total - (1.0 - math.exp(-4.5))) < 0.01
