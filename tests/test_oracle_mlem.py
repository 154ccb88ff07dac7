"""Pins of the oracle's MLEM iteration (Eq. 3 / Listing 1): invariants, special cases, brute force, and a
dense-matrix transcription of Eq. 3 in numpy on tiny grids (CPU only)."""
import numpy as np
import pytest

from paper_1502_07478_b200 import synth

R, L = 450.0, 500.0


def dense_eq3(oracle, events, sz, sdl, n_y, n_z, pixel, rho):
    """Eq. 3 as a dense [N, M] matrix product; P from oracle.kernel (pinned in
    test_oracle_pins.py), truncated to the 3-sigma ellipse with oracle.bCb."""
    ys = (np.arange(n_y) - 0.5 * (n_y - 1)) * pixel
    zs = (np.arange(n_z) - 0.5 * (n_z - 1)) * pixel
    s = oracle.sensitivity_image(R, L, n_y, n_z, pixel).ravel()
    P = np.zeros((len(events), n_y * n_z))
    for j, ev in enumerate(np.asarray(events, dtype=np.float32).astype(np.float64)):
        tan_t, y_t, z_t = oracle.eq2(ev[0], ev[1], ev[2], R)
        for iy, y in enumerate(ys):
            for iz, z in enumerate(zs):
                if oracle.bCb(y - y_t, z - z_t, tan_t, sz, sdl) <= 9.0:
                    P[j, iy * n_z + iz] = oracle.kernel(y, z, tan_t, y_t, z_t, R, sz, sdl)
    rho = rho.ravel()
    denom = P @ (s * rho)                       # sum_i P(e_j|i) s(i) rho(i)
    ok = denom > 0
    out = rho * (P[ok] / denom[ok, None]).sum(axis=0)
    out[s <= 0] = 0.0
    return out.reshape(n_y, n_z), int((P > 0).sum()), int((~ok).sum())


@pytest.mark.parametrize("n_y,n_z,pixel,sz,sdl", [(8, 8, 20.0, 10.0, 40.0), (16, 12, 10.0, 10.0, 40.0)])
def test_iterate_equals_dense_eq3(oracle, n_y, n_z, pixel, sz, sdl):
    cfg = synth.CONFIGS["cfg1"]
    ev = synth.generate_events(cfg.phantom, 60, R, L, sz, sdl, seed=5)
    ev = ev * np.float32(0.5)  # pull events towards the tiny grid
    rng = np.random.default_rng(0)
    rho = rng.uniform(0.5, 2.0, (n_y, n_z))
    want, evals, skipped = dense_eq3(oracle, ev, sz, sdl, n_y, n_z, pixel, rho)
    for brute in (False, True):
        got, ne, ns = oracle.mlem_iterate(ev, R, L, sz, sdl, n_y, n_z, pixel, rho, brute=brute, n_threads=2)
        assert ne == evals and ns == skipped
        assert np.max(np.abs(got - want)) <= 1e-12 * np.max(want)


def test_bbox_loop_equals_full_image_scan_cfg1(oracle):
    """Listing 1's bbox-restricted loop == brute-force scan with the same centre-in-ellipse rule (R10)."""
    cfg = synth.CONFIGS["cfg1"]
    ev = synth.config_events(cfg, n=3000)
    rho = np.ones((cfg.n_y, cfg.n_z))
    a, ne_a, ns_a = oracle.mlem_iterate(ev, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel, rho)
    b, ne_b, ns_b = oracle.mlem_iterate(ev, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel, rho,
                                        brute=True)
    assert (ne_a, ns_a) == (ne_b, ns_b)
    assert np.max(np.abs(a - b)) <= 1e-13 * np.max(a)


def test_count_conservation(oracle):
    """sum_l s(l) rho_out(l) = N - n_skipped for any positive rho_in (multiply Eq. 3 by s(l), sum over l)."""
    cfg = synth.CONFIGS["cfg1"]
    ev = synth.config_events(cfg)
    s = oracle.sensitivity_image(cfg.R, cfg.L, cfg.n_y, cfg.n_z, cfg.pixel)
    rng = np.random.default_rng(1)
    for rho in (np.ones((cfg.n_y, cfg.n_z)), rng.uniform(0.1, 3.0, (cfg.n_y, cfg.n_z))):
        out, ne, ns = oracle.mlem_iterate(ev, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel, rho)
        assert ns == 0
        assert abs((s * out).sum() - (len(ev) - ns)) < 1e-8 * len(ev)
        assert 140 * len(ev) < ne < 170 * len(ev)   # 154.6 px/event for config 1


def test_single_event_closed_form(oracle):
    """One event, uniform rho_in: rho_out(i) = P_i / sum_k P_k s(k) on the ellipse, 0 elsewhere; independent
    of the value of rho_in and of the kernel's constant prefactor (SURVEY.md 8(c) special case)."""
    n_y = n_z = 64
    pixel, sz, sdl = 5.0, 10.0, 40.0
    ev = np.array([[120.0, -60.0, -80.0]], dtype=np.float32)
    tan_t, y_t, z_t = oracle.eq2(120.0, -60.0, -80.0, R)
    s = oracle.sensitivity_image(R, L, n_y, n_z, pixel)
    P = np.zeros((n_y, n_z))
    for iy in range(n_y):
        for iz in range(n_z):
            y, z = (iy - 31.5) * pixel, (iz - 31.5) * pixel
            if oracle.bCb(y - y_t, z - z_t, tan_t, sz, sdl) <= 9.0:
                P[iy, iz] = oracle.kernel(y, z, tan_t, y_t, z_t, R, sz, sdl)
    want = P / (P * s).sum()
    for c in (1.0, 7.5):
        got, ne, ns = oracle.mlem_iterate(ev, R, L, sz, sdl, n_y, n_z, pixel, np.full((n_y, n_z), c))
        assert ne == int((P > 0).sum()) and ns == 0
        assert np.max(np.abs(got - want)) < 1e-12 * want.max()
        assert abs((s * got).sum() - 1.0) < 1e-12
    # ellipse area / pixel area ~ pixel count (3920.94 mm^2 / 25 mm^2 = 156.8; centre-in test => within a few)
    assert abs(int((P > 0).sum()) - 3920.944638 / 25.0) < 8


def test_mirror_symmetries(oracle):
    """(z_u, z_d, dl) -> (z_d, z_u, -dl) mirrors the image in y; z -> -z mirrors it in z (centred grid)."""
    cfg = synth.CONFIGS["cfg1"]
    ev = synth.config_events(cfg, n=2000)
    args = (cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel, np.ones((cfg.n_y, cfg.n_z)))
    base, _, _ = oracle.mlem_iterate(ev, *args)
    ev_y = np.stack([ev[:, 1], ev[:, 0], -ev[:, 2]], axis=1)
    my, _, _ = oracle.mlem_iterate(ev_y, *args)
    assert np.max(np.abs(my - base[::-1, :])) < 1e-12 * base.max()
    ev_z = np.stack([-ev[:, 0], -ev[:, 1], ev[:, 2]], axis=1)
    mz, _, _ = oracle.mlem_iterate(ev_z, *args)
    assert np.max(np.abs(mz - base[:, ::-1])) < 1e-12 * base.max()


def test_order_thread_and_scale_invariance(oracle):
    cfg = synth.CONFIGS["cfg1"]
    ev = synth.config_events(cfg, n=4000)
    rng = np.random.default_rng(2)
    rho = rng.uniform(0.2, 2.0, (cfg.n_y, cfg.n_z))
    args = (cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel)
    a, _, _ = oracle.mlem_iterate(ev, *args, rho, n_threads=1)
    b, _, _ = oracle.mlem_iterate(ev[rng.permutation(len(ev))], *args, rho, n_threads=3)
    c, _, _ = oracle.mlem_iterate(ev, *args, 10.0 * rho, n_threads=2)
    assert np.max(np.abs(a - b)) < 1e-12 * a.max()
    assert np.max(np.abs(a - c)) < 1e-12 * a.max()   # Eq. 3 is homogeneous of degree 0: rho_out(c rho) = rho_out(rho)


def test_skips_and_degenerate_inputs(oracle):
    n_y = n_z = 16
    args = (R, L, 10.0, 40.0, n_y, n_z, 5.0)
    ones = np.ones((n_y, n_z))
    # no events: empty sum over j => rho_out = 0
    out, ne, ns = oracle.mlem_iterate(np.zeros((0, 3), np.float32), *args, ones)
    assert (out == 0).all() and ne == 0 and ns == 0
    # an event far outside the grid, a NaN event, and an event under an all-zero rho are skipped and counted
    far = np.array([[200.0, 200.0, 0.0], [np.nan, 0.0, 0.0]], dtype=np.float32)
    out, ne, ns = oracle.mlem_iterate(far, *args, ones)
    assert (out == 0).all() and ns == 2
    out, ne, ns = oracle.mlem_iterate(np.array([[0.0, 0.0, 0.0]], np.float32), *args, np.zeros((n_y, n_z)))
    assert (out == 0).all() and ns == 1 and ne > 0


def test_reconstruct_is_repeated_iterate(oracle):
    cfg = synth.CONFIGS["cfg1"]
    ev = synth.config_events(cfg, n=3000)
    args = (cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel)
    rho = np.ones((cfg.n_y, cfg.n_z))
    for _ in range(3):
        rho, _, _ = oracle.mlem_iterate(ev, *args, rho)
    rec, _, _ = oracle.reconstruct(ev, *args, 3)
    assert np.max(np.abs(rec - rho)) < 1e-13 * rho.max()
    rec0, _, _ = oracle.reconstruct(ev, *args, 0, rho_init=2 * np.ones((cfg.n_y, cfg.n_z)))
    assert (rec0 == 2).all()
    s = oracle.sensitivity_image(cfg.R, cfg.L, cfg.n_y, cfg.n_z, cfg.pixel)
    assert abs((s * rec).sum() - len(ev)) < 1e-8 * len(ev)


def test_mlem_sharpens_towards_phantom(oracle):
    """Sanity of the whole chain: after a few iterations the hot insert of config 1 (intensity 4 inside a
    30 mm circle) is brighter than the surrounding ellipse, which is brighter than the empty corners."""
    cfg = synth.CONFIGS["cfg1"]
    ev = synth.config_events(cfg)
    rec, _, _ = oracle.reconstruct(ev, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel, 5)
    ys = (np.arange(cfg.n_y) - 31.5) * cfg.pixel
    zs = (np.arange(cfg.n_z) - 31.5) * cfg.pixel
    Y, Z = np.meshgrid(ys, zs, indexing="ij")
    truth = synth.phantom_intensity(cfg.phantom, Y, Z)
    hot = rec[(Y**2 + Z**2) < 20**2].mean()
    body = rec[(truth == 1.0) & ((Y**2 + Z**2) > 50**2)].mean()
    empty = rec[(np.abs(Y) > 130) & (truth == 0)].mean()
    assert hot > 2.0 * body > 10.0 * empty


def test_paper_shaped_workload_fig4(oracle):
    """Fig. 4 geometry with the Table 2 phantom.  The phantom is
    transcribed with x = z (reading R21): each ellipse's centre carries its own density unless a row above covers
    it; Eq. 3 conserves counts on this geometry as well (strips at R = 130 mm, |tan theta| up to 1.2)."""
    cfg = synth.CONFIGS["fig4"]
    table2 = [(0, 0, 0.3), (50, -62, 0.3), (-50, -63, 0.5), (60, 65, 0.5), (35, 55, 0.7)]        # (x, y, rho)
    for x, y, rho in table2:
        assert synth.phantom_intensity(cfg.phantom, np.array([float(y)]), np.array([float(x)]))[0] == rho
    assert synth.phantom_intensity(cfg.phantom, np.array([0.0]), np.array([100.0]))[0] == 0.1    # background, a = 120 along x
    assert synth.phantom_intensity(cfg.phantom, np.array([115.0]), np.array([0.0]))[0] == 0.0    # b = 110 along y
    ev = synth.config_events(cfg, n=20000)
    assert np.all(np.abs(ev[:, :2]) < cfg.L / 2 + 6 * cfg.sigma_z)
    g = (cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel)
    out, n_evals, n_skipped = oracle.mlem_iterate(ev, *g, np.ones((cfg.n_y, cfg.n_z)))
    s = oracle.sensitivity_image(cfg.R, cfg.L, cfg.n_y, cfg.n_z, cfg.pixel)
    assert abs(float((s * out).sum()) - (len(ev) - n_skipped)) <= 1e-8 * len(ev)
    assert 150 < n_evals / len(ev) < 260           # 9 pi sigma_z sigma_dl cos(theta) / (2 sqrt 2 pixel^2) <= 250
