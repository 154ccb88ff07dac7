"""Host logic of the CUDA path, no GPU: the plan jpet_mlem_begin would choose (kernel shape, degree of the exponent
polynomial, tiling, shared memory) and the host-built task table (csrc/task_table.h) that maps the lanes of an event
group to pieces of ellipse rows.  Read through the C-ABI call jpet_plan_describe."""
import math

import numpy as np
import pytest

import paper_1502_07478_b200 as jp
from paper_1502_07478_b200 import synth

VALID = 1 << 15


def plan_of(cfg):
    return jp.jpet_plan_describe(cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel)


def decode(entry):
    return {"row": entry & 0xFF, "part": (entry >> 8) & 3, "sh": (entry >> 10) & 3} if entry & VALID else None


@pytest.mark.parametrize("name,shape,low,degree,warps", [("cfg1", "small_deg3", "", 3, 1), ("cfg2", "mid18_deg4", "mid18_deg3", 4, 1),
                                                         ("cfg3", "mid18_deg3", "", 3, 1), ("cfg4", "large_deg4", "large_deg3", 4, 4),
                                                         ("cfg5", "xl_deg4", "", 4, 4), ("fig4", "small_closed", "", 0, 1)])
def test_plan_of_every_workload(name, shape, low, degree, warps):
    """Shape and degree per workload - `low`: the degree-3 instance for the events whose own bound
    allows it - and the tiling identities the kernels rely on."""
    cfg = synth.CONFIGS[name]
    p = plan_of(cfg)
    assert (jp.jpet_shape_name(p["variant"]), p["degree"], p["warps_per_event"], p["tiled"]) == (shape, degree, warps, 1)
    assert jp.jpet_shape_name(p["variant_low"]) == low
    assert p["HS"] % 32 == 0 and p["HS"] >= 2 * p["Hy"] + 4          # region rows: bank-conflict-free stride, whole ellipse
    assert p["Sy"] == p["HS"] - 2 * p["Hy"] and p["WZ"] == p["Sz"] + 2 * p["Hz"]
    hy = 1.5 * cfg.sigma_dl / cfg.pixel
    t_max = (cfg.L + 8 * cfg.sigma_z) / (2 * cfg.R)
    hz = 3 * math.sqrt(cfg.sigma_z**2 / 2 + cfg.sigma_dl**2 * (t_max**2 / (1 + t_max**2)) / 4) / cfg.pixel
    assert p["Hy"] >= hy + 1 and p["Hz"] >= hz + 1 - 1e-9               # halo >= largest 3-sigma extents (App. B)
    regions = 1 + p["groups_per_cta"]
    assert p["smem_bytes"] == 4 * regions * p["HS"] * p["WZ"] + 4 * p["table"].size <= 227 * 1024
    assert p["nr_min"] <= math.floor(2 * hy / math.sqrt(1 + t_max**2)) and p["nr_max"] >= math.floor(2 * hy) + 1
    assert p["table"].shape == (p["nr_max"] - p["nr_min"] + 1, 32 * warps)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg4", "cfg5", "fig4"])
def test_task_table_covers_every_row_once_without_bank_conflicts(name):
    cfg = synth.CONFIGS[name]
    p = plan_of(cfg)
    for k, words in enumerate(p["table"]):
        n = p["nr_min"] + k
        whole, parts = {}, {}
        for lane, w in enumerate(words):
            a, b = decode(int(w) & 0xFFFF), decode(int(w) >> 16)
            if a:
                assert a["part"] == 0 and a["sh"] == 0 and a["row"] not in whole       # slot A holds whole rows
                whole[a["row"]] = lane
            if b:
                parts.setdefault(b["row"], []).append((b["part"], b["sh"]))
        assert not (set(whole) & set(parts))
        for row, lst in parts.items():
            sh = lst[0][1]
            assert sorted(q for q, _ in lst) == list(range(1 << sh)) and all(s == sh for _, s in lst)
        assert sorted(set(whole) | set(parts)) == list(range(n))                         # every row of the ellipse, once
        for warp in range(p["warps_per_event"]):                                         # rows of a warp: distinct banks
            rows = [r for r, lane in whole.items() if lane // 32 == warp]
            assert len({r % 32 for r in rows}) == len(rows)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "fig4"])
def test_pieces_fit_their_register_slots(name):
    """The table promises that no piece is longer than its slot (the kernels keep the kernel values of a piece in
    cap_a / cap_b registers): random ellipses of every row count, chords counted as the kernels count them."""
    cfg = synth.CONFIGS[name]
    p = plan_of(cfg)
    rng = np.random.default_rng(3)
    H0p = 9 * 0.5 * cfg.sigma_z**2 / cfg.pixel**2                      # half chord^2 at the centre row [px^2]
    hy_max = 1.5 * cfg.sigma_dl / cfg.pixel
    seen = set()
    for _ in range(4000):
        hy = hy_max / math.sqrt(1 + rng.uniform(0, ((cfg.L + 8 * cfg.sigma_z) / (2 * cfg.R)) ** 2))
        fy, zc0, tilt = rng.uniform(0, 1), rng.uniform(0, 1), rng.uniform(-1.5, 1.5)
        iy0 = math.ceil(fy - hy)
        n = math.floor(fy + hy) - iy0 + 1
        if not p["nr_min"] <= n <= p["nr_max"]:
            continue
        seen.add(n)
        words = p["table"][n - p["nr_min"]]
        for w in words:
            for entry, cap in ((int(w) & 0xFFFF, p["cap_a"]), (int(w) >> 16, p["cap_b"])):
                e = decode(entry)
                if not e:
                    continue
                d = (iy0 + e["row"] - fy) / hy
                hw2 = H0p * (1 - d * d)
                assert hw2 >= -1e-9
                hw, zc = math.sqrt(max(hw2, 0.0)), zc0 + tilt * (iy0 + e["row"] - fy)
                length = max(0, math.floor(zc + hw) - math.ceil(zc - hw) + 1)
                assert -(-length // (1 << e["sh"])) <= cap
    assert len(seen) >= (p["nr_max"] - p["nr_min"] + 1) // 2


def worst_truncation(cfg, ev, degrees):
    """max over sampled (event, row, pixel) of |series cut after u^d - exact| * P / P_peak in log2 units, for every d in
    `degrees` (see the test below).  Quadratic forms typed from Eq. 8-10 with the diagonal C^-1 (fp64)."""
    R, iz2, il2, k = cfg.R, 1 / cfg.sigma_z**2, 1 / cfg.sigma_dl**2, 2.0
    y_lim = 0.5 * cfg.n_y * cfg.pixel
    rng = np.random.default_rng(4)
    worst = {d: 0.0 for d in degrees}
    for zu, zd, dl in ev:
        t = (zu - zd) / (2 * R)
        sec2 = 1 + t * t
        sec = math.sqrt(sec2)
        yt = -0.5 * dl / sec
        dy = rng.uniform(-1, 1, 12) * 1.5 * cfg.sigma_dl / sec
        y = yt + dy
        dy, y = dy[np.abs(y) <= y_lim], y[np.abs(y) <= y_lim]          # rows outside the image are never evaluated
        if not len(dy):
            continue
        c2 = 4 * il2 * sec2 * dy * dy
        frac = np.where(np.arange(len(dy)) % 2 == 0, 1.0, rng.uniform(0, 1, len(dy)))     # chord ends and points inside
        u = rng.choice([-1.0, 1.0], len(dy)) * frac * np.sqrt(np.maximum(9 - c2, 0) / (2 * iz2))
        alpha, beta = -2 * iz2 * sec2 * y, 2 * k * il2 * sec2 * t * y * dy
        aa = 2 * iz2 * sec2**2 * (y * y + R * R) + k * k * il2 * sec2 * t * t * y * y
        eps, delta = -4 * iz2 * sec2 * t * y, aa + 4 * il2 * sec2 * (1 + 2 * t * t) * y * dy
        ba, D = alpha * u + beta, eps * u + delta
        exact = 0.5 * ba * ba / D - 0.5 * np.log(D)
        # P / P_peak: the peak of the event sits at its reconstructed point (dy = u = 0), where P = D_0^-1/2
        D0 = 2 * iz2 * sec2**2 * (yt * yt + R * R) + k * k * il2 * sec2 * t * t * yt * yt
        weight = np.sqrt(D0 / D) * np.exp(-0.5 * (2 * iz2 * u * u + c2 - ba * ba / D))
        kap = eps / delta
        e = [beta**2 / delta, 2 * alpha * beta / delta, alpha**2 / delta]
        e[1] = e[1] - kap * e[0]
        e[2] = e[2] - kap * e[1]
        for n in range(3, 6):
            e.append(-kap * e[-1])
        for d in worst:
            series = -0.5 * np.log(delta) + sum((0.5 * e[n] + (0 if n == 0 else -0.5 * (-1) ** (n + 1) * kap**n / n)) * u**n
                                                for n in range(d + 1))
            worst[d] = max(worst[d], float(np.max(np.abs(series - exact) * weight)) * 1.4427)
    return worst


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
def test_degree_of_the_exponent_polynomial_keeps_the_truncation_small(name):
    """along a row ln P = -1/2 (q - ba^2 / D) - 1/2 ln D with D = delta (1 + x) is expanded in x = eps u /
    delta and cut after u^degree.  What the plan bounds is the error of a kernel value against the event's largest one
    (the image tolerance is relative to the image maximum): the neglected terms, in log2 units, times P / P_peak.  The
    plan's degree must keep that below its own bound (2e-5) everywhere in the 3-sigma ellipse - on its boundary, where x is
    largest but P is e^-4.5 of the peak, and inside, where P is large but x small; one degree less must be worse."""
    cfg = synth.CONFIGS[name]
    deg = plan_of(cfg)["degree"]
    assert deg in (3, 4, 5)
    worst = worst_truncation(cfg, synth.config_events(cfg, n=1500).astype(np.float64), (deg - 1, deg))
    assert worst[deg] <= 2e-5, worst
    assert worst[deg - 1] > worst[deg]


def test_truncation_bound_holds_when_the_strips_are_longer_than_2R():
    """|x| = |eps u / delta| is proportional to |t| / (1 + t^2), which peaks at |t| = 1 - for L > 2 R the
    largest tilt t_max = (L + 8 sigma_z) / (2 R) is beyond the peak, and a bound evaluated at t_max under-estimates x.
    Brute force over unsmeared events of the forward model spanning all tilts (R = 100, L = 600: |t| up to 2.9): the degree
    the plan picks must keep the weighted truncation below the plan's 2e-5, and one degree less must not (the geometry is
    chosen at that edge: with the bound taken at t_max the plan picked degree 4, whose tail is 3e-5)."""
    from types import SimpleNamespace

    cfg = SimpleNamespace(R=100.0, L=600.0, n_y=60, n_z=240, pixel=2.5, sigma_z=6.0, sigma_dl=30.0)
    deg = plan_of(cfg)["degree"]
    ev, _ = synth.noise_free_events(3000, cfg.R, cfg.L, seed=1, y_max=0.5 * cfg.n_y * cfg.pixel)
    assert np.max(np.abs(ev[:, 0] - ev[:, 1]) / (2 * cfg.R)) > 2.5 and np.min(np.abs(ev[:, 0] - ev[:, 1]) / (2 * cfg.R)) < 0.05
    worst = worst_truncation(cfg, ev, (3, 4, 5))
    assert deg in (0, 3, 4, 5)
    if deg:
        assert worst[deg] <= 2e-5, (deg, worst)
    assert deg == 5 and worst[4] > 2e-5, (deg, worst)      # degree 4 is not enough here, degree 5 is (and has a shape that fits)


def test_forced_sub_tile_width_that_does_not_fit_goes_direct():
    """a forced "sub_tile_z" whose regions exceed shared memory used to be replaced silently by 4; now the
    plan keeps the caller's width and sends every event to the direct kernel (tiled = 0); a width that fits is used."""
    cfg = synth.CONFIGS["cfg5"]
    try:
        jp.jpet_set_option("sub_tile_z", 256)
        p = plan_of(cfg)
        assert p["tiled"] == 0 and p["smem_bytes"] == 0
        jp.jpet_set_option("sub_tile_z", 4)
        p = plan_of(cfg)
        assert p["tiled"] == 1 and p["Sz"] == 4
    finally:
        jp.jpet_set_option("sub_tile_z", 0)
    assert plan_of(cfg)["tiled"] == 1
