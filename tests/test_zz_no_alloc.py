"""jpet_mlem_iterate_noalloc - the iteration for callers that cannot allocate device memory when they need it.

Who they are: a monitoring loop that must answer within a fixed time (cudaMalloc / cudaFree stall the whole device, and
jpet_mlem_iterate grows its workspace on demand), a plug-in in a program whose own pool already holds all of HBM (cudaMalloc
fails there), a process that may not allocate after start-up.  The entry point keeps its scratch in a fixed array inside
libjpet.so (3 MiB + 256 bytes per GPU, images up to JPET_NOALLOC_MAX_PIXELS = 512 x 512) and runs the simple direct kernel.

What is checked here: its image against the one jpet_mlem_iterate (the allocating, tiled path) gives for the same events,
within the tolerance the parity tests use (1e-4 of the image maximum after one iteration; the two differ by fp32 summation
order only), on calls made one after another - the array is shared by all calls and keeps the last call's contents, so a
big grid is followed by a small one and by the big one again, each with a different start image.  The file sorts last on
purpose (pytest -x stops at the first failure); it resets the process-wide settings itself, so it gives the same result alone
in a fresh process and after the other test files.
"""
import ctypes

import numpy as np
import pytest

from paper_1502_07478_b200 import synth

TOL_1 = 1e-4    # one iteration, relative to the image maximum - the bound of tests/test_parity_gpu.py


@pytest.fixture()
def jp():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import paper_1502_07478_b200 as jp

    jp.binding.load(build_if_missing=False)   # the in-tree .so must be the one that runs
    # whatever an earlier test file left behind: back to the defaults both paths are compared under
    for name in ("force_direct", "chunk", "sub_tile_z", "exact_kernel", "stage_bytes", "poly_off", "degree_classes_off"):
        jp.jpet_set_option(name, 0)
    jp.jpet_set_option("variant", -1)
    jp.jpet_set_a3_coef(2.0)
    jp.jpet_set_gamma(0.0)
    jp.jpet_set_sigma_z_edge(0.0)
    yield jp
    jp.jpet_set_gamma(0.0)


def geom(cfg):
    return (cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel)


def both_paths(jp, ev_d, cfg, rho):
    """(image of the static-scratch call, image of jpet_mlem_iterate) for one start image, as float64 numpy arrays."""
    import torch

    rho_d = torch.from_numpy(np.ascontiguousarray(rho, dtype=np.float32)).cuda().reshape(-1)
    got, want = torch.empty_like(rho_d), torch.empty_like(rho_d)
    jp.jpet_mlem_iterate_noalloc(ev_d, *geom(cfg), rho_d, got)
    jp.jpet_mlem_iterate(ev_d, *geom(cfg), rho_d, want)
    torch.cuda.synchronize()
    return got.cpu().numpy().astype(np.float64), want.cpu().numpy().astype(np.float64)


def rel_err(got, want):
    return float(np.max(np.abs(got - want)) / np.max(want))


@pytest.mark.gpu
def test_calls_in_a_row_match_the_allocating_path(jp):
    import torch

    big, small = synth.CONFIGS["cfg2"], synth.CONFIGS["cfg1"]
    ev_big = torch.from_numpy(np.ascontiguousarray(synth.config_events(big, n=100_000))).cuda()
    ev_small = torch.from_numpy(np.ascontiguousarray(synth.config_events(small))).cuda()
    rng = np.random.default_rng(7)
    calls = [(ev_big, big, np.ones(big.n_y * big.n_z)),                                  # 200 x 200, fills 40 000 floats per part
             (ev_small, small, rng.uniform(0.2, 3.0, small.n_y * small.n_z)),             # 64 x 64 over the big call's leftovers
             (ev_big, big, rng.uniform(0.2, 3.0, big.n_y * big.n_z)),                     # and the big grid over the small one's
             (ev_big, big, np.ones(big.n_y * big.n_z))]                                   # the first call again
    images = []
    for ev_d, cfg, rho in calls:
        got, want = both_paths(jp, ev_d, cfg, rho)
        assert np.isfinite(got).all() and want.max() > 0
        assert rel_err(got, want) <= TOL_1
        assert ((got == 0) == (want == 0)).all()          # the s = 0 mask of Eq. 3
        images.append(got)
    assert rel_err(images[3], images[0]) <= TOL_1         # nothing of the calls in between is left in the result


@pytest.mark.gpu
def test_gamma_and_aliasing_and_no_events(jp):
    import torch

    cfg = synth.CONFIGS["cfg1"]
    ev_d = torch.from_numpy(np.ascontiguousarray(synth.config_events(cfg))).cuda()
    jp.jpet_set_gamma(2e-4)                                # Eq. 12's off-diagonal term is read by this path as well
    got, want = both_paths(jp, ev_d, cfg, np.ones(cfg.n_y * cfg.n_z))
    assert rel_err(got, want) <= TOL_1
    jp.jpet_set_gamma(0.0)
    plain, _ = both_paths(jp, ev_d, cfg, np.ones(cfg.n_y * cfg.n_z))
    assert rel_err(got, plain) > 1e-6                      # and changes the image
    rho = torch.ones(cfg.n_y * cfg.n_z, device="cuda")
    jp.jpet_mlem_iterate_noalloc(ev_d, *geom(cfg), rho, rho)          # in place
    assert rel_err(rho.cpu().numpy().astype(np.float64), plain) <= TOL_1
    out = torch.full((cfg.n_y * cfg.n_z,), 5.0, device="cuda")
    jp.jpet_mlem_iterate_noalloc(ev_d[:0], *geom(cfg), torch.ones_like(out), out)   # the empty sum over events
    assert float(out.abs().max()) == 0.0


def test_sizes_beyond_the_static_scratch_are_refused():
    """No GPU needed: the size check comes before the first CUDA call."""
    from paper_1502_07478_b200 import binding

    lib = binding.load()
    g, s = binding.Geometry(450, 500), binding.Sigmas(10, 40)
    fake = ctypes.c_void_p(4096)                           # never dereferenced: the call is refused first
    too_big = binding.Grid(513, 512, 1.0)
    assert too_big.n_y * too_big.n_z > binding.NOALLOC_MAX_PIXELS
    assert lib.jpet_mlem_iterate_noalloc(None, 0, g, s, too_big, fake, fake, None) == binding.JPET_E_INVAL
    text = lib.jpet_last_error().decode()
    assert "JPET_NOALLOC_MAX_PIXELS" in text and str(binding.NOALLOC_MAX_PIXELS) in text
    assert lib.jpet_mlem_iterate_noalloc(fake, 2**31, g, s, binding.Grid(64, 64, 5.0), fake, fake, None) == binding.JPET_E_INVAL
    assert lib.jpet_mlem_iterate_noalloc(None, 0, g, s, binding.Grid(64, 64, 5.0), None, fake, None) == binding.JPET_E_INVAL
    header = open(binding.os.path.join(binding.os.path.dirname(binding.os.path.dirname(binding.__file__)), "include", "jpet.h")).read()
    assert "#define JPET_NOALLOC_MAX_PIXELS (512 * 512)" in header
