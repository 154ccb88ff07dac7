"""GPU parity of the rows SURVEY.md section 8(f) added in round 2, through the C-ABI binding against the CPU oracle on the same
seeded inputs: per-event sigma_z (f1), the direct-reconstruction histogram (f2: equal to Eq. 2 in fp64 away from pixel borders), event sharding with the
accumulator sum fused into the finalise kernel (f3), the device event generator and the exact-kernel mode (f4); plus the
host ring path and the stream ordering of the workspace.  Run on the B200 box with  pytest -m gpu."""
import math
import os
import sys

import numpy as np
import pytest

from paper_1502_07478_b200 import synth

pytestmark = pytest.mark.gpu

TOL_1 = 1e-4


@pytest.fixture(scope="module")
def jp():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import paper_1502_07478_b200 as jp

    jp.binding.load(build_if_missing=False)
    yield jp
    for name in ("force_direct", "exact_kernel", "stage_bytes", "chunk"):
        jp.jpet_set_option(name, 0)
    jp.jpet_set_option("variant", -1)
    jp.jpet_set_sigma_z_edge(0.0)
    jp.jpet_set_gamma(0.0)


def geom(cfg):
    return (cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel)


def rel_err(got, want):
    return float(np.max(np.abs(got - want)) / np.max(want))


def gpu_iterate(jp, ev, cfg, rho_in, n_iter=1):
    import torch

    ev_d = torch.from_numpy(np.ascontiguousarray(ev)).cuda()
    rho = torch.from_numpy(np.ascontiguousarray(rho_in, dtype=np.float32)).cuda().reshape(-1)
    out = torch.empty_like(rho)
    if n_iter == 1:
        jp.jpet_mlem_iterate(ev_d, *geom(cfg), rho, out)
    else:
        jp.jpet_reconstruct(ev_d, *geom(cfg), rho, out, n_iter)
    return out.cpu().numpy().astype(np.float64).reshape(cfg.n_y, cfg.n_z), jp.jpet_get_counters()


# ---- (f1) sigma_z depending on the hit positions -------------------------------------------------------
@pytest.mark.parametrize("name,n,eta,frac", [("cfg1", 20000, 0.1, 0.0), ("cfg2", 200_000, 0.1, 0.0), ("cfg2", 100_000, 0.25, 0.3),
                                             ("cfg4", 20000, 0.1, 0.0), ("cfg5", 200_000, 0.1, -0.3), ("fig4", 100_000, 0.1, 0.0)])
def test_position_dependent_sigma_z(jp, oracle, name, n, eta, frac):
    """C^-1 = diag(1/sigma_z(z~u)^2, 1/sigma_z(z~d)^2, 1/sigma_dl^2) (+ gamma) per event on both sides: the tiled kernel (its VS
    instances: per-event Gaussian coefficient and chord), the direct kernel, one and several iterations.  Switching eta on
    moves the image by far more than the tolerance.  (Config 5's 512 x 512 grid needs 10^5 events or more for the image
    tolerance to be meaningful: on a sparser image single ellipse-boundary ties, R20, reach 1e-4 of the maximum.)"""
    cfg = synth.CONFIGS[name]
    ev = synth.config_events(cfg, n=n)
    ns_ = 100_000 if name == "cfg5" else 20000
    rho = np.random.default_rng(2).uniform(0.5, 2.0, (cfg.n_y, cfg.n_z)).astype(np.float32)
    gamma = frac / (math.sqrt(2.0) * (1 + eta) * cfg.sigma_z * cfg.sigma_dl)
    base, _ = gpu_iterate(jp, ev, cfg, rho)
    try:
        jp.jpet_set_sigma_z_edge(eta)
        jp.jpet_set_gamma(gamma)
        oracle.set_sigma_z_edge(jp.jpet_get_sigma_z_edge())
        oracle.set_gamma(jp.jpet_get_gamma())
        got, (ne, ns) = gpu_iterate(jp, ev, cfg, rho)
        tiled = jp.jpet_get_option("last_tiled")
        got3, _ = gpu_iterate(jp, ev[:ns_], cfg, rho, n_iter=3)
        jp.jpet_set_option("force_direct", 1)
        direct, (nd, _) = gpu_iterate(jp, ev[:ns_], cfg, rho)
        jp.jpet_set_option("force_direct", 0)
        want, one, ons = oracle.mlem_iterate(ev, *geom(cfg), rho)
        want_d, oned, _ = oracle.mlem_iterate(ev[:ns_], *geom(cfg), rho)
        want3, _, _ = oracle.reconstruct(ev[:ns_], *geom(cfg), 3, rho_init=rho)
    finally:
        jp.jpet_set_option("force_direct", 0)
        jp.jpet_set_sigma_z_edge(0.0)
        jp.jpet_set_gamma(0.0)
        oracle.set_sigma_z_edge(0.0)
        oracle.set_gamma(0.0)
    assert tiled == 1
    assert rel_err(got, want) <= TOL_1
    assert rel_err(direct, want_d) <= TOL_1 and rel_err(got3, want3) <= 3 * TOL_1
    assert ns == ons and abs(ne - one) <= 1e-5 * one + 2 and abs(nd - oned) <= 1e-5 * oned + 2
    assert rel_err(base, want) > 20 * TOL_1


# ---- (f2) direct reconstruction histogram (Eq. 2, Fig. 4b) -------------------------------------------------------------
def histogram_agrees_with_fp64(oracle, ev, cfg, got, got_outside, before=None):
    """The rule for an integer decided by floating point (R24).  The oracle is Eq. 2 in fp64 and a floor; the
    kernel computes in fp32, so a point closer to a pixel border than the fp32 rounding error may be counted on the other
    side.  With c = (c_y, c_z) the oracle's fp64 pixel coordinates, an event is BORDERLINE when a border b in {0 .. n}
    lies within eps = 2^-18 (|c| + 1) pixels of c on either axis (fp32 evaluates c to about 2^-21 (|c| + 1): eight times
    closer).  Then: (i) the counts of all other events equal the oracle's exactly - the kernel's histogram minus the
    oracle's histogram of the decided events is >= 0 everywhere and sums to the number of borderline events; (ii) every
    borderline event is in one of the pixels next to its border(s) - per pixel (and for "outside") the remainder does not
    exceed the number of borderline events that have it among their candidates.  Returns (borderline fraction, fraction
    counted in another pixel than the oracle's)."""
    n_y, n_z = cfg.n_y, cfg.n_z
    c = oracle.direct_pixel_coords(ev, cfg.R, n_y, n_z, cfg.pixel)
    finite = ~np.isnan(c).any(axis=1)
    cf = np.where(finite[:, None], c, -1e6)                                     # non-finite events: decidedly outside
    b = np.stack([np.clip(np.rint(cf[:, 0]), 0, n_y), np.clip(np.rint(cf[:, 1]), 0, n_z)], axis=1)
    near_ax = np.abs(cf - b) <= 2.0 ** -18 * (np.abs(cf) + 1.0)
    near = near_ax.any(axis=1)
    want_d, out_d = oracle.direct_histogram(ev[~near], cfg.R, n_y, n_z, cfg.pixel, hist=None if before is None else before.copy())
    resid = got.astype(np.int64) - want_d.astype(np.int64)
    resid_out = got_outside - out_d
    assert (resid >= 0).all() and resid_out >= 0
    assert int(resid.sum()) + resid_out == int(near.sum())
    cap = np.zeros((n_y, n_z), dtype=np.int64)
    cap_out = 0
    fl = np.floor(cf).astype(np.int64)
    for j in np.nonzero(near)[0]:
        cand = [([int(b[j, a]) - 1, int(b[j, a])] if near_ax[j, a] else [int(fl[j, a])]) for a in (0, 1)]
        pixels = {(iy, iz) if (0 <= iy < n_y and 0 <= iz < n_z) else None for iy in cand[0] for iz in cand[1]}
        for q in pixels:
            if q is None:
                cap_out += 1
            else:
                cap[q] += 1
    assert (resid <= cap).all() and resid_out <= cap_out
    want_all, out_all = oracle.direct_histogram(ev, cfg.R, n_y, n_z, cfg.pixel, hist=None if before is None else before.copy())
    moved = (int(np.abs(got.astype(np.int64) - want_all.astype(np.int64)).sum()) + abs(got_outside - out_all)) / 2
    n = max(len(ev), 1)
    return float(near.sum()) / n, moved / n


@pytest.mark.parametrize("name,n", [("fig4", 1_000_003), ("cfg2", 300_000), ("cfg5", 1_000_000), ("cfg1", 0)])
def test_direct_histogram_against_the_fp64_oracle(jp, oracle, name, n):
    """Integer work decided by floating point: every count equals the count of Eq. 2 in fp64 + floor, except for events within
    eps of a pixel border, which must sit in an adjacent pixel (histogram_agrees_with_fp64).  The borderline fraction is what
    eps predicts for points spread evenly over the pixels (about 4 eps: two axes, both sides of a border; at most
    4 x 2^-18 x (n_max + 1) x 1.5), and the events that really are counted across a border are at most a quarter of them.
    fig4's image fits the per-block shared-memory histogram, the others take global atomics; a slice at an odd offset takes
    the scalar loads; a second call increments."""
    import torch

    cfg = synth.CONFIGS[name]
    ev = synth.config_events(cfg, n=n)
    if n:
        ev[::1000, 0] = np.nan                    # non-finite events are outside
        ev[5::1000, 2] = 1e9                      # far outside the grid
    hist = torch.zeros(cfg.n_y * cfg.n_z, dtype=torch.int32, device="cuda")
    ev_d = torch.from_numpy(ev).cuda()
    outside = jp.jpet_direct_histogram(ev_d, cfg.R, cfg.L, cfg.n_y, cfg.n_z, cfg.pixel, hist)
    got = hist.cpu().numpy().view(np.uint32).reshape(cfg.n_y, cfg.n_z).copy()
    assert int(got.sum()) + outside == n
    near, moved = histogram_agrees_with_fp64(oracle, ev, cfg, got, outside)
    print(f"{name}: borderline fraction {near:.2e}, counted across a border {moved:.2e}")
    assert near <= 6.0 * 2.0 ** -18 * (max(cfg.n_y, cfg.n_z) + 1) and moved <= 0.25 * near + 2.0 / max(n, 1)
    if n:
        assert jp.jpet_direct_histogram(ev_d[1:70001], cfg.R, cfg.L, cfg.n_y, cfg.n_z, cfg.pixel, hist, count_outside=False) is None
        got2 = hist.cpu().numpy().view(np.uint32).reshape(cfg.n_y, cfg.n_z)
        assert int(got2.sum()) - int(got.sum()) <= 70000
        out2 = 70000 - (int(got2.sum()) - int(got.sum()))
        histogram_agrees_with_fp64(oracle, ev[1:70001], cfg, got2, out2, before=got)


def test_direct_histogram_beyond_2_30_events(jp):
    """The global-atomic path walks one tile per block, so its stride is about n: past 2^30 events a 32-bit tile offset
    wraps.  One call over 2^30 + 2^20 + 5 device-generated events (12.9 GB) must count every event once
    and give, count by count, the sum of two calls over the halves (each below 2^30)."""
    import torch

    cfg = synth.CONFIGS["cfg2"]
    n = (1 << 30) + (1 << 20) + 5
    ev_d = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    jp.jpet_generate_events(cfg.phantom, n, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, 11, ev_d)
    whole = torch.zeros(cfg.n_y * cfg.n_z, dtype=torch.int32, device="cuda")
    halves = torch.zeros_like(whole)
    out_whole = jp.jpet_direct_histogram(ev_d, cfg.R, cfg.L, cfg.n_y, cfg.n_z, cfg.pixel, whole)
    out_halves = sum(jp.jpet_direct_histogram(part, cfg.R, cfg.L, cfg.n_y, cfg.n_z, cfg.pixel, halves)
                     for part in (ev_d[: n // 2], ev_d[n // 2:]))
    assert int(whole.sum(dtype=torch.int64)) + out_whole == n
    assert out_whole == out_halves and bool((whole == halves).all())
    del ev_d
    torch.cuda.empty_cache()


# ---- (f3) event sharding: private accumulators summed in the finalise kernel ----------------------------
def test_two_shards_on_one_gpu_equal_one_call_and_the_oracle(jp, oracle):
    """Two halves of the events accumulated separately (begin / accumulate, the accumulator copied out through
    jpet_mlem_accumulator), then one jpet_mlem_end_peers over the two buffers == one jpet_mlem_iterate over all events ==
    the oracle.  This is the device-side part of the sharded path; the rank plumbing is tested with gloo on CPU."""
    import torch

    cfg = synth.CONFIGS["cfg2"]
    ev = synth.config_events(cfg, n=200_001)
    rho_np = np.random.default_rng(3).uniform(0.5, 2.0, (cfg.n_y, cfg.n_z)).astype(np.float32)
    rho = torch.from_numpy(rho_np).cuda().reshape(-1)
    ev_d = torch.from_numpy(ev).cuda()
    whole = torch.empty_like(rho)
    jp.jpet_mlem_iterate(ev_d, *geom(cfg), rho, whole)
    shards = []
    for lo, hi in ((0, 100_000), (100_000, 200_001)):
        jp.jpet_mlem_begin(*geom(cfg), rho)
        jp.jpet_mlem_accumulate(ev_d[lo:hi])
        acc = jp.jpet_mlem_accumulator()
        assert acc.numel() == cfg.n_y * cfg.n_z and acc.is_cuda
        shards.append(acc.clone())
        if lo == 0:
            jp.jpet_mlem_end(rho, torch.empty_like(rho))          # closes the iteration of the first shard
    out = torch.empty_like(rho)
    jp.jpet_mlem_end_peers(rho, out, shards)
    assert float((out - whole).abs().max() / whole.max()) <= 1e-5
    want, _, _ = oracle.mlem_iterate(ev, *geom(cfg), rho_np)
    assert rel_err(out.cpu().numpy().astype(np.float64).reshape(cfg.n_y, cfg.n_z), want) <= TOL_1
    # the view is the workspace's accumulator: summing the shards into it in place and a plain end gives the same image
    jp.jpet_mlem_begin(*geom(cfg), rho)
    jp.jpet_mlem_accumulator().copy_(shards[0] + shards[1])
    out2 = torch.empty_like(rho)
    jp.jpet_mlem_end(rho, out2)
    assert float((out2 - out).abs().max() / out.max()) <= 1e-6
    with pytest.raises(jp.JpetError):
        jp.jpet_mlem_accumulator()                                # no open iteration
    with pytest.raises(jp.JpetError):
        jp.jpet_mlem_end_peers(rho, out, shards)


def test_ipc_handle_round_trip_in_one_process(jp):
    """jpet_ipc_export gives a 64-byte handle; opening it in the exporting process is refused by CUDA (a handle is for
    another process) - the error must come back as JPET_E_CUDA, not as a crash."""
    import torch

    buf = torch.arange(1024, dtype=torch.float32, device="cuda")
    handle = jp.jpet_ipc_export(buf.data_ptr())
    assert len(handle) == 64 and any(handle)
    try:
        ptr = jp.jpet_ipc_open(handle)
    except jp.JpetError as e:
        assert e.code == -2
    else:
        view = jp.binding.device_view(ptr, 1024)
        assert float((view - buf).abs().max()) == 0.0
        del view
        jp.jpet_ipc_close(ptr)


# ---- (f4) event generator ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["cfg2", "cfg3", "fig4"])
def test_generator_matches_the_oracle_slot_by_slot(jp, oracle, name):
    """Same counter-based streams on both sides: every slot is the same event up to fp32 rounding of the arithmetic
    (1e-2 mm), except the few slots where an accept / inside / hit decision falls on the other side of a boundary in
    fp32 (they are a different, equally valid event); slots do not depend on n or first."""
    import torch

    cfg = synth.CONFIGS[name]
    n = 300_000
    ev = torch.empty((n, 3), device="cuda")
    jp.jpet_generate_events(cfg.phantom, n, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, 42, ev)
    got = ev.cpu().numpy()
    want = oracle.generate_events(cfg.phantom, n, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, 42)
    assert np.isfinite(got).all()
    close = np.max(np.abs(got.astype(np.float64) - want), axis=1) <= 1e-2
    assert close.mean() >= 1 - 2e-4, close.mean()
    part = torch.empty((1000, 3), device="cuda")
    jp.jpet_generate_events(cfg.phantom, 1000, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, 42, part, first=123_456)
    assert (part.cpu().numpy() == got[123_456:124_456]).all()


def test_generated_events_reconstruct_like_the_numpy_ones(jp, oracle):
    """The device generator feeds the same pipeline: moments and the direct-reconstruction histogram agree statistically
    with synth.py's events (the statistical pin of VERDICT item 6), and an MLEM iteration on them matches the oracle."""
    import torch

    cfg = synth.CONFIGS["cfg2"]
    n = 400_000
    ev = torch.empty((n, 3), device="cuda")
    jp.jpet_generate_events(cfg.phantom, n, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, 7, ev)
    got = ev.cpu().numpy()
    ref = synth.config_events(cfg, n=n)
    for c in range(3):
        sd = ref[:, c].std()
        assert abs(got[:, c].mean() - ref[:, c].mean()) < 5 * sd * math.sqrt(2.0 / n)
        assert abs(got[:, c].std() / sd - 1) < 0.01
    ha, _ = oracle.direct_histogram(got, cfg.R, 20, 20, 10 * cfg.pixel)
    hb, _ = oracle.direct_histogram(ref, cfg.R, 20, 20, 10 * cfg.pixel)
    ha, hb = ha.ravel().astype(float), hb.ravel().astype(float)
    m = (ha + hb) >= 40
    chi2, dof = float(np.sum((ha[m] - hb[m]) ** 2 / (ha[m] + hb[m]))), int(m.sum()) - 1
    assert chi2 < dof + 5 * math.sqrt(2 * dof), (chi2, dof)
    ones = np.ones((cfg.n_y, cfg.n_z))
    out, (ne, ns) = gpu_iterate(jp, got[:100_000], cfg, ones)
    want, one, ons = oracle.mlem_iterate(got[:100_000], *geom(cfg), ones)
    assert rel_err(out, want) <= TOL_1 and ns == ons


# ---- (f4) exact-kernel mode ---------------------------------------------------------------------------------
@pytest.mark.parametrize("eta", [0.0, 0.1])
def test_exact_kernel_mode(jp, oracle, eta):
    """The theta integral instead of Eq. 7 on the same pixel sets: the GPU's 64-node trapezoid in tan(theta) around the
    integrand's peak against the oracle's trapezoid over the whole interval; the mode moves the image measurably."""
    cfg = synth.CONFIGS["cfg1"]
    ev = synth.config_events(cfg, n=3000)
    rho = np.random.default_rng(4).uniform(0.5, 2.0, (cfg.n_y, cfg.n_z)).astype(np.float32)
    eq7, _ = gpu_iterate(jp, ev, cfg, rho)
    try:
        jp.jpet_set_sigma_z_edge(eta)
        oracle.set_sigma_z_edge(eta)
        jp.jpet_set_option("exact_kernel", 64)
        got, (ne, ns) = gpu_iterate(jp, ev, cfg, rho)
        assert jp.jpet_get_option("last_tiled") == 0
        oracle.set_exact_kernel(4001)
        want, one, ons = oracle.mlem_iterate(ev, *geom(cfg), rho)
    finally:
        jp.jpet_set_option("exact_kernel", 0)
        jp.jpet_set_sigma_z_edge(0.0)
        oracle.set_exact_kernel(0)
        oracle.set_sigma_z_edge(0.0)
    assert rel_err(got, want) <= TOL_1
    assert ns == ons and abs(ne - one) <= 2
    if eta == 0.0:
        assert 1e-5 < rel_err(eq7, want) < 2e-2


# ---- host ring path and stream ordering -----------------------------------------------------------------------------------
def test_host_ring_path_over_several_iterations(jp, oracle):
    """when the events exceed the staging budget they are streamed through two ring slots once per
    iteration; the slots must not be overwritten while the previous iteration's kernels still read them.  The
    stage_bytes option forces the path with a small input."""
    import torch

    cfg = synth.CONFIGS["cfg2"]
    ev = synth.config_events(cfg, n=150_000)
    want, _, _ = oracle.reconstruct(ev, *geom(cfg), 4)
    try:
        jp.jpet_set_option("stage_bytes", 12 * 20_000)            # 7.5 chunks of 20 000 events
        out = torch.empty(cfg.n_y * cfg.n_z).pin_memory()
        for _ in range(3):                                        # repeated: a race would show as run-to-run differences
            jp.jpet_reconstruct_host(torch.from_numpy(ev).pin_memory(), *geom(cfg), None, out, 4, chunk_events=20_000)
            assert rel_err(out.numpy().astype(np.float64).reshape(cfg.n_y, cfg.n_z), want) <= 3 * TOL_1
    finally:
        jp.jpet_set_option("stage_bytes", 0)


def test_calls_on_different_streams_are_ordered(jp, oracle):
    """include/jpet.h: the workspace is used by one stream at a time - back-to-back iterations on two streams (the second
    reads what the first wrote) give the same result as on one stream."""
    import torch

    cfg = synth.CONFIGS["cfg2"]
    ev = torch.from_numpy(synth.config_events(cfg, n=300_000)).cuda()
    rho = torch.ones(cfg.n_y * cfg.n_z, device="cuda")
    a, b = torch.empty_like(rho), torch.empty_like(rho)
    jp.jpet_mlem_iterate(ev, *geom(cfg), rho, a)
    jp.jpet_mlem_iterate(ev, *geom(cfg), a, b)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    a2, b2 = torch.empty_like(rho), torch.empty_like(rho)
    jp.jpet_mlem_iterate(ev, *geom(cfg), rho, a2, stream=s1)
    jp.jpet_mlem_iterate(ev, *geom(cfg), a2, b2, stream=s2)
    ne, _ = jp.jpet_get_counters(stream=s2)
    torch.cuda.synchronize()
    assert ne > 0 and float((b2 - b).abs().max() / b.max()) <= 1e-5


def test_an_error_return_leaves_the_stream_ordering_intact(jp):
    """every way out of a call that has entered the workspace records the ordering event, error returns
    included, and keeps the text of the error that caused it.  An accumulate that fails its argument check on a second
    stream, in the middle of an iteration that runs on two streams, must not disturb the iteration."""
    import ctypes

    import torch

    cfg = synth.CONFIGS["cfg2"]
    ev = torch.from_numpy(synth.config_events(cfg, n=200_000)).cuda()
    rho = torch.ones(cfg.n_y * cfg.n_z, device="cuda")
    want, got = torch.empty_like(rho), torch.empty_like(rho)
    jp.jpet_mlem_iterate(ev, *geom(cfg), rho, want)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    lib = jp.binding.load()
    jp.jpet_mlem_begin(*geom(cfg), rho, stream=s1)
    jp.jpet_mlem_accumulate(ev[:100_000], stream=s1)
    assert lib.jpet_mlem_accumulate(None, 5, ctypes.c_void_p(s2.cuda_stream)) == jp.binding.JPET_E_INVAL
    assert "NULL events" in jp.jpet_last_error()
    jp.jpet_mlem_accumulate(ev[100_000:], stream=s2)
    jp.jpet_mlem_end(rho, got, stream=s1)
    torch.cuda.synchronize()
    assert float((got - want).abs().max() / want.max()) <= 1e-5


# ---- (f3) the sharded iteration across two PROCESSES (one GPU: the ranks' kernels never wait on one another) ------------
def _p2p_worker(rank, world, port, n_events, n_iter, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK="0", WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import torch
    import torch.distributed as dist

    from paper_1502_07478_b200.sharding import ShardedMlem, shard_range

    torch.cuda.set_device(0)
    dist.init_process_group("gloo")                                 # host plumbing only: handles, barriers
    cfg = synth.CONFIGS["cfg2"]
    events = synth.config_events(cfg, n=n_events)                   # every rank draws the same list and takes its shard
    lo, hi = shard_range(len(events), rank, world)
    sm = ShardedMlem(dist, mode="p2p")                              # accumulators mapped with cudaIpc, summed in the finalise kernel
    rho = torch.ones(cfg.n_y * cfg.n_z, device="cuda")
    out = torch.empty_like(rho)
    sm.reconstruct(torch.from_numpy(events[lo:hi]).cuda(), geom(cfg), rho, out, n_iter)
    torch.cuda.synchronize()
    img = out.cpu().numpy().reshape(cfg.n_y, cfg.n_z)
    sm.close()
    dist.destroy_process_group()
    q.put((rank, lo, hi, img))


def test_two_processes_share_accumulators_through_cuda_ipc(jp, oracle):
    """ShardedMlem(mode="p2p") as bench.py --gpus N runs it, with two processes on this one GPU and gloo for the handle exchange
    and the barriers: each rank accumulates its half of the events, maps the other rank's accumulator with cudaIpc and
    finalises over both - every rank must hold the image one process computes from all events (and the oracle's)."""
    import socket

    import torch.multiprocessing as mp

    n_events, n_iter = 60_001, 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_p2p_worker, args=(r, 2, port, n_events, n_iter, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=600) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert (got[0][1], got[0][2], got[1][1], got[1][2]) == (0, n_events // 2, n_events // 2, n_events)
    assert (got[0][3] == got[1][3]).all()                           # peers are read in rank order: identical bits on every rank
    cfg = synth.CONFIGS["cfg2"]
    want, _, _ = oracle.reconstruct(synth.config_events(cfg, n=n_events), *geom(cfg), n_iter)
    assert rel_err(got[0][3].astype(np.float64), want) <= 1e-4


# ---- degree classes: the events whose own truncation bound allows it are walked with the degree-3 exponent polynomial ----
@pytest.mark.parametrize("name,n,low", [("cfg4", 120_000, "large_deg3"), ("cfg2", 150_000, "mid18_deg3"), ("cfg5", 60_000, "")])
def test_degree_classes_do_not_change_the_image(jp, oracle, name, n, low):
    """with a degree-4 plan the sort puts the events that pass low_degree_ok into a second set of bins and
    the degree-3 instance of the kernel shape walks them.  Same image as with one class (the truncation error is far below
    fp32 summation noise), same counters, and both match the oracle; config 5's shape has no degree-3 instance."""
    cfg = synth.CONFIGS[name]
    ev = synth.config_events(cfg, n=n)
    rho = np.random.default_rng(7).uniform(0.5, 2.0, (cfg.n_y, cfg.n_z)).astype(np.float32)
    got, (ne, ns) = gpu_iterate(jp, ev, cfg, rho)
    assert jp.jpet_shape_name(jp.jpet_get_option("last_variant_low")) == low
    jp.jpet_set_option("degree_classes_off", 1)
    try:
        one, (ne1, ns1) = gpu_iterate(jp, ev, cfg, rho)
        assert jp.jpet_get_option("last_variant_low") == -1
    finally:
        jp.jpet_set_option("degree_classes_off", 0)
    want, one_evals, one_skipped = oracle.mlem_iterate(ev, *geom(cfg), rho)
    assert (ne, ns) == (ne1, ns1) and ns == one_skipped and abs(ne - one_evals) <= 1e-5 * one_evals + 2
    assert np.max(np.abs(got - one)) <= 5e-6 * one.max()
    assert rel_err(got, want) <= TOL_1 and rel_err(one, want) <= TOL_1
