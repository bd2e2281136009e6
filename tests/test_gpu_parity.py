"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerances (BASELINE.json north_star): per-iteration exit-wave and object relative L2 <= 1e-4,
<= 1e-3 after 50 iterations.  Integer/bit-exact parts: frame order bookkeeping (fetch by index).
"""
import numpy as np
import pytest

from paper_2202_03144_b200 import synth

pytestmark = pytest.mark.gpu

TOL_ITER = 1e-4
TOL_RUN = 1e-3


def rel(a, b):
    a, b = np.asarray(a, np.complex128).ravel(), np.asarray(b, np.complex128).ravel()
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2202_03144_b200 import binding
    binding.lib()
    return binding


def make(B, s, **par):
    return B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(**par))


def well_lit(s, frac=0.1):
    """SURVEY.md 8(c) parity protocol: the region d_O > frac * max d_O, d_O = sum_j sum_k |P_k|^2 placed at r_j."""
    d = np.zeros(s.obj0.shape)
    p2 = np.sum(np.abs(np.asarray(s.probe0).reshape(-1, s.n, s.n)) ** 2, 0)
    for y, x in s.pos:
        d[y:y + s.n, x:x + s.n] += p2
    return d > frac * d.max()


# ------------------------------------------------------------------------------ T2: FFT alone
@pytest.mark.parametrize("n", [64, 128, 256, 512])
def test_fft2_vs_oracle(B, oracle_mod, n):
    import torch
    rng = np.random.default_rng(n)
    x = (rng.standard_normal((5, n, n)) + 1j * rng.standard_normal((5, n, n))).astype(np.complex64)
    d = torch.from_numpy(x).cuda()
    f = B.test_fft2(d.clone()).cpu().numpy()
    want = np.stack([oracle_mod.fft2(v) for v in x])
    assert rel(f, want) < 2e-6
    back = B.test_fft2(torch.from_numpy(want.astype(np.complex64)).cuda(), inverse=True).cpu().numpy()
    assert rel(back, x) < 2e-6


@pytest.mark.parametrize("impl,n", [(0, 64), (0, 128), (0, 256), (0, 512), (1, 256)])
def test_fft_rows_both_implementations_vs_library(B, n, impl):
    """The row pass alone: the product's packed-fp32 line FFT (impl 0) and the tensor-core DFT micro-benchmark kernel (impl 1,
    csrc/fft_mma.cuh: two radix-16 stages in mma.sync TF32 with a 3-term split) against numpy's FFT in double, at the FFT tolerance
    north_star sets for the DFT-as-GEMM question (2e-6)."""
    import torch
    rng = np.random.default_rng(100 + n + impl)
    x = (rng.standard_normal((6, n, n)) + 1j * rng.standard_normal((6, n, n))).astype(np.complex64)
    x[0, 0] = 0; x[0, 0, 3] = 1.0                                           # a delta: one pure twiddle per output, catches index slips
    d = torch.from_numpy(x).cuda()
    got = B.test_fft_rows(d, impl=impl).cpu().numpy()
    want = np.fft.fft(x.astype(np.complex128), axis=-1)
    assert rel(got, want) < 2e-6, rel(got, want)
    assert np.abs(got[0, 0] - want[0, 0]).max() < 2e-6
    if impl == 1:
        with pytest.raises(B.PtychoError):
            B.test_fft_rows(torch.zeros((1, 128, 128), dtype=torch.complex64, device="cuda"), impl=1)


# ------------------------------------------------------------- T3/T4 on config 0 (full size)
@pytest.mark.parametrize("probe_start", [10 ** 9, 0])
def test_cfg0_dm_free_running(B, oracle_mod, probe_start):
    s = synth.make_config(0)
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(probe_start=probe_start))
    g = make(B, s, probe_start=probe_start)
    for it in range(10):
        o.iterate("DM", 1)
        g.iterate("DM", 1)
        assert rel(g.fetch_object(), o.O) < TOL_RUN, it
    assert rel(g.fetch_exit_waves(), o.psi) < TOL_RUN
    assert rel(g.fetch_probe(), o.P) < TOL_RUN
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)
    sel = np.array([5, 63, 0, 17], np.int32)                 # caller numbering survives the sort
    assert rel(g.fetch_exit_waves(sel), o.psi[sel]) < TOL_RUN


def test_cfg0_dm_teacher_forced(B, oracle_mod):
    s = synth.make_config(0)
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities)
    g = make(B, s)
    o.iterate("DM", 1)
    g.iterate("DM", 1)
    for it in range(1, 6):
        g.set_object(o.O)
        g.set_probe(o.P)
        g.set_exit_waves(o.psi.astype(np.complex64))
        o.iterate("DM", 1)
        g.iterate("DM", 1)
        assert rel(g.fetch_exit_waves(), o.psi) < TOL_ITER, it
        assert rel(g.fetch_object(), o.O) < TOL_ITER, it
        assert rel(g.fetch_probe(), o.P) < TOL_ITER, it


@pytest.mark.parametrize("alg", ["EPIE_MB", "LSQML"])
def test_cfg0_minibatch(B, oracle_mod, alg):
    s = synth.make_config(0)
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(batch_size=16), keep_revised=True)
    g = make(B, s, batch_size=16)
    for it in range(10):
        o.iterate(alg, 1)
        g.iterate(alg, 1)
        assert rel(g.fetch_object(), o.O) < TOL_RUN, it
        assert rel(g.fetch_probe(), o.P) < TOL_RUN, it
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3, atol=1e-9)
    if alg == "LSQML":
        assert np.allclose(g.fetch_steps(), np.array(o.steps), rtol=2e-3)
    assert g.eval_error() == pytest.approx(o.eval_error(), rel=2e-3)


def test_revised_waves_teacher_forced(B, oracle_mod):
    """Full-batch ePIE: the oracle's revised waves of iteration t belong to the state before it."""
    s = synth.make_config(0)
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, keep_revised=True)
    g = make(B, s)
    for it in range(3):
        g.set_object(o.O)
        g.set_probe(o.P)
        rv = g.revised_waves()
        o.iterate("EPIE_MB", 1)
        g.iterate("EPIE_MB", 1)
        assert rel(rv, o.revised) < TOL_ITER
        assert rel(g.fetch_object(), o.O) < TOL_ITER and rel(g.fetch_probe(), o.P) < TOL_ITER


# -------------------------------------------------- every size, modes, uint16, masks, pbound
@pytest.mark.parametrize("n,h,side,step,k,alg,kw", [
    (64, 160, 5, 13, 1, "DM", dict(pbound=0.2)),
    (64, 160, 5, 13, 3, "LSQML", dict(batch_size=7)),
    (64, 160, 5, 13, 2, "DM", dict(pbound=0.1)),
    (128, 300, 5, 31, 1, "EPIE_MB", dict(batch_size=10)),
    (128, 300, 5, 31, 1, "DM", dict(pbound=0.12)),
    (256, 520, 4, 61, 1, "DM", dict(pbound=0.5)),
    (256, 520, 4, 61, 3, "LSQML", dict(batch_size=6)),
    (256, 520, 3, 90, 1, "EPIE_MB", dict(batch_size=4, probe_start=2)),
    (512, 900, 3, 150, 1, "DM", dict(pbound=0.5)),
    (512, 900, 2, 200, 2, "LSQML", dict()),
])
def test_sizes_modes_uint16(B, oracle_mod, n, h, side, step, k, alg, kw):
    s = synth.make_custom(n, h, side, step, k=k, peak=2e4, dtype=np.uint16, jitter=3, seed=n + k,
                          probe_kind="zone" if alg == "DM" else "disk")
    s.intensities[1, 3, 5] = 65535                             # a masked pixel (R3)
    s.intensities[2, 0, 0] = 65535
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, kw)
    g = make(B, s, **kw)
    for it in range(4):
        o.iterate(alg, 1)
        g.iterate(alg, 1)
        assert rel(g.fetch_object(), o.O) < TOL_ITER * (it + 1), it
        assert rel(g.fetch_probe(), o.P) < TOL_ITER * (it + 1), it
    if alg == "DM":
        assert rel(g.fetch_exit_waves(), o.psi) < 4 * TOL_ITER
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)


def test_switching_algorithms_and_state(B, oracle_mod):
    """DM after a minibatch algorithm re-initialises psi = P O_j; the counter is global."""
    s = synth.make_config(0)
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(batch_size=16, probe_start=3))
    g = make(B, s, batch_size=16, probe_start=3)
    for alg, n in (("DM", 2), ("EPIE_MB", 2), ("DM", 2), ("LSQML", 1)):
        o.iterate(alg, n)
        g.iterate(alg, n)
    assert rel(g.fetch_object(), o.O) < TOL_RUN and rel(g.fetch_probe(), o.P) < TOL_RUN
    assert len(g.fetch_error()) == 7
    with pytest.raises(B.PtychoError):
        g.fetch_exit_waves()                                   # ESTATE: a minibatch ran last


def test_error_codes(B):
    s = synth.make_config(0)
    bad = s.pos.copy()
    bad[3, 1] = 192 - 63
    with pytest.raises(B.PtychoError, match="EBOUNDS"):
        B.Ptycho(s.obj0, s.probe0, bad, s.intensities)
    with pytest.raises(B.PtychoError):
        B.Ptycho(s.obj0, s.probe0[:, :48, :48], s.pos, s.intensities[:, :48, :48])
    g = B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(disable_dm=1))
    with pytest.raises(B.PtychoError, match="ESTATE"):
        g.iterate("DM", 1)
    g.iterate("EPIE_MB", 1)
    assert g.launch_count() > 0


def test_device_resident_inputs(B, oracle_mod):
    """Device pointers are accepted everywhere (intensities borrowed, state fetched to device)."""
    import torch
    s = synth.make_config(0)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    g = B.Ptycho(dev(s.obj0.astype(np.complex64)), dev(s.probe0.astype(np.complex64)), s.pos,
                 dev(s.intensities), B.default_params())
    g.iterate("DM", 3)
    out = torch.empty((192, 192), dtype=torch.complex64, device="cuda")
    g.fetch_object(out)
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities).iterate("DM", 3)
    assert rel(out.cpu().numpy(), o.O) < TOL_RUN


# ------------------------------------------------- full size, in the configuration bench.py times
def test_cfg2_full_size_sampled_frames_and_object(B, oracle_mod):
    """Config 2 as `bench.py` runs it (DM, 256x256, J = 10 000, uint16, pbound 0.5, default queue
    geometry).  In the first DM iteration psi_j' depends only on (O0, P0, I_j), so the oracle can
    compute sampled frames one by one: an oracle built from the sampled positions alone must give
    the GPU's exit waves for those frames.  The object is checked on everything the oracle can
    afford: where the host has the memory, one full oracle iteration; in any case the closed form
    of step 5 on a window, from the GPU's own exit waves of the frames that cover it."""
    import psutil
    s = synth.make_config(2)
    par = dict(pbound=s.params["pbound"])
    g = make(B, s, **par)
    g.iterate("DM", 1)
    J, n = s.n_pos, s.n
    rng = np.random.default_rng(7)
    idx = np.sort(rng.choice(J, 24, replace=False)).astype(np.int32)
    idx[0], idx[-1] = 0, J - 1                                   # first and last frame of the scan
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos[idx], s.intensities[idx], par)
    o.iterate("DM", 1)
    psi_g = g.fetch_exit_waves(idx)
    for k in range(len(idx)):
        assert rel(psi_g[k], o.psi[k]) < TOL_ITER, (k, idx[k])
    assert np.isfinite(g.fetch_error()[0])
    O_g, P_g = g.fetch_object(), g.fetch_probe()

    # window check: O_new = (sum_j conj(P0) psi_j' + eps O0) / (sum_j |P0|^2 + eps), eps = delta max|P0|^2 (R5)
    y0, x0, w = 2000, 2010, 48
    cover = np.where((s.pos[:, 0] <= y0) & (s.pos[:, 0] + n >= y0 + w) & (s.pos[:, 1] <= x0) & (s.pos[:, 1] + n >= x0 + w))[0]
    part = np.where((s.pos[:, 0] < y0 + w) & (s.pos[:, 0] + n > y0) & (s.pos[:, 1] < x0 + w) & (s.pos[:, 1] + n > x0))[0]
    assert len(cover) > 5
    P0 = s.probe0[0].astype(np.complex128)
    num = np.zeros((w, w), np.complex128)
    den = np.zeros((w, w))
    psi_w = g.fetch_exit_waves(part.astype(np.int32))
    for k, j in enumerate(part):
        py, px = int(s.pos[j, 0]), int(s.pos[j, 1])
        ys, xs = max(y0, py), max(x0, px)
        ye, xe = min(y0 + w, py + n), min(x0 + w, px + n)
        sl = (slice(ys - py, ye - py), slice(xs - px, xe - px))
        num[ys - y0:ye - y0, xs - x0:xe - x0] += np.conj(P0[sl]) * psi_w[k, 0][sl]
        den[ys - y0:ye - y0, xs - x0:xe - x0] += np.abs(P0[sl]) ** 2
    eps = 1e-2 * np.max(np.abs(P0) ** 2)
    expect = (num + eps * s.obj0[y0:y0 + w, x0:x0 + w]) / (den + eps)
    assert rel(O_g[y0:y0 + w, x0:x0 + w], expect) < TOL_ITER

    if psutil.virtual_memory().available > 40 * 2 ** 30:         # psi in double: 10.5 GB
        of = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, par)
        of.iterate("DM", 1)
        assert rel(O_g, of.O) < TOL_ITER and rel(P_g, of.P) < TOL_ITER
        assert np.allclose(g.fetch_error(), of.err, rtol=2e-3)
    g.destroy()


def test_dm_queue_geometry_does_not_change_the_result(B, oracle_mod, monkeypatch):
    """The megakernel's wave size, lag and ring slack are scheduling only: any legal setting gives the
    oracle's result (ragged last wave, ring wrap-around and J smaller than a wave included)."""
    s = synth.make_custom(128, 420, 7, 37, k=1, peak=2e4, dtype=np.uint16, jitter=3, seed=5, probe_kind="zone")
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(pbound=0.3)).iterate("DM", 3)
    for M, D, X in ((1, 2, 0), (3, 2, 1), (5, 3, 4), (64, 2, 0)):
        monkeypatch.setenv("PTYCHO_MEGA_M", str(M))
        monkeypatch.setenv("PTYCHO_MEGA_D", str(D))
        monkeypatch.setenv("PTYCHO_MEGA_X", str(X))
        g = make(B, s, pbound=0.3)
        g.iterate("DM", 3)
        assert rel(g.fetch_object(), o.O) < 3 * TOL_ITER, (M, D, X)
        assert rel(g.fetch_exit_waves(), o.psi) < 3 * TOL_ITER, (M, D, X)
        g.destroy()


def test_deterministic_mode_is_bit_reproducible_and_matches_the_oracle(B, oracle_mod):
    """deterministic = 1: the overlap sums are formed by owner-computes kernels in slot order
    (dm_det.cuh), no floating-point atomics: two runs agree bit for bit; the atomic mode agrees with
    both within the parity tolerance; minibatch algorithms and K > 1 are refused."""
    s = synth.make_custom(128, 420, 7, 37, k=1, peak=2e4, dtype=np.uint16, jitter=3, seed=9, probe_kind="zone")
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(pbound=0.3)).iterate("DM", 4)
    runs = []
    for _ in range(2):
        g = make(B, s, pbound=0.3, deterministic=1)
        g.iterate("DM", 4)
        runs.append((g.fetch_object(), g.fetch_probe(), g.fetch_exit_waves(), g.fetch_error()))
        with pytest.raises(B.PtychoError, match="EUNSUPPORTED"):
            g.iterate("EPIE_MB", 1)
        g.destroy()
    for a, b in zip(*runs):
        assert np.array_equal(a.view(np.uint8), b.view(np.uint8))
    assert rel(runs[0][0], o.O) < 4 * TOL_ITER and rel(runs[0][1], o.P) < 4 * TOL_ITER and rel(runs[0][2], o.psi) < 4 * TOL_ITER
    assert np.allclose(runs[0][3], o.err, rtol=2e-3)
    s3 = synth.make_custom(64, 160, 5, 13, k=2, peak=2e4, dtype=np.uint16, jitter=3, seed=3)
    with pytest.raises(B.PtychoError, match="EUNSUPPORTED"):
        make(B, s3, deterministic=1)


# --------------------------------------- the other configurations of BASELINE.json at their own sizes
def _free_run(B, oracle_mod, s, alg, iters, par, tol, check_psi=False):
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, par)
    g = make(B, s, **par)
    o.iterate(alg, iters)
    g.iterate(alg, iters)
    ro, rp = rel(g.fetch_object(), o.O), rel(g.fetch_probe(), o.P)
    assert ro < tol and rp < tol, (ro, rp)
    if check_psi:
        assert rel(g.fetch_exit_waves(), o.psi) < tol
    assert np.allclose(g.fetch_error(), o.err, rtol=5e-3)
    g.destroy()


def test_cfg1_full_50_iterations_epie_and_dm(B, oracle_mod):
    """Config 1 as written (128x128, 1024 positions, fp32 Poisson counts, batch 256): 50 free-running
    iterations of ePIE-minibatch and of DM (pbound 0.12) within the 1e-3 bound of north_star."""
    s = synth.make_config(1)
    _free_run(B, oracle_mod, s, "EPIE_MB", 50, dict(batch_size=256), TOL_RUN)
    _free_run(B, oracle_mod, s, "DM", 50, dict(pbound=s.params["pbound_dm"]), TOL_RUN, check_psi=True)


def test_cfg3_lsqml_three_modes_truncated_scan(B, oracle_mod):
    """Config 3 (LSQML-style, 256x256, 3 modes, uint16, 6144^2 object, batch 512) on the first 2048
    positions of its scan (4 batches): 5 free-running iterations.  The full 20 000-position scan is
    timed but not compared: one oracle iteration of it takes minutes."""
    s = synth.make_config(3, n_pos=2048)
    _free_run(B, oracle_mod, s, "LSQML", 5, dict(batch_size=512), TOL_RUN)


def test_cfg4_dm_512_truncated_scan(B, oracle_mod):
    """Config 4 (DM, 512x512, uint16, 8192^2 object, pbound 0.5) on the first 1024 positions of its
    Fermat spiral: 3 free-running iterations, exit waves included (the oracle's psi of the full
    16 384 positions would need 69 GB)."""
    s = synth.make_config(4, n_pos=1024)
    _free_run(B, oracle_mod, s, "DM", 3, dict(pbound=s.params["pbound"]), 3 * TOL_ITER, check_psi=True)


# ------------------------------------------------------------------- frame preparation (S:8(f) f2)
@pytest.mark.parametrize("in_dt,out_dt", [(np.uint16, np.uint16), (np.uint16, np.float32), (np.float32, np.uint16), (np.float32, np.float32)])
def test_prepare_frames_bit_exact(B, oracle_mod, in_dt, out_dt):
    """Integer / byte work: the GPU result equals the oracle bit for bit -- centred crop with the window
    hanging over the detector edge, threshold, saturation, sentinels; host and device pointers."""
    import torch
    rng = np.random.default_rng(11)
    raw = rng.integers(0, 70000, (5, 150, 170)).clip(0, 65535).astype(np.uint16)
    raw = raw if in_dt == np.uint16 else (raw.astype(np.float32) * 1.37 - 20.0).astype(np.float32)
    for center, n in (((75, 85), 128), ((10, 160), 64), ((149, 0), 32), ((3, 168), 6),
                      ((40, 50), 8), ((70, 90), 24), ((60, 20), 40), ((80, 80), 72)):   # n = 6 and n % 16 == 8: the scalar path
        ref = oracle_mod.prepare_frames(raw, center, n, threshold=300.0, saturation=60000.0, out_dtype=out_dt)
        got = B.prepare_frames(raw, center, n, threshold=300.0, saturation=60000.0, out_dtype=out_dt)
        assert got.dtype == ref.dtype and np.array_equal(got, ref), (center, n)
        got_d = B.prepare_frames(torch.from_numpy(raw).cuda(), center, n, threshold=300.0, saturation=60000.0, out_dtype=out_dt)
        assert np.array_equal(got_d.cpu().numpy(), ref), (center, n)
    plain = B.prepare_frames(raw, (75, 85), 64, out_dtype=out_dt)        # no threshold, no saturation
    assert np.array_equal(plain, oracle_mod.prepare_frames(raw, (75, 85), 64, out_dtype=out_dt))
    scale = (0.5 + rng.random(5)).astype(np.float32)                     # R23 rotation, R24 normalisation
    for rot in range(4):
        for center, n in (((75, 85), 64), ((3, 160), 32), ((70, 90), 24)):
            ref = oracle_mod.prepare_frames(raw, center, n, threshold=300.0, saturation=60000.0, out_dtype=out_dt, rot90=rot, frame_scale=scale)
            got = B.prepare_frames(raw, center, n, threshold=300.0, saturation=60000.0, out_dtype=out_dt, rot90=rot, frame_scale=scale)
            assert np.array_equal(got, ref), (rot, center, n)


# ------------------------------------------------- the steady-state path bench.py times, at full size
def test_cfg2_full_size_steady_state_teacher_forced(B, oracle_mod, record_property):
    """Config 2 as `bench.py` times it AFTER the first iteration: psi_j is read from the 5.2 GB store, the reflector is not
    the identity, the ring wraps ~70 times.  psi_j' of a DM iteration depends only on (O, P, psi_j, I_j), so it is teacher-forced:
    a perturbed object, psi_j = Q O_j for a perturbed probe Q (built on the device), ONE iteration, then 48 sampled frames (first,
    last, random: both sides of many ring wraps) against oracles holding just those frames with the same psi_j.  The object is
    compared with the oracle on a window, from an oracle that holds every frame overlapping the window."""
    import torch
    s = synth.make_config(2)
    par = dict(pbound=s.params["pbound"])
    J, n = s.n_pos, s.n
    rng = np.random.default_rng(21)
    obj = (s.obj_true * (1 + 0.05 * (rng.standard_normal(s.obj_true.shape) + 1j * rng.standard_normal(s.obj_true.shape)))).astype(np.complex64)
    q = (s.probe0[0] * (1 + 0.03 * (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))))).astype(np.complex64)
    g = make(B, s, **par)
    g.set_object(obj)
    od, qd = torch.from_numpy(obj).cuda(), torch.from_numpy(q).cuda()
    psi = torch.empty((J, 1, n, n), dtype=torch.complex64, device="cuda")
    for j, (y, x) in enumerate(s.pos):
        psi[j, 0] = qd * od[y:y + n, x:x + n]
    g.set_exit_waves(psi)
    g.iterate("DM", 1)                                           # steady-state branch: psi is valid, nothing is re-initialised
    idx = np.sort(rng.choice(J, 48, replace=False)).astype(np.int32)
    idx[0], idx[-1] = 0, J - 1
    psi_g = g.fetch_exit_waves(idx)
    o = oracle_mod.Oracle(obj, s.probe0, s.pos[idx], s.intensities[idx], par)
    o.psi = np.stack([(q * obj[y:y + n, x:x + n])[None] for y, x in s.pos[idx]]).astype(np.complex128)
    o.iterate("DM", 1)
    worst = max(rel(psi_g[k], o.psi[k]) for k in range(len(idx)))
    assert worst < TOL_ITER, worst
    # object on a window, against an oracle that holds all frames overlapping it
    y0, x0, w = 2000, 2100, 48
    cover = np.array([j for j, (y, x) in enumerate(s.pos) if y < y0 + w and y + n > y0 and x < x0 + w and x + n > x0], np.int32)
    assert len(cover) > 20
    ow = oracle_mod.Oracle(obj, s.probe0, s.pos[cover], s.intensities[cover], par)
    ow.psi = np.stack([(q * obj[y:y + n, x:x + n])[None] for y, x in s.pos[cover]]).astype(np.complex128)
    ow.iterate("DM", 1)
    O_g = g.fetch_object()
    assert rel(O_g[y0:y0 + w, x0:x0 + w], ow.O[y0:y0 + w, x0:x0 + w]) < TOL_ITER
    assert np.isfinite(g.fetch_error()[-1])
    # The same check in the regime most of bench.py's iterations are in: after 14 iterations every frame is inside its power bound,
    # the kernel runs its split form and the short pass 3.  Iteration 15 is teacher-forced from the GPU's own state.
    gs = make(B, s, **par)
    gs.iterate("DM", 14)
    O14, P14, psi14 = gs.fetch_object(), gs.fetch_probe(), gs.fetch_exit_waves(idx)
    gs.iterate("DM", 1)
    o15 = oracle_mod.Oracle(O14, P14, s.pos[idx], s.intensities[idx], par)
    o15.psi = psi14.astype(np.complex128)
    o15.iterate("DM", 1)
    psi15 = gs.fetch_exit_waves(idx)
    assert max(rel(psi15[k], o15.psi[k]) for k in range(len(idx))) < TOL_ITER
    mean_e = o15.err[0] * o15.sum_I / (len(idx) * n * n)
    assert mean_e < par["pbound"], mean_e                        # the sampled frames are inside the bound: this WAS the short path
    ow15 = oracle_mod.Oracle(O14, P14, s.pos[cover], s.intensities[cover], par)
    ow15.psi = gs.fetch_exit_waves(cover).astype(np.complex128)  # (already iteration 15's waves: the object step uses the NEW waves)
    O15 = gs.fetch_object()
    # object window from the closed form of step 5 with the new waves: O + sum_j conj(P)(psi'_j - P O_j) / (d_O + eps)
    num = np.zeros((w, w), complex); den = np.zeros((w, w))
    for k, j in enumerate(cover):
        py, px = s.pos[j]
        ys, ye, xs, xe = max(y0, py), min(y0 + w, py + n), max(x0, px), min(x0 + w, px + n)
        sl = (slice(ys - py, ye - py), slice(xs - px, xe - px))
        num[ys - y0:ye - y0, xs - x0:xe - x0] += np.conj(P14[0][sl]) * ow15.psi[k, 0][sl]
        den[ys - y0:ye - y0, xs - x0:xe - x0] += np.abs(P14[0][sl]) ** 2
    eps = 1e-2 * np.max(np.abs(s.probe0) ** 2)
    assert rel(O15[y0:y0 + w, x0:x0 + w], (num + eps * O14[y0:y0 + w, x0:x0 + w]) / (den + eps)) < TOL_ITER
    gs.destroy()
    # three free-running iterations against the full oracle, where the host can hold psi in double (10.5 GB)
    import psutil
    ran_full = psutil.virtual_memory().available > 40 * 2 ** 30
    record_property("cfg2_full_oracle_branch_ran", ran_full)
    print(f"cfg2 full-size free-running oracle branch ran: {ran_full}")
    if ran_full:
        g2 = make(B, s, **par)
        of = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, par)
        g2.iterate("DM", 3)
        of.iterate("DM", 3)
        lit = well_lit(s)
        O2 = g2.fetch_object()
        assert rel(O2, of.O) < 3 * TOL_ITER and rel(O2[lit], of.O[lit]) < 3 * TOL_ITER and rel(g2.fetch_probe(), of.P) < 3 * TOL_ITER
        assert rel(g2.fetch_exit_waves(idx), of.psi[idx]) < 3 * TOL_ITER
        assert np.allclose(g2.fetch_error(), of.err, rtol=2e-3)
        g2.destroy()
    g.destroy()


def test_cfg4_full_size_second_iteration_teacher_forced(B, oracle_mod):
    """Config 4 at FULL size (N = 512, J = 16 384: a 34 GB exit-wave store, 4.3 G complex elements -- indices beyond 2^31 -- and
    the ring capped at 96 MB), as `bench.py --config 4` runs it.  The first iteration forms psi in pass 1; the SECOND reads the
    store, so it is the one checked: teacher-forced from the GPU's state after iteration 1 on 24 sampled frames (first, last,
    random), and the object on a window from the closed form of the overlap update with the new waves of every frame over it."""
    s = synth.make_config(4)
    par = dict(pbound=s.params["pbound"])
    J, n = s.n_pos, s.n
    assert J == 16384 and n == 512
    rng = np.random.default_rng(44)
    idx = np.sort(rng.choice(J, 24, replace=False)).astype(np.int32)
    idx[0], idx[-1] = 0, J - 1
    g = make(B, s, **par)
    g.iterate("DM", 1)
    O1, P1, psi1 = g.fetch_object(), g.fetch_probe(), g.fetch_exit_waves(idx)
    g.iterate("DM", 1)
    o = oracle_mod.Oracle(O1, P1, s.pos[idx], s.intensities[idx], par)
    o.psi = psi1.astype(np.complex128)
    o.iterate("DM", 1)
    psi2 = g.fetch_exit_waves(idx)
    worst = max(rel(psi2[k], o.psi[k]) for k in range(len(idx)))
    assert worst < TOL_ITER, worst
    cy, cx = s.obj0.shape[0] // 2, s.obj0.shape[1] // 2
    y0, x0, w = cy - 40, cx + 25, 32
    cover = np.array([j for j, (y, x) in enumerate(s.pos) if y < y0 + w and y + n > y0 and x < x0 + w and x + n > x0], np.int32)
    assert len(cover) > 20
    psi_c = g.fetch_exit_waves(cover)                            # iteration 2's waves
    num = np.zeros((w, w), complex); den = np.zeros((w, w))
    for k, j in enumerate(cover):
        py, px = s.pos[j]
        ys, ye, xs, xe = max(y0, py), min(y0 + w, py + n), max(x0, px), min(x0 + w, px + n)
        sl = (slice(ys - py, ye - py), slice(xs - px, xe - px))
        num[ys - y0:ye - y0, xs - x0:xe - x0] += np.conj(P1[0][sl]) * psi_c[k, 0][sl].astype(complex)
        den[ys - y0:ye - y0, xs - x0:xe - x0] += np.abs(P1[0][sl]) ** 2
    eps = 1e-2 * np.max(np.abs(s.probe0) ** 2)                   # R5, fixed at init
    O2 = g.fetch_object()
    assert rel(O2[y0:y0 + w, x0:x0 + w], (num + eps * O1[y0:y0 + w, x0:x0 + w]) / (den + eps)) < TOL_ITER
    e = g.fetch_error()
    assert np.all(np.isfinite(e)) and e[1] < e[0]
    g.destroy()


def test_dm_inside_the_power_bound_paths(B, oracle_mod):
    """Frames whose error is inside the power bound (R6, rb = 1) take the short pass 3 (psi' = P O_j, no transform, no
    scatter), and once most frames are there the megakernel switches to its split form (error-only column pass, the full pass
    only for the frames that need it).  A bound chosen so that the frames cross it during the run exercises every combination;
    the oracle knows none of this."""
    s = synth.make_custom(128, 420, 7, 37, k=1, peak=2e4, dtype=np.uint16, jitter=3, seed=31, probe_kind="zone")
    lit = well_lit(s)
    for pb in (0.6, 3.0):
        o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(pbound=pb))
        g = make(B, s, pbound=pb)
        inside = []
        for it in range(14):
            o.iterate("DM", 1)
            g.iterate("DM", 1)
            tol = TOL_ITER * (it + 1)
            Og = g.fetch_object()
            assert rel(Og, o.O) < tol and rel(Og[lit], o.O[lit]) < tol and rel(g.fetch_probe(), o.P) < tol, (pb, it)
            inside.append(float(o.err[-1] * o.sum_I / (o.J * s.n * s.n)))
        assert rel(g.fetch_exit_waves(), o.psi) < 14 * TOL_ITER
        assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)
        assert inside[0] > pb and inside[-1] < pb, inside          # the run really crossed the bound
        g.destroy()


@pytest.mark.parametrize("n,h,side,step", [(256, 520, 4, 61), (512, 900, 3, 150)])
def test_dm_fp32_intensities_large_frames(B, oracle_mod, n, h, side, step):
    """The float-intensity instantiations of the megakernel at 256^2 and 512^2 (every other test of these sizes uses uint16)."""
    s = synth.make_custom(n, h, side, step, k=1, peak=2e4, dtype=np.float32, jitter=3, seed=n + 7, probe_kind="zone")
    s.intensities[1, 3, 5] = -1.0                              # a masked pixel (R3)
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(pbound=0.4))
    g = make(B, s, pbound=0.4)
    lit = well_lit(s)
    for it in range(4):
        o.iterate("DM", 1)
        g.iterate("DM", 1)
        Og = g.fetch_object()
        assert rel(Og, o.O) < TOL_ITER * (it + 1) and rel(Og[lit], o.O[lit]) < TOL_ITER * (it + 1), it
        assert rel(g.fetch_probe(), o.P) < TOL_ITER * (it + 1), it
    assert rel(g.fetch_exit_waves(), o.psi) < 4 * TOL_ITER
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)


@pytest.mark.parametrize("alg,k", [("DM", 1), ("EPIE_MB", 1), ("LSQML", 2), ("DM", 2)])
def test_zero_amplitude_branch_R2(B, oracle_mod, alg, k):
    """R2: where the transformed wave is exactly zero the projection gives sqrt(I) with zero phase (mode 0) and 0 (other modes).
    One frame sits on an object patch that is exactly 0, so its whole spectrum takes that branch -- in the megakernel (K = 1 DM)
    and in the three-pass kernels (everything else), which share the threshold |Phi|^2 <= 1e-30."""
    s = synth.make_custom(64, 200, 4, 30, k=k, peak=2e4, dtype=np.float32, jitter=0, seed=5, probe_kind="disk")
    y, x = s.pos[5]
    obj = s.obj0.copy()
    obj[y:y + 64, x:x + 64] = 0
    kw = {}                                                    # full batch: every frame sees the initial object
    o = oracle_mod.Oracle(obj, s.probe0, s.pos, s.intensities, kw, keep_revised=True)
    g = B.Ptycho(obj, s.probe0, s.pos, s.intensities, B.default_params(**kw))
    if alg != "DM":
        rv = g.revised_waves(np.array([5], np.int32))
    o.iterate(alg, 1)
    g.iterate(alg, 1)
    if alg != "DM":
        assert rel(rv[0], o.revised[5]) < TOL_ITER             # F^-1[sqrt(I)] in mode 0, zero in the others
        if k > 1:
            assert np.abs(rv[0, 1:]).max() == 0
    else:
        assert rel(g.fetch_exit_waves(np.array([5], np.int32)), o.psi[5:6]) < TOL_ITER
    o.iterate(alg, 1)
    g.iterate(alg, 1)
    assert rel(g.fetch_object(), o.O) < 2 * TOL_ITER and rel(g.fetch_probe(), o.P) < 2 * TOL_ITER
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)


def test_lsqml_teacher_forced_256_three_modes(B, oracle_mod):
    """Per-iteration parity (<= 1e-4) of the LSQML-style step at 256^2 with three probe modes: the GPU is reset to the oracle's
    state before every iteration; revised waves, object, probe modes and the (a, b) steps are compared."""
    s = synth.make_custom(256, 520, 4, 61, k=3, peak=2e4, dtype=np.uint16, jitter=3, seed=259, probe_kind="disk")
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(batch_size=6), keep_revised=True)
    g = make(B, s, batch_size=6)
    lit = well_lit(s)
    for it in range(3):
        g.set_object(o.O)
        g.set_probe(o.P)
        n_before = len(o.steps)
        o.iterate("LSQML", 1)
        g.iterate("LSQML", 1)
        Og = g.fetch_object()
        assert rel(Og, o.O) < TOL_ITER and rel(Og[lit], o.O[lit]) < TOL_ITER and rel(g.fetch_probe(), o.P) < TOL_ITER, it
        assert np.allclose(g.fetch_steps()[n_before:], np.array(o.steps[n_before:]), rtol=1e-3), it
    g.set_object(o.O)
    g.set_probe(o.P)
    sel = np.array([0, 3, 15], np.int32)                       # frames of the first batch (16 frames, 3 strided batches): they see this state
    rv = g.revised_waves(sel)
    o.iterate("LSQML", 1)
    assert rel(rv, o.revised[sel]) < TOL_ITER


def test_handoff_stress_deterministic_bitwise(B, monkeypatch):
    """The cross-CTA hand-off of the megakernel (relaxed polls, release increments, ring reuse) under many queue geometries:
    in deterministic mode the result does not depend on timing, so 10 random (M, D, X) x 20 iterations must reproduce the default
    geometry BIT FOR BIT (object, probe, exit waves).  A missed dependency would read a half-written frame and break equality."""
    s = synth.make_custom(64, 260, 9, 21, k=1, peak=2e4, dtype=np.uint16, jitter=3, seed=77, probe_kind="zone")
    def run():
        g = B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(pbound=0.3, deterministic=1))
        g.iterate("DM", 20)
        out = (g.fetch_object(), g.fetch_probe(), g.fetch_exit_waves(), g.fetch_error())
        g.destroy()
        return out
    ref = run()
    rng = np.random.default_rng(3)
    for _ in range(10):
        M, D, X = int(rng.integers(1, 9)), int(rng.integers(2, 7)), int(rng.integers(0, 5))
        monkeypatch.setenv("PTYCHO_MEGA_M", str(M))
        monkeypatch.setenv("PTYCHO_MEGA_D", str(D))
        monkeypatch.setenv("PTYCHO_MEGA_X", str(X))
        got = run()
        for a, b in zip(got, ref):
            assert np.array_equal(a, b), (M, D, X)


# ------------------------------------------------------------------ f1: textbook variants
@pytest.mark.parametrize("sweeps", [1, 2])
def test_sequential_dm_overlap_projection(B, oracle_mod, sweeps):
    """dm_sweeps = n: object from the new exit waves, then the probe from the same waves and the NEW object, n sweeps."""
    s = synth.make_custom(128, 420, 7, 37, k=1, peak=2e4, dtype=np.uint16, jitter=3, seed=41, probe_kind="zone")
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(pbound=0.3, dm_sweeps=sweeps))
    g = make(B, s, pbound=0.3, dm_sweeps=sweeps)
    lit = well_lit(s)
    for it in range(5):
        if it:                                                  # teacher-forced: per-iteration tolerance
            g.set_object(o.O); g.set_probe(o.P); g.set_exit_waves(o.psi.astype(np.complex64))
        o.iterate("DM", 1)
        g.iterate("DM", 1)
        Og = g.fetch_object()
        assert rel(Og, o.O) < TOL_ITER and rel(Og[lit], o.O[lit]) < TOL_ITER and rel(g.fetch_probe(), o.P) < TOL_ITER, it
        assert rel(g.fetch_exit_waves(), o.psi) < TOL_ITER, it
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)
    with pytest.raises(B.PtychoError, match="EUNSUPPORTED"):
        B.Ptycho(s.obj0, np.concatenate([s.probe0, s.probe0]), s.pos, s.intensities, B.default_params(dm_sweeps=1))


def test_position_sequential_epie(B, oracle_mod):
    """B = 1: the paper's position-sequential ePIE through the minibatch path, one frame per batch."""
    s = synth.make_custom(64, 200, 5, 24, k=1, peak=2e4, dtype=np.float32, jitter=2, seed=43, probe_kind="disk")
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(batch_size=1))
    g = make(B, s, batch_size=1)
    for it in range(3):
        o.iterate("EPIE_MB", 1)
        g.iterate("EPIE_MB", 1)
        assert rel(g.fetch_object(), o.O) < TOL_ITER * (it + 1) and rel(g.fetch_probe(), o.P) < TOL_ITER * (it + 1), it
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)


# ------------------------------------------------------------------ f3: streaming ingestion
@pytest.mark.parametrize("dtype", [np.uint16, np.float32])
def test_streaming_ingestion(B, oracle_mod, dtype):
    """Frames arrive in three pieces while the reconstruction runs: every ptycho_iterate works on the frames
    present, with the batches of R8 formed over them.  The oracle sees the same thing as a chain of runs on the growing prefix,
    each continuing from the object and probe of the last."""
    import torch
    s = synth.make_custom(64, 220, 6, 24, k=1, peak=2e4, dtype=dtype, jitter=2, seed=51, probe_kind="disk")
    J = len(s.pos)
    g = B.Ptycho(s.obj0, s.probe0, s.pos, None, B.default_params(batch_size=5), stream_dtype=dtype)
    with pytest.raises(B.PtychoError, match="ESTATE"):
        g.iterate("EPIE_MB", 1)                                  # nothing present yet
    O, P = s.obj0.astype(complex), s.probe0.astype(complex)
    errs = []
    pinned = torch.from_numpy(s.intensities).pin_memory()
    for lo, hi in ((0, 10), (10, 23), (23, J)):
        with pytest.raises(B.PtychoError, match="EINVAL"):
            g.append_frames(lo + 1, s.intensities[lo + 1:hi])    # a gap
        g.append_frames(lo, pinned[lo:hi] if lo else s.intensities[lo:hi])   # pinned torch slice and plain numpy
        assert g.frames_present() == hi
        if hi < J:
            with pytest.raises(B.PtychoError, match="ESTATE"):
                g.iterate("DM", 1)                               # DM wants every frame
        g.iterate("EPIE_MB", 2)
        o = oracle_mod.Oracle(O, P, s.pos[:hi], s.intensities[:hi], dict(batch_size=5)).iterate("EPIE_MB", 2)
        O, P = o.O, o.P
        errs += o.err
        assert rel(g.fetch_object(), O) < 4 * TOL_ITER and rel(g.fetch_probe(), P) < 4 * TOL_ITER, hi
    g.wait_frames()
    assert np.allclose(g.fetch_error(), errs, rtol=2e-3)
    g.iterate("DM", 2)                                           # complete now
    o = oracle_mod.Oracle(O, P, s.pos, s.intensities)
    first = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities)
    o.eps_O, o.eps_P = first.eps_O, first.eps_P                 # R5: the blend constants were fixed at init, from the initial state
    o.iterate("DM", 2)
    assert rel(g.fetch_object(), o.O) < 8 * TOL_ITER
    assert g.eval_error() == pytest.approx(o.eval_error(), rel=2e-3)


@pytest.mark.parametrize("n,h,side,step,k,batch", [(64, 200, 5, 24, 1, 7), (128, 300, 5, 31, 3, 0), (256, 520, 4, 61, 2, 6)])
def test_lsqml_per_frame_steps(B, oracle_mod, n, h, side, step, k, batch):
    """LSQML_PF (R25): one (a_j, b_j) per frame, weighted second scatter, mean probe step -- against the oracle, free-running."""
    s = synth.make_custom(n, h, side, step, k=k, peak=2e4, dtype=np.uint16, jitter=3, seed=n + 3 * k, probe_kind="disk")
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(batch_size=batch))
    g = make(B, s, batch_size=batch)
    lit = well_lit(s)
    for it in range(4):
        o.iterate("LSQML_PF", 1)
        g.iterate("LSQML_PF", 1)
        Og = g.fetch_object()
        assert rel(Og, o.O) < TOL_ITER * (it + 1) and rel(Og[lit], o.O[lit]) < TOL_ITER * (it + 1), it
        assert rel(g.fetch_probe(), o.P) < TOL_ITER * (it + 1), it
    gs, os_ = g.fetch_steps(), np.array(o.steps)               # one pair per frame; inside a batch the library visits frames in its
    assert gs.shape == os_.shape                               # own (spatial) order, so batches are compared as sets
    sizes = [len(b) for b in oracle_mod.batches(len(s.pos), batch)] * 4
    i0 = 0
    for sz in sizes:
        a, b = gs[i0:i0 + sz], os_[i0:i0 + sz]
        assert np.allclose(a[np.lexsort(a.T)], b[np.lexsort(b.T)], rtol=2e-3, atol=1e-5), i0
        i0 += sz
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)


# ------------------------------------------------------------------ f4 (part): probe-mode orthogonalisation (R26)
def test_mode_orthogonalisation(B, oracle_mod):
    """After a few LSQML-style iterations the three modes are no longer orthogonal; ptycho_orthogonalize_modes must give the
    oracle's mixing of the SAME modes (Gram eigen-decomposition, phase convention), leave sum_k |P_k|^2 alone, and mix stored DM
    exit waves alike."""
    s = synth.make_custom(64, 200, 5, 24, k=3, peak=2e4, dtype=np.float32, jitter=2, seed=61, probe_kind="disk")
    g = make(B, s, batch_size=8)
    g.iterate("LSQML", 3)
    g.iterate("DM", 1)                                           # fills the exit-wave store (K = 3: three-pass DM path)
    p_before, psi_before = g.fetch_probe(), g.fetch_exit_waves()
    flat = p_before.reshape(3, -1).astype(np.complex128)
    gram = flat @ flat.conj().T
    assert np.abs(gram[0, 1]) > 1e-4 * gram[0, 0].real           # really non-orthogonal now
    want_p, want_psi = oracle_mod.orthogonalize_modes(p_before, psi_before)
    g.orthogonalize_modes()
    p_after = g.fetch_probe()
    assert rel(p_after, want_p) < 2e-6 and rel(g.fetch_exit_waves(), want_psi) < 2e-6
    assert np.allclose(np.sum(np.abs(p_after) ** 2, 0), np.sum(np.abs(p_before) ** 2, 0), rtol=1e-5)
    g.iterate("LSQML", 1)                                        # and the run goes on
    assert np.isfinite(g.fetch_error()[-1])
    one = make(B, synth.make_config(0))
    one.orthogonalize_modes()                                    # K = 1: no-op


def test_split_form_under_queue_geometries(B, oracle_mod, monkeypatch):
    """The split form of the DM queue (error-only column pass, one pass-2b item per wave, short pass 3) under several queue
    geometries, ragged last wave and ring wrap included: with a wide power bound the frames are inside it after a few
    iterations, so the later ones run in that form; the oracle's result must come out whatever M, D, X are."""
    s = synth.make_custom(128, 420, 7, 37, k=1, peak=2e4, dtype=np.uint16, jitter=3, seed=71, probe_kind="zone")
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(pbound=3.0)).iterate("DM", 12)
    assert o.err[6] * o.sum_I / (o.J * 128 * 128) < 3.0          # inside the bound half-way: the later iterations used the split form
    for M, D, X in ((1, 2, 0), (3, 2, 1), (5, 3, 4), (64, 2, 0), (6, 6, 5)):
        monkeypatch.setenv("PTYCHO_MEGA_M", str(M))
        monkeypatch.setenv("PTYCHO_MEGA_D", str(D))
        monkeypatch.setenv("PTYCHO_MEGA_X", str(X))
        g = make(B, s, pbound=3.0)
        g.iterate("DM", 12)
        assert rel(g.fetch_object(), o.O) < 10 * TOL_ITER and rel(g.fetch_probe(), o.P) < 10 * TOL_ITER, (M, D, X)
        assert rel(g.fetch_exit_waves(), o.psi) < 10 * TOL_ITER, (M, D, X)
        assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)
        g.destroy()


@pytest.mark.parametrize("size", ["small", pytest.param("cfg2_full", marks=pytest.mark.skipif(
    not __import__("os").environ.get("PTYCHO_LONG_TESTS"), reason="opt-in (PTYCHO_LONG_TESTS=1): builds N = 256 twice, config 2 at full size"))])
def test_strict_sync_build_is_bit_identical(tmp_path, size):
    """The megakernel's hand-off polls with relaxed loads (DESIGN.md section 5.2 says what that assumes).  A build with
    -DPTYCHO_STRICT_SYNC polls with ld.acquire.gpu instead; in deterministic mode the two builds must agree bit for bit over a
    multi-iteration run with ring wrap-around -- a reordering the relaxed protocol allowed would show up as a difference.
    "cfg2_full" (opt-in) does the same at the size bench.py times: J = 10 000 frames of 256^2, 12 iterations, default geometry."""
    import hashlib, os, subprocess, sys
    script = tmp_path / "run.py"
    make_scan = ('s = synth.make_custom(64, 260, 9, 21, k=1, peak=2e4, dtype=np.uint16, jitter=3, seed=77, probe_kind="zone"); pb, its = 0.3, 25'
                 if size == "small" else 's = synth.make_config(2); pb, its = s.params["pbound"], 12')
    script.write_text(('''
import hashlib, sys, numpy as np
sys.path.insert(0, %r)
from paper_2202_03144_b200 import binding, synth
binding.build()
MAKE_SCAN
g = binding.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, binding.default_params(pbound=pb, deterministic=1))
g.iterate("DM", its)
'''.replace("MAKE_SCAN", make_scan) + '''
h = hashlib.sha1()
for a in (g.fetch_object(), g.fetch_probe(), g.fetch_exit_waves(), g.fetch_error()):
    h.update(np.ascontiguousarray(a).tobytes())
print("HASH", h.hexdigest())
''') % os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    out = {}
    for tag, defs in (("relaxed", ""), ("strict", "-DPTYCHO_STRICT_SYNC")):
        env = dict(os.environ, PTYCHO_BUILD_TAG=tag, PTYCHO_BUILD_DEFS=defs)
        if size == "small":
            env.update(PTYCHO_BUILD_ONLY_N="64", PTYCHO_MEGA_M="2", PTYCHO_MEGA_D="2", PTYCHO_MEGA_X="1")
        else:
            env.update(PTYCHO_BUILD_ONLY_N="256")
        r = subprocess.run([sys.executable, str(script)], env=env, capture_output=True, text=True, timeout=1800)
        assert r.returncode == 0, r.stderr[-2000:]
        out[tag] = [l for l in r.stdout.splitlines() if l.startswith("HASH")][0]
    assert out["relaxed"] == out["strict"]


# ------------------------------------------------------------- one scan over several GPUs (reading R27)
@pytest.mark.parametrize("world,n,h,side,step,jitter,dtype,pbound", [
    (2, 64, 420, 16, 21, 3, np.uint16, 0.3),       # two bands, frames cross the power bound on the way
    (3, 64, 420, 16, 21, 3, np.float32, 0.0),      # three bands: the middle one exchanges with both neighbours
    (5, 128, 400, 9, 30, 2, np.uint16, 0.3),       # thin bands (a band is lower than a frame): every rank overlaps several others
    (1, 64, 300, 9, 21, 0, np.float32, 0.0)])      # one shard: the two-call form of the plain iteration
def test_sharded_scan_matches_the_single_device_oracle(B, oracle_mod, world, n, h, side, step, jitter, dtype, pbound):
    """The frames are split over `world` shards (row bands), every shard is its own C-ABI context holding only its frames, and the
    overlap sums are completed by the exchange step between ptycho_shard_begin and ptycho_shard_end (sharded.py).  The result has
    a plain definition -- the single-device iteration over ALL frames -- so the oracle is the ordinary one, which knows nothing of
    shards.  All shards run in one process on this one GPU, stepped in lockstep (LocalGroup): the same calls, exchange code and
    order of additions as the distributed run, whose communication layer is covered by the gloo test in test_abi_and_host.py."""
    from paper_2202_03144_b200 import sharded
    s = synth.make_custom(n, h, side, step, k=1, peak=2e4 if dtype == np.uint16 else None, dtype=dtype, jitter=jitter, seed=31,
                          probe_kind="zone")
    par = dict(pbound=pbound, probe_start=2)
    plan = sharded.shard_plan(s.pos, n, h, h, world)
    if world == 5:
        assert max(len(e) for e in plan.exchange) >= 3      # the thin-band case really has many-way overlaps
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, par)
    grp = sharded.LocalGroup(plan, s.obj0, s.probe0, s.pos, s.intensities, **par)
    lit = well_lit(s)
    for it in range(12):
        o.iterate("DM", 1)
        grp.iterate(1)
        O = grp.fetch_object()
        assert rel(O, o.O) < TOL_RUN and rel(O[lit], o.O[lit]) < TOL_RUN, it
    assert rel(grp.fetch_exit_waves(), o.psi) < TOL_RUN
    assert rel(grp.fetch_probe(), o.P) < TOL_RUN
    assert np.allclose(grp.fetch_error(), o.err, rtol=2e-3)
    # every shard holds the same probe (the sums were completed before the blend), and on rows two shards cover their objects agree
    P0 = grp.shards[0].core.fetch_probe()
    objs = [sh.core.fetch_object() for sh in grp.shards]
    for r, sh in enumerate(grp.shards):
        assert np.array_equal(sh.core.fetch_probe(), P0)
        for q, lo, hi in plan.exchange[r]:
            assert rel(objs[r][lo:hi], objs[q][lo:hi]) < 1e-6
    # the plain single-context run of the same scan, for scale: the sharded result is as close to the oracle as it is
    g = make(B, s, **par)
    g.iterate("DM", 12)
    assert rel(O, g.fetch_object()) < 1e-4
    g.destroy()
    grp.destroy()


def test_shard_contexts_refuse_what_they_do_not_support(B):
    s = synth.make_custom(64, 300, 6, 21, k=1, seed=3)
    with pytest.raises(B.PtychoError):                      # K > 1
        s2 = synth.make_custom(64, 300, 6, 21, k=2, seed=3)
        B.Ptycho(s2.obj0, s2.probe0, s2.pos, s2.intensities, B.default_params(shard_total_pos=len(s2.pos)))
    with pytest.raises(B.PtychoError):                      # deterministic mode
        B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(shard_total_pos=len(s.pos), deterministic=1))
    with pytest.raises(B.PtychoError):                      # fewer frames in the scan than in the shard
        B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(shard_total_pos=3))
    g = B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(shard_total_pos=len(s.pos)))
    with pytest.raises(B.PtychoError):
        g.iterate("DM", 1)                                  # a shard is driven by begin / end
    with pytest.raises(B.PtychoError):
        g.shard_end()                                       # ... which alternate
    g.shard_begin()
    with pytest.raises(B.PtychoError):
        g.shard_begin()
    g.shard_end()
    plain = make(B, s)
    with pytest.raises(B.PtychoError):
        plain.shard_begin()                                 # and an ordinary context is not a shard
    plain.destroy()
    g.destroy()


# ------------------------------------------------------------- sub-pixel scan positions (reading R28)
@pytest.mark.parametrize("n,h,side,step,k,dtype,pbound,batch", [
    (64, 300, 6, 21, 1, np.float32, 0.0, 9),
    (64, 300, 6, 21, 2, np.uint16, 0.3, 0),
    (128, 420, 5, 40, 3, np.uint16, 0.0, 7),
    (256, 600, 3, 90, 1, np.float32, 0.0, 4)])
def test_subpixel_positions_epie_minibatch(B, oracle_mod, n, h, side, step, k, dtype, pbound, batch):
    """ePIE-minibatch with fractional positions: the probe every frame sees is the Fourier-shifted one, the probe term is shifted
    back before it is summed.  Against oracle/subpixel.py (fp64 numpy, pinned in test_oracle_pins.py), free-running."""
    from oracle import subpixel
    s = synth.make_custom(n, h, side, step, k=k, peak=2e4 if dtype == np.uint16 else None, dtype=dtype, jitter=2, seed=41,
                          probe_kind="zone")
    rng = np.random.default_rng(17)
    frac = rng.uniform(0, 1, (len(s.pos), 2)).astype(np.float32)
    frac[0] = 0.0                                            # an exactly integer position among them
    par = dict(batch_size=batch, probe_start=1, pbound=pbound, alpha_obj=0.9, alpha_probe=0.8)
    o = subpixel.SubpixelOracle(s.obj0, s.probe0, s.pos, frac, s.intensities, par)
    g = B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(subpixel_yx=frac, **par))
    for it in range(4):
        o.iterate(1)
        g.iterate("EPIE_MB", 1)
        ro, rp = rel(g.fetch_object(), o.O), rel(g.fetch_probe(), o.P)
        assert ro < TOL_ITER * (it + 1) and rp < TOL_ITER * (it + 1), (it, ro, rp)
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)
    assert np.isclose(g.eval_error(), o.eval_error(), rtol=2e-3)          # the data-fit error of the CURRENT O, P, shifted probes
    # the fractions matter at this tolerance: the ordinary path on the same input is far away
    z = B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(**par))
    z.iterate("EPIE_MB", 4)
    assert rel(z.fetch_object(), o.O) > 50 * TOL_ITER
    z.destroy()
    with pytest.raises(B.PtychoError):                       # not with per-frame LSQML steps
        g.iterate("LSQML_PF", 1)
    with pytest.raises(B.PtychoError):
        g.revised_waves(np.arange(2, dtype=np.int32))
    g.destroy()


@pytest.mark.parametrize("n,h,side,step,k,dtype,batch,probe_start", [
    (64, 300, 6, 21, 1, np.float32, 9, 0),
    (64, 300, 6, 21, 3, np.uint16, 12, 1),
    (256, 600, 3, 90, 2, np.uint16, 0, 0)])
def test_subpixel_positions_lsqml(B, oracle_mod, n, h, side, step, k, dtype, batch, probe_start):
    """The LSQML-style joint step with fractional positions: A11, b1, b2 from the canvas closed forms (exact with shifted probes),
    A22 and A12 from the per-frame gather with shifted probes and shifted probe directions.  Objects, probes, error history and the
    step lengths (a, b) of every batch against oracle/subpixel.py."""
    from oracle import subpixel
    s = synth.make_custom(n, h, side, step, k=k, peak=2e4 if dtype == np.uint16 else None, dtype=dtype, jitter=2, seed=47,
                          probe_kind="zone")
    rng = np.random.default_rng(19)
    frac = rng.uniform(0, 1, (len(s.pos), 2)).astype(np.float32)
    par = dict(batch_size=batch, probe_start=probe_start, lsq_lambda=0.1)
    o = subpixel.SubpixelOracle(s.obj0, s.probe0, s.pos, frac, s.intensities, par)
    g = B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(subpixel_yx=frac, **par))
    for it in range(3):
        o.iterate(1, "LSQML")
        g.iterate("LSQML", 1)
        ro, rp = rel(g.fetch_object(), o.O), rel(g.fetch_probe(), o.P)
        assert ro < TOL_ITER * (it + 1) and rp < TOL_ITER * (it + 1), (it, ro, rp)
    assert np.allclose(g.fetch_steps(), np.array(o.steps), rtol=2e-3, atol=1e-6)
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)
    g.destroy()


@pytest.mark.parametrize("n,h,side,step,k,dtype,pbound,probe_start", [
    (64, 300, 6, 21, 1, np.uint16, 0.3, 2),
    (64, 300, 6, 21, 2, np.float32, 0.0, 0),
    (256, 600, 3, 90, 1, np.uint16, 0.4, 1)])
def test_subpixel_positions_dm(B, oracle_mod, n, h, side, step, k, dtype, pbound, probe_start):
    """DM with fractional positions (the three-pass kernels with per-frame probes: the megakernel shares one probe among the frames
    of an item): exit waves, object, probe and error history against oracle/subpixel.py over six free-running iterations, the
    first of which forms psi_j = P_jk O_j."""
    from oracle import subpixel
    s = synth.make_custom(n, h, side, step, k=k, peak=2e4 if dtype == np.uint16 else None, dtype=dtype, jitter=2, seed=53,
                          probe_kind="zone")
    rng = np.random.default_rng(29)
    frac = rng.uniform(0, 1, (len(s.pos), 2)).astype(np.float32)
    par = dict(pbound=pbound, probe_start=probe_start)
    o = subpixel.SubpixelOracle(s.obj0, s.probe0, s.pos, frac, s.intensities, par)
    g = B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(subpixel_yx=frac, **par))
    for it in range(6):
        o.iterate(1, "DM")
        g.iterate("DM", 1)
        ro, rp = rel(g.fetch_object(), o.O), rel(g.fetch_probe(), o.P)
        assert ro < TOL_RUN and rp < TOL_RUN, (it, ro, rp)
    assert rel(g.fetch_exit_waves(), o.psi) < TOL_RUN
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)
    # switching algorithms keeps working: a minibatch iteration invalidates psi, the next DM iteration re-forms it with the shifted probes
    o.iterate(1, "EPIE_MB"); g.iterate("EPIE_MB", 1)
    o.iterate(1, "DM"); g.iterate("DM", 1)
    assert rel(g.fetch_object(), o.O) < TOL_RUN and rel(g.fetch_exit_waves(), o.psi) < TOL_RUN
    g.destroy()


def test_subpixel_zero_fractions_reproduce_the_ordinary_path(B):
    """delta_j = 0: the per-frame probes are F^-1 F P = P up to fp32 rounding, so the sub-pixel path must track the ordinary one."""
    s = synth.make_custom(64, 300, 6, 21, k=2, seed=43, jitter=2)
    par = dict(batch_size=9, probe_start=0)
    g = B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(subpixel_yx=np.zeros((len(s.pos), 2), np.float32), **par))
    z = B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(**par))
    g.iterate("EPIE_MB", 3); z.iterate("EPIE_MB", 3)
    assert rel(g.fetch_object(), z.fetch_object()) < 1e-5 and rel(g.fetch_probe(), z.fetch_probe()) < 1e-5
    with pytest.raises(B.PtychoError):                       # a fraction outside [0, 1)
        B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(subpixel_yx=np.full((len(s.pos), 2), 1.0, np.float32)))
    with pytest.raises(B.PtychoError):
        B.Ptycho(s.obj0, s.probe0, s.pos, s.intensities, B.default_params(subpixel_yx=np.zeros((len(s.pos), 2), np.float32), deterministic=1))
    g.destroy(); z.destroy()


# ------------------------------------------------------------- degenerate and extreme inputs (task brief: "the degenerate cases the method has")
def _scan_from(obj, probe, pos, dtype=np.float32, peak=None, seed=3):
    """Intensities of an arbitrary (object, probe, positions) through the package's seeded generator."""
    _, inten, _ = synth.simulate(obj, probe, np.asarray(pos, np.int32), peak, seed, dtype, 2)
    return inten


@pytest.mark.parametrize("alg", ["DM", "EPIE_MB", "LSQML"])
def test_single_frame_on_an_object_of_exactly_the_frame_size(B, oracle_mod, alg):
    """J = 1 and H = W = N: one wave (a ragged one: M = 6 slots per item), one minibatch of one frame, every object pixel covered
    once, the position (0, 0) the only legal one."""
    n = 64
    obj = synth.make_object(n, n, 8)
    probe = synth.probe_disk(n, n * 0.3125)[None]
    pos = np.zeros((1, 2), np.int32)
    inten = _scan_from(obj, probe, pos)
    par = dict(batch_size=1, pbound=0.0)
    obj0 = np.ones_like(obj)
    o = oracle_mod.Oracle(obj0, probe, pos, inten, par)
    g = B.Ptycho(obj0, probe, pos, inten, B.default_params(**par))
    for it in range(4):
        o.iterate(alg, 1)
        g.iterate(alg, 1)
        assert rel(g.fetch_object(), o.O) < TOL_RUN and rel(g.fetch_probe(), o.P) < TOL_RUN, (alg, it)
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3, atol=1e-12)
    with pytest.raises(B.PtychoError):                      # (0, 1) would hang over the edge: no wrap-around, no clamping
        B.Ptycho(obj0, probe, np.array([[0, 1]], np.int32), inten)
    g.destroy()


@pytest.mark.parametrize("alg", ["DM", "LSQML", "EPIE_MB"])
def test_eight_probe_modes(B, oracle_mod, alg):
    """K = PTYCHO_MAX_MODES = 8 at N = 64 (the column pass loops the modes and parks their spectra in S); K = 9 is refused."""
    n, K = 64, 8
    rng = np.random.default_rng(23)
    base = synth.probe_disk(n, n * 0.3125)
    yy, xx = np.mgrid[0:n, 0:n] - n / 2
    modes = np.stack([base * (1 + 0.0 * yy) if k == 0 else base * (np.cos(0.07 * k * yy) + 1j * np.sin(0.05 * k * xx)) * 0.6 ** k for k in range(K)])
    obj = synth.make_object(170, 170, 9)
    pos = synth.raster_positions(5, 5, 21, (8, 8), jitter=2, seed=4)
    inten = _scan_from(obj, modes, pos, dtype=np.uint16, peak=2e4)
    par = dict(batch_size=9, pbound=0.2)
    probe0 = (modes * (1 + 0.02 * (rng.standard_normal(modes.shape) + 1j * rng.standard_normal(modes.shape)))).astype(np.complex64)
    obj0 = np.ones_like(obj)
    o = oracle_mod.Oracle(obj0, probe0, pos, inten, par)
    g = B.Ptycho(obj0, probe0, pos, inten, B.default_params(**par))
    o.iterate(alg, 3); g.iterate(alg, 3)
    assert rel(g.fetch_object(), o.O) < TOL_RUN and rel(g.fetch_probe(), o.P) < TOL_RUN
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)
    g.destroy()
    with pytest.raises(B.PtychoError):
        B.Ptycho(obj0, np.concatenate([probe0, probe0[:1]]), pos, inten)


@pytest.mark.parametrize("alg,dtype", [("DM", np.uint16), ("EPIE_MB", np.uint16), ("DM", np.float32), ("LSQML", np.float32)])
def test_dead_frames_and_frames_on_every_border(B, oracle_mod, alg, dtype):
    """One frame with every pixel masked (R3: it must pass through the cycle unchanged and add nothing to the error), one frame
    with all-zero counts (sqrt I = 0 everywhere: the projection sends the wave to zero), frames flush with all four borders of
    the object, and a relaxed projection whose bound some frames are inside of from the first iteration."""
    n, h = 64, 150
    obj = synth.make_object(h, h, 10)
    probe = synth.probe_zone(n, n * 0.3125)[None]
    pos = np.array([[0, 0], [0, h - n], [h - n, 0], [h - n, h - n], [0, 40], [43, 0], [h - n, 37], [41, h - n], [40, 40], [50, 30], [30, 52]], np.int32)
    inten = _scan_from(obj, probe, pos, dtype=dtype, peak=5e3)
    inten[8] = 65535 if dtype == np.uint16 else -1.0         # fully masked frame
    inten[9] = 0                                             # dead frame
    par = dict(batch_size=4, pbound=0.3)
    obj0 = np.ones_like(obj)
    o = oracle_mod.Oracle(obj0, probe, pos, inten, par)
    g = B.Ptycho(obj0, probe, pos, inten, B.default_params(**par))
    for it in range(5):
        o.iterate(alg, 1); g.iterate(alg, 1)
        assert rel(g.fetch_object(), o.O) < TOL_RUN and rel(g.fetch_probe(), o.P) < TOL_RUN, (alg, it)
    if alg == "DM":
        assert rel(g.fetch_exit_waves(), o.psi) < TOL_RUN
    assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)
    g.destroy()


def test_more_than_65535_frames(B, oracle_mod):
    """J = 70 000 small frames: every launch that carries a frame index in a grid dimension has to cope with more than 65 535 of them
    (gridDim.y is capped there), the three-pass kernels cut the batch into several launches, the DM counters and tile lists index
    beyond 2^16.  DM (megakernel) and full-batch ePIE against the oracle."""
    n, h, J = 64, 700, 70000
    rng = np.random.default_rng(61)
    obj = synth.make_object(h, h, 12)
    probe = synth.probe_disk(n, n * 0.3125)[None]
    pos = rng.integers(0, h - n + 1, (J, 2)).astype(np.int32)
    _, inten, _ = synth.simulate(obj, probe, pos, 2e3, 5, np.uint16, 8)
    obj0 = np.ones_like(obj)
    for alg, par in (("DM", dict(pbound=0.3)), ("EPIE_MB", dict(batch_size=0))):
        o = oracle_mod.Oracle(obj0, probe, pos, inten, par)
        g = B.Ptycho(obj0, probe, pos, inten, B.default_params(**par))
        o.iterate(alg, 2); g.iterate(alg, 2)
        assert rel(g.fetch_object(), o.O) < TOL_RUN and rel(g.fetch_probe(), o.P) < TOL_RUN, alg
        assert np.allclose(g.fetch_error(), o.err, rtol=2e-3)
        if alg == "DM":
            sel = np.array([0, 65535, 65536, J - 1], np.int32)
            assert rel(g.fetch_exit_waves(sel), o.psi[sel]) < TOL_RUN
        g.destroy()


@pytest.mark.skipif(not __import__("os").environ.get("PTYCHO_LONG_TESTS"), reason="opt-in (PTYCHO_LONG_TESTS=1): thousands of iterations at full size")
@pytest.mark.parametrize("cfg,iters", [(2, 3000), (4, 400), (1, 20000)])
def test_soak_thousands_of_dm_iterations(B, cfg, iters):
    """The persistent queue over many launches at full size: no hang (the call returns), finite and non-increasing error tail."""
    import torch
    s = synth.make_config(cfg)
    g = B.Ptycho(s.obj0, s.probe0, s.pos, torch.from_numpy(s.intensities).cuda(),
                 B.default_params(pbound=s.params.get("pbound", s.params.get("pbound_dm", 0.0))))
    g.iterate("DM", iters)
    e = g.fetch_error()
    assert len(e) == iters and np.isfinite(e).all() and e[-1] < e[0] and e[-1] <= 1.05 * e[iters // 2]
    g.destroy()
