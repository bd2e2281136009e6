"""Pins of the CPU oracle against things other than itself (SURVEY.md 8(c) "Pins").

Every test here runs on CPU.  The independent references are: the DFT definition typed out with
numpy on tiny inputs, numpy's library FFT, closed forms, invariants and symmetries of the
method, a generic least-squares solver, and data simulated by `synth` with the library FFT.
"""
import numpy as np
import pytest

from paper_2202_03144_b200 import synth

RNG = np.random.default_rng(12345)


def crandn(*shape):
    return RNG.standard_normal(shape) + 1j * RNG.standard_normal(shape)


def rel(a, b):
    return float(np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300))


# ------------------------------------------------------------------------------------- FFT pins
def test_fft_vs_dft_definition_8x8(oracle_mod):
    x = crandn(8, 8)
    u = np.arange(8)
    w = np.exp(-2j * np.pi * np.outer(u, u) / 8)            # the definition, typed here
    want = w @ x @ w.T
    assert rel(oracle_mod.dft2_naive(x), want) < 1e-14
    assert rel(oracle_mod.fft2(x), want) < 1e-14
    assert rel(oracle_mod.fft2(want, inverse=True), x) < 1e-14
    assert rel(oracle_mod.dft2_naive(want, inverse=True), x) < 1e-14


def test_fft_rows_vs_naive_64(oracle_mod):
    x = crandn(16, 16)
    assert rel(oracle_mod.fft2(x), oracle_mod.dft2_naive(x)) < 1e-13


@pytest.mark.parametrize("n", [64, 128, 256, 512])
def test_fft_vs_library(oracle_mod, n):
    x = crandn(n, n)
    assert rel(oracle_mod.fft2(x), np.fft.fft2(x)) < 1e-13
    assert rel(oracle_mod.fft2(x, inverse=True), np.fft.ifft2(x)) < 1e-13


def test_fft_asymmetric_input_not_transposed(oracle_mod):
    """A transposed or sign-flipped transform fails here: single off-axis plane wave."""
    n = 32
    y, x = np.mgrid[0:n, 0:n]
    wave = np.exp(2j * np.pi * (3 * y + 5 * x) / n)         # peak must land at [3, 5], value n^2
    f = oracle_mod.fft2(wave)
    want = np.zeros((n, n), complex)
    want[3, 5] = n * n
    assert np.abs(f - want).max() < 1e-9
    d = np.zeros((n, n), complex)
    d[2, 7] = 1.0                                           # shifted delta -> pure phase ramp
    assert np.abs(oracle_mod.fft2(d) - np.exp(-2j * np.pi * (2 * y + 7 * x) / n)).max() < 1e-12


def test_fft_parseval_roundtrip_linearity(oracle_mod):
    n = 64
    a, b = crandn(n, n), crandn(n, n)
    fa, fb = oracle_mod.fft2(a), oracle_mod.fft2(b)
    assert abs(np.sum(np.abs(fa) ** 2) / (n * n * np.sum(np.abs(a) ** 2)) - 1) < 1e-14
    assert rel(oracle_mod.fft2(fa, inverse=True), a) < 1e-14
    assert rel(oracle_mod.fft2(2.5 * a - 1j * b), 2.5 * fa - 1j * fb) < 1e-14


# ------------------------------------------------------------------------- modulus projection
def test_projection_modulus_phase_idempotent(oracle_mod):
    n, k = 16, 3
    phi = crandn(k, n, n)
    inten = RNG.random((n, n)) * 50
    out, err = oracle_mod.modulus_project(phi, inten)
    assert np.allclose(np.sum(np.abs(out) ** 2, 0), inten, rtol=1e-13)          # |Phi'|^2 = I
    assert np.abs(np.angle(out * np.conj(phi))).max() < 1e-12                   # phases kept
    ratio = np.abs(out) / np.abs(phi)
    assert np.allclose(ratio, ratio[0][None], rtol=1e-12)                       # one scale per pixel
    out2, err2 = oracle_mod.modulus_project(out, inten)
    assert rel(out2, out) < 1e-14 and err2 < 1e-20                              # idempotent
    a = np.sqrt(np.sum(np.abs(phi) ** 2, 0))
    assert abs(err - np.sum((np.sqrt(inten) - a) ** 2)) < 1e-10 * err


def test_projection_mask_and_zero_amplitude(oracle_mod):
    n = 8
    phi = crandn(2, n, n)
    phi[:, 1, 2] = 0                                                            # A = 0 pixel (R2)
    inten = RNG.random((n, n)) * 9 + 1
    inten[3, 4] = -1.0                                                          # masked (R3)
    out, err = oracle_mod.modulus_project(phi, inten)
    assert np.array_equal(out[:, 3, 4], phi[:, 3, 4])
    assert out[0, 1, 2] == np.sqrt(inten[1, 2]) and out[1, 1, 2] == 0
    a = np.sqrt(np.sum(np.abs(phi) ** 2, 0))
    ok = inten >= 0
    assert abs(err - np.sum((np.sqrt(inten[ok]) - a[ok]) ** 2)) < 1e-12 * err
    # uint16 sentinel is the same mask
    cnt = np.full((n, n), 7, np.uint16)
    cnt[3, 4] = 65535
    out_u, _ = oracle_mod.modulus_project(phi, cnt)
    assert np.array_equal(out_u[:, 3, 4], phi[:, 3, 4])
    assert np.allclose(np.sum(np.abs(out_u) ** 2, 0)[cnt < 65535], 7.0)


def test_projection_relaxed_closed_form(oracle_mod):
    n = 16
    phi = crandn(1, n, n) * 3
    inten = RNG.random((n, n)) * 20
    exact, err = oracle_mod.modulus_project(phi, inten, 0.0)
    e = err / (n * n)
    same, _ = oracle_mod.modulus_project(phi, inten, pbound=e * 1.01)           # inside the bound
    assert np.array_equal(same, phi)
    pb = e * 0.3
    out, _ = oracle_mod.modulus_project(phi, inten, pbound=pb)
    _, err_after = oracle_mod.modulus_project(out, inten, 0.0)
    assert abs(err_after / (n * n) - pb) < 1e-12 * pb                           # lands on the bound
    r = np.sqrt(pb / e)
    assert rel(out, (1 - r) * exact + r * phi) < 1e-14


# ------------------------------------------------------------------- whole-cycle invariants
def f64_scan(n=16, h=40, side=4, step=6, k=1, probe_kind="disk"):
    s = synth.make_custom(n, h, side, step, k=k, probe_kind=probe_kind)
    lam = np.concatenate([l for _, l in synth.model_intensity(s.obj_true, s.probe_true, s.pos, 1)])
    return s, lam                                           # float64 noiseless intensities


@pytest.mark.parametrize("alg,k", [("DM", 1), ("EPIE_MB", 1), ("LSQML", 1), ("LSQML", 3), ("DM", 2)])
def test_ground_truth_is_fixed_point_with_zero_error(oracle_mod, alg, k):
    s, lam = f64_scan(k=k)
    o = oracle_mod.Oracle(s.obj_true, s.probe_true, s.pos, lam, dict(batch_size=5))
    o.iterate(alg, 2)
    assert max(o.err) < 1e-25
    assert rel(o.O, s.obj_true) < 1e-13 and rel(o.P, s.probe_true) < 1e-13
    assert o.eval_error() < 1e-25
    if alg == "DM":
        want = np.stack([s.probe_true * s.obj_true[None, y:y + s.n, x:x + s.n] for y, x in s.pos])
        assert rel(o.psi, want) < 1e-13


def test_dm_all_masked_closed_forms(oracle_mod):
    """With no Fourier constraint Pi_M = id, so psi_new = P O_j, O is unchanged, and the lagged
    probe update from incoming psi_j = Q O_j is the closed form (d_P Q + eps P)/(d_P + eps)."""
    s, lam = f64_scan()
    n = s.n
    obj = s.obj_true * (1 + 0.1 * crandn(*s.obj_true.shape))
    q = s.probe_true * (1 + 0.2 * crandn(*s.probe_true.shape))
    o = oracle_mod.Oracle(obj, s.probe_true, s.pos, -np.ones_like(lam))
    o.psi = np.stack([q * obj[None, y:y + n, x:x + n] for y, x in s.pos]).astype(complex)
    p_old, eps = o.P.copy(), o.eps_P
    o.iterate("DM", 1)
    want_psi = np.stack([p_old * obj[None, y:y + n, x:x + n] for y, x in s.pos])
    assert rel(o.psi, want_psi) < 1e-14
    assert rel(o.O, obj) < 1e-14
    d_p = sum(np.abs(obj[y:y + n, x:x + n]) ** 2 for y, x in s.pos)
    assert rel(o.P, (d_p * q + eps * p_old) / (d_p + eps)) < 1e-14
    assert eps == pytest.approx(1e-2 * len(s.pos) * np.max(np.abs(obj) ** 2))   # R5 constants
    assert o.eps_O == pytest.approx(1e-2 * np.max(np.abs(p_old) ** 2))


def test_epie_single_frame_closed_form_with_library_fft(oracle_mod):
    """J = 1, alpha = 1, delta -> 0, probe frozen: O_new = psi_F / P on the probe support, with
    psi_F = ifft2(fft2(P O) sqrt(I) / |fft2(P O)|) evaluated here with numpy's FFT."""
    s, lam = f64_scan(side=1)
    obj0 = 1 + 0.05 * crandn(*s.obj_true.shape)
    o = oracle_mod.Oracle(obj0, s.probe_true, s.pos, lam,
                          dict(delta_obj=1e-30, probe_start=10 ** 9), keep_revised=True)
    o.iterate("EPIE_MB", 1)
    (y, x), n, p = s.pos[0], s.n, s.probe_true[0]
    f = np.fft.fft2(p * obj0[y:y + n, x:x + n])
    psi_f = np.fft.ifft2(f * np.sqrt(lam[0]) / np.abs(f))
    assert rel(o.revised[0, 0], psi_f) < 1e-12
    sup = np.abs(p) > 0
    assert rel(o.O[y:y + n, x:x + n][sup], (psi_f / np.where(sup, p, 1))[sup]) < 1e-10
    assert np.array_equal(o.O[y:y + n, x:x + n][~sup], obj0[y:y + n, x:x + n][~sup])
    assert o.err[0] == pytest.approx(np.sum((np.sqrt(lam[0]) - np.abs(f)) ** 2) / lam.sum(), rel=1e-12)


def test_dm_first_iteration_equals_full_batch_epie(oracle_mod):
    """From psi0 = P O_j the reflector is the identity, so DM's first iteration and one full-batch
    ePIE step (alpha 1) give the same revised waves and, with delta_obj = delta_blend, the same
    object; DM's lagged probe update returns P unchanged.  Two code paths, one answer."""
    s, lam = f64_scan(n=16, h=48, side=5, step=5)
    cnt = RNG.poisson(lam * 50).astype(np.float64)
    p0 = s.probe_true * np.sqrt(50)
    dm = oracle_mod.Oracle(s.obj0, p0, s.pos, cnt, dict(delta_blend=0.37), keep_revised=True)
    ep = oracle_mod.Oracle(s.obj0, p0, s.pos, cnt, dict(delta_obj=0.37, probe_start=10 ** 9), keep_revised=True)
    dm.iterate("DM", 1)
    ep.iterate("EPIE_MB", 1)
    assert rel(dm.revised, ep.revised) < 1e-14
    assert rel(dm.psi, ep.revised) < 1e-14
    assert rel(dm.O, ep.O) < 1e-13
    assert rel(dm.P, p0) < 1e-13
    assert dm.err[0] == pytest.approx(ep.err[0], rel=1e-12)
    # the overlap formula applied to the revised waves, summed here with plain numpy slices
    n = s.n
    num = np.zeros_like(s.obj0)
    den = np.zeros(s.obj0.shape)
    for j, (y, x) in enumerate(s.pos):
        num[y:y + n, x:x + n] += np.conj(p0[0]) * ep.revised[j, 0]
        den[y:y + n, x:x + n] += np.abs(p0[0]) ** 2
    eps = 0.37 * np.max(np.abs(p0) ** 2)
    assert rel(dm.O, (num + eps * s.obj0) / (den + eps)) < 1e-13


def test_lsqml_direction_and_step_vs_generic_least_squares(oracle_mod):
    """LSQML-style moves along the ePIE directions (O_l - O = a dO, P_l - P = b dP_k) and (a, b)
    solves the Tikhonov-regularised real least-squares problem of reading R9, here handed as an
    explicit stacked system to numpy.linalg.lstsq (J = 4, N = 8, K = 2)."""
    s, lam = f64_scan(n=8, h=20, side=2, step=4, k=2)
    cnt = RNG.poisson(lam * 30).astype(np.float64)
    p0 = s.probe_true * np.sqrt(30)
    obj0 = 1 + 0.1 * crandn(*s.obj_true.shape)
    lam_t = 0.1
    ep = oracle_mod.Oracle(obj0, p0, s.pos, cnt, keep_revised=True)
    ls = oracle_mod.Oracle(obj0, p0, s.pos, cnt, dict(lsq_lambda=lam_t))
    ep.iterate("EPIE_MB", 1)
    ls.iterate("LSQML", 1)
    d_o, d_p = ep.O - obj0, ep.P - p0
    a, b = ls.steps[0]
    assert rel(ls.O - obj0, a * d_o) < 1e-12 and rel(ls.P - p0, b * d_p) < 1e-12
    n = s.n
    u, v, c = [], [], []
    for j, (y, x) in enumerate(s.pos):
        oj, doj = obj0[y:y + n, x:x + n], d_o[y:y + n, x:x + n]
        u.append(p0 * doj[None])
        v.append(d_p * oj[None])
        c.append(ep.revised[j] - p0 * oj[None])
    u, v, c = (np.ravel(np.stack(z)) for z in (u, v, c))
    ri = lambda z: np.concatenate([z.real, z.imag])
    a11, a22 = np.vdot(u, u).real, np.vdot(v, v).real
    m = np.stack([np.concatenate([ri(u), [np.sqrt(lam_t * a11), 0]]),
                  np.concatenate([ri(v), [0, np.sqrt(lam_t * a22)]])], 1)
    sol = np.linalg.lstsq(m, np.concatenate([ri(c), [0, 0]]), rcond=None)[0]
    assert a == pytest.approx(sol[0], rel=1e-10) and b == pytest.approx(sol[1], rel=1e-10)
    # frozen probe: a = b1 / (A11 (1 + lambda)), b = 0
    lf = oracle_mod.Oracle(obj0, p0, s.pos, cnt, dict(lsq_lambda=lam_t, probe_start=10 ** 9))
    lf.iterate("LSQML", 1)
    assert lf.steps[0][1] == 0
    assert lf.steps[0][0] == pytest.approx(np.vdot(u, c).real / (a11 * (1 + lam_t)), rel=1e-10)
    assert rel(lf.P, p0) == 0


def test_zero_modes_reduce_to_single_mode(oracle_mod):
    s, lam = f64_scan(k=1)
    cnt = RNG.poisson(lam * 20).astype(np.float64)
    p1 = s.probe_true * np.sqrt(20)
    p3 = np.concatenate([p1, np.zeros_like(p1), np.zeros_like(p1)])
    for alg in ("LSQML", "EPIE_MB", "DM"):
        a = oracle_mod.Oracle(s.obj0, p1, s.pos, cnt, dict(batch_size=6)).iterate(alg, 3)
        b = oracle_mod.Oracle(s.obj0, p3, s.pos, cnt, dict(batch_size=6)).iterate(alg, 3)
        assert rel(b.O, a.O) < 1e-13 and rel(b.P[0], a.P[0]) < 1e-13 and np.abs(b.P[1:]).max() == 0
        assert np.allclose(a.err, b.err, rtol=1e-12)


# ------------------------------------------------------------------------------- symmetries
@pytest.mark.parametrize("alg", ["DM", "EPIE_MB", "LSQML"])
def test_symmetries(oracle_mod, alg):
    s, lam = f64_scan(n=16, h=44, side=4, step=6)
    cnt = RNG.poisson(lam * 40).astype(np.float64)
    p0 = s.probe_true * np.sqrt(40)
    obj0 = 1 + 0.05 * crandn(*s.obj_true.shape)
    par = dict(batch_size=4, pbound=0.05 if alg == "DM" else 0.0)
    base = oracle_mod.Oracle(obj0, p0, s.pos, cnt, par).iterate(alg, 3)
    # (1) translating positions and object together changes nothing
    big = np.ones((60, 60), complex)
    big[7:51, 9:53] = obj0
    sh = oracle_mod.Oracle(big, p0, s.pos + np.array([7, 9], np.int32), cnt, par).iterate(alg, 3)
    assert rel(sh.O[7:51, 9:53], base.O) < 1e-13 and rel(sh.P, base.P) < 1e-13
    # (2) global phase of a frozen probe comes out conjugated on the object
    th = np.exp(0.7j)
    fz = dict(par, probe_start=10 ** 9)
    b0 = oracle_mod.Oracle(obj0, p0, s.pos, cnt, fz).iterate(alg, 2)
    b1 = oracle_mod.Oracle(obj0 * np.conj(th), p0 * th, s.pos, cnt, fz).iterate(alg, 2)
    assert rel(b1.O * th, b0.O) < 1e-13
    # (3) uint16 and float copies of the same integer counts agree exactly
    u = oracle_mod.Oracle(obj0, p0, s.pos, cnt.astype(np.uint16), par).iterate(alg, 3)
    assert np.array_equal(u.O, base.O) and np.array_equal(u.P, base.P)
    # (4) frame order only changes summation rounding (full batch)
    perm = RNG.permutation(len(s.pos))
    fb = dict(par, batch_size=0)
    c0 = oracle_mod.Oracle(obj0, p0, s.pos, cnt, fb).iterate(alg, 2)
    c1 = oracle_mod.Oracle(obj0, p0, s.pos[perm], cnt[perm], fb).iterate(alg, 2)
    assert rel(c1.O, c0.O) < 1e-12 and rel(c1.P, c0.P) < 1e-12


def test_strided_batches(oracle_mod):
    b = oracle_mod.batches(10, 4)
    assert [list(x) for x in b] == [[0, 3, 6, 9], [1, 4, 7], [2, 5, 8]]                # n_b = 3
    assert [len(x) for x in oracle_mod.batches(20000, 512)] == [500] * 40            # cfg3
    assert [list(x) for x in oracle_mod.batches(5, 2, order=[4, 3, 2, 1, 0])] == [[4, 3], [2, 1], [0]]
    assert len(oracle_mod.batches(7, 0)) == 1


# ------------------------------------------------------------------------------ convergence
def test_cfg0_dm_error_history_against_survey_values(oracle_mod):
    s = synth.make_config(0)
    gold = np.loadtxt("tests/golden/survey_x12_cfg0.txt")[:, 1]
    for ps in (10 ** 9, 0):
        o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(probe_start=ps)).iterate("DM", 10)
        e = np.array(o.err)
        assert np.all(np.diff(e[:8]) < 0), e                 # decreasing while far from the floor
        assert e[-1] < 0.1 * e[0]
        assert np.all((e > gold / 2) & (e < gold * 2)), e    # same order as the survey prototype


@pytest.mark.parametrize("alg", ["EPIE_MB", "LSQML"])
def test_minibatch_monotone_on_noiseless_data(oracle_mod, alg):
    s = synth.make_config(0)
    o = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, dict(batch_size=16)).iterate(alg, 50)
    e = np.array(o.err)
    assert np.all(np.diff(e) < 0), e
    assert e[-1] < 1e-3 * e[0]


def test_float_build_tracks_double(oracle_mod):
    """Precision floor: the same oracle compiled in float stays within the parity tolerances."""
    s = synth.make_config(0)
    d = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities).iterate("DM", 10)
    f = oracle_mod.Oracle(s.obj0, s.probe0, s.pos, s.intensities, precision="f32").iterate("DM", 10)
    assert rel(f.O, d.O) < 1e-4 and rel(f.psi, d.psi) < 1e-4


# ------------------------------------------------------------------ frame preparation (S:8(f) f2)
def test_prepare_frames_hand_example_and_shift_involution(oracle_mod):
    """6 x 6 detector, n = 4, centre (3, 2): indices worked out by hand from the definition in the header
    (sy = cy + (ky < n/2 ? ky : ky - n)); out-of-detector pixels masked; threshold zeroes, saturation masks."""
    raw = (np.arange(36, dtype=np.uint16).reshape(1, 6, 6) * 10)
    out = oracle_mod.prepare_frames(raw, (3, 2), 4)
    # ky = 0,1,2,3 -> sy = 3,4,1,2 ; kx = 0,1,2,3 -> sx = 2,3,0,1
    expect = np.array([[raw[0, sy, sx] for sx in (2, 3, 0, 1)] for sy in (3, 4, 1, 2)], np.uint16)
    assert np.array_equal(out[0], expect)
    assert out[0, 0, 0] == raw[0, 3, 2]                                 # the centre pixel is the DC term
    edge = oracle_mod.prepare_frames(raw, (0, 5), 4)                     # window hangs over two detector edges
    # ky -> sy = 0,1,-2,-1 ; kx -> sx = 5,6,3,4
    assert edge[0, 0, 0] == raw[0, 0, 5] and edge[0, 0, 1] == 65535 and edge[0, 2, 0] == 65535 and edge[0, 1, 3] == raw[0, 1, 4]
    th = oracle_mod.prepare_frames(raw, (3, 2), 4, threshold=185.0, saturation=260.0)
    assert th[0, 2, 2] == 0 and th[0, 0, 0] == 200 and th[0, 1, 0] == 65535 and th[0, 1, 1] == 65535   # 60 -> 0; 260, 270 saturated
    f32 = oracle_mod.prepare_frames(raw.astype(np.float32), (3, 2), 4, saturation=260.0, out_dtype=np.float32)
    assert f32.dtype == np.float32 and f32[0, 1, 0] == -1.0 and f32[0, 0, 0] == 200.0
    # fftshift of the result is the plain centred crop (involution of the shift for even n)
    rng = np.random.default_rng(0)
    big = rng.integers(0, 60000, (3, 40, 50)).astype(np.uint16)
    o = oracle_mod.prepare_frames(big, (20, 25), 16)
    assert np.array_equal(np.fft.fftshift(o, axes=(1, 2)), big[:, 12:28, 17:33])


# ------------------------------------------------- pins asked for by the round-1 review
def test_eval_error_off_zero_against_numpy(oracle_mod):
    """orc_eval_error_num away from the ground truth (R7, C3): sum_j sum_q (sqrt I - sqrt(sum_k |fft2(P_k O_j)|^2))^2
    / sum I, typed here with numpy's FFT; J = 4, K in {1, 2}, O != truth, one masked pixel per frame."""
    for k in (1, 2):
        s, lam = f64_scan(n=8, h=20, side=2, step=4, k=k)
        cnt = RNG.poisson(lam * 25).astype(np.float64)
        cnt[:, 2, 5] = -1.0                                                      # masked (R3): excluded from both sums
        obj = s.obj_true * (1 + 0.3 * crandn(*s.obj_true.shape))
        p0 = s.probe_true * np.sqrt(25) * (1 + 0.1 * crandn(*s.probe_true.shape))
        o = oracle_mod.Oracle(obj, p0, s.pos, cnt)
        n, num, den = s.n, 0.0, 0.0
        for j, (y, x) in enumerate(s.pos):
            a = np.sqrt(sum(np.abs(np.fft.fft2(p0[m] * obj[y:y + n, x:x + n])) ** 2 for m in range(k)))
            ok = cnt[j] >= 0
            num += np.sum((np.sqrt(cnt[j][ok]) - a[ok]) ** 2)
            den += np.sum(cnt[j][ok])
        assert num / den > 1e-3                                                  # really off zero
        assert o.eval_error() == pytest.approx(num / den, rel=1e-12)
        assert o.sum_I == pytest.approx(den, rel=1e-14)


def test_epie_probe_direction_against_numpy(oracle_mod):
    """Probe side of the minibatch step (R8): one full-batch ePIE step, alpha_P = 1, delta_probe = 0.37:
    P_new - P = n_P / (d_P + 0.37 max_r d_P), n_P = sum_j conj(O_j)(revised_j - P O_j), d_P = sum_j |O_j|^2,
    summed here with numpy slices; K = 2 so that d_P is shared by the modes."""
    s, lam = f64_scan(n=8, h=20, side=2, step=4, k=2)
    cnt = RNG.poisson(lam * 30).astype(np.float64)
    p0 = s.probe_true * np.sqrt(30)
    obj0 = 1 + 0.2 * crandn(*s.obj_true.shape)
    o = oracle_mod.Oracle(obj0, p0, s.pos, cnt, dict(delta_probe=0.37, delta_obj=0.61), keep_revised=True)
    o.iterate("EPIE_MB", 1)
    n = s.n
    n_p, d_p = np.zeros_like(p0), np.zeros((n, n))
    n_o, d_o = np.zeros_like(obj0), np.zeros(obj0.shape)
    for j, (y, x) in enumerate(s.pos):
        oj = obj0[y:y + n, x:x + n]
        chi = o.revised[j] - p0 * oj[None]
        n_p += np.conj(oj)[None] * chi
        d_p += np.abs(oj) ** 2
        n_o[y:y + n, x:x + n] += np.sum(np.conj(p0) * chi, 0)
        d_o[y:y + n, x:x + n] += np.sum(np.abs(p0) ** 2, 0)
    assert rel(o.P - p0, n_p / (d_p + 0.37 * d_p.max())[None]) < 1e-12
    assert rel(o.O - obj0, n_o / (d_o + 0.61 * np.max(np.sum(np.abs(p0) ** 2, 0)))) < 1e-12


def test_masked_pixels_are_excluded_from_sum_intensity(oracle_mod):
    """R3: masked pixels count neither in the error terms nor in sum I.  err[0] * sum(I unmasked) must equal
    the numpy sum over unmasked pixels; including the masked counts in sum I would fail this."""
    s, lam = f64_scan(n=8, h=20, side=2, step=4)
    cnt = np.minimum(RNG.poisson(lam * 400), 65534).astype(np.uint16)
    cnt[:, 0, 0] = 65535                                                         # the brightest pixel of every frame
    cnt[1, 3, 4] = 65535
    p0 = s.probe_true * np.sqrt(400)
    o = oracle_mod.Oracle(s.obj0, p0, s.pos, cnt, dict(probe_start=10 ** 9))
    o.iterate("EPIE_MB", 1)
    ok = cnt < 65535
    n, num = s.n, 0.0
    for j, (y, x) in enumerate(s.pos):
        a = np.abs(np.fft.fft2(p0[0] * s.obj0[y:y + n, x:x + n]))
        num += np.sum((np.sqrt(cnt[j][ok[j]].astype(float)) - a[ok[j]]) ** 2)
    unmasked = float(np.sum(cnt[ok].astype(np.float64)))
    assert o.sum_I == unmasked
    assert o.err[0] * unmasked == pytest.approx(num, rel=1e-12)
    assert abs(o.err[0] * float(cnt.astype(np.float64).sum()) - num) > 1e-3 * num   # the wrong denominator is far off


# --------------------------------------------------------------------- f1: textbook variants
def test_sequential_dm_overlap_closed_forms(oracle_mod):
    """One sweep of the sequential overlap projection against the closed forms of S:8(c) "Overlap update": for consistent
    waves psi_j = Q O*_j the object step returns (d_O O* + eps O_old)/(d_O + eps) -- with the probe it is given, Q -- and the
    probe step, run with the NEW object, returns (d_P Q' + eps P_old)/(d_P + eps) where Q' solves psi_j = Q' O_new,j pixel by
    pixel in the least-squares sense; here everything is typed with numpy slices.  All pixels masked: Pi_M = id."""
    s, lam = f64_scan(n=8, h=22, side=3, step=4)
    n = s.n
    ostar = s.obj_true * (1 + 0.2 * crandn(*s.obj_true.shape))
    q = s.probe_true * (1 + 0.3 * crandn(*s.probe_true.shape))
    o_old = 1 + 0.1 * crandn(*s.obj_true.shape)
    o = oracle_mod.Oracle(o_old, q, s.pos, -np.ones_like(lam), dict(dm_sweeps=1))
    o.psi = np.stack([q * ostar[None, y:y + n, x:x + n] for y, x in s.pos]).astype(complex)
    eps_o, eps_p = o.eps_O, o.eps_P
    o.iterate("DM", 1)
    # all-masked Fourier step: psi_new = psi + P O_old,j - P O_old,j ... = P O_old,j (reflector and update cancel, see the DM closed-form pin)
    psi_new = np.stack([q * o_old[None, y:y + n, x:x + n] for y, x in s.pos])
    assert rel(o.psi, psi_new) < 1e-13
    d_o, n_o = np.zeros(o_old.shape), np.zeros_like(o_old)
    for j, (y, x) in enumerate(s.pos):
        d_o[y:y + n, x:x + n] += np.abs(q[0]) ** 2
        n_o[y:y + n, x:x + n] += np.conj(q[0]) * psi_new[j, 0]
    o_new = (n_o + eps_o * o_old) / (d_o + eps_o)
    assert rel(o.O, o_new) < 1e-13
    n_p, d_p = np.zeros_like(q[0]), np.zeros((n, n))
    for j, (y, x) in enumerate(s.pos):
        oj = o_new[y:y + n, x:x + n]                                             # the NEW object: sequential, not lagged
        n_p += np.conj(oj) * psi_new[j, 0]
        d_p += np.abs(oj) ** 2
    assert rel(o.P[0], (n_p + eps_p * q[0]) / (d_p + eps_p)) < 1e-13
    # two sweeps: the object is formed once more from the same waves with the new probe
    o2 = oracle_mod.Oracle(o_old, q, s.pos, -np.ones_like(lam), dict(dm_sweeps=2))
    o2.psi = np.stack([q * ostar[None, y:y + n, x:x + n] for y, x in s.pos]).astype(complex)
    o2.iterate("DM", 1)
    p1 = (n_p + eps_p * q[0]) / (d_p + eps_p)
    d2, n2 = np.zeros(o_old.shape), np.zeros_like(o_old)
    for j, (y, x) in enumerate(s.pos):
        d2[y:y + n, x:x + n] += np.abs(p1) ** 2
        n2[y:y + n, x:x + n] += np.conj(p1) * psi_new[j, 0]
    assert rel(o2.O, (n2 + eps_o * o_new) / (d2 + eps_o)) < 1e-13


def test_sequential_dm_fixed_point_and_decrease(oracle_mod):
    s, lam = f64_scan()
    o = oracle_mod.Oracle(s.obj_true, s.probe_true, s.pos, lam, dict(dm_sweeps=2)).iterate("DM", 2)
    assert max(o.err) < 1e-25 and rel(o.O, s.obj_true) < 1e-13 and rel(o.P, s.probe_true) < 1e-13
    c = synth.make_config(0)
    e = np.array(oracle_mod.Oracle(c.obj0, c.probe0, c.pos, c.intensities, dict(dm_sweeps=1)).iterate("DM", 10).err)
    assert np.all(np.diff(e[:8]) < 0) and e[-1] < 0.1 * e[0], e                  # the sequential form is monotone on cfg0


def test_position_sequential_epie_is_single_frame_steps_in_sequence(oracle_mod):
    """B = 1 (the paper's position-sequential ePIE): one iteration equals J single-frame oracles applied one
    after the other to the running state, in scan order."""
    s, lam = f64_scan(n=8, h=20, side=2, step=4)
    cnt = RNG.poisson(lam * 30).astype(np.float64)
    p0 = s.probe_true * np.sqrt(30)
    obj0 = 1 + 0.1 * crandn(*s.obj_true.shape)
    seq = oracle_mod.Oracle(obj0, p0, s.pos, cnt, dict(batch_size=1)).iterate("EPIE_MB", 1)
    O, P = obj0.copy(), p0.copy()
    for j in range(len(s.pos)):
        one = oracle_mod.Oracle(O, P, s.pos[j:j + 1], cnt[j:j + 1]).iterate("EPIE_MB", 1)
        O, P = one.O, one.P
    assert rel(seq.O, O) < 1e-13 and rel(seq.P, P) < 1e-13


def test_prepare_frames_rotation_and_normalisation_by_hand(oracle_mod):
    """rot90 (R23) and frame_scale (R24) on a 7 x 7 detector indexed by hand.  Centre (3, 3), n = 4.  A quarter turn
    counter-clockwise (numpy.rot90 convention: the pixel to the RIGHT of the centre moves to ABOVE it) means the output pixel at
    centred offset (dy, dx) comes from the source pixel at offset (dx, -dy); two turns: (-dy, -dx); three: (-dx, dy)."""
    raw = (np.arange(49, dtype=np.uint16).reshape(1, 7, 7) + 100)
    c = (3, 3)
    off = [0, 1, -2, -1]                                   # centred offset of FFT-order index 0..3
    src = {0: lambda dy, dx: (dy, dx), 1: lambda dy, dx: (dx, -dy), 2: lambda dy, dx: (-dy, -dx), 3: lambda dy, dx: (-dx, dy)}
    for k in range(4):
        out = oracle_mod.prepare_frames(raw, c, 4, rot90=k)
        want = np.array([[raw[0, 3 + src[k](dy, dx)[0], 3 + src[k](dy, dx)[1]] for dx in off] for dy in off], np.uint16)
        assert np.array_equal(out[0], want), k
    # the defining property, on one pixel: right of the centre (offset (0, +1), value raw[3, 4]) lands above it (offset (-1, 0))
    assert oracle_mod.prepare_frames(raw, c, 4, rot90=1)[0, 3, 0] == raw[0, 3, 4]
    # rotation about an off-centre pixel near the edge: what leaves the detector is masked
    edge = oracle_mod.prepare_frames(raw, (0, 6), 4, rot90=1)
    # (dy, dx) = (1, 0) <- source offset (0, -1) = raw[0, 5]; (0, 1) <- (1, 0) = raw[1, 6]; (0, -1) <- (-1, 0): row -1, off the detector
    assert edge[0, 0, 0] == raw[0, 0, 6] and edge[0, 1, 0] == raw[0, 0, 5] and edge[0, 0, 1] == raw[0, 1, 6] and edge[0, 0, 3] == 65535
    # normalisation: one factor per frame, after the threshold, fp32 product rounded to nearest for uint16
    two = np.concatenate([raw, raw])
    sc = oracle_mod.prepare_frames(two, c, 4, threshold=125.0, frame_scale=np.array([1.0, 0.5], np.float32))
    assert sc[1, 0, 1] == round(float(raw[0, 3, 4]) * 0.5) and sc[0, 0, 1] == raw[0, 3, 4]       # 125 -> 62 (round half to even: 62.5 -> 62)
    assert sc[1, 0, 0] == 0 and sc[0, 0, 0] == 0                                                    # 124 < threshold -> 0 in both
    f32 = oracle_mod.prepare_frames(two.astype(np.float32), c, 4, frame_scale=np.array([2.0, 0.25], np.float32), out_dtype=np.float32)
    assert f32[0, 0, 0] == 248.0 and f32[1, 0, 0] == 31.0


def test_lsqml_per_frame_steps_against_per_frame_lstsq(oracle_mod):
    """LSQML_PF (R25): (a_j, b_j) of every frame against numpy.linalg.lstsq of that frame's own stacked system; the object update
    against the weighted-scatter formula typed with numpy slices; the probe moves by the mean b_j.  J = 4, N = 8, K = 2."""
    s, lam = f64_scan(n=8, h=20, side=2, step=4, k=2)
    cnt = RNG.poisson(lam * 30).astype(np.float64)
    p0 = s.probe_true * np.sqrt(30)
    obj0 = 1 + 0.1 * crandn(*s.obj_true.shape)
    lam_t, n = 0.1, s.n
    ep = oracle_mod.Oracle(obj0, p0, s.pos, cnt, keep_revised=True).iterate("EPIE_MB", 1)   # directions (alpha = 1) and revised waves
    pf = oracle_mod.Oracle(obj0, p0, s.pos, cnt, dict(lsq_lambda=lam_t)).iterate("LSQML_PF", 1)
    d_o, d_p = ep.O - obj0, ep.P - p0
    ri = lambda z: np.concatenate([z.real.ravel(), z.imag.ravel()])
    aw, ww, bs = np.zeros(obj0.shape), np.zeros(obj0.shape), []
    for j, (y, x) in enumerate(s.pos):
        oj, doj = obj0[y:y + n, x:x + n], d_o[y:y + n, x:x + n]
        u, v, c = p0 * doj[None], d_p * oj[None], ep.revised[j] - p0 * oj[None]
        a11, a22 = np.vdot(u, u).real, np.vdot(v, v).real
        m = np.stack([np.concatenate([ri(u), [np.sqrt(lam_t * a11), 0]]), np.concatenate([ri(v), [0, np.sqrt(lam_t * a22)]])], 1)
        sol = np.linalg.lstsq(m, np.concatenate([ri(c), [0, 0]]), rcond=None)[0]
        assert pf.steps[j][0] == pytest.approx(sol[0], rel=1e-9) and pf.steps[j][1] == pytest.approx(sol[1], rel=1e-9), j
        w = np.sum(np.abs(p0) ** 2, 0)
        aw[y:y + n, x:x + n] += sol[0] * w
        ww[y:y + n, x:x + n] += w
        bs.append(sol[1])
    want_o = obj0 + np.where(ww > 0, aw / np.where(ww > 0, ww, 1), 0) * d_o
    assert rel(pf.O, want_o) < 1e-12 and rel(pf.P, p0 + np.mean(bs) * d_p) < 1e-12
    assert pf.err[0] == pytest.approx(ep.err[0], rel=1e-12)


def test_lsqml_per_frame_reduces_to_joint_step_for_one_frame(oracle_mod):
    """J = 1: the per-frame step IS the joint step of R9 (two code paths, one answer); ground truth stays a fixed point."""
    s, lam = f64_scan(n=8, h=14, side=1, step=4, k=2)
    cnt = RNG.poisson(lam * 30).astype(np.float64)
    p0, obj0 = s.probe_true * np.sqrt(30), 1 + 0.1 * crandn(*s.obj_true.shape)
    a = oracle_mod.Oracle(obj0, p0, s.pos, cnt).iterate("LSQML", 1)
    b = oracle_mod.Oracle(obj0, p0, s.pos, cnt).iterate("LSQML_PF", 1)
    assert rel(b.O, a.O) < 1e-12 and rel(b.P, a.P) < 1e-12 and b.steps[0] == pytest.approx(a.steps[0], rel=1e-10)
    s4, lam4 = f64_scan(k=3)
    t = oracle_mod.Oracle(s4.obj_true, s4.probe_true, s4.pos, lam4, dict(batch_size=5)).iterate("LSQML_PF", 2)
    assert max(t.err) < 1e-25 and rel(t.O, s4.obj_true) < 1e-13 and rel(t.P, s4.probe_true) < 1e-13
    c = synth.make_config(0)
    e = np.array(oracle_mod.Oracle(c.obj0, c.probe0, c.pos, c.intensities, dict(batch_size=16)).iterate("LSQML_PF", 30).err)
    assert np.all(np.diff(e) < 0) and e[-1] < 1e-2 * e[0], e                    # R22: monotone on noiseless data


def test_mode_orthogonalisation_pins(oracle_mod):
    """R26: the mixed modes have a diagonal Gram matrix with the eigenvalues of the old one (numpy.linalg.eigvalsh, a different
    routine) in descending order; the incoherent sum sum_k |P_k|^2 is unchanged at every pixel; modes that are already orthogonal
    with distinct powers come back unchanged; two identical modes collapse into one; exit waves mixed alike stay P'_k O_j."""
    p = crandn(3, 12, 12) * np.array([1.0, 0.6, 0.3])[:, None, None]
    p[1] += 0.5 * p[0]                                                           # make them clearly non-orthogonal
    q = oracle_mod.orthogonalize_modes(p)
    g = q.reshape(3, -1) @ q.reshape(3, -1).conj().T
    lam = np.linalg.eigvalsh(p.reshape(3, -1) @ p.reshape(3, -1).conj().T)[::-1]
    assert np.abs(g - np.diag(np.diag(g))).max() < 1e-10 * lam[0]
    assert np.allclose(np.diag(g).real, lam, rtol=1e-12) and np.all(np.diff(np.diag(g).real) <= 0)
    assert np.allclose(np.sum(np.abs(q) ** 2, 0), np.sum(np.abs(p) ** 2, 0), rtol=1e-12)
    s, _ = f64_scan(k=3)                                                         # synth's modes: Gram-Schmidt, powers 0.80 / 0.15 / 0.05
    assert rel(oracle_mod.orthogonalize_modes(s.probe_true), s.probe_true) < 1e-12
    twin = np.stack([p[0], p[0]])
    t = oracle_mod.orthogonalize_modes(twin)
    assert rel(t[0], np.sqrt(2) * p[0]) < 1e-12 and np.abs(t[1]).max() < 1e-12 * np.abs(p).max()
    obj = crandn(20, 20)
    psi = np.stack([p * obj[None, y:y + 12, x:x + 12] for y, x in ((0, 0), (3, 5), (8, 8))])
    q2, psi2 = oracle_mod.orthogonalize_modes(p, psi)
    want = np.stack([q2 * obj[None, y:y + 12, x:x + 12] for y, x in ((0, 0), (3, 5), (8, 8))])
    assert rel(psi2, want) < 1e-12


# ------------------------------------------------------------------ sub-pixel positions (reading R28; oracle/subpixel.py)
def test_subpixel_shift_closed_form_roll_and_adjoint(oracle_mod):
    from oracle import subpixel
    n = 16
    yy, xx = np.mgrid[0:n, 0:n]
    dy, dx = 0.3, 0.85
    for ay, ax in [(1, 0), (0, 1), (3, -5), (-7, 2)]:                     # a Fourier mode moved by (dy, dx): the closed form
        f = np.exp(2j * np.pi * (ay * yy + ax * xx) / n)
        want = np.exp(2j * np.pi * (ay * (yy - dy) + ax * (xx - dx)) / n)
        assert np.allclose(subpixel.shift(f, dy, dx), want, atol=1e-12)
    f = crandn(2, n, n)
    g = subpixel.shift(subpixel.shift(f, dy, 0.0), 1 - dy, 0.0)           # dy then 1 - dy = one whole row DOWN (+y), columns untouched
    assert np.allclose(g, np.roll(f, 1, axis=-2), atol=1e-12)
    g = subpixel.shift(subpixel.shift(f, 0.0, dx), 0.0, 1 - dx)
    assert np.allclose(g, np.roll(f, 1, axis=-1), atol=1e-12)
    assert np.allclose(subpixel.shift(f, 0.0, 0.0), f, atol=1e-13)
    a, b = crandn(n, n), crandn(n, n)                                      # S_{-d} is the adjoint of S_d
    assert np.isclose(np.vdot(b, subpixel.shift(a, dy, dx)), np.vdot(subpixel.shift(b, -dy, -dx), a), atol=1e-10)


@pytest.mark.parametrize("k,dtype,pbound", [(1, np.float32, 0.0), (2, np.uint16, 0.4)])
def test_subpixel_zero_shift_is_the_ordinary_minibatch_step(oracle_mod, k, dtype, pbound):
    """delta_j = 0 for every frame: oracle/subpixel.py (numpy) must give what orc_minibatch_step (C) gives -- masks, relaxed
    projection, several modes, strided batches, probe update from iteration 1 on."""
    from oracle import subpixel
    s = synth.make_custom(16, 44, 4, 6, k=k, peak=3e3 if dtype == np.uint16 else None, dtype=dtype, seed=12, jitter=1)
    inten = s.intensities.copy()
    inten[3, 2, 5] = 65535 if dtype == np.uint16 else -1.0                 # a masked pixel (R3)
    par = dict(batch_size=5, probe_start=1, pbound=pbound, alpha_obj=0.9, alpha_probe=0.7)
    O0 = s.obj0 * (1 + 0.05 * crandn(*s.obj0.shape))
    o = oracle_mod.Oracle(O0, s.probe0, s.pos, inten, par).iterate("EPIE_MB", 3)
    q = subpixel.SubpixelOracle(O0, s.probe0, s.pos, np.zeros((len(s.pos), 2)), inten, par).iterate(3)
    assert rel(q.O, o.O) < 1e-11 and rel(q.P, o.P) < 1e-11
    assert np.allclose(q.err, o.err, rtol=1e-10)


def test_subpixel_common_shift_equals_a_preshifted_probe(oracle_mod):
    """Every frame shifted by the same delta: the object step must be the ordinary (C oracle) step taken with the probe
    S_delta[P]; and with a huge regulariser the probe step reduces to alpha n_P / (delta_P max d_P), whose numerators must be
    related by the BACK-shift S_{-delta} (catches a forward shift, or none, in the probe term)."""
    from oracle import subpixel
    s = synth.make_custom(16, 44, 4, 6, k=2, seed=5, jitter=1)
    d = (0.35, 0.6)
    frac = np.tile(np.array(d), (len(s.pos), 1))
    O0 = s.obj0 * (1 + 0.05 * crandn(*s.obj0.shape))
    Ps = subpixel.shift(s.probe0, *d)
    big = 1e9
    par = dict(batch_size=0, probe_start=0, delta_probe=big, alpha_probe=big)
    o = oracle_mod.Oracle(O0, Ps, s.pos, s.intensities, par).iterate("EPIE_MB", 1)
    # The object regulariser is delta_O max_r sum_k |P_k|^2: of the UNSHIFTED probe in the sub-pixel step (R28), of the probe it is
    # given in the ordinary one.  The two runs differ only through that scalar, so it is matched through delta_obj.
    mo, mq = np.max(np.sum(np.abs(Ps) ** 2, 0)), np.max(np.sum(np.abs(s.probe0) ** 2, 0))
    par2 = dict(par, delta_obj=mo / mq)
    q = subpixel.SubpixelOracle(O0, s.probe0, s.pos, frac, s.intensities, par2).iterate(1)
    assert rel(q.O, o.O) < 1e-11
    dq, do = q.P - s.probe0, o.P - Ps                                      # alpha n_P / (d_P + delta_P max d_P) -> n_P / max d_P
    assert rel(dq, subpixel.shift(do, -d[0], -d[1])) < 1e-7
    assert rel(dq, subpixel.shift(do, d[0], d[1])) > 1e-2 and rel(dq, do) > 1e-2
    assert np.allclose(q.err, o.err, rtol=1e-10)


def test_subpixel_positions_matter_and_the_true_ones_fit_best(oracle_mod):
    """Data simulated (here, with numpy) from fractional positions: the ground truth is a fixed point of the sub-pixel step with
    zero error, and it is NOT one when the fractions are dropped."""
    from oracle import subpixel
    s = synth.make_custom(16, 44, 4, 6, k=1, seed=9, jitter=1)
    rng = np.random.default_rng(3)
    frac = rng.uniform(0, 1, (len(s.pos), 2))
    n = 16
    inten = np.empty((len(s.pos), n, n), np.float32)
    for j, (y, x) in enumerate(s.pos):
        inten[j] = np.abs(np.fft.fft2(subpixel.shift(s.probe_true, *frac[j])[0] * s.obj_true[y:y + n, x:x + n])) ** 2
    q = subpixel.SubpixelOracle(s.obj_true, s.probe_true, s.pos, frac, inten, dict(batch_size=4)).iterate(2)
    assert q.err[0] < 1e-12 and rel(q.O, s.obj_true) < 1e-6 and rel(q.P, s.probe_true) < 1e-6
    assert q.eval_error() < 1e-12
    z = subpixel.SubpixelOracle(s.obj_true, s.probe_true, s.pos, 0 * frac, inten, dict(batch_size=4)).iterate(1)
    assert z.err[0] > 1e-4
    z2 = subpixel.SubpixelOracle(s.obj_true, s.probe_true, s.pos, 0 * frac, inten)      # eval_error with zero fractions = the C oracle's
    assert np.isclose(z2.eval_error(), oracle_mod.Oracle(s.obj_true, s.probe_true, s.pos, inten).eval_error(), rtol=1e-10) and z2.eval_error() > 1e-4


@pytest.mark.parametrize("k,probe_start", [(1, 0), (3, 1)])
def test_subpixel_lsqml_zero_shift_is_the_ordinary_joint_step(oracle_mod, k, probe_start):
    """The LSQML-style joint step of oracle/subpixel.py with every fraction zero: objects, probes, error history AND the step
    lengths (a, b) of every batch must be those of orc_minibatch_step(LSQML), with and without the probe update."""
    from oracle import subpixel
    s = synth.make_custom(16, 44, 4, 6, k=k, seed=21, jitter=1)
    par = dict(batch_size=6, probe_start=probe_start, pbound=0.0, lsq_lambda=0.1)
    O0 = s.obj0 * (1 + 0.05 * crandn(*s.obj0.shape))
    o = oracle_mod.Oracle(O0, s.probe0, s.pos, s.intensities, par).iterate("LSQML", 3)
    q = subpixel.SubpixelOracle(O0, s.probe0, s.pos, np.zeros((len(s.pos), 2)), s.intensities, par).iterate(3, "LSQML")
    assert rel(q.O, o.O) < 1e-10 and rel(q.P, o.P) < 1e-10
    assert np.allclose(q.steps, o.steps, rtol=1e-9, atol=1e-14) and np.allclose(q.err, o.err, rtol=1e-10)
    assert any(b != 0 for _, b in q.steps) and (probe_start == 0 or q.steps[0][1] == 0.0)


def test_subpixel_lsqml_step_minimises_the_linearised_residual(oracle_mod):
    """With fractions: the (a, b) applied must be the Tikhonov-regularised least-squares solution of
    sum_jk || chi_jk - a P_jk dO_j - b S_delta_j[dP_k] O_j ||^2, found here by numpy's lstsq on the stacked real system."""
    from oracle import subpixel
    s = synth.make_custom(16, 44, 3, 7, k=2, seed=22, jitter=1)
    rng = np.random.default_rng(4)
    frac = rng.uniform(0, 1, (len(s.pos), 2))
    par = dict(oracle_mod.DEFAULTS, batch_size=0, probe_start=0, lsq_lambda=0.0)
    O0 = (s.obj0 * (1 + 0.05 * crandn(*s.obj0.shape))).astype(np.complex128)
    P0 = np.array(s.probe0, np.complex128)
    # the directions, from one ePIE-type step with unit steps and the probe updated: dO = O' - O, dP = P' - P
    Oe, Pe = O0.copy(), P0.copy()
    subpixel.epie_mb_step(Oe, Pe, s.pos, frac, s.intensities, np.arange(len(s.pos)), True, dict(par, alpha_obj=1.0, alpha_probe=1.0))
    dO, dP = Oe - O0, Pe - P0
    n = 16
    cols_u, cols_v, rhs = [], [], []
    for j, (y, x) in enumerate(s.pos):
        Pj = subpixel.shift(P0, *frac[j]); Oj = O0[y:y + n, x:x + n]
        psi = Pj * Oj[None]
        chi = np.fft.ifft2(oracle_mod.modulus_project(np.fft.fft2(psi), s.intensities[j], 0.0)[0]) - psi
        cols_u.append((Pj * dO[None, y:y + n, x:x + n]).ravel()); cols_v.append((subpixel.shift(dP, *frac[j]) * Oj[None]).ravel()); rhs.append(chi.ravel())
    u, v, c = np.concatenate(cols_u), np.concatenate(cols_v), np.concatenate(rhs)
    A = np.stack([np.concatenate([u.real, u.imag]), np.concatenate([v.real, v.imag])], 1)
    ab = np.linalg.lstsq(A, np.concatenate([c.real, c.imag]), rcond=None)[0]
    Ol, Pl, steps = O0.copy(), P0.copy(), []
    subpixel.epie_mb_step(Ol, Pl, s.pos, frac, s.intensities, np.arange(len(s.pos)), True, par, lsqml=True, steps_out=steps)
    assert np.allclose(steps[0], ab, rtol=1e-8)
    assert rel(Ol, O0 + ab[0] * dO) < 1e-12 and rel(Pl, P0 + ab[1] * dP) < 1e-12


def test_subpixel_dm_pins(oracle_mod):
    """DM with sub-pixel positions (oracle/subpixel.py dm_iteration): zero fractions = orc_dm_iteration (K = 2, relaxed projection,
    probe update from iteration 1, exit waves included); a common shift with the probe frozen = the ordinary DM run with the
    pre-shifted probe; data simulated at fractional positions keep the ground truth fixed with zero error (probe frozen), and do not
    when the fractions are dropped."""
    from oracle import subpixel
    s = synth.make_custom(16, 44, 4, 6, k=2, peak=3e3, dtype=np.uint16, seed=31, jitter=1)
    par = dict(probe_start=1, pbound=0.4)
    O0 = s.obj0 * (1 + 0.05 * crandn(*s.obj0.shape))
    o = oracle_mod.Oracle(O0, s.probe0, s.pos, s.intensities, par).iterate("DM", 4)
    q = subpixel.SubpixelOracle(O0, s.probe0, s.pos, np.zeros((len(s.pos), 2)), s.intensities, par).iterate(4, "DM")
    assert rel(q.O, o.O) < 1e-11 and rel(q.P, o.P) < 1e-11 and rel(q.psi, o.psi) < 1e-11 and np.allclose(q.err, o.err, rtol=1e-10)
    d = (0.4, 0.75)
    frac = np.tile(np.array(d), (len(s.pos), 1))
    Ps = subpixel.shift(s.probe0, *d)
    frozen = dict(probe_start=10 ** 9, pbound=0.0)
    o = oracle_mod.Oracle(O0, Ps, s.pos, s.intensities, frozen)
    q = subpixel.SubpixelOracle(O0, s.probe0, s.pos, frac, s.intensities, frozen)
    q.eps_O = o.eps_O                                                       # (R5 takes eps_O from the probe it is given: matched)
    o.iterate("DM", 3); q.iterate(3, "DM")
    assert rel(q.O, o.O) < 1e-11 and rel(q.psi, o.psi) < 1e-11
    s1 = synth.make_custom(16, 44, 4, 6, k=1, seed=9, jitter=1)
    rng = np.random.default_rng(3)
    fr = rng.uniform(0, 1, (len(s1.pos), 2))
    inten = np.stack([np.abs(np.fft.fft2(subpixel.shift(s1.probe_true, *fr[j])[0] * s1.obj_true[y:y + 16, x:x + 16])) ** 2
                      for j, (y, x) in enumerate(s1.pos)]).astype(np.float32)
    q = subpixel.SubpixelOracle(s1.obj_true, s1.probe_true, s1.pos, fr, inten, dict(probe_start=10 ** 9)).iterate(2, "DM")
    assert q.err[-1] < 1e-12 and rel(q.O, s1.obj_true) < 1e-6           # (probe frozen: with d_P = sum |O_j|^2 unshifted the probe
    z = subpixel.SubpixelOracle(s1.obj_true, s1.probe_true, s1.pos, 0 * fr, inten, dict(probe_start=10 ** 9)).iterate(2, "DM")
    assert z.err[-1] > 1e-4                                                # update keeps the truth only approximately, see the docstring)
