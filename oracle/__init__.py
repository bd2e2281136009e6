"""ctypes driver of the CPU oracle (oracle/ptycho_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: imported only by tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py.  Nothing here imports the CUDA package.

The arithmetic lives in the C file; this module only (a) compiles it with gcc, (b) keeps the
reconstruction state (O, P, psi, iteration counter, error history) between calls the way the
paper's step mode does (init / step / fetch at any iteration), and (c) sequences
iterations and minibatches (SURVEY.md 8(c) readings R8, R20: strided batches, one iteration = one
pass over all positions; P:L52 probe_start).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
ALG = {"EPIE_MB": 0, "DM": 1, "LSQML": 2, "LSQML_PF": 3}
DEFAULTS = dict(batch_size=0, probe_start=0, delta_blend=1e-2, delta_obj=1.0, delta_probe=1.0,
                alpha_obj=1.0, alpha_probe=1.0, lsq_lambda=0.1, pbound=0.0, batch_order=None, dm_sweeps=0)


def build(force: bool = False) -> None:
    """gcc the oracle in double (liboracle_f64.so) and float (liboracle_f32.so)."""
    src = os.path.join(_HERE, "ptycho_oracle.c")
    for name, flag in (("f64", []), ("f32", ["-DORACLE_FLOAT"])):
        out = os.path.join(_HERE, f"liboracle_{name}.so")
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
            subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", *flag,
                                   src, "-o", out, "-lm"])


_libs: dict = {}


def lib(precision: str = "f64"):
    if precision not in _libs:
        build()
        l = C.CDLL(os.path.join(_HERE, f"liboracle_{precision}.so"))
        l.orc_modulus_project.restype = C.c_double if precision == "f64" else C.c_float
        for f in ("orc_sum_intensity", "orc_eval_error_num", "orc_dm_iteration", "orc_minibatch_step", "orc_minibatch_step_perframe"):
            getattr(l, f).restype = C.c_double
        _libs[precision] = l
    return _libs[precision]


def _types(precision):
    return (np.float64, np.complex128, C.c_double) if precision == "f64" else (np.float32, np.complex64, C.c_float)


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def to_real_intensity(inten: np.ndarray, rdt) -> np.ndarray:
    """uint16 65535 or negative float = masked (R3) -> negative value in the oracle's real type."""
    out = inten.astype(rdt)
    if inten.dtype == np.uint16:
        out[inten == 65535] = -1
    return np.ascontiguousarray(out)


def fft2(a: np.ndarray, inverse: bool = False, precision="f64") -> np.ndarray:
    rdt, cdt, _ = _types(precision)
    x = np.ascontiguousarray(a, cdt).copy()
    lib(precision).orc_fft2(C.c_int(x.shape[-1]), _p(x), C.c_int(int(inverse)))
    return x


def dft2_naive(a: np.ndarray, inverse: bool = False, precision="f64") -> np.ndarray:
    rdt, cdt, _ = _types(precision)
    x = np.ascontiguousarray(a, cdt)
    out = np.empty_like(x)
    lib(precision).orc_dft2_naive(C.c_int(x.shape[-1]), _p(x), _p(out), C.c_int(int(inverse)))
    return out


def modulus_project(phi: np.ndarray, inten: np.ndarray, pbound: float = 0.0, precision="f64"):
    """phi (K, n, n), inten (n, n) -> (phi', error term)."""
    rdt, cdt, cr = _types(precision)
    x = np.ascontiguousarray(phi, cdt)
    out = np.empty_like(x)
    it = to_real_intensity(inten, rdt)
    e = lib(precision).orc_modulus_project(C.c_int(x.shape[-1]), C.c_int(x.shape[0]), _p(x), _p(it),
                                           cr(pbound), _p(out))
    return out, float(e)


def batches(n_pos: int, batch_size: int, order=None):
    """R8: strided batches (n_b = ceil(J/B); batch b = {j : j mod n_b = b}) or, with a caller
    permutation, consecutive runs of B of it."""
    if batch_size <= 0 or batch_size >= n_pos:
        base = np.arange(n_pos, dtype=np.int32) if order is None else np.asarray(order, np.int32)
        return [base]
    if order is not None:
        order = np.asarray(order, np.int32)
        return [order[s:s + batch_size] for s in range(0, n_pos, batch_size)]
    nb = -(-n_pos // batch_size)
    return [np.arange(b, n_pos, nb, dtype=np.int32) for b in range(nb)]


class Oracle:
    """State + sequencing around the C oracle; mirrors the C-ABI semantics of include/ptycho_b200.h."""

    def __init__(self, obj, probe, pos, intensities, params=None, precision="f64", keep_revised=False):
        self.precision = precision
        self.rdt, self.cdt, self.cr = _types(precision)
        self.l = lib(precision)
        self.par = dict(DEFAULTS)
        self.par.update(params or {})
        self.O = np.ascontiguousarray(obj, self.cdt).copy()
        self.P = np.ascontiguousarray(probe, self.cdt).copy()
        if self.P.ndim == 2:
            self.P = self.P[None]
        self.pos = np.ascontiguousarray(pos, np.int32)
        self.I = to_real_intensity(intensities, self.rdt)
        self.K, self.n = self.P.shape[0], self.P.shape[-1]
        self.J = self.pos.shape[0]
        self.H, self.W = self.O.shape
        assert self.I.shape == (self.J, self.n, self.n)
        d = self.par["delta_blend"]
        self.eps_O = d * float(np.max(np.sum(np.abs(self.P) ** 2, axis=0)))       # R5
        self.eps_P = d * self.J * float(np.max(np.abs(self.O) ** 2))
        self.sum_I = float(self.l.orc_sum_intensity(C.c_long(self.I.size), _p(self.I)))
        self.psi = None
        self.t = 0
        self.err: list[float] = []
        self.steps: list[tuple[float, float]] = []
        self.keep_revised = keep_revised
        self.revised = None

    def _dims(self):
        return [C.c_int(v) for v in (self.H, self.W, self.n, self.K)]

    def init_exit_waves(self):
        """psi_j = P O_j (R4 initial psi)."""
        n = self.n
        self.psi = np.empty((self.J, self.K, n, n), self.cdt)
        for j, (y, x) in enumerate(self.pos):
            self.psi[j] = self.P * self.O[None, y:y + n, x:x + n]

    def eval_error(self) -> float:
        num = self.l.orc_eval_error_num(*self._dims(), C.c_int(self.J), _p(self.O), _p(self.P),
                                        _p(self.pos), _p(self.I))
        return float(num) / (self.sum_I if self.sum_I > 0 else 1.0)

    def iterate(self, alg: str, n_iters: int = 1):
        p = self.par
        for _ in range(n_iters):
            upd = int(self.t >= p["probe_start"])
            rev = None
            if self.keep_revised:
                rev = np.empty((self.J, self.K, self.n, self.n), self.cdt)
            if alg == "DM":
                if self.psi is None:
                    self.init_exit_waves()
                sweeps = int(p["dm_sweeps"])
                # dm_sweeps = 0: reading R4 (lagged probe sums, one pass).  dm_sweeps = n >= 1: the textbook sequential overlap
                # projection: Fourier step and object from the new psi (probe untouched), then the probe from the
                # same psi and the NEW object; n - 1 more object/probe sweeps.
                num = self.l.orc_dm_iteration(*self._dims(), C.c_int(self.J), _p(self.O), _p(self.P),
                                              _p(self.psi), _p(self.pos), _p(self.I), self.cr(self.eps_O),
                                              self.cr(self.eps_P), C.c_int(upd if sweeps == 0 else 0), self.cr(p["pbound"]), _p(rev))
                for sw in range(sweeps):
                    if sw > 0:
                        self.l.orc_object_from_waves(*self._dims(), C.c_int(self.J), _p(self.O), _p(self.P), _p(self.psi),
                                                     _p(self.pos), self.cr(self.eps_O))
                    if upd:
                        self.l.orc_probe_from_waves(*self._dims(), C.c_int(self.J), _p(self.O), _p(self.P), _p(self.psi),
                                                    _p(self.pos), self.cr(self.eps_P))
            else:
                self.psi = None
                num = 0.0
                for fr in batches(self.J, p["batch_size"], p["batch_order"]):
                    fr = np.ascontiguousarray(fr, np.int32)
                    if alg == "LSQML_PF":                      # per-frame step lengths; steps: one pair per frame
                        stf = np.zeros((len(fr), 2))
                        num += self.l.orc_minibatch_step_perframe(
                            *self._dims(), _p(self.O), _p(self.P), _p(self.pos), _p(self.I), _p(fr), C.c_int(len(fr)), C.c_int(upd),
                            self.cr(p["delta_obj"]), self.cr(p["delta_probe"]), self.cr(p["lsq_lambda"]), self.cr(p["pbound"]), _p(stf))
                        self.steps += [tuple(v) for v in stf]
                        continue
                    st = (C.c_double * 2)()
                    rb = np.empty((len(fr), self.K, self.n, self.n), self.cdt) if rev is not None else None
                    num += self.l.orc_minibatch_step(
                        C.c_int(ALG[alg]), *self._dims(), _p(self.O), _p(self.P), _p(self.pos), _p(self.I),
                        _p(fr), C.c_int(len(fr)), C.c_int(upd), self.cr(p["alpha_obj"]),
                        self.cr(p["alpha_probe"]), self.cr(p["delta_obj"]), self.cr(p["delta_probe"]),
                        self.cr(p["lsq_lambda"]), self.cr(p["pbound"]), st, _p(rb))
                    self.steps.append((st[0], st[1]))
                    if rev is not None:
                        rev[fr] = rb
            self.revised = rev
            self.err.append(float(num) / (self.sum_I if self.sum_I > 0 else 1.0))
            self.t += 1
        return self


# --------------------------------------------------------------------------------------------------
# Frame preparation (centre, crop, threshold, saturation from the bit depth).
# TEST INFRASTRUCTURE like the rest of this package.  The definition written out: a centred crop of n x n
# pixels around (cy, cx), the noise threshold, the saturation mask, then numpy's ifftshift to put the centre
# pixel at [0, 0] (reading R1: FFT order).  Pinned in tests/test_oracle_pins.py against index arithmetic done by
# hand on a 6 x 6 example and against the fftshift/ifftshift involution.
def prepare_frames(raw, center, n, threshold=0.0, saturation=0.0, out_dtype=np.uint16, rot90=0, frame_scale=None):
    """rot90 = k ("the rotation angles of the diffraction patterns"; multiples of 90 degrees only, R23): the
    pattern is rotated counter-clockwise by k quarter turns about the centre pixel before the crop -- written here as numpy.rot90
    of a window that has the centre pixel in its middle.  frame_scale ("diffraction pattern normalization", R24): one
    factor per frame, applied to the counts that survive the threshold; masks are decided on the raw counts."""
    raw = np.asarray(raw)
    assert raw.ndim == 3 and n % 2 == 0
    f, dh, dw = raw.shape
    cy, cx = int(center[0]), int(center[1])
    h = n // 2
    if rot90 % 4:
        # window of (2n + 1)^2 pixels centred on (cy, cx), outside the detector = masked; rotate it; go on with the rotated window
        m = n
        big = np.full((f, 2 * m + 1, 2 * m + 1), 65535 if raw.dtype == np.uint16 else -1, raw.dtype)
        for iy in range(2 * m + 1):
            sy = cy - m + iy
            if 0 <= sy < dh:
                for ix in range(2 * m + 1):
                    sx = cx - m + ix
                    if 0 <= sx < dw:
                        big[:, iy, ix] = raw[:, sy, sx]
        raw, (cy, cx) = np.rot90(big, rot90 % 4, axes=(1, 2)), (m, m)
        dh = dw = 2 * m + 1
    val = np.zeros((f, n, n), np.float64)
    masked = np.ones((f, n, n), bool)                      # outside the detector: masked
    for iy in range(n):                                    # plain loops over the crop window (slow, obvious)
        sy = cy - h + iy
        if sy < 0 or sy >= dh:
            continue
        for ix in range(n):
            sx = cx - h + ix
            if sx < 0 or sx >= dw:
                continue
            v = raw[:, sy, sx].astype(np.float64)
            m = (v == 65535) if raw.dtype == np.uint16 else (v < 0)     # already the sentinel (R3)
            if saturation > 0:
                m = m | (v >= np.float32(saturation))
            if threshold > 0:
                v = np.where(v < np.float32(threshold), 0.0, v)
            if frame_scale is not None:
                v = (v.astype(np.float32) * np.asarray(frame_scale, np.float32)).astype(np.float64)   # fp32 product, like any fp32 path
            val[:, iy, ix] = v
            masked[:, iy, ix] = m
    val = np.fft.ifftshift(val, axes=(1, 2))               # centre pixel (index h) -> index 0
    masked = np.fft.ifftshift(masked, axes=(1, 2))
    if np.dtype(out_dtype) == np.uint16:
        out = np.minimum(np.rint(val), 65534).astype(np.uint16)
        out[masked] = 65535
    else:
        out = val.astype(np.float32)
        out[masked] = -1.0
    return out


# --------------------------------------------------------------------------------------------------
# Probe-mode orthogonalisation (reading R26; "several probe modes").  TEST INFRASTRUCTURE.
# The K modes are mixed by the unitary that diagonalises their Gram matrix G_ij = sum_r P_i(r) conj(P_j(r)): P' = V^H P with
# G = V diag(lambda) V^H, lambda descending (numpy.linalg.eigh is the library step).  Each eigenvector's phase is fixed by making its
# largest-magnitude component real and positive.  sum_k |P'_k(r)|^2 = sum_k |P_k(r)|^2 at every pixel, so the model intensities do not
# change; the same mixing applied to stored exit waves keeps them consistent.
def mode_mixing_matrix(P):
    K = P.shape[0]
    flat = np.asarray(P, np.complex128).reshape(K, -1)
    G = flat @ flat.conj().T
    lam, V = np.linalg.eigh(G)
    order = np.argsort(-lam, kind="stable")
    V = V[:, order]
    for m in range(K):
        i = int(np.argmax(np.abs(V[:, m])))
        V[:, m] *= np.exp(-1j * np.angle(V[i, m]))
    return V.conj().T                                      # U = V^H: P' = U P


def orthogonalize_modes(P, psi=None):
    U = mode_mixing_matrix(P)
    P2 = np.tensordot(U, np.asarray(P, np.complex128), axes=(1, 0))
    if psi is None:
        return P2
    return P2, np.einsum("mk,jkyx->jmyx", U, np.asarray(psi, np.complex128))
